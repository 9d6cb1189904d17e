// coils_h.cuh -- multi-coil receive on tcgen05 with FP16 operands (kind::f16, K = 16): half the instructions of the
// 3xTF32 kernel of coils_tc.cuh for the same contraction
//     S[n][c] = sum_i C[n][i] * W[i][c]        (reading C1; [samples x spins] x [spins x coils], complex)
// and the same structure: a generator thread owns one sample (one TMEM lane), evaluates its contributions from 8 spins,
// writes them into TENSOR MEMORY as the A operand (tcgen05.st), B tiles (the weights) arrive by TMA, accumulators in
// TMEM, one control thread issues the MMAs.  What changes is the arithmetic of the operands.  A tcgen05.mma of this
// shape costs ~74 clocks whatever N and K, so the instruction count decides:
//   * K = 16 halves per instruction: the complex product is stacked along K, A = [Cr(8 spins) | Ci(8 spins)],
//     B = [[Wr, Wi], [-Wi, Wr]], so ONE instruction covers 8 spins completely (two with TF32: K = 8).
//   * Every value is split into two FP16 pieces x s = hi + lo (hi = fp16(x s), lo = fp16(x s - hi): 22 significant
//     bits, what hi + lo TF32 pieces carry), and hi x [B hi | B lo] is one instruction of N = 4 NC with the two B tiles
//     side by side along N; lo x B hi is the second.  2 instructions per 8 spins and 128 samples (TF32: 4).
//   * FP16 has 5 exponent bits: both operands are scaled by powers of two taken from measured maxima (coil_scales_kernel:
//     the largest |M| a spin can reach, max(M0, |M(0)|), and the largest weight component), so that the largest value
//     sits in [2^13, 2^14).  A piece is then exact to max(2^-11 of itself, 3e-8) -- the FP16 subnormal spacing, 2^-38 of
//     the largest value --, so lo needs no scale of its own: it goes subnormal only for values below 2^-17 of the
//     largest, where the absolute error stays at 3e-8.  hi x hi lands in accumulator columns [0, 2 NC), the cross
//     products in [2 NC, 4 NC); the epilogue returns (hh + mix) / (s_A s_B).  lo x lo (2^-22 relative) is dropped, as
//     in 3xTF32.
// B operand layout (no swizzle, K-major): 8-row x 16-byte core matrices (8 halves per row), contiguous 128 B each;
//     byte offset of element (row n, k) = (n / 8) * 256 + (k / 8) * 128 + (n % 8) * 16 + (k % 8) * 2,  rows [B hi | B lo]
// A operand in TMEM: row m = lane m, K = 16 halves = 8 consecutive 32-bit columns (k = 2 j in the low half of column j);
// a stage (16 spins) = 2 groups x [hi (8 columns) | lo (8 columns)] = 32 columns, after the 4 NC accumulator columns
// (up to 32 coils per pass take the wide instruction), as many stages as the CTA's 256 columns hold (at most 7).
#pragma once
#include <cuda_fp16.h>

#include "coils_tc.cuh"

namespace bloch {

constexpr int kScalMMax = 6;          // scal[]: bound on |M| of any spin (float bits), coil_scales_kernel
constexpr int kScalWMax = 7;          // scal[]: largest |re|, |im| of a coil weight
constexpr int kHAStageCols = kTcGroups * 16;   // per 8-spin group: hi (8 columns) | lo (8 columns)
// TMEM (256 columns per CTA, two CTAs per SM): 4 NC accumulator columns, the rest A stages: 7 / 6 / 4 for 8 / 16 / 32 coils
__host__ __device__ constexpr int h_dcols(int nc) { return 4 * nc; }
__host__ __device__ constexpr int h_astages(int nc) { return (kTcCols - 4 * nc) / kHAStageCols < 7 ? (kTcCols - 4 * nc) / kHAStageCols : 7; }
constexpr int kHSlots = 8;
__host__ __device__ constexpr int h_btile(int nc) { return 4 * nc * 32; }   // per 8-spin group: 4 NC rows x 16 halves
__host__ __device__ constexpr int h_slot(int nc) { return kTcStageSpins * 32 + kTcGroups * h_btile(nc); }
__host__ __device__ constexpr size_t h_smem(int nc) { return kHSlots * (size_t)h_slot(nc) + 256; }

// 2^(13 - floor(log2 vmax)): the largest scaled value lies in [2^13, 2^14)
__device__ __forceinline__ float h_scale(unsigned vmax_bits) {
    const int e = (int)((vmax_bits >> 23) & 0xffu);  // biased exponent; 0 (zero / denormal maximum): no scaling
    if (e == 0 || e == 255) return 1.0f;
    const int se = min(max(127 + 13 - (e - 127), 1), 254);
    return __uint_as_float((unsigned)se << 23);
}

// maxima that fix the operand scales: every |Cr|, |Ci| <= |Mxy| <= max(M0, |M(0)|) (relaxation only shrinks the
// excess over M0), every B entry is a weight component.  Integer max of float bit patterns: order-independent.
__global__ void __launch_bounds__(256)
coil_scales_kernel(int n, const float4 *__restrict__ Cc, const float4 *__restrict__ S, const float2 *__restrict__ coil,
                   long long n_w, unsigned *__restrict__ scal) {
    float m = 0.f, w = 0.f;
    const long long stride = (long long)gridDim.x * blockDim.x, t0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    for (long long i = t0; i < n; i += stride) {
        const float4 s = S[i];
        m = fmaxf(m, fmaxf(fabsf(Cc[i].z), sqrtf(fmaf(s.x, s.x, fmaf(s.y, s.y, s.z * s.z)))));
    }
    for (long long j = t0; j < n_w; j += stride) {
        const float2 c = coil[j];
        w = fmaxf(w, fmaxf(fabsf(c.x), fabsf(c.y)));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
        w = fmaxf(w, __shfl_xor_sync(0xffffffffu, w, o));
    }
    if ((threadIdx.x & 31) == 0) {
        atomicMax(scal + kScalMMax, __float_as_uint(fminf(fmaxf(m, 0.f), 3.0e38f)));
        atomicMax(scal + kScalWMax, __float_as_uint(fminf(fmaxf(w, 0.f), 3.0e38f)));
    }
}

// Block-start state in polar form for the generators: (|Mxy|, arg Mxy, Mz, e2).  A contribution is then
// |Mxy| e^{-tau/T2} (cos, sin)(theta + arg Mxy): the argument rides in the phase's FMA chain for free and the complex
// rotation (6 instructions per (spin, sample)) becomes 3 multiplies.  One small launch per block.
__global__ void __launch_bounds__(256)
coil_polar_kernel(int n, const float4 *__restrict__ S, float4 *__restrict__ Sp) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float4 s = S[i];
    Sp[i] = make_float4(hypotf(s.x, s.y), atan2f(s.y, s.x), s.z, s.w);
}

__device__ __forceinline__ void h_split(float x, __half &hi, __half &lo) {
    hi = __float2half_rn(x);
    lo = __float2half_rn(x - __half2float(hi));
}

// Weights -> B tiles.  Bt[pass][group][4 NC rows x 16 halves], group = spin / 8 over the spins padded to a multiple of 16.
template <int NC>
__global__ void __launch_bounds__(256)
pack_coils_h_kernel(int n, int n_pad, int n_coils, const float2 *__restrict__ coil, const unsigned *__restrict__ scal,
                    unsigned char *__restrict__ Bt) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;  // spin (padded range)
    const int pass = blockIdx.y;
    if (i >= n_pad) return;
    const float sB = h_scale(scal[kScalWMax]);
    unsigned char *grp = Bt + ((size_t)pass * (n_pad / 8) + (size_t)(i / 8)) * h_btile(NC);
    const int k = i & 7;
    for (int c = 0; c < NC; ++c) {
        const int cc = pass * NC + c;
        float2 w = make_float2(0.f, 0.f);
        if (i < n && cc < n_coils) w = coil[(size_t)cc * n + i];
        // stacked B: rows n < NC give the real part of the sum, n >= NC the imaginary part; k < 8 meets Cr, k >= 8 Ci
        const float vals[2][2] = {{w.x, -w.y}, {w.y, w.x}};  // [row block re / im][k block cr / ci]
        for (int rb = 0; rb < 2; ++rb)
            for (int kb = 0; kb < 2; ++kb) {
                __half hi, lo;
                h_split(vals[rb][kb] * sB, hi, lo);
                const int nn = c + NC * rb, kk = k + 8 * kb;
                const int off_h = (nn / 8) * 256 + (kk / 8) * 128 + (nn % 8) * 16 + (kk % 8) * 2;
                const int nl = nn + 2 * NC;
                const int off_l = (nl / 8) * 256 + (kk / 8) * 128 + (nl % 8) * 16 + (kk % 8) * 2;
                *reinterpret_cast<__half *>(grp + off_h) = hi;
                *reinterpret_cast<__half *>(grp + off_l) = lo;
            }
    }
}

// instruction descriptor: D = F32, A = B = F16, both K-major, N columns, M = 128
__host__ __device__ constexpr uint32_t h_idesc(int n) {
    return (1u << 4) | ((uint32_t)(n >> 3) << 17) | ((128u >> 4) << 24);
}

__device__ __forceinline__ void h_mma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t"
        "}\n" ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}

template <int NC>
__global__ void __launch_bounds__(kTcThreads, 2)
signal_coils_h_kernel(const float4 *__restrict__ recs, int n_pts, const float4 *__restrict__ A,
                      const float4 *__restrict__ S /* polar states, coil_polar_kernel */,
                      const unsigned char *__restrict__ Bt /* this pass */,
                      int n_spins, int spins_per_chunk /* multiple of 16 */, const unsigned *__restrict__ scal,
                      float2 *__restrict__ partial /* [NC][chunks][n_pts] */) {
    constexpr int kBTile = h_btile(NC), kSlotBytes = h_slot(NC);
    constexpr uint32_t kIdescW = h_idesc(4 * NC), kIdescN = h_idesc(2 * NC);
    constexpr int kHDCols = h_dcols(NC), kHAStages = h_astages(NC);
    static_assert(kHDCols + kHAStages * kHAStageCols <= kTcCols && kHAStages >= 2, "TMEM columns");
    extern __shared__ __align__(1024) unsigned char smem[];
    unsigned char *slots = smem;                                    // [kHSlots][spin A (256 B) | spin S (256 B) | B tiles]
    uint64_t *full = reinterpret_cast<uint64_t *>(slots + kHSlots * kSlotBytes);    // [kHSlots] TMA landed
    uint64_t *a_full = full + kHSlots;                                              // [kHAStages] generators done with an A stage
    uint64_t *mma_done = a_full + kHAStages;                                        // [kHAStages] tensor core done with an A stage
    uint64_t *all_done = mma_done + kHAStages;                                      // every MMA of the CTA has completed
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(all_done + 1);
    const int tid = threadIdx.x, warp = tid >> 5;
    const int s0 = blockIdx.y * spins_per_chunk;
    const int s1 = min(n_spins, s0 + spins_per_chunk);
    const int n_stages = (s1 - s0 + kTcStageSpins - 1) / kTcStageSpins;
    auto issue = [&](int st) {  // control thread: stage st -> ring slot st % kHSlots
        const int sl = st % kHSlots;
        unsigned char *dst = slots + sl * kSlotBytes;
        const int base = s0 + st * kTcStageSpins;
        const uint32_t cnt = (uint32_t)min(kTcStageSpins, s1 - base);
        mbar_expect_tx(&full[sl], cnt * 32u + (uint32_t)(kTcGroups * kBTile));
        bulk_g2s(dst, A + base, cnt * 16u, &full[sl]);
        bulk_g2s(dst + kTcStageSpins * 16, S + base, cnt * 16u, &full[sl]);
        bulk_g2s(dst + kTcStageSpins * 32, Bt + (size_t)(base / 8) * kBTile, (uint32_t)(kTcGroups * kBTile), &full[sl]);
    };
    // the spin-record area of every ring slot starts as zeros (a ragged last stage must hold finite values; its B rows
    // are zero, pack_coils_h_kernel)
    for (int k = tid; k < kHSlots * kTcStageSpins * 2; k += kTcThreads)
        reinterpret_cast<float4 *>(slots + (k / (kTcStageSpins * 2)) * kSlotBytes)[k % (kTcStageSpins * 2)] = make_float4(0.f, 0.f, 0.f, 0.f);
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    if (tid == 0) {
        for (int k = 0; k < kHSlots; ++k) mbar_init(&full[k], 1);
        for (int k = 0; k < kHAStages; ++k) {
            mbar_init(&a_full[k], 128);  // the four generator warps of the stage's set
            mbar_init(&mma_done[k], 1);
        }
        mbar_init(all_done, 1);
        mbar_init_fence();
    }
    if (warp == 0) {
        __syncwarp();
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "n"(kTcCols) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = *tmem_slot;

    if (warp == kTcGenWarps) {
        // ------------------------------------------------------------ control warp: TMA ring + MMA issue (lane 0)
        if (tid == 32 * kTcGenWarps) {
            for (int st = 0; st < kHSlots - 1 && st < n_stages; ++st) issue(st);
            for (int st = 0; st < n_stages; ++st) {
                const int ab = st % kHAStages, sl = st % kHSlots;
                mbar_wait(&a_full[ab], (uint32_t)((st / kHAStages) & 1));
                mbar_wait(&full[sl], (uint32_t)((st / kHSlots) & 1));
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const uint32_t a0 = tmem + (uint32_t)(kHDCols + ab * kHAStageCols);
                const uint32_t b0 = smem_u32(slots + sl * kSlotBytes + kTcStageSpins * 32);
#pragma unroll
                for (int gq = 0; gq < kTcGroups; ++gq) {
                    const uint32_t ag = a0 + gq * 16, bg = b0 + gq * kBTile;  // A parts: columns +0 hi, +8 lo
                    const uint32_t first = (st == 0 && gq == 0) ? 0u : 1u;
                    h_mma_ts(tmem, ag + 0, tc_desc(bg), kIdescW, first);          // hi x [B hi | B lo] -> [hh | hl]
                    h_mma_ts(tmem + 2 * NC, ag + 8, tc_desc(bg), kIdescN, 1u);    // lo x B hi          ->      [lh]
                }
                asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(&mma_done[ab])) : "memory");
                if (st + kHSlots - 1 < n_stages) {  // the slot of stage st + kHSlots - 1 held stage st - 1
                    if (st >= 1) mbar_wait(&mma_done[(st - 1) % kHAStages], (uint32_t)(((st - 1) / kHAStages) & 1));
                    issue(st + kHSlots - 1);
                }
            }
            asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(all_done)) : "memory");
        }
    } else {
        // ------------------------------------------------------------ generator warps: one sample (TMEM lane) per thread
        const int set = warp >> 2;
        const int row = 32 * (warp & 3) + (tid & 31);
        const uint32_t lane_addr = tmem + ((uint32_t)(32 * (warp & 3)) << 16);
        float4 r = make_float4(0.f, 0.f, 0.f, 0.f);
        {
            const int p = blockIdx.x * kTcM + row;
            if (p < n_pts) r = recs[p];
        }
        const float kx = r.x, ky = r.y, kz = r.z, tau = r.w;
        const float sA = h_scale(scal[kScalMMax]);
        const float lsA = (float)((int)((__float_as_uint(sA) >> 23) & 0xffu) - 127);  // log2 s_A, folded into the decay's exponent
        for (int st = set; st < n_stages; st += kTcGenWarps / 4) {
            const int ab = st % kHAStages, sl = st % kHSlots;
            if (st >= kHAStages) {  // the MMAs that read this A stage kHAStages stages ago are complete
                mbar_wait(&mma_done[ab], (uint32_t)(((st / kHAStages) - 1) & 1));
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            }
            mbar_wait(&full[sl], (uint32_t)((st / kHSlots) & 1));
            const unsigned char *slot = slots + sl * kSlotBytes;
            const float4 *spA = reinterpret_cast<const float4 *>(slot);
            const float4 *spS = reinterpret_cast<const float4 *>(slot + kTcStageSpins * 16);
            uint32_t v[32];  // per group: [hi: cr pairs (4) ci pairs (4) | lo: cr pairs (4) ci pairs (4)]
#pragma unroll
            for (int gq = 0; gq < kTcGroups; ++gq) {
#pragma unroll
                for (int m = 0; m < 4; ++m) {
                    float cr[2], ci[2];
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const int sp = 8 * gq + 2 * m + h;
                        const float4 a = spA[sp];
                        const float4 sv = spS[sp];  // polar: (|Mxy|, arg Mxy, Mz, e2 = -log2(e)/T2)
                        const float th = fmaf(kx, a.x, fmaf(ky, a.y, fmaf(kz, a.z, fmaf(tau, a.w, sv.y))));  // radians
                        const float sn = __sinf(th), cs = __cosf(th);
                        const float me = sv.x * ex2_approx(fmaf(tau, sv.w, lsA));  // s_A |Mxy| exp(-tau / T2)
                        cr[h] = me * cs;
                        ci[h] = me * sn;
                    }
                    const __half2 hr = __floats2half2_rn(cr[0], cr[1]), hi_ = __floats2half2_rn(ci[0], ci[1]);
                    const float2 fr = __half22float2(hr), fi = __half22float2(hi_);
                    const __half2 lr = __floats2half2_rn(cr[0] - fr.x, cr[1] - fr.y);
                    const __half2 li = __floats2half2_rn(ci[0] - fi.x, ci[1] - fi.y);
                    v[16 * gq + m] = *reinterpret_cast<const uint32_t *>(&hr);
                    v[16 * gq + 4 + m] = *reinterpret_cast<const uint32_t *>(&hi_);
                    v[16 * gq + 8 + m] = *reinterpret_cast<const uint32_t *>(&lr);
                    v[16 * gq + 12 + m] = *reinterpret_cast<const uint32_t *>(&li);
                }
            }
            tc_st32(lane_addr + (uint32_t)(kHDCols + ab * kHAStageCols), v);
            asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            mbar_arrive(&a_full[ab]);
        }
        // all MMAs complete -> epilogue (warps 0-3: TMEM lanes 32 w .. 32 w + 31 = sample rows)
        if (warp < 4) {
            float acc[2 * NC];
#pragma unroll
            for (int c = 0; c < 2 * NC; ++c) acc[c] = 0.f;
            if (n_stages > 0) {
                mbar_wait(all_done, 0u);
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const float inv = 1.0f / (sA * h_scale(scal[kScalWMax]));
#pragma unroll
                for (int c0 = 0; c0 < 2 * NC; c0 += 16) {
                    uint32_t hh[16], mx[16];
                    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                                 : "=r"(hh[0]), "=r"(hh[1]), "=r"(hh[2]), "=r"(hh[3]), "=r"(hh[4]), "=r"(hh[5]), "=r"(hh[6]), "=r"(hh[7]),
                                   "=r"(hh[8]), "=r"(hh[9]), "=r"(hh[10]), "=r"(hh[11]), "=r"(hh[12]), "=r"(hh[13]), "=r"(hh[14]), "=r"(hh[15])
                                 : "r"(lane_addr + (uint32_t)c0));
                    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                                 : "=r"(mx[0]), "=r"(mx[1]), "=r"(mx[2]), "=r"(mx[3]), "=r"(mx[4]), "=r"(mx[5]), "=r"(mx[6]), "=r"(mx[7]),
                                   "=r"(mx[8]), "=r"(mx[9]), "=r"(mx[10]), "=r"(mx[11]), "=r"(mx[12]), "=r"(mx[13]), "=r"(mx[14]), "=r"(mx[15])
                                 : "r"(lane_addr + (uint32_t)(2 * NC + c0)));
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                    for (int c = 0; c < 16; ++c)
                        acc[c0 + c] = (__uint_as_float(hh[c]) + __uint_as_float(mx[c])) * inv;
                }
            }
            const int pp = blockIdx.x * kTcM + row;
            if (pp < n_pts) {
                const size_t coil_stride = (size_t)gridDim.y * (size_t)n_pts;
#pragma unroll
                for (int c = 0; c < NC; ++c)
                    partial[(size_t)c * coil_stride + (size_t)blockIdx.y * n_pts + pp] = make_float2(acc[c], acc[NC + c]);
            }
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(kTcCols) : "memory");
}

}  // namespace bloch
