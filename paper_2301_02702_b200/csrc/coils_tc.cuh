// coils_tc.cuh -- multi-coil receive on the 5th-generation tensor cores (tcgen05 + TMEM).
//
// With several coils the receive sum is a dense contraction (reading C1):
//     S[n][c] = sum_i C[n][i] * W[i][c],     C[n][i] = Mxy_i(0) exp(-tau_n/T2_i) exp(i theta_in)
// [samples x spins] x [spins x coils], complex.  C is generated on the fly and never leaves the SM: the threads
// evaluate it (same arithmetic as signal_kernel), split every value into TF32 hi + lo and store it straight into
// shared memory in the canonical K-major operand layout; one elected thread issues tcgen05.mma (kind::tf32,
// M = 128 samples, N = 16 = 8 coils x {re, im}, K = 8 spins per instruction) with the FP32 accumulators in TMEM.
// The complex product is made real by stacking K:  A = [Cr | Ci],  B = [[Wr, Wi], [-Wi, Wr]]  ->  D = [Dr | Di],
// and every product runs as hi*hi + lo*hi + hi*lo ("3xTF32", ~2^-21 relative), because plain TF32 (2^-11) breaks
// the 1e-5 NRMSE bound on small phantoms: 6 MMA instructions per 8 spins and 128 samples, negligible next to the
// MUFU-bound generation of C.  B tiles (weights, negated / swapped / split as above) are prepared once per
// simulation by pack_coils_tc_kernel in exactly the shared-memory layout and arrive by bulk copies (TMA).
//
// Operand layout (no swizzle, K-major): 8-row x 16-byte core matrices (4 TF32 per row), contiguous 128 B each;
//     byte offset of element (row r, k) = (r / 8) * 256 + (k / 4) * 128 + (r % 8) * 16 + (k % 4) * 4
// i.e. leading-dimension (K) byte offset 128, stride-dimension (M / N) byte offset 256 in the matrix descriptors.
// CTA = 8 generator warps + 1 control warp, 128 samples; a stage = 16 spins (two 8-spin groups); generator thread =
// (samples m2 and m2 + 64, spin quad tid / 64) evaluates 8 contributions per stage and writes 16-byte vectors, then
// arrives on the stage's mbarrier; lane 0 of the control warp waits for it, issues the 12 MMAs and commits them to
// the mbarrier that frees the (double-buffered) A stage.  No CTA-wide barrier in the loop.  Spin records and B tiles
// ride a 4-slot TMA ring refilled by the control thread.  Epilogue: tcgen05.ld 32 lanes x 16 columns per warp -> P[coil][chunk][sample].
#pragma once
#include "coils.cuh"

namespace bloch {

constexpr int kTcM = 128;             // samples per CTA (MMA M)
constexpr int kTcStageSpins = 16;     // spins per stage
constexpr int kTcGroups = kTcStageSpins / 8;
constexpr int kTcSlots = 4;           // TMA ring: spin records + B tiles
constexpr int kTcATile = kTcM * 32;   // one A tile: 128 rows x 8 TF32 = 4096 B
// NC = coils per pass (8, 16 or 32): N = 2 NC columns (re | im)
__host__ __device__ constexpr int tc_btile(int nc) { return 2 * nc * 32; }     // one B tile: 2 NC rows x 8 TF32
__host__ __device__ constexpr int tc_bgroup(int nc) { return 4 * tc_btile(nc); }  // per 8-spin group: cr hi, cr lo, ci hi, ci lo
__host__ __device__ constexpr int tc_slot(int nc) { return kTcStageSpins * 32 + kTcGroups * tc_bgroup(nc); }  // spin records + B tiles
constexpr int kTcAStage = kTcGroups * 4 * kTcATile;                       // 32 KB
__host__ __device__ constexpr size_t tc_smem(int nc) { return 2 * (size_t)kTcAStage + kTcSlots * (size_t)tc_slot(nc) + 256; }
// the MMA count per stage does not depend on N, so more coils per pass are nearly free; 32 per pass need 132 KB of
// shared memory (one CTA per SM, which the tensor-pipe-bound kernel does not mind)
__host__ __device__ inline int tc_coils_per_pass(int n_coils) { return n_coils > 16 ? 32 : (n_coils > 8 ? 16 : 8); }

__device__ __forceinline__ uint32_t tc_tf32(float x) {
    uint32_t r;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
    return r;
}

// Weights -> B tiles.  Bt[pass][group][part][512 B], group = spin / 8 over the spins padded to a multiple of 16.
template <int NC>
__global__ void __launch_bounds__(256)
pack_coils_tc_kernel(int n, int n_pad, int n_coils, const float2 *__restrict__ coil, unsigned char *__restrict__ Bt) {
    constexpr int kTcBTile = tc_btile(NC), kTcBGroup = tc_bgroup(NC);
    const int i = blockIdx.x * blockDim.x + threadIdx.x;  // spin (padded range)
    const int pass = blockIdx.y;
    if (i >= n_pad) return;
    unsigned char *grp = Bt + ((size_t)pass * (n_pad / 8) + (size_t)(i / 8)) * kTcBGroup;
    const int k = i & 7;
    for (int c = 0; c < NC; ++c) {
        const int cc = pass * NC + c;
        float2 w = make_float2(0.f, 0.f);
        if (i < n && cc < n_coils) w = coil[(size_t)cc * n + i];
        // column n of the stacked B: cr-part [Wr | Wi], ci-part [-Wi | Wr]
        const float vals[2][2] = {{w.x, w.y}, {-w.y, w.x}};  // [part cr/ci][n < NC / n >= NC]
        for (int part = 0; part < 2; ++part)
            for (int hi8 = 0; hi8 < 2; ++hi8) {
                const int nn = c + NC * hi8;
                const float x = vals[part][hi8];
                const uint32_t h = tc_tf32(x);
                const uint32_t l = tc_tf32(x - __uint_as_float(h));
                const int off = (nn / 8) * 256 + (k / 4) * 128 + (nn % 8) * 16 + (k % 4) * 4;
                *reinterpret_cast<uint32_t *>(grp + (2 * part + 0) * kTcBTile + off) = h;
                *reinterpret_cast<uint32_t *>(grp + (2 * part + 1) * kTcBTile + off) = l;
            }
    }
}

// shared-memory matrix descriptor: no swizzle, K-major, LBO = 128 B, SBO = 256 B, descriptor version 1 (sm_100)
__device__ __forceinline__ uint64_t tc_desc(uint32_t smem_addr) {
    return (uint64_t)((smem_addr >> 4) & 0x3fffu) | ((uint64_t)(128u >> 4) << 16) | ((uint64_t)(256u >> 4) << 32) |
           ((uint64_t)1 << 46);
}
// instruction descriptor: D = F32, A = B = TF32, both K-major, N columns, M = 128
__host__ __device__ constexpr uint32_t tc_idesc(int n) {
    return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(n >> 3) << 17) | ((128u >> 4) << 24);
}

__device__ __forceinline__ void tc_mma(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t"
        "}\n" ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}

constexpr int kTcThreads = 288;  // 8 generator warps + 1 control warp (TMA + MMA issue by its lane 0)

template <int NC>
__global__ void __launch_bounds__(kTcThreads, NC == 32 ? 1 : 2)
signal_coils_tc_kernel(const float4 *__restrict__ recs, int n_pts, const float4 *__restrict__ A,
                       const float4 *__restrict__ S, const unsigned char *__restrict__ Bt /* this pass */,
                       int n_spins, int spins_per_chunk /* multiple of 16 */, const float *__restrict__ scal,
                       float2 *__restrict__ partial /* [NC][chunks][n_pts] */) {
    constexpr int kTcBTile = tc_btile(NC), kTcBGroup = tc_bgroup(NC), kTcSlotBytes = tc_slot(NC);
    constexpr uint32_t kIdesc = tc_idesc(2 * NC);
    constexpr int kCols = 2 * NC < 32 ? 32 : 2 * NC;  // TMEM columns (power of two >= 32)
    extern __shared__ __align__(1024) unsigned char smem[];
    unsigned char *a_tiles = smem;                                  // [2][groups][4 parts][4096]
    unsigned char *slots = smem + 2 * kTcAStage;                    // [kTcSlots][spin A (256 B) | spin S (256 B) | B tiles]
    uint64_t *full = reinterpret_cast<uint64_t *>(slots + kTcSlots * kTcSlotBytes);  // [kTcSlots] TMA landed
    uint64_t *a_full = full + kTcSlots;                                              // [2] generators done with an A stage
    uint64_t *mma_done = a_full + 2;                                                 // [2] tensor core done with an A stage
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(mma_done + 2);
    const int tid = threadIdx.x, warp = tid >> 5;
    const int s0 = blockIdx.y * spins_per_chunk;
    const int s1 = min(n_spins, s0 + spins_per_chunk);
    const int n_stages = (s1 - s0 + kTcStageSpins - 1) / kTcStageSpins;
    auto issue = [&](int st) {  // control thread: stage st -> ring slot st % kTcSlots
        const int sl = st % kTcSlots;
        unsigned char *dst = slots + sl * kTcSlotBytes;
        const int base = s0 + st * kTcStageSpins;
        const uint32_t cnt = (uint32_t)min(kTcStageSpins, s1 - base);
        mbar_expect_tx(&full[sl], cnt * 32u + (uint32_t)(kTcGroups * kTcBGroup));
        bulk_g2s(dst, A + base, cnt * 16u, &full[sl]);
        bulk_g2s(dst + kTcStageSpins * 16, S + base, cnt * 16u, &full[sl]);
        bulk_g2s(dst + kTcStageSpins * 32, Bt + (size_t)(base / 8) * kTcBGroup, (uint32_t)(kTcGroups * kTcBGroup), &full[sl]);
    };
    if (tid == 0) {
        for (int k = 0; k < kTcSlots; ++k) mbar_init(&full[k], 1);
        for (int k = 0; k < 2; ++k) {
            mbar_init(&a_full[k], 256);
            mbar_init(&mma_done[k], 1);
        }
        mbar_init_fence();
    }
    if (warp == 0) {  // TMEM: 32 columns (128 lanes x 16 FP32 columns used)
        __syncwarp();
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "n"(kCols) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = *tmem_slot;

    if (warp == 8) {
        // ------------------------------------------------------------ control warp: TMA ring + MMA issue (lane 0)
        if (tid == 256) {
            for (int st = 0; st < kTcSlots - 1 && st < n_stages; ++st) issue(st);
            for (int st = 0; st < n_stages; ++st) {
                const int ab = st & 1, sl = st % kTcSlots;
                mbar_wait(&a_full[ab], (uint32_t)((st >> 1) & 1));   // the generators have written this A stage
                mbar_wait(&full[sl], (uint32_t)((st / kTcSlots) & 1));  // (the B tiles landed; the generators saw it too)
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const uint32_t a0 = smem_u32(a_tiles + ab * kTcAStage);
                const uint32_t b0 = smem_u32(slots + sl * kTcSlotBytes + kTcStageSpins * 32);
#pragma unroll
                for (int gq = 0; gq < kTcGroups; ++gq) {
                    const uint32_t ag = a0 + gq * (4 * kTcATile), bg = b0 + gq * kTcBGroup;
                    const uint32_t first = (st == 0 && gq == 0) ? 0u : 1u;
                    tc_mma(tmem, tc_desc(ag + 0 * kTcATile), tc_desc(bg + 0 * kTcBTile), kIdesc, first);  // cr hi x B hi
                    tc_mma(tmem, tc_desc(ag + 1 * kTcATile), tc_desc(bg + 0 * kTcBTile), kIdesc, 1u);     // cr lo x B hi
                    tc_mma(tmem, tc_desc(ag + 0 * kTcATile), tc_desc(bg + 1 * kTcBTile), kIdesc, 1u);     // cr hi x B lo
                    tc_mma(tmem, tc_desc(ag + 2 * kTcATile), tc_desc(bg + 2 * kTcBTile), kIdesc, 1u);     // ci hi x B' hi
                    tc_mma(tmem, tc_desc(ag + 3 * kTcATile), tc_desc(bg + 2 * kTcBTile), kIdesc, 1u);     // ci lo x B' hi
                    tc_mma(tmem, tc_desc(ag + 2 * kTcATile), tc_desc(bg + 3 * kTcBTile), kIdesc, 1u);     // ci hi x B' lo
                }
                asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(&mma_done[ab])) : "memory");
                // refill the ring: slot (st + 3) % 4 held stage st - 1, whose MMAs must be complete
                if (st + kTcSlots - 1 < n_stages) {
                    if (st >= 1) mbar_wait(&mma_done[(st - 1) & 1], (uint32_t)(((st - 1) >> 1) & 1));
                    issue(st + kTcSlots - 1);
                }
            }
        }
    } else {
        // ------------------------------------------------------------ generator warps: 2 samples x 1 spin quad per thread
        const int m2 = tid & 63, quad = tid >> 6;  // rows m2 and m2 + 64 of the CTA's 128 samples; spins 4 quad .. 4 quad + 3
        float kx[2], ky[2], kz[2], tau[2];
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            const int p = blockIdx.x * kTcM + m2 + 64 * j;
            float4 r = make_float4(0.f, 0.f, 0.f, j ? tau[0] : 0.f);
            if (p < n_pts) r = recs[p];
            kx[j] = r.x; ky[j] = r.y; kz[j] = r.z; tau[j] = r.w;
        }
        const float cj1 = (tau[1] - tau[0]) * 0.6931471805599453f;
        // sample 1's decay from sample 0's by the cubic series when (tau_1 - tau_0)/T2 <= 0.02 for every spin
        const bool series = __all_sync(0xffffffffu, fabsf(cj1) * (scal[0] * kLog2e) <= 0.02f);
        for (int st = 0; st < n_stages; ++st) {
            const int ab = st & 1, sl = st % kTcSlots;
            if (st >= 2) {  // the MMAs that read A buffer ab two stages ago are complete
                mbar_wait(&mma_done[ab], (uint32_t)(((st - 2) >> 1) & 1));
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            }
            mbar_wait(&full[sl], (uint32_t)((st / kTcSlots) & 1));
            const unsigned char *slot = slots + sl * kTcSlotBytes;
            const float4 *spA = reinterpret_cast<const float4 *>(slot);
            const float4 *spS = reinterpret_cast<const float4 *>(slot + kTcStageSpins * 16);
            const int cnt = min(kTcStageSpins, s1 - (s0 + st * kTcStageSpins));
            float cr[2][4], ci[2][4];
#pragma unroll
            for (int j4 = 0; j4 < 4; ++j4) {
                const int sp = 4 * quad + j4;
                const bool ok = sp < cnt;
                const float4 a = spA[ok ? sp : 0];
                float4 sv = spS[ok ? sp : 0];  // (Mxy.re, Mxy.im, Mz, e2 = -log2(e)/T2)
                if (!ok) { sv.x = 0.f; sv.y = 0.f; }
                float er0 = 0.f, ei0 = 0.f;
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    const float th = fmaf(kx[j], a.x, fmaf(ky[j], a.y, fmaf(kz[j], a.z, tau[j] * a.w)));  // radians
                    const float sn = __sinf(th), cs = __cosf(th);
                    float er, ei;
                    if (j == 0 || !series) {
                        const float e = ex2_approx(tau[j] * sv.w);
                        er = sv.x * e;
                        ei = sv.y * e;
                        if (j == 0) { er0 = er; ei0 = ei; }
                    } else {
                        const float y = cj1 * sv.w;
                        const float pe = fmaf(y, fmaf(y, fmaf(y, 1.0f / 6.0f, 0.5f), 1.0f), 1.0f);
                        er = er0 * pe;
                        ei = ei0 * pe;
                    }
                    cr[j][j4] = fmaf(er, cs, -ei * sn);
                    ci[j][j4] = fmaf(er, sn, ei * cs);
                }
            }
            // hi = x rounded to TF32 by integer ops (add half an ulp of the 10-bit mantissa, clear the low 13 bits):
            // cvt.rna.tf32 would put two more operations per value on the 16-lane conversion pipe next to the MUFU
            // work.  lo = x - hi is exact; the tensor core ignores its low 13 bits (2^-22 of x).
            auto split = [](float x, uint32_t &hi, uint32_t &lo) {
                hi = (__float_as_uint(x) + 0x1000u) & 0xffffe000u;
                lo = __float_as_uint(x - __uint_as_float(hi));
            };
            unsigned char *abuf = a_tiles + ab * kTcAStage + (quad >> 1) * (4 * kTcATile) + (quad & 1) * 128;
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                uint4 crh, crl, cih, cil;
                split(cr[j][0], crh.x, crl.x); split(cr[j][1], crh.y, crl.y); split(cr[j][2], crh.z, crl.z); split(cr[j][3], crh.w, crl.w);
                split(ci[j][0], cih.x, cil.x); split(ci[j][1], cih.y, cil.y); split(ci[j][2], cih.z, cil.z); split(ci[j][3], cih.w, cil.w);
                const int row = m2 + 64 * j;
                unsigned char *gbase = abuf + (row >> 3) * 256 + (row & 7) * 16;
                *reinterpret_cast<uint4 *>(gbase + 0 * kTcATile) = crh;
                *reinterpret_cast<uint4 *>(gbase + 1 * kTcATile) = crl;
                *reinterpret_cast<uint4 *>(gbase + 2 * kTcATile) = cih;
                *reinterpret_cast<uint4 *>(gbase + 3 * kTcATile) = cil;
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // generic-proxy stores -> visible to the tensor core
            mbar_arrive(&a_full[ab]);
        }
        // all MMAs complete -> epilogue (warps 0-3: TMEM lanes 32 w .. 32 w + 31 = sample rows)
        if (warp < 4) {
            uint32_t v[2 * NC];
#pragma unroll
            for (int c = 0; c < 2 * NC; ++c) v[c] = 0u;
            if (n_stages > 0) {
                const int last = n_stages - 1;
                mbar_wait(&mma_done[last & 1], (uint32_t)((last >> 1) & 1));
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const uint32_t taddr = tmem + ((uint32_t)(32 * warp) << 16);
#pragma unroll
                for (int c0 = 0; c0 < 2 * NC; c0 += 16)
                    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                                 : "=r"(v[c0 + 0]), "=r"(v[c0 + 1]), "=r"(v[c0 + 2]), "=r"(v[c0 + 3]), "=r"(v[c0 + 4]), "=r"(v[c0 + 5]),
                                   "=r"(v[c0 + 6]), "=r"(v[c0 + 7]), "=r"(v[c0 + 8]), "=r"(v[c0 + 9]), "=r"(v[c0 + 10]), "=r"(v[c0 + 11]),
                                   "=r"(v[c0 + 12]), "=r"(v[c0 + 13]), "=r"(v[c0 + 14]), "=r"(v[c0 + 15])
                                 : "r"(taddr + (uint32_t)c0));
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            }
            const int pp = blockIdx.x * kTcM + 32 * warp + (tid & 31);
            if (pp < n_pts) {
                const size_t coil_stride = (size_t)gridDim.y * (size_t)n_pts;
#pragma unroll
                for (int c = 0; c < NC; ++c)
                    partial[(size_t)c * coil_stride + (size_t)blockIdx.y * n_pts + pp] =
                        make_float2(__uint_as_float(v[c]), __uint_as_float(v[NC + c]));
            }
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(kCols) : "memory");
}

}  // namespace bloch
