// coils_tc.cuh -- multi-coil receive on the 5th-generation tensor cores (tcgen05 + TMEM).
//
// With several coils the receive sum is a dense contraction (reading C1):
//     S[n][c] = sum_i C[n][i] * W[i][c],     C[n][i] = Mxy_i(0) exp(-tau_n/T2_i) exp(i theta_in)
// [samples x spins] x [spins x coils], complex.  C is generated on the fly and never leaves the SM -- it does not even
// pass through shared memory: a generator thread owns ONE sample (= one TMEM lane, one row of the MMA's M = 128),
// evaluates its contributions from 8 spins (same arithmetic as signal_kernel), splits every value into TF32 hi + lo and
// writes the 32 values straight from its registers into TENSOR MEMORY (tcgen05.st.32x32b.x32), where they are the A
// operand of tcgen05.mma (kind::tf32, M = 128 samples, N = 2 x coils, K = 8 spins per instruction, FP32 accumulators
// in TMEM as well).  Only B (the weights) comes from shared memory.  With A in TMEM an M128 N16 K8 instruction costs its
// floor of 8 clocks (128 N / 256); with both operands in shared memory (round 1) it cost ~100 and the kernel lost to the
// FFMA kernel at 8 coils.
// The complex product is made real by stacking K:  A = [Cr | Ci],  B = [[Wr, Wi], [-Wi, Wr]]  ->  D = [Dr | Di],
// and every product runs as hi*hi + lo*hi + hi*lo ("3xTF32", ~2^-21 relative), because plain TF32 (2^-11) breaks
// the 1e-5 NRMSE bound on small phantoms: 6 MMA instructions per 8 spins and 128 samples -- 4 for up to 16 coils per
// pass, where the B tiles of a group lie [B hi | B lo] side by side along N and the hi part of A meets both in ONE
// instruction of N = 4 NC (its halves land in two accumulator column groups, added in the epilogue): an instruction of
// this shape costs ~74 clocks whatever N, so the count is what matters (8 coils: 105.9 -> 93.3 ms on config 4).  B
// tiles (weights, negated / swapped / split as above) are prepared once per simulation by pack_coils_tc_kernel in
// exactly the shared-memory operand layout and arrive by bulk copies (TMA).
//
// B operand layout (no swizzle, K-major): 8-row x 16-byte core matrices (4 TF32 per row), contiguous 128 B each;
//     byte offset of element (row r, k) = (r / 8) * 256 + (k / 4) * 128 + (r % 8) * 16 + (k % 4) * 4
// i.e. leading-dimension (K) byte offset 128, stride-dimension (N) byte offset 256 in the matrix descriptor.
// A operand in TMEM: row m = lane m, K = 8 consecutive 32-bit columns; a stage (16 spins) is 2 groups x 4 parts
// (cr hi, cr lo, ci hi, ci lo) x 8 columns = 64 columns, three stages deep; the accumulators take the first 2 NC columns.
// CTA = 8 generator warps + 1 control warp, 128 samples, two CTAs per SM; a stage = 16 spins.  Warps w and w + 4
// own the TMEM lanes 32 (w % 4) .. + 31 (a warp reaches only its lane quarter): warps 0-3 generate the even stages,
// warps 4-7 the odd ones, each thread its sample's
// row of the stage, then tcgen05.wait::st, fence, arrive on the stage's mbarrier; lane 0 of the control warp waits for it,
// issues the stage's 8 (32 coils per pass: 12) MMAs and commits them to the mbarrier that frees the A stage.  No
// CTA-wide barrier in the loop.  Spin records and B tiles ride an 8-slot (32 coils: 6-slot) TMA ring refilled by the
// control thread.  Epilogue: tcgen05.ld 32 lanes x 16
// columns per warp -> P[coil][chunk][sample].
#pragma once
#include "coils.cuh"

namespace bloch {

constexpr int kTcM = 128;             // samples per CTA (MMA M)
constexpr int kTcStageSpins = 16;     // spins per stage (two K = 8 groups)
constexpr int kTcGroups = kTcStageSpins / 8;
// TMA ring of spin records + B tiles.  A slot is refilled when the MMAs that read its B tiles are complete, so the copy
// for stage st + slots - 1 starts after the MMAs of stage st - 1: with 4 slots the generators (up to kTcAStages ahead of
// the tensor core) found their spins not yet landed on every stage (ncu: 19 % of all warp samples on that wait, 42 % on
// the A-stage wait behind it).  8 slots (32 coils per pass: 6 x 17 KB, so that two CTAs still share an SM).
__host__ __device__ constexpr int tc_slots(int nc) { return nc > 16 ? 6 : 8; }
// A stages in TMEM: each generator set fills one while the tensor core works through the others.  Measured on workload
// 4c (signal kernels, 8 coils): two CTAs of 8 generator warps (two sets) per SM with three 16-spin stages each 120 ms;
// six 8-spin stages 140 ms (twice the hand-shakes per evaluation); ONE CTA of 16 generator warps (four sets) per SM with
// seven 16-spin stages 182 ms (a single accumulator chain per SM: the MMAs of one CTA into one accumulator serialise).
constexpr int kTcAStages = 3;
constexpr int kTcAStageCols = kTcGroups * 4 * 8;  // 64 columns per stage: groups x (cr hi, cr lo, ci hi, ci lo) x K = 8
constexpr int kTcDCols = 64;          // accumulator columns reserved (2 NC <= 64; two accumulators when 4 NC <= 64)
constexpr int kTcCols = 256;          // TMEM allocation: 64 + 3 x 64 = 256 columns (two CTAs share an SM's 512)
static_assert(kTcDCols + kTcAStages * kTcAStageCols <= kTcCols, "TMEM columns");
// NC = coils per pass (8, 16 or 32): N = 2 NC columns (re | im)
__host__ __device__ constexpr int tc_btile(int nc) { return 2 * nc * 32; }     // one B tile: 2 NC rows x 8 TF32
__host__ __device__ constexpr int tc_bgroup(int nc) { return 4 * tc_btile(nc); }  // per 8-spin group: cr hi, cr lo, ci hi, ci lo
__host__ __device__ constexpr int tc_slot(int nc) { return kTcStageSpins * 32 + kTcGroups * tc_bgroup(nc); }  // spin records + B tiles
__host__ __device__ constexpr size_t tc_smem(int nc) { return tc_slots(nc) * (size_t)tc_slot(nc) + 256; }
// the MMA count per stage does not depend on N, so more coils per pass are nearly free (the floor of an instruction
// grows with N: 8 / 16 / 32 clocks for 8 / 16 / 32 coils)
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

__device__ __forceinline__ void tc_mma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t"
        "}\n" ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}

// 32 consecutive TMEM columns of the thread's lane <- 32 registers
__device__ __forceinline__ void tc_st32(uint32_t taddr, const uint32_t (&v)[32]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,"
        "%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};"
        ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]),
          "r"(v[9]), "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]), "r"(v[16]), "r"(v[17]),
          "r"(v[18]), "r"(v[19]), "r"(v[20]), "r"(v[21]), "r"(v[22]), "r"(v[23]), "r"(v[24]), "r"(v[25]), "r"(v[26]),
          "r"(v[27]), "r"(v[28]), "r"(v[29]), "r"(v[30]), "r"(v[31]) : "memory");
}

constexpr int kTcGenWarps = 8;   // two sets of four: set s generates the stages s, s + 2, ...; warp w owns TMEM lanes 32 (w % 4) ..
constexpr int kTcThreads = 32 * (kTcGenWarps + 1);  // + 1 control warp (TMA + MMA issue by its lane 0)

template <int NC>
__global__ void __launch_bounds__(kTcThreads, 2)
signal_coils_tc_kernel(const float4 *__restrict__ recs, int n_pts, const float4 *__restrict__ A,
                       const float4 *__restrict__ S, const unsigned char *__restrict__ Bt /* this pass */,
                       int n_spins, int spins_per_chunk /* multiple of 16 */, const float *__restrict__ scal,
                       float2 *__restrict__ partial /* [NC][chunks][n_pts] */) {
    constexpr int kTcBTile = tc_btile(NC), kTcBGroup = tc_bgroup(NC), kTcSlotBytes = tc_slot(NC), kTcSlots = tc_slots(NC);
    constexpr uint32_t kIdesc = tc_idesc(2 * NC);
    static_assert(2 * NC <= kTcDCols, "accumulator columns");
    // Accumulator columns, in groups of 2 NC that the epilogue adds up.  Up to 16 coils per pass the wide scheme is used
    // (kWide, see the MMA issue loop): 8 coils: [Cr: hh + lh | Cr: hl | Ci: hh + lh | Ci: hl], 16 coils: [hh + lh | hl];
    // 32 coils: one group.  (Separate accumulator chains by themselves change nothing: 8 coils on four chains 106.8 ms,
    // 32 coils on one 107.7 ms.)
    constexpr bool kWide = 4 * NC <= kTcDCols;
    constexpr int kAcc = kTcDCols / (2 * NC) >= 4 ? 4 : (kTcDCols / (2 * NC) >= 2 ? 2 : 1);
    constexpr uint32_t kCi = kAcc == 4 ? 4 * NC : 0;        // the Ci products' own accumulator when there is room
    constexpr uint32_t kIdescW = tc_idesc(4 * NC);          // N = 4 NC: [B hi | B lo]
    extern __shared__ __align__(1024) unsigned char smem[];
    unsigned char *slots = smem;                                    // [kTcSlots][spin A (256 B) | spin S (256 B) | B tiles]
    uint64_t *full = reinterpret_cast<uint64_t *>(slots + kTcSlots * kTcSlotBytes);  // [kTcSlots] TMA landed
    uint64_t *a_full = full + kTcSlots;                                              // [kTcAStages] generators done with an A stage
    uint64_t *mma_done = a_full + kTcAStages;                                        // [kTcAStages] tensor core done with an A stage
    uint64_t *all_done = mma_done + kTcAStages;                                      // every MMA of the CTA has completed
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(all_done + 1);
    const int tid = threadIdx.x, warp = tid >> 5;
    const int s0 = blockIdx.y * spins_per_chunk;
    const int s1 = min(n_spins, s0 + spins_per_chunk);
    const int n_stages = (s1 - s0 + kTcStageSpins - 1) / kTcStageSpins;
    (void)scal;
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
    // the spin-record area of every ring slot starts as zeros: the last stage of the phantom may hold fewer than 16
    // spins, and what the bulk copy does not overwrite must be finite (its B rows are zero, pack_coils_tc_kernel)
    for (int k = tid; k < kTcSlots * kTcStageSpins * 2; k += kTcThreads)
        reinterpret_cast<float4 *>(slots + (k / (kTcStageSpins * 2)) * kTcSlotBytes)[k % (kTcStageSpins * 2)] = make_float4(0.f, 0.f, 0.f, 0.f);
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // generic-proxy stores before the async-proxy bulk copies
    if (tid == 0) {
        for (int k = 0; k < kTcSlots; ++k) mbar_init(&full[k], 1);
        for (int k = 0; k < kTcAStages; ++k) {
            mbar_init(&a_full[k], 128);  // the four generator warps of the stage's half
            mbar_init(&mma_done[k], 1);
        }
        mbar_init(all_done, 1);
        mbar_init_fence();
    }
    if (warp == 0) {  // TMEM: accumulators + three A stages
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
            for (int st = 0; st < kTcSlots - 1 && st < n_stages; ++st) issue(st);
            for (int st = 0; st < n_stages; ++st) {
                const int ab = st % kTcAStages, sl = st % kTcSlots;
                mbar_wait(&a_full[ab], (uint32_t)((st / kTcAStages) & 1));  // the generators have written this A stage
                mbar_wait(&full[sl], (uint32_t)((st / kTcSlots) & 1));      // (the B tiles landed; the generators saw it too)
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const uint32_t a0 = tmem + (uint32_t)(kTcDCols + ab * kTcAStageCols);
                const uint32_t b0 = smem_u32(slots + sl * kTcSlotBytes + kTcStageSpins * 32);
#pragma unroll
                for (int gq = 0; gq < kTcGroups; ++gq) {
                    const uint32_t ag = a0 + gq * 32, bg = b0 + gq * kTcBGroup;  // A parts: columns +0 cr hi, +8 cr lo, +16 ci hi, +24 ci lo
                    const uint32_t first = (st == 0 && gq == 0) ? 0u : 1u;  // 0: the accumulator's first MMA overwrites
                    if (kWide) {
                        // An instruction costs the same for any N (~74 clocks), and the B tiles [B hi | B lo] lie side by
                        // side along N: ONE instruction of N = 4 NC gives hi x B hi in the accumulator's first 2 NC
                        // columns and hi x B lo in the next 2 NC; the lo x B hi product adds into the first 2 NC.
                        // 4 instructions per 8 spins instead of 6; the column groups are added in the epilogue.
                        tc_mma_ts(tmem, ag + 0, tc_desc(bg + 0 * kTcBTile), kIdescW, first);                      // cr hi x [B hi | B lo]
                        tc_mma_ts(tmem + kCi, ag + 16, tc_desc(bg + 2 * kTcBTile), kIdescW, kCi ? first : 1u);    // ci hi x [B' hi | B' lo]
                        tc_mma_ts(tmem, ag + 8, tc_desc(bg + 0 * kTcBTile), kIdesc, 1u);                          // cr lo x B hi
                        tc_mma_ts(tmem + kCi, ag + 24, tc_desc(bg + 2 * kTcBTile), kIdesc, 1u);                   // ci lo x B' hi
                    } else {
                        tc_mma_ts(tmem, ag + 0, tc_desc(bg + 0 * kTcBTile), kIdesc, first);    // cr hi x B hi
                        tc_mma_ts(tmem, ag + 16, tc_desc(bg + 2 * kTcBTile), kIdesc, 1u);      // ci hi x B' hi
                        tc_mma_ts(tmem, ag + 8, tc_desc(bg + 0 * kTcBTile), kIdesc, 1u);       // cr lo x B hi
                        tc_mma_ts(tmem, ag + 24, tc_desc(bg + 2 * kTcBTile), kIdesc, 1u);      // ci lo x B' hi
                        tc_mma_ts(tmem, ag + 0, tc_desc(bg + 1 * kTcBTile), kIdesc, 1u);       // cr hi x B lo
                        tc_mma_ts(tmem, ag + 16, tc_desc(bg + 3 * kTcBTile), kIdesc, 1u);      // ci hi x B' lo
                    }
                }
                asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(&mma_done[ab])) : "memory");
                // refill the ring: the slot of stage st + kTcSlots - 1 held stage st - 1, whose MMAs must be complete
                if (st + kTcSlots - 1 < n_stages) {
                    if (st >= 1) mbar_wait(&mma_done[(st - 1) % kTcAStages], (uint32_t)(((st - 1) / kTcAStages) & 1));
                    issue(st + kTcSlots - 1);
                }
            }
            // the epilogue warps finish their own (even) stages up to two stages before the last one: they wait on a
            // barrier of their own, not on a stage barrier that may still be a phase behind (parity waits would alias)
            asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(all_done)) : "memory");
        }
    } else {
        // ------------------------------------------------------------ generator warps: one sample (TMEM lane) per thread
        const int set = warp >> 2;                        // warps 4 s .. 4 s + 3 generate the stages s, s + 4, s + 8, ...
        const int row = 32 * (warp & 3) + (tid & 31);     // the thread's row of the 128 samples = its TMEM lane
        const uint32_t lane_addr = tmem + ((uint32_t)(32 * (warp & 3)) << 16);
        float4 r = make_float4(0.f, 0.f, 0.f, 0.f);
        {
            const int p = blockIdx.x * kTcM + row;
            if (p < n_pts) r = recs[p];
        }
        const float kx = r.x, ky = r.y, kz = r.z, tau = r.w;
        // The tensor core reads the upper 19 bits of a TF32 operand, i.e. it truncates: hi is x as it stands, and
        // lo = x - trunc(x) is exact (one LOP, one FADD); the tensor core truncates lo in turn, leaving 2^-20 of x.
        auto split = [](float x, uint32_t &hi, uint32_t &lo) {
            hi = __float_as_uint(x);
            lo = __float_as_uint(x - __uint_as_float(hi & 0xffffe000u));
        };
        for (int st = set; st < n_stages; st += kTcGenWarps / 4) {
            const int ab = st % kTcAStages, sl = st % kTcSlots;
            if (st >= kTcAStages) {  // the MMAs that read this A stage kTcAStages stages ago are complete
                mbar_wait(&mma_done[ab], (uint32_t)(((st / kTcAStages) - 1) & 1));
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            }
            mbar_wait(&full[sl], (uint32_t)((st / kTcSlots) & 1));
            const unsigned char *slot = slots + sl * kTcSlotBytes;
            const float4 *spA = reinterpret_cast<const float4 *>(slot);
            const float4 *spS = reinterpret_cast<const float4 *>(slot + kTcStageSpins * 16);
#pragma unroll
            for (int gq = 0; gq < kTcGroups; ++gq) {
                uint32_t v[32];  // [cr hi (8) | cr lo (8) | ci hi (8) | ci lo (8)] for the group's 8 spins
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    const int sp = 8 * gq + k;
                    const float4 a = spA[sp];
                    const float4 sv = spS[sp];  // (Mxy.re, Mxy.im, Mz, e2 = -log2(e)/T2)
                    const float th = fmaf(kx, a.x, fmaf(ky, a.y, fmaf(kz, a.z, tau * a.w)));  // radians
                    const float sn = __sinf(th), cs = __cosf(th);
                    const float e = ex2_approx(tau * sv.w);
                    const float er = sv.x * e, ei = sv.y * e;
                    split(fmaf(er, cs, -ei * sn), v[k], v[8 + k]);
                    split(fmaf(er, sn, ei * cs), v[16 + k], v[24 + k]);
                }
                tc_st32(lane_addr + (uint32_t)(kTcDCols + ab * kTcAStageCols + gq * 32), v);
            }
            asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            mbar_arrive(&a_full[ab]);
        }
        // all MMAs complete -> epilogue (warps 0-3: TMEM lanes 32 w .. 32 w + 31 = sample rows)
        if (warp < 4) {
            uint32_t v[2 * NC];
#pragma unroll
            for (int c = 0; c < 2 * NC; ++c) v[c] = 0u;
            if (n_stages > 0) {
                mbar_wait(all_done, 0u);
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
                for (int c0 = 0; c0 < 2 * NC; c0 += 16)
                    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                                 : "=r"(v[c0 + 0]), "=r"(v[c0 + 1]), "=r"(v[c0 + 2]), "=r"(v[c0 + 3]), "=r"(v[c0 + 4]), "=r"(v[c0 + 5]),
                                   "=r"(v[c0 + 6]), "=r"(v[c0 + 7]), "=r"(v[c0 + 8]), "=r"(v[c0 + 9]), "=r"(v[c0 + 10]), "=r"(v[c0 + 11]),
                                   "=r"(v[c0 + 12]), "=r"(v[c0 + 13]), "=r"(v[c0 + 14]), "=r"(v[c0 + 15])
                                 : "r"(lane_addr + (uint32_t)c0));
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                for (int acc = 1; acc < kAcc; ++acc) {  // add the other accumulators
                    uint32_t u[2 * NC];
#pragma unroll
                    for (int c0 = 0; c0 < 2 * NC; c0 += 16)
                        asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                                     : "=r"(u[c0 + 0]), "=r"(u[c0 + 1]), "=r"(u[c0 + 2]), "=r"(u[c0 + 3]), "=r"(u[c0 + 4]), "=r"(u[c0 + 5]),
                                       "=r"(u[c0 + 6]), "=r"(u[c0 + 7]), "=r"(u[c0 + 8]), "=r"(u[c0 + 9]), "=r"(u[c0 + 10]), "=r"(u[c0 + 11]),
                                       "=r"(u[c0 + 12]), "=r"(u[c0 + 13]), "=r"(u[c0 + 14]), "=r"(u[c0 + 15])
                                     : "r"(lane_addr + (uint32_t)(acc * 2 * NC + c0)));
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                    for (int c = 0; c < 2 * NC; ++c) v[c] = __float_as_uint(__uint_as_float(v[c]) + __uint_as_float(u[c]));
                }
            }
            const int pp = blockIdx.x * kTcM + row;
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
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(kTcCols) : "memory");
}

}  // namespace bloch
