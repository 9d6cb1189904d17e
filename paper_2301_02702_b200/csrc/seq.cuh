// seq.cuh -- whole-sequence kernel (a5-a8 in ONE launch) for plans with few spins and many blocks (MRF, GRE).
//
// With 65,536 spins an excitation launch holds 3.5 warps per SM sub-partition and is bound by the latency of
// its own dependent chain, and the signal launch that follows leaves the FMA pipe half idle; launched one
// after the other neither fills the machine (profiles/r01_v2_cfg5.md).  Spins are independent,
// so here ONE persistent CTA per SM owns a fixed chunk of spins for the whole sequence and its warps are
// specialised:
//   warp 0              producer: streams the RF step tiles of ALL excitation blocks, in sequence order, through a
//                       4-stage shared-memory ring with 1-D bulk copies (TMA) -- across block boundaries, so the
//                       first tile of the next pulse is already resident when the RF warps get there
//   warps 1 .. R        RF warps: one spin per thread, magnetisation in registers for the WHOLE SEQUENCE (a8:
//                       rf_tile of rf.cuh; block-end free precession by propagate()); at the start of every
//                       precession block that serves ADC samples they publish (Mxy, e2) to a double-buffered
//                       shared array and carry straight on with the next pulse
//   warps R+1 .. R+G    signal warps: for every published state evaluate the block's ADC samples (a6: a thread
//                       owns P adjacent samples and walks the chunk's spins in shared memory, arithmetic as
//                       signal_kernel) and write the CTA's partial sums of that block into a RING of partial rows
//                       ring[block % R][cta][sample] (a7).  The sum over the CTAs is made inside the same launch,
//                       a few blocks later: CTA c adds, in CTA order, rows 0 .. n_ctas-1 of ITS slice of
//                       the block's samples and writes the signal -- no float atomics, a fixed order whatever the
//                       timing, so still bitwise reproducible; integer tickets (arrive / reduced, one pair per block)
//                       say when a block's rows are complete and when its ring slot may be written again.  The
//                       signal warp that finishes a block last in its CTA raises the CTA's ticket and makes the
//                       CTA's sum of the block kSeqReduceLag blocks back.  The
//                       block's samples are cut into items of 32 x P samples which the warps take from a
//                       shared counter, so a sub-partition that holds fewer RF warps serves more items; a
//                       sample's sum is one thread's walk over the chunk in spin order whichever warp takes it
// so the FMA-bound excitation of pulse k+1 and the MUFU-bound readout of block k share the SM's issue slots.
// The roles meet only at mbarriers (tile full/empty, state full/empty); there is no CTA-wide barrier after set-up.
// The published states go through a ring of kSeqStateBufs buffers: the signal warps may lag that many blocks.
// The state is rounded to one float per component at the end of every RF block exactly as rf_kernel stores it,
// so the final magnetisation is bitwise equal to the per-block path.
#pragma once
#include <type_traits>

#include "internal.h"
#include "kernels.cuh"
#include "rf.cuh"
#include "signal.cuh"
#include "tma.cuh"

namespace bloch {

constexpr int kSeqStages = 4;
constexpr int kSeqTileStride = 4224;  // >= kRfHdrBytes + kRfTileSteps * 32 (static plans), multiple of 128
constexpr int kSeqMaxThreads = 1024;
constexpr int kSeqStateBufs = 4;
constexpr int kSeqBarBytes = 256;
// Partial-row ring: kSeqRingSlots blocks may lie between "partial row written" and "summed over the CTAs", and a CTA
// sums its slice of block g - kSeqReduceLag when it has finished block g, so the CTAs may drift kSeqRingSlots -
// kSeqReduceLag blocks apart before anyone waits for a ticket.  Measured alternatives (config 5 / config 2, against
// 124.2 / 2.237 ms with one partial row per CTA over the whole sequence, summed by a second kernel): this layout 125.2 /
// 2.217; tickets looked at every fourth block (2 blocks of drift) 127.0 / 2.254; 26 to 64 slots with a lag of a quarter
// of them 127.0 / 2.334 (the last `lag` blocks are summed after the sequence's end: a tail short sequences feel); a
// dedicated reducer warp polling every 200 ns 126.1 / 2.42, every 2 us 125.3 / 2.33, asleep on an mbarrier 128.5 /
// 2.34; the roles as separate non-inlined functions 133.8 / 3.06 (spills under the 64-register cap).
constexpr int kSeqReduceLag = 3;
constexpr int kSeqRingSlots = 8;
static_assert(kSeqRingSlots > kSeqReduceLag + 1, "ring too short");

// Role of each warp of the CTA, chosen on the host (api.cu seq_shape) so that every SM sub-partition (warp id mod 4)
// carries about the same load: >= 0: RF warp with that index (spins 32 i .. 32 i + 31 of the chunk), -1: producer,
// -2: signal warp, -3: idle (exits at once).
struct SeqRoles {
    signed char role[kSeqMaxThreads / 32];
    int n_sig_warps;
};
constexpr int kRoleProducer = -1, kRoleSignal = -2, kRoleIdle = -3;
static_assert(kSeqTileStride >= kRfHdrBytes + kRfTileSteps * 32 && kSeqTileStride % 128 == 0, "tile stride");

// dynamic shared memory: [ring: kSeqStages x kSeqTileStride][barriers + item counters: 256 B][shA: chunk float4]
// [shS: kSeqStateBufs x chunk float4]
// [shW: chunk x NC float2] with NC receive coils
__host__ __device__ inline size_t seq_smem_bytes(int chunk, int nc = 0) {
    return size_t(kSeqStages) * kSeqTileStride + kSeqBarBytes + size_t(1 + kSeqStateBufs) * chunk * sizeof(float4) +
           size_t(chunk) * nc * sizeof(float2);
}
static_assert((2 * kSeqStages + 2 * kSeqStateBufs) * 8 + 2 * kSeqStateBufs * 4 <= kSeqBarBytes, "barrier area");

// cross-CTA tickets of the partial-row ring (integers only)
__device__ __forceinline__ int ld_acquire_gpu(const int *p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void wait_ticket(const int *ctr, int target, int lane) {
    if (lane == 0)
        while (ld_acquire_gpu(ctr) < target) __nanosleep(200);
    __syncwarp();
}

// One CTA's share of the sum over CTAs for one block: samples [cta n_pts / n_ctas, (cta + 1) n_pts / n_ctas) of the
// block, rows added in CTA order (lane r takes rows r, r + 32, ...; fixed butterfly across lanes).
__device__ __forceinline__ void seq_reduce_slice(const float2 *slot, int slot_stride, int n_ctas, int cta, int n_pts,
                                                 float2 *__restrict__ sig, int lane, const int *arrive, int *reduced) {
    wait_ticket(arrive, n_ctas, lane);  // every CTA's row of this block is written and visible
    const int p_lo = (int)((long long)cta * n_pts / n_ctas), p_hi = (int)((long long)(cta + 1) * n_pts / n_ctas);
    for (int p = p_lo; p < p_hi; ++p) {
        float re = 0.f, im = 0.f;
        for (int r = lane; r < n_ctas; r += 32) {
            const float2 v = __ldcg(slot + (size_t)r * slot_stride + p);  // L2: the slot is rewritten by other SMs
            re += v.x;
            im += v.y;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            re += __shfl_xor_sync(0xffffffffu, re, o);
            im += __shfl_xor_sync(0xffffffffu, im, o);
        }
        if (lane == 0) sig[p] = make_float2(re, im);
    }
    __syncwarp();
    if (lane == 0) {
        __threadfence();  // this CTA's reads of the slot are done before the slot is declared free
        atomicAdd(reduced, 1);
    }
}

// One item (32 x P adjacent ADC samples starting at `base`) of a precession block for the chunk's spins.
template <int P>
__device__ __forceinline__ void seq_signal_item(const float4 *__restrict__ recs, int n_pts, int base, const float4 *shA,
                                                const float4 *shS, int cnt, int lane, float r2max_log2e,
                                                float2 *__restrict__ out) {
    const int p0 = base + lane * P;
    float kx[P], ky[P], kz[P], tau[P], cj[P], ar[P], ai[P];
    float cmax = 0.f;
#pragma unroll
    for (int j = 0; j < P; ++j) {
        const int p = p0 + j;
        float4 r = make_float4(0.f, 0.f, 0.f, j ? tau[0] : 0.f);
        if (p < n_pts) r = recs[p];
        kx[j] = r.x; ky[j] = r.y; kz[j] = r.z; tau[j] = r.w;
        cj[j] = (r.w - tau[0]) * 0.6931471805599453f;
        cmax = fmaxf(cmax, fabsf(cj[j]));
        ar[j] = 0.f; ai[j] = 0.f;
    }
    // exp(-tau_j/T2), j > 0, from the j = 0 value by a cubic series when (tau_j - tau_0)/T2 <= 0.02 for every spin
    const bool series = P > 1 && __all_sync(0xffffffffu, cmax * r2max_log2e <= 0.02f);
    // equally spaced samples: decay of sample j = decay of sample j-1 times q = exp(-dwell/T2) (signal.cuh)
    float dev = 0.f;
#pragma unroll
    for (int j = 2; j < P; ++j) dev = fmaxf(dev, fabsf(cj[j] - (float)j * cj[1]));
    const bool geom = P > 2 && series && __all_sync(0xffffffffu, dev * r2max_log2e <= 1e-6f);
    auto run = [&](auto mode_tag) {
        constexpr int MODE = decltype(mode_tag)::value;  // 0: MUFU.EX2 per sample, 1: series per sample, 2: geometric
#pragma unroll 2
        for (int s = 0; s < cnt; ++s) signal_spin_fp32<P, MODE>(kx, ky, kz, tau, cj, shA[s], shS[s], ar, ai);
    };
    if (geom) run(std::integral_constant<int, 2>{});
    else if (series) run(std::integral_constant<int, 1>{});
    else run(std::integral_constant<int, 0>{});
#pragma unroll
    for (int j = 0; j < P; ++j)
        if (p0 + j < n_pts) out[p0 + j] = make_float2(ar[j], ai[j]);
}

// A signal warp's share of one block: items taken from the block's shared counter until none is left.
template <int P>
__device__ __forceinline__ void seq_signal_block(const float4 *__restrict__ recs, int n_pts, const float4 *shA,
                                                 const float4 *shS, int cnt, int lane, int *item_ctr,
                                                 float r2max_log2e, float2 *__restrict__ out) {
    for (;;) {
        int item = 0;
        if (lane == 0) item = atomicAdd(item_ctr, 1);
        item = __shfl_sync(0xffffffffu, item, 0);
        const int base = item * (32 * P);
        if (base >= n_pts) break;
        seq_signal_item<P>(recs, n_pts, base, shA, shS, cnt, lane, r2max_log2e, out);
    }
}

// The same for n_coils receive coils: a CTA's row of a block is [NC][slot_stride] (coil-major), the signal [n_coils][n_adc].
__device__ __forceinline__ void seq_reduce_slice_coils(const float2 *slot, int slot_stride, int nc, int n_ctas, int cta,
                                                       int n_pts, float2 *__restrict__ sig, long long n_adc, int n_coils,
                                                       int lane, const int *arrive, int *reduced) {
    wait_ticket(arrive, n_ctas, lane);
    const int p_lo = (int)((long long)cta * n_pts / n_ctas), p_hi = (int)((long long)(cta + 1) * n_pts / n_ctas);
    const size_t row = (size_t)nc * slot_stride;
    for (int c = 0; c < n_coils; ++c) {
        for (int p = p_lo; p < p_hi; ++p) {
            float re = 0.f, im = 0.f;
            for (int r = lane; r < n_ctas; r += 32) {
                const float2 v = __ldcg(slot + (size_t)r * row + (size_t)c * slot_stride + p);
                re += v.x;
                im += v.y;
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                re += __shfl_xor_sync(0xffffffffu, re, o);
                im += __shfl_xor_sync(0xffffffffu, im, o);
            }
            if (lane == 0) sig[(size_t)c * (size_t)n_adc + p] = make_float2(re, im);
        }
    }
    __syncwarp();
    if (lane == 0) {
        __threadfence();
        atomicAdd(reduced, 1);
    }
}

// Multi-coil item (reading C1): 32 x P adjacent samples, P per lane, NC coil sums per sample.  A spin's
// contribution (phase, sin / cos, decay: signal_spin_fp32) does not depend on the coil; every coil adds one complex
// multiply-add with the spin's weight (shW: NC float2 per spin, read as warp-wide broadcasts, shared by the P samples).
// P = 2 for up to 4 coils (16 accumulators); 8 coils keep P = 1 under the kernel's 64-register cap.
template <int NC, int P>
__device__ __forceinline__ void seq_signal_item_coils(const float4 *__restrict__ recs, int n_pts, int base,
                                                      const float4 *shA, const float4 *shS, const float4 *shW, int cnt,
                                                      int lane, float r2max_log2e, int slot_stride,
                                                      float2 *__restrict__ out) {
    const int p0 = base + lane * P;
    float kx[P], ky[P], kz[P], tau[P], cj[P];
    float cmax = 0.f;
#pragma unroll
    for (int j = 0; j < P; ++j) {
        const int p = p0 + j;
        float4 r = make_float4(0.f, 0.f, 0.f, j ? tau[0] : 0.f);
        if (p < n_pts) r = recs[p];
        kx[j] = r.x; ky[j] = r.y; kz[j] = r.z; tau[j] = r.w;
        cj[j] = (r.w - tau[0]) * 0.6931471805599453f;
        cmax = fmaxf(cmax, fabsf(cj[j]));
    }
    const bool series = P > 1 && __all_sync(0xffffffffu, cmax * r2max_log2e <= 0.02f);  // as seq_signal_item
    // coil sums in pairs (coils 2k, 2k + 1): the complex multiply-adds run as packed FP32 (fma.rn.f32x2: one issue slot
    // for two coils; each lane rounds as fmaf does)
    float2 ar[P][NC / 2], ai[P][NC / 2];
#pragma unroll
    for (int j = 0; j < P; ++j)
#pragma unroll
        for (int k = 0; k < NC / 2; ++k) { ar[j][k] = make_float2(0.f, 0.f); ai[j][k] = make_float2(0.f, 0.f); }
    auto run = [&](auto mode_tag) {
        constexpr int MODE = decltype(mode_tag)::value;  // 0: MUFU.EX2 per sample, 1: series from sample 0
#pragma unroll 2
        for (int s = 0; s < cnt; ++s) {
            float cr[P], ci[P];
#pragma unroll
            for (int j = 0; j < P; ++j) { cr[j] = 0.f; ci[j] = 0.f; }
            signal_spin_fp32<P, MODE>(kx, ky, kz, tau, cj, shA[s], shS[s], cr, ci);
#pragma unroll
            for (int k = 0; k < NC / 2; ++k) {
                const float4 w = shW[s * (NC / 2) + k];  // two coils' weights as (re, re', im, im')
                const float2 wr = make_float2(w.x, w.y), wi = make_float2(w.z, w.w);
#pragma unroll
                for (int j = 0; j < P; ++j) {
                    const float2 c2 = make_float2(cr[j], cr[j]), d2 = make_float2(ci[j], ci[j]),
                                 n2 = make_float2(-ci[j], -ci[j]);
                    ar[j][k] = __ffma2_rn(c2, wr, __ffma2_rn(n2, wi, ar[j][k]));
                    ai[j][k] = __ffma2_rn(c2, wi, __ffma2_rn(d2, wr, ai[j][k]));
                }
            }
        }
    };
    if (series) run(std::integral_constant<int, 1>{});
    else run(std::integral_constant<int, 0>{});
#pragma unroll
    for (int j = 0; j < P; ++j)
        if (p0 + j < n_pts) {
#pragma unroll
            for (int k = 0; k < NC / 2; ++k) {
                out[(size_t)(2 * k) * slot_stride + p0 + j] = make_float2(ar[j][k].x, ai[j][k].x);
                out[(size_t)(2 * k + 1) * slot_stride + p0 + j] = make_float2(ar[j][k].y, ai[j][k].y);
            }
        }
}

template <int NC, int P>
__device__ __forceinline__ void seq_signal_block_coils(const float4 *__restrict__ recs, int n_pts, const float4 *shA,
                                                       const float4 *shS, const float4 *shW, int cnt, int lane,
                                                       int *item_ctr, float r2max_log2e, int slot_stride,
                                                       float2 *__restrict__ out) {
    for (;;) {
        int item = 0;
        if (lane == 0) item = atomicAdd(item_ctr, 1);
        item = __shfl_sync(0xffffffffu, item, 0);
        const int base = item * (32 * P);
        if (base >= n_pts) break;
        seq_signal_item_coils<NC, P>(recs, n_pts, base, shA, shS, shW, cnt, lane, r2max_log2e, slot_stride, out);
    }
}

// PS: PER_SPIN plans (a separate instantiation so that the SUM_ALL kernel keeps its 64 registers without spills)
// NC: receive coils per spin record (0: none; 4 or 8: SUM_ALL plans with up to NC coils, sums per coil in the same launch)
template <bool PS, int NC>
__global__ void __launch_bounds__(kSeqMaxThreads, 1)
seq_kernel(const unsigned char *__restrict__ tables, const SeqOp *__restrict__ ops, int n_ops,
           const float4 *__restrict__ A, const float4 *__restrict__ Cc, float4 *__restrict__ S, int n, int chunk,
           int rf_warps, SeqRoles roles, int min_items, const float *__restrict__ scal,
           float2 *__restrict__ prow /* [ring_slots][n_ctas][slot_stride] partial rows */, int ring_slots, int slot_stride,
           int *__restrict__ tickets /* [2][n_adc_blocks]: arrive, reduced; zeroed before the launch */, int n_adc_blocks,
           const SeqAdcBlock *__restrict__ adc_blocks /* [n_adc_blocks] */,
           float2 *__restrict__ sig /* SUM_ALL: signal[n_adc] */,
           long long n_adc, int final_state, float2 *__restrict__ out_ps /* PER_SPIN plans: out[spin][adc], else NULL */,
           const float4 *__restrict__ Wc /* NC > 0: NC / 2 float4 of coil weights per spin (pack_coils_kernel) */,
           int n_coils /* NC > 0: rows of sig, [n_coils][n_adc] */) {
    static_assert(NC == 0 || ((NC == 4 || NC == 8) && !PS), "coils: SUM_ALL plans, 4 or 8 weights per spin record");
    extern __shared__ __align__(128) unsigned char smem[];
    unsigned char *ring = smem;
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + kSeqStages * kSeqTileStride);
    uint64_t *tile_full = bars, *tile_empty = bars + kSeqStages, *st_full = bars + 2 * kSeqStages,
             *st_empty = bars + 2 * kSeqStages + kSeqStateBufs;
    int *item_ctr = reinterpret_cast<int *>(bars + 2 * kSeqStages + 2 * kSeqStateBufs);  // [kSeqStateBufs]
    int *fin_ctr = item_ctr + kSeqStateBufs;  // [kSeqStateBufs]: signal warps that have finished the block
    float4 *shA = reinterpret_cast<float4 *>(smem + kSeqStages * kSeqTileStride + kSeqBarBytes);
    float4 *shS = shA + chunk;  // [kSeqStateBufs][chunk]
    float4 *shW = shS + kSeqStateBufs * chunk;  // NC > 0: [chunk][NC / 2]
    const int tid = threadIdx.x, warp = tid >> 5;
    const int n_rf_thr = rf_warps * 32;
    const int nsig = roles.n_sig_warps * 32;
    const int my_role = roles.role[warp];
    const int s0 = blockIdx.x * chunk;
    const int cnt = min(chunk, n - s0);
    if (tid == 0) {
        for (int k = 0; k < kSeqStages; ++k) {
            mbar_init(&tile_full[k], 1);
            mbar_init(&tile_empty[k], n_rf_thr);
        }
        for (int k = 0; k < kSeqStateBufs; ++k) {
            mbar_init(&st_full[k], n_rf_thr);
            mbar_init(&st_empty[k], max(nsig, 1));
            item_ctr[k] = 0;
            fin_ctr[k] = 0;
        }
        mbar_init_fence();
    }
    __syncthreads();  // the only CTA-wide barrier: from here on the roles meet at mbarriers
    if (my_role == kRoleIdle) return;

    if (my_role == kRoleProducer) {
        // ---------------------------------------------------------------- producer
        if ((tid & 31) != 0) return;
        int g = 0;
        for (int oi = 0; oi < n_ops; ++oi) {
            const int2 tn = *reinterpret_cast<const int2 *>(&ops[oi]);
            if (tn.x != kBlockRF) continue;
            const unsigned char *tbl = tables + ops[oi].table_off;
            const int2 *dir = reinterpret_cast<const int2 *>(tbl);
            for (int t = 0; t < tn.y; ++t, ++g) {
                const int st = g % kSeqStages, use = g / kSeqStages;
                if (use > 0) mbar_wait(&tile_empty[st], (uint32_t)((use - 1) & 1));
                const int2 d = dir[t];
                mbar_expect_tx(&tile_full[st], (uint32_t)d.y);
                bulk_g2s(ring + st * kSeqTileStride, tbl + d.x, (uint32_t)d.y, &tile_full[st]);
            }
        }
        return;
    }

    if (my_role >= 0) {
        // ---------------------------------------------------------------- RF warps: one spin per thread
        const int r = my_role * 32 + (tid & 31);
        const bool active = r < cnt;
        const int i = s0 + r;
        float4 a = make_float4(0.f, 0.f, 0.f, 0.f), c = make_float4(1.f, 1.f, 0.f, 0.f),
               s = make_float4(0.f, 0.f, 0.f, 0.f);
        const float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
        if (active) {
            a = A[i];
            c = Cc[i];
            s = S[i];
            shA[r] = a;
            if constexpr (NC > 0) {  // visible to the signal warps with the first published state (st_full)
#pragma unroll
                for (int k = 0; k < NC / 2; ++k) {  // (re, im, re', im') of coils 2k, 2k + 1 -> (re, re', im, im')
                    const float4 w = Wc[(size_t)i * (NC / 2) + k];
                    shW[r * (NC / 2) + k] = make_float4(w.x, w.z, w.y, w.w);
                }
            }
        }
        float hx = s.x, hy = s.y, hz = s.z, lx = 0.f, ly = 0.f, lz = 0.f;
        const RfSpin sp{a.x, a.y, a.z, c.w, c.x, c.y, c.z, 0.f, 0.f, 0.f};
        const float ax = fabsf(sp.x), ay = fabsf(sp.y), az = fabsf(sp.z), adw = fabsf(sp.dw);
        bool pending = false;
        PropRec prop{0, 0, 0, 0, 0, 0, 0};
        int g = 0, pub = 0;
        for (int oi = 0; oi < n_ops; ++oi) {
            const int2 tn = *reinterpret_cast<const int2 *>(&ops[oi]);
            if (pending) {  // end transform of the precession block before this one (Eq 10-11 in closed form)
                propagate(prop, a, c, v, hx, hy, hz);
                pending = false;
            }
            if (tn.x == kBlockRF) {
                for (int t = 0; t < tn.y; ++t, ++g) {
                    const int st = g % kSeqStages;
                    mbar_wait(&tile_full[st], (uint32_t)((g / kSeqStages) & 1));
                    const unsigned char *tile = ring + st * kSeqTileStride;
                    const RfTileHdr hd = *reinterpret_cast<const RfTileHdr *>(tile);
                    RfRelax rx;
                    rx.D1 = -expm1f(-hd.dt * sp.r1);
                    rx.D2 = -expm1f(-hd.dt * sp.r2);
                    rx.E1 = 1.0f - rx.D1;
                    rx.E2 = 1.0f - rx.D2;
                    rx.D1m0 = rx.D1 * sp.m0;
                    const float wzb = fmaf(hd.gx_max, ax, fmaf(hd.gy_max, ay, fmaf(hd.gz_max, az, hd.dt * adw)));
                    const float qb = fmaf(wzb, wzb, hd.wxy2_max);
                    const bool uni = (hd.flags & kRfFlagUniformG) != 0;
                    const int tier = __all_sync(0xffffffffu, qb <= kRfQLin) ? -1
                                     : (__all_sync(0xffffffffu, qb <= 0.00390625f) ? 0
                                        : (__all_sync(0xffffffffu, qb <= 0.25f) ? 1 : 2));
#define BLOCH_SEQ_TILE(T)                                                          \
    do {                                                                           \
        if (uni) rf_tile<T, 0>(tile, hd, sp, rx, hx, hy, hz, lx, ly, lz);          \
        else rf_tile<T, 1>(tile, hd, sp, rx, hx, hy, hz, lx, ly, lz);              \
    } while (0)
                    if (tier == -1) BLOCH_SEQ_TILE(-1);
                    else if (tier == 0) BLOCH_SEQ_TILE(0);
                    else if (tier == 1) BLOCH_SEQ_TILE(1);
                    else BLOCH_SEQ_TILE(2);
#undef BLOCH_SEQ_TILE
                    mbar_arrive(&tile_empty[st]);  // this thread is done reading the stage
                }
                // round the state to one float per component, as rf_kernel stores it between launches
                hx += lx; hy += ly; hz += lz;
                lx = 0.f; ly = 0.f; lz = 0.f;
            } else {
                if (PS && tn.y > 0) {
                    // PER_SPIN output (dictionary mode; blocks of a few samples): the spin's own thread evaluates
                    // them with the accurate functions and fp64 phase of perspin_kernel -- no signal warps
                    const void *recs = tables + ops[oi].table_off;
                    float2 *row = out_ps + (size_t)i * (size_t)n_adc + ops[oi].adc_first;
                    const float4 now = make_float4(hx, hy, hz, s.w);
                    for (int p = 0; p < tn.y; ++p) {
                        const float2 w = accurate_contribution(load_point<false>(recs, p, false), a, c, now, nullptr);
                        if (active) row[p] = w;
                    }
                } else if (tn.y > 0) {  // publish the block-start state for the signal warps
                    const int b = pub % kSeqStateBufs, use = pub / kSeqStateBufs;
                    if (use > 0) mbar_wait(&st_empty[b], (uint32_t)((use - 1) & 1));
                    if (active) shS[b * chunk + r] = make_float4(hx, hy, hz, s.w);
                    if (r == 0) { item_ctr[b] = 0; fin_ctr[b] = 0; }  // every signal warp is past its last atomicAdd of the previous use
                    mbar_arrive(&st_full[b]);
                    ++pub;
                }
                const double4 k4 = *reinterpret_cast<const double4 *>(&ops[oi].kend[0]);
                prop.kx = k4.x; prop.ky = k4.y; prop.kz = k4.z; prop.tau = k4.w;
                pending = k4.w != 0.0;  // an empty block (an ADC sample inside an RF run) has nothing to propagate
            }
        }
        if (final_state) {
            if (pending) propagate(prop, a, c, v, hx, hy, hz);
            if (active) S[i] = make_float4(hx, hy, hz, s.w);
        }
        return;
    }

    // -------------------------------------------------------------------- signal warps
    {
        const int lane = tid & 31;
        const float r2max_log2e = scal[0] * kLog2e;
        const int n_ctas = gridDim.x, cta = blockIdx.x;
        int *arrive = tickets, *reduced = tickets + n_adc_blocks;
        const size_t row_elems = (size_t)(NC > 0 ? NC : 1) * slot_stride;  // one CTA's row(s) of a block
        const size_t slot_elems = (size_t)n_ctas * row_elems;
        int pub = 0;  // = index of the block among the ADC-bearing precession blocks (adc_blocks[pub])
        for (int oi = 0; oi < n_ops; ++oi) {
            const int2 tn = *reinterpret_cast<const int2 *>(&ops[oi]);
            if (tn.x != kBlockPrecession || tn.y == 0) continue;
            const float4 *recs = reinterpret_cast<const float4 *>(tables + ops[oi].table_off);
            // the ring slot is free once every CTA has summed its slice of the block that used it before
            if (pub >= ring_slots) wait_ticket(&reduced[pub - ring_slots], n_ctas, lane);
            float2 *out = prow + (size_t)(pub % ring_slots) * slot_elems + (size_t)cta * row_elems;
            const int b = pub % kSeqStateBufs;
            mbar_wait(&st_full[b], (uint32_t)((pub / kSeqStateBufs) & 1));
            const float4 *stS = shS + b * chunk;
            // item size: the largest P that still leaves min_items items (about one per signal warp)
            if constexpr (NC > 0) {
                // two samples per lane with up to 4 coils when that still leaves an item for every signal warp
                if (NC == 4 && tn.y >= 64 * roles.n_sig_warps)
                    seq_signal_block_coils<NC, NC == 4 ? 2 : 1>(recs, tn.y, shA, stS, shW, cnt, lane, &item_ctr[b], r2max_log2e, slot_stride, out);
                else
                    seq_signal_block_coils<NC, 1>(recs, tn.y, shA, stS, shW, cnt, lane, &item_ctr[b], r2max_log2e, slot_stride, out);
            } else if (tn.y >= 128 * min_items) seq_signal_block<4>(recs, tn.y, shA, stS, cnt, lane, &item_ctr[b], r2max_log2e, out);
            else if (tn.y >= 64 * min_items) seq_signal_block<2>(recs, tn.y, shA, stS, cnt, lane, &item_ctr[b], r2max_log2e, out);
            else seq_signal_block<1>(recs, tn.y, shA, stS, cnt, lane, &item_ctr[b], r2max_log2e, out);
            // the warp that finishes the block last in this CTA announces the CTA's row and takes the CTA's reduce duty
            __syncwarp();
            int last = 0;
            if (lane == 0) {
                __threadfence();  // this warp's partial sums are visible before it counts itself done
                last = atomicAdd(&fin_ctr[b], 1) == roles.n_sig_warps - 1;
            }
            last = __shfl_sync(0xffffffffu, last, 0);
            mbar_arrive(&st_empty[b]);
            if (last) {
                if (lane == 0) {
                    __threadfence();
                    atomicAdd(&arrive[pub], 1);
                }
                // this CTA's slice of the block finished kSeqReduceLag blocks ago; after the last block, of the rest too
                const int h_hi = pub == n_adc_blocks - 1 ? pub : pub - kSeqReduceLag;
                for (int h = max(pub - kSeqReduceLag, 0); h <= h_hi; ++h) {
                    const SeqAdcBlock ab = adc_blocks[h];
                    if constexpr (NC > 0)
                        seq_reduce_slice_coils(prow + (size_t)(h % ring_slots) * slot_elems, slot_stride, NC, n_ctas, cta,
                                               ab.n, sig + ab.adc_first, n_adc, n_coils, lane, &arrive[h], &reduced[h]);
                    else
                        seq_reduce_slice(prow + (size_t)(h % ring_slots) * slot_elems, slot_stride, n_ctas, cta, ab.n,
                                         sig + ab.adc_first, lane, &arrive[h], &reduced[h]);
                }
            }
            ++pub;
        }
    }
}

}  // namespace bloch
