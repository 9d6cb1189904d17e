// rf.cuh -- a8: RF (excitation) kernel for sm_100a.  One thread = one spin; the magnetisation stays in
// registers for the whole excitation block; the block's step table is streamed through shared memory tile
// by tile with 1-D bulk copies (TMA) into a two-stage mbarrier ring and broadcast to all threads.
//
// Per step the Cayley-Klein rotation of Eq 6-9 is applied in its increment form.  With
// the rotation vector w = gamma * (B1x, B1y, Bz) * dt (so phi = -|w| in Eq 8),
//     alpha = cos(|w|/2) + i (wz/|w|) sin(|w|/2),   beta = i ((wx + i wy)/|w|) sin(|w|/2),
// Eq 9 expanded in real components is identically
//     M+ = M + a (w x M) + b (w x (w x M)),     a = -sin|w| / |w|,     b = (1 - cos|w|) / |w|^2
// (tests/test_host_plan.py checks the identity against Eq 9 numerically).  a and b are even series in
// q = |w|^2: no sqrt, no division, no 0/0 at |B| = 0 (reading G10), and 1 - cos is never formed by
// cancellation (SURVEY.md hard parts H1/H2).  Relaxation (Eq 11, :160-163) follows the rotation in the same
// increment form with D = -expm1(-dt/T):   M++ = M + [E d - D M (+ D1 M0 z)],  d the rotation increment.
//
// The work per step is chosen per tile and per warp from a bound on q (tile header maxima x the spin's own
// |x|, |y|, |z|, |dw|), so the hot loops are branch-free:
//   tier -1 q <= 2^-14: series through q only (the q^2 terms are below q^2.5 / 120 = 2.4e-13 |M| per step: 2.4e-7 over the
//                       1e6 steps of an MRF schedule), otherwise as tier 0 -- every pulse of the five configs
//   tier 0  q <= 2^-8 : series through q^2 (truncation < 1.2e-11), state carried as hi + lo with the
//                       increments summed in lo and folded into hi every 8 steps (error-free Fast2Sum)
//   tier 1  q <= 1/4  : series through q^3 (truncation < 1.1e-8), Kahan-compensated state
//   tier 2  otherwise : sqrt + sincos per step where needed, Kahan-compensated state
// Tiles whose gradient part is the same for every step (compact records) hoist wz out of the step loop.
#pragma once
#include "internal.h"
#include "kernels.cuh"
#include "tma.cuh"

namespace bloch {

struct RfSpin {
    float x, y, z, dw, r1, r2, m0;
    float vx, vy, vz;  // motion plans (x(t) = x + v t); zero otherwise
};
struct RfRelax {
    float E1, E2, D1, D2, D1m0;
};

template <int TIER>
__device__ __forceinline__ void rf_series(float q, float &ca, float &cb) {
    if (TIER == -1) {
        ca = fmaf(q, 1.0f / 6.0f, -1.0f);
        cb = fmaf(q, -1.0f / 24.0f, 0.5f);
    } else if (TIER == 0) {
        ca = fmaf(q, fmaf(q, -1.0f / 120.0f, 1.0f / 6.0f), -1.0f);
        cb = fmaf(q, fmaf(q, 1.0f / 720.0f, -1.0f / 24.0f), 0.5f);
    } else if (TIER == 1) {
        ca = fmaf(q, fmaf(q, fmaf(q, 1.0f / 5040.0f, -1.0f / 120.0f), 1.0f / 6.0f), -1.0f);
        cb = fmaf(q, fmaf(q, fmaf(q, -1.0f / 40320.0f, 1.0f / 720.0f), -1.0f / 24.0f), 0.5f);
    } else {
        if (q <= 0.25f) {
            ca = fmaf(q, fmaf(q, fmaf(q, 1.0f / 5040.0f, -1.0f / 120.0f), 1.0f / 6.0f), -1.0f);
            cb = fmaf(q, fmaf(q, fmaf(q, -1.0f / 40320.0f, 1.0f / 720.0f), -1.0f / 24.0f), 0.5f);
        } else {
            const float t = sqrtf(q);
            float sh, ch;
            sincosf(0.5f * t, &sh, &ch);
            ca = -2.0f * sh * ch / t;  // -sin t / t
            cb = 2.0f * sh * sh / q;   // (1 - cos t) / t^2
        }
    }
}

// increment of one step (rotation Eq 9, then relaxation Eq 11) for the state (mx, my, mz)
template <int TIER>
__device__ __forceinline__ void rf_increment(float wx, float wy, float wz, float q, float mx, float my, float mz,
                                             const RfRelax &r, float &tx, float &ty, float &tz) {
    float ca, cb;
    rf_series<TIER>(q, ca, cb);
    const float ux = fmaf(wy, mz, -wz * my);  // u = w x M
    const float uy = fmaf(wz, mx, -wx * mz);
    const float uz = fmaf(wx, my, -wy * mx);
    const float vx = fmaf(wy, uz, -wz * uy);  // v = w x u
    const float vy = fmaf(wz, ux, -wx * uz);
    const float vz = fmaf(wx, uy, -wy * ux);
    const float dx = fmaf(ca, ux, cb * vx);
    const float dy = fmaf(ca, uy, cb * vy);
    const float dz = fmaf(ca, uz, cb * vz);
    tx = fmaf(r.E2, dx, -r.D2 * mx);
    ty = fmaf(r.E2, dy, -r.D2 * my);
    tz = fmaf(r.E1, dz, fmaf(-r.D1, mz, r.D1m0));
}

// The same step for the hi + lo tiers (TIER <= 0), added straight into the low part: l <- l + E d - D m (+ D1 M0 z),
// the sum folded into the FMAs that form the increment (two instructions per component instead of three).
template <int TIER>
__device__ __forceinline__ void rf_accumulate(float wx, float wy, float wz, float q, float mx, float my, float mz,
                                              const RfRelax &r, float &lx, float &ly, float &lz) {
    float ca, cb;
    rf_series<TIER>(q, ca, cb);
    const float ux = fmaf(wy, mz, -wz * my);  // u = w x M
    const float uy = fmaf(wz, mx, -wx * mz);
    const float uz = fmaf(wx, my, -wy * mx);
    const float vx = fmaf(wy, uz, -wz * uy);  // v = w x u
    const float vy = fmaf(wz, ux, -wx * uz);
    const float vz = fmaf(wx, uy, -wy * ux);
    const float dx = fmaf(ca, ux, cb * vx);
    const float dy = fmaf(ca, uy, cb * vy);
    const float dz = fmaf(ca, uz, cb * vz);
    lx = fmaf(r.E2, dx, fmaf(-r.D2, mx, lx));
    ly = fmaf(r.E2, dy, fmaf(-r.D2, my, ly));
    lz = fmaf(r.E1, dz, fmaf(-r.D1, mz, lz + r.D1m0));
}

__device__ __forceinline__ void kahan_add(float &m, float &c, float d) {
    const float yv = d - c;
    const float t = m + yv;
    c = (t - m) - yv;
    m = t;
}

// hi <- fl(hi + lo), lo <- the rounding error of that sum (Fast2Sum; |lo| << |hi| here, and where it is not
// the residual is below an ulp of lo)
__device__ __forceinline__ void fold(float &hi, float &lo) {
    const float s = hi + lo;
    lo -= (s - hi);
    hi = s;
}

// Hi + lo tiers (TIER <= 0): the step loop is unrolled rf_fold(TIER) deep and the low part is folded into the high part
// once per trip.  The loop is instruction-bound, so the loop overhead (9 instructions per trip) and the folds (9 per fold)
// both show.  Measured with tier -1 (every pulse of the configs), rf ms per step of config 4 / whole-sequence ms of
// config 5 / 5b: 4 steps per fold: 43.2; 8: 39.1 / 119.3 / 136.3; 16: 37.9 / 118.7 / 132.0; 24: 37.9 / 116.9 / 133.7;
// 32: 37.6 / 115.0 / 131.6 (unrolled 32 deep but folded every 16: 37.9 / 119.0 / 134.5; every 8: 38.4 / 118.1 / 134.7).
// |l| stays below fold |w| |M|: tier -1 (|w| <= 2^-7) takes 32, so that |l| <= |M| / 4 and the sums into l round at
// 2^-26 |M| or finer (2^-28 |M| with 8: the final magnetisation of config 5, 1e6 steps, moved from NRMSE 3.3e-7 to
// 5.2e-7 against the whole oracle, tolerance 1e-5; every signal unchanged to the digits printed); tier 0
// (|w| <= 2^-4) keeps 8, |l| <= |M| / 2.
__host__ __device__ constexpr int rf_fold(int tier) { return tier < 0 ? 32 : 8; }

// One tile of steps.  State in and out as (h, l) with h + l the magnetisation.
// MODE 0: compact records (uniform gradient part), 1: general records, 2: general + motion records.
template <int TIER, int MODE>
__device__ __forceinline__ void rf_tile(const unsigned char *tile, const RfTileHdr &hd, const RfSpin &sp,
                                        const RfRelax &rx, float &hx, float &hy, float &hz, float &lx, float &ly,
                                        float &lz) {
    const float4 *rec = reinterpret_cast<const float4 *>(tile + kRfHdrBytes);
    const int n = hd.n_steps;
    const float dtdw = hd.dt * sp.dw;
    // Eq 2: gamma Bz dt = g . x + dw dt
    const float wz_u = fmaf(hd.gx, sp.x, fmaf(hd.gy, sp.y, fmaf(hd.gz, sp.z, dtdw)));
    const float wz2_u = __fmul_rn(wz_u, wz_u);  // __fmul_rn / __fadd_rn: no contraction, rf_kernel and seq_kernel round alike
#define BLOCH_RF_LOAD(k)                                                              \
    float wx, wy, wz, q;                                                              \
    if (MODE == 0) {                                                                  \
        const float4 a = rec[k];                                                      \
        wx = a.x; wy = a.y; wz = wz_u; q = __fadd_rn(a.z, wz2_u);                              \
    } else if (MODE == 1) {                                                           \
        const float4 a = rec[2 * (k)], g = rec[2 * (k) + 1];                          \
        wx = a.x; wy = a.y;                                                           \
        wz = fmaf(g.x, sp.x, fmaf(g.y, sp.y, fmaf(g.z, sp.z, dtdw)));                 \
        q = fmaf(wz, wz, a.z);                                                        \
    } else {                                                                          \
        const float4 a = rec[3 * (k)], g = rec[3 * (k) + 1], h = rec[3 * (k) + 2];    \
        wx = a.x; wy = a.y;                                                           \
        wz = fmaf(g.x, sp.x, fmaf(g.y, sp.y, fmaf(g.z, sp.z, dtdw)));                 \
        wz = fmaf(h.x, sp.vx, fmaf(h.y, sp.vy, fmaf(h.z, sp.vz, wz)));                \
        q = fmaf(wz, wz, a.z);                                                        \
    }
    if (TIER <= 0) {
        int k = 0;
        constexpr int kFold = rf_fold(TIER);
        for (; k + kFold <= n; k += kFold) {
#pragma unroll
            for (int j = 0; j < kFold; ++j) {
                BLOCH_RF_LOAD(k + j)
                rf_accumulate<TIER>(wx, wy, wz, q, hx + lx, hy + ly, hz + lz, rx, lx, ly, lz);
            }
            fold(hx, lx); fold(hy, ly); fold(hz, lz);
        }
        for (; k < n; ++k) {
            BLOCH_RF_LOAD(k)
            rf_accumulate<TIER>(wx, wy, wz, q, hx + lx, hy + ly, hz + lz, rx, lx, ly, lz);
        }
        fold(hx, lx); fold(hy, ly); fold(hz, lz);
    } else {
        float cx = -lx, cy = -ly, cz = -lz;  // Kahan carries the negated low part
#pragma unroll 4
        for (int k = 0; k < n; ++k) {
            BLOCH_RF_LOAD(k)
            float tx, ty, tz;
            rf_increment<TIER>(wx, wy, wz, q, hx, hy, hz, rx, tx, ty, tz);
            kahan_add(hx, cx, tx);
            kahan_add(hy, cy, ty);
            kahan_add(hz, cz, tz);
        }
        lx = -cx; ly = -cy; lz = -cz;
    }
#undef BLOCH_RF_LOAD
}

// Tier-0 tile for TWO spins per thread (static plans).  The step record (wx, wy, wx^2 + wy^2 and, on general tiles, g)
// is warp-uniform and the same for both spins, so it is loaded once, and the two spins' cross products sit next to
// each other in the instruction stream with wx, wy in the same operand slot (the operand-reuse cache can then serve
// the second read: the RF step is bound by register-file operand bandwidth).  Each spin's own
// arithmetic is rf_accumulate<TIER> exactly as in rf_tile<TIER, MODE>, so the result is bitwise that of one spin per thread.
template <int TIER, int MODE>
__device__ __forceinline__ void rf_tile0_pair(const unsigned char *tile, const RfTileHdr &hd, const RfSpin &sa,
                                              const RfSpin &sb, const RfRelax &ra, const RfRelax &rb, float (&h)[6],
                                              float (&l)[6]) {
    const float4 *rec = reinterpret_cast<const float4 *>(tile + kRfHdrBytes);
    const int n = hd.n_steps;
    const float dtdw_a = hd.dt * sa.dw, dtdw_b = hd.dt * sb.dw;
    const float wz_ua = fmaf(hd.gx, sa.x, fmaf(hd.gy, sa.y, fmaf(hd.gz, sa.z, dtdw_a)));
    const float wz_ub = fmaf(hd.gx, sb.x, fmaf(hd.gy, sb.y, fmaf(hd.gz, sb.z, dtdw_b)));
    const float wz2_ua = __fmul_rn(wz_ua, wz_ua), wz2_ub = __fmul_rn(wz_ub, wz_ub);
#define BLOCH_RF_PAIR_STEP(k)                                                                          \
    {                                                                                                  \
        float wx, wy, wza, wzb, qa, qb;                                                                \
        if (MODE == 0) {                                                                               \
            const float4 a = rec[k];                                                                   \
            wx = a.x; wy = a.y; wza = wz_ua; wzb = wz_ub;                                              \
            qa = __fadd_rn(a.z, wz2_ua); qb = __fadd_rn(a.z, wz2_ub);                                  \
        } else {                                                                                       \
            const float4 a = rec[2 * (k)], g = rec[2 * (k) + 1];                                       \
            wx = a.x; wy = a.y;                                                                        \
            wza = fmaf(g.x, sa.x, fmaf(g.y, sa.y, fmaf(g.z, sa.z, dtdw_a)));                           \
            wzb = fmaf(g.x, sb.x, fmaf(g.y, sb.y, fmaf(g.z, sb.z, dtdw_b)));                           \
            qa = fmaf(wza, wza, a.z); qb = fmaf(wzb, wzb, a.z);                                        \
        }                                                                                              \
        rf_accumulate<TIER>(wx, wy, wza, qa, h[0] + l[0], h[1] + l[1], h[2] + l[2], ra, l[0], l[1], l[2]);    \
        rf_accumulate<TIER>(wx, wy, wzb, qb, h[3] + l[3], h[4] + l[4], h[5] + l[5], rb, l[3], l[4], l[5]);    \
    }
    int k = 0;
    constexpr int kFold = rf_fold(TIER);  // as rf_tile: bitwise the one-spin kernel
    for (; k + kFold <= n; k += kFold) {
#pragma unroll
        for (int j = 0; j < kFold; ++j) BLOCH_RF_PAIR_STEP(k + j)
#pragma unroll
        for (int c = 0; c < 6; ++c) fold(h[c], l[c]);
    }
    for (; k < n; ++k) BLOCH_RF_PAIR_STEP(k)
#pragma unroll
    for (int c = 0; c < 6; ++c) fold(h[c], l[c]);
#undef BLOCH_RF_PAIR_STEP
}

constexpr int kRfMaxThreads = 128;
constexpr float kRfQLin = 6.103515625e-05f;  // 2^-14: below it the series of a, b stop at the term linear in q (tier -1)

// MO: motion plans (48-B step records, velocities); the static instantiation keeps its registers and shared
// memory (48 registers, 8.3 KB) so that 10 CTAs of 128 threads fit an SM.
template <bool MO>
__global__ void __launch_bounds__(kRfMaxThreads)
rf_kernel(const unsigned char *__restrict__ tbl, int n_tiles, PropRec prop, int has_prop,
          const float4 *__restrict__ A, const float4 *__restrict__ Cc, float4 *__restrict__ S,
          const float4 *__restrict__ V /* motion plans, else NULL */, int n) {
    __shared__ __align__(128) unsigned char buf[2][kRfHdrBytes + kRfTileSteps * (MO ? 48 : 32)];
    __shared__ __align__(8) uint64_t bar[2];
    const int tid = threadIdx.x;
    const int2 *dir = reinterpret_cast<const int2 *>(tbl);
    if (tid == 0 && n_tiles > 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        mbar_init_fence();
        for (int b = 0; b < 2 && b < n_tiles; ++b) {
            const int2 d = dir[b];
            mbar_expect_tx(&bar[b], (uint32_t)d.y);
            bulk_g2s(buf[b], tbl + d.x, (uint32_t)d.y, &bar[b]);
        }
    }
    const int i = blockIdx.x * blockDim.x + tid;
    const bool active = i < n;
    float4 a = make_float4(0.f, 0.f, 0.f, 0.f), c = make_float4(1.f, 1.f, 0.f, 0.f),
           s = make_float4(0.f, 0.f, 0.f, 0.f);
    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
    if (active) {
        a = A[i];
        c = Cc[i];
        s = S[i];
        if (MO) v = V[i];
    }
    float hx = s.x, hy = s.y, hz = s.z;
    if (has_prop) propagate(prop, a, c, v, hx, hy, hz);
    float lx = 0.f, ly = 0.f, lz = 0.f;
    const RfSpin sp{a.x, a.y, a.z, c.w, c.x, c.y, c.z, v.x, v.y, v.z};
    const float ax = fabsf(sp.x), ay = fabsf(sp.y), az = fabsf(sp.z), adw = fabsf(sp.dw);
    const float avx = fabsf(v.x), avy = fabsf(v.y), avz = fabsf(v.z);
    __syncthreads();  // barrier initialisation visible to every waiter

    for (int t = 0; t < n_tiles; ++t) {
        const int b = t & 1;
        mbar_wait(&bar[b], (uint32_t)((t >> 1) & 1));
        const unsigned char *tile = buf[b];
        const RfTileHdr hd = *reinterpret_cast<const RfTileHdr *>(tile);
        RfRelax rx;
        rx.D1 = -expm1f(-hd.dt * sp.r1);
        rx.D2 = -expm1f(-hd.dt * sp.r2);
        rx.E1 = 1.0f - rx.D1;
        rx.E2 = 1.0f - rx.D2;
        rx.D1m0 = rx.D1 * sp.m0;
        // bound on q = |w|^2 over the tile for this spin -> tier, decided per warp
        float wzb = fmaf(hd.gx_max, ax, fmaf(hd.gy_max, ay, fmaf(hd.gz_max, az, hd.dt * adw)));
        if (MO) wzb = fmaf(hd.hx_max, avx, fmaf(hd.hy_max, avy, fmaf(hd.hz_max, avz, wzb)));
        const float qb = fmaf(wzb, wzb, hd.wxy2_max);
        const int mode = MO ? 2 : ((hd.flags & kRfFlagUniformG) ? 0 : 1);  // motion plans hold motion tiles only
        const int tier = __all_sync(0xffffffffu, qb <= kRfQLin) ? -1
                         : (__all_sync(0xffffffffu, qb <= 0.00390625f) ? 0 : (__all_sync(0xffffffffu, qb <= 0.25f) ? 1 : 2));
#define BLOCH_RF_TILE(T, M) rf_tile<T, M>(tile, hd, sp, rx, hx, hy, hz, lx, ly, lz)
#define BLOCH_RF_MODES(T)                       \
    do {                                        \
        if (MO) BLOCH_RF_TILE(T, 2);            \
        else if (mode == 0) BLOCH_RF_TILE(T, 0);\
        else BLOCH_RF_TILE(T, 1);               \
    } while (0)
        if (tier == -1) BLOCH_RF_MODES(-1);
        else if (tier == 0) BLOCH_RF_MODES(0);
        else if (tier == 1) BLOCH_RF_MODES(1);
        else BLOCH_RF_MODES(2);
#undef BLOCH_RF_MODES
#undef BLOCH_RF_TILE
        __syncthreads();  // every thread is done reading buf[b]
        if (tid == 0 && t + 2 < n_tiles) {
            const int2 d = dir[t + 2];
            mbar_expect_tx(&bar[b], (uint32_t)d.y);
            bulk_g2s(buf[b], tbl + d.x, (uint32_t)d.y, &bar[b]);
        }
    }
    if (active) S[i] = make_float4(hx + lx, hy + ly, hz + lz, s.w);
}

// One compact tile whose step records come from the kernel's parameter space (constant bank): the arithmetic of
// rf_tile<TIER, 0>, operation for operation, so the result is bitwise that of rf_kernel.
template <int TIER>
__device__ __forceinline__ void rf_ctile(const RfConstArgs &args, int base, const RfConstTile &hd, const RfSpin &sp,
                                         const RfRelax &rx, float &hx, float &hy, float &hz, float &lx, float &ly,
                                         float &lz) {
    const int n = hd.n_steps;
    const float dtdw = hd.dt * sp.dw;
    const float wz_u = fmaf(hd.gx, sp.x, fmaf(hd.gy, sp.y, fmaf(hd.gz, sp.z, dtdw)));
    const float wz2_u = __fmul_rn(wz_u, wz_u);
#define BLOCH_RFC_LOAD(k)                                                                         \
    const float wx = args.rec[4 * (base + (k))], wy = args.rec[4 * (base + (k)) + 1], wz = wz_u,    \
                q = __fadd_rn(args.rec[4 * (base + (k)) + 2], wz2_u);
    if (TIER <= 0) {
        int k = 0;
        constexpr int kFold = rf_fold(TIER);
        for (; k + kFold <= n; k += kFold) {
            const int o = 4 * (base + k);  // one uniform offset per trip; the unrolled steps are immediates from it
#pragma unroll
            for (int j = 0; j < kFold; ++j) {
                const float wx = args.rec[o + 4 * j], wy = args.rec[o + 4 * j + 1], wz = wz_u,
                            q = __fadd_rn(args.rec[o + 4 * j + 2], wz2_u);
                rf_accumulate<TIER>(wx, wy, wz, q, hx + lx, hy + ly, hz + lz, rx, lx, ly, lz);
            }
            fold(hx, lx); fold(hy, ly); fold(hz, lz);
        }
        for (; k < n; ++k) {
            BLOCH_RFC_LOAD(k)
            rf_accumulate<TIER>(wx, wy, wz, q, hx + lx, hy + ly, hz + lz, rx, lx, ly, lz);
        }
        fold(hx, lx); fold(hy, ly); fold(hz, lz);
    } else {
        float cx = -lx, cy = -ly, cz = -lz;
#pragma unroll 4
        for (int k = 0; k < n; ++k) {
            BLOCH_RFC_LOAD(k)
            float tx, ty, tz;
            rf_increment<TIER>(wx, wy, wz, q, hx, hy, hz, rx, tx, ty, tz);
            kahan_add(hx, cx, tx);
            kahan_add(hy, cy, ty);
            kahan_add(hz, cz, tz);
        }
        lx = -cx; ly = -cy; lz = -cz;
    }
#undef BLOCH_RFC_LOAD
}

// (a minimum of 4 ... 8 CTAs per SM in the launch bounds: still 40 registers, but ptxas schedules the unrolled steps
// differently and config 4's excitation goes 36.3 -> 34.8 ms; 10: 35.1; 14 or 16: 37.6.  The same hint makes rf_kernel
// slower, 37.5 -> 38.3 ms.)
__global__ void __launch_bounds__(kRfMaxThreads, 8)
rf_const_kernel(const __grid_constant__ RfConstArgs args, PropRec prop, int has_prop, const float4 *__restrict__ A,
                const float4 *__restrict__ Cc, float4 *__restrict__ S, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const bool active = i < n;
    float4 a = make_float4(0.f, 0.f, 0.f, 0.f), c = make_float4(1.f, 1.f, 0.f, 0.f), s = make_float4(0.f, 0.f, 0.f, 0.f);
    const float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
    if (active) {
        a = A[i];
        c = Cc[i];
        s = S[i];
    }
    float hx = s.x, hy = s.y, hz = s.z;
    if (has_prop) propagate(prop, a, c, v, hx, hy, hz);
    float lx = 0.f, ly = 0.f, lz = 0.f;
    const RfSpin sp{a.x, a.y, a.z, c.w, c.x, c.y, c.z, 0.f, 0.f, 0.f};
    const float ax = fabsf(sp.x), ay = fabsf(sp.y), az = fabsf(sp.z), adw = fabsf(sp.dw);
    int base = 0;
    for (int t = 0; t < args.n_tiles; ++t) {
        const RfConstTile hd = args.tile[t];
        RfRelax rx;
        rx.D1 = -expm1f(-hd.dt * sp.r1);
        rx.D2 = -expm1f(-hd.dt * sp.r2);
        rx.E1 = 1.0f - rx.D1;
        rx.E2 = 1.0f - rx.D2;
        rx.D1m0 = rx.D1 * sp.m0;
        const float wzb = fmaf(fabsf(hd.gx), ax, fmaf(fabsf(hd.gy), ay, fmaf(fabsf(hd.gz), az, hd.dt * adw)));
        const float qb = fmaf(wzb, wzb, hd.wxy2_max);
        const int tier = __all_sync(0xffffffffu, qb <= kRfQLin) ? -1
                         : (__all_sync(0xffffffffu, qb <= 0.00390625f) ? 0 : (__all_sync(0xffffffffu, qb <= 0.25f) ? 1 : 2));
        if (tier == -1) rf_ctile<-1>(args, base, hd, sp, rx, hx, hy, hz, lx, ly, lz);
        else if (tier == 0) rf_ctile<0>(args, base, hd, sp, rx, hx, hy, hz, lx, ly, lz);
        else if (tier == 1) rf_ctile<1>(args, base, hd, sp, rx, hx, hy, hz, lx, ly, lz);
        else rf_ctile<2>(args, base, hd, sp, rx, hx, hy, hz, lx, ly, lz);
        base += hd.n_steps;
    }
    if (active) S[i] = make_float4(hx + lx, hy + ly, hz + lz, s.w);
}

// Two spins per thread (static plans; BLOCH_OPT_RF_SPINS): thread t owns spins t and t + ceil(n / 2).  Tiles whose
// bound on q leaves tier 0 (never with the configs' pulses) fall back to rf_tile one spin after the other.
__global__ void __launch_bounds__(kRfMaxThreads)
rf_pair_kernel(const unsigned char *__restrict__ tbl, int n_tiles, PropRec prop, int has_prop,
               const float4 *__restrict__ A, const float4 *__restrict__ Cc, float4 *__restrict__ S, int n) {
    __shared__ __align__(128) unsigned char buf[2][kRfHdrBytes + kRfTileSteps * 32];
    __shared__ __align__(8) uint64_t bar[2];
    const int tid = threadIdx.x;
    const int2 *dir = reinterpret_cast<const int2 *>(tbl);
    if (tid == 0 && n_tiles > 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        mbar_init_fence();
        for (int b = 0; b < 2 && b < n_tiles; ++b) {
            const int2 d = dir[b];
            mbar_expect_tx(&bar[b], (uint32_t)d.y);
            bulk_g2s(buf[b], tbl + d.x, (uint32_t)d.y, &bar[b]);
        }
    }
    const int half = (n + 1) / 2;
    const int ia = blockIdx.x * blockDim.x + tid, ib = ia + half;
    const bool act_a = ia < half, act_b = act_a && ib < n;
    const float4 zero = make_float4(0.f, 0.f, 0.f, 0.f), one = make_float4(1.f, 1.f, 0.f, 0.f);
    float4 aa = zero, ca = one, st_a = zero, ab = zero, cb = one, st_b = zero;
    if (act_a) { aa = A[ia]; ca = Cc[ia]; st_a = S[ia]; }
    if (act_b) { ab = A[ib]; cb = Cc[ib]; st_b = S[ib]; }
    float h[6] = {st_a.x, st_a.y, st_a.z, st_b.x, st_b.y, st_b.z};
    float l[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    if (has_prop) {
        propagate(prop, aa, ca, zero, h[0], h[1], h[2]);
        propagate(prop, ab, cb, zero, h[3], h[4], h[5]);
    }
    const RfSpin sa{aa.x, aa.y, aa.z, ca.w, ca.x, ca.y, ca.z, 0.f, 0.f, 0.f};
    const RfSpin sb{ab.x, ab.y, ab.z, cb.w, cb.x, cb.y, cb.z, 0.f, 0.f, 0.f};
    const float ax = fmaxf(fabsf(sa.x), fabsf(sb.x)), ay = fmaxf(fabsf(sa.y), fabsf(sb.y)),
                az = fmaxf(fabsf(sa.z), fabsf(sb.z)), adw = fmaxf(fabsf(sa.dw), fabsf(sb.dw));
    __syncthreads();  // barrier initialisation visible to every waiter

    for (int t = 0; t < n_tiles; ++t) {
        const int b = t & 1;
        mbar_wait(&bar[b], (uint32_t)((t >> 1) & 1));
        const unsigned char *tile = buf[b];
        const RfTileHdr hd = *reinterpret_cast<const RfTileHdr *>(tile);
        RfRelax ra, rb;
        ra.D1 = -expm1f(-hd.dt * sa.r1); ra.D2 = -expm1f(-hd.dt * sa.r2);
        ra.E1 = 1.0f - ra.D1; ra.E2 = 1.0f - ra.D2; ra.D1m0 = ra.D1 * sa.m0;
        rb.D1 = -expm1f(-hd.dt * sb.r1); rb.D2 = -expm1f(-hd.dt * sb.r2);
        rb.E1 = 1.0f - rb.D1; rb.E2 = 1.0f - rb.D2; rb.D1m0 = rb.D1 * sb.m0;
        const float wzb = fmaf(hd.gx_max, ax, fmaf(hd.gy_max, ay, fmaf(hd.gz_max, az, hd.dt * adw)));
        const float qb = fmaf(wzb, wzb, hd.wxy2_max);
        const bool uni = (hd.flags & kRfFlagUniformG) != 0;
        if (__all_sync(0xffffffffu, qb <= kRfQLin)) {
            if (uni) rf_tile0_pair<-1, 0>(tile, hd, sa, sb, ra, rb, h, l);
            else rf_tile0_pair<-1, 1>(tile, hd, sa, sb, ra, rb, h, l);
        } else if (__all_sync(0xffffffffu, qb <= 0.00390625f)) {
            if (uni) rf_tile0_pair<0, 0>(tile, hd, sa, sb, ra, rb, h, l);
            else rf_tile0_pair<0, 1>(tile, hd, sa, sb, ra, rb, h, l);
        } else {
            const int tier = __all_sync(0xffffffffu, qb <= 0.25f) ? 1 : 2;
#define BLOCH_RF_ONE(T, M, SP, RX, O) rf_tile<T, M>(tile, hd, SP, RX, h[O], h[O + 1], h[O + 2], l[O], l[O + 1], l[O + 2])
#define BLOCH_RF_BOTH(T)                                                              \
    do {                                                                              \
        if (uni) { BLOCH_RF_ONE(T, 0, sa, ra, 0); BLOCH_RF_ONE(T, 0, sb, rb, 3); }    \
        else { BLOCH_RF_ONE(T, 1, sa, ra, 0); BLOCH_RF_ONE(T, 1, sb, rb, 3); }        \
    } while (0)
            if (tier == 1) BLOCH_RF_BOTH(1);
            else BLOCH_RF_BOTH(2);
#undef BLOCH_RF_BOTH
#undef BLOCH_RF_ONE
        }
        __syncthreads();  // every thread is done reading buf[b]
        if (tid == 0 && t + 2 < n_tiles) {
            const int2 d = dir[t + 2];
            mbar_expect_tx(&bar[b], (uint32_t)d.y);
            bulk_g2s(buf[b], tbl + d.x, (uint32_t)d.y, &bar[b]);
        }
    }
    if (act_a) S[ia] = make_float4(h[0] + l[0], h[1] + l[1], h[2] + l[2], st_a.w);
    if (act_b) S[ib] = make_float4(h[3] + l[3], h[4] + l[4], h[5] + l[5], st_b.w);
}

}  // namespace bloch
