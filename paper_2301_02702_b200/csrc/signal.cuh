// signal.cuh -- a6 + a7: free-precession signal kernels (SUM_ALL) for sm_100a.
//
// Free precession is evaluated in closed form from the block start (Eq 10-11, are diagonal
// in (Mxy, Mz) and commute, so the step-by-step product collapses exactly; :132 "exact solution"):
//     c_in = Mxy_i(0) * exp(-tau_n / T2_i) * exp(i theta_in),    theta_in = k'_n . x_i + f'_i tau_n
// with k' = -gamma K(t) the cumulative gradient moment of the block (Eq 12-13, :173-180) and f' = -dw.
//
// Grid = (point tiles, spin chunks).  A thread OWNS P adjacent evaluated points (k', tau in registers) and
// walks the spins of its chunk.  Spin tiles (x, y, z, f') and (Mxy, e2) are staged global -> shared by 1-D bulk copies
// (TMA) into a two-stage mbarrier ring by one elected thread and then broadcast to all threads (every lane
// reads the same address: conflict-free LDS.128).  The sum over spins is therefore thread-local: no
// shuffles, no atomics.  Each CTA writes its partial sums P[chunk][point]; reduce_kernel adds the chunks in
// index order (deterministic two-pass reduction, :194 "add them later").
//
// fp32 phase: tables and f' in radians; per evaluation 4 FMA (phase), 1 FMUL (MUFU pre-scale to turns),
// MUFU sin + cos, 1 FMUL + MUFU ex2 (T2 decay), 2 FMUL + 4 FMA (complex multiply-accumulate) = 16 issue
// slots, 3 of them on the 16-lane MUFU pipe -- the bound.  Because a thread's P points are adjacent samples,
// exp(-tau_j/T2) for j > 0 is the j = 0 value times a cubic series in (tau_j - tau_0)/T2 on the FMA pipe
// whenever that ratio is <= 0.02 for every spin (bound from max 1/T2, found by pack_kernel): 2 + 1/P MUFU
// operations and 17.9 instructions per evaluation.  Consecutive blocks of one batch write their partials
// side by side (row_stride, p_off) so that one second-pass launch serves the whole batch.  No explicit range reduction: MUFU.SIN/COS take
// their argument in turns and wrap it themselves; the planner keeps |theta| below 256 turns in this mode,
// where the fp32 rounding of theta (~1e-4 rad) is already the error floor.
// fp64 phase (north_star item 4): k', tau, x, f' in double, theta in turns by 4 DFMA; adding 1.5 * 2^20
// leaves frac(theta) as a 32-bit fixed-point number in the low word of the double, which is turned into a
// float in [0, 1) with two integer ops and one FADD -- no F2F (it would be a fourth op on the MUFU pipe).
#pragma once
#include <type_traits>

#include "internal.h"
#include "kernels.cuh"
#include "tma.cuh"

namespace bloch {

constexpr int kSigThreads = 256;
constexpr int kSigTile = 256;  // spins per staged tile

// fp32 phase, static spins: the contributions of ONE spin to a thread's P adjacent samples, added into (ar, ai).  The one
// copy of this arithmetic: signal_kernel and the signal warps of the whole-sequence kernel (seq.cuh) both call it.
// MODE 0: one MUFU.EX2 per sample, 1: decay of sample j from sample 0 by the cubic series, 2: geometric decay.
// a = (x, y, z, f'), st = (Mxy.re, Mxy.im, Mz, e2 = -log2(e)/T2); k' in rad/m, cj[j] = (tau_j - tau_0) ln 2.
template <int P, int MODE>
__device__ __forceinline__ void signal_spin_fp32(const float (&kx)[P], const float (&ky)[P], const float (&kz)[P],
                                                 const float (&tau)[P], const float (&cj)[P], const float4 &a,
                                                 const float4 &st, float (&ar)[P], float (&ai)[P]) {
    float er0 = 0.f, ei0 = 0.f, qd = 1.f;
    if (MODE == 2) {
        const float y = cj[1] * st.w;  // -dwell/T2
        qd = fmaf(y, fmaf(y, fmaf(y, 1.0f / 6.0f, 0.5f), 1.0f), 1.0f);
    }
#pragma unroll
    for (int j = 0; j < P; ++j) {
        const float th = fmaf(kx[j], a.x, fmaf(ky[j], a.y, fmaf(kz[j], a.z, tau[j] * a.w)));  // radians
        const float sn = __sinf(th), cs = __cosf(th);  // FMUL by 1/(2 pi) + MUFU.SIN / MUFU.COS
        float er, ei;
        if (j == 0 || MODE == 0) {
            const float e = ex2_approx(tau[j] * st.w);  // MUFU.EX2: exp(-tau/T2)
            er = st.x * e;
            ei = st.y * e;
            if (j == 0) { er0 = er; ei0 = ei; }
        } else if (MODE == 2) {
            er0 *= qd;  // running product: exp(-(tau_0 + j dwell)/T2)
            ei0 *= qd;
            er = er0;
            ei = ei0;
        } else {
            const float y = cj[j] * st.w;  // -(tau_j - tau_0)/T2
            const float pe = fmaf(y, fmaf(y, fmaf(y, 1.0f / 6.0f, 0.5f), 1.0f), 1.0f);
            er = er0 * pe;
            ei = ei0 * pe;
        }
        ar[j] = fmaf(er, cs, fmaf(-ei, sn, ar[j]));
        ai[j] = fmaf(er, sn, fmaf(ei, cs, ai[j]));
    }
}

// MO (motion plans): every record (k', tau) is followed by (mu', 0), the spins' velocities are a third staged
// tile, and the phase gains mu' . v (x(t) = x + v t).
// fp32 phase, static plans: held to 64 registers (P <= 4: 4 CTAs per SM) or 85 (P = 8: 3 CTAs per SM); ptxas otherwise
// drifts to 72 / 100 registers and loses a resident CTA
template <int P, bool PH64, bool MO>
__global__ void __launch_bounds__(kSigThreads, (PH64 || MO) ? 1 : (P == 8 ? 3 : 4))
signal_kernel(const void *__restrict__ recs_, int n_pts, const void *__restrict__ A_, const void *__restrict__ V_,
              const float4 *__restrict__ S, int n_spins, int spins_per_chunk,
              const float *__restrict__ scal /* [0] = max 1/T2, from pack_kernel */, float2 *__restrict__ partial,
              int row_stride /* points of the whole batch */, int p_off /* this block's first point in the batch */,
              int allow_lin /* 0: never take the rotation recurrence (BLOCH_SIGNAL_LIN=0, diagnostics) */) {
    using RecT = typename std::conditional<PH64, double4, float4>::type;   // (k'x, k'y, k'z, tau)
    using PosT = typename std::conditional<PH64, double4, float4>::type;   // (x, y, z, f')
    using real = typename std::conditional<PH64, double, float>::type;
    __shared__ __align__(128) PosT shA[2][kSigTile];
    __shared__ __align__(128) float4 shS[2][kSigTile];
    __shared__ __align__(128) PosT shV[MO ? 2 : 1][MO ? kSigTile : 1];
    __shared__ __align__(8) uint64_t bar[2];
    const RecT *recs = reinterpret_cast<const RecT *>(recs_);
    const PosT *A = reinterpret_cast<const PosT *>(A_);
    const PosT *V = reinterpret_cast<const PosT *>(V_);
    constexpr int RS = MO ? 2 : 1;
    const int tid = threadIdx.x;
    const int s0 = blockIdx.y * spins_per_chunk;
    const int s1 = min(n_spins, s0 + spins_per_chunk);
    const int n_tiles = (s1 - s0 + kSigTile - 1) / kSigTile;
    auto issue = [&](int t) {
        const int b = t & 1;
        const int base = s0 + t * kSigTile;
        const uint32_t cnt = (uint32_t)min(kSigTile, s1 - base);
        mbar_expect_tx(&bar[b], cnt * (uint32_t)((MO ? 2 : 1) * sizeof(PosT) + sizeof(float4)));
        bulk_g2s(shA[b], A + base, cnt * (uint32_t)sizeof(PosT), &bar[b]);
        bulk_g2s(shS[b], S + base, cnt * (uint32_t)sizeof(float4), &bar[b]);
        if (MO) bulk_g2s(shV[b], V + base, cnt * (uint32_t)sizeof(PosT), &bar[b]);
    };
    if (tid == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        mbar_init_fence();
        if (n_tiles > 0) issue(0);
        if (n_tiles > 1) issue(1);
    }
    // the thread's P points are ADJACENT ADC samples, so tau_j - tau_0 is a few dwell times
    const int p0 = (blockIdx.x * (int)blockDim.x + tid) * P;  // blockDim.x < kSigThreads for blocks of few samples
    real kx[P], ky[P], kz[P], tau[P], ux[MO ? P : 1], uy[MO ? P : 1], uz[MO ? P : 1];
    float tf[P], cj[P], ar[P], ai[P];
    float cmax = 0.f;
#pragma unroll
    for (int j = 0; j < P; ++j) {
        const int p = p0 + j;
        RecT r;
        r.x = 0; r.y = 0; r.z = 0; r.w = j ? tau[0] : (real)0;
        if (p < n_pts) r = recs[RS * p];
        kx[j] = r.x; ky[j] = r.y; kz[j] = r.z; tau[j] = r.w;
        if (MO) {
            RecT m;
            m.x = 0; m.y = 0; m.z = 0; m.w = 0;
            if (p < n_pts) m = recs[RS * p + 1];
            ux[j] = m.x; uy[j] = m.y; uz[j] = m.z;
        }
        tf[j] = (float)r.w;
        cj[j] = (float)(r.w - tau[0]) * 0.6931471805599453f;  // (tau_j - tau_0) ln 2; times e2 = -(tau_j - tau_0)/T2
        cmax = fmaxf(cmax, fabsf(cj[j]));
        ar[j] = 0.f; ai[j] = 0.f;
    }
    // exp(-tau_j/T2) for j > 0 from the j = 0 value by a cubic series in (tau_j - tau_0)/T2 when that ratio is
    // <= 0.02 for every spin (truncation < 7e-9); decided per warp, otherwise every point takes its own MUFU.EX2
    const bool series = P > 1 && __all_sync(0xffffffffu, cmax * (scal[0] * kLog2e) <= 0.02f);
    // ... and when the thread's samples are equally spaced (one dwell apart: every readout of the configs), the
    // decay of sample j is the decay of sample j-1 times q = exp(-dwell/T2): q by the same cubic series once per spin,
    // then two FMUL per sample instead of six instructions.  Taken when |tau_j - tau_0 - j dwell| / T2 <= 1e-6 for
    // every spin (the fp32 rounding of tau alone is a few 1e-9 s late in a block).
    float dev = 0.f;
#pragma unroll
    for (int j = 2; j < P; ++j) dev = fmaxf(dev, fabsf(cj[j] - (float)j * cj[1]));
    const bool geom = P > 2 && series && __all_sync(0xffffffffu, dev * (scal[0] * kLog2e) <= 1e-6f);
    // ... and when k' itself advances by the same step from sample to sample (a Cartesian / EPI readout on its
    // plateau), the whole factor exp(-tau_j/T2) exp(i theta_j) of sample j is that of sample j-1 times
    // zeta = q exp(i delta), delta = dk' . x + f' dwell: one sincos for theta_0 and one for delta per spin, then one
    // complex multiply per sample on the FMA pipe -- (5 MUFU + ~74 issue slots) / P instead of 2 + 1/P MUFU per
    // evaluation.  dk' is the slope through the thread's first and last sample; the mode is taken when every
    // sample in between lies on that line to within the rounding of the table itself (2.5e-7 relative to the larger
    // end in fp32, i.e. 2-4 ulp; 1e-13 in fp64), so the phase it reconstructs differs from the tabulated one by no more
    // than the table's own rounding.  Not for motion plans (the first-moment term is quadratic in time).
    real dkx = 0, dky = 0, dkz = 0, dta = 0;
    bool lin = false;
    if (!MO && P > 2 && allow_lin) {
        constexpr real inv = (real)1 / (real)(P - 1);
        constexpr real rel = PH64 ? (real)1e-13 : (real)2.5e-7;  // fp32: 1 ulp of table rounding + 1 ulp of this check's own arithmetic
        dkx = (kx[P - 1] - kx[0]) * inv;
        dky = (ky[P - 1] - ky[0]) * inv;
        dkz = (kz[P - 1] - kz[0]) * inv;
        dta = (tau[P - 1] - tau[0]) * inv;
        // fp64 tables (turns / m): the ADC times themselves are equally spaced only to the rounding of t (7e-18 s in
        // 4e-6 s: 2e-12 of a step), so allow 1e-8 turns / m absolute -- below 1e-8 turns of phase for |x| < 1 m, an
        // order under the 2^-23-turn granularity of the reduced phase
        constexpr real fl = PH64 ? (real)1e-8 : (real)0;
        const real tx = rel * fmax(fabs(kx[0]), fabs(kx[P - 1])) + fl, ty = rel * fmax(fabs(ky[0]), fabs(ky[P - 1])) + fl;
        const real tz = rel * fmax(fabs(kz[0]), fabs(kz[P - 1])) + fl, tt = rel * fmax(fabs(tau[0]), fabs(tau[P - 1]));
        bool ok = true;
#pragma unroll
        for (int j = 1; j < P - 1; ++j) {
            ok = ok && fabs(kx[j] - (kx[0] + (real)j * dkx)) <= tx && fabs(ky[j] - (ky[0] + (real)j * dky)) <= ty &&
                 fabs(kz[j] - (kz[0] + (real)j * dkz)) <= tz && fabs(tau[j] - (tau[0] + (real)j * dta)) <= tt;
        }
        lin = geom && __all_sync(0xffffffffu, ok);
    }
    __syncthreads();  // barrier initialisation visible to every waiter
    // sin and cos of the phase k . x + w tau (fp32: radians; fp64: turns, reduced as described in the header)
    auto phase_sincos = [&](real qx, real qy, real qz, real qt, const PosT &a, float &sn, float &cs) {
        if (PH64) {
            double th = fma((double)qx, (double)a.x, fma((double)qy, (double)a.y,
                            fma((double)qz, (double)a.z, (double)qt * (double)a.w)));  // turns
            th += 1572864.0;  // 1.5 * 2^20: ulp = 2^-32, low word = frac(theta) in 0.32 fixed point
            const unsigned lo = (unsigned)__double2loint(th);
            const float fr = __uint_as_float(0x3f800000u | (lo >> 9)) - 1.0f;  // [0, 1) turns
            const float ang = fr * 6.283185307179586f;
            sn = __sinf(ang);
            cs = __cosf(ang);
        } else {
            const float th = fmaf((float)qx, (float)a.x, fmaf((float)qy, (float)a.y,
                                  fmaf((float)qz, (float)a.z, (float)qt * (float)a.w)));  // radians
            sn = __sinf(th);
            cs = __cosf(th);
        }
    };
    auto run = [&](auto mode_tag) {
    // 0: one MUFU.EX2 per sample, 1: series per sample, 2: geometric decay, 3: geometric decay and rotation
    constexpr int MODE = decltype(mode_tag)::value;
    constexpr bool SERIES = MODE != 0;
    for (int t = 0; t < n_tiles; ++t) {
        const int b = t & 1;
        mbar_wait(&bar[b], (uint32_t)((t >> 1) & 1));
        const int cnt = min(kSigTile, s1 - (s0 + t * kSigTile));
#pragma unroll 2
        for (int s = 0; s < cnt; ++s) {
            const PosT a = shA[b][s];
            const float4 st = shS[b][s];  // (Mxy.re, Mxy.im, Mz, e2 = -log2(e)/T2)
            PosT vv;
            vv.x = 0; vv.y = 0; vv.z = 0; vv.w = 0;
            if (MO) vv = shV[b][s];
            float er0 = 0.f, ei0 = 0.f, qd = 1.f;
            if (MODE >= 2) {
                const float y = cj[1] * st.w;  // -dwell/T2
                qd = fmaf(y, fmaf(y, fmaf(y, 1.0f / 6.0f, 0.5f), 1.0f), 1.0f);
            }
            if (MODE == 3) {
                float sn, cs, sd, cd;
                phase_sincos(kx[0], ky[0], kz[0], tau[0], a, sn, cs);
                phase_sincos(dkx, dky, dkz, dta, a, sd, cd);
                const float e = ex2_approx(tf[0] * st.w);  // MUFU.EX2: exp(-tau_0/T2)
                const float zr = qd * cd, zi = qd * sd;    // zeta
                const float er = st.x * e, ei = st.y * e;
                // w_j = w_0 zeta^j through zeta^2, zeta^4: dependency depth log2(P) instead of P - 1
                float wr[P], wi[P];
                wr[0] = fmaf(er, cs, -ei * sn);
                wi[0] = fmaf(er, sn, ei * cs);
                float pr = zr, pi = zi;  // zeta^(2^m)
#pragma unroll
                for (int h = 1; h < P; h *= 2) {
#pragma unroll
                    for (int j = 0; j < h; ++j) {
                        wr[h + j] = fmaf(wr[j], pr, -wi[j] * pi);
                        wi[h + j] = fmaf(wr[j], pi, wi[j] * pr);
                    }
                    if (2 * h < P) {
                        const float t2 = fmaf(pr, pr, -pi * pi);
                        pi = 2.0f * pr * pi;
                        pr = t2;
                    }
                }
#pragma unroll
                for (int j = 0; j < P; ++j) {
                    ar[j] += wr[j];
                    ai[j] += wi[j];
                }
                continue;
            }
            if constexpr (!PH64 && !MO) {
                if (MODE < 3) {
                    signal_spin_fp32<P, MODE < 3 ? MODE : 0>(kx, ky, kz, tau, cj, a, st, ar, ai);
                    continue;
                }
            }
#pragma unroll
            for (int j = 0; j < P; ++j) {
                float sn, cs;
                if (PH64) {
                    double th = fma((double)kx[j], (double)a.x, fma((double)ky[j], (double)a.y,
                                    fma((double)kz[j], (double)a.z, (double)tau[j] * (double)a.w)));  // turns
                    if (MO) th = fma((double)ux[j], (double)vv.x, fma((double)uy[j], (double)vv.y,
                                     fma((double)uz[j], (double)vv.z, th)));
                    th += 1572864.0;  // 1.5 * 2^20: ulp = 2^-32, low word = frac(theta) in 0.32 fixed point
                    const unsigned lo = (unsigned)__double2loint(th);
                    const float fr = __uint_as_float(0x3f800000u | (lo >> 9)) - 1.0f;  // [0, 1) turns
                    const float ang = fr * 6.283185307179586f;
                    sn = __sinf(ang);
                    cs = __cosf(ang);
                } else {
                    float th = fmaf((float)kx[j], (float)a.x, fmaf((float)ky[j], (float)a.y,
                                    fmaf((float)kz[j], (float)a.z, (float)tau[j] * (float)a.w)));  // radians
                    if (MO) th = fmaf((float)ux[j], (float)vv.x, fmaf((float)uy[j], (float)vv.y,
                                      fmaf((float)uz[j], (float)vv.z, th)));
                    sn = __sinf(th);  // FMUL by 1/(2 pi) + MUFU.SIN
                    cs = __cosf(th);
                }
                float er, ei;
                if (j == 0 || !SERIES) {
                    const float e = ex2_approx(tf[j] * st.w);  // MUFU.EX2: exp(-tau/T2)
                    er = st.x * e;
                    ei = st.y * e;
                    if (j == 0) { er0 = er; ei0 = ei; }
                } else if (MODE == 2) {
                    er0 *= qd;  // running product: exp(-(tau_0 + j dwell)/T2)
                    ei0 *= qd;
                    er = er0;
                    ei = ei0;
                } else {
                    const float y = cj[j] * st.w;  // -(tau_j - tau_0)/T2
                    const float pe = fmaf(y, fmaf(y, fmaf(y, 1.0f / 6.0f, 0.5f), 1.0f), 1.0f);
                    er = er0 * pe;
                    ei = ei0 * pe;
                }
                ar[j] = fmaf(er, cs, fmaf(-ei, sn, ar[j]));
                ai[j] = fmaf(er, sn, fmaf(ei, cs, ai[j]));
            }
        }
        __syncthreads();  // every thread is done with stage b
        if (tid == 0 && t + 2 < n_tiles) issue(t + 2);
    }
    };
    if (lin) run(std::integral_constant<int, 3>{});
    else if (geom) run(std::integral_constant<int, 2>{});
    else if (series) run(std::integral_constant<int, 1>{});
    else run(std::integral_constant<int, 0>{});
#pragma unroll
    for (int j = 0; j < P; ++j) {
        const int p = p0 + j;
        if (p < n_pts) partial[(size_t)blockIdx.y * row_stride + p_off + p] = make_float2(ar[j], ai[j]);
    }
}

// Cartesian readouts: the rotation recurrence alone (see signal_kernel, mode 3), launched instead of signal_kernel for
// precession blocks whose table the PLANNER found to advance by a constant step inside every aligned group of kLinP
// samples (Block::lin_pts of them; fp64 check on the untruncated table, plan.cpp).  A thread keeps only its group's first
// record and the step, so the fp64-phase variant needs ~1/2 of signal_kernel<8, true>'s registers and two or three CTAs
// fit on an SM; 5 MUFU and ~136 issue slots per 16 evaluations.  The block's remaining n_pts % kLinP samples go
// through signal_kernel with the same chunking (one more launch, same partial rows).
constexpr int kLinP = 16;
constexpr int kLinMid = 8;  // motion: the third record that fixes the quadratic of mu'

// MO (motion plans, x(t) = x + v t): on a plateau the first moment mu' is a quadratic in the sample index, so
// theta_j = theta_0 + j alpha + j^2 beta with alpha = dk' . x + a . v + f' dwell, beta = b . v (a, b from the group's
// records 0, kLinMid, kLinP - 1), and w_{j+1} = w_j zeta_j, zeta_{j+1} = zeta_j rho with zeta_0 = q exp(i (alpha + beta)),
// rho = exp(2 i beta): three sincos per spin and two complex multiplies per sample.  2 beta is tiny (1e-5 rad at
// 0.1 m/s), so rho comes from its series and adds no MUFU error to the j^2 term.
template <bool PH64, bool MO>
__global__ void __launch_bounds__(kSigThreads, 2)
signal_lin_kernel(const void *__restrict__ recs_, int n_groups, const void *__restrict__ A_, const void *__restrict__ V_,
                  const float4 *__restrict__ S, int n_spins, int spins_per_chunk,
                  const float *__restrict__ scal /* [0] = max 1/T2 */, float2 *__restrict__ partial, int row_stride,
                  int p_off) {
    constexpr int P = kLinP;
    constexpr int RS = MO ? 2 : 1;
    using RecT = typename std::conditional<PH64, double4, float4>::type;
    using PosT = typename std::conditional<PH64, double4, float4>::type;
    using real = typename std::conditional<PH64, double, float>::type;
    __shared__ __align__(128) PosT shA[2][kSigTile];
    __shared__ __align__(128) float4 shS[2][kSigTile];
    __shared__ __align__(128) PosT shV[MO ? 2 : 1][MO ? kSigTile : 1];
    __shared__ __align__(8) uint64_t bar[2];
    const RecT *recs = reinterpret_cast<const RecT *>(recs_);
    const PosT *A = reinterpret_cast<const PosT *>(A_);
    const PosT *V = reinterpret_cast<const PosT *>(V_);
    const int tid = threadIdx.x;
    const int s0 = blockIdx.y * spins_per_chunk;
    const int s1 = min(n_spins, s0 + spins_per_chunk);
    const int n_tiles = (s1 - s0 + kSigTile - 1) / kSigTile;
    auto issue = [&](int t) {
        const int b = t & 1;
        const int base = s0 + t * kSigTile;
        const uint32_t cnt = (uint32_t)min(kSigTile, s1 - base);
        mbar_expect_tx(&bar[b], cnt * (uint32_t)((MO ? 2 : 1) * sizeof(PosT) + sizeof(float4)));
        bulk_g2s(shA[b], A + base, cnt * (uint32_t)sizeof(PosT), &bar[b]);
        bulk_g2s(shS[b], S + base, cnt * (uint32_t)sizeof(float4), &bar[b]);
        if (MO) bulk_g2s(shV[b], V + base, cnt * (uint32_t)sizeof(PosT), &bar[b]);
    };
    if (tid == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        mbar_init_fence();
        if (n_tiles > 0) issue(0);
        if (n_tiles > 1) issue(1);
    }
    const int g = blockIdx.x * (int)blockDim.x + tid;
    const bool live = g < n_groups;
    RecT r0, r1, m0, m8, m15;
    r0.x = 0; r0.y = 0; r0.z = 0; r0.w = 0;
    r1 = r0; m0 = r0; m8 = r0; m15 = r0;
    if (live) {
        r0 = recs[(size_t)RS * g * P];
        r1 = recs[(size_t)RS * (g * P + P - 1)];
        if (MO) {
            m0 = recs[(size_t)RS * g * P + 1];
            m8 = recs[(size_t)RS * (g * P + kLinMid) + 1];
            m15 = recs[(size_t)RS * (g * P + P - 1) + 1];
        }
    }
    constexpr real inv = (real)1 / (real)(P - 1);
    const real dkx = (r1.x - r0.x) * inv, dky = (r1.y - r0.y) * inv, dkz = (r1.z - r0.z) * inv, dta = (r1.w - r0.w) * inv;
    // mu'(j) = m0 + a j + b j^2 through j = 0, kLinMid, P - 1
    constexpr real i8 = (real)1 / (real)kLinMid, i7 = (real)1 / (real)(P - 1 - kLinMid);
    const real bx = MO ? ((m15.x - m0.x) * inv - (m8.x - m0.x) * i8) * i7 : (real)0;
    const real by = MO ? ((m15.y - m0.y) * inv - (m8.y - m0.y) * i8) * i7 : (real)0;
    const real bz = MO ? ((m15.z - m0.z) * inv - (m8.z - m0.z) * i8) * i7 : (real)0;
    // a + b (the first step's moment increment)
    const real abx = MO ? (m8.x - m0.x) * i8 - (real)(kLinMid - 1) * bx : (real)0;
    const real aby = MO ? (m8.y - m0.y) * i8 - (real)(kLinMid - 1) * by : (real)0;
    const real abz = MO ? (m8.z - m0.z) * i8 - (real)(kLinMid - 1) * bz : (real)0;
    const float tf0 = (float)r0.w;
    const float cd = (float)dta * 0.6931471805599453f;  // dwell ln 2; times e2 = -log2(e)/T2 gives -dwell/T2
    // q = exp(-dwell/T2) by the cubic series when dwell/T2 <= 0.02 for every spin (as in signal_kernel), else MUFU.EX2
    const bool series = __all_sync(0xffffffffu, fabsf(cd) * (scal[0] * kLog2e) <= 0.02f);
    float ar[P], ai[P];
#pragma unroll
    for (int j = 0; j < P; ++j) { ar[j] = 0.f; ai[j] = 0.f; }
    // sin and cos of k . x + w tau (+ u . v); fp32: radians, fp64: turns reduced as described in the file header
    auto phase_sincos = [&](real qx, real qy, real qz, real qt, real ux, real uy, real uz, const PosT &a, const PosT &vv,
                            float &sn, float &cs, bool accurate) {
        if (PH64) {
            double th = fma((double)qx, (double)a.x, fma((double)qy, (double)a.y,
                            fma((double)qz, (double)a.z, (double)qt * (double)a.w)));  // turns
            if (MO) th = fma((double)ux, (double)vv.x, fma((double)uy, (double)vv.y, fma((double)uz, (double)vv.z, th)));
            th += 1572864.0;  // 1.5 * 2^20: low word = frac(theta) in 0.32 fixed point
            const unsigned lo = (unsigned)__double2loint(th);
            if (accurate) {
                // the step's rotation is applied up to P - 1 times: full-precision sincos of the signed fraction
                const float fs = (float)(int)lo * 2.3283064365386963e-10f;  // [-0.5, 0.5) turns
                sincospif(2.0f * fs, &sn, &cs);
            } else {
                const float fr = __uint_as_float(0x3f800000u | (lo >> 9)) - 1.0f;
                const float ang = fr * 6.283185307179586f;
                sn = __sinf(ang);
                cs = __cosf(ang);
            }
        } else {
            float th = fmaf((float)qx, (float)a.x, fmaf((float)qy, (float)a.y,
                            fmaf((float)qz, (float)a.z, (float)qt * (float)a.w)));  // radians
            if (MO) th = fmaf((float)ux, (float)vv.x, fmaf((float)uy, (float)vv.y, fmaf((float)uz, (float)vv.z, th)));
            if (accurate) {
                float r = th * 0.15915494309189535f;  // turns; the step's phase is a few radians at most
                r -= rintf(r);
                sincospif(2.0f * r, &sn, &cs);
            } else {
                sn = __sinf(th);
                cs = __cosf(th);
            }
        }
    };
    __syncthreads();
    for (int t = 0; t < n_tiles; ++t) {
        const int b = t & 1;
        mbar_wait(&bar[b], (uint32_t)((t >> 1) & 1));
        const int cnt = min(kSigTile, s1 - (s0 + t * kSigTile));
#pragma unroll 2
        for (int s = 0; s < cnt; ++s) {
            const PosT a = shA[b][s];
            const float4 st = shS[b][s];  // (Mxy.re, Mxy.im, Mz, e2 = -log2(e)/T2)
            PosT vv;
            vv.x = 0; vv.y = 0; vv.z = 0; vv.w = 0;
            if (MO) vv = shV[b][s];
            float sn, cs, sd, cdl;
            phase_sincos(r0.x, r0.y, r0.z, r0.w, m0.x, m0.y, m0.z, a, vv, sn, cs, false);
            phase_sincos(dkx, dky, dkz, dta, abx, aby, abz, a, vv, sd, cdl, true);
            const float e = ex2_approx(tf0 * st.w);
            const float y = cd * st.w;  // -dwell/T2
            float qd = fmaf(y, fmaf(y, fmaf(y, 1.0f / 6.0f, 0.5f), 1.0f), 1.0f);
            if (!series) qd = ex2_approx((float)dta * st.w);
            float pr = qd * cdl, pi = qd * sd;  // zeta (MO: zeta_0), then zeta^(2^m) (static) or zeta_j (MO)
            const float er = st.x * e, ei = st.y * e;
            float wr[P], wi[P];
            wr[0] = fmaf(er, cs, -ei * sn);
            wi[0] = fmaf(er, sn, ei * cs);
            if (MO) {
                // rho = exp(2 i beta): beta = b . v in turns (fp64) or radians (fp32)
                float ang = 2.0f * (float)(bx * vv.x + by * vv.y + bz * vv.z);
                if (PH64) ang *= 6.283185307179586f;
                const float a2 = ang * ang;
                float rr = fmaf(a2, fmaf(a2, 1.0f / 24.0f, -0.5f), 1.0f);
                float ri = ang * fmaf(a2, fmaf(a2, 1.0f / 120.0f, -1.0f / 6.0f), 1.0f);
                if (fabsf(ang) > 0.05f) { rr = __cosf(ang); ri = __sinf(ang); }  // series truncation 2e-11 below that
#pragma unroll
                for (int j = 1; j < P; ++j) {
                    wr[j] = fmaf(wr[j - 1], pr, -wi[j - 1] * pi);
                    wi[j] = fmaf(wr[j - 1], pi, wi[j - 1] * pr);
                    const float t2 = fmaf(pr, rr, -pi * ri);
                    pi = fmaf(pr, ri, pi * rr);
                    pr = t2;
                }
            } else {
                // w_j = w_0 zeta^j through zeta^2, zeta^4, zeta^8: dependency depth log2(P)
#pragma unroll
                for (int h = 1; h < P; h *= 2) {
#pragma unroll
                    for (int j = 0; j < h; ++j) {
                        wr[h + j] = fmaf(wr[j], pr, -wi[j] * pi);
                        wi[h + j] = fmaf(wr[j], pi, wi[j] * pr);
                    }
                    if (2 * h < P) {
                        const float t2 = fmaf(pr, pr, -pi * pi);
                        pi = 2.0f * pr * pi;
                        pr = t2;
                    }
                }
            }
#pragma unroll
            for (int j = 0; j < P; ++j) {
                ar[j] += wr[j];
                ai[j] += wi[j];
            }
        }
        __syncthreads();
        if (tid == 0 && t + 2 < n_tiles) issue(t + 2);
    }
    if (live) {
        float2 *dst = partial + (size_t)blockIdx.y * row_stride + p_off + (size_t)g * P;
#pragma unroll
        for (int j = 0; j < P; ++j) dst[j] = make_float2(ar[j], ai[j]);
    }
}

// Second pass of a7: fixed-order sum over the spin chunks.  blockDim = (32, 8): x = point, y = chunk lane.
__global__ void __launch_bounds__(256)
reduce_kernel(const float2 *__restrict__ partial, int n_chunks, int n_pts, float2 *__restrict__ out) {
    __shared__ float2 sh[8][33];
    const int p = blockIdx.x * 32 + threadIdx.x;
    float re = 0.f, im = 0.f;
    if (p < n_pts) {
        for (int c = threadIdx.y; c < n_chunks; c += 8) {
            const float2 v = partial[(size_t)c * n_pts + p];
            re += v.x;
            im += v.y;
        }
    }
    sh[threadIdx.y][threadIdx.x] = make_float2(re, im);
    __syncthreads();
    if (threadIdx.y == 0 && p < n_pts) {
#pragma unroll
        for (int k = 1; k < 8; ++k) {
            re += sh[k][threadIdx.x].x;
            im += sh[k][threadIdx.x].y;
        }
        out[p] = make_float2(re, im);
    }
}

}  // namespace bloch
