// coils.cuh -- multi-coil receive (SURVEY.md 8(f) f2 "per-coil weights"; reading C1):
//     S_c(t_n) = sum_i C_c(x_i) * Mxy_i(t_n),     C_c complex, given per spin by the caller.
//
// The expensive part of an evaluation -- the phase, MUFU sin / cos / ex2, the decay -- does not depend on the
// coil, so one kernel evaluates c_in = Mxy_i(0) exp(-tau_n/T2_i) exp(i theta_in) ONCE (arithmetic of
// signal_kernel, signal.cuh) and accumulates it into NC coil sums with 4 FMA per coil: an extra coil costs 4
// FMA-pipe instructions per evaluation instead of a second pass of 18.  NC = 4 coils per pass for up to 4 coils,
// 8 beyond (the shared part is then amortised over twice the coils; 96 registers, 2 CTAs per SM); more coils take
// ceil(n_coils / NC) passes over the block.  The weights are repacked once per simulation into one record of NC
// float2 per spin per pass so that a spin tile's weights arrive by ONE bulk copy (TMA) next to its position and
// state tiles; unused slots of the last pass hold zeros.  Partials P[coil][chunk][point], second pass in
// chunk order (no float atomics, bitwise reproducible), as a7.
#pragma once
#include <type_traits>

#include "internal.h"
#include "kernels.cuh"
#include "signal.cuh"
#include "tma.cuh"

namespace bloch {

constexpr int kCoilsPerPassMax = 8;
__host__ __device__ inline int coils_per_pass(int n_coils) { return n_coils > 4 ? 8 : 4; }

// caller layout coil[c][i] (float2) -> W[pass][i][k] (float2), k = c - ncp pass
__global__ void __launch_bounds__(256)
pack_coils_kernel(int n, int n_coils, int ncp, const float2 *__restrict__ coil, float2 *__restrict__ W) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int pass = blockIdx.y;
    if (i >= n) return;
    float4 *dst = reinterpret_cast<float4 *>(W + ((size_t)pass * n + i) * ncp);
    for (int k = 0; k < ncp; k += 2) {
        const int c = pass * ncp + k;
        const float2 a = c < n_coils ? coil[(size_t)c * n + i] : make_float2(0.f, 0.f);
        const float2 b = c + 1 < n_coils ? coil[(size_t)(c + 1) * n + i] : make_float2(0.f, 0.f);
        dst[k / 2] = make_float4(a.x, a.y, b.x, b.y);
    }
}

// MO (motion plans, x(t) = x + v u(t)): every record (k', tau) is followed by (mu', 0), the spins' velocities /
// amplitudes are one more staged tile, and the phase gains mu' . v, exactly as in signal_kernel.
template <int P, int NC, bool PH64, bool MO>
__global__ void __launch_bounds__(kSigThreads, (NC == 8 || MO) ? 2 : 4)
signal_coils_kernel(const void *__restrict__ recs_, int n_pts, const void *__restrict__ A_, const void *__restrict__ V_,
                    const float4 *__restrict__ S, const float4 *__restrict__ W /* this pass: NC / 2 float4 per spin */,
                    int n_spins, int spins_per_chunk, const float *__restrict__ scal,
                    float2 *__restrict__ partial /* [NC][chunks][n_pts] */) {
    using RecT = typename std::conditional<PH64, double4, float4>::type;
    using PosT = typename std::conditional<PH64, double4, float4>::type;
    using real = typename std::conditional<PH64, double, float>::type;
    constexpr int TILE = (NC == 8 || MO) ? 128 : kSigTile;  // spins per staged tile (static shared memory stays < 48 KB)
    __shared__ __align__(128) PosT shA[2][TILE];
    __shared__ __align__(128) float4 shS[2][TILE];
    constexpr int WQ = NC / 2;  // float4 per spin
    __shared__ __align__(128) float4 shW[2][WQ * TILE];
    __shared__ __align__(128) PosT shV[MO ? 2 : 1][MO ? TILE : 1];
    __shared__ __align__(8) uint64_t bar[2];
    const RecT *recs = reinterpret_cast<const RecT *>(recs_);
    const PosT *A = reinterpret_cast<const PosT *>(A_);
    const PosT *V = reinterpret_cast<const PosT *>(V_);
    constexpr int RS = MO ? 2 : 1;
    const int tid = threadIdx.x;
    const int s0 = blockIdx.y * spins_per_chunk;
    const int s1 = min(n_spins, s0 + spins_per_chunk);
    const int n_tiles = (s1 - s0 + TILE - 1) / TILE;
    auto issue = [&](int t) {
        const int b = t & 1;
        const int base = s0 + t * TILE;
        const uint32_t cnt = (uint32_t)min(TILE, s1 - base);
        mbar_expect_tx(&bar[b], cnt * (uint32_t)((MO ? 2 : 1) * sizeof(PosT) + (1 + WQ) * sizeof(float4)));
        bulk_g2s(shA[b], A + base, cnt * (uint32_t)sizeof(PosT), &bar[b]);
        bulk_g2s(shS[b], S + base, cnt * (uint32_t)sizeof(float4), &bar[b]);
        bulk_g2s(shW[b], W + WQ * (size_t)base, cnt * (uint32_t)(WQ * sizeof(float4)), &bar[b]);
        if (MO) bulk_g2s(shV[b], V + base, cnt * (uint32_t)sizeof(PosT), &bar[b]);
    };
    if (tid == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        mbar_init_fence();
        if (n_tiles > 0) issue(0);
        if (n_tiles > 1) issue(1);
    }
    const int p0 = (blockIdx.x * (int)blockDim.x + tid) * P;  // blockDim.x < kSigThreads for blocks of few samples
    real kx[P], ky[P], kz[P], tau[P], ux[MO ? P : 1], uy[MO ? P : 1], uz[MO ? P : 1];
    float tf[P], cj[P], ar[NC][P], ai[NC][P];
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
        cj[j] = (float)(r.w - tau[0]) * 0.6931471805599453f;
        cmax = fmaxf(cmax, fabsf(cj[j]));
#pragma unroll
        for (int k = 0; k < NC; ++k) { ar[k][j] = 0.f; ai[k][j] = 0.f; }
    }
    const bool series = P > 1 && __all_sync(0xffffffffu, cmax * (scal[0] * kLog2e) <= 0.02f);
    __syncthreads();  // barrier initialisation visible to every waiter
    for (int t = 0; t < n_tiles; ++t) {
        const int b = t & 1;
        mbar_wait(&bar[b], (uint32_t)((t >> 1) & 1));
        const int cnt = min(TILE, s1 - (s0 + t * TILE));
#pragma unroll 2
        for (int s = 0; s < cnt; ++s) {
            const PosT a = shA[b][s];
            const float4 st = shS[b][s];  // (Mxy.re, Mxy.im, Mz, e2 = -log2(e)/T2)
            PosT vv;
            vv.x = 0; vv.y = 0; vv.z = 0; vv.w = 0;
            if (MO) vv = shV[b][s];
            float wr[NC], wi[NC];
#pragma unroll
            for (int q = 0; q < WQ; ++q) {
                const float4 w2 = shW[b][WQ * s + q];
                wr[2 * q] = w2.x; wi[2 * q] = w2.y; wr[2 * q + 1] = w2.z; wi[2 * q + 1] = w2.w;
            }
            float er0 = 0.f, ei0 = 0.f;
#pragma unroll
            for (int j = 0; j < P; ++j) {
                float sn, cs;
                if (PH64) {
                    double th = fma((double)kx[j], (double)a.x, fma((double)ky[j], (double)a.y,
                                    fma((double)kz[j], (double)a.z, (double)tau[j] * (double)a.w)));  // turns
                    if (MO) th = fma((double)ux[j], (double)vv.x, fma((double)uy[j], (double)vv.y,
                                     fma((double)uz[j], (double)vv.z, th)));
                    th += 1572864.0;  // 1.5 * 2^20: the low word is frac(theta) in 0.32 fixed point (signal.cuh)
                    const unsigned lo = (unsigned)__double2loint(th);
                    const float fr = __uint_as_float(0x3f800000u | (lo >> 9)) - 1.0f;
                    const float ang = fr * 6.283185307179586f;
                    sn = __sinf(ang);
                    cs = __cosf(ang);
                } else {
                    float th = fmaf((float)kx[j], (float)a.x, fmaf((float)ky[j], (float)a.y,
                                    fmaf((float)kz[j], (float)a.z, (float)tau[j] * (float)a.w)));  // radians
                    if (MO) th = fmaf((float)ux[j], (float)vv.x, fmaf((float)uy[j], (float)vv.y,
                                      fmaf((float)uz[j], (float)vv.z, th)));
                    sn = __sinf(th);
                    cs = __cosf(th);
                }
                float er, ei;
                if (j == 0 || !series) {
                    const float e = ex2_approx(tf[j] * st.w);
                    er = st.x * e;
                    ei = st.y * e;
                    if (j == 0) { er0 = er; ei0 = ei; }
                } else {
                    const float y = cj[j] * st.w;
                    const float pe = fmaf(y, fmaf(y, fmaf(y, 1.0f / 6.0f, 0.5f), 1.0f), 1.0f);
                    er = er0 * pe;
                    ei = ei0 * pe;
                }
                const float cr = fmaf(er, cs, -ei * sn);  // c_in, once for all coils
                const float ci = fmaf(er, sn, ei * cs);
#pragma unroll
                for (int k = 0; k < NC; ++k) {
                    ar[k][j] = fmaf(wr[k], cr, fmaf(-wi[k], ci, ar[k][j]));
                    ai[k][j] = fmaf(wr[k], ci, fmaf(wi[k], cr, ai[k][j]));
                }
            }
        }
        __syncthreads();  // every thread is done with stage b
        if (tid == 0 && t + 2 < n_tiles) issue(t + 2);
    }
    const size_t coil_stride = (size_t)gridDim.y * (size_t)n_pts;
#pragma unroll
    for (int j = 0; j < P; ++j) {
        const int p = p0 + j;
        if (p < n_pts) {
#pragma unroll
            for (int k = 0; k < NC; ++k)
                partial[k * coil_stride + (size_t)blockIdx.y * n_pts + p] = make_float2(ar[k][j], ai[k][j]);
        }
    }
}

// Second pass: blockIdx.y = coil of the pass; chunks added in index order.  out row stride = n_adc_total.
__global__ void __launch_bounds__(256)
reduce_coils_kernel(const float2 *__restrict__ partial, int n_chunks, int n_pts, float2 *__restrict__ out,
                    long long n_adc_total) {
    __shared__ float2 sh[8][33];
    const int p = blockIdx.x * 32 + threadIdx.x;
    const float2 *src = partial + (size_t)blockIdx.y * (size_t)n_chunks * (size_t)n_pts;
    float re = 0.f, im = 0.f;
    if (p < n_pts) {
        for (int c = threadIdx.y; c < n_chunks; c += 8) {
            const float2 v = src[(size_t)c * n_pts + p];
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
        out[(size_t)blockIdx.y * (size_t)n_adc_total + p] = make_float2(re, im);
    }
}

}  // namespace bloch
