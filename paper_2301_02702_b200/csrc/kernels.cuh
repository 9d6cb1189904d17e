// kernels.cuh -- device code of the hot path for sm_100a.
//
// Internal spin layout (built once per bloch_simulate by pack_kernel, 48 B per spin; +32 B with fp64 phase):
//   A[i] = (x, y, z, f')        f' = -dw  [rad/s]                  constant
//   V[i]  = (vx, vy, vz, 0)     velocity [m/s], motion plans only (Vd[i]: the same as doubles, fp64 phase)
//   Ad[i] = (x, y, z, f') as doubles, f' = -dw / (2 pi) [turns/s]  constant, fp64-phase plans only
//   C[i] = (1/T1, 1/T2, M0, dw)                                   constant
//   S[i] = (Mxy.re, Mxy.im, Mz, e2)   e2 = -(1/T2) log2(e)        state (e2 rides along for the signal kernel)
//
// Phase convention (reading G3): Mxy(t) = Mxy(0) exp(-t/T2) exp(-i (2 pi gamma_bar K.x + dw t)); the tables
// hold k' = -gamma K [rad/m] (fp32 phase) or -gamma_bar K [turns/m] (fp64 phase, block-end records), so that
// the phase is theta = k'.x + f' tau.
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>

#include "internal.h"

namespace bloch {

constexpr float kInv2Pi = 0.15915494309189535f;
constexpr float kTwoPi = 6.283185307179586f;
constexpr float kLog2e = 1.4426950408889634f;

__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// ------------------------------------------------------------------------------------------------
// a5: spin state init / pack, and a9: unpack
// ------------------------------------------------------------------------------------------------
__global__ void pack_kernel(int n, const float *__restrict__ x, const float *__restrict__ y,
                            const float *__restrict__ z, const float *__restrict__ M0,
                            const float *__restrict__ T1, const float *__restrict__ T2,
                            const float *__restrict__ dw, const float2 *__restrict__ Mxy,
                            const float *__restrict__ Mz, int init_eq, float4 *__restrict__ A,
                            float4 *__restrict__ Cc, float4 *__restrict__ S, double4 *__restrict__ Ad,
                            unsigned *__restrict__ scal, const float *__restrict__ vx,
                            const float *__restrict__ vy, const float *__restrict__ vz, float4 *__restrict__ V,
                            double4 *__restrict__ Vd) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    // scal[kScalR2Max] = max 1/T2 over the spins (the signal kernels bound their series with it), and what
    // bloch_plan_status reports about the phantom: max |x|^2, max |dw|, max |v|^2, and flags for T1 / T2 <= 0 or
    // non-finite input.  The bit pattern of a non-negative float orders like the unsigned integer and an integer
    // max / or is order-independent, so all of this stays reproducible.
    float r2w = 0.f, x2w = 0.f, dww = 0.f, v2w = 0.f;
    unsigned bad = 0;
    if (i < n) {
        const float t1 = T1[i], t2 = T2[i], px = x[i], py = y[i], pz = z[i], w = dw[i], m0 = M0[i];
        r2w = 1.0f / t2;
        x2w = fmaf(px, px, fmaf(py, py, pz * pz));
        dww = fabsf(w);
        const float a = vx ? vx[i] : 0.f, b = vy ? vy[i] : 0.f, c = vz ? vz[i] : 0.f;
        v2w = fmaf(a, a, fmaf(b, b, c * c));
        if (!(t1 > 0.f) || !(t2 > 0.f) || isinf(t1) || isinf(t2)) bad |= BLOCH_STATUS_BAD_RELAXATION;  // NaN fails t > 0
        if (!isfinite(x2w) || !isfinite(w) || !isfinite(m0) || !isfinite(v2w)) bad |= BLOCH_STATUS_NONFINITE;
        if (!init_eq) {
            const float2 m = Mxy[i];
            if (!isfinite(m.x) || !isfinite(m.y) || !isfinite(Mz[i])) bad |= BLOCH_STATUS_NONFINITE;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        r2w = fmaxf(r2w, __shfl_xor_sync(0xffffffffu, r2w, o));
        x2w = fmaxf(x2w, __shfl_xor_sync(0xffffffffu, x2w, o));
        dww = fmaxf(dww, __shfl_xor_sync(0xffffffffu, dww, o));
        v2w = fmaxf(v2w, __shfl_xor_sync(0xffffffffu, v2w, o));
    }
    bad = __reduce_or_sync(0xffffffffu, bad);
    if ((threadIdx.x & 31) == 0) {
        // fmaxf drops NaNs and the clamp keeps +inf / negative values out of the integer ordering's way
        atomicMax(scal + kScalR2Max, __float_as_uint(fminf(fmaxf(r2w, 0.f), 3.0e38f)));
        atomicMax(scal + kScalX2Max, __float_as_uint(fminf(fmaxf(x2w, 0.f), 3.0e38f)));
        atomicMax(scal + kScalDwMax, __float_as_uint(fminf(fmaxf(dww, 0.f), 3.0e38f)));
        atomicMax(scal + kScalV2Max, __float_as_uint(fminf(fmaxf(v2w, 0.f), 3.0e38f)));
        if (bad) atomicOr(scal + kScalFlags, bad);
        if (i == 0) scal[kScalValid] = 1u;
    }
    if (i >= n) return;
    const float r1 = 1.0f / T1[i], r2 = 1.0f / T2[i], m0 = M0[i], w = dw[i];
    A[i] = make_float4(x[i], y[i], z[i], -w);
    if (Ad) Ad[i] = make_double4((double)x[i], (double)y[i], (double)z[i], -(double)w * 0.15915494309189535);
    if (V) {  // motion plan: zero velocity when the caller gave none
        const float a = vx ? vx[i] : 0.f, b = vy ? vy[i] : 0.f, c = vz ? vz[i] : 0.f;
        V[i] = make_float4(a, b, c, 0.f);
        if (Vd) Vd[i] = make_double4((double)a, (double)b, (double)c, 0.0);
    }
    Cc[i] = make_float4(r1, r2, m0, w);
    float4 s;
    if (init_eq) {
        s = make_float4(0.f, 0.f, m0, 0.f);  // reading G8: thermal equilibrium
    } else {
        const float2 m = Mxy[i];
        s = make_float4(m.x, m.y, Mz[i], 0.f);
    }
    s.w = -r2 * kLog2e;
    S[i] = s;
}

__global__ void unpack_kernel(int n, const float4 *__restrict__ S, float2 *__restrict__ Mxy,
                              float *__restrict__ Mz) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float4 s = S[i];
    Mxy[i] = make_float2(s.x, s.y);
    Mz[i] = s.z;
}

// ------------------------------------------------------------------------------------------------
// Free precession over a whole block, closed form from the block start (Eq 10-11 are diagonal in
// (Mxy, Mz) and commute, so the step-by-step product collapses exactly; "exact solution").
// Used once per spin per block -> accurate functions, phase in fp64 turns.
// ------------------------------------------------------------------------------------------------
struct PropRec {
    double kx, ky, kz, tau;  // k' = -gamma_bar K(T) [turns/m], tau = T [s]
    double mx, my, mz;       // motion: first moment mu'(T) [turns s/m]
};

__device__ __forceinline__ void propagate(const PropRec &p, const float4 &a, const float4 &c, const float4 &v,
                                          float &mx, float &my, float &mz) {
    // every contraction is written out (__fma_rn / __fmaf_rn / __fmul_rn), so rf_kernel and seq_kernel round alike
    double th = __fma_rn(p.kx, (double)a.x, __fma_rn(p.ky, (double)a.y, __fma_rn(p.kz, (double)a.z,
                         -__dmul_rn(__dmul_rn((double)c.w, 0.15915494309189535), p.tau))));
    th = __fma_rn(p.mx, (double)v.x, __fma_rn(p.my, (double)v.y, __fma_rn(p.mz, (double)v.z, th)));  // x(t) = x + v t
    th -= rint(th);
    float sn, cs;
    sincospif(2.0f * (float)th, &sn, &cs);
    const float tau = (float)p.tau;
    const float e2 = expf(-__fmul_rn(tau, c.y)), e1 = expf(-__fmul_rn(tau, c.x));
    const float ax = __fmul_rn(mx, e2), ay = __fmul_rn(my, e2);
    mx = __fmaf_rn(ax, cs, -__fmul_rn(ay, sn));
    my = __fmaf_rn(ax, sn, __fmul_rn(ay, cs));
    mz = __fmaf_rn(__fsub_rn(mz, c.z), e1, c.z);  // Eq 11
}

// One evaluated point of a precession block for the accurate (per-spin / grouped) readouts: its record as doubles in
// turns/m and seconds, whatever the table's format (fp64-phase tables hold turns/m, fp32-phase tables rad/m), and the
// first-moment record that follows it in motion plans.
struct PointRec {
    double kx, ky, kz, tau, ux, uy, uz;
};
template <bool PH64>
__device__ __forceinline__ PointRec load_point(const void *__restrict__ recs_, int p, bool motion) {
    PointRec r;
    r.ux = 0.; r.uy = 0.; r.uz = 0.;
    const int rs = motion ? 2 : 1;  // motion plans: (k', tau) is followed by (mu', 0)
    if (PH64) {
        const double4 q = reinterpret_cast<const double4 *>(recs_)[rs * p];
        r.kx = q.x; r.ky = q.y; r.kz = q.z; r.tau = q.w;
        if (motion) {
            const double4 m = reinterpret_cast<const double4 *>(recs_)[rs * p + 1];
            r.ux = m.x; r.uy = m.y; r.uz = m.z;
        }
    } else {
        const float4 q = reinterpret_cast<const float4 *>(recs_)[rs * p];
        r.kx = (double)q.x * 0.15915494309189535; r.ky = (double)q.y * 0.15915494309189535;
        r.kz = (double)q.z * 0.15915494309189535; r.tau = q.w;
        if (motion) {
            const float4 m = reinterpret_cast<const float4 *>(recs_)[rs * p + 1];
            r.ux = (double)m.x * 0.15915494309189535; r.uy = (double)m.y * 0.15915494309189535;
            r.uz = (double)m.z * 0.15915494309189535;
        }
    }
    return r;
}

// c_in = Mxy(0) exp(-tau/T2) exp(i theta) of one spin at one point, accurate functions, phase in fp64 turns
__device__ __forceinline__ float2 accurate_contribution(const PointRec &r, const float4 &a, const float4 &c, const float4 &s,
                                                        const float4 *v) {
    double th = r.kx * (double)a.x + r.ky * (double)a.y + r.kz * (double)a.z - (double)c.w * 0.15915494309189535 * r.tau;
    if (v) th += r.ux * (double)v->x + r.uy * (double)v->y + r.uz * (double)v->z;
    th -= rint(th);
    float sn, cs;
    sincospif(2.0f * (float)th, &sn, &cs);
    const float e = expf(-(float)r.tau * c.y);
    const float er = s.x * e, ei = s.y * e;
    return make_float2(er * cs - ei * sn, er * sn + ei * cs);
}

// PER_SPIN output (dictionary mode): one thread per (spin, point); accurate functions because nothing
// averages the per-evaluation error; phase in fp64 turns.  recs are float4 or double4 by PH64.
template <bool PH64>
__global__ void __launch_bounds__(256)
perspin_kernel(const void *__restrict__ recs_, int n_pts, const float4 *__restrict__ A,
               const float4 *__restrict__ Cc, const float4 *__restrict__ S, const float4 *__restrict__ V,
               int n_spins, long long n_adc_total, long long adc_first, float2 *__restrict__ out) {
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= (long long)n_spins * n_pts) return;
    const int sp = (int)(gid / n_pts), p = (int)(gid % n_pts);
    const PointRec r = load_point<PH64>(recs_, p, V != nullptr);
    const float4 a = A[sp], c = Cc[sp], s = S[sp];
    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
    if (V) v = V[sp];
    out[(size_t)sp * n_adc_total + adc_first + p] = accurate_contribution(r, a, c, s, V ? &v : nullptr);
}

// GROUPED output: one warp per group of `gs` consecutive spins (an isochromat ensemble);
// the lanes take the group's spins, evaluate the block's points one after the other with the accurate
// functions of perspin_kernel, and add up with a fixed butterfly (bitwise reproducible); lane 0 writes
// out[group][adc].
template <bool PH64>
__global__ void __launch_bounds__(256)
grouped_kernel(const void *__restrict__ recs_, int n_pts, const float4 *__restrict__ A,
               const float4 *__restrict__ Cc, const float4 *__restrict__ S, const float4 *__restrict__ V,
               int n_groups, int gs, long long n_adc_total, long long adc_first, float2 *__restrict__ out) {
    const int warp = (int)(((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
    if (warp >= n_groups) return;
    const long long s0 = (long long)warp * gs;
    for (int p = 0; p < n_pts; ++p) {
        const PointRec r = load_point<PH64>(recs_, p, V != nullptr);
        float re = 0.f, im = 0.f;
        for (int k = lane; k < gs; k += 32) {
            const float4 a = A[s0 + k], c = Cc[s0 + k], s = S[s0 + k];
            float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
            if (V) v = V[s0 + k];
            const float2 w = accurate_contribution(r, a, c, s, V ? &v : nullptr);
            re += w.x;
            im += w.y;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            re += __shfl_xor_sync(0xffffffffu, re, o);
            im += __shfl_xor_sync(0xffffffffu, im, o);
        }
        if (lane == 0) out[(size_t)warp * n_adc_total + adc_first + p] = make_float2(re, im);
    }
}

// ------------------------------------------------------------------------------------------------
// pipe micro-benchmarks (roofline denominators)
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) mb_mufu(int iters, float *out) {
    float v[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) v[k] = 0.001f * (threadIdx.x + k);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            v[k] = __sinf(v[k]);
            v[k] = __cosf(v[k]);
            v[k] = ex2_approx(v[k]);
        }
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += v[k];
    if (s == 123.456f) out[0] = s;
}
__global__ void __launch_bounds__(256) mb_ffma(int iters, float *out) {
    float v[8];
    const float a = 1.0f + 1e-7f * threadIdx.x, b = 1e-9f * blockIdx.x;
#pragma unroll
    for (int k = 0; k < 8; ++k) v[k] = 0.001f * (threadIdx.x + k);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int k = 0; k < 8; ++k) v[k] = fmaf(v[k], a, b);
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += v[k];
    if (s == 123.456f) out[0] = s;
}
// FFMA whose three source operands are three different, changing registers (no operand reuse, no immediate):
// the form most FFMAs of the RF step have (cross products).  The register file delivers about two 32-bit operands
// per lane per clock, so this runs at ~2/3 of the mb_ffma rate.
__global__ void __launch_bounds__(256) mb_ffma3(int iters, float *out) {
    float v[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) v[k] = 0.5f + 0.001f * (threadIdx.x + k);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int k = 0; k < 8; ++k)
                asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(v[k]) : "f"(v[(k + 3) & 7]), "f"(v[(k + 5) & 7]));
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += v[k];
    if (s == 123.456f) out[0] = s;
}
__global__ void __launch_bounds__(256) mb_dfma(int iters, float *out) {
    double v[8];
    const double a = 1.0 + 1e-12 * threadIdx.x, b = 1e-15 * blockIdx.x;
#pragma unroll
    for (int k = 0; k < 8; ++k) v[k] = 0.001 * (threadIdx.x + k);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int k = 0; k < 8; ++k) v[k] = fma(v[k], a, b);
    }
    double s = 0.;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += v[k];
    if (s == 123.456) out[0] = (float)s;
}

}  // namespace bloch
