// kernels.cuh -- device code of the hot path for sm_100a.
//
// Internal spin layout (built once per bloch_simulate by pack_kernel, 48 B per spin):
//   A[i] = (x, y, z, f')        f' = -dw / (2 pi)  [turns/s]     constant
//   C[i] = (1/T1, 1/T2, M0, dw)                                   constant
//   S[i] = (Mxy.re, Mxy.im, Mz, e2)   e2 = -(1/T2) log2(e)        state (e2 rides along for the signal kernel)
//
// Phase convention (reading G3): Mxy(t) = Mxy(0) exp(-t/T2) exp(-i (2 pi gamma_bar K.x + dw t)); the tables
// hold k' = -gamma_bar K [turns/m] so that the phase in turns is theta = k'.x + f' tau.
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>

namespace bloch {

constexpr float kInv2Pi = 0.15915494309189535f;
constexpr float kTwoPi = 6.283185307179586f;
constexpr float kLog2e = 1.4426950408889634f;

// ------------------------------------------------------------------------------------------------
// a5: spin state init / pack, and a9: unpack
// ------------------------------------------------------------------------------------------------
__global__ void pack_kernel(int n, const float *__restrict__ x, const float *__restrict__ y,
                            const float *__restrict__ z, const float *__restrict__ M0,
                            const float *__restrict__ T1, const float *__restrict__ T2,
                            const float *__restrict__ dw, const float2 *__restrict__ Mxy,
                            const float *__restrict__ Mz, int init_eq, float4 *__restrict__ A,
                            float4 *__restrict__ Cc, float4 *__restrict__ S) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float r1 = 1.0f / T1[i], r2 = 1.0f / T2[i], m0 = M0[i], w = dw[i];
    A[i] = make_float4(x[i], y[i], z[i], -w * kInv2Pi);
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
};

__device__ __forceinline__ void propagate(const PropRec &p, const float4 &a, const float4 &c, float &mx,
                                          float &my, float &mz) {
    double th = p.kx * (double)a.x + p.ky * (double)a.y + p.kz * (double)a.z -
                (double)c.w * 0.15915494309189535 * p.tau;
    th -= rint(th);
    float sn, cs;
    sincospif(2.0f * (float)th, &sn, &cs);
    const float tau = (float)p.tau;
    const float e2 = expf(-tau * c.y), e1 = expf(-tau * c.x);
    const float ax = mx * e2, ay = my * e2;
    mx = ax * cs - ay * sn;
    my = ax * sn + ay * cs;
    mz = c.z + (mz - c.z) * e1;  // Eq 11
}

// ------------------------------------------------------------------------------------------------
// a6 + a7: free-precession signal kernel (SUM_ALL).
//
// Grid = (point tiles, spin chunks).  A thread OWNS P evaluated points (k', tau in registers) and walks the
// spins of its chunk, which are staged through shared memory and broadcast to all threads (every lane
// reads the same address: conflict-free LDS.128).  The sum over spins is therefore thread-local: no
// shuffles, no atomics.  Each CTA writes its partial sums P[chunk][point]; reduce_kernel adds the chunks
// in index order (deterministic two-pass reduction, "add them later").
// Per evaluation: 4 FMA phase, 3 ops range reduction to [-1/2, 1/2] turns, MUFU sin + cos, MUFU ex2,
// 2 mul + 4 FMA complex multiply-accumulate.
// ------------------------------------------------------------------------------------------------
constexpr int kSigThreads = 256;

__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

template <int P>
__global__ void __launch_bounds__(kSigThreads)
signal_kernel_f32(const float4 *__restrict__ recs, int n_pts, const float4 *__restrict__ A,
                  const float4 *__restrict__ S, int n_spins, int spins_per_chunk,
                  float2 *__restrict__ partial) {
    __shared__ float4 shA[kSigThreads];
    __shared__ float4 shB[kSigThreads];
    const int tid = threadIdx.x;
    const int p0 = blockIdx.x * (kSigThreads * P) + tid;
    float kx[P], ky[P], kz[P], tau[P], ar[P], ai[P];
#pragma unroll
    for (int j = 0; j < P; ++j) {
        const int p = p0 + j * kSigThreads;
        const float4 r = p < n_pts ? recs[p] : make_float4(0.f, 0.f, 0.f, 0.f);
        kx[j] = r.x; ky[j] = r.y; kz[j] = r.z; tau[j] = r.w;
        ar[j] = 0.f; ai[j] = 0.f;
    }
    const int s0 = blockIdx.y * spins_per_chunk;
    const int s1 = min(n_spins, s0 + spins_per_chunk);
    for (int base = s0; base < s1; base += kSigThreads) {
        __syncthreads();
        {
            const int idx = base + tid;
            float4 a = make_float4(0.f, 0.f, 0.f, 0.f), b = a;
            if (idx < s1) {
                a = A[idx];
                const float4 st = S[idx];
                b = make_float4(st.w, st.x, st.y, 0.f);
            }
            shA[tid] = a;
            shB[tid] = b;
        }
        __syncthreads();
        const int cnt = min(kSigThreads, s1 - base);
#pragma unroll 2
        for (int s = 0; s < cnt; ++s) {
            const float4 a = shA[s];
            const float4 b = shB[s];
#pragma unroll
            for (int j = 0; j < P; ++j) {
                float th = fmaf(kx[j], a.x, fmaf(ky[j], a.y, fmaf(kz[j], a.z, tau[j] * a.w)));
                th -= (th + 12582912.0f) - 12582912.0f;          // th - rint(th): [-1/2, 1/2] turns
                const float ang = th * kTwoPi;
                const float sn = __sinf(ang), cs = __cosf(ang);  // MUFU.SIN / MUFU.COS
                const float e = ex2_approx(tau[j] * b.x);        // MUFU.EX2: exp(-tau/T2)
                const float er = b.y * e, ei = b.z * e;
                ar[j] = fmaf(er, cs, fmaf(-ei, sn, ar[j]));
                ai[j] = fmaf(er, sn, fmaf(ei, cs, ai[j]));
            }
        }
    }
#pragma unroll
    for (int j = 0; j < P; ++j) {
        const int p = p0 + j * kSigThreads;
        if (p < n_pts) partial[(size_t)blockIdx.y * n_pts + p] = make_float2(ar[j], ai[j]);
    }
}

// fp64 phase accumulation (north_star item 4): k', tau, x, f' in double; the fractional turn goes to
// fp32 for MUFU sin/cos.  4 DFMA + 3 DADD + 1 F2F per evaluation on top of the fp32 work.
template <int P>
__global__ void __launch_bounds__(kSigThreads)
signal_kernel_f64(const double4 *__restrict__ recs, int n_pts, const float4 *__restrict__ A,
                  const float4 *__restrict__ Cc, const float4 *__restrict__ S, int n_spins,
                  int spins_per_chunk, float2 *__restrict__ partial) {
    __shared__ double4 shA[kSigThreads];
    __shared__ float4 shB[kSigThreads];
    const int tid = threadIdx.x;
    const int p0 = blockIdx.x * (kSigThreads * P) + tid;
    double kx[P], ky[P], kz[P], tau[P];
    float tf[P], ar[P], ai[P];
#pragma unroll
    for (int j = 0; j < P; ++j) {
        const int p = p0 + j * kSigThreads;
        const double4 r = p < n_pts ? recs[p] : make_double4(0., 0., 0., 0.);
        kx[j] = r.x; ky[j] = r.y; kz[j] = r.z; tau[j] = r.w;
        tf[j] = (float)r.w;
        ar[j] = 0.f; ai[j] = 0.f;
    }
    const int s0 = blockIdx.y * spins_per_chunk;
    const int s1 = min(n_spins, s0 + spins_per_chunk);
    for (int base = s0; base < s1; base += kSigThreads) {
        __syncthreads();
        {
            const int idx = base + tid;
            double4 a = make_double4(0., 0., 0., 0.);
            float4 b = make_float4(0.f, 0.f, 0.f, 0.f);
            if (idx < s1) {
                const float4 af = A[idx];
                const float4 st = S[idx];
                a = make_double4((double)af.x, (double)af.y, (double)af.z,
                                 -(double)Cc[idx].w * 0.15915494309189535);
                b = make_float4(st.w, st.x, st.y, 0.f);
            }
            shA[tid] = a;
            shB[tid] = b;
        }
        __syncthreads();
        const int cnt = min(kSigThreads, s1 - base);
        for (int s = 0; s < cnt; ++s) {
            const double4 a = shA[s];
            const float4 b = shB[s];
#pragma unroll
            for (int j = 0; j < P; ++j) {
                double th = fma(kx[j], a.x, fma(ky[j], a.y, fma(kz[j], a.z, tau[j] * a.w)));
                th -= (th + 6755399441055744.0) - 6755399441055744.0;   // th - rint(th)
                const float ang = (float)th * kTwoPi;
                const float sn = __sinf(ang), cs = __cosf(ang);
                const float e = ex2_approx(tf[j] * b.x);
                const float er = b.y * e, ei = b.z * e;
                ar[j] = fmaf(er, cs, fmaf(-ei, sn, ar[j]));
                ai[j] = fmaf(er, sn, fmaf(ei, cs, ai[j]));
            }
        }
    }
#pragma unroll
    for (int j = 0; j < P; ++j) {
        const int p = p0 + j * kSigThreads;
        if (p < n_pts) partial[(size_t)blockIdx.y * n_pts + p] = make_float2(ar[j], ai[j]);
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

// PER_SPIN output (dictionary mode): one thread per (spin, point); accurate functions because nothing
// averages the per-evaluation error; phase in fp64 turns.  recs are float4 or double4 by PH64.
template <bool PH64>
__global__ void __launch_bounds__(256)
perspin_kernel(const void *__restrict__ recs_, int n_pts, const float4 *__restrict__ A,
               const float4 *__restrict__ Cc, const float4 *__restrict__ S, int n_spins,
               long long n_adc_total, long long adc_first, float2 *__restrict__ out) {
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= (long long)n_spins * n_pts) return;
    const int sp = (int)(gid / n_pts), p = (int)(gid % n_pts);
    double kx, ky, kz, tau;
    if (PH64) {
        const double4 r = reinterpret_cast<const double4 *>(recs_)[p];
        kx = r.x; ky = r.y; kz = r.z; tau = r.w;
    } else {
        const float4 r = reinterpret_cast<const float4 *>(recs_)[p];
        kx = r.x; ky = r.y; kz = r.z; tau = r.w;
    }
    const float4 a = A[sp], c = Cc[sp], s = S[sp];
    double th = kx * (double)a.x + ky * (double)a.y + kz * (double)a.z - (double)c.w * 0.15915494309189535 * tau;
    th -= rint(th);
    float sn, cs;
    sincospif(2.0f * (float)th, &sn, &cs);
    const float e = expf(-(float)tau * c.y);
    const float er = s.x * e, ei = s.y * e;
    out[(size_t)sp * n_adc_total + adc_first + p] = make_float2(er * cs - ei * sn, er * sn + ei * cs);
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
