// Line FFT machinery of the own transform kernels (se_zfft.cuh): complex type, in-register radix-2/4/8/16 butterflies
// and one Stockham stage on a shared-memory line (the 3-D transforms of PAPER.md Sec. 3.1 L265 and L326 are separable;
// these are their 1-D factors).  A line of M complex values is transformed by the M/16 threads of ONE warp: a thread owns
// 16 values per stage, loads them, the warp synchronises, and it writes them to their autosort positions; twiddles come
// from a table made on the host.
#pragma once
#include "se_common.cuh"

struct __align__(16) cplx { double x, y; };

// position of x inside a line: one extra slot per 2^LV values, so that the stride-2^LV writes of the first stage
// (x = V j + r over consecutive j) fall in distinct banks
template <int LV> __host__ __device__ inline int xf_sk(int x) { return x + (x >> LV); }

__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return { a.x + b.x, a.y + b.y }; }
__device__ __forceinline__ cplx csub(cplx a, cplx b) { return { a.x - b.x, a.y - b.y }; }
__device__ __forceinline__ cplx cmul(cplx a, cplx b) { return { a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x }; }
// multiply by -i (forward) or +i (inverse)
template <bool INV> __device__ __forceinline__ cplx cmuli(cplx a) { return INV ? cplx{ -a.y, a.x } : cplx{ a.y, -a.x }; }

// exp(-+ 2 pi i k / 16), k = 0..7, as compile-time constants
template <bool INV> __device__ __forceinline__ cplx w16(int k)
{
    constexpr double C[8] = { 1.0, 0.92387953251128674, 0.70710678118654752, 0.38268343236508977,
                              0.0, -0.38268343236508977, -0.70710678118654752, -0.92387953251128674 };
    constexpr double S[8] = { 0.0, 0.38268343236508977, 0.70710678118654752, 0.92387953251128674,
                              1.0, 0.92387953251128674, 0.70710678118654752, 0.38268343236508977 };
    return { C[k], INV ? S[k] : -S[k] };
}

// In-register FFT of R values v[0], v[S], ..., v[(R-1) S] (decimation in time, natural order out).
template <int R, int S, bool INV> struct RegFft {
    static __device__ __forceinline__ void run(cplx *v)
    {
        RegFft<R / 2, 2 * S, INV>::run(v);            // even samples
        RegFft<R / 2, 2 * S, INV>::run(v + S);        // odd samples
        cplx e[R / 2], o[R / 2];
#pragma unroll
        for (int k = 0; k < R / 2; ++k) { e[k] = v[2 * k * S]; o[k] = v[(2 * k + 1) * S]; }
#pragma unroll
        for (int k = 0; k < R / 2; ++k) {
            const int tw = k * (16 / R);
            const cplx t = tw == 0 ? o[k] : (tw == 4 ? cmuli<INV>(o[k]) : cmul(o[k], w16<INV>(tw)));
            v[k * S] = cadd(e[k], t);
            v[(k + R / 2) * S] = csub(e[k], t);
        }
    }
};
template <int S, bool INV> struct RegFft<1, S, INV> {
    static __device__ __forceinline__ void run(cplx *) {}
};

// One Stockham stage of radix R on one line (M complex values, contiguous), in place.  The M/16 threads of a
// line sit in one warp: each loads its 16 values (x = jj + q M/16, q = 0..15), the warp synchronises, then the
// 16/R butterflies j = jj + u M/16 are twiddled, transformed in registers and written to their autosort positions
//   out[(j / Ns) Ns R + (j mod Ns) + r Ns] = v_r          (Ns = product of the radices of earlier stages).
template <int LV, int R, bool INV>
__device__ __forceinline__ void xf_stage(cplx *__restrict__ line, const cplx *__restrict__ W, int M, int lNs, int jj)
{
    constexpr int V = 1 << LV, NB = V / R;           // values, butterflies per thread
    const int M16 = M >> LV, Ns = 1 << lNs;          // M / V
    cplx v[V];
#pragma unroll
    for (int q = 0; q < V; ++q) v[q] = line[xf_sk<LV>(jj + q * M16)];
    __syncwarp();
    const int twstep = M >> (lNs + (R == 16 ? 4 : R == 8 ? 3 : R == 4 ? 2 : 1));       // M / (Ns R)
#pragma unroll
    for (int u = 0; u < NB; ++u) {
        const int j = jj + u * M16, k = j & (Ns - 1);
        if (lNs > 0) {
#pragma unroll
            for (int r = 1; r < R; ++r) {
                cplx w = W[r * k * twstep];
                if (INV) w.y = -w.y;
                v[u + r * NB] = cmul(v[u + r * NB], w);
            }
        }
        RegFft<R, NB, INV>::run(v + u);
        const int base = ((j >> lNs) << lNs) * R + k;
#pragma unroll
        for (int r = 0; r < R; ++r) line[xf_sk<LV>(base + r * Ns)] = v[u + r * NB];
    }
    __syncwarp();
}

// Length-M transform of one line, in place (M = 2^lM, 32 <= M <= 512); warp-local synchronisation only.
template <int LV, bool INV>
__device__ __forceinline__ void xf_fft(cplx *__restrict__ line, const cplx *__restrict__ W, int M, int lM, int jj)
{
    int lNs = 0;
    while (lM - lNs >= LV) { xf_stage<LV, (1 << LV), INV>(line, W, M, lNs, jj); lNs += LV; }
    const int rem = lM - lNs;
    if (LV > 3 && rem == 3) xf_stage<LV, (LV > 3 ? 8 : 2), INV>(line, W, M, lNs, jj);
    else if (rem == 2) xf_stage<LV, 4, INV>(line, W, M, lNs, jj);
    else if (rem == 1) xf_stage<LV, 2, INV>(line, W, M, lNs, jj);
}

// power-of-two grids the own transform kernels support
static inline bool xf_supported(int M) { return M >= 32 && M <= 512 && (M & (M - 1)) == 0; }
