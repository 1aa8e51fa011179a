// a4/a5/a6 fused along x: forward FFT over the slowest grid axis, the k-space pass, and the inverse FFT over
// the same axis in ONE kernel and ONE pass over HBM (Eq. 43 with Eq. 36, hybrid Eq. 50-51; the 3-D
// transforms of Sec. 3.1 L265 and L326 are separable).  cuFFT then only does the batched 2-D (y,z) transforms:
//
//   cuFFT D2Z 2-D x 3M planes:  H(x,y,z)       -> H'(x, ky, kz)
//   k_xfused (this file):       H'(x, ky, kz)  -> FFT_x -> H_k -> u_k, w_k = -k^2 u_k -> FFT_x^-1 -> u'(x,ky,kz), w'(x,ky,kz)
//   cuFFT Z2D 2-D x 6M planes:  u', w'         -> u~(x,y,z), w~(x,y,z)
//
// instead of three passes (x transform, k_kspace, x transform back) that read and write the 3 + 6 spectra three
// times.  A CTA owns XF_T consecutive modes of the flattened (ky,kz) plane (contiguous in memory for every x)
// and all M values of x: 3 T lines of M complex values in shared memory (M T = 1024), each transformed in place by
// the M/16 threads of ONE warp with a Stockham FFT whose stages are radix-16 butterflies held in registers (a
// thread owns 16 values per stage: loads them, the warp synchronises, and it writes them to their autosort
// positions), twiddles from a table made on the host.  u_k overwrites H_k, w_k goes to a second buffer; CTA-wide
// barriers only around the load, the k-space pass and the store.
// Opt-in (flag SE_FUSED_X), for power-of-two 32 <= M <= 512 and without the compressible extension; the default is
// own z transforms + 2-D cuFFT + k_kspace (se_zfft.cuh, se_kspace.cuh).  Results agree to FFT round-off.  On B200 the
// kernel is bound by shared memory and registers (103 KB and 168 registers per CTA: 12 warps per SM), not by HBM:
// 0.65 ms at M = 256 against the 0.18 ms HBM floor, which does not yet pay for cuFFT's slower 2-D plans.
#pragma once
#include "se_common.cuh"

#define XF_ELEMS 1024                      // complex values per component and CTA: M * T
// LV = log2 of the values a thread holds per stage: 4 (radix-16 stages, 192 threads; used) or 3 (radix-8 stages,
// 384 threads, M <= 256 only: a line's M/8 threads must fit one warp)
#define XF_THREADS(LV) (3 * XF_ELEMS >> (LV))

struct __align__(16) cplx { double x, y; };

// pad of a shared-memory line (complex values): with T = 1024 / M modes per row of the global arrays, a
// quarter-warp touches T lines x 8/T values; pad = max(1, 8/T) keeps those eight 16-byte words in distinct banks
// position of x inside a line: one extra slot per XF_V values, so that the stride-XF_V writes of the first stage
// (x = V j + r over consecutive j) fall in distinct banks
template <int LV> __host__ __device__ inline int xf_sk(int x) { return x + (x >> LV); }
__host__ __device__ inline int xf_pad(int M) { const int T = XF_ELEMS / M; return T >= 8 ? 1 : 8 / T; }

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

// Hk2: [3][M][M*Zc] complex, the 2-D (y,z) spectra of the spread grids for every x (cuFFT D2Z, batched).
// Gk2: [6][M][M*Zc] complex, out: u' (3) and w' (3), ready for the batched 2-D inverse transforms.
// Wtab: [M] complex, exp(-2 pi i q / M).   Grid: M*Zc / T CTAs of XF_THREADS threads; dynamic smem xf_smem_bytes(M).
// Shared memory: two buffers of 3 T lines (component-major, then the T modes), line pitch M + pad complex values.
template <int LV>
__global__ void __launch_bounds__(XF_THREADS(LV), 2) k_xfused(SeConst c, int lM, const double2 *__restrict__ Hk2, double2 *__restrict__ Gk2,
                                                          const double2 *__restrict__ Wtab)
{
    extern __shared__ __align__(16) unsigned char xf_smem[];
    const int M = c.M, lT = 10 - lM, T = 1 << lT, Zc = M / 2 + 1;          // M = 2^lM, T = 1024 / M: shifts, no divisions
    constexpr int NT = XF_THREADS(LV);
    const int LP = xf_sk<LV>(M) + xf_pad(M);               // line pitch: conflict-free row-wise phases
    const size_t plane = (size_t)M * Zc;                   // complex values per x
    cplx *A = reinterpret_cast<cplx *>(xf_smem), *B = A + 3 * T * LP, *W = B + 3 * T * LP;
    const int tid = threadIdx.x;
    const size_t idx0 = (size_t)blockIdx.x * T;            // first flattened (ky,kz) mode of this CTA
    constexpr int NLD = 3 * XF_ELEMS / NT;                 // 2^LV values per thread and buffer
    // load: rows (comp, x) of T contiguous complex values; consecutive threads take consecutive 16-byte values;
    // all 16 loads of a thread are in flight before the first is stored
    {
        double2 h[NLD];
#pragma unroll
        for (int n = 0; n < NLD; ++n) {
            const int e = tid + n * NT, row = e >> lT, tt = e & (T - 1);
            h[n] = __ldcs(Hk2 + (size_t)row * plane + idx0 + tt);
        }
        for (int q = tid; q < M; q += NT) { const double2 w = Wtab[q]; W[q] = { w.x, w.y }; }
#pragma unroll
        for (int n = 0; n < NLD; ++n) {
            const int e = tid + n * NT, row = e >> lT, tt = e & (T - 1);
            const int cc = row >> lM, x = row & (M - 1);
            A[(cc * T + tt) * LP + xf_sk<LV>(x)] = { h[n].x, h[n].y };
        }
    }
    __syncthreads();
    const int M16 = M >> LV, myline = tid >> (lM - LV), jj = tid & (M16 - 1);      // 3 T lines x M/16 threads = 192
    xf_fft<LV, false>(A + myline * LP, W, M, lM, jj);
    __syncthreads();

    // k-space pass: u_k in place of H_k (buffer A), w_k = -k^2 u_k in buffer B
    const int iy0 = (int)(idx0 / Zc), iz0 = (int)(idx0 - (size_t)iy0 * Zc);
    for (int e = tid; e < XF_ELEMS; e += NT) {
        const int ix = e >> lT, t2 = e & (T - 1);
        int iy = iy0, iz = iz0 + t2;
        while (iz >= Zc) { iz -= Zc; ++iy; }
        cplx u0 = { 0.0, 0.0 }, u1 = u0, u2 = u0, w0 = u0, w1 = u0, w2 = u0;
        const int a0 = t2 * LP + xf_sk<LV>(ix), a1 = a0 + T * LP, a2 = a1 + T * LP;
        const bool zero = (ix == 0 && iy == 0 && iz == 0) || ix == M / 2 || iy == M / 2 || iz == M / 2;
        if (!zero) {
            const int jx = ix < M / 2 ? ix : ix - M, jy = iy < M / 2 ? iy : iy - M;
            const double kx = c.twopiL * jx, ky = c.twopiL * jy, kz = c.twopiL * iz;
            const double k2 = kx * kx + ky * ky + kz * kz;
            const double sc = c.scale0 * (1.0 + k2 * c.inv4xi2) * exp(-c.dec * k2) / k2;
            const cplx h0 = A[a0], h1 = A[a1], h2 = A[a2];
            const double pr = (kx * h0.x + ky * h1.x + kz * h2.x) / k2, pi = (kx * h0.y + ky * h1.y + kz * h2.y) / k2;
            u0 = { sc * (h0.x - kx * pr), sc * (h0.y - kx * pi) };
            u1 = { sc * (h1.x - ky * pr), sc * (h1.y - ky * pi) };
            u2 = { sc * (h2.x - kz * pr), sc * (h2.y - kz * pi) };
            w0 = { -k2 * u0.x, -k2 * u0.y }; w1 = { -k2 * u1.x, -k2 * u1.y }; w2 = { -k2 * u2.x, -k2 * u2.y };
        }
        A[a0] = u0; A[a1] = u1; A[a2] = u2;
        B[a0] = w0; B[a1] = w1; B[a2] = w2;
    }
    __syncthreads();
    xf_fft<LV, true>(A + myline * LP, W, M, lM, jj);
    xf_fft<LV, true>(B + myline * LP, W, M, lM, jj);
    __syncthreads();
#pragma unroll
    for (int pass = 0; pass < 2; ++pass) {
        const cplx *__restrict__ S = pass ? B : A;
#pragma unroll
        for (int n = 0; n < NLD; ++n) {
            const int e = tid + n * NT, row = e >> lT, tt = e & (T - 1);
            const int cc = row >> lM, x = row & (M - 1);
            const cplx v = S[(cc * T + tt) * LP + xf_sk<LV>(x)];
            __stcs(Gk2 + ((size_t)pass * 3 * M + row) * plane + idx0 + tt, make_double2(v.x, v.y));
        }
    }
}

// radix-16 register blocks for every supported M: the radix-8 variant (twice the warps, three stages instead of two at
// M = 256) measured slower on B200 (0.80 against 0.65 ms at c4)
static inline int xf_lv(int M) { (void)M; return 4; }
static inline size_t xf_smem_bytes(int M)
{
    const int T = XF_ELEMS / M, LP = (xf_lv(M) == 4 ? xf_sk<4>(M) : xf_sk<3>(M)) + xf_pad(M);
    return (size_t)(6 * T * LP + M) * 16;
}
// M (M/2 + 1) must be a multiple of T = 1024 / M: true for every power of two from 32 on
static inline bool xf_supported(int M) { return M >= 32 && M <= 512 && (M & (M - 1)) == 0; }
