// a4 / a6 along z by hand, with TRANSPOSED spectra (opt-in path SE_ZT; power-of-two 32 <= M <= 512).
//
// cuFFT's 3-D real transforms spend 0.62 of their 1.43 ms (c4) in the two kernels of the contiguous z axis
// (vector_fft_r2c / vector_fft_c2r, ~3.9 TB/s), and its strided 2-D plans are three times slower than its contiguous
// ones.  Here the z transforms are own kernels that write / read the half spectra with kz as the SLOWEST index,
//     spec[g][kz][x][y],   kz = 0 .. M/2,
// so that the remaining (x,y) transforms are cuFFT's fast contiguous batched 2-D complex plans (in place), and the
// k-space pass indexes the same layout (k_kspace<true>).  Same transforms as cuFFT's D2Z / Z2D (signs, no scaling).
//
// A real line h[0..M) is transformed as the complex line z_n = h[2n] + i h[2n+1] of length Nh = M/2 (a Stockham FFT of
// radix-16 register butterflies, one warp-local group of Nh/16 threads per line; se_xfft.cuh) plus the split step
//   forward:  X_k = 1/2 [ (Z_k + conj Z_{Nh-k}) - i w^k (Z_k - conj Z_{Nh-k}) ],  w = e^{-2 pi i / M},  k = 0 .. Nh  (Z_Nh = Z_0)
//   inverse:  Z_k = (X_k + conj X_{Nh-k}) + i w^{-k} (X_k - conj X_{Nh-k}),       k = 0 .. Nh-1,  z = FFT^-1_Nh Z.
// A CTA owns ZT_LINES consecutive y of one (grid, x): rows are read / written coalesced in z on the real side and
// as 512-byte runs in y on the spectral side (through shared memory, odd line pitch: conflict-free both ways).
#pragma once
#include "se_xfft.cuh"

#ifndef ZT_LINES
#define ZT_LINES 16
#endif

// pitch of a line in shared memory (complex values): skewed positions of Nh + 1 values, made odd
__host__ __device__ inline int zt_pitch(int Nh) { return (xf_sk<4>(Nh) + 1) | 1; }
static inline size_t zt_smem_bytes(int M) { return (size_t)(ZT_LINES * zt_pitch(M / 2) + M / 2 + M / 2 + 1) * 16; }
static inline int zt_threads(int M) { return ZT_LINES * (M / 2) / 16; }

// H: [ng][M][M][M] real -> spec: [ng][M/2+1][M][M] complex.  Wtab: [M] complex, exp(-2 pi i q / M).
// Grid: ng * M * (M / ZT_LINES) CTAs of ZT_LINES * Nh / 16 threads.
__global__ void __launch_bounds__(ZT_LINES * 16) k_zfft_r2c(int M, int lNh, const double *__restrict__ H, double2 *__restrict__ spec,
                                                           const double2 *__restrict__ Wtab)
{
    extern __shared__ __align__(16) unsigned char zt_smem[];
    const int Nh = M >> 1, Zc = Nh + 1, LP = zt_pitch(Nh), nt = blockDim.x, tid = threadIdx.x;
    cplx *L = reinterpret_cast<cplx *>(zt_smem), *WN = L + ZT_LINES * LP, *WP = WN + Nh;
    const int nyb = M / ZT_LINES;
    const int yb = blockIdx.x % nyb, gx = blockIdx.x / nyb;               // gx = g * M + x
    const int y0 = yb * ZT_LINES, g = gx / M, x = gx - g * M;
    for (int q = tid; q < Nh; q += nt) { const double2 w = Wtab[2 * q]; WN[q] = { w.x, w.y }; }
    for (int q = tid; q <= Nh; q += nt) { const double2 w = q < M ? Wtab[q] : make_double2(1.0, 0.0); WP[q] = { w.x, w.y }; }
    const double2 *__restrict__ rows = reinterpret_cast<const double2 *>(H + ((size_t)gx * M + y0) * M);
    {   // ZT_LINES * Nh = 16 nt values: all sixteen loads of a thread in flight before the first is stored
        double2 v[16];
#pragma unroll
        for (int q = 0; q < 16; ++q) v[q] = __ldcs(rows + tid + q * nt);          // the block's rows are contiguous
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            const int e = tid + q * nt, r = e >> lNh, n = e & (Nh - 1);
            L[r * LP + xf_sk<4>(n)] = { v[q].x, v[q].y };
        }
    }
    __syncthreads();
    {
        const int tpl = Nh >> 4, line = tid / tpl, jj = tid - line * tpl;
        xf_fft<4, false>(L + line * LP, WN, Nh, lNh, jj);
    }
    __syncthreads();
    double2 *__restrict__ out = spec + (((size_t)g * Zc) * M + x) * M + y0;
    const size_t kstride = (size_t)M * M;
    for (int e = tid; e < Zc * ZT_LINES; e += nt) {
        const int k = e / ZT_LINES, r = e - k * ZT_LINES;
        const cplx zk = L[r * LP + xf_sk<4>(k & (Nh - 1))], zm = L[r * LP + xf_sk<4>((Nh - k) & (Nh - 1))];
        const cplx w = WP[k];
        const double sr = zk.x + zm.x, si = zk.y - zm.y;          // Z_k + conj Z_{Nh-k}
        const double dr = zk.x - zm.x, di = zk.y + zm.y;          // Z_k - conj Z_{Nh-k}
        // -i w d = -i (wr + i wi)(dr + i di) = (wr di + wi dr) - i (wr dr - wi di)
        const double tr = w.x * di + w.y * dr, ti = -(w.x * dr - w.y * di);
        __stcs(out + (size_t)k * kstride + r, make_double2(0.5 * (sr + tr), 0.5 * (si + ti)));
    }
}

// spec: [ng][M/2+1][M][M] complex -> R: [ng][M][M][M] real (unnormalised inverse).
__global__ void __launch_bounds__(ZT_LINES * 16) k_zfft_c2r(int M, int lNh, const double2 *__restrict__ spec, double *__restrict__ R,
                                                           const double2 *__restrict__ Wtab)
{
    extern __shared__ __align__(16) unsigned char zt_smem[];
    const int Nh = M >> 1, Zc = Nh + 1, LP = zt_pitch(Nh), nt = blockDim.x, tid = threadIdx.x;
    cplx *L = reinterpret_cast<cplx *>(zt_smem), *WN = L + ZT_LINES * LP, *WP = WN + Nh;
    const int nyb = M / ZT_LINES;
    const int yb = blockIdx.x % nyb, gx = blockIdx.x / nyb;
    const int y0 = yb * ZT_LINES, g = gx / M, x = gx - g * M;
    for (int q = tid; q < Nh; q += nt) { const double2 w = Wtab[2 * q]; WN[q] = { w.x, w.y }; }
    for (int q = tid; q <= Nh; q += nt) { const double2 w = q < M ? Wtab[q] : make_double2(1.0, 0.0); WP[q] = { w.x, -w.y }; }   // w^{-k}
    const double2 *__restrict__ in = spec + (((size_t)g * Zc) * M + x) * M + y0;
    const size_t kstride = (size_t)M * M;
    // X_k of the ZT_LINES lines, k = 0 .. Nh (position Nh sits one past the skewed Nh - 1)
    {   // Zc * ZT_LINES = 16 nt + ZT_LINES values: sixteen batched loads per thread, then the k = Nh row
        double2 v[16];
#pragma unroll
        for (int q = 0; q < 16; ++q) { const int e = tid + q * nt; v[q] = __ldcs(in + (size_t)(e / ZT_LINES) * kstride + (e % ZT_LINES)); }
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            const int e = tid + q * nt, k = e / ZT_LINES, r = e - k * ZT_LINES;
            L[r * LP + xf_sk<4>(k)] = { v[q].x, v[q].y };
        }
        if (tid < ZT_LINES) {
            const double2 w = __ldcs(in + (size_t)Nh * kstride + tid);
            L[tid * LP + xf_sk<4>(Nh - 1) + 1] = { w.x, w.y };
        }
    }
    __syncthreads();
    // split step in place: the pair (k, Nh - k) is read and written by one thread
    for (int e = tid; e < (Nh / 2 + 1) * ZT_LINES; e += nt) {
        const int k = e / ZT_LINES, r = e - k * ZT_LINES, km = Nh - k;
        cplx *ln = L + r * LP;
        const int pk = xf_sk<4>(k), pm = km < Nh ? xf_sk<4>(km) : xf_sk<4>(Nh - 1) + 1;
        const cplx xk = ln[pk], xm = ln[pm];
        auto zfrom = [&](cplx a, cplx b, cplx w) {                // (a + conj b) + i w (a - conj b)
            const double sr = a.x + b.x, si = a.y - b.y, dr = a.x - b.x, di = a.y + b.y;
            return cplx{ sr - (w.x * di + w.y * dr), si + (w.x * dr - w.y * di) };
        };
        const cplx zk = zfrom(xk, xm, WP[k]);
        const cplx zm = zfrom(xm, xk, WP[km]);
        ln[pk] = zk;
        if (km < Nh && km != k) ln[pm] = zm;
    }
    __syncthreads();
    {
        const int tpl = Nh >> 4, line = tid / tpl, jj = tid - line * tpl;
        xf_fft<4, true>(L + line * LP, WN, Nh, lNh, jj);
    }
    __syncthreads();
    double2 *__restrict__ rows = reinterpret_cast<double2 *>(R + ((size_t)gx * M + y0) * M);
    for (int e = tid; e < ZT_LINES * Nh; e += nt) {
        const int r = e >> lNh, n = e & (Nh - 1);
        const cplx v = L[r * LP + xf_sk<4>(n)];
        __stcs(rows + (size_t)r * Nh + n, make_double2(v.x, v.y));
    }
}
