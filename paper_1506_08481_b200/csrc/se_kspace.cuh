// a5: fused k-space pass (Eq. 43 with the kernel g1 of Eq. 36; hybrid variant Eq. 50-51 with the
// bracket replaced by H_k, L326).  One HBM pass: reads the three spectra H_k, writes the six spectra
//   u_k = s(k) (H_k - k (k.H_k)/k^2),   s(k) = [Delta^3/(eta0 V)] (1 + k^2/4xi^2) exp(-(1-eta_se) k^2/4xi^2)/k^2
//   w_k = -k^2 u_k
// (Green's function scale and Gaussian deconvolution e^{+eta_se k^2/4xi^2} folded into one factor);
// zero at k = 0 (Eq. 43) and on the Nyquist planes (reading 13).
// Layout: half spectra [M][M][M/2+1] complex (cuFFT D2Z), last index fastest.
// Compressible extension (a9; Eq. 33-34, 29-31), optional spectra Hs_k (in) and p_k (out).  cuFFT's forward
// transform carries e^{-ik.x} where the paper's (and the oracle's) carries e^{+ik.x}; for real grids that is a
// complex conjugation of everything, so the odd multipliers i k change sign here:
//   u_k += [Delta^3/(4 eta0 V)] (-i k/k^2) e^{-(1-eta_se) k^2/4xi^2} Hs_k     (before w_k = -k^2 u_k is formed)
//   p_k  = [Delta^3/V] (-i k.H_k/k^2) e^{-(1-eta_se) k^2/4xi^2}
#pragma once
#include "se_common.cuh"

#define KSPACE_THREADS 256

// Used on the cuFFT 3-D path only (grids that are not powers of two, or flag SE_CUFFT3D); power-of-two grids run k_xmid
// (se_xyfft.cuh), which fuses this arithmetic with the x transforms.
__global__ void __launch_bounds__(KSPACE_THREADS) k_kspace(SeConst c, const double2 *__restrict__ Hk, double2 *__restrict__ Gk,
                                                           const double2 *__restrict__ Hsk, double2 *__restrict__ Pk)
{
    const int M = c.M, Zc = M / 2 + 1;
    const size_t Gc = (size_t)M * M * Zc;
    const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= Gc) return;
    int ix, iy, iz;
    { iz = (int)(q % Zc); const size_t t = q / Zc; iy = (int)(t % M); ix = (int)(t / M); }
    const int jx = ix < M / 2 ? ix : ix - M, jy = iy < M / 2 ? iy : iy - M, jz = iz;
    double2 u0 = make_double2(0.0, 0.0), u1 = u0, u2 = u0, w0 = u0, w1 = u0, w2 = u0, pk = u0;
    const bool zero = (ix == 0 && iy == 0 && iz == 0) || ix == M / 2 || iy == M / 2 || iz == M / 2;
    if (!zero) {
        // sheared lattice: k = (2 pi/L)(jx, jy - gamma jx, jz); deconvolution in the fractional wave number kq (se_xyfft.cuh)
        const double kx = c.twopiL * jx, ky = c.twopiL * ((double)jy - c.gamma * (double)jx), kz = c.twopiL * jz;
        const double k2 = kx * kx + ky * ky + kz * kz;
        const double kq2 = c.twopiL * c.twopiL * ((double)jx * jx + (double)jy * jy + (double)jz * jz);
        const double dec = c.gamma == 0.0 ? exp(-c.dec * k2) : exp(-k2 * c.inv4xi2 + c.eta_se * kq2 * c.inv4xi2);
        const double sc = c.scale0 * (1.0 + k2 * c.inv4xi2) * dec / k2;
        const double2 h0 = Hk[q], h1 = Hk[Gc + q], h2 = Hk[2 * Gc + q];
        const double pr = (kx * h0.x + ky * h1.x + kz * h2.x) / k2, pi = (kx * h0.y + ky * h1.y + kz * h2.y) / k2;
        u0 = make_double2(sc * (h0.x - kx * pr), sc * (h0.y - kx * pi));
        u1 = make_double2(sc * (h1.x - ky * pr), sc * (h1.y - ky * pi));
        u2 = make_double2(sc * (h2.x - kz * pr), sc * (h2.y - kz * pi));
        if (Hsk) {                                   // -i (x + i y) = y - i x
            const double2 hs = Hsk[q];
            const double cs = 0.25 * c.scale0 * dec / k2;
            u0.x += cs * kx * hs.y; u0.y -= cs * kx * hs.x;
            u1.x += cs * ky * hs.y; u1.y -= cs * ky * hs.x;
            u2.x += cs * kz * hs.y; u2.y -= cs * kz * hs.x;
        }
        if (Pk) {
            const double cp = c.scale0 * c.eta0 * dec;                  // Delta^3/V
            pk = make_double2(cp * pi, -cp * pr);
        }
        w0 = make_double2(-k2 * u0.x, -k2 * u0.y);
        w1 = make_double2(-k2 * u1.x, -k2 * u1.y);
        w2 = make_double2(-k2 * u2.x, -k2 * u2.y);
    }
    Gk[q] = u0; Gk[Gc + q] = u1; Gk[2 * Gc + q] = u2;
    Gk[3 * Gc + q] = w0; Gk[4 * Gc + q] = w1; Gk[5 * Gc + q] = w2;
    if (Pk) Pk[q] = pk;
}
