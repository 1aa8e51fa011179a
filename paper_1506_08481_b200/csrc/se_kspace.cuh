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
// T2 = double2, or float2 for the single-precision mesh (SE_OPT_GRID_FP32): the spectra are then stored in fp32, the
// factors are still formed in fp64.
template <typename T2> __device__ __forceinline__ double2 ks_load(const T2 *p, size_t i) { const T2 v = p[i]; return make_double2((double)v.x, (double)v.y); }
template <typename T2> __device__ __forceinline__ void ks_store(T2 *p, size_t i, double2 v);
template <> __device__ __forceinline__ void ks_store<double2>(double2 *p, size_t i, double2 v) { p[i] = v; }
template <> __device__ __forceinline__ void ks_store<float2>(float2 *p, size_t i, double2 v) { p[i] = make_float2((float)v.x, (float)v.y); }

template <typename T2>
__global__ void __launch_bounds__(KSPACE_THREADS) k_kspace(SeConst c, const T2 *__restrict__ Hk, T2 *__restrict__ Gk,
                                                           const T2 *__restrict__ Hsk, T2 *__restrict__ Pk)
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
        const double2 h0 = ks_load(Hk, q), h1 = ks_load(Hk, Gc + q), h2 = ks_load(Hk, 2 * Gc + q);
        const double pr = (kx * h0.x + ky * h1.x + kz * h2.x) / k2, pi = (kx * h0.y + ky * h1.y + kz * h2.y) / k2;
        u0 = make_double2(sc * (h0.x - kx * pr), sc * (h0.y - kx * pi));
        u1 = make_double2(sc * (h1.x - ky * pr), sc * (h1.y - ky * pi));
        u2 = make_double2(sc * (h2.x - kz * pr), sc * (h2.y - kz * pi));
        if (Hsk) {                                   // -i (x + i y) = y - i x
            const double2 hs = ks_load(Hsk, q);
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
    ks_store(Gk, q, u0); ks_store(Gk, Gc + q, u1); ks_store(Gk, 2 * Gc + q, u2);
    ks_store(Gk, 3 * Gc + q, w0); ks_store(Gk, 4 * Gc + q, w1); ks_store(Gk, 5 * Gc + q, w2);
    if (Pk) ks_store(Pk, q, pk);
}

// Single-precision mesh: H (fp64, plain [n][M][M][M]) -> fp32 copy for the transforms.
__global__ void k_grid_to_f32(const double *__restrict__ src, float *__restrict__ dst, size_t n)
{
    const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q < n) dst[q] = (float)src[q];
}

// Single-precision mesh: returned fp32 grids (plain [n][M][M][M]) -> the padded fp64 planes [MYp][MZp] the gather reads,
// periodic halo included (rows M .. M+halo-1 and columns M .. M+halo repeat the first ones, as k_halo_fill writes them).
__global__ void k_grid_from_f32(const float *__restrict__ src, double *__restrict__ Rg, int M, int MYp, int MZp, int halo, size_t nplanes)
{
    const size_t per = (size_t)MYp * MZp;
    const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= nplanes * per) return;
    const size_t pl = q / per;
    const int r = (int)(q - pl * per), y = r / MZp, z = r - y * MZp;
    if (y >= M + halo || z >= M + halo + 1) return;
    Rg[q] = (double)src[(pl * M + (size_t)(y % M)) * M + (z % M)];
}

// Wave-space size variant (Eq. 49-52; SE_OPT_SIZE_VARIANT = 2): only the Gaussian itself is spread and
// gathered, every derivative of the Faxen laws and of the multipole expansion is a wave-vector factor here.  In place on 24
// half spectra of the cuFFT layout:
//   in : 0-2 F, 3-5 a^2 F, 6-8 T, 9-14 S (xx,xy,xz,yy,yz,zz), 15-20 a^2 S                      (Eq. 49)
//        Heff = (F - (k^2/6) a^2F) + (i/2) k x T - i (S - (k^2/10) a^2S).k                      (bracket of Eq. 50)
//        u_k as in k_kspace from Heff
//   out: 0-2 u, 3-5 w = -k^2 u (Eq. 51), 6-8 om = (i/2) k x u, 9-14 e0[ab] = (i/2)(k_a u_b + k_b u_a), 15-20 e2 = -k^2 e0, 21-23 zero.
// The signs of the odd factors are those of cuFFT's e^{-ik.x} forward transform (see k_kspace): the conjugates of the oracle's.
__global__ void __launch_bounds__(KSPACE_THREADS) k_kspace_wave(SeConst c, double2 *__restrict__ Wk, const double2 *__restrict__ Hsk,
                                                                double2 *__restrict__ Pk)
{
    const int M = c.M, Zc = M / 2 + 1;
    const size_t Gc = (size_t)M * M * Zc;
    const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= Gc) return;
    int ix, iy, iz;
    { iz = (int)(q % Zc); const size_t t = q / Zc; iy = (int)(t % M); ix = (int)(t / M); }
    const int jx = ix < M / 2 ? ix : ix - M, jy = iy < M / 2 ? iy : iy - M, jz = iz;
    const double2 z0 = make_double2(0.0, 0.0);
    double2 out[21], pk = z0;
#pragma unroll
    for (int g = 0; g < 21; ++g) out[g] = z0;
    const bool zero = (ix == 0 && iy == 0 && iz == 0) || ix == M / 2 || iy == M / 2 || iz == M / 2;
    if (!zero) {
        // sheared lattice: k = (2 pi/L)(jx, jy - gamma jx, jz) in every factor; deconvolution in the fractional wave number (k_kspace)
        const double k[3] = { c.twopiL * jx, c.twopiL * ((double)jy - c.gamma * (double)jx), c.twopiL * jz };
        const double k2 = k[0] * k[0] + k[1] * k[1] + k[2] * k[2];
        const double kq2 = c.twopiL * c.twopiL * ((double)jx * jx + (double)jy * jy + (double)jz * jz);
        const double dec = c.gamma == 0.0 ? exp(-c.dec * k2) : exp(-k2 * c.inv4xi2 + c.eta_se * kq2 * c.inv4xi2);
        const double sc = c.scale0 * (1.0 + k2 * c.inv4xi2) * dec / k2;
        const int PA[6] = { 0, 0, 0, 1, 1, 2 }, PB[6] = { 0, 1, 2, 1, 2, 2 };
        double2 h[3], Tk[3], Sk[3][3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const double2 f = Wk[a * Gc + q], f2 = Wk[(3 + a) * Gc + q];
            h[a] = make_double2(f.x - (k2 / 6.0) * f2.x, f.y - (k2 / 6.0) * f2.y);
            Tk[a] = Wk[(6 + a) * Gc + q];
        }
#pragma unroll
        for (int e = 0; e < 6; ++e) {
            const double2 s1 = Wk[(9 + e) * Gc + q], s2 = Wk[(15 + e) * Gc + q];
            const double2 v = make_double2(s1.x - (k2 / 10.0) * s2.x, s1.y - (k2 / 10.0) * s2.y);
            Sk[PA[e]][PB[e]] = v; Sk[PB[e]][PA[e]] = v;
        }
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const int b = (a + 1) % 3, d = (a + 2) % 3;
            const double2 kxT = make_double2(k[b] * Tk[d].x - k[d] * Tk[b].x, k[b] * Tk[d].y - k[d] * Tk[b].y);
            const double2 Sdk = make_double2(Sk[a][0].x * k[0] + Sk[a][1].x * k[1] + Sk[a][2].x * k[2],
                                             Sk[a][0].y * k[0] + Sk[a][1].y * k[1] + Sk[a][2].y * k[2]);
            // (i/2) z = (-z.y, z.x)/2;  -i z = (z.y, -z.x)
            h[a].x += -0.5 * kxT.y + Sdk.y;
            h[a].y += 0.5 * kxT.x - Sdk.x;
        }
        const double pr = (k[0] * h[0].x + k[1] * h[1].x + k[2] * h[2].x) / k2, pi = (k[0] * h[0].y + k[1] * h[1].y + k[2] * h[2].y) / k2;
        double2 u[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) u[a] = make_double2(sc * (h[a].x - k[a] * pr), sc * (h[a].y - k[a] * pi));
        if (Hsk) {
            const double2 hs = Hsk[q];
            const double cs = 0.25 * c.scale0 * dec / k2;
#pragma unroll
            for (int a = 0; a < 3; ++a) { u[a].x += cs * k[a] * hs.y; u[a].y -= cs * k[a] * hs.x; }
        }
        if (Pk) {
            const double cp = c.scale0 * c.eta0 * dec;
            pk = make_double2(cp * pi, -cp * pr);
        }
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const int b = (a + 1) % 3, d = (a + 2) % 3;
            out[a] = u[a];
            out[3 + a] = make_double2(-k2 * u[a].x, -k2 * u[a].y);
            const double2 kxu = make_double2(k[b] * u[d].x - k[d] * u[b].x, k[b] * u[d].y - k[d] * u[b].y);
            out[6 + a] = make_double2(-0.5 * kxu.y, 0.5 * kxu.x);
        }
#pragma unroll
        for (int e = 0; e < 6; ++e) {
            const int a = PA[e], b = PB[e];
            const double2 t = make_double2(k[a] * u[b].x + k[b] * u[a].x, k[a] * u[b].y + k[b] * u[a].y);
            out[9 + e] = make_double2(-0.5 * t.y, 0.5 * t.x);
            out[15 + e] = make_double2(-k2 * out[9 + e].x, -k2 * out[9 + e].y);
        }
    }
#pragma unroll
    for (int g = 0; g < 21; ++g) Wk[g * Gc + q] = out[g];
    Wk[21 * Gc + q] = z0; Wk[22 * Gc + q] = z0; Wk[23 * Gc + q] = z0;
    if (Pk) Pk[q] = pk;
}

// Spreading records of one pass of the wave-space variant: a copy of the particle's record with the size polynomials of
// the plain Gaussian (f0 = 1, f1 = s0 = s1 = 0), no torque and stresslet, and in the force slots the three values the
// pass spreads: 0 F, 1 a^2 F, 2 T, 3 (Sxx,Sxy,Sxz), 4 (Syy,Syz,Szz), 5 and 6 the same two rows times a^2.
__global__ void k_plain_recs(SeConst c, const double *__restrict__ recs, double *__restrict__ wrecs, int pass)
{
    const int i = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (i >= c.N) return;
    const double *__restrict__ r = recs + (size_t)i * c.rec_stride;
    double *__restrict__ w = wrecs + (size_t)i * c.rec_stride;
    for (int k = lane; k < c.rec_stride; k += 32) {
        double v = r[k];
        if (k >= REC_POLY && k < REC_SP) {
            v = 0.0;
            if (k == REC_POLY) v = 1.0;
            if (k >= REC_F && k < REC_F + 3) {
                const int a = k - REC_F;
                const double a2F = 6.0 * r[REC_CF], a2S = 10.0 * r[REC_CS];
                switch (pass) {
                case 0: v = r[REC_F + a]; break;
                case 1: v = a2F * r[REC_F + a]; break;
                case 2: v = r[REC_T + a]; break;
                case 3: v = r[REC_S + a]; break;
                case 4: v = r[REC_S + 3 + a]; break;
                case 5: v = a2S * r[REC_S + a]; break;
                default: v = a2S * r[REC_S + 3 + a]; break;
                }
            }
        }
        w[k] = v;
    }
}
