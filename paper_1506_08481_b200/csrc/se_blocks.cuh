// f4: self-image Ewald blocks (Sec. 4.2: "the mobility tensor is approximated by its block-diagonal
// components using direct Ewald summation, i.e., for each particle, the approximation only considers the interactions
// with its periodic images"): for every particle the 11 x 11 matrix that maps its own (F,T,S) to its own (U,Omega,E)
// when only the particle and its periodic images are present,
//     B_i = one-body terms (Eq. 13-15)  -  wave-space self terms (Eq. 37)
//           + sum_{n != 0} real-space Ewald block(R_n; a_i, a_i)  +  (1/eta0 V) sum_{k != 0} wave-space block(k; a_i, a_i),
// by DIRECT Ewald sums (no grid).  Everything but the one-body terms is, entry by entry, a polynomial of degree two in
// t = a_i^2: the size operators enter as (1 + c_i lap)(1 + c_j lap) with c proportional to a^2 (Eq. 13-17), i.e. the
// radial functions are Psi = Phi + (c_i+c_j) B + c_i c_j C in real space and the factors (1 - c_i k^2)(1 - c_j k^2) in wave
// space.  So the lattice sums are done for THREE reference radii only (k_block_lattice, 33 CTAs), and a second kernel
// evaluates, per particle, the Lagrange interpolant through them -- exact up to round-off -- and adds the one-body and self
// terms (k_block_eval): O(N), as the paper asks of the preconditioner.  The sums use their own splitting parameter
// xi_b = sqrt(pi)/L (the result does not depend on it), images |n_d| <= 4 and wave vectors |j_d| <= 7: truncation < 1e-20.
//
// Wave-space block for a single particle (all phases e^{ik.(r_i - r_j)} = 1), with f = 1 - cF k^2, s = 1 - cS k^2,
// G = (1 + k^2/4xi^2) e^{-k^2/4xi^2} / (eta0 V k^2), P = I - khat khat, and grad -> -ik acting on e^{-ik.x}:
//     source  Fcal = f F + (i/2) T x k + i s S.k                                                   [from Eq. 17]
//     U = f G P.Re(Fcal),   w = G P.Im(Fcal),   Omega = (1/2) k x w,   E = (s/2)(k w + w k)          [Eq. 13-15]
// (the other combinations are purely imaginary and cancel between k and -k).
#pragma once
#include "se_real.cuh"

#define BLK_THREADS 256
#define BLK_NIMG 4
#define BLK_KMAX 7

// W[ref][row][col], ref < 3, row, col < 11: real-space image sum + wave-space sum of the self pair at radius sqrt(tref[ref]).
__global__ void __launch_bounds__(BLK_THREADS) k_block_lattice(SeConst cb, double t0, double t1, double t2, double *__restrict__ W)
{
    __shared__ double red[BLK_THREADS / 32][11];
    const int col = blockIdx.x, ref = blockIdx.y, tid = threadIdx.x;
    const double t = ref == 0 ? t0 : (ref == 1 ? t1 : t2), a = sqrt(t);
    const double cF = t * (1.0 / 6.0), cS = t * 0.1;
    double mj[12];
#pragma unroll
    for (int q = 0; q < 12; ++q) mj[q] = q == col ? 1.0 : 0.0;
    double acc[12], accw[11];
#pragma unroll
    for (int q = 0; q < 12; ++q) acc[q] = 0.0;
#pragma unroll
    for (int q = 0; q < 11; ++q) accw[q] = 0.0;
    // real-space images R_n = L n, n != 0: separation x = r_i - r_j - R_n = -R_n
    // sheared lattice: R_n = L (n0 + gamma n1, n1, n2); the x range is widened so that the cube still holds the cutoff sphere
    constexpr int NI = 2 * BLK_NIMG + 1;
    const int wx = (int)ceil(fabs(cb.gamma) * BLK_NIMG), NX = NI + 2 * wx;
    for (int q = tid; q < NX * NI * NI; q += BLK_THREADS) {
        const int nx = q / (NI * NI) - BLK_NIMG - wx, ny = (q / NI) % NI - BLK_NIMG, nz = q % NI - BLK_NIMG;
        if (nx == 0 && ny == 0 && nz == 0) continue;
        const double x = -cb.L * (nx + cb.gamma * ny), y = -cb.L * ny, z = -cb.L * nz;
        pair_real<false>(cb, x, y, z, x * x + y * y + z * z, cF, cS, a, mj, acc);
    }
    // wave vectors k = (2 pi / L) j, j != 0
    const double Fx = mj[0], Fy = mj[1], Fz = mj[2], Tx = mj[3], Ty = mj[4], Tz = mj[5];
    const double Sxx = mj[6], Sxy = mj[7], Sxz = mj[8], Syy = mj[9], Syz = mj[10], Szz = -(Sxx + Syy);
    const double V = cb.L * cb.L * cb.L;
    // k = (2 pi/L)(j0, j1 - gamma j0, j2); the j1 range is widened likewise
    constexpr int NK = 2 * BLK_KMAX + 1;
    const int wy = (int)ceil(fabs(cb.gamma) * BLK_KMAX), NY = NK + 2 * wy;
    for (int q = tid; q < NK * NY * NK; q += BLK_THREADS) {
        const int jx = q / (NY * NK) - BLK_KMAX, jy = (q / NK) % NY - BLK_KMAX - wy, jz = q % NK - BLK_KMAX;
        if (jx == 0 && jy == 0 && jz == 0) continue;
        const double kx = cb.twopiL * jx, ky = cb.twopiL * (jy - cb.gamma * jx), kz = cb.twopiL * jz;
        const double k2 = kx * kx + ky * ky + kz * kz, e = k2 * cb.inv4xi2;
        const double G = (1.0 + e) * exp(-e) / (cb.eta0 * V * k2);
        const double f = 1.0 - cF * k2, s = 1.0 - cS * k2;
        // U from the real part of the source
        const double kF = (kx * Fx + ky * Fy + kz * Fz) / k2, fG = f * f * G;
        accw[0] += fG * (Fx - kx * kF); accw[1] += fG * (Fy - ky * kF); accw[2] += fG * (Fz - kz * kF);
        // imaginary part of the source: (1/2) T x k + s S.k, projected
        double ix = 0.5 * (Ty * kz - Tz * ky) + s * (Sxx * kx + Sxy * ky + Sxz * kz);
        double iy = 0.5 * (Tz * kx - Tx * kz) + s * (Sxy * kx + Syy * ky + Syz * kz);
        double iz = 0.5 * (Tx * ky - Ty * kx) + s * (Sxz * kx + Syz * ky + Szz * kz);
        const double kI = (kx * ix + ky * iy + kz * iz) / k2;
        const double wx = G * (ix - kx * kI), wy = G * (iy - ky * kI), wz = G * (iz - kz * kI);
        accw[3] += 0.5 * (ky * wz - kz * wy); accw[4] += 0.5 * (kz * wx - kx * wz); accw[5] += 0.5 * (kx * wy - ky * wx);
        const double hs = 0.5 * s;
        accw[6] += hs * 2.0 * kx * wx;
        accw[7] += hs * (kx * wy + wx * ky);
        accw[8] += hs * (kx * wz + wx * kz);
        accw[9] += hs * 2.0 * ky * wy;
        accw[10] += hs * (ky * wz + wy * kz);
    }
    const int lane = tid & 31, w = tid >> 5;
#pragma unroll
    for (int r = 0; r < 11; ++r) {
        double v = cb.k0 * acc[r] + accw[r];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) red[w][r] = v;
    }
    __syncthreads();
    if (tid < 11) {
        double v = 0.0;
        for (int q = 0; q < BLK_THREADS / 32; ++q) v += red[q][tid];
        W[(ref * 11 + tid) * 11 + col] = v;
    }
}

// out[i][row][col] = sum_m l_m(a_i^2) W[m][row][col]  (+ one-body - self on the diagonal); l_m: Lagrange basis on t0, t1, t2.
__global__ void k_block_eval(SeConst cb, double t0, double t1, double t2, const double *__restrict__ W, const double *__restrict__ radii,
                             double *__restrict__ out)
{
    const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= (size_t)cb.N * 121) return;
    const size_t i = q / 121;
    const int e = (int)(q - i * 121), row = e / 11, col = e - row * 11;
    const double a = radii[i], t = a * a;
    const double l0 = (t - t1) * (t - t2) / ((t0 - t1) * (t0 - t2));
    const double l1 = (t - t0) * (t - t2) / ((t1 - t0) * (t1 - t2));
    const double l2 = (t - t0) * (t - t1) / ((t2 - t0) * (t2 - t1));
    double v = l0 * W[e] + l1 * W[121 + e] + l2 * W[242 + e];
    if (row == col) {
        const double PI = 3.14159265358979323846, p32 = PI * sqrt(PI);
        const double a3 = a * t, ax2 = t * cb.xi * cb.xi, xi3 = cb.xi * cb.xi * cb.xi;
        if (row < 3) v += 1.0 / (6.0 * PI * cb.eta0 * a) - cb.xi * (9.0 - 10.0 * ax2 + 7.0 * ax2 * ax2) / (18.0 * p32 * cb.eta0);
        else if (row < 6) v += 1.0 / (8.0 * PI * cb.eta0 * a3) - 5.0 * xi3 / (12.0 * p32 * cb.eta0);
        else v += 1.0 / ((20.0 / 3.0) * PI * cb.eta0 * a3) - xi3 * (25.0 - 42.0 * ax2 + 27.0 * ax2 * ax2) / (50.0 * p32 * cb.eta0);
    }
    out[q] = v;
}
