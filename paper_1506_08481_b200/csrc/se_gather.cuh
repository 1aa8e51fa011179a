// a7: Gaussian gather (Eq. 45 / Eq. 52 by the trapezoidal rule, L280) and a8: epilogue.
//   U_i  = D^3 sum_n gamma(d) (u~ + cF_i w~)
//   Om_i = D^3 sum_n al gamma(d) d x u~
//   E_i  = traceless part of D^3 sum_n al gamma(d) (d q + q d),  q = u~ + cS_i w~,   d = x_n - r_i
// over the same P^3 support as the spreading.  One warp per particle (tile order, so that neighbouring
// warps read overlapping footprints from L1/L2); a lane takes (y,z) columns of the footprint and reduces
// along x first: per grid g it needs only  m0 = sum_k gx(k) g  and  m1 = sum_k gx(k) dx_k g.
#pragma once
#include "se_common.cuh"

#define GATHER_WARPS 4

template <int P>
__global__ void __launch_bounds__(GATHER_WARPS * 32) k_gather(SeConst c, const double *__restrict__ recs,
                                                               const double *__restrict__ Gr, double *__restrict__ out_wave)
{
    const int lane = threadIdx.x & 31;
    const int slot = blockIdx.x * GATHER_WARPS + (threadIdx.x >> 5);
    if (slot >= c.N) return;
    const double *__restrict__ rec = recs + (size_t)slot * c.rec_stride;
    const int M = c.M;
    const size_t G = (size_t)M * M * M;
    const int2 yz = reinterpret_cast<const int2 *>(rec)[0], xo = reinterpret_cast<const int2 *>(rec)[1];
    const double d0x = rec[REC_D0], d0y = rec[REC_D0 + 1], d0z = rec[REC_D0 + 2];
    const double cF = rec[REC_CF], cS = rec[REC_CS], Delta = c.Delta;

    double aU[3] = { 0, 0, 0 }, aW[3] = { 0, 0, 0 }, aE[6] = { 0, 0, 0, 0, 0, 0 };   // E: xx,xy,xz,yy,yz,zz
    for (int col = lane; col < P * P; col += 32) {
        const int ry = col / P, rz = col - ry * P;
        int yw = yz.x + ry, zw = yz.y + rz;
        yw -= yw >= M ? M : 0;
        zw -= zw >= M ? M : 0;
        const size_t colbase = (size_t)yw * M + zw;
        double m0[6], m1[6];
#pragma unroll
        for (int g = 0; g < 6; ++g) { m0[g] = 0.0; m1[g] = 0.0; }
#pragma unroll 4
        for (int k = 0; k < P; ++k) {
            int xw = xo.x + k;
            xw -= xw >= M ? M : 0;
            const size_t idx = (size_t)xw * M * M + colbase;
            const double gx = rec[SE_REC_HDR + k];
            const double gxd = gx * (d0x + k * Delta);
#pragma unroll
            for (int g = 0; g < 6; ++g) {
                const double v = Gr[g * G + idx];
                m0[g] = fma(gx, v, m0[g]);
                m1[g] = fma(gxd, v, m1[g]);
            }
        }
        const double dy = d0y + ry * Delta, dz = d0z + rz * Delta;
        const double gyz = rec[SE_REC_HDR + P + ry] * rec[SE_REC_HDR + 2 * P + rz];
        const double ga = gyz * c.alpha;
#pragma unroll
        for (int a = 0; a < 3; ++a) aU[a] = fma(gyz, m0[a] + cF * m0[3 + a], aU[a]);
        // d x u~ summed over x: (dy uz - dz uy, dz ux - dx uz, dx uy - dy ux) with dx-moments m1
        aW[0] = fma(ga, dy * m0[2] - dz * m0[1], aW[0]);
        aW[1] = fma(ga, dz * m0[0] - m1[2], aW[1]);
        aW[2] = fma(ga, m1[1] - dy * m0[0], aW[2]);
        double Q0[3], Q1[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) { Q0[a] = m0[a] + cS * m0[3 + a]; Q1[a] = m1[a] + cS * m1[3 + a]; }
        // (d q + q d)_ab summed over x: d_x -> Q1, d_y -> dy Q0, d_z -> dz Q0
        aE[0] = fma(ga, 2.0 * Q1[0], aE[0]);
        aE[1] = fma(ga, Q1[1] + dy * Q0[0], aE[1]);
        aE[2] = fma(ga, Q1[2] + dz * Q0[0], aE[2]);
        aE[3] = fma(ga, 2.0 * dy * Q0[1], aE[3]);
        aE[4] = fma(ga, dy * Q0[2] + dz * Q0[1], aE[4]);
        aE[5] = fma(ga, 2.0 * dz * Q0[2], aE[5]);
    }
    double r[12] = { aU[0], aU[1], aU[2], aW[0], aW[1], aW[2], aE[0], aE[1], aE[2], aE[3], aE[4], aE[5] };
#pragma unroll
    for (int k = 0; k < 12; ++k) {
        double v = r[k];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        r[k] = v;
    }
    if (lane == 0) {
        double *o = out_wave + 11 * (size_t)xo.y;
        const double tr3 = (r[6] + r[9] + r[11]) * (1.0 / 3.0);
        o[0] = c.D3 * r[0]; o[1] = c.D3 * r[1]; o[2] = c.D3 * r[2];
        o[3] = c.D3 * r[3]; o[4] = c.D3 * r[4]; o[5] = c.D3 * r[5];
        o[6] = c.D3 * (r[6] - tr3); o[7] = c.D3 * r[7]; o[8] = c.D3 * r[8];
        o[9] = c.D3 * (r[9] - tr3); o[10] = c.D3 * r[10];
    }
}

// a8: out = real + wave + (one-body - self) * input, in caller order (Eq. 13-15 one-body terms;
// Eq. 37 and its Omega-T / E-S analogues for the wave-space self terms).
__global__ void k_epilogue(SeConst c, unsigned flags, const double *__restrict__ radii,
                           const double *__restrict__ F, const double *__restrict__ T, const double *__restrict__ S,
                           const double *__restrict__ out_real, const double *__restrict__ out_wave,
                           double *__restrict__ U, double *__restrict__ W, double *__restrict__ E)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= c.N) return;
    const double a = radii[i], a3 = a * a * a;
    const double PI = 3.14159265358979323846;
    const double p32 = PI * sqrt(PI);
    const double ax2 = a * a * c.xi * c.xi, xi3 = c.xi * c.xi * c.xi;
    double cU = 0.0, cW = 0.0, cE = 0.0;
    if (!(flags & 0x4u)) {                                   // SE_SKIP_SELF
        cU -= c.xi * (9.0 - 10.0 * ax2 + 7.0 * ax2 * ax2) / (18.0 * p32 * c.eta0);
        cW -= 5.0 * xi3 / (12.0 * p32 * c.eta0);
        cE -= xi3 * (25.0 - 42.0 * ax2 + 27.0 * ax2 * ax2) / (50.0 * p32 * c.eta0);
    }
    if (!(flags & 0x8u)) {                                   // SE_SKIP_ONEBODY
        cU += 1.0 / (6.0 * PI * c.eta0 * a);
        cW += 1.0 / (8.0 * PI * c.eta0 * a3);
        cE += 1.0 / ((20.0 / 3.0) * PI * c.eta0 * a3);
    }
    const bool real = !(flags & 0x1u), wave = !(flags & 0x2u);
    const double *orl = out_real + 11 * (size_t)i, *owv = out_wave + 11 * (size_t)i;
#pragma unroll
    for (int k = 0; k < 11; ++k) {
        double v = 0.0;
        if (real) v += orl[k];
        if (wave) v += owv[k];
        if (k < 3) U[3 * (size_t)i + k] = v + cU * F[3 * (size_t)i + k];
        else if (k < 6) W[3 * (size_t)i + k - 3] = v + cW * T[3 * (size_t)i + k - 3];
        else E[5 * (size_t)i + k - 6] = v + cE * S[5 * (size_t)i + k - 6];
    }
}
