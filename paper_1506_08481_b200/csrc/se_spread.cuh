// a3: Gaussian spreading of (F,T,S) onto three M^3 grids (Eq. 42 with the Gaussian derivatives of
// Eq. 48 carried out analytically; P^3 support, Sec. 3.1):
//   H(x_n) = sum_j gamma(d) [ F_j (1 + cF_j (4 al^2 d^2 - 6 al)) - al d x T_j
//                             + 2 al (S_j.d) (1 + cS_j (4 al^2 d^2 - 10 al)) ],   d = x_n - r_j.
//
// Design ("register sweep", no atomics, every grid point written exactly once, zeros included):
// a thread owns one grid column (y,z) and sweeps along x (the slowest grid axis).  It keeps a window of
// P partial sums per component in registers: window slot k is plane p+k.  At plane p it adds, for every
// particle whose support STARTS at plane p and covers the column, that particle's contribution to all P
// slots (statically indexed), then stores slot 0 (plane p is now final), shifts the window and moves on.
// A warp owns a 4 (y) x 8 (z) patch of columns so that its stores are 64-byte rows; candidates come from
// the plane-thin tile bins (x-plane, y/4, z/8) of the counting sort.  For a fixed column the summand is a
// cubic in dx = x_n - x_j times the x-Gaussian:
//   H_c = gyz gx(k) [ c0 + dx (c1 + dx (c2 + dx c3)) ]_c      -> 4 FMA per component and grid point.
// The sweep is cut into segments along x for parallelism; a segment starts P-1 planes early to pick up the
// particles whose support reaches into it.
#pragma once
#include "se_common.cuh"

#define SPREAD_WARPS 4

template <int P>
__global__ void __launch_bounds__(SPREAD_WARPS * 32) k_spread(SeConst c, const double *__restrict__ recs,
                                                               const int *__restrict__ start_s, double *__restrict__ H)
{
    const int lane = threadIdx.x & 31;
    const int wid = blockIdx.x * SPREAD_WARPS + (threadIdx.x >> 5);
    const int npatch = c.NBY * c.NBZ;
    const int seg = wid / npatch, patch = wid - seg * npatch;
    if (seg >= c.nseg) return;
    const int M = c.M;
    const int py = patch / c.NBZ, pz = patch - py * c.NBZ;
    const int Y0 = py * SE_TILE_Y, Z0 = pz * SE_TILE_Z;
    const int y = Y0 + (lane >> 3), z = Z0 + (lane & 7);
    const bool active = (y < M) && (z < M);

    // bins that can hold particles covering this patch: y0w in [Y0-P+1, Y0+3], z0w in [Z0-P+1, Z0+7] (mod M)
    int by_lo[2], by_hi[2], bz_lo[2], bz_hi[2], nyr, nzr;
    {
        const int ylo = Y0 - (P - 1), yhi = min(Y0 + SE_TILE_Y - 1, M - 1);
        if (yhi - ylo + 1 >= M) { nyr = 1; by_lo[0] = 0; by_hi[0] = c.NBY - 1; }
        else if (ylo < 0) { nyr = 2; by_lo[0] = 0; by_hi[0] = yhi / SE_TILE_Y; by_lo[1] = (ylo + M) / SE_TILE_Y; by_hi[1] = c.NBY - 1;
                            if (by_lo[1] <= by_hi[0]) { nyr = 1; by_hi[0] = c.NBY - 1; } }
        else { nyr = 1; by_lo[0] = ylo / SE_TILE_Y; by_hi[0] = yhi / SE_TILE_Y; }
        const int zlo = Z0 - (P - 1), zhi = min(Z0 + SE_TILE_Z - 1, M - 1);
        if (zhi - zlo + 1 >= M) { nzr = 1; bz_lo[0] = 0; bz_hi[0] = c.NBZ - 1; }
        else if (zlo < 0) { nzr = 2; bz_lo[0] = 0; bz_hi[0] = zhi / SE_TILE_Z; bz_lo[1] = (zlo + M) / SE_TILE_Z; bz_hi[1] = c.NBZ - 1;
                            if (bz_lo[1] <= bz_hi[0]) { nzr = 1; bz_hi[0] = c.NBZ - 1; } }
        else { nzr = 1; bz_lo[0] = zlo / SE_TILE_Z; bz_hi[0] = zhi / SE_TILE_Z; }
    }

    double acc[P][3];
#pragma unroll
    for (int k = 0; k < P; ++k) { acc[k][0] = 0.0; acc[k][1] = 0.0; acc[k][2] = 0.0; }

    const int seg_start = seg * c.seg_len, seg_end = min(seg_start + c.seg_len, M);
    const size_t G = (size_t)M * M * M;
    const double Delta = c.Delta, al = c.alpha;

    for (int p = seg_start - (P - 1); p < seg_end; ++p) {
        const int px = p < 0 ? p + M : p;
        for (int yr = 0; yr < nyr; ++yr)
            for (int by = by_lo[yr]; by <= by_hi[yr]; ++by) {
                const int rowbase = (px * c.NBY + by) * c.NBZ;
                for (int zr = 0; zr < nzr; ++zr) {
                    const int js = start_s[rowbase + bz_lo[zr]], je = start_s[rowbase + bz_hi[zr] + 1];
                    for (int j = js; j < je; ++j) {
                        const double *__restrict__ rec = recs + (size_t)j * c.rec_stride;
                        const int2 yz = *reinterpret_cast<const int2 *>(rec);
                        int ry = y - yz.x, rz = z - yz.y;
                        ry += ry < 0 ? M : 0;
                        rz += rz < 0 ? M : 0;
                        if (active && ry < P && rz < P) {
                            const double dy = rec[REC_D0 + 1] + ry * Delta, dz = rec[REC_D0 + 2] + rz * Delta;
                            const double d0x = rec[REC_D0];
                            const double gyz = rec[SE_REC_HDR + P + ry] * rec[SE_REC_HDR + 2 * P + rz];
                            const double rho2 = dy * dy + dz * dz;
                            const double f1 = rec[REC_POLY + 1], s1 = rec[REC_POLY + 3];
                            const double fa = rec[REC_POLY] + f1 * rho2;          // (1 - 6 al cF) + 4 al^2 cF rho^2
                            const double sa = rec[REC_POLY + 2] + s1 * rho2;      // 2 al (1 - 10 al cS) + 8 al^3 cS rho^2
                            const double Fx = rec[REC_F], Fy = rec[REC_F + 1], Fz = rec[REC_F + 2];
                            const double Tx = rec[REC_T], Ty = rec[REC_T + 1], Tz = rec[REC_T + 2];
                            const double Sxx = rec[REC_S], Sxy = rec[REC_S + 1], Sxz = rec[REC_S + 2];
                            const double Syy = rec[REC_S + 3], Syz = rec[REC_S + 4], Szz = rec[REC_S + 5];
                            // S.d = S_cx dx + sig_c;  d x T = tau0 + dx tau1 with tau1 = (0, -Tz, Ty)
                            const double sg0 = Sxy * dy + Sxz * dz, sg1 = Syy * dy + Syz * dz, sg2 = Syz * dy + Szz * dz;
                            const double t00 = dy * Tz - dz * Ty, t01 = dz * Tx, t02 = -dy * Tx;
                            double c0[3], c1[3], c2[3], c3[3];
                            c0[0] = gyz * (fa * Fx - al * t00 + sa * sg0);
                            c0[1] = gyz * (fa * Fy - al * t01 + sa * sg1);
                            c0[2] = gyz * (fa * Fz - al * t02 + sa * sg2);
                            c1[0] = gyz * (sa * Sxx);
                            c1[1] = gyz * (sa * Sxy + al * Tz);
                            c1[2] = gyz * (sa * Sxz - al * Ty);
                            c2[0] = gyz * (f1 * Fx + s1 * sg0);
                            c2[1] = gyz * (f1 * Fy + s1 * sg1);
                            c2[2] = gyz * (f1 * Fz + s1 * sg2);
                            c3[0] = gyz * s1 * Sxx; c3[1] = gyz * s1 * Sxy; c3[2] = gyz * s1 * Sxz;
#pragma unroll
                            for (int k = 0; k < P; ++k) {
                                const double dx = d0x + k * Delta;
                                const double gx = rec[SE_REC_HDR + k];
#pragma unroll
                                for (int a = 0; a < 3; ++a)
                                    acc[k][a] = fma(gx, fma(dx, fma(dx, fma(dx, c3[a], c2[a]), c1[a]), c0[a]), acc[k][a]);
                            }
                        }
                    }
                }
            }
        if (p >= seg_start && active) {
            const size_t idx = ((size_t)p * M + y) * M + z;
            H[idx] = acc[0][0];
            H[G + idx] = acc[0][1];
            H[2 * G + idx] = acc[0][2];
        }
#pragma unroll
        for (int k = 0; k < P - 1; ++k) { acc[k][0] = acc[k + 1][0]; acc[k][1] = acc[k + 1][1]; acc[k][2] = acc[k + 1][2]; }
        acc[P - 1][0] = 0.0; acc[P - 1][1] = 0.0; acc[P - 1][2] = 0.0;
    }
}
