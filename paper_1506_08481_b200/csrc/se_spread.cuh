// a3: Gaussian spreading of (F,T,S) onto three M^3 grids (Eq. 42 with the Gaussian derivatives of
// Eq. 48 carried out analytically; P^3 support, Sec. 3.1):
//   H(x_n) = sum_j gamma(d) [ F_j (1 + cF_j (4 al^2 d^2 - 6 al)) - al d x T_j
//                             + 2 al (S_j.d) (1 + cS_j (4 al^2 d^2 - 10 al)) ],   d = x_n - r_j.
//
// Design ("register sweep", se_sweep.cuh; no atomics, every grid point written exactly once, zeros included):
// a thread owns one grid column (y,z) and sweeps along x.  It keeps a window of P partial sums per component
// in registers: window slot k is plane p+k.  At plane p it adds, for every particle whose support STARTS at
// plane p and covers the column, that particle's contribution to all P slots (statically indexed), then
// stores slot 0 (plane p is now final), shifts the window and moves on.  For a fixed column the summand is
// a cubic in dx = x_n - x_j times the x-Gaussian:
//   H_c = gx(k) [ c0 + dx c1 + dx^2 c2 + dx^3 c3 ]_c      -> 4 FMA per component and grid point (Horner),
// with the (y,z) Gaussian folded into the four coefficients and gx tabulated per particle (a1).  The sweep is cut into
// segments along x for parallelism; a segment starts P-1 planes early to pick up the particles whose support reaches into it.
#pragma once
#include "se_sweep.cuh"

// NC = 3: the three force-density grids; NC = 4: plus the scalar grid of the pressure moments (a9),
// Hs(x_n) = sum_j gamma(d) s_j, one more FMA per grid point.
// SHEAR: sheared lattice (Eq. 48).  The Gaussian is isotropic in the grid offsets (dx, dy, dz) = fractional
// offsets times L; its physical gradient is -2 al D gam with the metric vector D = (dx, dy - g dx, dz), lap gam =
// (4 al^2 D.D - 2 al (3 + g^2)) gam and grad lap gam carries the extra term 8 al^2 Mt.D, Mt = [[1,-g,0],[-g,1+g^2,0],[0,0,1]]:
//   H = gam { F [f0 + f1 D.D] - al D x T + (S.D) [s0 + s1 D.D] - 8 al^2 cS S.(Mt.D) },   f0, s0 with the trace 3 + g^2 (a1),
// still a cubic in dx for a fixed column: D = D0 + dx D1, D0 = (0, dy, dz), D1 = (1, -g, 0).
template <int P, int NC, bool SHEAR>
__device__ __forceinline__ void spread_hit(const SeConst &c, const double *__restrict__ rec, int y, int z, bool active,
                                           double (&acc)[P][NC])
{
    const int M = c.M;
    const int2 yz = *reinterpret_cast<const int2 *>(rec);
    int ry = y - yz.x, rz = z - yz.y;
    ry += ry < 0 ? M : 0;
    rz += rz < 0 ? M : 0;
    if (active && ry < P && rz < P) {
        const double Delta = c.Delta, al = c.alpha;
        const double dy = rec[REC_D0 + 1] + ry * Delta, dz = rec[REC_D0 + 2] + rz * Delta;
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
        if (SHEAR) {
            const double g = c.gamma, g1 = 1.0 + g * g, kap = 8.0 * al * al * rec[REC_CS];
            const double A1 = -2.0 * g * dy * f1, A2 = g1 * f1, B1 = -2.0 * g * dy * s1, B2 = g1 * s1;
            const double Fv[3] = { Fx, Fy, Fz };
            const double Sx_[3] = { Sxx, Sxy, Sxz }, Sy_[3] = { Sxy, Syy, Syz }, Sz_[3] = { Sxz, Syz, Szz };
            const double t0v[3] = { t00, t01, t02 };                                  // D0 x T
            const double t1v[3] = { -g * Tz, -Tz, Ty + g * Tx };                      // D1 x T
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const double sg = Sy_[a] * dy + Sz_[a] * dz;                          // (S.D0)_a
                const double sd = Sx_[a] - g * Sy_[a];                                // (S.D1)_a
                const double m0 = -g * dy * Sx_[a] + g1 * dy * Sy_[a] + dz * Sz_[a];  // (S.Mt.D0)_a
                const double m1 = g1 * Sx_[a] - g * (2.0 + g * g) * Sy_[a];           // (S.Mt.D1)_a
                c0[a] = gyz * (fa * Fv[a] - al * t0v[a] + sa * sg - kap * m0);
                c1[a] = gyz * (A1 * Fv[a] - al * t1v[a] + B1 * sg + sa * sd - kap * m1);
                c2[a] = gyz * (A2 * Fv[a] + B2 * sg + B1 * sd);
                c3[a] = gyz * (B2 * sd);
            }
        }
        // acc[k][a] += gx(k) ((c3 dx + c2) dx + c1) dx + c0)[a], dx = d0x + k Delta: 3P independent chains of four FMAs,
        // one table value per plane
        const double *__restrict__ X0 = rec + SE_REC_HDR;
        const double d0x = rec[REC_D0];
        const double gsp = NC == 4 ? gyz * rec[REC_SP] : 0.0;
#pragma unroll
        for (int k = 0; k < P; ++k) {
            const double gx = X0[k], dx = fma((double)k, Delta, d0x);
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                double t = fma(c3[a], dx, c2[a]);
                t = fma(t, dx, c1[a]);
                t = fma(t, dx, c0[a]);
                acc[k][a] = fma(gx, t, acc[k][a]);
            }
            if (NC == 4) acc[k][NC - 1] = fma(gx, gsp, acc[k][NC - 1]);
        }
    }
}

template <int P, int NC, bool SHEAR>
__global__ void __launch_bounds__(SWEEP_WARPS * 32, (NC == 3 && !SHEAR) ? SWEEP_MIN_BLOCKS : 2) k_spread(SeConst c, const double *__restrict__ recs,
                                                              const int *__restrict__ start_s, double *__restrict__ H,
                                                              double *__restrict__ Hs)
{
    extern __shared__ __align__(16) unsigned char sweep_smem[];
    const int lane = threadIdx.x & 31, wl = threadIdx.x >> 5;
    const int wid = blockIdx.x * SWEEP_WARPS + wl;
    const int npatch = c.NBY * c.NBZ;
    const int seg = wid / npatch, patch = wid - seg * npatch;
    if (seg >= c.nseg) return;
    const int M = c.M, stride = c.rec_stride;
    const int py = patch / c.NBZ, pz = patch - py * c.NBZ;
    const int Y0 = py * SE_TILE_Y, Z0 = pz * SE_TILE_Z;
    const int y = Y0 + (lane >> 3), z = Z0 + (lane & 7);
    const bool active = (y < M) && (z < M);

    double *slot0 = reinterpret_cast<double *>(sweep_smem) + (size_t)wl * 2 * SWEEP_CAP * stride;
    double *slot1 = slot0 + (size_t)SWEEP_CAP * stride;
    const uint32_t bar0 = smem_u32(sweep_smem + (size_t)SWEEP_WARPS * 2 * SWEEP_CAP * stride * 8 + wl * 16), bar1 = bar0 + 8;
    if (lane == 0) {
        mbar_init(bar0, 1);
        mbar_init(bar1, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();

    const SweepRanges rg = sweep_ranges<P>(c, Y0, Z0, lane);

    double acc[P][NC];
#pragma unroll
    for (int k = 0; k < P; ++k)
#pragma unroll
        for (int a = 0; a < NC; ++a) acc[k][a] = 0.0;

    const int seg_start = seg * c.seg_len, seg_end = min(seg_start + c.seg_len, M);
    const size_t G = (size_t)M * M * M;
    int p = seg_start - (P - 1);
    auto binbase = [&](int q) { return (q < 0 ? q + M : q) * npatch; };
    SweepList cur = sweep_scan(sweep_load(rg, start_s, binbase(p), lane), lane);
    sweep_stage(cur, recs, stride, smem_u32(slot0), bar0, lane);
    int2 raw = sweep_load(rg, start_s, binbase(min(p + 1, seg_end - 1)), lane);     // ranges of plane p+1
    unsigned parity = 0;
    for (int buf = 0; p < seg_end; ++p, buf ^= 1) {
        SweepList nxt;
        nxt.js = 0; nxt.cnt = 0; nxt.off = 0; nxt.n = 0;
        if (p + 1 < seg_end) {
            nxt = sweep_scan(raw, lane);
            sweep_stage(nxt, recs, stride, smem_u32(buf ? slot0 : slot1), buf ? bar0 : bar1, lane);
            raw = sweep_load(rg, start_s, binbase(min(p + 2, seg_end - 1)), lane);   // used one iteration later
        }
        if (cur.n > 0) {
            mbar_wait(buf ? bar1 : bar0, (parity >> buf) & 1u);
            parity ^= 1u << buf;
            const double *__restrict__ sl = buf ? slot1 : slot0;
            const int ns = min(cur.n, SWEEP_CAP);
            for (int ci = 0; ci < ns; ++ci) spread_hit<P, NC, SHEAR>(c, sl + (size_t)ci * stride, y, z, active, acc);
            for (int ci = SWEEP_CAP; ci < cur.n; ++ci) {
                const int j = sweep_overflow_index(cur, ci);
                spread_hit<P, NC, SHEAR>(c, recs + (size_t)j * stride, y, z, active, acc);
            }
            __syncwarp();                           // slot fully read before it is refilled
        }
        if (p >= seg_start && active) {
            const size_t idx = ((size_t)p * M + y) * M + z;
            H[idx] = acc[0][0];
            H[G + idx] = acc[0][1];
            H[2 * G + idx] = acc[0][2];
            if (NC == 4) Hs[idx] = acc[0][NC - 1];
        }
#pragma unroll
        for (int k = 0; k < P - 1; ++k)
#pragma unroll
            for (int a = 0; a < NC; ++a) acc[k][a] = acc[k + 1][a];
#pragma unroll
        for (int a = 0; a < NC; ++a) acc[P - 1][a] = 0.0;
        cur = nxt;
    }
}

static inline size_t sweep_smem_bytes(int rec_stride)
{
    return (size_t)SWEEP_WARPS * 2 * SWEEP_CAP * rec_stride * 8 + SWEEP_WARPS * 16;
}
