// a3: Gaussian spreading of (F,T,S) onto three M^3 grids (Eq. 42 with the Gaussian derivatives of
// Eq. 48 carried out analytically; P^3 support, Sec. 3.1):
//   H(x_n) = sum_j gamma(d) [ F_j (1 + cF_j (4 al^2 d^2 - 6 al)) - al d x T_j
//                             + 2 al (S_j.d) (1 + cS_j (4 al^2 d^2 - 10 al)) ],   d = x_n - r_j.
//
// Design ("register sweep", se_sweep.cuh; no atomics, every grid point written exactly once, zeros included):
// a thread owns one grid column (y,z) and sweeps along x.  It keeps a window of P partial sums per component
// in registers: window slot s is the plane q = s (mod P).  At plane p it adds, for every particle whose support
// STARTS at plane p and covers the column, that particle's contribution to all P slots (statically indexed; the
// rotation is taken by the address of the doubled x tables), then stores and clears slot p mod P (plane p is
// now final) and moves on -- the window is never shifted.  For a fixed column the summand is
// a cubic in dx = x_n - x_j times the x-Gaussian:
//   H_c = gx(k) [ c0 + dx c1 + dx^2 c2 + dx^3 c3 ]_c      -> 4 FMA per component and grid point,
// with the (y,z) Gaussian folded into the four coefficients and gx dx^n tabulated per particle (a1).  The sweep is cut into segments along x for
// parallelism; a segment starts P-1 planes early to pick up the particles whose support reaches into it.
#pragma once
#include "se_sweep.cuh"

// NC = 3: the three force-density grids; NC = 4: plus the scalar grid of the pressure moments (a9),
// Hs(x_n) = sum_j gamma(d) s_j, one more FMA per grid point.
// The register window is ROTATING: slot s holds the plane q with q = s (mod P); a particle whose support starts at
// plane p (p0 = p mod P) adds its k-th support plane to slot (p0 + k) mod P, i.e. slot s takes entry s + P - p0 of the
// x tables, which the record stores twice (se_common.cuh) -- X points at entry P - p0, the slot index is static.
template <int P, int NC>
__device__ __forceinline__ void spread_hit(const SeConst &c, const double *__restrict__ rec, int xrot, int y, int z, bool active,
                                           double (&acc)[P][NC])
{
    const int M = c.M;
    const int2 yz = *reinterpret_cast<const int2 *>(rec);
    int ry = y - yz.x, rz = z - yz.y;
    ry += ry < 0 ? M : 0;
    rz += rz < 0 ? M : 0;
    if (active && ry < P && rz < P) {
        const double Delta = c.Delta;
        const double dy = rec[REC_D0Y] + ry * Delta, dz = rec[REC_D0Z] + rz * Delta;
        const double g = rec[SE_REC_HDR + ry] * rec[SE_REC_HDR + P + rz];
        const double rho2 = dy * dy + dz * dz;
        const double2 pf = *reinterpret_cast<const double2 *>(rec + REC_POLY), ps = *reinterpret_cast<const double2 *>(rec + REC_POLY + 2);
        // the (y,z) Gaussian folded into the five scalars the coefficients are made of
        const double gfa = g * (pf.x + pf.y * rho2);           // g [(1 - 6 al cF) + 4 al^2 cF rho^2]
        const double gsa = g * (ps.x + ps.y * rho2);           // g [2 al (1 - 10 al cS) + 8 al^3 cS rho^2]
        const double gal = g * c.alpha, gf1 = g * pf.y, gs1 = g * ps.y;
        const double2 m0 = *reinterpret_cast<const double2 *>(rec + REC_F), m1 = *reinterpret_cast<const double2 *>(rec + REC_F + 2),
                      m2 = *reinterpret_cast<const double2 *>(rec + REC_F + 4), m3 = *reinterpret_cast<const double2 *>(rec + REC_F + 6),
                      m4 = *reinterpret_cast<const double2 *>(rec + REC_F + 8), m5 = *reinterpret_cast<const double2 *>(rec + REC_F + 10);
        const double Fx = m0.x, Fy = m0.y, Fz = m1.x, Tx = m1.y, Ty = m2.x, Tz = m2.y;
        const double Sxx = m3.x, Sxy = m3.y, Sxz = m4.x, Syy = m4.y, Syz = m5.x, Szz = m5.y;
        // S.d = S_cx dx + sig_c;  d x T = tau0 + dx tau1 with tau1 = (0, -Tz, Ty)
        const double sg0 = Sxy * dy + Sxz * dz, sg1 = Syy * dy + Syz * dz, sg2 = Syz * dy + Szz * dz;
        const double t00 = dy * Tz - dz * Ty, t01 = dz * Tx, t02 = -dy * Tx;
        double c0[3], c1[3], c2[3], c3[3];
        c0[0] = gfa * Fx - gal * t00 + gsa * sg0;
        c0[1] = gfa * Fy - gal * t01 + gsa * sg1;
        c0[2] = gfa * Fz - gal * t02 + gsa * sg2;
        c1[0] = gsa * Sxx;
        c1[1] = gsa * Sxy + gal * Tz;
        c1[2] = gsa * Sxz - gal * Ty;
        c2[0] = gf1 * Fx + gs1 * sg0;
        c2[1] = gf1 * Fy + gs1 * sg1;
        c2[2] = gf1 * Fz + gs1 * sg2;
        c3[0] = gs1 * Sxx; c3[1] = gs1 * Sxy; c3[2] = gs1 * Sxz;
        const double gsp = NC == 4 ? g * rec[REC_SP] : 0.0;
        // acc[s][a] += sum_n X[s][n] c_n[a]: 3P independent chains of four FMAs
        const double2 *__restrict__ X = reinterpret_cast<const double2 *>(rec + xrot);
#pragma unroll
        for (int s = 0; s < P; ++s) {
            const double2 x01 = X[2 * s], x23 = X[2 * s + 1];
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                double t = acc[s][a];
                t = fma(x01.x, c0[a], t);
                t = fma(x01.y, c1[a], t);
                t = fma(x23.x, c2[a], t);
                acc[s][a] = fma(x23.y, c3[a], t);
            }
            if (NC == 4) acc[s][NC - 1] = fma(x01.x, gsp, acc[s][NC - 1]);
        }
    }
}

// Store window slot p0 (now final: the plane whose index is p0 mod P) if `st`, and clear it for the plane P further on.
template <int P, int NC>
__device__ __forceinline__ void spread_flush(int p0, bool st, size_t idx, size_t G, double *__restrict__ H, double *__restrict__ Hs,
                                             double (&acc)[P][NC])
{
#define SE_SLOT(S)                                                                  \
    case S:                                                                         \
        if (S < P) {                                                                \
            constexpr int s_ = S < P ? S : 0;                                       \
            if (st) {                                                               \
                H[idx] = acc[s_][0]; H[G + idx] = acc[s_][1]; H[2 * G + idx] = acc[s_][2]; \
                if (NC == 4) Hs[idx] = acc[s_][NC - 1];                             \
            }                                                                       \
            _Pragma("unroll") for (int a = 0; a < NC; ++a) acc[s_][a] = 0.0;        \
        }                                                                           \
        break;
    switch (p0) {
        SE_SLOT(0) SE_SLOT(1) SE_SLOT(2) SE_SLOT(3) SE_SLOT(4) SE_SLOT(5) SE_SLOT(6) SE_SLOT(7)
        SE_SLOT(8) SE_SLOT(9) SE_SLOT(10) SE_SLOT(11) SE_SLOT(12) SE_SLOT(13) SE_SLOT(14) SE_SLOT(15)
        SE_SLOT(16) SE_SLOT(17) SE_SLOT(18) SE_SLOT(19) SE_SLOT(20) SE_SLOT(21) SE_SLOT(22) SE_SLOT(23)
    }
#undef SE_SLOT
}

template <int P, int NC>
__global__ void __launch_bounds__(SWEEP_WARPS * 32, NC == 3 ? SWEEP_MIN_BLOCKS : 2) k_spread(SeConst c, const double *__restrict__ recs,
                                                              const int *__restrict__ start_s, double *__restrict__ H,
                                                              double *__restrict__ Hs)
{
    extern __shared__ __align__(32) unsigned char sweep_smem[];
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
    constexpr int XOFF = (SE_REC_HDR + 2 * P + 3) & ~3;
    int p = seg_start - (P - 1);
    int p0 = (p % P + P) % P;                            // window slot of plane p
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
            const int xrot = XOFF + 4 * (P - p0);
            for (int ci = 0; ci < ns; ++ci) spread_hit<P, NC>(c, sl + (size_t)ci * stride, xrot, y, z, active, acc);
            for (int ci = SWEEP_CAP; ci < cur.n; ++ci) {
                const int j = sweep_overflow_index(cur, ci);
                spread_hit<P, NC>(c, recs + (size_t)j * stride, xrot, y, z, active, acc);
            }
            __syncwarp();                           // slot fully read before it is refilled
        }
        // plane p is final: no later particle of this sweep reaches it
        spread_flush<P, NC>(p0, p >= seg_start && active, ((size_t)max(p, 0) * M + y) * M + z, G, H, Hs, acc);
        p0 = p0 + 1 == P ? 0 : p0 + 1;
        cur = nxt;
    }
}

static inline size_t sweep_smem_bytes(int rec_stride)
{
    return (size_t)SWEEP_WARPS * 2 * SWEEP_CAP * rec_stride * 8 + SWEEP_WARPS * 16;
}
