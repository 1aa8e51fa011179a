// a2: real-space Ewald pair sum, matrix-free (Sec. 3.3; Eq. 22 with Eq. 13-15 and Eq. 17).
//
// Every coupling is a Cartesian derivative of two radial functions built from the Hasimoto screening
// function Phi(r) = r erfc(xi r) - exp(-xi^2 r^2)/(xi sqrt(pi)) (Eq. 22):
//     Psi = Phi + (ci+cj) B + ci cj C,   Lambda = lap Psi = B + (ci+cj) C + ci cj D,
//     B = lap Phi, C = lap^2 Phi, D = lap^3 Phi,   ci, cj in {a^2/6, a^2/10, 0} per coupling.
// Here the derivative tensors are contracted by hand with x, F, T, S (f_n = ((1/r) d/dr)^n f):
//   U  = k0 { (L0-Ps1) F - Ps2 (x.F) x            [UF: (cFi,cFj)]
//            + (1/2) L1 x^T                        [UT: (cFi,0)]
//            - (L1-2Ps2) S.x + Ps3 (x.S.x) x }     [US: (cFi,cSj)]
//   Om = k0 { (1/2) L1 x^F                         [OF: (0,cFj)]
//            + (1/4) [(B1-C0) T + B2 (x.T) x]      [OT]
//            - (1/2) L2 x^(S.x) }                  [OS: (0,cSj)]
//   E  = k0 { x w + w x + a4 S + beta x x + kappa I },  w = a1 F + a2 (x^T) + a3 S.x
//        a1 = L1/2 - Ps2, beta -= Ps3 (x.F), kappa -= Ps2 (x.F)       [EF: (cSi,cFj)]
//        a2 = L2/4                                                     [ET: (cSi,0)]
//        a3 = -(L2/2 - 2 Ps3), a4 = -(L1 - 2 Ps2), beta += Ps4 (x.S.x), kappa += Ps3 (x.S.x)   [ES: (cSi,cSj)]
// with x = r_i - r_j (minimum image), k0 = 1/(8 pi eta0).
//
// Compressible extension (a9; Eq. 24-34), template flag COMP: with chi = erfc(xi r)/r (so that
// chi_n = Phi_{n+1}) and lap chi = 2 xi^2 q g, q_n(c) = chi_n + c (lap chi)_n:
//   U  += -(k0/2) q_1(cFi) s_j x                                   [U <- s, psi_R = -chi/(16 pi eta0)]
//   E  += -(k0/2) s_j [ q_2(cSi) x x + q_1(cSi) I ], trace removed  [E <- s]
//   p   = (1/4pi) [ q_2(cSj) (x.S.x) - q_1(cFj) (x.F) ]            [p <- F, p <- S; Eq. 29-31]
#pragma once
#include "se_common.cuh"

#define REAL_WARPS 4
#define REAL_QCAP 64
#ifndef REAL_MINB1
#define REAL_MINB1 3                // resident CTAs per SM the single right-hand-side kernel is compiled for
#endif

// The radial part of a pair: everything that does not depend on the moments.  Evaluated once per pair and then applied
// to one or several right-hand sides (far_mobility_apply_batch).
template <bool COMP> struct PairS {
    double uf_a, uf_b, ut, us_a, us_b;          // U:  uf_a F + (uf_b x.F + us_b x.S.x) x + ut x^T + us_a S.x
    double of, ot_a, ot_b, os;                  // Om: of x^F + ot_a T + ot_b (x.T) x + os x^(S.x)
    double a1, a2, a3, a4, ef2, ef3, es3, es4;  // E:  w = a1 F + a2 x^T + a3 S.x; beta = es4 xSx - ef3 xF; kappa = es3 xSx - ef2 xF
    double cu, ce1, ce2, ctr, pS, pF;           // a9 (COMP): U <- s, E <- s, p <- S, p <- F
};

template <bool COMP>
__device__ __forceinline__ PairS<COMP> pair_scalars(const SeConst &c, double r2, double cFi, double cSi, double aj)
{
    const double cFj = aj * aj * (1.0 / 6.0), cSj = aj * aj * 0.1;
    const double ir = rsqrt(r2), r = r2 * ir, ir2 = ir * ir;      // one reciprocal square root instead of a root and a division
    const double xr = c.xi * r;
    const double Ec = erfc(xr), qg = c.q * exp(-xr * xr);
    const double ir3 = ir2 * ir, ir4 = ir2 * ir2, ir5 = ir4 * ir, ir6 = ir4 * ir2, ir7 = ir6 * ir, ir8 = ir4 * ir4, ir9 = ir8 * ir;
    // Phi_n = ((1/r) d/dr)^n Phi
    const double P1 = Ec * ir;
    const double P2 = -(Ec * ir3 + qg * ir2);
    const double P3 = 3.0 * Ec * ir5 + qg * (3.0 * ir4 + 2.0 * c.x2 * ir2);
    const double P4 = -(15.0 * Ec * ir7 + qg * (15.0 * ir6 + 10.0 * c.x2 * ir4 + 4.0 * c.x4 * ir2));
    const double P5 = 105.0 * Ec * ir9 + qg * (105.0 * ir8 + 70.0 * c.x2 * ir6 + 28.0 * c.x4 * ir4 + 8.0 * c.x6 * ir2);
    // B_n: B = 2 Phi_1 - q g
    const double B0 = 2.0 * P1 - qg;
    const double B1 = 2.0 * P2 + 2.0 * c.x2 * qg;
    const double B2 = 2.0 * P3 - 4.0 * c.x4 * qg;
    const double B3 = 2.0 * P4 + 8.0 * c.x6 * qg;
    const double B4 = 2.0 * P5 - 16.0 * c.x8 * qg;
    // C_n, D_n: polynomials in s = r^2 times q g
    const double C0 = qg * (10.0 * c.x2 - 4.0 * c.x4 * r2);
    const double C1 = qg * (-28.0 * c.x4 + 8.0 * c.x6 * r2);
    const double C2 = qg * (72.0 * c.x6 - 16.0 * c.x8 * r2);
    const double C3 = qg * (-176.0 * c.x8 + 32.0 * c.x10 * r2);
    const double C4 = qg * (416.0 * c.x10 - 64.0 * c.x12 * r2);
    const double D0 = qg * (-84.0 * c.x4 + (96.0 * c.x6 - 16.0 * c.x8 * r2) * r2);
    const double D1 = qg * (360.0 * c.x6 + (-256.0 * c.x8 + 32.0 * c.x10 * r2) * r2);
    const double D2 = qg * (-1232.0 * c.x8 + (640.0 * c.x10 - 64.0 * c.x12 * r2) * r2);

    PairS<COMP> o;
    double s, p;
    // ---- U ----
    s = cFi + cFj; p = cFi * cFj;
    o.uf_a = (B0 + s * C0 + p * D0) - (P1 + s * B1 + p * C1);
    o.uf_b = -(P2 + s * B2 + p * C2);
    o.ut = 0.5 * (B1 + cFi * C1);
    s = cFi + cSj; p = cFi * cSj;
    const double us_Ps2 = P2 + s * B2 + p * C2;
    o.us_a = -((B1 + s * C1 + p * D1) - 2.0 * us_Ps2);
    o.us_b = P3 + s * B3 + p * C3;
    // ---- Omega ----
    o.of = 0.5 * (B1 + cFj * C1);
    o.ot_a = 0.25 * (B1 - C0);
    o.ot_b = 0.25 * B2;
    o.os = -0.5 * (B2 + cSj * C2);
    // ---- E ----
    s = cSi + cFj; p = cSi * cFj;
    o.ef2 = P2 + s * B2 + p * C2;
    o.ef3 = P3 + s * B3 + p * C3;
    o.a1 = 0.5 * (B1 + s * C1 + p * D1) - o.ef2;
    o.a2 = 0.25 * (B2 + cSi * C2);
    s = cSi + cSj; p = cSi * cSj;
    const double es_Ps2 = P2 + s * B2 + p * C2;
    o.es3 = P3 + s * B3 + p * C3;
    o.es4 = P4 + s * B4 + p * C4;
    o.a3 = -(0.5 * (B2 + s * C2 + p * D2) - 2.0 * o.es3);
    o.a4 = -((B1 + s * C1 + p * D1) - 2.0 * es_Ps2);
    if (COMP) {
        const double L1c = -4.0 * c.x4 * qg, L2c = 8.0 * c.x6 * qg;          // (lap chi)_n, n = 1, 2
        o.cu = -0.5 * (P2 + cFi * L1c);
        o.ce1 = -0.5 * (P2 + cSi * L1c);
        o.ce2 = -0.5 * (P3 + cSi * L2c);
        o.ctr = (3.0 * o.ce1 + o.ce2 * r2) * (1.0 / 3.0);
        o.pS = 0.07957747154594767 * (P3 + cSj * L2c);                       // 1/(4 pi)
        o.pF = 0.07957747154594767 * (P2 + cFj * L1c);
    }
    return o;
}

// acc[0..2] U, [3..5] Omega, [6..10] E (xx,xy,xz,yy,yz), still to be multiplied by k0; acc[11] pressure p (COMP).
template <bool COMP>
__device__ __forceinline__ void pair_apply(const PairS<COMP> &o, double x, double y, double z, double r2,
                                           const double *__restrict__ mj, double acc[12])
{
    const double Fx = mj[0], Fy = mj[1], Fz = mj[2], Tx = mj[3], Ty = mj[4], Tz = mj[5];
    const double Sxx = mj[6], Sxy = mj[7], Sxz = mj[8], Syy = mj[9], Syz = mj[10], Szz = -(Sxx + Syy);
    const double xF = x * Fx + y * Fy + z * Fz, xT = x * Tx + y * Ty + z * Tz;
    const double Sx0 = Sxx * x + Sxy * y + Sxz * z, Sx1 = Sxy * x + Syy * y + Syz * z, Sx2 = Sxz * x + Syz * y + Szz * z;
    const double xSx = x * Sx0 + y * Sx1 + z * Sx2;
    const double cT0 = y * Tz - z * Ty, cT1 = z * Tx - x * Tz, cT2 = x * Ty - y * Tx;       // x ^ T
    const double cF0 = y * Fz - z * Fy, cF1 = z * Fx - x * Fz, cF2 = x * Fy - y * Fx;       // x ^ F
    const double cS0 = y * Sx2 - z * Sx1, cS1 = z * Sx0 - x * Sx2, cS2 = x * Sx1 - y * Sx0; // x ^ (S.x)
    const double ux = o.uf_b * xF + o.us_b * xSx;
    acc[0] += o.uf_a * Fx + ux * x + o.ut * cT0 + o.us_a * Sx0;
    acc[1] += o.uf_a * Fy + ux * y + o.ut * cT1 + o.us_a * Sx1;
    acc[2] += o.uf_a * Fz + ux * z + o.ut * cT2 + o.us_a * Sx2;
    const double otb = o.ot_b * xT;
    acc[3] += o.of * cF0 + o.ot_a * Tx + otb * x + o.os * cS0;
    acc[4] += o.of * cF1 + o.ot_a * Ty + otb * y + o.os * cS1;
    acc[5] += o.of * cF2 + o.ot_a * Tz + otb * z + o.os * cS2;
    const double beta = o.es4 * xSx - o.ef3 * xF;
    const double kappa = o.es3 * xSx - o.ef2 * xF;
    const double w0 = o.a1 * Fx + o.a2 * cT0 + o.a3 * Sx0, w1 = o.a1 * Fy + o.a2 * cT1 + o.a3 * Sx1, w2 = o.a1 * Fz + o.a2 * cT2 + o.a3 * Sx2;
    acc[6] += 2.0 * x * w0 + o.a4 * Sxx + beta * x * x + kappa;
    acc[7] += x * w1 + y * w0 + o.a4 * Sxy + beta * x * y;
    acc[8] += x * w2 + z * w0 + o.a4 * Sxz + beta * x * z;
    acc[9] += 2.0 * y * w1 + o.a4 * Syy + beta * y * y + kappa;
    acc[10] += y * w2 + z * w1 + o.a4 * Syz + beta * y * z;
    if (COMP) {
        const double sj = mj[11];
        const double us = o.cu * sj;
        acc[0] += us * x; acc[1] += us * y; acc[2] += us * z;
        const double e1 = o.ce1 * sj, e2 = o.ce2 * sj, tr3 = o.ctr * sj;
        acc[6] += e2 * x * x + e1 - tr3;
        acc[7] += e2 * x * y;
        acc[8] += e2 * x * z;
        acc[9] += e2 * y * y + e1 - tr3;
        acc[10] += e2 * y * z;
        acc[11] += o.pS * xSx - o.pF * xF;
        (void)r2;
    }
}

template <bool COMP>
__device__ __forceinline__ void pair_real(const SeConst &c, double x, double y, double z, double r2,
                                          double cFi, double cSi, double aj, const double *__restrict__ mj,
                                          double acc[12])
{
    const PairS<COMP> o = pair_scalars<COMP>(c, r2, cFi, cSi, aj);
    pair_apply<COMP>(o, x, y, z, r2, mj, acc);
}

// One CTA per real-space cell (or, when the box holds fewer than 3 cells per axis, per slice of all
// particles).  The positions and radii of the particles of the 27 neighbour cells are staged once in
// shared memory (chunks of REAL_STAGE), then each warp takes target particles of the cell in turn: its lanes
// scan the staged candidates, hits are compacted through a per-warp shared-memory queue so that the expensive
// pair evaluation always runs on full warps, and the 11 sums are reduced over the warp at the end.
// Minimum image as in the oracle, x = d - L rint(d/L), with d/L formed as d * (1/L).
#define REAL_STAGE 1024

// NR right-hand sides at once (far_mobility_apply_batch): moments rs_mom[r][N][12], results out_real[r][N][12],
// r < NR, `rhs_stride` doubles apart; the radial part of a pair is evaluated once and applied NR times.
template <bool COMP, int NR>
__global__ void __launch_bounds__(REAL_WARPS * 32, (NR == 1 ? REAL_MINB1 : (NR == 2 ? 3 : 2))) k_real(SeConst c, const double4 *__restrict__ rs_pos,
                                                          const double *__restrict__ rs_mom, const int *__restrict__ rs_orig,
                                                          const int *__restrict__ start_r, double *__restrict__ out_real,
                                                          size_t rhs_stride)
{
    __shared__ double4 cand[REAL_STAGE];               // (x, y, z, a) of staged candidates
    __shared__ int cand_j[REAL_STAGE];                 // their index in cell order
    __shared__ double4 qd[REAL_WARPS][REAL_QCAP];      // (dx, dy, dz, a_j)
    __shared__ int qj[REAL_WARPS][REAL_QCAP];
    __shared__ int seg_s[27], seg_o[28];               // neighbour cell ranges: first particle, exclusive offsets
    const int wl = threadIdx.x >> 5, lane = threadIdx.x & 31, tid = threadIdx.x;
    const int nc = c.ncr;

    // Work items: the cells (grid-stride loop, so that a small persistent grid can run beside the HBM-bound
    // wave-space kernels without taking their SM resources), or one slice of all particles per CTA.
    const int nitems = nc > 1 ? nc * nc * nc : (int)gridDim.x;
    for (int item = blockIdx.x; item < nitems; item += gridDim.x) {
    __syncthreads();                                   // the previous item's shared tables are no longer read
    // targets of this item and its candidate segments
    int t0, t1, nsegs;
    if (nc > 1) {
        const int cell = item;
        t0 = start_r[cell]; t1 = start_r[cell + 1];
        if (t0 == t1) continue;
        nsegs = 27;
        if (tid < 27) {
            const int cz = cell % nc, cy = (cell / nc) % nc, cx = cell / (nc * nc);
            const int nx = se_mod(cx + tid / 9 - 1, nc), ny = se_mod(cy + (tid / 3) % 3 - 1, nc), nz = se_mod(cz + tid % 3 - 1, nc);
            const int nb = (nx * nc + ny) * nc + nz;
            seg_s[tid] = start_r[nb];
            seg_o[tid + 1] = start_r[nb + 1] - start_r[nb];
        }
    } else {
        const int per = (c.N + gridDim.x - 1) / gridDim.x;
        t0 = item * per; t1 = min(t0 + per, c.N);
        if (t0 >= t1) continue;
        nsegs = 1;
        if (tid == 0) { seg_s[0] = 0; seg_o[1] = c.N; }
    }
    __syncthreads();
    if (tid == 0) {
        int run = 0;
        seg_o[0] = 0;
        for (int k = 0; k < nsegs; ++k) { const int n = seg_o[k + 1]; seg_o[k + 1] = run + n; run += n; }
        // now seg_o[k] = exclusive offset of segment k, seg_o[nsegs] = total
    }
    __syncthreads();
    const int ncand = seg_o[nsegs];
    const int ntgt = t1 - t0;
    const int rounds = (ntgt + REAL_WARPS - 1) / REAL_WARPS;

    for (int base = 0; base < ncand; base += REAL_STAGE) {
        const int nst = min(REAL_STAGE, ncand - base);
        __syncthreads();                               // previous chunk fully consumed
        for (int q = tid; q < nst; q += REAL_WARPS * 32) {
            const int f = base + q;
            int k = 0;
            while (k + 1 < nsegs && seg_o[k + 1] <= f) ++k;
            const int j = seg_s[k] + (f - seg_o[k]);
            cand[q] = rs_pos[j];
            cand_j[q] = j;
        }
        __syncthreads();

        for (int rd = 0; rd < rounds; ++rd) {
            const int i = t0 + rd * REAL_WARPS + wl;
            if (i >= t1) break;
            const double4 pi = rs_pos[i];
            const double cFi = pi.w * pi.w * (1.0 / 6.0), cSi = pi.w * pi.w * 0.1;
            constexpr int NA = COMP ? 12 : 11;
            double acc[NR][12];
#pragma unroll
            for (int r = 0; r < NR; ++r)
#pragma unroll
                for (int k = 0; k < 12; ++k) acc[r][k] = 0.0;
            auto pair = [&](const double4 &d, int jj) {
                const double r2 = d.x * d.x + d.y * d.y + d.z * d.z;
                const PairS<COMP> o = pair_scalars<COMP>(c, r2, cFi, cSi, d.w);
#pragma unroll
                for (int r = 0; r < NR; ++r) pair_apply<COMP>(o, d.x, d.y, d.z, r2, rs_mom + r * rhs_stride + 12 * (size_t)jj, acc[r]);
            };
            int qn = 0;
            for (int qb = 0; qb < nst; qb += 32) {
                const int q = qb + lane;
                bool hit = false;
                double dx = 0, dy = 0, dz = 0, aj = 0;
                int j = -1;
                if (q < nst) {
                    const double4 pj = cand[q];
                    j = cand_j[q];
                    dx = pi.x - pj.x; dy = pi.y - pj.y; dz = pi.z - pj.z;
                    se_min_image(c, dx, dy, dz);
                    const double r2 = dx * dx + dy * dy + dz * dz;
                    hit = (j != i) && (r2 < c.rc2) && (r2 > 0.0);
                    aj = pj.w;
                }
                const unsigned mask = __ballot_sync(0xffffffffu, hit);
                if (hit) {
                    const int slot = qn + __popc(mask & ((1u << lane) - 1u));
                    qd[wl][slot] = make_double4(dx, dy, dz, aj);
                    qj[wl][slot] = j;
                }
                qn += __popc(mask);
                __syncwarp();
                if (qn >= 32) {
                    pair(qd[wl][qn - 32 + lane], qj[wl][qn - 32 + lane]);
                    qn -= 32;
                    __syncwarp();
                }
            }
            if (lane < qn) pair(qd[wl][lane], qj[wl][lane]);
            __syncwarp();
            const int io = rs_orig[i];
#pragma unroll
            for (int r = 0; r < NR; ++r) {
#pragma unroll
                for (int k = 0; k < NA; ++k) {
                    double v = acc[r][k];
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
                    acc[r][k] = v;
                }
                if (lane == 0) {
                    double *o = out_real + r * rhs_stride + 12 * (size_t)io;
                    if (COMP) acc[r][11] *= 1.0 / c.k0;               // p carries its own prefactor
                    if (base == 0) {
#pragma unroll
                        for (int k = 0; k < NA; ++k) o[k] = c.k0 * acc[r][k];
                    } else {
#pragma unroll
                        for (int k = 0; k < NA; ++k) o[k] += c.k0 * acc[r][k];
                    }
                }
            }
        }
    }
    // a cell without any candidate at all cannot occur (it contains its own targets), so every target was written
    }
}

// ------------------------------------------------------------------------------------------------------------
// Cached pairs (the paper prebuilds its real-space matrix once per configuration for the same reason):
// with the configuration fixed by se_plan_set_positions, the neighbour search and every pair's erfc/exp and radial scalars
// are done ONCE; every later product only streams the pair list and contracts it with the new moments.
//   k_pairs<false>  counts the pairs r < r_c of every target (cell order);   k_pairs<true>  fills, per target i, its row
//   of the list: pj[row + p] = partner (cell order), pd[row * PAIR_F + f * n_i + p] = field f of pair p (row-local
//   structure of arrays: x, y, z, then the 17 scalars of PairS<false>), n_i = pairs of the target.
//   k_real_cached   half a warp per target: lanes stride over the row (coalesced field loads), gather the partner's
//   moments, apply, reduce over the 16 lanes.
// Same scan machinery as k_real (27 staged neighbour cells or all pairs, chunks of REAL_STAGE candidates).
// ------------------------------------------------------------------------------------------------------------
#define PAIR_F 20

template <bool FILL>
__global__ void __launch_bounds__(REAL_WARPS * 32) k_pairs(SeConst c, const double4 *__restrict__ rs_pos, const int *__restrict__ start_r,
                                                           int *__restrict__ cnt,              // [N] pairs per target (count mode: written)
                                                           const int *__restrict__ row_start,  // [N+1] (fill mode)
                                                           int *__restrict__ cursor,           // [N] pairs of the target written so far (fill mode; zeroed)
                                                           int *__restrict__ pj, double *__restrict__ pd)
{
    __shared__ double4 cand[REAL_STAGE];
    __shared__ int cand_j[REAL_STAGE];
    __shared__ double4 qd[REAL_WARPS][REAL_QCAP];
    __shared__ int qj[REAL_WARPS][REAL_QCAP];
    __shared__ int seg_s[27], seg_o[28];
    const int wl = threadIdx.x >> 5, lane = threadIdx.x & 31, tid = threadIdx.x;
    const int nc = c.ncr;
    const int nitems = nc > 1 ? nc * nc * nc : (int)gridDim.x;
    for (int item = blockIdx.x; item < nitems; item += gridDim.x) {
    __syncthreads();
    int t0, t1, nsegs;
    if (nc > 1) {
        const int cell = item;
        t0 = start_r[cell]; t1 = start_r[cell + 1];
        if (t0 == t1) continue;
        nsegs = 27;
        if (tid < 27) {
            const int cz = cell % nc, cy = (cell / nc) % nc, cx = cell / (nc * nc);
            const int nx = se_mod(cx + tid / 9 - 1, nc), ny = se_mod(cy + (tid / 3) % 3 - 1, nc), nz = se_mod(cz + tid % 3 - 1, nc);
            const int nb = (nx * nc + ny) * nc + nz;
            seg_s[tid] = start_r[nb];
            seg_o[tid + 1] = start_r[nb + 1] - start_r[nb];
        }
    } else {
        const int per = (c.N + gridDim.x - 1) / gridDim.x;
        t0 = item * per; t1 = min(t0 + per, c.N);
        if (t0 >= t1) continue;
        nsegs = 1;
        if (tid == 0) { seg_s[0] = 0; seg_o[1] = c.N; }
    }
    __syncthreads();
    if (tid == 0) {
        int run = 0;
        seg_o[0] = 0;
        for (int k = 0; k < nsegs; ++k) { const int n = seg_o[k + 1]; seg_o[k + 1] = run + n; run += n; }
    }
    __syncthreads();
    const int ncand = seg_o[nsegs];
    const int rounds = (t1 - t0 + REAL_WARPS - 1) / REAL_WARPS;
    for (int base = 0; base < ncand; base += REAL_STAGE) {
        const int nst = min(REAL_STAGE, ncand - base);
        __syncthreads();
        for (int q = tid; q < nst; q += REAL_WARPS * 32) {
            const int f = base + q;
            int k = 0;
            while (k + 1 < nsegs && seg_o[k + 1] <= f) ++k;
            const int j = seg_s[k] + (f - seg_o[k]);
            cand[q] = rs_pos[j];
            cand_j[q] = j;
        }
        __syncthreads();
        for (int rd = 0; rd < rounds; ++rd) {
            const int i = t0 + rd * REAL_WARPS + wl;
            if (i >= t1) break;
            const double4 pi = rs_pos[i];
            const double cFi = pi.w * pi.w * (1.0 / 6.0), cSi = pi.w * pi.w * 0.1;
            int done = 0, row = 0, ni = 0;
            if (FILL) { row = row_start[i]; ni = row_start[i + 1] - row; done = cursor[i]; }
            auto emit = [&](const double4 &d, int jj, int p) {          // pair p of the row
                const PairS<false> o = pair_scalars<false>(c, d.x * d.x + d.y * d.y + d.z * d.z, cFi, cSi, d.w);
                pj[row + p] = jj;
                double *f = pd + (size_t)row * PAIR_F + p;
                const double v[PAIR_F] = { d.x, d.y, d.z, o.uf_a, o.uf_b, o.ut, o.us_a, o.us_b, o.of, o.ot_a, o.ot_b, o.os,
                                           o.a1, o.a2, o.a3, o.a4, o.ef2, o.ef3, o.es3, o.es4 };
#pragma unroll
                for (int q = 0; q < PAIR_F; ++q) f[(size_t)q * ni] = v[q];
            };
            int qn = 0;
            for (int qb = 0; qb < nst; qb += 32) {
                const int q = qb + lane;
                bool hit = false;
                double dx = 0, dy = 0, dz = 0, aj = 0;
                int j = -1;
                if (q < nst) {
                    const double4 pjv = cand[q];
                    j = cand_j[q];
                    dx = pi.x - pjv.x; dy = pi.y - pjv.y; dz = pi.z - pjv.z;
                    se_min_image(c, dx, dy, dz);
                    const double r2 = dx * dx + dy * dy + dz * dz;
                    hit = (j != i) && (r2 < c.rc2) && (r2 > 0.0);
                    aj = pjv.w;
                }
                const unsigned mask = __ballot_sync(0xffffffffu, hit);
                if (!FILL) { qn += __popc(mask); continue; }
                if (hit) {
                    const int slot = qn + __popc(mask & ((1u << lane) - 1u));
                    qd[wl][slot] = make_double4(dx, dy, dz, aj);
                    qj[wl][slot] = j;
                }
                qn += __popc(mask);
                __syncwarp();
                if (qn >= 32) {
                    emit(qd[wl][qn - 32 + lane], qj[wl][qn - 32 + lane], done + lane);
                    done += 32;
                    qn -= 32;
                    __syncwarp();
                }
            }
            if (FILL) {
                if (lane < qn) emit(qd[wl][lane], qj[wl][lane], done + lane);
                done += qn;
                __syncwarp();
                if (lane == 0) cursor[i] = done;
            } else if (lane == 0) {
                if (base == 0) cnt[i] = qn; else cnt[i] += qn;
            }
        }
    }
    }
}

// out_real[r][rs_orig[i]][0..10] = k0 * sum over the cached pairs of target i (cell order) applied to the moments rs_mom[r],
// r < NR right-hand sides `rhs_stride` doubles apart: the list is streamed once for all of them.
template <int NR>
__global__ void __launch_bounds__(128) k_real_cached(SeConst c, const int *__restrict__ row_start, const int *__restrict__ pj,
                                                     const double *__restrict__ pd, const double *__restrict__ rs_mom,
                                                     const int *__restrict__ rs_orig, double *__restrict__ out_real, size_t rhs_stride)
{
    const int hl = threadIdx.x & 15;
    const int nhw = (int)(gridDim.x * blockDim.x) >> 4;
    for (int i0 = (int)(blockIdx.x * blockDim.x + threadIdx.x) >> 4; ; i0 += nhw) {
        // the two halves of a warp walk in step (shuffles below are warp-wide); a half past the end idles
        const bool live = i0 < c.N;
        if (!__any_sync(0xffffffffu, live)) break;
        const int i = live ? i0 : c.N - 1;
        const int row = row_start[i], n = live ? row_start[i + 1] - row : 0;
        const double *__restrict__ f = pd + (size_t)row * PAIR_F;
        double acc[NR][12];
#pragma unroll
        for (int r = 0; r < NR; ++r)
#pragma unroll
            for (int k = 0; k < 12; ++k) acc[r][k] = 0.0;
        for (int p = hl; p < n; p += 16) {
            PairS<false> o;
            const double x = f[p], y = f[(size_t)n + p], z = f[2 * (size_t)n + p];
            o.uf_a = f[3 * (size_t)n + p]; o.uf_b = f[4 * (size_t)n + p]; o.ut = f[5 * (size_t)n + p]; o.us_a = f[6 * (size_t)n + p];
            o.us_b = f[7 * (size_t)n + p]; o.of = f[8 * (size_t)n + p]; o.ot_a = f[9 * (size_t)n + p]; o.ot_b = f[10 * (size_t)n + p];
            o.os = f[11 * (size_t)n + p]; o.a1 = f[12 * (size_t)n + p]; o.a2 = f[13 * (size_t)n + p]; o.a3 = f[14 * (size_t)n + p];
            o.a4 = f[15 * (size_t)n + p]; o.ef2 = f[16 * (size_t)n + p]; o.ef3 = f[17 * (size_t)n + p]; o.es3 = f[18 * (size_t)n + p];
            o.es4 = f[19 * (size_t)n + p];
            const double *__restrict__ mj = rs_mom + 12 * (size_t)pj[row + p];
#pragma unroll
            for (int r = 0; r < NR; ++r) {
                double m[12];
                const double2 *__restrict__ m2 = reinterpret_cast<const double2 *>(mj + r * rhs_stride);     // rows of 96 bytes: 16-byte aligned
#pragma unroll
                for (int q = 0; q < 6; ++q) { const double2 t = m2[q]; m[2 * q] = t.x; m[2 * q + 1] = t.y; }
                pair_apply<false>(o, x, y, z, 0.0, m, acc[r]);
            }
        }
        const int io = rs_orig[i];
#pragma unroll
        for (int r = 0; r < NR; ++r) {
#pragma unroll
            for (int k = 0; k < 11; ++k) {
                double v = acc[r][k];
#pragma unroll
                for (int s = 8; s > 0; s >>= 1) v += __shfl_xor_sync(0xffffffffu, v, s);
                acc[r][k] = v;
            }
            if (live && hl == 0) {
                double *o = out_real + r * rhs_stride + 12 * (size_t)io;
#pragma unroll
                for (int k = 0; k < 11; ++k) o[k] = c.k0 * acc[r][k];
            }
        }
    }
}
