// a7: Gaussian gather (Eq. 45 / Eq. 52 by the trapezoidal rule, L280) and a8: epilogue.
//   U_i  = D^3 sum_n gamma(d) (u~ + cF_i w~)
//   Om_i = D^3 sum_n al gamma(d) d x u~
//   E_i  = traceless part of D^3 sum_n al gamma(d) (d q + q d),  q = u~ + cS_i w~,   d = x_n - r_i
// over the same P^3 support as the spreading.  All of it follows from four sums per returned grid g,
//     A0[g] = sum gamma g,  A1[g] = sum gamma dx g,  Ay[g] = sum gamma dy g,  Az[g] = sum gamma dz g,
// which this kernel writes to moments[N][24] (caller order); a8 combines them per particle.
//
// Design ("plane ring", persistent): one CTA per SM walks over work items (returned grid, x segment, (y,z) tile of
// TY x TZ support origins).  The planes of the item's haloed tile, WY x WZ columns, stream through a ring of R planes
// in shared memory, filled by ONE TMA tensor-box copy per plane (cp.async.bulk.tensor.3d issued by one elected
// thread, completion counted in bytes by the slot's "full" mbarrier).  The returned grids are stored with P-1
// periodic halo rows and columns (written by the inverse z transform itself), so every box lies inside the padded
// plane: there is no seam path.  The producer runs across item boundaries, so the ring never drains between items.
// Consumers: the particles whose support starts in the tile are sorted by starting plane (a1); a consumer warp takes
// TWO particles at a time for P <= 16, one per half-warp (one per warp for larger P).  The 16 lanes of a particle
// form a 4 x 4 grid (by, bz) and own the footprint columns (by + 4a, bz + 4b): with rows padded to WZ = 4 (mod 8)
// doubles the sixteen columns of one load fall in sixteen different banks, all other addresses of a lane differ
// from its first by compile-time constants, and for P = 12 every lane owns exactly nine columns.  A lane reduces
// along x in registers,   m0 = sum_k gx(k) g(x0+k),   m1 = sum_k gx(k) dx_k g(x0+k),
// weights with the (y,z) Gaussians and the four sums are reduced over the 16 (32) lanes once per particle.  Every
// (particle, grid) pair is produced by exactly one half-warp in a fixed order: no atomics, bitwise reproducible.
// Planes are released through per-slot "empty" mbarriers (one arrival per consumer warp), so warps run up to R-P
// planes apart without CTA-wide barriers.  Gather records (se_common.cuh) arrive by bulk copies, double-buffered.
#pragma once
#include <cuda.h>                  // CUtensorMap (type only; the encoder is fetched through the runtime)
#include "se_sweep.cuh"
#include "se_sort.cuh"

#define GATHER_SUMS 24             // per particle: slot (g/3)*12 + kind*3 + g%3, kind = 0 (1), 1 (dx), 2 (dy), 3 (dz)
#ifndef GR_WARPS
#define GR_WARPS 12                // consumer warps; warp GR_WARPS is the producer
#endif

#ifndef GR_PREFETCH
#define GR_PREFETCH 16             // planes the producer's L2 prefetch cursor runs ahead of its loads
#endif
#ifndef GT_TZ12
#define GT_TZ12 32                 // tile width along z for P <= 12
#endif
#ifndef GT_RS12
#define GT_RS12 7                  // ring slack for P <= 12: R = P + GT_RS12 planes
#endif
// Compile-time geometry of the gather for support P.
template <int P> struct GatherTraits {
    static constexpr bool HALF = P <= 16;                       // two particles per warp
    static constexpr int LP = HALF ? 16 : 32;                   // lanes per particle
    static constexpr int LZ = LP / 4;                           // lane grid 4 x LZ
    static constexpr int CY = (P + 3) / 4, CZ = (P + LZ - 1) / LZ;   // footprint columns per lane: CY x CZ
    static constexpr int TY = P <= 16 ? 16 : (P <= 20 ? 8 : 2);
    static constexpr int TZ = P <= 12 ? GT_TZ12 : (P <= 16 ? 16 : 8);
    static constexpr int R = P <= 12 ? P + GT_RS12 : (P <= 16 ? P + 4 : (P <= 20 ? P + 3 : P + 1));
    static constexpr int WY = TY + 4 * CY - 1;                  // rows of the haloed tile (>= TY + P - 1)
    static constexpr int WZ0 = TZ + LZ * CZ - 1;
    // row pitch = 4 (mod 8) [half-warp particles] or 8 (mod 16) [warp particles]: conflict-free column loads
    static constexpr int WZ = HALF ? ((WZ0 + 3) / 8) * 8 + 4 : ((WZ0 + 7) / 16) * 16 + 8;
    static constexpr int SLOT = (WY * WZ + 15) & ~15;           // doubles per ring slot (a multiple of 128 bytes)
    static constexpr int PP = (P + 7) & ~7;
    static constexpr int GSTRIDE = 4 + 2 * PP + 2 * P;          // = se_grec_stride(P)
    static constexpr int NPW = HALF ? 2 : 1;                    // particles per warp pass
    static constexpr size_t SMEM = (size_t)R * SLOT * 8 + (size_t)GR_WARPS * 2 * NPW * GSTRIDE * 8 + (size_t)R * 16 + GR_WARPS * 16;
};

__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ bool mbar_test(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile("{\n.reg .pred P1;\nmbarrier.try_wait.parity.shared::cta.b64 P1, [%1], %2;\nselp.u32 %0, 1, 0, P1;\n}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}

// One box of the tensor `tmap` at element coordinates (c0 fastest, c1, c2) into shared memory at `dst`.
__device__ __forceinline__ void tma_box3(uint32_t dst, const CUtensorMap *tmap, int c0, int c1, int c2, uint32_t bar)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"(dst), "l"(tmap), "r"(c0), "r"(c1), "r"(c2), "r"(bar) : "memory");
}

// Ask for the same box to be brought into L2 (no shared-memory destination, no completion to wait for).
__device__ __forceinline__ void tma_prefetch3(const CUtensorMap *tmap, int c0, int c1, int c2)
{
    asm volatile("cp.async.bulk.prefetch.tensor.3d.L2.global.tile [%0, {%1, %2, %3}];" ::"l"(tmap), "r"(c0), "r"(c1), "r"(c2) : "memory");
}

// Work of the launch: items = (returned grid, (y,z) tile), tiles of one grid consecutive, M planes each.  They are dealt
// to the persistent CTAs round-robin, so that at any moment the CTAs work on neighbouring tiles of the same planes and the
// halo re-reads hit L2.  The items of the last, incomplete round (768 items on 148 SMs: 28 left after five rounds) are cut
// along x into floor(gridDim / left) segments each, so that every CTA gets a share of it instead of 28 CTAs a whole sixth
// item.  A sub-item (item, [x0, x1)): the planes x0 .. x1 + P - 2 stream through the ring, the particles whose support
// starts in [x0, x1) are gathered.
struct GatherItem { int grid, seg_start, nplanes, Y0, Z0, i0, i1; };
struct GatherWalk {
    int round, nfull, nitems, left, nsplit;
    __device__ __forceinline__ GatherWalk(const GatherGeom &g, int ngrids)
    {
        nitems = g.NTY * g.NTZ * ngrids;
        nfull = nitems / (int)gridDim.x;
        left = nitems - nfull * (int)gridDim.x;
        nsplit = left > 0 ? (int)gridDim.x / left : 1;
        round = 0;
    }
    // next sub-item with particles; false at the end of this CTA's work
    __device__ __forceinline__ bool next(GatherItem &r, const SeConst &c, const GatherGeom &g, const int *__restrict__ start_g)
    {
        const int M = c.M, ntile = g.NTY * g.NTZ, b = (int)blockIdx.x;
        while (round <= nfull) {
            int it, x0 = 0, x1 = M;
            if (round < nfull) it = round * (int)gridDim.x + b;
            else {
                if (b >= left * nsplit) { ++round; break; }
                const int q = b % nsplit, len = (M + nsplit - 1) / nsplit;
                it = nfull * (int)gridDim.x + b / nsplit;
                x0 = q * len; x1 = min(x0 + len, M);
                if (x0 >= x1) { ++round; break; }
            }
            ++round;
            const int gi = it / ntile, tile = it - gi * ntile;
            r.i0 = start_g[tile * M + x0];
            r.i1 = start_g[tile * M + x1];
            if (r.i0 == r.i1) continue;                               // no support starts here: skipped by everybody
            r.grid = gi;
            r.seg_start = x0;
            r.nplanes = x1 - x0 + c.P - 1;
            const int ty = tile / g.NTZ, tz = tile - ty * g.NTZ;
            r.Y0 = ty * g.TY; r.Z0 = tz * g.TZ;
            return true;
        }
        return false;
    }
};

// RV (real-space size variant): the Faxen operators act on the Gaussian of the gather, (1 + cF lap) gamma
// = gamma (1 + cF (4 al^2 d^2 - 6 al)) and its gradient, so four more sums per grid are needed,
//     Q0[g] = sum gamma d^2 g,  Q1[g] = sum gamma d^2 dx g,  Qy[g], Qz[g],
// from the x moments m2 = sum gx dx^2 g and m3 = sum gx dx^3 g: d^2 = dx^2 + dy^2 + dz^2.  Slot of (kind, g): kind*3 + g, g < 3.
template <int P, bool RV>
__global__ void __launch_bounds__((GR_WARPS + 1) * 32, 1)
k_gather(SeConst c, GatherGeom g, const double *__restrict__ grecs, const int *__restrict__ start_g,
         const __grid_constant__ CUtensorMap tmap, int ngrids, double *__restrict__ moments, int mstride)
{
    using GT = GatherTraits<P>;
    constexpr int R = GT::R, SLOT = GT::SLOT, WZ = GT::WZ, CY = GT::CY, CZ = GT::CZ, LZ = GT::LZ, LP = GT::LP, NPW = GT::NPW;
    constexpr int GS = GT::GSTRIDE, PP = GT::PP;
    extern __shared__ __align__(128) unsigned char gsm[];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int M = c.M;

    double *ring = reinterpret_cast<double *>(gsm);
    double *rbuf = ring + (size_t)R * SLOT;                            // [GR_WARPS][2][NPW][GS] record buffers
    const uint32_t bars = smem_u32(rbuf + GR_WARPS * 2 * NPW * GS);
    auto full_bar = [&](int sl) { return bars + 16u * (uint32_t)sl; };
    auto empty_bar = [&](int sl) { return bars + 16u * (uint32_t)sl + 8u; };
    const uint32_t rbars = bars + 16u * R;                             // per consumer warp: two record barriers
    if (threadIdx.x == 0) {
        for (int sl = 0; sl < R; ++sl) { mbar_init(full_bar(sl), 1); mbar_init(empty_bar(sl), GR_WARPS); }
        for (int q = 0; q < 2 * GR_WARPS; ++q) mbar_init(rbars + 8u * q, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    if (w == GR_WARPS) {
        // ---- producer (one elected thread): plane after plane of item after item; global plane n goes to slot n % R
        // once every consumer has released plane n - R; one tensor-box copy per plane.
        if (lane == 0) {
            const uint32_t ring_a = smem_u32(ring);
            constexpr uint32_t box_bytes = (uint32_t)(GT::WY * WZ * 8);
            int sl = 0;
            uint32_t par = 1;                                          // passes at once in round 0
            // A second cursor runs GR_PREFETCH planes ahead of the loads (across item boundaries) and asks for the boxes
            // to be brought into L2, so that the ring fill itself sees L2 latency only: the ring's slack of R - P planes
            // is too short to cover a DRAM miss under load.
            int pj = 0, ahead = 0;
            GatherWalk pw(g, ngrids);
            GatherItem PI;
            bool phave = pw.next(PI, c, g, start_g);
            auto prefetch_step = [&]() {                               // prefetch one plane, advance the cursor
                while (phave && pj >= PI.nplanes) { phave = pw.next(PI, c, g, start_g); pj = 0; }
                if (!phave) return;
                int x = PI.seg_start + pj;
                if (x >= M) x -= M;
                tma_prefetch3(&tmap, PI.Z0, PI.Y0, PI.grid * M + x);
                ++pj;
            };
            GatherWalk lw(g, ngrids);
            GatherItem I;
            while (lw.next(I, c, g, start_g)) {
                int x = I.seg_start;
                for (int j = 0; j < I.nplanes; ++j) {
                    while (ahead < GR_PREFETCH + 1) { prefetch_step(); ++ahead; }
                    mbar_wait(empty_bar(sl), par);
                    mbar_expect_tx(full_bar(sl), box_bytes);
                    tma_box3(ring_a + 8u * (uint32_t)(sl * SLOT), &tmap, I.Z0, I.Y0, I.grid * M + x, full_bar(sl));
                    --ahead;
                    if (++sl == R) { sl = 0; par ^= 1u; }
                    if (++x == M) x = 0;
                }
            }
        }
        return;
    }

    // ---- consumers ----
    // ring state: planes of the current item below jdone are known loaded (slot / parity of plane jdone: sdone, pdone),
    // planes below jrel are released by this warp (slot of plane jrel: srel).  Every consumer observes every phase of
    // every slot in order and releases a plane only after having observed it: the parity waits can never alias.
    int sdone = 0, srel = 0;
    uint32_t pdone = 0;
    const int half = NPW == 2 ? lane >> 4 : 0, hl = lane & (LP - 1);
    const int by = hl / LZ, bz = hl - by * LZ;
    double *rb = rbuf + (size_t)w * 2 * NPW * GS;
    const uint32_t rbar0 = rbars + 16u * (uint32_t)w;
    uint32_t rpar = 0;                                                 // bit b: parity of record buffer b
    const double Delta = c.Delta;

    GatherWalk cw(g, ngrids);
    GatherItem I;
    while (cw.next(I, c, g, start_g)) {
        int jdone = 0, jrel = 0;
        auto observe_next = [&]() {
            mbar_wait(full_bar(sdone), pdone);
            ++jdone;
            if (++sdone == R) { sdone = 0; pdone ^= 1u; }
        };
        auto release_below = [&](int jto) {
            while (jrel < jto) {
                if (jrel == jdone) observe_next();
                __syncwarp();
                if (lane == 0) mbar_arrive(empty_bar(srel));
                ++jrel;
                if (++srel == R) srel = 0;
            }
        };
        // passes of this warp: particles i0 + NPW (w + GR_WARPS t) [+ 1]
        const int npass = (I.i1 - I.i0 + NPW - 1) / NPW;
        auto stage = [&](int t, int b) {                               // records of pass t into buffer b
            if (lane == 0) {
                const int i = I.i0 + NPW * t, n = min(NPW, I.i1 - i);
                const uint32_t bytes = (uint32_t)(n * GS * 8);
                mbar_expect_tx(rbar0 + 8u * b, bytes);
                bulk_g2s(smem_u32(rb + (size_t)b * NPW * GS), grecs + (size_t)i * GS, bytes, rbar0 + 8u * b);
            }
        };
        int b = 0;
        if (w < npass) stage(w, 0);
        for (int t = w; t < npass; t += GR_WARPS, b ^= 1) {
            __syncwarp();                                              // buffer b^1 no longer read by any lane
            if (t + GR_WARPS < npass) stage(t + GR_WARPS, b ^ 1);
            mbar_wait(rbar0 + 8u * b, (rpar >> b) & 1u);
            rpar ^= 1u << b;
            const bool valid = NPW == 1 || I.i0 + NPW * t + half < I.i1;       // the odd particle out has no partner
            const double *__restrict__ rs = rb + (size_t)(b * NPW + (valid ? half : 0)) * GS;
            const int2 yz = reinterpret_cast<const int2 *>(rs)[0], xo = reinterpret_cast<const int2 *>(rs)[1];
            const int j0 = xo.x - I.seg_start;
            int jlo = j0, jhi = j0;
            if (NPW == 2) {
                const int o = __shfl_xor_sync(0xffffffffu, j0, 16);
                jlo = min(j0, o); jhi = max(j0, o);
            }
            // Two particles whose windows do not fit the ring together take one turn each (then jlo < jhi strictly).
            const int nturn = (NPW == 2 && jhi - jlo + P > R) ? 2 : 1;
            for (int turn = 0; turn < nturn; ++turn) {
                const bool mine = nturn == 1 || j0 == (turn == 0 ? jlo : jhi);
                const int ja = (nturn == 2 && turn == 1) ? jhi : jlo, jb = (nturn == 2 && turn == 0) ? jlo : jhi;
                release_below(ja);                                     // now jrel == ja, srel = slot of plane ja
                while (jdone < jb + P) observe_next();
                int sl = srel + (mine ? j0 - ja : 0);                  // slot of my first plane (idle lanes: any loaded one)
                if (sl >= R) sl -= R;
                const double *__restrict__ col = ring + ((yz.x - I.Y0 + by) * WZ + (yz.y - I.Z0 + bz));
                double m0[CY][CZ], m1[CY][CZ], m2[RV ? CY : 1][RV ? CZ : 1], m3[RV ? CY : 1][RV ? CZ : 1];
#pragma unroll
                for (int a = 0; a < CY; ++a)
#pragma unroll
                    for (int q = 0; q < CZ; ++q) {
                        m0[a][q] = 0.0; m1[a][q] = 0.0;
                        if (RV) { m2[a][q] = 0.0; m3[a][q] = 0.0; }
                    }
                const double2 *__restrict__ GX = reinterpret_cast<const double2 *>(rs + 4 + 2 * PP);
                const double d0x = RV ? GX[0].y / GX[0].x : 0.0;      // the table holds (gx, gx dx); gx(0) >= e^{-m^2/2} > 0
#pragma unroll
                for (int k = 0; k < P; ++k) {
                    const double *__restrict__ pl = col + sl * SLOT;
                    const double2 gx = GX[k];
                    const double dxk = fma((double)k, Delta, d0x), gx2 = gx.y * dxk, gx3 = gx2 * dxk;
#pragma unroll
                    for (int a = 0; a < CY; ++a)
#pragma unroll
                        for (int q = 0; q < CZ; ++q) {
                            const double v = pl[4 * a * WZ + LZ * q];
                            m0[a][q] = fma(gx.x, v, m0[a][q]);
                            m1[a][q] = fma(gx.y, v, m1[a][q]);
                            if (RV) {
                                m2[a][q] = fma(gx2, v, m2[a][q]);
                                m3[a][q] = fma(gx3, v, m3[a][q]);
                            }
                        }
                    sl = sl + 1 == R ? 0 : sl + 1;
                }
                // weights: sums over this lane's columns of gy gz {m0, m1, dy m0, dz m0}; gy, gz are zero beyond P
                const double d0y = rs[2] + by * Delta, d0z = rs[3] + bz * Delta;
                constexpr int B1 = LP / 2, B2 = LP / 4, B3 = LP / 8;
                if (!RV) {
                double gz[CZ], gzd[CZ];
#pragma unroll
                for (int q = 0; q < CZ; ++q) { gz[q] = rs[4 + PP + bz + LZ * q]; gzd[q] = gz[q] * (d0z + (LZ * q) * Delta); }
                double s0 = 0.0, s1 = 0.0, sy = 0.0, sz = 0.0;
#pragma unroll
                for (int a = 0; a < CY; ++a) {
                    double r0 = 0.0, r1 = 0.0, rz = 0.0;
#pragma unroll
                    for (int q = 0; q < CZ; ++q) {
                        r0 = fma(gz[q], m0[a][q], r0);
                        r1 = fma(gz[q], m1[a][q], r1);
                        rz = fma(gzd[q], m0[a][q], rz);
                    }
                    const double gy = rs[4 + by + 4 * a], gr0 = gy * r0;
                    s0 += gr0;
                    s1 = fma(gy, r1, s1);
                    sy = fma(d0y + (4 * a) * Delta, gr0, sy);
                    sz = fma(gy, rz, sz);
                }
                // reduce-scatter of the four sums over the LP lanes of the particle: the two highest lane bits select
                // the kind (00 s0, 01 s1, 10 sy, 11 sz), the remaining bits are summed
                {
                    const bool hi = (hl & B1) != 0;
                    const double a = (hi ? sy : s0) + __shfl_xor_sync(0xffffffffu, hi ? s0 : sy, B1);
                    const double bb = (hi ? sz : s1) + __shfl_xor_sync(0xffffffffu, hi ? s1 : sz, B1);
                    const bool h2 = (hl & B2) != 0;
                    double tt = (h2 ? bb : a) + __shfl_xor_sync(0xffffffffu, h2 ? a : bb, B2);
#pragma unroll
                    for (int o = B2 / 2; o > 0; o >>= 1) tt += __shfl_xor_sync(0xffffffffu, tt, o);
                    if ((hl & (B2 - 1)) == 0 && valid && mine) {
                        const int kind = (hi ? 2 : 0) | (h2 ? 1 : 0);
                        moments[(size_t)xo.y * mstride + (I.grid / 3) * 12 + kind * 3 + (I.grid % 3)] = tt;
                    }
                }
                } else {
                    // eight sums: kind 0 gamma, 1 gamma dx, 2 gamma dy, 3 gamma dz, 4..7 the same times D.D (d^2 in the cubic box)
                    const double g1 = 1.0 + c.gamma * c.gamma, gdy2 = -2.0 * c.gamma;
                    double sm[8];
#pragma unroll
                    for (int i = 0; i < 8; ++i) sm[i] = 0.0;
#pragma unroll
                    for (int a = 0; a < CY; ++a) {
                        const double gy = rs[4 + by + 4 * a], dy = d0y + (4 * a) * Delta;
#pragma unroll
                        for (int q = 0; q < CZ; ++q) {
                            const double dz = d0z + (LZ * q) * Delta, w = gy * rs[4 + PP + bz + LZ * q];
                            const double rho2 = fma(dy, dy, dz * dz);
                            const double t0 = w * m0[a][q], t1 = w * m1[a][q];
                            // weight D.D = (1 + g^2) dx^2 - 2 g dx dy + dy^2 + dz^2 (sheared lattice; g = 0: d^2)
                            const double u0 = w * fma(rho2, m0[a][q], fma(gdy2 * dy, m1[a][q], g1 * m2[a][q]));
                            const double u1 = w * fma(rho2, m1[a][q], fma(gdy2 * dy, m2[a][q], g1 * m3[a][q]));
                            sm[0] += t0; sm[1] += t1; sm[2] = fma(dy, t0, sm[2]); sm[3] = fma(dz, t0, sm[3]);
                            sm[4] += u0; sm[5] += u1; sm[6] = fma(dy, u0, sm[6]); sm[7] = fma(dz, u0, sm[7]);
                        }
                    }
                    // reduce-scatter over the LP lanes: the three highest lane bits select the kind, the rest is summed
                    const bool h1 = (hl & B1) != 0, h2 = (hl & B2) != 0, h3 = (hl & B3) != 0;
                    double v4[4], v2[2];
#pragma unroll
                    for (int i = 0; i < 4; ++i) v4[i] = (h1 ? sm[i + 4] : sm[i]) + __shfl_xor_sync(0xffffffffu, h1 ? sm[i] : sm[i + 4], B1);
#pragma unroll
                    for (int i = 0; i < 2; ++i) v2[i] = (h2 ? v4[i + 2] : v4[i]) + __shfl_xor_sync(0xffffffffu, h2 ? v4[i] : v4[i + 2], B2);
                    double tt = (h3 ? v2[1] : v2[0]) + __shfl_xor_sync(0xffffffffu, h3 ? v2[0] : v2[1], B3);
#pragma unroll
                    for (int o = B3 / 2; o > 0; o >>= 1) tt += __shfl_xor_sync(0xffffffffu, tt, o);
                    if ((hl & (B3 - 1)) == 0 && valid && mine) {
                        const int kind = (h1 ? 4 : 0) | (h2 ? 2 : 0) | (h3 ? 1 : 0);
                        moments[(size_t)xo.y * mstride + kind * 3 + I.grid] = tt;
                    }
                }
            }
        }
        __syncwarp();
        release_below(I.nplanes);
    }
}

// a8: out = real + wave + (one-body - self) * input, in caller order (Eq. 13-15 one-body terms;
// Eq. 37 and its Omega-T / E-S analogues for the wave-space self terms).  The wave part is combined here from
// the 24 gathered sums of the particle: with A = sums of u~ (A0 = gamma u, A1 = gamma dx u, Ay, Az) and
// B the same for w~,
//   U = D^3 (A0 + cF B0),  Om = al D^3 (Ay[2]-Az[1], Az[0]-A1[2], A1[1]-Ay[0]),
//   E = al D^3 traceless(d q + q d) with the d-moments C1 = A1 + cS B1, Cy = Ay + cS By, Cz = Az + cS Bz.
__global__ void k_epilogue(SeConst c, unsigned flags, const double *__restrict__ radii,
                           const double *__restrict__ F, const double *__restrict__ T, const double *__restrict__ S,
                           const double *__restrict__ out_real, const double *__restrict__ moments, int mstride,
                           const double *__restrict__ pmom,     // gathered pressure sums [N][12], slot 0 used (a9), or NULL
                           double *__restrict__ U, double *__restrict__ W, double *__restrict__ E,
                           double *__restrict__ s_out,           // 4 pi a^3 p'(r_i), Eq. 28 (a9), or NULL
                           int variant)                          // 0 hybrid, 1 real-space, 2 wave-space size terms (Sec. 3.2)
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
    double v[11];
#pragma unroll
    for (int k = 0; k < 11; ++k) v[k] = 0.0;
    if (!(flags & 0x1u)) {                                   // real-space part
        const double *orl = out_real + 12 * (size_t)i;
#pragma unroll
        for (int k = 0; k < 11; ++k) v[k] += orl[k];
    }
    if (!(flags & 0x2u)) {                                   // wave-space part
        const double *m = moments + (size_t)mstride * i;
        const double cF = a * a / 6.0, cS = a * a / 10.0, D3 = c.D3, aD3 = c.alpha * c.D3;
        double A0[3], A1[3], Ay[3], Az[3], C1[3], Cy[3], Cz[3];
        // sheared lattice: the gathered offsets are fractional (times L); the physical gradient of the Gaussian carries the
        // metric vector D = (dx, dy - gamma dx, dz) (se_spread.cuh), so only the y moments change
        const double gm = c.gamma;
        // real-space variant: slots 12.. hold the D.D-weighted sums Q of u~ instead of the sums of w~ (D.D = d^2 in the cubic box):
        // lap gamma = (4 al^2 D.D - 2 al tr) gamma for U; for E the gradient of (1 + cS lap) gamma is
        // -2 al D (1 + cS (4 al^2 D.D - 2 al tr)) gamma + 8 al^2 cS Mt.D gamma, tr = 3 + g^2 (se_spread.cuh); with g = 0, Mt.D = D and
        // the last term turns -6 al into the -10 al of the cubic formula
        const double tr = 3.0 + gm * gm, g1 = 1.0 + gm * gm;
        const double q2 = 4.0 * c.alpha * c.alpha, qU = variant == 1 ? -2.0 * c.alpha * tr : 0.0, qE = qU, qM = variant == 1 ? -4.0 * c.alpha : 0.0;
        const double qs = variant == 1 ? q2 : 1.0;
#pragma unroll
        for (int g = 0; g < 3; ++g) {
            A0[g] = m[g]; A1[g] = m[3 + g]; Ay[g] = m[6 + g] - gm * m[3 + g]; Az[g] = m[9 + g];
            v[g] += D3 * (A0[g] + cF * (qs * m[12 + g] + qU * A0[g]));
            // Mt.D from the raw first moments (d = grid offsets): ((1+g^2) dx - g dy, -g (2+g^2) dx + (1+g^2) dy, dz)
            const double M1 = g1 * m[3 + g] - gm * m[6 + g], My = -gm * (2.0 + gm * gm) * m[3 + g] + g1 * m[6 + g], Mz = m[9 + g];
            C1[g] = A1[g] + cS * (qs * m[15 + g] + qE * A1[g] + qM * M1);
            Cy[g] = Ay[g] + cS * (qs * (m[18 + g] - gm * m[15 + g]) + qE * Ay[g] + qM * My);
            Cz[g] = Az[g] + cS * (qs * m[21 + g] + qE * Az[g] + qM * Mz);
        }
        if (variant == 2) {
            // wave-space variant: plain sums of om~ (slots 24..26), e0~ (36..38, 48..50) and e2~ (60..62, 72..74)
            v[3] += D3 * m[24]; v[4] += D3 * m[25]; v[5] += D3 * m[26];
            const double exx = m[36] + cS * m[60], exy = m[37] + cS * m[61], exz = m[38] + cS * m[62];
            const double eyy = m[48] + cS * m[72], eyz = m[49] + cS * m[73], ezz = m[50] + cS * m[74];
            const double tr3 = (exx + eyy + ezz) * (1.0 / 3.0);
            v[6] += D3 * (exx - tr3); v[7] += D3 * exy; v[8] += D3 * exz; v[9] += D3 * (eyy - tr3); v[10] += D3 * eyz;
        } else {
        v[3] += aD3 * (Ay[2] - Az[1]);
        v[4] += aD3 * (Az[0] - A1[2]);
        v[5] += aD3 * (A1[1] - Ay[0]);
        const double exx = 2.0 * C1[0], eyy = 2.0 * Cy[1], ezz = 2.0 * Cz[2];
        const double tr3 = (exx + eyy + ezz) * (1.0 / 3.0);
        v[6] += aD3 * (exx - tr3);
        v[7] += aD3 * (C1[1] + Cy[0]);
        v[8] += aD3 * (C1[2] + Cz[0]);
        v[9] += aD3 * (eyy - tr3);
        v[10] += aD3 * (Cy[2] + Cz[1]);
        }
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        U[3 * (size_t)i + k] = v[k] + cU * F[3 * (size_t)i + k];
        W[3 * (size_t)i + k] = v[3 + k] + cW * T[3 * (size_t)i + k];
    }
#pragma unroll
    for (int k = 0; k < 5; ++k) E[5 * (size_t)i + k] = v[6 + k] + cE * S[5 * (size_t)i + k];
    if (s_out) {
        double pv = 0.0;
        if (!(flags & 0x1u)) pv += out_real[12 * (size_t)i + 11];
        if (!(flags & 0x2u) && pmom) pv += c.D3 * pmom[12 * (size_t)i];
        s_out[i] = 4.0 * PI * a3 * pv;
    }
}
