// a7: Gaussian gather (Eq. 45 / Eq. 52 by the trapezoidal rule, L280) and a8: epilogue.
//   U_i  = D^3 sum_n gamma(d) (u~ + cF_i w~)
//   Om_i = D^3 sum_n al gamma(d) d x u~
//   E_i  = traceless part of D^3 sum_n al gamma(d) (d q + q d),  q = u~ + cS_i w~,   d = x_n - r_i
// over the same P^3 support as the spreading.  All of it follows from four sums per returned grid g,
//     A0[g] = sum gamma g,  A1[g] = sum gamma dx g,  Ay[g] = sum gamma dy g,  Az[g] = sum gamma dz g,
// which this kernel writes to moments[N][24] (caller order); a8 combines them per particle.
//
// Design ("plane ring"): a CTA owns one returned grid, one (y,z) tile of TY x TZ support origins and one
// segment of x.  It streams the planes of its haloed tile, (TY+P-1) x (TZ+P-1) columns, through a ring of R
// planes in shared memory, R-P planes ahead of the consumers, so every grid value crosses L2->SM once per tile
// and is then read from shared memory.  The fill has two paths with the same slot layout.  A tile whose halo
// stays inside the grid takes ONE TMA tensor-box copy per plane (cp.async.bulk.tensor.3d issued by one elected
// thread, completion counted in bytes by the slot's mbarrier).  A tile whose halo crosses the periodic seam (the
// last tile row and column) copies the plane with 16-byte cp.async through a table that wraps the coordinates
// (two producer warps, completion counted by deferred mbarrier arrivals).  Measured on B200: the cp.async path
// sustains only ~10 B/clk/SM and bounded the whole kernel when every tile used it; a box copy per plane is
// ~6 times faster, and per-row bulk copies were slower than either.  The particles whose support starts in the tile are sorted by starting plane (a1,
// second counting sort); the eight consumer warps take them round-robin, ONE WARP PER PARTICLE: the lanes
// own the P^2 columns of the footprint (all lanes busy), reduce along x in registers,
//     m0 = sum_k gx(k) g(x0+k),   m1 = sum_k gx(k) dx_k g(x0+k),
// weight with the (y,z) Gaussian and reduce over the warp once per particle.  Every (particle, grid) pair
// is produced by exactly one warp in a fixed order: no atomics, no zero-fill, bitwise reproducible.
// Rows are padded to WZ = P (mod 16) doubles so that the footprint columns of a half-warp fall in
// distinct shared-memory banks.  Planes are released through per-slot "empty" mbarriers (one arrival per
// consumer warp), so warps run up to R-P planes apart without CTA-wide barriers.
#pragma once
#include <cuda.h>                  // CUtensorMap (type only; the encoder is fetched through the runtime)
#include "se_sweep.cuh"
#include "se_sort.cuh"

#define GATHER_SUMS 24             // per particle: slot (g/3)*12 + kind*3 + g%3, kind = 0 (1), 1 (dx), 2 (dy), 3 (dz)
#ifndef GR_WARPS
#define GR_WARPS 8                 // consumer warps
#endif
// Two CTAs per SM hide each other's pipeline bubbles; supports up to GR_P2MAX keep the register budget for it.
#ifndef GR_P2MAX
#define GR_P2MAX 14
#endif
#define GR_PROD 2                  // producer warps (GR_WARPS, GR_WARPS + 1)

__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}

__device__ __forceinline__ void cp_async16(uint32_t dst, const void *src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
// Arrive on `bar` once all cp.async of this thread issued so far have landed (counted in the barrier's init count).
__device__ __forceinline__ void cp_async_arrive(uint32_t bar)
{
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(bar) : "memory");
}

// One box of the tensor `tmap` at element coordinates (c0 fastest, c1, c2) into shared memory at `dst`.
__device__ __forceinline__ void tma_box3(uint32_t dst, const CUtensorMap *tmap, int c0, int c1, int c2, uint32_t bar)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"(dst), "l"(tmap), "r"(c0), "r"(c1), "r"(c2), "r"(bar) : "memory");
}

template <int P>
__global__ void __launch_bounds__((GR_WARPS + GR_PROD) * 32, (P <= GR_P2MAX ? 2 : 1))
k_gather(SeConst c, GatherGeom g, const double *__restrict__ recs, const int *__restrict__ gperm,
         const int *__restrict__ start_g, const double *__restrict__ Gr, const __grid_constant__ CUtensorMap tmap, int ngrids,
         double *__restrict__ moments, int mstride)
{
    extern __shared__ __align__(128) unsigned char gsm[];
    constexpr int PP = P * P, NI = (PP + 31) / 32;
    constexpr int NREC = SE_REC_HDR + 4 * P, NR = (NREC + 31) / 32;      // record prefix the gather needs
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int M = c.M, stride = c.rec_stride, R = g.R;
    // Work items in launch order: tile slowest, and the seam tiles (last tile row and column: the slow cp.async
    // fill, see below) first, so that they do not form the tail of the launch.
    const int per_tile = ngrids * g.nseg;
    const int q = blockIdx.x / per_tile, rest = blockIdx.x - q * per_tile;
    const int grid = rest % ngrids, seg = rest / ngrids;
    const int nseam = g.NTY + g.NTZ - 1;
    int ty, tz;
    if (q < g.NTZ) { ty = g.NTY - 1; tz = q; }
    else if (q < nseam) { ty = q - g.NTZ; tz = g.NTZ - 1; }
    else { const int r = q - nseam; ty = r / (g.NTZ - 1); tz = r - ty * (g.NTZ - 1); }
    const int tile = ty * g.NTZ + tz;
    const int seg_start = seg * g.seg_len, seg_end = min(seg_start + g.seg_len, M);
    const int i0 = start_g[tile * M + seg_start], i1 = start_g[tile * M + seg_end];
    if (i0 == i1) return;                                              // no support starts here
    const int Y0 = ty * g.TY, Z0 = tz * g.TZ;
    const int nplanes = seg_end - seg_start + P - 1;
    const int plane_d = g.slot_d;                                      // doubles per ring slot (a multiple of 128 bytes)
    // the box [Y0, Y0+WY) x [Z0, Z0+WZ) may reach beyond the grid only in its unused pad columns (zero-filled)
    const bool use_tma = (Y0 + g.TY + P - 1 <= M) && (Z0 + g.TZ + P - 1 <= M);
    const int cw = g.WZL >> 1, nch = g.WY * cw;                        // 16-byte chunks per row, per plane

    double *ring = reinterpret_cast<double *>(gsm);
    double *rslots = ring + (size_t)R * plane_d;                       // per consumer warp: one record prefix
    int2 *table = reinterpret_cast<int2 *>(rslots + GR_WARPS * NR * 32);   // per chunk: (offset in a grid plane, offset in a slot)
    const uint32_t bars = smem_u32(table + nch);
    auto full_bar = [&](int sl) { return bars + 16u * (uint32_t)sl; };
    auto empty_bar = [&](int sl) { return bars + 16u * (uint32_t)sl + 8u; };
    if (threadIdx.x == 0) {
        for (int sl = 0; sl < R; ++sl) { mbar_init(full_bar(sl), use_tma ? 1 : GR_PROD * 32); mbar_init(empty_bar(sl), GR_WARPS); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    if (!use_tma) for (int ch = threadIdx.x; ch < nch; ch += blockDim.x) {   // periodic wrap along y and z, once per CTA
        const int r = ch / cw, col = ch - r * cw;
        table[ch] = make_int2(((Y0 + r) % M) * M + (Z0 + 2 * col) % M, r * g.WZ + 2 * col);
    }
    __syncthreads();

    if (w >= GR_WARPS && use_tma) {
        // ---- producer, interior tile (one elected thread): plane j of the segment goes to slot j % R once every
        // consumer has released plane j - R; one tensor-box copy per plane.
        if (w == GR_WARPS && lane == 0) {
            const uint32_t ring_a = smem_u32(ring), box_bytes = (uint32_t)(g.WY * g.WZ * 8);
            int sl = 0, x = seg_start;
            uint32_t par = 1;                                          // passes at once in round 0
            for (int j = 0; j < nplanes; ++j) {
                mbar_wait(empty_bar(sl), par);
                mbar_expect_tx(full_bar(sl), box_bytes);
                tma_box3(ring_a + 8u * (uint32_t)(sl * plane_d), &tmap, Z0, Y0, grid * M + x, full_bar(sl));
                if (++sl == R) { sl = 0; par ^= 1u; }
                if (++x == M) x = 0;
            }
        }
        return;
    }
    if (w >= GR_WARPS) {
        // ---- producers, seam tile: as above, with the periodic wrap done by the chunk table.
        // 16-byte cp.async per chunk (rows are too short for bulk copies to pay); completion is counted by the
        // slot's "full" mbarrier, one deferred arrival per producer lane.
        const double *__restrict__ G0 = Gr + (size_t)grid * M * M * M;
        const int pl = (w - GR_WARPS) * 32 + lane;
        const uint32_t ring_a = smem_u32(ring);
        int sl = 0;
        uint32_t par = 1;                                              // passes at once in round 0
        int x = seg_start;
        for (int j = 0; j < nplanes; ++j) {
            mbar_wait(empty_bar(sl), par);
            const double *__restrict__ src = G0 + (size_t)x * M * M;
            const uint32_t dst = ring_a + 8u * (uint32_t)(sl * plane_d);
            for (int ch = pl; ch < nch; ch += GR_PROD * 32) {
                const int2 e = table[ch];
                cp_async16(dst + 8u * (uint32_t)e.y, src + e.x);
            }
            cp_async_arrive(full_bar(sl));
            if (++sl == R) { sl = 0; par ^= 1u; }
            if (++x == M) x = 0;
        }
        asm volatile("cp.async.wait_all;" ::: "memory");
        return;
    }

    // ---- consumers: particle i0 + w, i0 + w + 8, ... (non-decreasing starting plane per warp) ----
    double *rs = rslots + w * NR * 32;
    // planes [0, jdone) are known loaded (slot/parity of plane jdone: sdone, pdone); planes [0, jrel) released
    int jdone = 0, sdone = 0, jrel = 0, srel = 0;
    uint32_t pdone = 0;
    double pre[NR];
    auto fetch = [&](int ii) {
        const double *__restrict__ rec = recs + (size_t)gperm[ii] * stride;
#pragma unroll
        for (int q = 0; q < NR; ++q) pre[q] = (q * 32 + lane < NREC) ? rec[q * 32 + lane] : 0.0;
    };
    auto observe_next = [&]() {
        mbar_wait(full_bar(sdone), pdone);
        ++jdone;
        if (++sdone == R) { sdone = 0; pdone ^= 1u; }
    };
    // Every consumer observes every phase of every slot, in order, and releases a plane only after having
    // observed it: the parity waits can then never alias, however far apart the starting planes are.
    auto release_below = [&](int jto) {
        while (jrel < jto) {
            if (jrel == jdone) observe_next();
            __syncwarp();
            if (lane == 0) mbar_arrive(empty_bar(srel));
            ++jrel;
            if (++srel == R) srel = 0;
        }
    };
    // lane constants: footprint column lane + 32 q -> (ry, rz), its offset in a slot, its distance from the origin
    int colof[NI], colry[NI], colrz[NI];
    bool colok[NI];
    double coldy[NI], coldz[NI];
#pragma unroll
    for (int q = 0; q < NI; ++q) {
        const int cc = lane + 32 * q;
        colok[q] = cc < PP;
        const int cl = min(cc, PP - 1);
        colry[q] = cl / P; colrz[q] = cl - colry[q] * P;
        colof[q] = colry[q] * g.WZ + colrz[q];
        coldy[q] = colry[q] * c.Delta; coldz[q] = colrz[q] * c.Delta;
    }
    int i = i0 + w;
    if (i < i1) fetch(i);
    for (; i < i1; i += GR_WARPS) {
        __syncwarp();
#pragma unroll
        for (int q = 0; q < NR; ++q) rs[q * 32 + lane] = pre[q];
        __syncwarp();
        if (i + GR_WARPS < i1) fetch(i + GR_WARPS);                    // next record in flight during the sums
        const int2 yz = reinterpret_cast<const int2 *>(rs)[0], xo = reinterpret_cast<const int2 *>(rs)[1];
        const int j0 = xo.x - seg_start;
        release_below(j0);                                             // now jrel == j0 and srel == j0 % R
        while (jdone < j0 + P) observe_next();

        const int cb = (yz.x - Y0) * g.WZ + (yz.y - Z0);
        double m0[NI], m1[NI];
#pragma unroll
        for (int q = 0; q < NI; ++q) { m0[q] = 0.0; m1[q] = 0.0; }
        int sl = srel;
        const double *__restrict__ X0 = rs + SE_REC_HDR, *__restrict__ X1 = rs + SE_REC_HDR + 3 * P;
        double gxr[P], gxdr[P];                                        // x tables: loaded before the sums start
#pragma unroll
        for (int k = 0; k < P; ++k) { gxr[k] = X0[k]; gxdr[k] = X1[k]; }
#pragma unroll
        for (int k = 0; k < P; ++k) {
            const double *__restrict__ pl = ring + sl * plane_d;
            const double gx = gxr[k], gxd = gxdr[k];
#pragma unroll
            for (int q = 0; q < NI; ++q) {
                const double v = pl[cb + colof[q]];
                m0[q] = fma(gx, v, m0[q]);
                m1[q] = fma(gxd, v, m1[q]);
            }
            sl = sl + 1 == R ? 0 : sl + 1;
        }
        double s0 = 0.0, s1 = 0.0, sy = 0.0, sz = 0.0;
        const double d0y = rs[REC_D0 + 1], d0z = rs[REC_D0 + 2];
        const double *__restrict__ GY = rs + SE_REC_HDR + P, *__restrict__ GZ = rs + SE_REC_HDR + 2 * P;
#pragma unroll
        for (int q = 0; q < NI; ++q) {
            const double gyz = colok[q] ? GY[colry[q]] * GZ[colrz[q]] : 0.0;
            const double a0 = gyz * m0[q];
            s0 += a0;
            s1 = fma(gyz, m1[q], s1);
            sy = fma(d0y + coldy[q], a0, sy);
            sz = fma(d0z + coldz[q], a0, sz);
        }
        // reduce-scatter of the four sums: lane bits (16, 8) select the kind: 00 s0, 01 s1, 10 sy, 11 sz
        {
            const bool hi = (lane & 16) != 0;
            const double a = (hi ? sy : s0) + __shfl_xor_sync(0xffffffffu, hi ? s0 : sy, 16);
            const double b = (hi ? sz : s1) + __shfl_xor_sync(0xffffffffu, hi ? s1 : sz, 16);
            const bool h8 = (lane & 8) != 0;
            double t = (h8 ? b : a) + __shfl_xor_sync(0xffffffffu, h8 ? a : b, 8);
            t += __shfl_xor_sync(0xffffffffu, t, 4);
            t += __shfl_xor_sync(0xffffffffu, t, 2);
            t += __shfl_xor_sync(0xffffffffu, t, 1);
            if ((lane & 7) == 0) {
                const int kind = ((lane >> 4) << 1) | ((lane >> 3) & 1);
                moments[(size_t)xo.y * mstride + (grid / 3) * 12 + kind * 3 + (grid % 3)] = t;
            }
        }
    }
    __syncwarp();
    release_below(nplanes);
}

static inline size_t gather_smem_bytes(const GatherGeom &g, int P)
{
    const int NR = (SE_REC_HDR + 4 * P + 31) / 32;
    return (size_t)g.R * g.slot_d * 8 + (size_t)GR_WARPS * NR * 32 * 8 + (size_t)g.WY * (g.WZL / 2) * 8 + (size_t)g.R * 16;
}

// a8: out = real + wave + (one-body - self) * input, in caller order (Eq. 13-15 one-body terms;
// Eq. 37 and its Omega-T / E-S analogues for the wave-space self terms).  The wave part is combined here from
// the 24 gathered sums of the particle: with A = sums of u~ (A0 = gamma u, A1 = gamma dx u, Ay, Az) and
// B the same for w~,
//   U = D^3 (A0 + cF B0),  Om = al D^3 (Ay[2]-Az[1], Az[0]-A1[2], A1[1]-Ay[0]),
//   E = al D^3 traceless(d q + q d) with the d-moments C1 = A1 + cS B1, Cy = Ay + cS By, Cz = Az + cS Bz.
__global__ void k_epilogue(SeConst c, unsigned flags, const double *__restrict__ radii,
                           const double *__restrict__ F, const double *__restrict__ T, const double *__restrict__ S,
                           const double *__restrict__ out_real, const double *__restrict__ moments,
                           const double *__restrict__ pmom,     // gathered pressure sums [N][12], slot 0 used (a9), or NULL
                           double *__restrict__ U, double *__restrict__ W, double *__restrict__ E,
                           double *__restrict__ s_out)           // 4 pi a^3 p'(r_i), Eq. 28 (a9), or NULL
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
        const double *m = moments + (size_t)GATHER_SUMS * i;
        const double cF = a * a / 6.0, cS = a * a / 10.0, D3 = c.D3, aD3 = c.alpha * c.D3;
        double A0[3], A1[3], Ay[3], Az[3], C1[3], Cy[3], Cz[3];
#pragma unroll
        for (int g = 0; g < 3; ++g) {
            A0[g] = m[g]; A1[g] = m[3 + g]; Ay[g] = m[6 + g]; Az[g] = m[9 + g];
            v[g] += D3 * (A0[g] + cF * m[12 + g]);
            C1[g] = A1[g] + cS * m[15 + g];
            Cy[g] = Ay[g] + cS * m[18 + g];
            Cz[g] = Az[g] + cS * m[21 + g];
        }
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
