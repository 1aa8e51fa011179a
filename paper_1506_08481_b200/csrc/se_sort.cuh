// a1: wrap, counting sorts (by real-space cell and by spreading tile), packed per-particle records.
// PAPER.md Sec. 3.3 (cells slightly larger than r_c, 27-cell search) and Sec. 3.4 (per-grid-point
// particle lists, replaced here by a counting sort by grid tile).
#pragma once
#include "se_common.cuh"

// Geometry of the ring gather (se_gather.cuh).  The tile shape, ring depth and slot layout are compile-time functions
// of P (GatherTraits); this struct carries them, and the run-time tile / segment counts, to the kernels.
struct GatherGeom {
    int TY, TZ;                    // support origins per tile along y, z
    int NTY, NTZ;                  // tiles per axis
    int nseg, seg_len;             // segments of the sweep along x
    int MYp, MZp;                  // padded extents of the returned real grids: rows M + P - 1, row pitch >= M + P - 1
};

__device__ __forceinline__ double se_wrap(double x, double L) { return x - L * floor(x / L); }

// One thread per particle: cell keys and the rank inside each cell (atomic counter).
__global__ void k_keys(SeConst c, GatherGeom g, const double *__restrict__ pos, int *__restrict__ key_r, int *__restrict__ rank_r,
                       int *__restrict__ cnt_r, int *__restrict__ key_s, int *__restrict__ rank_s, int *__restrict__ cnt_s,
                       int *__restrict__ key_g, int *__restrict__ rank_g, int *__restrict__ cnt_g)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= c.N) return;
    int cc[3], n0[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        double xw;
        const double u = se_grid_coord(c, pos + 3 * (size_t)i, d, &xw);
        cc[d] = se_mod((int)floor(xw / c.hr), c.ncr);                 // sheared: cells in the fractional coordinate (xw = t L)
        n0[d] = se_mod(se_support_start(u, c.P), c.M);
    }
    const int kr = (cc[0] * c.ncr + cc[1]) * c.ncr + cc[2];
    const int ks = (n0[0] * c.NBY + n0[1] / SE_TILE_Y) * c.NBZ + n0[2] / SE_TILE_Z;
    key_r[i] = kr;
    key_s[i] = ks;
    rank_r[i] = atomicAdd(&cnt_r[kr], 1);
    rank_s[i] = atomicAdd(&cnt_s[ks], 1);
    // gather order: (y,z) tile of the support origin major, starting plane minor
    const int kg = ((n0[1] / g.TY) * g.NTZ + n0[2] / g.TZ) * c.M + n0[0];
    key_g[i] = kg;
    rank_g[i] = atomicAdd(&cnt_g[kg], 1);
}

// ---- exclusive prefix sum over n ints (three small kernels; n up to a few million) ----
#define SCAN_THREADS 256
#define SCAN_ITEMS 8
#define SCAN_BLOCK (SCAN_THREADS * SCAN_ITEMS)

__device__ __forceinline__ int block_exclusive_scan(int v, int *total)
{
    __shared__ int wsum[SCAN_THREADS / 32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) wsum[w] = inc;
    __syncthreads();
    if (w == 0) {
        int s = lane < SCAN_THREADS / 32 ? wsum[lane] : 0;
#pragma unroll
        for (int o = 1; o < SCAN_THREADS / 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, s, o);
            if (lane >= o) s += t;
        }
        if (lane < SCAN_THREADS / 32) wsum[lane] = s;
    }
    __syncthreads();
    const int base = w ? wsum[w - 1] : 0;
    *total = wsum[SCAN_THREADS / 32 - 1];
    __syncthreads();
    return base + inc - v;
}

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_local(const int *__restrict__ in, int *__restrict__ out,
                                                            int *__restrict__ bsum, int n)
{
    const int base = blockIdx.x * SCAN_BLOCK + threadIdx.x * SCAN_ITEMS;
    int v[SCAN_ITEMS], s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) { v[k] = (base + k < n) ? in[base + k] : 0; s += v[k]; }
    int total;
    int off = block_exclusive_scan(s, &total);
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) { if (base + k < n) out[base + k] = off; off += v[k]; }
    if (threadIdx.x == 0) bsum[blockIdx.x] = total;
}

// Second pass of the scan.  The three count arrays are concatenated, each followed by one zero pad element:
//   [cnt_r (n1-1) 0 | cnt_s (n2-n1-1) 0 | cnt_g ... 0],  every array summing to N,
// so ONE exclusive scan gives all three start tables, each with its sentinel (= N) in the pad slot, after
// subtracting N (2N) from the second (third) table.  Each block adds the totals of the blocks before it.
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_add(int *__restrict__ out, const int *__restrict__ bsum, int n,
                                                          int n1, int n2, int N)
{
    __shared__ int red[SCAN_THREADS / 32];
    int part = 0;
    for (int b = threadIdx.x; b < blockIdx.x; b += SCAN_THREADS) part += bsum[b];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = part;
    __syncthreads();
    int add = 0;
#pragma unroll
    for (int k = 0; k < SCAN_THREADS / 32; ++k) add += red[k];
    const int base = blockIdx.x * SCAN_BLOCK + threadIdx.x * SCAN_ITEMS;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        const int q = base + k;
        if (q < n) out[q] += add - (q >= n1 ? N : 0) - (q >= n2 ? N : 0);
    }
}

#define SCATTER_PART 64             // particles per CTA
#define SCATTER_THREADS (3 * SCATTER_PART)
// Three threads per particle, one per axis: write the real-space packed copy (cell order), the spreading record (tile
// order) and the gather record (gather order) with the per-axis Gaussian tables (Eq. 41 in physical coordinates; the
// paper's fast Gaussian gridding, Eq. 47, is replaced by P direct exponentials per axis, done once here).
// The record is built in shared memory (one row per particle, odd row pitch) and copied out by whole warps, contiguous
// doubles at a time: per-thread stores of whole records were the whole cost of a1.
__global__ void __launch_bounds__(SCATTER_THREADS)
k_scatter(SeConst c, const double *__restrict__ pos, const double *__restrict__ radii,
          const double *__restrict__ F, const double *__restrict__ T, const double *__restrict__ S,
          const double *__restrict__ s_in,      // pressure moments (a9) or NULL
          const int *__restrict__ key_r, const int *__restrict__ rank_r, const int *__restrict__ start_r,
          const int *__restrict__ key_s, const int *__restrict__ rank_s, const int *__restrict__ start_s,
          const int *__restrict__ key_g, const int *__restrict__ rank_g, const int *__restrict__ start_g,
          double *__restrict__ grecs, double4 *__restrict__ rs_pos, double *__restrict__ rs_mom, int *__restrict__ rs_orig,
          double *__restrict__ recs, int2 *__restrict__ dst_rs)   // dst_rs[i] = (cell-order index, record index)
{
    extern __shared__ __align__(16) double sc_rows[];          // [SCATTER_PART][(rec_stride + P) | 1] then int dst[2][SCATTER_PART]
    const int P = c.P, pitch = (c.rec_stride + P) | 1;          // a row: the spreading record, then gx dx (gather record only)
    int *sc_dst = reinterpret_cast<int *>(sc_rows + SCATTER_PART * pitch), *sc_dg = sc_dst + SCATTER_PART;
    const int pl = threadIdx.x / 3, d = threadIdx.x - 3 * pl;   // local particle, axis
    const int i = blockIdx.x * SCATTER_PART + pl;
    if (d == 0) sc_dst[pl] = -1;
    if (i < c.N) {
        const size_t i3 = 3 * (size_t)i, i5 = 5 * (size_t)i;
        double *r = sc_rows + pl * pitch, *gxd = r + c.rec_stride;
        const int dr = start_r[key_r[i]] + rank_r[i];
        // this thread's axis: wrapped coordinate, support start, Gaussian table
        double xw;
        const double u = se_grid_coord(c, pos + i3, d, &xw), al = c.alpha;
        if (c.gamma != 0.0 && d == 0) {                     // real-space copy: a physical position, x = L (t1 + gamma t2)
            double yw;
            se_grid_coord(c, pos + i3, 1, &yw);
            reinterpret_cast<double *>(rs_pos + dr)[0] = xw + c.gamma * yw;
        } else reinterpret_cast<double *>(rs_pos + dr)[d] = xw;
        const int n0 = se_support_start(u, P);
        r[REC_D0 + d] = ((double)n0 - u) * c.Delta;
        reinterpret_cast<int *>(r)[d == 0 ? 2 : d - 1] = se_mod(n0, c.M);            // int2 (y0w, z0w), int2 (x0w, orig)
        double *g = r + SE_REC_HDR + d * P;
        for (int k = 0; k < P; ++k) {
            const double dk = ((double)(n0 + k) - u) * c.Delta;
            const double e = exp(-al * dk * dk);
            g[k] = d == 0 ? c.gnorm * e : e;
            if (d == 0) gxd[k] = g[k] * dk;                     // gx dx of the gather record
        }
        if (d == 0) {
            const double a = radii[i];
            reinterpret_cast<double *>(rs_pos + dr)[3] = a;
            // F == NULL: positions only (se_plan_set_positions); the moments are filled in later by k_moments
            double f[3] = { 0.0, 0.0, 0.0 }, t[3] = { 0.0, 0.0, 0.0 }, s[5] = { 0.0, 0.0, 0.0, 0.0, 0.0 };
            if (F) {
                f[0] = F[i3]; f[1] = F[i3 + 1]; f[2] = F[i3 + 2]; t[0] = T[i3]; t[1] = T[i3 + 1]; t[2] = T[i3 + 2];
                s[0] = S[i5]; s[1] = S[i5 + 1]; s[2] = S[i5 + 2]; s[3] = S[i5 + 3]; s[4] = S[i5 + 4];
            }
            // real-space copy
            double *m = rs_mom + 12 * (size_t)dr;
            m[0] = f[0]; m[1] = f[1]; m[2] = f[2]; m[3] = t[0]; m[4] = t[1]; m[5] = t[2];
            const double sp = s_in ? s_in[i] : 0.0;
            m[6] = s[0]; m[7] = s[1]; m[8] = s[2]; m[9] = s[3]; m[10] = s[4]; m[11] = sp;
            rs_orig[dr] = i;
            // spreading / gather records
            const int ds = start_s[key_s[i]] + rank_s[i];
            dst_rs[i] = make_int2(dr, ds);
            sc_dst[pl] = ds;
            sc_dg[pl] = start_g[key_g[i]] + rank_g[i];
            const double cF = a * a / 6.0, cS = a * a / 10.0;
            if (c.rec_stride > SE_REC_HDR + 3 * P) r[SE_REC_HDR + 3 * P] = 0.0;
            reinterpret_cast<int *>(r)[3] = i;
            if (c.gamma == 0.0) {
                r[REC_POLY] = 1.0 - 6.0 * al * cF;
                r[REC_POLY + 2] = 2.0 * al * (1.0 - 10.0 * al * cS);
            } else {                                        // metric trace 3 + gamma^2 (Eq. 48); the anisotropic S term is separate (k_spread)
                const double trM = 3.0 + c.gamma * c.gamma;
                r[REC_POLY] = 1.0 - 2.0 * al * trM * cF;
                r[REC_POLY + 2] = 2.0 * al * (1.0 - 2.0 * al * trM * cS);
            }
            r[REC_POLY + 1] = 4.0 * al * al * cF;
            r[REC_POLY + 3] = 8.0 * al * al * al * cS;
            r[REC_F] = f[0]; r[REC_F + 1] = f[1]; r[REC_F + 2] = f[2];
            r[REC_T] = t[0]; r[REC_T + 1] = t[1]; r[REC_T + 2] = t[2];
            r[REC_S] = s[0]; r[REC_S + 1] = s[1]; r[REC_S + 2] = s[2]; r[REC_S + 3] = s[3]; r[REC_S + 4] = s[4];
            r[REC_S + 5] = -(s[0] + s[3]);
            r[REC_CF] = cF; r[REC_CS] = cS; r[REC_SP] = sp;
        }
    }
    __syncthreads();
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int PP = se_grec_pp(P), gstride = c.grec_stride;
    for (int rr = w; rr < SCATTER_PART; rr += SCATTER_THREADS / 32) {
        const int ds = sc_dst[rr];
        if (ds < 0) continue;
        const double *__restrict__ src = sc_rows + rr * pitch;
        double *__restrict__ dst = recs + (size_t)ds * c.rec_stride;
        for (int q = lane; q < c.rec_stride; q += 32) dst[q] = src[q];
        double *__restrict__ dg = grecs + (size_t)sc_dg[rr] * gstride;
        for (int q = lane; q < gstride; q += 32) {
            double v;
            if (q < 2) v = src[q];
            else if (q < 4) v = src[REC_D0 + q - 1];
            else if (q < 4 + 2 * PP) { const int ax = (q - 4) / PP, k = (q - 4) - ax * PP; v = k < P ? src[SE_REC_HDR + (ax + 1) * P + k] : 0.0; }
            else { const int e = q - 4 - 2 * PP; v = (e & 1) ? src[c.rec_stride + (e >> 1)] : src[SE_REC_HDR + (e >> 1)]; }
            dg[q] = v;
        }
    }
}

// Positions unchanged since se_plan_set_positions: only the moments of the spreading records and of the real-space
// copy are refreshed (the sorts, indices and Gaussian tables, and the gather records, are reused).
__global__ void k_moments(SeConst c, const double *__restrict__ F, const double *__restrict__ T, const double *__restrict__ S,
                          const double *__restrict__ s_in, const int2 *__restrict__ dst_rs, double *__restrict__ rs_mom,
                          double *__restrict__ recs)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= c.N) return;
    const size_t i3 = 3 * (size_t)i, i5 = 5 * (size_t)i;
    const int2 d = dst_rs[i];
    const double sp = s_in ? s_in[i] : 0.0;
    double *m = rs_mom + 12 * (size_t)d.x;
    const double f0 = F[i3], f1 = F[i3 + 1], f2 = F[i3 + 2], t0 = T[i3], t1 = T[i3 + 1], t2 = T[i3 + 2];
    const double s0 = S[i5], s1 = S[i5 + 1], s2 = S[i5 + 2], s3 = S[i5 + 3], s4 = S[i5 + 4];
    m[0] = f0; m[1] = f1; m[2] = f2; m[3] = t0; m[4] = t1; m[5] = t2;
    m[6] = s0; m[7] = s1; m[8] = s2; m[9] = s3; m[10] = s4; m[11] = sp;
    if (!recs) return;                                  // batch: the real-space copy only
    double *r = recs + (size_t)d.y * c.rec_stride;
    r[REC_F] = f0; r[REC_F + 1] = f1; r[REC_F + 2] = f2;
    r[REC_T] = t0; r[REC_T + 1] = t1; r[REC_T + 2] = t2;
    r[REC_S] = s0; r[REC_S + 1] = s1; r[REC_S + 2] = s2; r[REC_S + 3] = s3; r[REC_S + 4] = s4; r[REC_S + 5] = -(s0 + s3);
    r[REC_SP] = sp;
}

static inline size_t scatter_smem_bytes(int P)
{
    return (size_t)SCATTER_PART * ((se_rec_stride(P) + P) | 1) * 8 + 2 * SCATTER_PART * 4;
}
