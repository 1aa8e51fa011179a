// Common machinery of the two particle<->grid kernels (a3 spreading, a7 gather): the "register sweep".
//
// A thread owns one grid column (y,z) and sweeps along x, the slowest grid axis; a warp owns a
// 4 (y) x 8 (z) patch of columns so that its global rows are 64 bytes.  The particles whose P^3 support
// STARTS at plane p and overlaps the patch are found through the plane-thin tile bins (x-plane, y/4, z/8)
// of the counting sort (a1): for a patch they are a handful of contiguous record ranges per plane.
// Each warp stages those records one plane ahead into its own shared-memory slot with bulk asynchronous
// copies (TMA, cp.async.bulk + mbarrier), so the per-particle arithmetic never waits on global memory.
// Slots hold SWEEP_CAP records; the rare excess is read straight from global memory.
#pragma once
#include "se_common.cuh"

#define SWEEP_WARPS 4
#define SWEEP_CAP 8
#ifndef SWEEP_MIN_BLOCKS
#define SWEEP_MIN_BLOCKS 3             // resident CTAs per SM the register allocation aims at
#endif

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
// suspend-time hint of try_wait: the waiting warp sleeps in hardware instead of polling shared memory
#ifndef SE_WAIT_HINT_NS
#define SE_WAIT_HINT_NS 20000u
#endif
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile("{\n"
                 ".reg .pred P1;\n"
                 "LAB_WAIT:\n"
                 "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1, %2;\n"
                 "@P1 bra DONE;\n"
                 "bra LAB_WAIT;\n"
                 "DONE:\n"
                 "}" ::"r"(bar), "r"(parity), "r"(SE_WAIT_HINT_NS) : "memory");
}

// Per-lane description of the candidate ranges of a patch: lane r < nr owns the bins
// [rowoff, rowoff + len) of every plane (add plane * NBY * NBZ), contiguous in the sorted records.
struct SweepRanges { int nr, rowoff, len; };

// Bins that can hold particles covering the patch with first column (Y0, Z0):
// y0w in [Y0-P+1, Y0+3], z0w in [Z0-P+1, Z0+7] (mod M).  At most 2 row ranges x 2 bin ranges.
template <int P>
__device__ __forceinline__ SweepRanges sweep_ranges(const SeConst &c, int Y0, int Z0, int lane)
{
    const int M = c.M;
    int by_lo[2], by_hi[2], bz_lo[2], bz_hi[2], nyr, nzr;
    const int ylo = Y0 - (P - 1), yhi = min(Y0 + SE_TILE_Y - 1, M - 1);
    if (yhi - ylo + 1 >= M) { nyr = 1; by_lo[0] = 0; by_hi[0] = c.NBY - 1; }
    else if (ylo < 0) {
        nyr = 2; by_lo[0] = 0; by_hi[0] = yhi / SE_TILE_Y; by_lo[1] = (ylo + M) / SE_TILE_Y; by_hi[1] = c.NBY - 1;
        if (by_lo[1] <= by_hi[0]) { nyr = 1; by_hi[0] = c.NBY - 1; }
    } else { nyr = 1; by_lo[0] = ylo / SE_TILE_Y; by_hi[0] = yhi / SE_TILE_Y; }
    const int zlo = Z0 - (P - 1), zhi = min(Z0 + SE_TILE_Z - 1, M - 1);
    if (zhi - zlo + 1 >= M) { nzr = 1; bz_lo[0] = 0; bz_hi[0] = c.NBZ - 1; }
    else if (zlo < 0) {
        nzr = 2; bz_lo[0] = 0; bz_hi[0] = zhi / SE_TILE_Z; bz_lo[1] = (zlo + M) / SE_TILE_Z; bz_hi[1] = c.NBZ - 1;
        if (bz_lo[1] <= bz_hi[0]) { nzr = 1; bz_hi[0] = c.NBZ - 1; }
    } else { nzr = 1; bz_lo[0] = zlo / SE_TILE_Z; bz_hi[0] = zhi / SE_TILE_Z; }
    const int rows0 = by_hi[0] - by_lo[0] + 1, rows = rows0 + (nyr == 2 ? by_hi[1] - by_lo[1] + 1 : 0);
    SweepRanges r;
    r.nr = rows * nzr;                               // <= 16 for P <= 24 (host checks)
    const int row = lane / nzr, zr = lane - row * nzr;
    const int by = row < rows0 ? by_lo[0] + row : by_lo[nyr - 1] + (row - rows0);
    r.rowoff = by * c.NBZ + bz_lo[zr];
    r.len = bz_hi[zr] - bz_lo[zr] + 1;
    if (lane >= r.nr) { r.rowoff = 0; r.len = 0; }
    return r;
}

// Candidate list of one plane, as seen by a warp: lane r holds the first record js and the exclusive
// offset off of its range; n is the total (warp-uniform).
struct SweepList { int js, cnt, off, n; };

// Raw (first record, one-past-last record) of this lane's range in the plane whose bins start at binbase.
// Kept apart from sweep_scan so that the loads can be issued a whole plane before their use.
__device__ __forceinline__ int2 sweep_load(const SweepRanges &rg, const int *__restrict__ start_s, int binbase, int lane)
{
    int2 r = make_int2(0, 0);
    if (lane < rg.nr) {
        r.x = start_s[binbase + rg.rowoff];
        r.y = start_s[binbase + rg.rowoff + rg.len];
    }
    return r;
}

__device__ __forceinline__ SweepList sweep_scan(int2 raw, int lane)
{
    const int cnt = raw.y - raw.x;
    int inc = cnt;
#pragma unroll
    for (int o = 1; o < 16; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    SweepList l;
    l.js = raw.x;
    l.cnt = cnt;
    l.off = inc - cnt;
    l.n = __shfl_sync(0xffffffffu, inc, 15);         // ranges live in lanes 0..15
    return l;
}

// Issue the bulk copies of the first min(n, CAP) records of list l into the slot at shared address `slot`.
__device__ __forceinline__ void sweep_stage(const SweepList &l, const double *__restrict__ recs, int rec_stride,
                                            uint32_t slot, uint32_t bar, int lane)
{
    const uint32_t rb = (uint32_t)rec_stride * 8u;
    if (l.n > 0) {
        if (lane == 0) mbar_expect_tx(bar, (uint32_t)min(l.n, SWEEP_CAP) * rb);
        __syncwarp();
        if (l.cnt > 0 && l.off < SWEEP_CAP) {
            const int nc = min(l.cnt, SWEEP_CAP - l.off);
            bulk_g2s(slot + (uint32_t)l.off * rb, recs + (size_t)l.js * rec_stride, (uint32_t)nc * rb, bar);
        }
    }
}

// Record index of candidate ci >= CAP of list l (warp-uniform ci).
__device__ __forceinline__ int sweep_overflow_index(const SweepList &l, int ci)
{
    const unsigned m = __ballot_sync(0xffffffffu, l.cnt > 0 && l.off <= ci);
    const int r = 31 - __clz((int)m);
    return __shfl_sync(0xffffffffu, l.js, r) + ci - __shfl_sync(0xffffffffu, l.off, r);
}
