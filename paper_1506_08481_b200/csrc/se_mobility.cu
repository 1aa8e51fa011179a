// C-ABI of the far-field mobility product (include/se_mobility.h): plan, orchestration, cuFFT calls.
// Hand-written CUDA for sm_100a; cuFFT is used only for grids that are not powers of two (batched 3-D real plans, a4 / a6).
#include "../../include/se_mobility.h"

#include <cuda_runtime.h>
#include <cufft.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <cmath>
#include <mutex>

#include "se_common.cuh"
#include "se_sort.cuh"
#include "se_real.cuh"
#include "se_spread.cuh"
#include "se_kspace.cuh"
#include "se_xfft.cuh"
#include "se_xyfft.cuh"
#include "se_zfft.cuh"
#include "se_gather.cuh"
#include "se_blocks.cuh"

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

struct se_plan {
    SeConst c;
    double m;                      // Gaussian shape parameter
    unsigned flags;
    int debug_stop;
    int last_launches;
    size_t bytes;
    char err[256];
    // device buffers
    double *d_radii;
    double a2min, a2max;           // range of a_i^2 (reference radii of the self-image blocks)
    double *d_blockW;              // [3][11][11] lattice sums of se_self_image_blocks at the reference radii
    int *d_key_r, *d_rank_r, *d_cnt_r, *d_start_r;
    int *d_key_s, *d_rank_s, *d_cnt_s, *d_start_s;
    int *d_key_g, *d_rank_g, *d_cnt_g, *d_start_g;
    double *d_grecs;               // gather records [N][grec_stride], gather order
    int2 *d_dst_rs;                // per particle (caller order): index in cell order, record index
    bool have_positions;           // a1 was run by se_plan_set_positions and is reused while pos == NULL
    int *d_cnt_all, *d_start_all;  // the three count / start tables, concatenated (one pad element after each)
    int *d_bsum;
    int ncell_r, ncell_s, ncell_g, ncell_all;
    int ncell_r_alloc;             // cells the count / start tables were laid out for (strain 0)
    double r_c;
    cudaStream_t side;             // the real-space sum runs here, beside the wave-space pipeline
    cudaEvent_t ev_fork, ev_join;
    bool have_side;
    int real_side_ctas;            // grid of k_real when it runs beside the wave pipeline (0 = one CTA per cell)
    int real_overlap;              // SE_OPT_REAL_OVERLAP
    int sms;                       // multiprocessors of the plan's device (grid sizing)
    GatherGeom gg;                 // ring gather geometry (spreading's segments are in c.nseg, c.seg_len)
    CUtensorMap tmap, tmap_p;      // TMA descriptors of the six returned grids / of the pressure grid (se_gather.cuh)
    size_t gather_smem;
    int gWY, gWZ;                  // TMA box of the gather: rows, columns of the haloed tile
    size_t Gp;                     // doubles per padded returned grid: M * MYp * MZp
    bool real_p_padded;            // d_real_p currently holds the returned pressure grid (padded layout)
    double4 *d_rs_pos;
    double *d_rs_mom;
    int *d_rs_orig;
    double *d_recs;
    double *d_real;                // [6][M][MYp][MZp] returned grids with periodic halo; the first 3 M^3 doubles double as the spread grids H
    double2 *d_Hk;                 // [3][M][M][M/2+1]
    double2 *d_Gk;                 // [6][M][M][M/2+1]
    double *d_out_real;            // [N][12] real-space part in caller order (slot 11: pressure, a9)
    // cached pairs of the real-space sum (se_real.cuh), built by se_plan_set_positions when SE_OPT_PAIR_CACHE is on
    int pair_cache;                // SE_OPT_PAIR_CACHE
    bool have_pairs;               // the list below belongs to the cached configuration
    int *d_pair_start, *d_pair_cursor, *d_pair_bsum, *d_pj;   // [N+1] row starts (count, then scanned), [N], scan scratch, partners
    double *d_pd;                  // [pairs][PAIR_F] in row-local structure-of-arrays form
    size_t pair_cap, npairs;
    const double *ext_out_real;    // far_mobility_apply_batch: real-space part already computed (k_real is skipped)
    double *d_mom_b, *d_out_real_b; // batch: moments in cell order and real-space results, [nrhs][N][12]
    int batch_cap;                 // right-hand sides the batch buffers hold
    // compressible extension (a9): allocated by the first apply that passes s_in or s_out
    double *d_real_p;              // [M][MYp][MZp]: scalar spread grid Hs (first M^3 doubles), then the returned pressure grid p~ (padded)
    double2 *d_Hk_s, *d_Gk_p;      // their spectra
    double *d_pmom;                // [N][12] gathered pressure sums
    cufftHandle fft_fwd1, fft_inv1;
    bool have_comp;
    double *d_moments;             // [N][24] gathered wave-space sums in caller order
    double *d_wrecs;               // wave-space variant: spreading records of the current pass [N][rec_stride]
    double2 *d_Wk;                 // wave-space variant: 24 half spectra (cuFFT layout), transformed in place by k_kspace_wave
    double *d_wmom;                // wave-space variant: gathered sums [N][96] (four batches of six returned grids)
    int grid_fp32;                 // SE_OPT_GRID_FP32: mesh (H, spectra, transforms, returned grids) in single precision
    float *d_realf;                // fp32 mesh: [7][M^3] real grids (6 + pressure)
    float2 *d_Hkf, *d_Gkf;         // fp32 mesh: [4][Gc] and [7][Gc] half spectra (3 + pressure moment, 6 + pressure)
    cufftHandle fftf_fwd, fftf_inv, fftf_fwd1, fftf_inv1;
    bool have_f32;
    int size_variant;              // SE_OPT_SIZE_VARIANT: 0 hybrid (default), 1 real-space, 2 wave-space size terms (Sec. 3.2)
    // host-API staging
    double *d_io;                  // pos3 F3 T3 S5 U3 W3 E5 = 25 N doubles
    cufftHandle fft_fwd, fft_inv;  // 3-D batched plans (unfused path), made when first needed
    bool have_fwd, have_inv, have_fft1;
    bool have_zt;
    int lM;
    double2 *d_wtab;               // exp(-2 pi i q / M), q < M
    double *d_etab;                // exp(-(1 - eta_se) k_q^2 / 4 xi^2), q < M (k-space pass of se_xyfft.cuh)
    // plan-owned CUDA graph of the whole product (SE_OPT_GRAPH): replayed while the same pointers, flags and options come back
    int use_graph;                 // 0 off, 1 on (default: on for M <= 128, where launch latency dominates)
    bool have_graph;
    cudaGraphExec_t gexec;
    const void *gkey[10];          // pos F T S s_in U Omega E s_out stream
    unsigned gflags;
    long gepoch, epoch;            // epoch: bumped by every setter that changes what apply_impl enqueues
    int graph_launches;
    bool warmed[2];                // a plain apply (lazy allocations done) was made: [0] without, [1] with the a9 arguments
    int yz_fused;                  // SE_OPT_YZ_FUSED: (y,z) transforms in one cluster kernel per direction (se_zfft.cuh)
    size_t fft_bytes;
    cudaEvent_t ev[SE_NUM_STAGES + 1];
    bool have_events, timed;
};

static se_status fail(se_plan *p, se_status st, const char *what, const char *detail)
{
    if (p) snprintf(p->err, sizeof(p->err), "%s: %s", what, detail ? detail : "");
    return st;
}

#define CUDA_TRY(p, call)                                                              \
    do {                                                                               \
        cudaError_t e_ = (call);                                                       \
        if (e_ != cudaSuccess) return fail((p), SE_ERR_CUDA, #call, cudaGetErrorString(e_)); \
    } while (0)

#define CUFFT_TRY(p, call)                                                             \
    do {                                                                               \
        cufftResult r_ = (call);                                                       \
        if (r_ != CUFFT_SUCCESS) {                                                     \
            char b_[32]; snprintf(b_, sizeof(b_), "cufftResult %d", (int)r_);          \
            return fail((p), SE_ERR_CUFFT, #call, b_);                                 \
        }                                                                              \
    } while (0)

template <typename Tp>
static se_status dev_alloc(se_plan *p, Tp **ptr, size_t count)
{
    *ptr = nullptr;
    const size_t nb = count * sizeof(Tp);
    cudaError_t e = cudaMalloc((void **)ptr, nb ? nb : 16);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(p, e == cudaErrorMemoryAllocation ? SE_ERR_ALLOC : SE_ERR_CUDA, "cudaMalloc", cudaGetErrorString(e));
    }
    p->bytes += nb;
    return SE_OK;
}

// Derived constants (oracle step 1 restated independently): Delta = L/M,
// eta_se = (P Delta xi/m)^2 [= theta L^2/4pi^2 of Eq. 46], alpha = 2 xi^2/eta_se (Eq. 41).
static void derive_constants(se_plan *p)
{
    SeConst &c = p->c;
    c.MoverL = (double)c.M / c.L;
    c.Delta = c.L / c.M;
    const double t = c.P * c.Delta * c.xi / p->m;
    c.eta_se = t * t;
    c.alpha = 2.0 * c.xi * c.xi / c.eta_se;
    c.gnorm = pow(c.alpha / M_PI, 1.5);
    c.q = 2.0 * c.xi / sqrt(M_PI);
    c.x2 = c.xi * c.xi; c.x4 = c.x2 * c.x2; c.x6 = c.x4 * c.x2; c.x8 = c.x4 * c.x4; c.x10 = c.x8 * c.x2; c.x12 = c.x6 * c.x6;
    c.k0 = 1.0 / (8.0 * M_PI * c.eta0);
    const double V = c.L * c.L * c.L;
    c.D3 = c.Delta * c.Delta * c.Delta;
    c.scale0 = c.D3 / (c.eta0 * V);
    c.inv4xi2 = 1.0 / (4.0 * c.xi * c.xi);
    c.dec = (1.0 - c.eta_se) / (4.0 * c.xi * c.xi);
    c.twopiL = 2.0 * M_PI / c.L;
    c.invL = 1.0 / c.L;
}

// Real-space cell grid: cells of edge >= r_c in the cubic box; on the sheared lattice the cells live in the fractional
// coordinate, where a separation r < r_c has |dt1| <= r_c sqrt(1 + gamma^2)/L, |dt2|, |dt3| <= r_c/L.
static void choose_real_cells(se_plan *p)
{
    SeConst &c = p->c;
    int ncr = (int)floor(c.L / (p->r_c * sqrt(1.0 + c.gamma * c.gamma)));
    if (ncr < 3) ncr = 1;
    if (ncr > 1024) ncr = 1024;
    c.ncr = ncr;
    c.hr = c.L / ncr;
    p->ncell_r = ncr * ncr * ncr;
}

// Sweep segments along x.  Spreading re-processes the particles of the P-1 planes before a segment, the
// gather re-reads P-1 planes per segment, so segments are long; they exist only to fill the machine:
// aim at >= 16 resident warps per SM, segments no shorter than 32 planes.
static void choose_segments(se_plan *p, int spread_segments, int gather_segments)
{
    SeConst &c = p->c;
    const int npatch = c.NBY * c.NBZ, M = c.M;
    int ns = spread_segments;
    if (ns <= 0) {
        const int slots = p->sms * 3 * SWEEP_WARPS;          // warps the device holds at once (three CTAs per SM at P = 12)
        if (npatch < slots) {
            // small grids: the sweep of a patch is a serial chain of planes and the machine is not full -- as many segments
            // as fit in one round, down to two planes each (c1: 0.029 -> 0.012 ms, c2: 0.041 -> 0.025 ms)
            ns = slots / npatch;
            if (ns > M / 2) ns = M / 2;
        } else {
            // large grids: >= 16 warps per SM, segments no shorter than 32 planes
            const int maxseg = M / 32 > 1 ? M / 32 : 1;
            ns = (p->sms * 16 + npatch - 1) / npatch;
            if (ns > maxseg) ns = maxseg;
        }
    }
    if (ns > M) ns = M;
    if (ns < 1) ns = 1;
    c.seg_len = (M + ns - 1) / ns;
    c.nseg = (M + c.seg_len - 1) / c.seg_len;
    (void)gather_segments;                        // the gather balances its own work (GatherWalk, se_gather.cuh)
}

#ifndef FOR_EACH_P                 // a development build may define a shorter list on the command line
#define FOR_EACH_P(X) \
    X(2) X(3) X(4) X(5) X(6) X(7) X(8) X(9) X(10) X(11) X(12) X(13) X(14) X(15) X(16) X(17) X(18) X(19) X(20) X(21) X(22) X(23) X(24)
#endif

// Ring gather geometry (se_gather.cuh): tile, ring and box are compile-time functions of P (GatherTraits); the padded
// extents of the returned grids follow from M and P.
static bool choose_gather_geometry(se_plan *p)
{
    const int M = p->c.M, P = p->c.P;
    GatherGeom &g = p->gg;
    switch (P) {
#define X(v) case v: g.TY = GatherTraits<v>::TY; g.TZ = GatherTraits<v>::TZ; p->gWY = GatherTraits<v>::WY; p->gWZ = GatherTraits<v>::WZ; \
                     p->gather_smem = GatherTraits<v>::SMEM; break;
        FOR_EACH_P(X)
#undef X
        default: return false;
    }
    g.NTY = (M + g.TY - 1) / g.TY; g.NTZ = (M + g.TZ - 1) / g.TZ;
    g.MYp = M + P - 1;
    g.MZp = (M + P + 3) & ~3;                          // >= M + P, rows start on 32-byte boundaries
    g.nseg = 1; g.seg_len = M;
    p->Gp = (size_t)M * g.MYp * g.MZp;
    return p->gather_smem <= 227 * 1024;
}

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-kernel, process-wide limit: it is set to the device's opt-in
// maximum (minus the kernel's static shared memory), never to one plan's own need, so that a later plan with a smaller
// requirement cannot lower the limit an earlier plan still relies on.
template <typename K>
static cudaError_t raise_smem_limit(K kernel)
{
    int dev = 0, optin = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    cudaFuncAttributes fa;
    if (e == cudaSuccess) e = cudaFuncGetAttributes(&fa, kernel);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, optin - (int)fa.sharedSizeBytes);
    return e;
}

static cudaError_t dispatch_prepare(int P);

extern "C" const char *se_version(void) { return "se_mobility 0.2 (sm_100a)"; }

extern "C" const char *se_last_error(const se_plan *plan) { return plan ? plan->err : "null plan"; }

extern "C" se_status se_plan_destroy(se_plan *p)
{
    if (!p) return SE_OK;
    cudaFree(p->d_radii); cudaFree(p->d_blockW);
    cudaFree(p->d_pair_start); cudaFree(p->d_pair_cursor); cudaFree(p->d_pair_bsum); cudaFree(p->d_pj); cudaFree(p->d_pd);
    cudaFree(p->d_key_r); cudaFree(p->d_rank_r); cudaFree(p->d_key_s); cudaFree(p->d_rank_s);
    cudaFree(p->d_key_g); cudaFree(p->d_rank_g); cudaFree(p->d_grecs);
    cudaFree(p->d_cnt_all); cudaFree(p->d_start_all); cudaFree(p->d_dst_rs);
    if (p->have_graph) cudaGraphExecDestroy(p->gexec);
    if (p->have_side) { cudaStreamDestroy(p->side); cudaEventDestroy(p->ev_fork); cudaEventDestroy(p->ev_join); }
    cudaFree(p->d_bsum);
    cudaFree(p->d_rs_pos); cudaFree(p->d_rs_mom); cudaFree(p->d_rs_orig); cudaFree(p->d_recs);
    cudaFree(p->d_wrecs); cudaFree(p->d_Wk); cudaFree(p->d_wmom);
    cudaFree(p->d_realf); cudaFree(p->d_Hkf); cudaFree(p->d_Gkf);
    if (p->have_f32) { cufftDestroy(p->fftf_fwd); cufftDestroy(p->fftf_inv); cufftDestroy(p->fftf_fwd1); cufftDestroy(p->fftf_inv1); }
    cudaFree(p->d_real); cudaFree(p->d_Hk); cudaFree(p->d_Gk);
    cudaFree(p->d_out_real); cudaFree(p->d_moments); cudaFree(p->d_io); cudaFree(p->d_mom_b); cudaFree(p->d_out_real_b);
    if (p->have_comp) {
        cudaFree(p->d_real_p); cudaFree(p->d_Hk_s); cudaFree(p->d_Gk_p); cudaFree(p->d_pmom);
        if (p->have_fft1) { cufftDestroy(p->fft_fwd1); cufftDestroy(p->fft_inv1); }
    }
    cudaFree(p->d_wtab); cudaFree(p->d_etab);
    if (p->have_fwd) cufftDestroy(p->fft_fwd);
    if (p->have_inv) cufftDestroy(p->fft_inv);
    if (p->have_events) for (int k = 0; k <= SE_NUM_STAGES; ++k) cudaEventDestroy(p->ev[k]);
    cudaGetLastError();
    free(p);
    return SE_OK;
}

// TMA descriptor of nplanes padded grid planes [MYp][MZp] at `base`: 3-D tensor (z, y, plane), box = one haloed tile
// (parts of a box beyond the padded plane are zero-filled; they lie beyond every support).
// The encoder lives in the driver; it is fetched through the runtime so that the library links against cudart only.
static se_status make_tensor_map(se_plan *p, CUtensorMap *map, double *base, int nplanes)
{
    typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) != cudaSuccess || !fn ||
        qr != cudaDriverEntryPointSuccess) {
        cudaGetLastError();
        return fail(p, SE_ERR_CUDA, "cudaGetDriverEntryPoint", "cuTensorMapEncodeTiled");
    }
    const GatherGeom &g = p->gg;
    const cuuint64_t dims[3] = { (cuuint64_t)g.MZp, (cuuint64_t)g.MYp, (cuuint64_t)nplanes };
    const cuuint64_t strides[2] = { (cuuint64_t)g.MZp * 8, (cuuint64_t)g.MYp * g.MZp * 8 };
    const cuuint32_t box[3] = { (cuuint32_t)p->gWZ, (cuuint32_t)p->gWY, 1 };
    const cuuint32_t estr[3] = { 1, 1, 1 };
    const CUresult cr = ((encode_fn)fn)(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, base, dims, strides, box, estr,
                                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                        CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (cr != CUDA_SUCCESS) {
        char b[32]; snprintf(b, sizeof(b), "CUresult %d", (int)cr);
        return fail(p, SE_ERR_CUDA, "cuTensorMapEncodeTiled", b);
    }
    return SE_OK;
}

// Periodic halo of the padded returned grids after cuFFT's 3-D inverse transforms (which fill the M^3 interior only):
// rows / columns M .. M+P-2 repeat 0 .. P-2.  The own z transform (se_zfft.cuh) writes its halo itself.
__global__ void k_halo_fill(double *__restrict__ Rg, int M, int MYp, int MZp, int halo, size_t nplanes)
{
    const size_t per = (size_t)MYp * MZp;
    const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= nplanes * per) return;
    const size_t pl = q / per;
    const int r = (int)(q - pl * per), y = r / MZp, z = r - y * MZp;
    if ((y < M && z < M) || y >= M + halo || z >= M + halo + 1) return;
    Rg[q] = Rg[pl * per + (size_t)(y % M) * MZp + (z % M)];
}

// Batched 3-D cuFFT plans (other grid sizes than powers of two, or flag SE_CUFFT3D): D2Z (3 grids, contiguous) and
// Z2D (6 grids) into the padded layout of the returned grids; `single`: the one-grid plans of the compressible extension.
static se_status ensure_fft3d(se_plan *p, bool single)
{
    if (single ? p->have_fft1 : (p->have_fwd && p->have_inv)) return SE_OK;
    const int M = p->c.M;
    int n3[3] = { M, M, M }, ic[3] = { M, M, M / 2 + 1 }, orl[3] = { M, p->gg.MYp, p->gg.MZp };
    const int idist = M * M * (M / 2 + 1);
    const long long odist = (long long)p->Gp;
    if (odist > 0x7fffffffLL) return fail(p, SE_ERR_UNSUPPORTED, "ensure_fft3d", "grid too large for cuFFT's int distances");
    size_t ws = 0, tot = 0;
    cufftHandle *fw = single ? &p->fft_fwd1 : &p->fft_fwd, *iv = single ? &p->fft_inv1 : &p->fft_inv;
    const int nf = single ? 1 : 3, ni = single ? 1 : 6;
    cufftResult r = cufftCreate(fw);
    bool c1 = (r == CUFFT_SUCCESS), c2 = false;
    if (c1) { r = cufftMakePlanMany(*fw, 3, n3, NULL, 1, 0, NULL, 1, 0, CUFFT_D2Z, nf, &ws); tot += ws; }
    if (r == CUFFT_SUCCESS) { r = cufftCreate(iv); c2 = (r == CUFFT_SUCCESS); }
    if (r == CUFFT_SUCCESS) { r = cufftMakePlanMany(*iv, 3, n3, ic, 1, idist, orl, 1, (int)odist, CUFFT_Z2D, ni, &ws); tot += ws; }
    if (r != CUFFT_SUCCESS) {
        if (c1) cufftDestroy(*fw);
        if (c2) cufftDestroy(*iv);
        return fail(p, r == CUFFT_ALLOC_FAILED ? SE_ERR_ALLOC : SE_ERR_CUFFT, "cufftMakePlanMany", "3-D plans");
    }
    if (single) p->have_fft1 = true; else { p->have_fwd = true; p->have_inv = true; }
    p->fft_bytes += tot;
    p->bytes += tot;
    return SE_OK;
}

static se_status ensure_wtab(se_plan *p);

// Twiddle table exp(-2 pi i q / M), q < M (own z transforms).
static se_status ensure_wtab(se_plan *p)
{
    if (p->d_wtab) return SE_OK;
    const int M = p->c.M;
    double2 *wt = (double2 *)malloc(sizeof(double2) * (size_t)M);
    if (!wt) return fail(p, SE_ERR_ALLOC, "malloc", "twiddle table");
    se_status st = dev_alloc(p, &p->d_wtab, (size_t)M);
    if (st == SE_OK) {
        for (int q = 0; q < M; ++q) { const double a = 2.0 * M_PI * q / M; wt[q].x = cos(a); wt[q].y = -sin(a); }
        if (cudaMemcpy(p->d_wtab, wt, sizeof(double2) * (size_t)M, cudaMemcpyHostToDevice) != cudaSuccess) {
            cudaGetLastError(); cudaFree(p->d_wtab); p->d_wtab = nullptr;
            st = fail(p, SE_ERR_CUDA, "cudaMemcpy", "twiddle table");
        }
    }
    free(wt);
    return st;
}

// Per-axis table of the separable Gaussian factor of the k-space pass; depends on the shape parameter m.
static se_status upload_etab(se_plan *p)
{
    const int M = p->c.M;
    if (!p->d_etab) { se_status st = dev_alloc(p, &p->d_etab, (size_t)M); if (st != SE_OK) return st; }
    double *et = (double *)malloc(sizeof(double) * (size_t)M);
    if (!et) return fail(p, SE_ERR_ALLOC, "malloc", "exp table");
    for (int q = 0; q < M; ++q) {           // sheared lattice: only the deconvolution e^{+eta_se kq^2/4xi^2} is separable (se_xyfft.cuh)
        const double k = p->c.twopiL * (q < M / 2 ? q : q - M);
        et[q] = p->c.gamma == 0.0 ? exp(-p->c.dec * k * k) : exp(p->c.eta_se * p->c.inv4xi2 * k * k);
    }
    const cudaError_t e = cudaMemcpy(p->d_etab, et, sizeof(double) * (size_t)M, cudaMemcpyHostToDevice);
    free(et);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(p, SE_ERR_CUDA, "cudaMemcpy", "exp table"); }
    return SE_OK;
}

// y-batch of k_xmid: 4 columns (64-byte runs), 2 where the compressible variant would not fit the register file
#ifndef XM_YB8
#define XM_YB8 4                   // y-batch for M = 256
#endif
#ifndef XM_YB9
#define XM_YB9 4                   // y-batch for M = 512
#endif
template <int LM, bool COMP> struct XmChoice { static constexpr int YB = LM == 9 ? (COMP ? 2 : XM_YB9) : (LM == 8 && !COMP ? XM_YB8 : 4); };

template <int LM>
static cudaError_t prepare_xy()
{
    cudaError_t e = raise_smem_limit(k_yfft<LM, false>);
    if (e == cudaSuccess) e = raise_smem_limit(k_yfft<LM, true>);
    if (e == cudaSuccess) e = raise_smem_limit(k_xmid<LM, XmChoice<LM, false>::YB, false, false>);
    if (e == cudaSuccess) e = raise_smem_limit(k_xmid<LM, XmChoice<LM, true>::YB, true, false>);
    if (e == cudaSuccess) e = raise_smem_limit(k_xmid<LM, XmChoice<LM, false>::YB, false, true>);
    if (e == cudaSuccess) e = raise_smem_limit(k_xmid<LM, XmChoice<LM, true>::YB, true, true>);
    return e;
}

template <int LM>
static void launch_yfft(cudaStream_t s, double2 *spec, const double2 *wtab, int ngrids, bool inv)
{
    using TR = YfTraits<LM>;
    const size_t nlines = (size_t)ngrids * (TR::M / 2) * TR::M;
    const unsigned nb = (unsigned)((nlines + TR::LPC - 1) / TR::LPC);
    if (inv) k_yfft<LM, true><<<nb, YF_THREADS, TR::SMEM, s>>>(spec, wtab, ngrids);
    else k_yfft<LM, false><<<nb, YF_THREADS, TR::SMEM, s>>>(spec, wtab, ngrids);
}

template <int LM, bool COMP>
static void launch_xmid(const SeConst &c, cudaStream_t s, const double2 *Hk, const double2 *Hsk, double2 *Gk, double2 *Pk,
                        const double2 *wtab, const double *etab)
{
    constexpr int YB = XmChoice<LM, COMP>::YB;
    using TR = XmTraits<LM, YB, COMP>;
    const unsigned nb = (unsigned)((TR::M / 2 + 1) * (TR::M / YB));
    if (c.gamma != 0.0) k_xmid<LM, YB, COMP, true><<<nb, TR::NT, TR::SMEM, s>>>(c, Hk, Hsk, Gk, Pk, wtab, etab);
    else k_xmid<LM, YB, COMP, false><<<nb, TR::NT, TR::SMEM, s>>>(c, Hk, Hsk, Gk, Pk, wtab, etab);
}

#define FOR_EACH_LM(X) X(5) X(6) X(7) X(8) X(9)

// (y,z) transforms by thread-block clusters of M/32 CTAs (se_zfft.cuh); M = 512 needs the non-portable cluster size 16.
template <int LM>
static cudaError_t prepare_yz()
{
    cudaError_t e = raise_smem_limit(k_yz_r2c<LM>);
    if (e == cudaSuccess) e = raise_smem_limit(k_yz_c2r<LM>);
    if (e == cudaSuccess && YzTraits<LM>::CS > 8) {
        e = cudaFuncSetAttribute(k_yz_r2c<LM>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_yz_c2r<LM>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    }
    return e;
}

template <int LM>
static cudaError_t launch_yz(bool inv, cudaStream_t s, int ngrids, const double *H, double2 *spec, double *R, const double2 *wtab,
                             int MYp, int MZp, int halo)
{
    using TR = YzTraits<LM>;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(ngrids * TR::M * TR::CS));
    cfg.blockDim = dim3(TR::NT);
    cfg.dynamicSmemBytes = TR::SMEM;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = TR::CS; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    if (inv) return cudaLaunchKernelEx(&cfg, k_yz_c2r<LM>, (const double2 *)spec, R, wtab, MYp, MZp, halo);
    return cudaLaunchKernelEx(&cfg, k_yz_r2c<LM>, H, spec, wtab);
}

static cudaError_t dispatch_prepare_yz(int lM)
{
    switch (lM) {
#define X(v) case v: return prepare_yz<v>();
        FOR_EACH_LM(X)
#undef X
    }
    return cudaErrorInvalidValue;
}

static cudaError_t dispatch_yz(int lM, bool inv, cudaStream_t s, int ngrids, const double *H, double2 *spec, double *R,
                               const double2 *wtab, int MYp, int MZp, int halo)
{
    switch (lM) {
#define X(v) case v: return launch_yz<v>(inv, s, ngrids, H, spec, R, wtab, MYp, MZp, halo);
        FOR_EACH_LM(X)
#undef X
    }
    return cudaErrorInvalidValue;
}

static cudaError_t dispatch_prepare_xy(int lM)
{
    switch (lM) {
#define X(v) case v: return prepare_xy<v>();
        FOR_EACH_LM(X)
#undef X
    }
    return cudaErrorInvalidValue;
}

static void dispatch_yfft(int lM, cudaStream_t s, double2 *spec, const double2 *wtab, int ngrids, bool inv)
{
    switch (lM) {
#define X(v) case v: launch_yfft<v>(s, spec, wtab, ngrids, inv); break;
        FOR_EACH_LM(X)
#undef X
    }
}

static void dispatch_xmid(int lM, bool comp, const SeConst &c, cudaStream_t s, const double2 *Hk, const double2 *Hsk, double2 *Gk,
                          double2 *Pk, const double2 *wtab, const double *etab)
{
    switch (lM) {
#define X(v) case v: if (comp) launch_xmid<v, true>(c, s, Hk, Hsk, Gk, Pk, wtab, etab); else launch_xmid<v, false>(c, s, Hk, Hsk, Gk, Pk, wtab, etab); break;
        FOR_EACH_LM(X)
#undef X
    }
}

// Tables and kernel attributes of the own-transform path (se_zfft.cuh, se_xyfft.cuh): power-of-two grids, no cuFFT.
static se_status ensure_zt(se_plan *p)
{
    if (p->have_zt) return SE_OK;
    const int M = p->c.M;
    se_status st = ensure_wtab(p);
    if (st != SE_OK) return st;
    if (raise_smem_limit(k_zfft_r2c<128>) != cudaSuccess || raise_smem_limit(k_zfft_c2r<128>) != cudaSuccess ||
        raise_smem_limit(k_zfft_r2c<256>) != cudaSuccess || raise_smem_limit(k_zfft_c2r<256>) != cudaSuccess) {
        cudaGetLastError();
        return fail(p, SE_ERR_CUDA, "ensure_zt", "shared-memory limit");
    }
    p->lM = 0;
    while ((1 << p->lM) < M) ++p->lM;
    st = upload_etab(p);
    if (st == SE_OK && (dispatch_prepare_xy(p->lM) != cudaSuccess || dispatch_prepare_yz(p->lM) != cudaSuccess)) {
        cudaGetLastError();
        st = fail(p, SE_ERR_CUDA, "ensure_zt", "shared-memory limit");
    }
    if (st != SE_OK) return st;
    p->have_zt = true;
    p->yz_fused = M <= 128 ? 1 : 0;          // measured: clusters of 8 (M = 256) lose to the separate z and y kernels
    return SE_OK;
}

extern "C" se_status se_plan_create(se_plan **out, int64_t N, double L, const double *radii,
                                    double xi, double r_c, int M, int P, double eta0)
{
    if (!out) return SE_ERR_INVALID_ARG;
    *out = nullptr;
    if (!radii || N < 1 || N > (int64_t)1 << 30 || !(L > 0.0) || !(xi > 0.0) || !(r_c > 0.0) || r_c > 0.5 * L ||
        M < 2 || (M & 1) || M > 2048 || P < 2 || P > M || !(eta0 > 0.0))
        return SE_ERR_INVALID_ARG;
    if (P > SE_PMAX) return SE_ERR_UNSUPPORTED;
    double a2min = 1e300, a2max = 0.0;
    for (int64_t i = 0; i < N; ++i) {
        if (!(radii[i] > 0.0)) return SE_ERR_INVALID_ARG;
        const double t = radii[i] * radii[i];
        if (t < a2min) a2min = t;
        if (t > a2max) a2max = t;
    }

    se_plan *p = (se_plan *)aligned_alloc(64, (sizeof(se_plan) + 63) & ~(size_t)63);     // CUtensorMap members: 64-byte aligned
    if (!p) return SE_ERR_ALLOC;
    memset(p, 0, sizeof(se_plan));
    p->debug_stop = -1;
    SeConst &c = p->c;
    c.N = (int)N; c.M = M; c.P = P; c.L = L; c.xi = xi; c.rc2 = r_c * r_c; c.eta0 = eta0;
    p->m = sqrt(M_PI * P);
    p->a2min = a2min; p->a2max = a2max;
    derive_constants(p);
    {
        int dev = 0, sms = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) sms = 0;
        cudaGetLastError();
        p->sms = sms > 0 ? sms : 148;                  // without a device the allocations below fail anyway
    }

    // real-space cell grid: edge >= r_c, at least 3 cells per axis, else all pairs (one cell)
    p->r_c = r_c;
    choose_real_cells(p);
    p->ncell_r_alloc = p->ncell_r;                     // a strain only makes the cells larger
    // spreading tile bins (plane-thin): M x ceil(M/4) x ceil(M/8)
    c.NBY = (M + SE_TILE_Y - 1) / SE_TILE_Y;
    c.NBZ = (M + SE_TILE_Z - 1) / SE_TILE_Z;
    p->ncell_s = M * c.NBY * c.NBZ;
    c.rec_stride = se_rec_stride(P);
    c.grec_stride = se_grec_stride(P);
    if (!choose_gather_geometry(p)) { free(p); return SE_ERR_UNSUPPORTED; }
    p->ncell_g = p->gg.NTY * p->gg.NTZ * M;
    choose_segments(p, 0, 0);

    se_status st = SE_OK;
    const size_t Gc = (size_t)M * M * (M / 2 + 1);
    p->ncell_all = p->ncell_r + p->ncell_s + p->ncell_g + 3;
    const int nscan = p->ncell_all;
#define ALLOC(ptr, count) if (st == SE_OK) st = dev_alloc(p, &(ptr), (size_t)(count))
    ALLOC(p->d_radii, N);
    ALLOC(p->d_key_r, N); ALLOC(p->d_rank_r, N); ALLOC(p->d_key_s, N); ALLOC(p->d_rank_s, N);
    ALLOC(p->d_key_g, N); ALLOC(p->d_rank_g, N); ALLOC(p->d_grecs, (size_t)N * c.grec_stride);
    ALLOC(p->d_cnt_all, p->ncell_all); ALLOC(p->d_start_all, p->ncell_all); ALLOC(p->d_dst_rs, N);
    if (st == SE_OK) {
        p->d_cnt_r = p->d_cnt_all; p->d_cnt_s = p->d_cnt_r + p->ncell_r + 1; p->d_cnt_g = p->d_cnt_s + p->ncell_s + 1;
        p->d_start_r = p->d_start_all; p->d_start_s = p->d_start_r + p->ncell_r + 1; p->d_start_g = p->d_start_s + p->ncell_s + 1;
    }
    ALLOC(p->d_bsum, (nscan + SCAN_BLOCK - 1) / SCAN_BLOCK + 1);
    ALLOC(p->d_rs_pos, N); ALLOC(p->d_rs_mom, 12 * (size_t)N); ALLOC(p->d_rs_orig, N);
    ALLOC(p->d_recs, (size_t)N * c.rec_stride);
    ALLOC(p->d_real, 6 * p->Gp); ALLOC(p->d_Hk, 3 * Gc); ALLOC(p->d_Gk, 6 * Gc);
    ALLOC(p->d_out_real, 12 * (size_t)N); ALLOC(p->d_moments, GATHER_SUMS * (size_t)N);
    ALLOC(p->d_io, 25 * (size_t)N);
#undef ALLOC
    if (st != SE_OK) { se_plan_destroy(p); return st; }
    if (cudaMemcpy(p->d_radii, radii, sizeof(double) * (size_t)N, cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemset(p->d_out_real, 0, sizeof(double) * 12 * (size_t)N) != cudaSuccess ||
        cudaMemset(p->d_real, 0, sizeof(double) * 6 * p->Gp) != cudaSuccess ||       // alignment padding is read (with zero weight): keep it finite

        cudaMemset(p->d_moments, 0, sizeof(double) * GATHER_SUMS * (size_t)N) != cudaSuccess) {
        se_plan_destroy(p);
        return SE_ERR_CUDA;
    }

    // cuFFT: power-of-two grids use the own-z-transform path (2-D complex plans, made here); the batched 3-D real plans
    // are made by the first apply that needs them.
    {
        se_status stf = xf_supported(M) ? ensure_zt(p) : ensure_fft3d(p, false);
        if (stf == SE_OK) stf = make_tensor_map(p, &p->tmap, p->d_real, 6 * M);
        if (stf != SE_OK) { se_plan_destroy(p); return stf; }
    }

    for (int k = 0; k <= SE_NUM_STAGES; ++k)
        if (cudaEventCreate(&p->ev[k]) != cudaSuccess) { p->have_events = (k > 0); se_plan_destroy(p); return SE_ERR_CUDA; }
    p->have_events = true;
    int prio_lo = 0, prio_hi = 0;
    cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi);          // the side stream only fills what the wave pipeline leaves idle
    if (cudaStreamCreateWithPriority(&p->side, cudaStreamNonBlocking, prio_lo) != cudaSuccess) { cudaGetLastError(); se_plan_destroy(p); return SE_ERR_CUDA; }
    if (cudaEventCreateWithFlags(&p->ev_fork, cudaEventDisableTiming) != cudaSuccess) { cudaStreamDestroy(p->side); se_plan_destroy(p); return SE_ERR_CUDA; }
    if (cudaEventCreateWithFlags(&p->ev_join, cudaEventDisableTiming) != cudaSuccess) {
        cudaStreamDestroy(p->side); cudaEventDestroy(p->ev_fork); se_plan_destroy(p); return SE_ERR_CUDA;
    }
    p->have_side = true;
    {   // beside the wave pipeline a2 runs as a persistent grid of one CTA per SM (measured best on B200: it then
        // takes little from the HBM-bound kernels' occupancy; c4 step 3.57 -> 3.50 ms) -- as long as a CTA walks no more than
        // about 256 cells: beyond that the walk can outlast the wave pipeline and become the critical path (c5, 537 cells per
        // CTA: 26.8 ... 29.1 ms from run to run with one CTA per SM, 26.98 ms every time with two or three)
        const int per_sm = (p->ncell_r + 256 * p->sms - 1) / (256 * p->sms);
        p->real_side_ctas = p->sms * (per_sm < 1 ? 1 : (per_sm > 3 ? 3 : per_sm));
        p->real_overlap = 1;
        p->use_graph = M <= 128 ? 1 : 0;
        p->pair_cache = 1;
    }
    if (raise_smem_limit(k_scatter) != cudaSuccess || dispatch_prepare(P) != cudaSuccess) { cudaGetLastError(); se_plan_destroy(p); return SE_ERR_CUDA; }
    *out = p;
    return SE_OK;
}

extern "C" se_status se_plan_set_shape(se_plan *p, double m)
{
    if (!p || !(m > 0.0)) return SE_ERR_INVALID_ARG;
    p->m = m;
    ++p->epoch;
    derive_constants(p);
    p->have_positions = false;          // the cached Gaussian tables depend on the shape
    if (p->d_etab) return upload_etab(p);
    return SE_OK;
}

// Lees-Edwards strain of the lattice.  The count / start tables keep the layout of the unstrained box (their
// real-space part is only used up to the current number of cells).
extern "C" se_status se_plan_set_strain(se_plan *p, double gamma)
{
    if (!p || !(gamma == gamma) || fabs(gamma) > 1e6) return SE_ERR_INVALID_ARG;
    p->c.gamma = gamma;
    ++p->epoch;
    p->have_positions = false;
    p->have_pairs = false;
    choose_real_cells(p);
    if (p->ncell_r > p->ncell_r_alloc) return fail(p, SE_ERR_UNSUPPORTED, "se_plan_set_strain", "cell grid larger than allocated");
    if (p->d_etab) return upload_etab(p);
    return SE_OK;
}

extern "C" se_status se_plan_set_tuning(se_plan *p, int spread_segments, int gather_segments)
{
    if (!p || spread_segments < 0 || gather_segments < 0) return SE_ERR_INVALID_ARG;
    choose_segments(p, spread_segments, gather_segments);
    ++p->epoch;
    return SE_OK;
}

extern "C" se_status se_plan_set_option(se_plan *p, int key, int value)
{
    if (!p || value < 0) return SE_ERR_INVALID_ARG;
    ++p->epoch;
    switch (key) {
    case SE_OPT_REAL_OVERLAP: if (value > 2) return SE_ERR_INVALID_ARG; p->real_overlap = value; break;
    case SE_OPT_REAL_CTAS: p->real_side_ctas = value; break;
    case SE_OPT_YZ_FUSED: if (value > 1) return SE_ERR_INVALID_ARG; p->yz_fused = value; break;
    case SE_OPT_GRAPH: if (value > 1) return SE_ERR_INVALID_ARG; p->use_graph = value; break;
    case SE_OPT_PAIR_CACHE: if (value > 1) return SE_ERR_INVALID_ARG; p->pair_cache = value; if (!value) p->have_pairs = false; break;
    case SE_OPT_SIZE_VARIANT: if (value > 2) return SE_ERR_INVALID_ARG; p->size_variant = value; break;
    case SE_OPT_GRID_FP32: if (value > 1) return SE_ERR_INVALID_ARG; p->grid_fp32 = value; break;
    default: return SE_ERR_INVALID_ARG;
    }
    return SE_OK;
}

extern "C" se_status se_plan_set_flags(se_plan *p, unsigned flags)
{
    if (!p || (flags & ~0x5fu)) return SE_ERR_INVALID_ARG;
    p->flags = flags;
    ++p->epoch;
    return SE_OK;
}

extern "C" se_status se_plan_debug_stop(se_plan *p, int stage)
{
    if (!p || stage < -1 || stage >= SE_NUM_STAGES) return SE_ERR_INVALID_ARG;
    p->debug_stop = stage;
    ++p->epoch;
    return SE_OK;
}

extern "C" int se_plan_last_launch_count(const se_plan *p) { return p ? p->last_launches : 0; }
extern "C" size_t se_plan_workspace_bytes(const se_plan *p) { return p ? p->bytes : 0; }

extern "C" se_status se_plan_get_constants(const se_plan *p, double *out)
{
    if (!p || !out) return SE_ERR_INVALID_ARG;
    out[0] = p->c.Delta; out[1] = p->c.eta_se; out[2] = p->c.alpha; out[3] = p->m;
    out[4] = (double)p->c.ncr; out[5] = (double)p->c.nseg; out[6] = (double)p->gg.nseg;
    return SE_OK;
}

static se_status scan_cells(se_plan *p, cudaStream_t s)
{
    const int n = p->ncell_all, nb = (n + SCAN_BLOCK - 1) / SCAN_BLOCK;
    k_scan_local<<<nb, SCAN_THREADS, 0, s>>>(p->d_cnt_all, p->d_start_all, p->d_bsum, n);
    k_scan_add<<<nb, SCAN_THREADS, 0, s>>>(p->d_start_all, p->d_bsum, n, p->ncell_r_alloc + 1, p->ncell_r_alloc + p->ncell_s + 2, p->c.N);
    p->last_launches += 2;
    CUDA_TRY(p, cudaGetLastError());
    return SE_OK;
}

template <int P>
static void launch_spread(se_plan *p, cudaStream_t s, bool comp_in, const double *recs)
{
    const SeConst &c = p->c;
    const long long warps = (long long)c.NBY * c.NBZ * c.nseg;
    const int blocks = (int)((warps + SWEEP_WARPS - 1) / SWEEP_WARPS);
    const size_t sm = sweep_smem_bytes(c.rec_stride);
    if (c.gamma != 0.0) {
        if (comp_in) k_spread<P, 4, true><<<blocks, SWEEP_WARPS * 32, sm, s>>>(c, recs, p->d_start_s, p->d_real, p->d_real_p);
        else k_spread<P, 3, true><<<blocks, SWEEP_WARPS * 32, sm, s>>>(c, recs, p->d_start_s, p->d_real, nullptr);
    } else if (comp_in)
        k_spread<P, 4, false><<<blocks, SWEEP_WARPS * 32, sm, s>>>(c, recs, p->d_start_s, p->d_real, p->d_real_p);
    else
        k_spread<P, 3, false><<<blocks, SWEEP_WARPS * 32, sm, s>>>(c, recs, p->d_start_s, p->d_real, nullptr);
}

template <int P>
static void launch_gather(se_plan *p, cudaStream_t s, bool pressure, double *mom, int mstride)
{
    const GatherGeom &g = p->gg;
    const bool rv = !pressure && p->size_variant == 1;                            // real-space variant: u~ only, eight sums per grid
    const int ngrids = pressure ? 1 : (rv ? 3 : 6);
    const int items = g.NTY * g.NTZ * ngrids;
    const unsigned blocks = (unsigned)(items < p->sms ? items : p->sms);          // persistent: one CTA per SM (work split: GatherWalk)
    if (rv) {
        k_gather<P, true><<<blocks, (GR_WARPS + 1) * 32, p->gather_smem, s>>>(p->c, g, p->d_grecs, p->d_start_g, p->tmap, ngrids, p->d_moments, GATHER_SUMS);
        return;
    }
    k_gather<P, false><<<blocks, (GR_WARPS + 1) * 32, p->gather_smem, s>>>(p->c, g, p->d_grecs, p->d_start_g, pressure ? p->tmap_p : p->tmap, ngrids,
                                                             pressure ? p->d_pmom : (mom ? mom : p->d_moments), pressure ? 12 : (mom ? mstride : GATHER_SUMS));
}

template <int P>
static cudaError_t prepare_sweeps()
{
    cudaError_t e = raise_smem_limit(k_spread<P, 3, false>);
    if (e == cudaSuccess) e = raise_smem_limit(k_spread<P, 4, false>);
    if (e == cudaSuccess) e = raise_smem_limit(k_spread<P, 3, true>);
    if (e == cudaSuccess) e = raise_smem_limit(k_spread<P, 4, true>);
    if (e == cudaSuccess) e = raise_smem_limit(k_gather<P, false>);
    if (e == cudaSuccess) e = raise_smem_limit(k_gather<P, true>);
    return e;
}

static void dispatch_spread(se_plan *p, cudaStream_t s, bool comp_in, const double *recs = nullptr)
{
    if (!recs) recs = p->d_recs;
    switch (p->c.P) {
#define X(v) case v: launch_spread<v>(p, s, comp_in, recs); break;
        FOR_EACH_P(X)
#undef X
    }
}

static cudaError_t dispatch_prepare(int P)
{
    switch (P) {
#define X(v) case v: return prepare_sweeps<v>();
        FOR_EACH_P(X)
#undef X
    }
    return cudaErrorInvalidValue;
}

static void dispatch_gather(se_plan *p, cudaStream_t s, bool pressure, double *mom = nullptr, int mstride = 0)
{
    switch (p->c.P) {
#define X(v) case v: launch_gather<v>(p, s, pressure, mom, mstride); break;
        FOR_EACH_P(X)
#undef X
    }
}

// Buffers of the compressible extension (a9), made by the first apply that needs them; its cuFFT plans are made by
// ensure_comp_plans for the transform path actually taken.
static se_status ensure_compressible(se_plan *p)
{
    if (p->have_comp) return SE_OK;
    const int M = p->c.M;
    const size_t Gc = (size_t)M * M * (M / 2 + 1);
    se_status st = dev_alloc(p, &p->d_real_p, p->Gp);
    if (st == SE_OK) st = dev_alloc(p, &p->d_Hk_s, Gc);
    if (st == SE_OK) st = dev_alloc(p, &p->d_Gk_p, Gc);
    if (st == SE_OK) st = dev_alloc(p, &p->d_pmom, 12 * (size_t)p->c.N);
    if (st == SE_OK && cudaMemset(p->d_real_p, 0, sizeof(double) * p->Gp) != cudaSuccess) st = fail(p, SE_ERR_CUDA, "cudaMemset", "pressure grid");
    if (st == SE_OK) st = make_tensor_map(p, &p->tmap_p, p->d_real_p, M);
    if (st != SE_OK) {
        cudaFree(p->d_real_p); cudaFree(p->d_Hk_s); cudaFree(p->d_Gk_p); cudaFree(p->d_pmom);
        p->d_real_p = nullptr; p->d_Hk_s = nullptr; p->d_Gk_p = nullptr; p->d_pmom = nullptr;
        cudaGetLastError();
        return st;
    }
    p->have_comp = true;
    return SE_OK;
}

// Buffers and cuFFT plans of the single-precision mesh (SE_OPT_GRID_FP32), made by the first product that needs them.
static se_status ensure_f32(se_plan *p)
{
    if (p->have_f32) return SE_OK;
    const int M = p->c.M;
    const size_t G = (size_t)M * M * M, Gc = (size_t)M * M * (M / 2 + 1);
    se_status st = dev_alloc(p, &p->d_realf, 7 * G);
    if (st == SE_OK) st = dev_alloc(p, &p->d_Hkf, 4 * Gc);
    if (st == SE_OK) st = dev_alloc(p, &p->d_Gkf, 7 * Gc);
    int n3[3] = { M, M, M };
    cufftHandle *h[4] = { &p->fftf_fwd, &p->fftf_inv, &p->fftf_fwd1, &p->fftf_inv1 };
    const cufftType ty[4] = { CUFFT_R2C, CUFFT_C2R, CUFFT_R2C, CUFFT_C2R };
    const int nb[4] = { 3, 6, 1, 1 };
    int made = 0;
    size_t tot = 0;
    cufftResult r = CUFFT_SUCCESS;
    for (int i = 0; i < 4 && st == SE_OK && r == CUFFT_SUCCESS; ++i) {
        size_t ws = 0;
        r = cufftCreate(h[i]);
        if (r == CUFFT_SUCCESS) { ++made; r = cufftMakePlanMany(*h[i], 3, n3, NULL, 1, 0, NULL, 1, 0, ty[i], nb[i], &ws); tot += ws; }
    }
    if (st == SE_OK && r != CUFFT_SUCCESS) st = fail(p, r == CUFFT_ALLOC_FAILED ? SE_ERR_ALLOC : SE_ERR_CUFFT, "cufftMakePlanMany", "single-precision 3-D plans");
    if (st != SE_OK) {
        for (int i = 0; i < made; ++i) cufftDestroy(*h[i]);
        cudaFree(p->d_realf); cudaFree(p->d_Hkf); cudaFree(p->d_Gkf);
        p->d_realf = nullptr; p->d_Hkf = nullptr; p->d_Gkf = nullptr;
        cudaGetLastError();
        return st;
    }
    p->fft_bytes += tot;
    p->bytes += tot;
    p->have_f32 = true;
    return SE_OK;
}

// Buffers of the wave-space size variant (SE_OPT_SIZE_VARIANT = 2), made by the first product that needs them.
static se_status ensure_wave_variant(se_plan *p)
{
    if (p->d_Wk) return SE_OK;
    const int M = p->c.M;
    const size_t Gc = (size_t)M * M * (M / 2 + 1);
    se_status st = dev_alloc(p, &p->d_wrecs, (size_t)p->c.N * p->c.rec_stride);
    if (st == SE_OK) st = dev_alloc(p, &p->d_wmom, 96 * (size_t)p->c.N);
    if (st == SE_OK) st = dev_alloc(p, &p->d_Wk, 24 * Gc);
    if (st == SE_OK && cudaMemset(p->d_wmom, 0, sizeof(double) * 96 * (size_t)p->c.N) != cudaSuccess) st = fail(p, SE_ERR_CUDA, "cudaMemset", "wave-variant sums");
    if (st != SE_OK) {
        cudaFree(p->d_wrecs); cudaFree(p->d_wmom); cudaFree(p->d_Wk);
        p->d_wrecs = nullptr; p->d_wmom = nullptr; p->d_Wk = nullptr;
        cudaGetLastError();
    }
    return st;
}

// Single-grid cuFFT plans of the compressible extension (cuFFT 3-D path only; the own transforms need none).
static se_status ensure_comp_plans(se_plan *p, bool zt)
{
    return zt ? SE_OK : ensure_fft3d(p, true);
}

// a1: wrap, the three counting sorts, packed records and real-space copies (F == NULL: zero moments).
static se_status sort_and_pack(se_plan *p, const double *pos, const double *F, const double *T, const double *S,
                               const double *s_in, cudaStream_t s)
{
    const SeConst &c = p->c;
    const int TB = 128, nbN = (c.N + TB - 1) / TB;
    p->have_pairs = false;                            // a new configuration: the cached pair list is stale
    CUDA_TRY(p, cudaMemsetAsync(p->d_cnt_all, 0, sizeof(int) * (size_t)p->ncell_all, s));
    k_keys<<<nbN, TB, 0, s>>>(c, p->gg, pos, p->d_key_r, p->d_rank_r, p->d_cnt_r, p->d_key_s, p->d_rank_s, p->d_cnt_s,
                              p->d_key_g, p->d_rank_g, p->d_cnt_g);
    p->last_launches += 1;
    const se_status st = scan_cells(p, s);
    if (st != SE_OK) return st;
    k_scatter<<<(c.N + SCATTER_PART - 1) / SCATTER_PART, SCATTER_THREADS, scatter_smem_bytes(c.P), s>>>(
        c, pos, p->d_radii, F, T, S, s_in, p->d_key_r, p->d_rank_r, p->d_start_r, p->d_key_s, p->d_rank_s, p->d_start_s,
        p->d_key_g, p->d_rank_g, p->d_start_g, p->d_grecs, p->d_rs_pos, p->d_rs_mom, p->d_rs_orig, p->d_recs, p->d_dst_rs);
    p->last_launches += 1;
    CUDA_TRY(p, cudaGetLastError());
    return SE_OK;
}

// Neighbour search and radial scalars of the real-space sum, once per cached configuration (se_real.cuh, "Cached pairs"):
// count the pairs of every target, scan, size the list (one 8-byte read back: the stream is synchronised), fill.
static se_status build_pair_cache(se_plan *p, cudaStream_t s)
{
    const SeConst &c = p->c;
    const int N = c.N, n = N + 1, nb = (n + SCAN_BLOCK - 1) / SCAN_BLOCK;
    if (!p->d_pair_start) {
        se_status st = dev_alloc(p, &p->d_pair_start, (size_t)n);
        if (st == SE_OK) st = dev_alloc(p, &p->d_pair_cursor, (size_t)n);
        if (st == SE_OK) st = dev_alloc(p, &p->d_pair_bsum, (size_t)nb + 1);
        if (st != SE_OK) return st;
    }
    const unsigned grid = (unsigned)(c.ncr > 1 ? p->ncell_r : (c.N + 31) / 32);
    CUDA_TRY(p, cudaMemsetAsync(p->d_pair_cursor, 0, sizeof(int) * (size_t)n, s));
    k_pairs<false><<<grid, REAL_WARPS * 32, 0, s>>>(c, p->d_rs_pos, p->d_start_r, p->d_pair_cursor, nullptr, nullptr, nullptr, nullptr);
    k_scan_local<<<nb, SCAN_THREADS, 0, s>>>(p->d_pair_cursor, p->d_pair_start, p->d_pair_bsum, n);
    k_scan_add<<<nb, SCAN_THREADS, 0, s>>>(p->d_pair_start, p->d_pair_bsum, n, 0x7fffffff, 0x7fffffff, 0);
    p->last_launches += 3;
    int total = 0;
    CUDA_TRY(p, cudaMemcpyAsync(&total, p->d_pair_start + N, sizeof(int), cudaMemcpyDeviceToHost, s));
    CUDA_TRY(p, cudaStreamSynchronize(s));
    if (total < 0) return fail(p, SE_ERR_UNSUPPORTED, "build_pair_cache", "more than 2^31 pairs");
    if ((size_t)total > p->pair_cap) {
        cudaFree(p->d_pj); cudaFree(p->d_pd);
        p->d_pj = nullptr; p->d_pd = nullptr; p->pair_cap = 0;
        const size_t cap = (size_t)total + (size_t)total / 8 + 1024;
        se_status st = dev_alloc(p, &p->d_pj, cap);
        if (st == SE_OK) st = dev_alloc(p, &p->d_pd, cap * PAIR_F);
        if (st != SE_OK) { cudaFree(p->d_pj); p->d_pj = nullptr; cudaGetLastError(); p->err[0] = 0; return SE_OK; }   // no room: products fall back to k_real
        p->pair_cap = cap;
    }
    p->npairs = (size_t)total;
    CUDA_TRY(p, cudaMemsetAsync(p->d_pair_cursor, 0, sizeof(int) * (size_t)n, s));
    k_pairs<true><<<grid, REAL_WARPS * 32, 0, s>>>(c, p->d_rs_pos, p->d_start_r, nullptr, p->d_pair_start, p->d_pair_cursor, p->d_pj, p->d_pd);
    p->last_launches += 1;
    CUDA_TRY(p, cudaGetLastError());
    p->have_pairs = true;
    return SE_OK;
}

extern "C" se_status se_plan_set_positions(se_plan *p, const double *pos, void *cuda_stream)
{
    if (!p) return SE_ERR_INVALID_ARG;
    ++p->epoch;
    if (!pos) { p->have_positions = false; return SE_OK; }            // forget the cached configuration
    p->last_launches = 0;
    p->have_positions = false;
    const se_status st = sort_and_pack(p, pos, nullptr, nullptr, nullptr, nullptr, (cudaStream_t)cuda_stream);
    if (st != SE_OK) return st;
    p->have_positions = true;
    p->have_pairs = false;
    if (p->pair_cache) return build_pair_cache(p, (cudaStream_t)cuda_stream);
    return SE_OK;
}

static se_status apply_impl(se_plan *p, const double *pos, const double *F, const double *T, const double *S,
                            const double *s_in, double *U, double *Omega, double *E, double *s_out, void *cuda_stream,
                            const char *who)
{
    if (!p) return SE_ERR_INVALID_ARG;
    if (!F || !T || !S || !U || !Omega || !E) return fail(p, SE_ERR_INVALID_ARG, who, "null pointer");
    if (!pos && !p->have_positions) return fail(p, SE_ERR_INVALID_ARG, who, "pos is NULL and no positions were set (se_plan_set_positions)");
    const bool comp_in = s_in != nullptr, comp_out = s_out != nullptr, comp = comp_in || comp_out;
    if (comp) { se_status stc = ensure_compressible(p); if (stc != SE_OK) return stc; }
    const bool wv = p->size_variant == 2;
    const int nret = p->size_variant == 1 ? 3 : 6;          // returned grids: u~ (+ w~ in the hybrid approach)
    // wave-space variant: seven spreading passes of three plain grids each, cuFFT's 3-D transforms, one k-space pass on 24
    // spectra, four batches of six returned grids through the gather
    if (wv && p->debug_stop >= 0) return fail(p, SE_ERR_UNSUPPORTED, who, "se_plan_debug_stop with the wave-space size variant");
    if (wv) { se_status stw = ensure_wave_variant(p); if (stw != SE_OK) return stw; }
    // default for power-of-two grids: own z transforms with transposed spectra + contiguous 2-D complex cuFFT plans
    // (se_zfft.cuh); otherwise, and with SE_CUFFT3D, cuFFT's 3-D real transforms
    const bool f32 = p->grid_fp32 != 0 && !wv;
    if (p->grid_fp32 != 0 && wv) return fail(p, SE_ERR_UNSUPPORTED, who, "the single-precision mesh is built for the hybrid and real-space size variants");
    if (f32) { se_status st3 = ensure_f32(p); if (st3 != SE_OK) return st3; }
    const bool use_zt = !wv && !f32 && !(p->flags & SE_CUFFT3D) && xf_supported(p->c.M);
    if (use_zt) { se_status stf = ensure_zt(p); if (stf != SE_OK) return stf; }
    if (!use_zt && !f32) { se_status stf = ensure_fft3d(p, false); if (stf != SE_OK) return stf; }
    if (comp && !f32) { se_status stf = ensure_comp_plans(p, use_zt); if (stf != SE_OK) return stf; }
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const SeConst &c = p->c;
    const unsigned fl = p->flags;
    const bool timing = (fl & SE_TIMING) != 0;
    const bool do_real = !(fl & SE_SKIP_REAL) && !p->ext_out_real, do_wave = !(fl & SE_SKIP_WAVE);
    const int stop = p->debug_stop;
    auto on = [&](int stage) { return do_wave && !wv && (stop < 0 || stage <= stop); };
    p->last_launches = 0;
    p->timed = false;
    p->err[0] = 0;
    const int TB = 128, nbN = (c.N + TB - 1) / TB;
    int evi = 0;
#define MARK() do { if (timing) CUDA_TRY(p, cudaEventRecord(p->ev[evi], s)); ++evi; } while (0)
    MARK();
    // ---- a1: wrap + counting sorts + packing; with cached positions (pos == NULL) only the moments are refreshed ----
    if (pos) {
        p->have_positions = false;
        const se_status st = sort_and_pack(p, pos, F, T, S, s_in, s);
        if (st != SE_OK) return st;
    } else {
        k_moments<<<nbN, TB, 0, s>>>(c, F, T, S, s_in, p->d_dst_rs, p->d_rs_mom, p->d_recs);
        p->last_launches += 1;
        CUDA_TRY(p, cudaGetLastError());
    }
    MARK();
    // ---- a2: real-space pair sum ----
    // a2 is independent of the wave pipeline: it runs on the plan's (low-priority) side stream, forked here and
    // joined before the epilogue, and fills what the wave-space kernels leave idle (tails, the HBM-bound stages).
    // Measured gain on B200 is small (c4: 4 %).  When stage timings are asked for it runs on the caller's
    // stream, alone, so that every stage is timed by itself.
    const bool fork = do_real && do_wave && !timing && stop < 0 && p->real_overlap > 0;
    auto launch_real = [&](cudaStream_t sr) {
        if (!pos && !comp && p->have_pairs) {          // cached configuration: stream the pair list
            const unsigned nbc = (unsigned)((c.N + 7) / 8 < p->sms * 16 ? (c.N + 7) / 8 : p->sms * 16);   // 8 targets per CTA pass, 16 CTAs per SM
            k_real_cached<1><<<nbc, 128, 0, sr>>>(c, p->d_pair_start, p->d_pj, p->d_pd, p->d_rs_mom, p->d_rs_orig, p->d_out_real, 0);
            p->last_launches += 1;
            return;
        }
        unsigned nb = (unsigned)(c.ncr > 1 ? p->ncell_r : (c.N + 31) / 32);
        if (sr != s && c.ncr > 1 && p->real_side_ctas > 0 && nb > (unsigned)p->real_side_ctas) nb = (unsigned)p->real_side_ctas;
        if (comp) k_real<true, 1><<<nb, REAL_WARPS * 32, 0, sr>>>(c, p->d_rs_pos, p->d_rs_mom, p->d_rs_orig, p->d_start_r, p->d_out_real, 0);
        else k_real<false, 1><<<nb, REAL_WARPS * 32, 0, sr>>>(c, p->d_rs_pos, p->d_rs_mom, p->d_rs_orig, p->d_start_r, p->d_out_real, 0);
        p->last_launches += 1;
    };
    if (do_real && !fork) {
        launch_real(s);
        CUDA_TRY(p, cudaGetLastError());
    }
    auto fork_real = [&]() -> se_status {
        CUDA_TRY(p, cudaEventRecord(p->ev_fork, s));
        CUDA_TRY(p, cudaStreamWaitEvent(p->side, p->ev_fork, 0));
        launch_real(p->side);
        CUDA_TRY(p, cudaGetLastError());
        CUDA_TRY(p, cudaEventRecord(p->ev_join, p->side));
        return SE_OK;
    };
    if (fork && p->real_overlap == 1) { se_status sf = fork_real(); if (sf != SE_OK) return sf; }
    MARK();
    // ---- a3..a7: Spectral Ewald wave-space sum ----
    bool wave_done = false;
    if (on(SE_STAGE_SPREAD)) {
        if (comp_in) p->real_p_padded = false;
        dispatch_spread(p, s, comp_in);
        p->last_launches += 1;
        CUDA_TRY(p, cudaGetLastError());
    }
    if (wv && do_wave) {
        // stage "spread" of the timings holds all seven passes (records, spreading, transform to wave space)
        const size_t Gc = (size_t)c.M * c.M * (c.M / 2 + 1);
        if (comp_in) p->real_p_padded = false;
        CUFFT_TRY(p, cufftSetStream(p->fft_fwd, s));
        for (int pass = 0; pass < 7; ++pass) {
            k_plain_recs<<<(unsigned)((c.N + 3) / 4), 128, 0, s>>>(c, p->d_recs, p->d_wrecs, pass);
            dispatch_spread(p, s, comp_in && pass == 0, p->d_wrecs);
            p->last_launches += 2;
            CUDA_TRY(p, cudaGetLastError());
            CUFFT_TRY(p, cufftExecD2Z(p->fft_fwd, p->d_real, (cufftDoubleComplex *)(p->d_Wk + 3 * (size_t)pass * Gc)));
            if (comp_in && pass == 0) {
                CUFFT_TRY(p, cufftSetStream(p->fft_fwd1, s));
                CUFFT_TRY(p, cufftExecD2Z(p->fft_fwd1, p->d_real_p, (cufftDoubleComplex *)p->d_Hk_s));
            }
        }
    }
    if (fork && p->real_overlap == 2) { se_status sf = fork_real(); if (sf != SE_OK) return sf; }
    MARK();
    const bool yz = use_zt && p->yz_fused != 0;
    if (on(SE_STAGE_FFT_FWD) && yz) {
        CUDA_TRY(p, dispatch_yz(p->lM, false, s, 3, p->d_real, p->d_Hk, nullptr, p->d_wtab, 0, 0, 0));
        p->last_launches += 1;
        if (comp_in) {
            CUDA_TRY(p, dispatch_yz(p->lM, false, s, 1, p->d_real_p, p->d_Hk_s, nullptr, p->d_wtab, 0, 0, 0));
            p->last_launches += 1;
        }
    } else if (on(SE_STAGE_FFT_FWD) && use_zt) {
        const int M = c.M;
        if (zt_threads(M) <= 128) k_zfft_r2c<128><<<3 * M * (M / ZT_LINES), zt_threads(M), zt_smem_bytes(M), s>>>(M, p->lM - 1, p->d_real, p->d_Hk, p->d_wtab);
        else k_zfft_r2c<256><<<3 * M * (M / ZT_LINES), zt_threads(M), zt_smem_bytes(M), s>>>(M, p->lM - 1, p->d_real, p->d_Hk, p->d_wtab);
        p->last_launches += 1;
        CUDA_TRY(p, cudaGetLastError());
        dispatch_yfft(p->lM, s, p->d_Hk, p->d_wtab, 3, false);
        p->last_launches += 1;
        CUDA_TRY(p, cudaGetLastError());
        if (comp_in) {
            if (zt_threads(M) <= 128) k_zfft_r2c<128><<<M * (M / ZT_LINES), zt_threads(M), zt_smem_bytes(M), s>>>(M, p->lM - 1, p->d_real_p, p->d_Hk_s, p->d_wtab);
            else k_zfft_r2c<256><<<M * (M / ZT_LINES), zt_threads(M), zt_smem_bytes(M), s>>>(M, p->lM - 1, p->d_real_p, p->d_Hk_s, p->d_wtab);
            p->last_launches += 1;
            CUDA_TRY(p, cudaGetLastError());
            dispatch_yfft(p->lM, s, p->d_Hk_s, p->d_wtab, 1, false);
            p->last_launches += 1;
            CUDA_TRY(p, cudaGetLastError());
        }
    } else if (on(SE_STAGE_FFT_FWD) && f32) {
        const size_t G = (size_t)c.M * c.M * c.M;
        k_grid_to_f32<<<(unsigned)((3 * G + 255) / 256), 256, 0, s>>>(p->d_real, p->d_realf, 3 * G);
        p->last_launches += 1;
        CUFFT_TRY(p, cufftSetStream(p->fftf_fwd, s));
        CUFFT_TRY(p, cufftExecR2C(p->fftf_fwd, p->d_realf, (cufftComplex *)p->d_Hkf));
        if (comp_in) {
            const size_t Gc = (size_t)c.M * c.M * (c.M / 2 + 1);
            k_grid_to_f32<<<(unsigned)((G + 255) / 256), 256, 0, s>>>(p->d_real_p, p->d_realf + 6 * G, G);
            p->last_launches += 1;
            CUFFT_TRY(p, cufftSetStream(p->fftf_fwd1, s));
            CUFFT_TRY(p, cufftExecR2C(p->fftf_fwd1, p->d_realf + 6 * G, (cufftComplex *)(p->d_Hkf + 3 * Gc)));
        }
        CUDA_TRY(p, cudaGetLastError());
    } else if (on(SE_STAGE_FFT_FWD)) {
        CUFFT_TRY(p, cufftSetStream(p->fft_fwd, s));
        CUFFT_TRY(p, cufftExecD2Z(p->fft_fwd, p->d_real, (cufftDoubleComplex *)p->d_Hk));
        if (comp_in) {
            CUFFT_TRY(p, cufftSetStream(p->fft_fwd1, s));
            CUFFT_TRY(p, cufftExecD2Z(p->fft_fwd1, p->d_real_p, (cufftDoubleComplex *)p->d_Hk_s));
        }
    }
    MARK();
    if (on(SE_STAGE_KSPACE)) {
        const size_t Gc = (size_t)c.M * c.M * (c.M / 2 + 1);
        const unsigned nbk = (unsigned)((Gc + KSPACE_THREADS - 1) / KSPACE_THREADS);
        if (use_zt) dispatch_xmid(p->lM, comp, c, s, p->d_Hk, comp_in ? p->d_Hk_s : nullptr, p->d_Gk, comp_out ? p->d_Gk_p : nullptr,
                                  p->d_wtab, p->d_etab);
        else if (f32) k_kspace<float2><<<nbk, KSPACE_THREADS, 0, s>>>(c, p->d_Hkf, p->d_Gkf, comp_in ? p->d_Hkf + 3 * Gc : nullptr,
                                                                     comp_out ? p->d_Gkf + 6 * Gc : nullptr);
        else k_kspace<double2><<<nbk, KSPACE_THREADS, 0, s>>>(c, p->d_Hk, p->d_Gk, comp_in ? p->d_Hk_s : nullptr,
                                                            comp_out ? p->d_Gk_p : nullptr);
        p->last_launches += 1;
        CUDA_TRY(p, cudaGetLastError());
    }
    if (wv && do_wave) {
        const size_t Gc = (size_t)c.M * c.M * (c.M / 2 + 1);
        k_kspace_wave<<<(unsigned)((Gc + KSPACE_THREADS - 1) / KSPACE_THREADS), KSPACE_THREADS, 0, s>>>(c, p->d_Wk, comp_in ? p->d_Hk_s : nullptr,
                                                                                                    comp_out ? p->d_Gk_p : nullptr);
        p->last_launches += 1;
        CUDA_TRY(p, cudaGetLastError());
    }
    MARK();
    if (on(SE_STAGE_FFT_INV) && yz) {
        const int MYp = p->gg.MYp, MZp = p->gg.MZp, halo = c.P - 1;
        CUDA_TRY(p, dispatch_yz(p->lM, true, s, nret, nullptr, p->d_Gk, p->d_real, p->d_wtab, MYp, MZp, halo));
        p->last_launches += 1;
        if (comp_out) {
            CUDA_TRY(p, dispatch_yz(p->lM, true, s, 1, nullptr, p->d_Gk_p, p->d_real_p, p->d_wtab, MYp, MZp, halo));
            p->last_launches += 1;
            p->real_p_padded = true;
        }
    } else if (on(SE_STAGE_FFT_INV) && use_zt) {
        const int M = c.M, MYp = p->gg.MYp, MZp = p->gg.MZp, halo = c.P - 1;
        dispatch_yfft(p->lM, s, p->d_Gk, p->d_wtab, nret, true);
        p->last_launches += 1;
        CUDA_TRY(p, cudaGetLastError());
        if (zt_threads(M) <= 128) k_zfft_c2r<128><<<nret * M * (M / ZT_LINES), zt_threads(M), zt_smem_bytes(M), s>>>(M, p->lM - 1, p->d_Gk, p->d_real, p->d_wtab, MYp, MZp, halo);
        else k_zfft_c2r<256><<<nret * M * (M / ZT_LINES), zt_threads(M), zt_smem_bytes(M), s>>>(M, p->lM - 1, p->d_Gk, p->d_real, p->d_wtab, MYp, MZp, halo);
        p->last_launches += 1;
        CUDA_TRY(p, cudaGetLastError());
        if (comp_out) {
            dispatch_yfft(p->lM, s, p->d_Gk_p, p->d_wtab, 1, true);
            p->last_launches += 1;
            CUDA_TRY(p, cudaGetLastError());
            if (zt_threads(M) <= 128) k_zfft_c2r<128><<<M * (M / ZT_LINES), zt_threads(M), zt_smem_bytes(M), s>>>(M, p->lM - 1, p->d_Gk_p, p->d_real_p, p->d_wtab, MYp, MZp, halo);
            else k_zfft_c2r<256><<<M * (M / ZT_LINES), zt_threads(M), zt_smem_bytes(M), s>>>(M, p->lM - 1, p->d_Gk_p, p->d_real_p, p->d_wtab, MYp, MZp, halo);
            p->last_launches += 1;
            CUDA_TRY(p, cudaGetLastError());
            p->real_p_padded = true;
        }
    } else if (on(SE_STAGE_FFT_INV) && f32) {
        const int M = c.M, MYp = p->gg.MYp, MZp = p->gg.MZp, halo = c.P - 1;
        const size_t per = (size_t)MYp * MZp, G = (size_t)M * M * M, Gc = (size_t)M * M * (M / 2 + 1);
        CUFFT_TRY(p, cufftSetStream(p->fftf_inv, s));
        CUFFT_TRY(p, cufftExecC2R(p->fftf_inv, (cufftComplex *)p->d_Gkf, p->d_realf));       // all six; the real-space variant gathers three
        k_grid_from_f32<<<(unsigned)((nret * M * per + 255) / 256), 256, 0, s>>>(p->d_realf, p->d_real, M, MYp, MZp, halo, (size_t)nret * M);
        p->last_launches += 1;
        if (comp_out) {
            CUFFT_TRY(p, cufftSetStream(p->fftf_inv1, s));
            CUFFT_TRY(p, cufftExecC2R(p->fftf_inv1, (cufftComplex *)(p->d_Gkf + 6 * Gc), p->d_realf + 6 * G));
            k_grid_from_f32<<<(unsigned)((M * per + 255) / 256), 256, 0, s>>>(p->d_realf + 6 * G, p->d_real_p, M, MYp, MZp, halo, (size_t)M);
            p->last_launches += 1;
            p->real_p_padded = true;
        }
        CUDA_TRY(p, cudaGetLastError());
    } else if (on(SE_STAGE_FFT_INV)) {
        const int M = c.M, MYp = p->gg.MYp, MZp = p->gg.MZp, halo = c.P - 1;
        const size_t per = (size_t)MYp * MZp;
        CUFFT_TRY(p, cufftSetStream(p->fft_inv, s));
        CUFFT_TRY(p, cufftExecZ2D(p->fft_inv, (cufftDoubleComplex *)p->d_Gk, p->d_real));
        k_halo_fill<<<(unsigned)((6 * M * per + 255) / 256), 256, 0, s>>>(p->d_real, M, MYp, MZp, halo, (size_t)6 * M);
        p->last_launches += 1;
        if (comp_out) {
            CUFFT_TRY(p, cufftSetStream(p->fft_inv1, s));
            CUFFT_TRY(p, cufftExecZ2D(p->fft_inv1, (cufftDoubleComplex *)p->d_Gk_p, p->d_real_p));
            k_halo_fill<<<(unsigned)((M * per + 255) / 256), 256, 0, s>>>(p->d_real_p, M, MYp, MZp, halo, (size_t)M);
            p->last_launches += 1;
            p->real_p_padded = true;
        }
        CUDA_TRY(p, cudaGetLastError());
    }
    MARK();
    if (on(SE_STAGE_GATHER)) {
        dispatch_gather(p, s, false);
        p->last_launches += 1;
        if (comp_out) {
            dispatch_gather(p, s, true);
            p->last_launches += 1;
        }
        CUDA_TRY(p, cudaGetLastError());
        wave_done = true;
    }
    if (wv && do_wave) {
        // stage "gather" of the timings holds the four batches (transform back, halo, gather)
        const int M = c.M, MYp = p->gg.MYp, MZp = p->gg.MZp, halo = c.P - 1;
        const size_t Gc = (size_t)M * M * (M / 2 + 1), per = (size_t)MYp * MZp;
        CUFFT_TRY(p, cufftSetStream(p->fft_inv, s));
        for (int b = 0; b < 4; ++b) {
            CUFFT_TRY(p, cufftExecZ2D(p->fft_inv, (cufftDoubleComplex *)(p->d_Wk + 6 * (size_t)b * Gc), p->d_real));
            k_halo_fill<<<(unsigned)((6 * M * per + 255) / 256), 256, 0, s>>>(p->d_real, M, MYp, MZp, halo, (size_t)6 * M);
            dispatch_gather(p, s, false, p->d_wmom + 24 * b, 96);
            p->last_launches += 2;
            CUDA_TRY(p, cudaGetLastError());
        }
        if (comp_out) {
            CUFFT_TRY(p, cufftSetStream(p->fft_inv1, s));
            CUFFT_TRY(p, cufftExecZ2D(p->fft_inv1, (cufftDoubleComplex *)p->d_Gk_p, p->d_real_p));
            k_halo_fill<<<(unsigned)((M * per + 255) / 256), 256, 0, s>>>(p->d_real_p, M, MYp, MZp, halo, (size_t)M);
            dispatch_gather(p, s, true);
            p->last_launches += 2;
            p->real_p_padded = true;
            CUDA_TRY(p, cudaGetLastError());
        }
        wave_done = true;
    }
    MARK();
    // ---- a8: epilogue ----
    if (fork) CUDA_TRY(p, cudaStreamWaitEvent(s, p->ev_join, 0));
    k_epilogue<<<nbN, TB, 0, s>>>(c, fl | (wave_done ? 0u : SE_SKIP_WAVE), p->d_radii, F, T, S, p->ext_out_real ? p->ext_out_real : p->d_out_real, wv ? p->d_wmom : p->d_moments, wv ? 96 : GATHER_SUMS,
                                  comp_out && wave_done ? p->d_pmom : nullptr, U, Omega, E, s_out, p->size_variant);
    p->last_launches += 1;
    CUDA_TRY(p, cudaGetLastError());
    MARK();
#undef MARK
    p->timed = timing;
    return SE_OK;
}

// The product as a plan-owned CUDA graph (small systems are bound by the latency of ~15 launches): the first call with a
// given set of pointers runs plainly (lazy allocations), the second captures the same sequence on the caller's stream into
// a graph, later ones replay it.  Anything that changes what is enqueued (other pointers or stream, flags, options,
// se_plan_set_positions) captures again.  Not used on the legacy default stream, while the caller is capturing itself,
// or with SE_TIMING / se_plan_debug_stop.
static se_status apply_graphed(se_plan *p, const double *pos, const double *F, const double *T, const double *S,
                               const double *s_in, double *U, double *Omega, double *E, double *s_out, void *cuda_stream,
                               const char *who)
{
    if (!p) return SE_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const int cv = (s_in || s_out) ? 1 : 0;
    bool plain = !p->use_graph || s == nullptr || s == cudaStreamLegacy || (p->flags & SE_TIMING) || p->debug_stop >= 0 || !p->warmed[cv] ||
                 !F || !T || !S || !U || !Omega || !E || (!pos && !p->have_positions);
    if (!plain) {
        cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
        if (cudaStreamIsCapturing(s, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) { cudaGetLastError(); plain = true; }
    }
    if (plain) {
        const se_status st = apply_impl(p, pos, F, T, S, s_in, U, Omega, E, s_out, cuda_stream, who);
        if (st == SE_OK) p->warmed[cv] = true;
        return st;
    }
    const void *key[10] = { pos, F, T, S, s_in, U, Omega, E, s_out, cuda_stream };
    if (p->have_graph && p->gepoch == p->epoch && p->gflags == p->flags && memcmp(key, p->gkey, sizeof(key)) == 0) {
        CUDA_TRY(p, cudaGraphLaunch(p->gexec, s));
        p->last_launches = p->graph_launches;
        if (pos) p->have_positions = false;
        return SE_OK;
    }
    const bool had_pos = p->have_positions;
    CUDA_TRY(p, cudaStreamBeginCapture(s, cudaStreamCaptureModeThreadLocal));
    const se_status st = apply_impl(p, pos, F, T, S, s_in, U, Omega, E, s_out, cuda_stream, who);
    cudaGraph_t g = nullptr;
    const cudaError_t ec = cudaStreamEndCapture(s, &g);
    if (st != SE_OK || ec != cudaSuccess || !g) {
        if (g) cudaGraphDestroy(g);
        cudaGetLastError();
        p->have_positions = had_pos;
        if (st != SE_OK) return st;
        return fail(p, SE_ERR_CUDA, "cudaStreamEndCapture", cudaGetErrorString(ec));
    }
    if (p->have_graph) { cudaGraphExecDestroy(p->gexec); p->have_graph = false; }
    const cudaError_t ei = cudaGraphInstantiate(&p->gexec, g, 0);
    cudaGraphDestroy(g);
    if (ei != cudaSuccess) { cudaGetLastError(); return fail(p, SE_ERR_CUDA, "cudaGraphInstantiate", cudaGetErrorString(ei)); }
    p->have_graph = true;
    memcpy(p->gkey, key, sizeof(key));
    p->gflags = p->flags;
    p->gepoch = p->epoch;
    p->graph_launches = p->last_launches;
    CUDA_TRY(p, cudaGraphLaunch(p->gexec, s));
    return SE_OK;
}

extern "C" se_status far_mobility_apply(se_plan *p, const double *pos, const double *F, const double *T,
                                        const double *S, double *U, double *Omega, double *E, void *cuda_stream)
{
    return apply_graphed(p, pos, F, T, S, nullptr, U, Omega, E, nullptr, cuda_stream, "far_mobility_apply");
}

extern "C" se_status far_mobility_apply_compressible(se_plan *p, const double *pos, const double *F, const double *T,
                                                     const double *S, const double *s_in, double *U, double *Omega,
                                                     double *E, double *s_out, void *cuda_stream)
{
    return apply_graphed(p, pos, F, T, S, s_in, U, Omega, E, s_out, cuda_stream, "far_mobility_apply_compressible");
}

// Several right-hand sides on one configuration: a1 once; the real-space sum for up to four right-hand
// sides per launch, each pair's radial functions evaluated once (k_real<., NR>); the wave-space pipeline per right-hand side.
extern "C" se_status far_mobility_apply_batch(se_plan *p, const double *pos, int nrhs, const double *F, const double *T,
                                              const double *S, double *U, double *Omega, double *E, void *cuda_stream)
{
    if (!p) return SE_ERR_INVALID_ARG;
    if (nrhs < 1 || !F || !T || !S || !U || !Omega || !E) return fail(p, SE_ERR_INVALID_ARG, "far_mobility_apply_batch", "null pointer or nrhs < 1");
    if (!pos && !p->have_positions) return fail(p, SE_ERR_INVALID_ARG, "far_mobility_apply_batch", "pos is NULL and no positions were set");
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const SeConst &c = p->c;
    const size_t N = (size_t)c.N, rs = 12 * N;
    if (nrhs > p->batch_cap) {
        CUDA_TRY(p, cudaStreamSynchronize(s));                         // an earlier batch may still use the old buffers
        cudaFree(p->d_mom_b); cudaFree(p->d_out_real_b);
        p->d_mom_b = nullptr; p->d_out_real_b = nullptr; p->batch_cap = 0;
        se_status st = dev_alloc(p, &p->d_mom_b, (size_t)nrhs * rs);
        if (st == SE_OK) st = dev_alloc(p, &p->d_out_real_b, (size_t)nrhs * rs);
        if (st != SE_OK) return st;
        p->batch_cap = nrhs;
    }
    int launches = 0;
    if (pos) {
        const se_status st = se_plan_set_positions(p, pos, cuda_stream);
        if (st != SE_OK) return st;
        launches += p->last_launches;
    }
    const bool do_real = !(p->flags & SE_SKIP_REAL);
    const int TB = 128, nbN = (c.N + TB - 1) / TB;
    if (do_real) {
        for (int r = 0; r < nrhs; ++r)
            k_moments<<<nbN, TB, 0, s>>>(c, F + 3 * N * r, T + 3 * N * r, S + 5 * N * r, nullptr, p->d_dst_rs, p->d_mom_b + rs * r, nullptr);
        launches += nrhs;
        const unsigned nb = (unsigned)(c.ncr > 1 ? p->ncell_r : (c.N + 31) / 32);
        for (int r = 0; r < nrhs;) {
            const double *m = p->d_mom_b + rs * r;
            double *o = p->d_out_real_b + rs * r;
            if (p->have_pairs) {                      // cached pair list: one streaming pass for up to four right-hand sides
                const unsigned nbc = (unsigned)((c.N + 7) / 8 < p->sms * 16 ? (c.N + 7) / 8 : p->sms * 16);   // 8 targets per CTA pass, 16 CTAs per SM
                if (nrhs - r >= 4) { k_real_cached<4><<<nbc, 128, 0, s>>>(c, p->d_pair_start, p->d_pj, p->d_pd, m, p->d_rs_orig, o, rs); r += 4; }
                else if (nrhs - r >= 2) { k_real_cached<2><<<nbc, 128, 0, s>>>(c, p->d_pair_start, p->d_pj, p->d_pd, m, p->d_rs_orig, o, rs); r += 2; }
                else { k_real_cached<1><<<nbc, 128, 0, s>>>(c, p->d_pair_start, p->d_pj, p->d_pd, m, p->d_rs_orig, o, rs); r += 1; }
            } else if (nrhs - r >= 4) { k_real<false, 4><<<nb, REAL_WARPS * 32, 0, s>>>(c, p->d_rs_pos, m, p->d_rs_orig, p->d_start_r, o, rs); r += 4; }
            else if (nrhs - r >= 2) { k_real<false, 2><<<nb, REAL_WARPS * 32, 0, s>>>(c, p->d_rs_pos, m, p->d_rs_orig, p->d_start_r, o, rs); r += 2; }
            else { k_real<false, 1><<<nb, REAL_WARPS * 32, 0, s>>>(c, p->d_rs_pos, m, p->d_rs_orig, p->d_start_r, o, rs); r += 1; }
            launches += 1;
        }
        CUDA_TRY(p, cudaGetLastError());
    }
    se_status st = SE_OK;
    for (int r = 0; r < nrhs && st == SE_OK; ++r) {
        p->ext_out_real = do_real ? p->d_out_real_b + rs * r : nullptr;
        st = apply_impl(p, nullptr, F + 3 * N * r, T + 3 * N * r, S + 5 * N * r, nullptr, U + 3 * N * r, Omega + 3 * N * r, E + 5 * N * r,
                        nullptr, cuda_stream, "far_mobility_apply_batch");
        launches += p->last_launches;
    }
    p->ext_out_real = nullptr;
    p->last_launches = launches;
    return st;
}

extern "C" se_status far_mobility_apply_host_async(se_plan *p, const double *pos, const double *F, const double *T,
                                                   const double *S, double *U, double *Omega, double *E, void *cuda_stream)
{
    if (!p) return SE_ERR_INVALID_ARG;
    if (!pos || !F || !T || !S || !U || !Omega || !E) return fail(p, SE_ERR_INVALID_ARG, "far_mobility_apply_host", "null pointer");
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const size_t N = (size_t)p->c.N, B = sizeof(double);
    double *d = p->d_io;
    double *dpos = d, *dF = d + 3 * N, *dT = d + 6 * N, *dS = d + 9 * N, *dU = d + 14 * N, *dW = d + 17 * N, *dE = d + 20 * N;
    CUDA_TRY(p, cudaMemcpyAsync(dpos, pos, 3 * N * B, cudaMemcpyHostToDevice, s));
    CUDA_TRY(p, cudaMemcpyAsync(dF, F, 3 * N * B, cudaMemcpyHostToDevice, s));
    CUDA_TRY(p, cudaMemcpyAsync(dT, T, 3 * N * B, cudaMemcpyHostToDevice, s));
    CUDA_TRY(p, cudaMemcpyAsync(dS, S, 5 * N * B, cudaMemcpyHostToDevice, s));
    se_status st = far_mobility_apply(p, dpos, dF, dT, dS, dU, dW, dE, cuda_stream);
    if (st != SE_OK) return st;
    CUDA_TRY(p, cudaMemcpyAsync(U, dU, 3 * N * B, cudaMemcpyDeviceToHost, s));
    CUDA_TRY(p, cudaMemcpyAsync(Omega, dW, 3 * N * B, cudaMemcpyDeviceToHost, s));
    CUDA_TRY(p, cudaMemcpyAsync(E, dE, 5 * N * B, cudaMemcpyDeviceToHost, s));
    return SE_OK;
}

extern "C" se_status far_mobility_apply_host(se_plan *p, const double *pos, const double *F, const double *T,
                                             const double *S, double *U, double *Omega, double *E, void *cuda_stream)
{
    const se_status st = far_mobility_apply_host_async(p, pos, F, T, S, U, Omega, E, cuda_stream);
    if (st != SE_OK) return st;
    CUDA_TRY(p, cudaStreamSynchronize((cudaStream_t)cuda_stream));
    return SE_OK;
}

extern "C" se_status se_self_image_blocks(se_plan *p, double *out, void *cuda_stream)
{
    if (!p) return SE_ERR_INVALID_ARG;
    if (!out) return fail(p, SE_ERR_INVALID_ARG, "se_self_image_blocks", "null pointer");
    cudaStream_t s = (cudaStream_t)cuda_stream;
    if (!p->d_blockW) { se_status st = dev_alloc(p, &p->d_blockW, 3 * 121); if (st != SE_OK) return st; }
    // the sums use their own splitting parameter xi_b = sqrt(pi)/L: real and wave parts converge equally fast
    SeConst cb = p->c;
    cb.xi = sqrt(M_PI) / cb.L;
    cb.q = 2.0 * cb.xi / sqrt(M_PI);
    cb.x2 = cb.xi * cb.xi; cb.x4 = cb.x2 * cb.x2; cb.x6 = cb.x4 * cb.x2; cb.x8 = cb.x4 * cb.x4; cb.x10 = cb.x8 * cb.x2; cb.x12 = cb.x6 * cb.x6;
    cb.inv4xi2 = 1.0 / (4.0 * cb.xi * cb.xi);
    // three distinct reference values of t = a^2 spanning the radii (any three distinct values give the same quadratic)
    const double t0 = p->a2min, t2 = p->a2max > 1.0001 * p->a2min ? p->a2max : 2.0 * p->a2min, t1 = 0.5 * (t0 + t2);
    k_block_lattice<<<dim3(11, 3), BLK_THREADS, 0, s>>>(cb, t0, t1, t2, p->d_blockW);
    const size_t n = (size_t)cb.N * 121;
    k_block_eval<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(cb, t0, t1, t2, p->d_blockW, p->d_radii, out);
    p->last_launches = 2;
    CUDA_TRY(p, cudaGetLastError());
    return SE_OK;
}

extern "C" se_status se_plan_copy_grids(se_plan *p, int which, double *dst)
{
    if (!p || !dst || which < 0 || which > 2) return SE_ERR_INVALID_ARG;
    const int M = p->c.M;
    const size_t G = (size_t)M * M * M, per = (size_t)p->gg.MYp * p->gg.MZp;
    if (which == 2 && !p->have_comp) return fail(p, SE_ERR_INVALID_ARG, "se_plan_copy_grids", "no compressible apply was made");
    CUDA_TRY(p, cudaDeviceSynchronize());
    if (which == 0 || (which == 2 && !p->real_p_padded)) {              // spread grids: plain [M][M][M]
        CUDA_TRY(p, cudaMemcpy(dst, which == 0 ? p->d_real : p->d_real_p, sizeof(double) * (which == 0 ? 3 : 1) * G, cudaMemcpyDeviceToHost));
        return SE_OK;
    }
    // returned grids: strip the periodic halo of the padded layout, plane by plane
    const double *src = which == 1 ? p->d_real : p->d_real_p;
    const size_t nplanes = (size_t)(which == 1 ? 6 : 1) * M;
    for (size_t pl = 0; pl < nplanes; ++pl)
        CUDA_TRY(p, cudaMemcpy2D(dst + pl * M * M, sizeof(double) * M, src + pl * per, sizeof(double) * p->gg.MZp, sizeof(double) * M, M,
                                 cudaMemcpyDeviceToHost));
    return SE_OK;
}

// Independent DFMA chains: 8 accumulators per thread, 4096 rounds, 8 CTAs of 256 threads per SM.
__global__ void __launch_bounds__(256) k_fp64_peak(double *sink, double a, double b, int rounds)
{
    double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    for (int r = 0; r < rounds; ++r) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
            x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
        }
    }
    const double s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
    if (s == 123.456) sink[0] = s;           // never true; keeps the chains alive
}

extern "C" se_status se_measure_fp64_peak(double *tflops, void *cuda_stream)
{
    if (!tflops) return SE_ERR_INVALID_ARG;
    *tflops = 0.0;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        cudaGetLastError();
        return SE_ERR_CUDA;
    }
    double *sink = nullptr;
    cudaEvent_t e0, e1;
    if (cudaMalloc((void **)&sink, 8) != cudaSuccess) { cudaGetLastError(); return SE_ERR_CUDA; }
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int rounds = 4096, blocks = sms * 8;
    float best = 1e30f;
    cudaError_t e = cudaSuccess;
    for (int rep = 0; rep < 4 && e == cudaSuccess; ++rep) {       // first repetition warms up
        cudaEventRecord(e0, s);
        k_fp64_peak<<<blocks, 256, 0, s>>>(sink, 0.999999, 1e-9, rounds);
        cudaEventRecord(e1, s);
        e = cudaEventSynchronize(e1);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(sink);
    if (e != cudaSuccess) { cudaGetLastError(); return SE_ERR_CUDA; }
    const double fma_count = (double)blocks * 256.0 * rounds * 64.0;
    *tflops = 2.0 * fma_count / (best * 1e-3) / 1e12;
    return SE_OK;
}

extern "C" se_status se_plan_get_timings(se_plan *p, double *ms)
{
    if (!p || !ms) return SE_ERR_INVALID_ARG;
    if (!p->timed) return fail(p, SE_ERR_INVALID_ARG, "se_plan_get_timings", "last apply was not made with SE_TIMING");
    CUDA_TRY(p, cudaEventSynchronize(p->ev[SE_NUM_STAGES]));
    for (int k = 0; k < SE_NUM_STAGES; ++k) {
        float t = 0.f;
        CUDA_TRY(p, cudaEventElapsedTime(&t, p->ev[k], p->ev[k + 1]));
        ms[k] = (double)t;
    }
    return SE_OK;
}

// ------------------------------------------------------------------------------------------------------------
// far_mobility_real_noalloc: the real-space pair sum (a2) for callers that cannot allocate (CUDA graph capture, serving
// loops, harnesses that forbid cudaMalloc).  No plan, no cudaMalloc / cudaFree, no cuFFT: the packed copies the pair kernel
// reads (wrapped positions + radius, the 12 moments per particle, the index map) and the 12 sums per particle it writes
// live in ONE file-scope device array of fixed size, SE_NOALLOC_MAX_N particles (1.9 MB, held by every GPU that loads the
// library until the process exits).  All pairs are scanned (no cell list), which is what the plan's kernel does too when
// L < 3 r_c; the launch sequence is  k_noalloc_pack -> k_real<false,1> (the plan's own pair kernel, reading the scratch)
// -> k_epilogue (real part only).
// The array's name is a host-side stand-in in host code, not a device address: its device address is asked for once per
// device (cudaGetSymbolAddress with that device current) and handed to the kernels.
// ------------------------------------------------------------------------------------------------------------
#define SE_NOALLOC_DOUBLES_PER_PARTICLE 29          // 4 (x, y, z, a) + 12 moments + 12 sums + 1 (the int index map, padded)
static __device__ __align__(256) double g_noalloc_scratch[(size_t)SE_NOALLOC_MAX_N * SE_NOALLOC_DOUBLES_PER_PARTICLE];

#define SE_NOALLOC_MAX_DEVICES 64
static double *g_noalloc_addr[SE_NOALLOC_MAX_DEVICES];     // device address of g_noalloc_scratch, per device ordinal (0 = not asked yet)
static std::mutex g_noalloc_mutex;

// wrapped position + radius, moments in the pair kernel's layout (slot 11, the pressure moment, zero), identity index map
__global__ void k_noalloc_pack(SeConst c, const double *__restrict__ pos, const double *__restrict__ radii, const double *__restrict__ F,
                               const double *__restrict__ T, const double *__restrict__ S, double4 *__restrict__ rs_pos,
                               double *__restrict__ rs_mom, int *__restrict__ rs_orig)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= c.N) return;
    double xw[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) se_grid_coord(c, pos + 3 * (size_t)i, d, &xw[d]);
    rs_pos[i] = make_double4(xw[0], xw[1], xw[2], radii[i]);
    double *m = rs_mom + 12 * (size_t)i;
#pragma unroll
    for (int k = 0; k < 3; ++k) { m[k] = F[3 * (size_t)i + k]; m[3 + k] = T[3 * (size_t)i + k]; }
#pragma unroll
    for (int k = 0; k < 5; ++k) m[6 + k] = S[5 * (size_t)i + k];
    m[11] = 0.0;
    rs_orig[i] = i;
}

static se_status noalloc_fail(char *err, size_t err_len, se_status st, const char *what, const char *detail)
{
    if (err && err_len) snprintf(err, err_len, "far_mobility_real_noalloc: %s: %s", what, detail);
    return st;
}

extern "C" se_status far_mobility_real_noalloc(int64_t N, double L, double xi, double r_c, double eta0, const double *pos,
                                               const double *radii, const double *F, const double *T, const double *S, double *U,
                                               double *Omega, double *E, void *cuda_stream, char *err, size_t err_len)
{
    if (err && err_len) err[0] = 0;
    if (N < 1) return noalloc_fail(err, err_len, SE_ERR_INVALID_ARG, "N", "must be at least 1");
    if (N > SE_NOALLOC_MAX_N) {
        char b[96];
        snprintf(b, sizeof(b), "N = %lld exceeds SE_NOALLOC_MAX_N = %d (size of the static device scratch)", (long long)N, SE_NOALLOC_MAX_N);
        return noalloc_fail(err, err_len, SE_ERR_INVALID_ARG, "N", b);
    }
    if (!(L > 0.0) || !(xi > 0.0) || !(eta0 > 0.0) || !(r_c > 0.0) || r_c > 0.5 * L || !std::isfinite(L) || !std::isfinite(xi))
        return noalloc_fail(err, err_len, SE_ERR_INVALID_ARG, "parameters", "need L, xi, eta0 > 0 and 0 < r_c <= L/2");
    if (!pos || !radii || !F || !T || !S || !U || !Omega || !E) return noalloc_fail(err, err_len, SE_ERR_INVALID_ARG, "pointers", "null pointer");

    // set-up, once per device: the device address of the static scratch array on the CURRENT device
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { cudaGetLastError(); return noalloc_fail(err, err_len, SE_ERR_CUDA, "cudaGetDevice", cudaGetErrorString(e)); }
    if (dev < 0 || dev >= SE_NOALLOC_MAX_DEVICES) return noalloc_fail(err, err_len, SE_ERR_UNSUPPORTED, "device", "ordinal beyond SE_NOALLOC_MAX_DEVICES");
    double *base = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_noalloc_mutex);
        if (!g_noalloc_addr[dev]) {
            void *ptr = nullptr;
            e = cudaGetSymbolAddress(&ptr, g_noalloc_scratch);
            if (e != cudaSuccess || !ptr) {
                cudaGetLastError();
                return noalloc_fail(err, err_len, SE_ERR_CUDA, "cudaGetSymbolAddress", e != cudaSuccess ? cudaGetErrorString(e) : "null address");
            }
            g_noalloc_addr[dev] = (double *)ptr;
        }
        base = g_noalloc_addr[dev];
    }
    double4 *rs_pos = reinterpret_cast<double4 *>(base);                               // [MAX_N] 32-byte elements at a 256-byte aligned base
    double *rs_mom = base + 4 * (size_t)SE_NOALLOC_MAX_N;                              // [MAX_N][12]
    double *out_real = rs_mom + 12 * (size_t)SE_NOALLOC_MAX_N;                         // [MAX_N][12]
    int *rs_orig = reinterpret_cast<int *>(out_real + 12 * (size_t)SE_NOALLOC_MAX_N);  // [MAX_N]

    SeConst c;
    memset(&c, 0, sizeof(c));
    c.N = (int)N; c.L = L; c.invL = 1.0 / L; c.xi = xi; c.eta0 = eta0; c.rc2 = r_c * r_c;
    c.ncr = 1; c.hr = L; c.gamma = 0.0;
    c.q = 2.0 * xi / sqrt(M_PI);
    c.x2 = xi * xi; c.x4 = c.x2 * c.x2; c.x6 = c.x4 * c.x2; c.x8 = c.x4 * c.x4; c.x10 = c.x8 * c.x2; c.x12 = c.x6 * c.x6;
    c.k0 = 1.0 / (8.0 * M_PI * eta0);

    cudaStream_t s = (cudaStream_t)cuda_stream;
    const int TB = 128, nbN = (c.N + TB - 1) / TB;
    // nothing in the scratch has to start at zero: the pack kernel writes every field the pair kernel reads, the pair kernel
    // writes sums 0..10 of every particle (it assigns on its first candidate chunk), the epilogue reads only those
    k_noalloc_pack<<<nbN, TB, 0, s>>>(c, pos, radii, F, T, S, rs_pos, rs_mom, rs_orig);
    k_real<false, 1><<<(unsigned)((c.N + 31) / 32), REAL_WARPS * 32, 0, s>>>(c, rs_pos, rs_mom, rs_orig, nullptr, out_real, 0);
    k_epilogue<<<nbN, TB, 0, s>>>(c, SE_SKIP_WAVE | SE_SKIP_SELF | SE_SKIP_ONEBODY, radii, F, T, S, out_real, nullptr, GATHER_SUMS, nullptr,
                                  U, Omega, E, nullptr, 0);
    e = cudaGetLastError();
    if (e != cudaSuccess) return noalloc_fail(err, err_len, SE_ERR_CUDA, "kernel launch", cudaGetErrorString(e));
    return SE_OK;
}
