// a4 / a6 along z by hand, with TRANSPOSED spectra (the default for power-of-two 32 <= M <= 512; SE_CUFFT3D turns it off).
//
// cuFFT's 3-D real transforms spend 0.62 of their 1.43 ms (c4) in the two kernels of the contiguous z axis
// (vector_fft_r2c / vector_fft_c2r, ~3.9 TB/s), and its strided 2-D plans are three times slower than its contiguous
// ones.  Here the z transforms are own kernels that write / read the half spectra with kz as the SLOWEST index,
//     spec[g][kz][x][y],   kz = 0 .. M/2,
// so that the remaining (x,y) transforms are cuFFT's fast contiguous batched 2-D complex plans (in place), and the
// k-space pass indexes the same layout (k_kspace<true>).  Same transforms as cuFFT's D2Z / Z2D (signs, no scaling).
//
// A real line h[0..M) is transformed as the complex line z_n = h[2n] + i h[2n+1] of length Nh = M/2 (a Stockham FFT of
// radix-16 register butterflies, one warp-local group of Nh/16 threads per line; se_xfft.cuh) plus the split step
//   forward:  X_k = 1/2 [ (Z_k + conj Z_{Nh-k}) - i w^k (Z_k - conj Z_{Nh-k}) ],  w = e^{-2 pi i / M},  k = 0 .. Nh  (Z_Nh = Z_0)
//   inverse:  Z_k = (X_k + conj X_{Nh-k}) + i w^{-k} (X_k - conj X_{Nh-k}),       k = 0 .. Nh-1,  z = FFT^-1_Nh Z.
// A CTA owns ZT_LINES consecutive y of one (grid, x): rows are read / written coalesced in z on the real side and
// as 256-byte runs in y on the spectral side (through shared memory, odd line pitch: conflict-free both ways).
// Measured at M = 256 on B200: r2c 0.16 ms (5.1 TB/s), c2r 0.31 ms (5.3 TB/s) against cuFFT's 3.9 TB/s for these passes.
#pragma once
#include "se_xyfft.cuh"

#ifndef ZT_LINES
#define ZT_LINES 16             // lines (consecutive y) per CTA: 16 measured best (8, 32 slower)
#endif
#ifndef ZT_MINB
#define ZT_MINB 4               // resident CTAs per SM aimed at for blocks of <= 128 threads (M <= 256); 5 spills and is slower
#endif

// pitch of a line in shared memory (complex values): skewed positions of Nh + 1 values, made odd
__host__ __device__ inline int zt_pitch(int Nh) { return (xf_sk<4>(Nh) + 1) | 1; }
static inline size_t zt_smem_bytes(int M) { return (size_t)(ZT_LINES * zt_pitch(M / 2) + M / 2 + M / 2 + 1) * 16; }
static inline int zt_threads(int M) { return ZT_LINES * (M / 2) / 16; }

// One Stockham stage on one line as xf_stage<4, R, INV> (se_xfft.cuh), with the line's input taken straight from
// global memory (GIN: the first stage of the forward transform reads the real row as Nh complex values) or its
// output written straight to global memory (GOUT: the last stage of the inverse transform writes the real row):
// two shared-memory passes fewer per transform.
// GOUT rows may carry a periodic halo (the padded layout of the returned grids, se_gather.cuh): the first hz values are
// stored again M further on, and the whole row a second time at gout2 (the halo row y + M) when gout2 is not NULL.
template <int R, bool INV, bool GIN, bool GOUT>
__device__ __forceinline__ void zt_stage(cplx *__restrict__ line, const double2 *__restrict__ gin, double2 *__restrict__ gout,
                                         const cplx *__restrict__ W, int M, int lNs, int jj, int hz = 0, double2 *__restrict__ gout2 = nullptr)
{
    constexpr int V = 16, NB = V / R;
    const int M16 = M >> 4, Ns = 1 << lNs;
    cplx v[V];
#pragma unroll
    for (int q = 0; q < V; ++q) {
        if (GIN) { const double2 t = __ldcs(gin + jj + q * M16); v[q] = { t.x, t.y }; }
        else v[q] = line[xf_sk<4>(jj + q * M16)];
    }
    if (!GIN) __syncwarp();
    const int twstep = M >> (lNs + (R == 16 ? 4 : R == 8 ? 3 : R == 4 ? 2 : 1));
#pragma unroll
    for (int u = 0; u < NB; ++u) {
        const int j = jj + u * M16, k = j & (Ns - 1);
        if (lNs > 0) {
#pragma unroll
            for (int r = 1; r < R; ++r) {
                cplx w = W[r * k * twstep];
                if (INV) w.y = -w.y;
                v[u + r * NB] = cmul(v[u + r * NB], w);
            }
        }
        RegFft<R, NB, INV>::run(v + u);
        const int base = ((j >> lNs) << lNs) * R + k;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            if (GOUT) {
                const int e = base + r * Ns;
                const double2 val = make_double2(v[u + r * NB].x, v[u + r * NB].y);
                __stcs(gout + e, val);
                if (e < hz) __stcs(gout + e + M, val);                 // M complex pairs = one period of the real row
                if (gout2) { __stcs(gout2 + e, val); if (e < hz) __stcs(gout2 + e + M, val); }
            } else line[xf_sk<4>(base + r * Ns)] = v[u + r * NB];
        }
    }
    if (!GOUT) __syncwarp();
}

// Length-Nh transform of one line (Nh = 2^lNh >= 16): radix-16 stages, then one stage of the remaining radix.
template <bool INV, bool GIN, bool GOUT>
__device__ __forceinline__ void zt_fft(cplx *__restrict__ line, const double2 *__restrict__ gin, double2 *__restrict__ gout,
                                       const cplx *__restrict__ W, int Nh, int lNh, int jj, int hz = 0, double2 *__restrict__ gout2 = nullptr)
{
    int lNs = 0;
    while (lNh - lNs >= 4) {
        const bool first = lNs == 0, last = lNs + 4 == lNh;
        if (GIN && first && GOUT && last) zt_stage<16, INV, true, true>(line, gin, gout, W, Nh, lNs, jj, hz, gout2);
        else if (GIN && first) zt_stage<16, INV, true, false>(line, gin, gout, W, Nh, lNs, jj);
        else if (GOUT && last) zt_stage<16, INV, false, true>(line, gin, gout, W, Nh, lNs, jj, hz, gout2);
        else zt_stage<16, INV, false, false>(line, gin, gout, W, Nh, lNs, jj);
        lNs += 4;
    }
    const int rem = lNh - lNs;                     // 0 .. 3: the last stage, never the first (Nh >= 16)
    if (rem == 3) { if (GOUT) zt_stage<8, INV, false, true>(line, gin, gout, W, Nh, lNs, jj, hz, gout2); else zt_stage<8, INV, false, false>(line, gin, gout, W, Nh, lNs, jj); }
    else if (rem == 2) { if (GOUT) zt_stage<4, INV, false, true>(line, gin, gout, W, Nh, lNs, jj, hz, gout2); else zt_stage<4, INV, false, false>(line, gin, gout, W, Nh, lNs, jj); }
    else if (rem == 1) { if (GOUT) zt_stage<2, INV, false, true>(line, gin, gout, W, Nh, lNs, jj, hz, gout2); else zt_stage<2, INV, false, false>(line, gin, gout, W, Nh, lNs, jj); }
}

// H: [ng][M][M][M] real -> spec: [ng][M/2+1][M][M] complex.  Wtab: [M] complex, exp(-2 pi i q / M).
// Grid: ng * M * (M / ZT_LINES) CTAs of ZT_LINES * Nh / 16 threads.
template <int NT>
__global__ void __launch_bounds__(NT, NT <= 128 ? ZT_MINB : 2) k_zfft_r2c(int M, int lNh, const double *__restrict__ H, double2 *__restrict__ spec,
                                                           const double2 *__restrict__ Wtab)
{
    extern __shared__ __align__(16) unsigned char zt_smem[];
    const int Nh = M >> 1, Zc = Nh + 1, LP = zt_pitch(Nh), nt = blockDim.x, tid = threadIdx.x;
    cplx *L = reinterpret_cast<cplx *>(zt_smem), *WN = L + ZT_LINES * LP, *WP = WN + Nh;
    const int nyb = M / ZT_LINES;
    const int yb = blockIdx.x % nyb, gx = blockIdx.x / nyb;               // gx = g * M + x
    const int y0 = yb * ZT_LINES, g = gx / M, x = gx - g * M;
    for (int q = tid; q < Nh; q += nt) { const double2 w = Wtab[2 * q]; WN[q] = { w.x, w.y }; }
    for (int q = tid; q <= Nh; q += nt) { const double2 w = q < M ? Wtab[q] : make_double2(1.0, 0.0); WP[q] = { w.x, w.y }; }
    const double2 *__restrict__ rows = reinterpret_cast<const double2 *>(H + ((size_t)gx * M + y0) * M);
    __syncthreads();                                   // twiddle tables
    {   // the first stage reads the real rows straight from global memory (sixteen loads per thread in flight)
        const int tpl = Nh >> 4, line = tid / tpl, jj = tid - line * tpl;
        zt_fft<false, true, false>(L + line * LP, rows + (size_t)line * Nh, nullptr, WN, Nh, lNh, jj);
    }
    __syncthreads();
    double2 *__restrict__ out = spec + (((size_t)g * Zc) * M + x) * M + y0;
    const size_t kstride = (size_t)M * M;
    // split step on the fly, the pair (k, Nh - k) from one read of Z_k and Z_{Nh-k}: k = 0 also gives X_Nh
    for (int e = tid; e < (Nh / 2 + 1) * ZT_LINES; e += nt) {
        const int k = e / ZT_LINES, r = e - k * ZT_LINES, km = Nh - k;
        const cplx zk = L[r * LP + xf_sk<4>(k)], zm = L[r * LP + xf_sk<4>(km & (Nh - 1))];
        auto xfrom = [&](cplx a, cplx b, cplx w) {                // 1/2 [ (a + conj b) - i w (a - conj b) ]
            const double sr = a.x + b.x, si = a.y - b.y, dr = a.x - b.x, di = a.y + b.y;
            return make_double2(0.5 * (sr + (w.x * di + w.y * dr)), 0.5 * (si - (w.x * dr - w.y * di)));
        };
        __stcs(out + (size_t)k * kstride + r, xfrom(zk, zm, WP[k]));
        if (km != k) __stcs(out + (size_t)km * kstride + r, xfrom(zm, zk, WP[km]));
    }
}

// spec: [ng][M/2+1][M][M] complex -> R: [ng][M][MYp][MZp] real (unnormalised inverse), rows and columns M .. M+halo-1
// repeating 0 .. halo-1 (the periodic halo the gather's tensor boxes read; halo = P - 1, MYp >= M + halo,
// MZp >= M + halo + 1 and even).
template <int NT>
__global__ void __launch_bounds__(NT, NT <= 128 ? ZT_MINB : 2) k_zfft_c2r(int M, int lNh, const double2 *__restrict__ spec, double *__restrict__ R,
                                                           const double2 *__restrict__ Wtab, int MYp, int MZp, int halo)
{
    extern __shared__ __align__(16) unsigned char zt_smem[];
    const int Nh = M >> 1, Zc = Nh + 1, LP = zt_pitch(Nh), nt = blockDim.x, tid = threadIdx.x;
    cplx *L = reinterpret_cast<cplx *>(zt_smem), *WN = L + ZT_LINES * LP, *WP = WN + Nh;
    const int nyb = M / ZT_LINES;
    const int yb = blockIdx.x % nyb, gx = blockIdx.x / nyb;
    const int y0 = yb * ZT_LINES, g = gx / M, x = gx - g * M;
    for (int q = tid; q < Nh; q += nt) { const double2 w = Wtab[2 * q]; WN[q] = { w.x, w.y }; }
    for (int q = tid; q <= Nh; q += nt) { const double2 w = q < M ? Wtab[q] : make_double2(1.0, 0.0); WP[q] = { w.x, -w.y }; }   // w^{-k}
    const double2 *__restrict__ in = spec + (((size_t)g * Zc) * M + x) * M + y0;
    const size_t kstride = (size_t)M * M;
    __syncthreads();                                   // twiddle tables
    // load with the split step fused: the pair (X_k, X_{Nh-k}) gives Z_k and Z_{Nh-k}; nine pairs per thread in flight
    {
        constexpr int NPQ = 9;                             // (Nh/2 + 1) ZT_LINES = 8 nt + ZT_LINES pairs
        double2 a[NPQ], b[NPQ];
        const int npair = (Nh / 2 + 1) * ZT_LINES;
#pragma unroll
        for (int q = 0; q < NPQ; ++q) {
            const int e = tid + q * nt;
            if (e < npair) {
                const int k = e / ZT_LINES, r = e - k * ZT_LINES;
                a[q] = __ldcs(in + (size_t)k * kstride + r);
                b[q] = __ldcs(in + (size_t)(Nh - k) * kstride + r);
            }
        }
#pragma unroll
        for (int q = 0; q < NPQ; ++q) {
            const int e = tid + q * nt;
            if (e < npair) {
                const int k = e / ZT_LINES, r = e - k * ZT_LINES, km = Nh - k;
                auto zfrom = [&](double2 x, double2 y, cplx w) {      // (x + conj y) + i w (x - conj y)
                    const double sr = x.x + y.x, si = x.y - y.y, dr = x.x - y.x, di = x.y + y.y;
                    return cplx{ sr - (w.x * di + w.y * dr), si + (w.x * dr - w.y * di) };
                };
                cplx *ln = L + r * LP;
                ln[xf_sk<4>(k)] = zfrom(a[q], b[q], WP[k]);
                if (km < Nh && km != k) ln[xf_sk<4>(km)] = zfrom(b[q], a[q], WP[km]);
            }
        }
    }
    __syncthreads();
    {   // the last stage writes the real rows straight to global memory
        const int tpl = Nh >> 4, line = tid / tpl, jj = tid - line * tpl;
        double2 *__restrict__ row = reinterpret_cast<double2 *>(R + ((size_t)gx * MYp + y0 + line) * MZp);
        double2 *__restrict__ row2 = y0 + line < halo ? row + (size_t)M * (MZp >> 1) : nullptr;      // halo row y + M
        zt_fft<true, false, true>(L + line * LP, nullptr, row, WN, Nh, lNh, jj, (halo + 1) >> 1, row2);
    }
}

// ------------------------------------------------------------------------------------------------------------
// (y,z) transforms fused in ONE pass over HBM by a thread-block cluster (power-of-two 32 <= M <= 256).
//
// The CS = M/32 CTAs of a cluster own one (grid, x) plane.  Forward: CTA `rank` transforms the 32 real rows
// y = 32 rank .. 32 rank + 31 along z as k_zfft_r2c does (lines in its own shared memory, split step in place), the
// cluster synchronises, and the same CTA then transforms along y the 16 lines kz = 16 rank .. 16 rank + 15: its threads
// read the 16 inputs of their first radix-16 stage straight out of the other CTAs' shared memory (distributed shared
// memory, ld.shared::cluster), 16 bytes each, and after a second cluster barrier the line buffers are reused for the
// exchange between the stages; the last stage writes spec[g][kz][x][.] (4 KB lines).  The Nyquist plane kz = M/2 is
// neither made nor read anywhere (the k-space pass zeroes it, reading 13).  Inverse: the mirror image -- y
// transforms of 16 kz lines, results in natural order in shared memory, cluster barrier, every CTA pulls the pairs
// (X_k, X_{M/2-k}) of its 32 rows from the owners, second barrier, split step + z transform + halo as k_zfft_c2r.
// A half spectrum crosses HBM once per direction instead of three times.
// ------------------------------------------------------------------------------------------------------------
#define YZ_LINES 32             // real rows (y) per CTA
#define YZ_KZ 16                // kz lines per CTA

__device__ __forceinline__ void cluster_sync_all()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t cluster_rank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
// 16-byte load from the shared memory of CTA `rank` of the cluster, at the address that is `p` in this CTA
__device__ __forceinline__ cplx ld_remote(const cplx *p, uint32_t rank)
{
    uint32_t ra;
    cplx v;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"((uint32_t)__cvta_generic_to_shared(p)), "r"(rank));
    asm volatile("ld.shared::cluster.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(ra) : "memory");
    return v;
}

template <int LM> struct YzTraits {
    static constexpr int M = 1 << LM, Nh = M / 2, M16 = M / 16, CS = M / YZ_LINES;
    static constexpr int NT = YZ_LINES * (Nh / 16);                  // = YZ_KZ * M16
    static constexpr int LPZ = ((Nh + (Nh >> 4)) + 1) | 1;           // pitch of a z line (zt_pitch(Nh))
    static constexpr int LPY = (M + (M >> 4) + 1) | 1;               // pitch of a y line
    static constexpr int LBUF = (YZ_LINES * LPZ > YZ_KZ * LPY) ? YZ_LINES * LPZ : YZ_KZ * LPY;
    static constexpr size_t SMEM = (size_t)(LBUF + Nh + Nh + 1 + M) * 16;
    static_assert(Nh / 16 <= 32 && M16 <= 32, "a line's threads sit in one warp");
};

// H: [ng][M][M][M] real -> spec: [ng][M/2+1][M][M] complex, planes kz < M/2 fully transformed along z and y.
template <int LM>
__global__ void __launch_bounds__(YzTraits<LM>::NT, (YzTraits<LM>::NT <= 256 ? 2 : 1)) k_yz_r2c(const double *__restrict__ H, double2 *__restrict__ spec, const double2 *__restrict__ Wtab)
{
    using TR = YzTraits<LM>;
    constexpr int M = TR::M, Nh = TR::Nh, Zc = Nh + 1, M16 = TR::M16, nt = TR::NT, LP = TR::LPZ;
    extern __shared__ __align__(16) unsigned char yz_smem[];
    cplx *L = reinterpret_cast<cplx *>(yz_smem), *WN = L + TR::LBUF, *WP = WN + Nh, *WY = WP + Nh + 1;
    const int tid = threadIdx.x;
    const uint32_t rank = cluster_rank();
    const int gx = blockIdx.x / TR::CS;                                // g * M + x
    const int g = gx / M, x = gx - g * M, y0 = (int)rank * YZ_LINES;
    for (int q = tid; q < Nh; q += nt) { const double2 w = Wtab[2 * q]; WN[q] = { w.x, w.y }; }
    for (int q = tid; q <= Nh; q += nt) { const double2 w = q < M ? Wtab[q] : make_double2(1.0, 0.0); WP[q] = { w.x, w.y }; }
    for (int q = tid; q < M; q += nt) { const double2 w = Wtab[q]; WY[q] = { w.x, w.y }; }
    const double2 *__restrict__ rows = reinterpret_cast<const double2 *>(H + ((size_t)gx * M + y0) * M);
    __syncthreads();
    {
        constexpr int tpl = Nh >> 4;
        const int line = tid / tpl, jj = tid - line * tpl;
        zt_fft<false, true, false>(L + line * LP, rows + (size_t)line * Nh, nullptr, WN, Nh, LM - 1, jj);
    }
    __syncthreads();
    // split step in place: the pair (k, Nh - k) from Z_k and Z_{Nh-k}; X_Nh is dropped
    for (int e = tid; e < (Nh / 2 + 1) * YZ_LINES; e += nt) {
        const int k = e / YZ_LINES, r = e - k * YZ_LINES, km = Nh - k;
        cplx *ln = L + r * LP;
        const cplx zk = ln[xf_sk<4>(k)], zm = ln[xf_sk<4>(km & (Nh - 1))];
        auto xfrom = [&](cplx a, cplx b, cplx w) {                // 1/2 [ (a + conj b) - i w (a - conj b) ]
            const double sr = a.x + b.x, si = a.y - b.y, dr = a.x - b.x, di = a.y + b.y;
            return cplx{ 0.5 * (sr + (w.x * di + w.y * dr)), 0.5 * (si - (w.x * dr - w.y * di)) };
        };
        ln[xf_sk<4>(k)] = xfrom(zk, zm, WP[k]);
        if (km != k && km < Nh) ln[xf_sk<4>(km)] = xfrom(zm, zk, WP[km]);
    }
    cluster_sync_all();                                                // every CTA's X[y][kz] is in place
    const int kzl = tid / M16, jj = tid - kzl * M16;
    const int kz = (int)rank * YZ_KZ + kzl;
    cplx v[16];
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        const int y = jj + q * M16;
        v[q] = ld_remote(L + (y % YZ_LINES) * LP + xf_sk<4>(kz), (uint32_t)(y / YZ_LINES));
    }
    cluster_sync_all();                                                // all remote reads done: the buffers may be reused
    cplx *ln = L + kzl * TR::LPY;
    fft16<LM, false>(v, WY, jj,
                     [&](int pos, cplx val) { ln[xf_sk<4>(pos)] = val; },
                     [&](int pos) { return ln[xf_sk<4>(pos)]; },
                     [] { __syncwarp(); }, [] { __syncwarp(); });
    double2 *__restrict__ row = spec + (((size_t)g * Zc + kz) * M + x) * M;
#pragma unroll
    for (int q = 0; q < 16; ++q) row[jj + q * M16] = make_double2(v[q].x, v[q].y);
}

// spec: [ng][M/2+1][M][M] complex (planes kz < M/2) -> R: [ng][M][MYp][MZp] real with periodic halo (see k_zfft_c2r).
template <int LM>
__global__ void __launch_bounds__(YzTraits<LM>::NT, (YzTraits<LM>::NT <= 256 ? 2 : 1)) k_yz_c2r(const double2 *__restrict__ spec, double *__restrict__ R, const double2 *__restrict__ Wtab,
                                                                int MYp, int MZp, int halo)
{
    using TR = YzTraits<LM>;
    constexpr int M = TR::M, Nh = TR::Nh, Zc = Nh + 1, M16 = TR::M16, nt = TR::NT, LP = TR::LPZ;
    extern __shared__ __align__(16) unsigned char yz_smem[];
    cplx *L = reinterpret_cast<cplx *>(yz_smem), *WN = L + TR::LBUF, *WP = WN + Nh, *WY = WP + Nh + 1;
    const int tid = threadIdx.x;
    const uint32_t rank = cluster_rank();
    const int gx = blockIdx.x / TR::CS;
    const int g = gx / M, x = gx - g * M, y0 = (int)rank * YZ_LINES;
    for (int q = tid; q < Nh; q += nt) { const double2 w = Wtab[2 * q]; WN[q] = { w.x, w.y }; }
    for (int q = tid; q <= Nh; q += nt) { const double2 w = q < M ? Wtab[q] : make_double2(1.0, 0.0); WP[q] = { w.x, -w.y }; }   // w^{-k}
    for (int q = tid; q < M; q += nt) { const double2 w = Wtab[q]; WY[q] = { w.x, w.y }; }
    __syncthreads();
    {   // inverse y transforms of this CTA's kz lines; results in natural order in the line buffers
        const int kzl = tid / M16, jj = tid - kzl * M16;
        const int kz = (int)rank * YZ_KZ + kzl;
        const double2 *__restrict__ row = spec + (((size_t)g * Zc + kz) * M + x) * M;
        cplx v[16];
#pragma unroll
        for (int q = 0; q < 16; ++q) { const double2 t = row[jj + q * M16]; v[q] = { t.x, t.y }; }
        cplx *ln = L + kzl * TR::LPY;
        fft16<LM, true>(v, WY, jj,
                        [&](int pos, cplx val) { ln[xf_sk<4>(pos)] = val; },
                        [&](int pos) { return ln[xf_sk<4>(pos)]; },
                        [] { __syncwarp(); }, [] { __syncwarp(); });
        __syncwarp();
#pragma unroll
        for (int q = 0; q < 16; ++q) ln[xf_sk<4>(jj + q * M16)] = v[q];
    }
    cluster_sync_all();
    // pull the pairs (X_k, X_{Nh-k}) of this CTA's rows from their owners; X_Nh = 0
    constexpr int NPQ = 9, npair = (Nh / 2 + 1) * YZ_LINES;              // npair = 8 nt + YZ_LINES
    cplx a[NPQ], b[NPQ];
#pragma unroll
    for (int q = 0; q < NPQ; ++q) {
        const int e = tid + q * nt;
        if (e < npair) {
            const int k = e / YZ_LINES, r = e - k * YZ_LINES, km = Nh - k, yy = xf_sk<4>(y0 + r);
            a[q] = ld_remote(L + (k % YZ_KZ) * TR::LPY + yy, (uint32_t)(k / YZ_KZ));
            b[q] = km < Nh ? ld_remote(L + (km % YZ_KZ) * TR::LPY + yy, (uint32_t)(km / YZ_KZ)) : cplx{ 0.0, 0.0 };
        }
    }
    cluster_sync_all();                                                // all remote reads done: the buffers may be reused
#pragma unroll
    for (int q = 0; q < NPQ; ++q) {
        const int e = tid + q * nt;
        if (e < npair) {
            const int k = e / YZ_LINES, r = e - k * YZ_LINES, km = Nh - k;
            auto zfrom = [&](cplx p, cplx s, cplx w) {              // (p + conj s) + i w (p - conj s)
                const double sr = p.x + s.x, si = p.y - s.y, dr = p.x - s.x, di = p.y + s.y;
                return cplx{ sr - (w.x * di + w.y * dr), si + (w.x * dr - w.y * di) };
            };
            cplx *ln = L + r * LP;
            ln[xf_sk<4>(k)] = zfrom(a[q], b[q], WP[k]);
            if (km < Nh && km != k) ln[xf_sk<4>(km)] = zfrom(b[q], a[q], WP[km]);
        }
    }
    __syncthreads();
    {
        constexpr int tpl = Nh >> 4;
        const int line = tid / tpl, jj = tid - line * tpl;
        double2 *__restrict__ row = reinterpret_cast<double2 *>(R + ((size_t)gx * MYp + y0 + line) * MZp);
        double2 *__restrict__ row2 = y0 + line < halo ? row + (size_t)M * (MZp >> 1) : nullptr;      // halo row y + M
        zt_fft<true, false, true>(L + line * LP, nullptr, row, WN, Nh, LM - 1, jj, (halo + 1) >> 1, row2);
    }
}
