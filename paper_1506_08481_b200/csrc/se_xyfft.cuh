// a4 / a5 / a6 in the (x,y) directions by hand, on the TRANSPOSED half spectra spec[g][kz][x][y] of se_zfft.cuh
// (power-of-two 32 <= M <= 512).  Two kernels replace cuFFT's batched 2-D plans and the separate k-space pass:
//
//   k_yfft   the y transforms: lines of M contiguous complex values, in place, one smem round trip per radix-16 stage
//            boundary (the first stage reads global memory, the last writes it).
//   k_xmid   ONE pass over HBM for: forward x transform of the three spectra H_k, the k-space scaling of
//            PAPER.md Eq. 43 with the kernel of Eq. 36 and the hybrid Laplacian of Eq. 50-51 (L326)
//                u_k = s(k) (H_k - k (k.H_k)/k^2),   w_k = -k^2 u_k,
//                s(k) = [Delta^3/(eta0 V)] (1 + k^2/4xi^2) exp(-(1-eta_se) k^2/4xi^2)/k^2,
//            zero at k = 0 and on the Nyquist planes (reading 13), and the six inverse x transforms.
//            A CTA owns one kz and YB consecutive y: lines along x (stride M) with YB-wide contiguous runs; a thread
//            owns 16 points of one line of one component.  The forward result stays in registers in natural order,
//            which is exactly the register order the first inverse stage wants, so the k-space arithmetic and both
//            inverse transforms (u first, then w = -k^2 u from a register copy) need no extra pass over shared memory
//            beyond one exchange of the three components.  exp(-(1-eta_se) k^2/4xi^2) is separable and comes from a
//            per-axis table.  Compressible extension (a9; Eq. 33-34, 29-31): a fourth thread group transforms the
//            scalar spectrum Hs_k, adds its source term to u_k and makes the pressure spectrum
//                u_k += [Delta^3/(4 eta0 V)] (-i k/k^2) e^{...} Hs_k,   p_k = [Delta^3/V] (-i k.H_k/k^2) e^{...}
//            (signs for the e^{-ik.x} forward transform used here; see se_kspace.cuh).
//
// Stockham autosort stages of radix 16 (then one of the remaining radix 2/4/8) on 16 values per thread: before a stage
// a thread holds v[q] = x[jj + q M/16]; after the last stage v[q] = X[jj + q M/16] (natural order).
#pragma once
#include "se_xfft.cuh"

// twiddles and butterflies of the stage with Ns = 2^LNS (product of earlier radices), radix R
template <int LM, int LNS, int R, bool INV>
__device__ __forceinline__ void fs_core(cplx (&v)[16], const cplx *__restrict__ W, int jj)
{
    constexpr int M = 1 << LM, M16 = M >> 4, NB = 16 / R, Ns = 1 << LNS;
    constexpr int LR = R == 16 ? 4 : R == 8 ? 3 : R == 4 ? 2 : 1;
    constexpr int twstep = M >> (LNS + LR);                           // M / (Ns R)
#pragma unroll
    for (int u = 0; u < NB; ++u) {
        const int k = (jj + u * M16) & (Ns - 1);
        if (LNS > 0) {
#pragma unroll
            for (int r = 1; r < R; ++r) {
                cplx w = W[r * k * twstep];
                if (INV) w.y = -w.y;
                v[u + r * NB] = cmul(v[u + r * NB], w);
            }
        }
        RegFft<R, NB, INV>::run(v + u);
    }
}

// autosort position of output r of butterfly u
template <int LM, int LNS, int R>
__device__ __forceinline__ int fs_dst(int jj, int u, int r)
{
    constexpr int M16 = (1 << LM) >> 4, Ns = 1 << LNS;
    const int j = jj + u * M16, k = j & (Ns - 1);
    return ((j >> LNS) << LNS) * R + k + r * Ns;
}

// between two stages: store to the exchange line (st(pos, value)), synchronise, load the next stage's inputs (ld(pos)).
// syw() is called before the stores (the line may still be read by others), syr() after them.
template <int LM, int LNS, int R, typename St, typename Ld, typename SyW, typename SyR>
__device__ __forceinline__ void fs_exchange(cplx (&v)[16], int jj, St st, Ld ld, SyW syw, SyR syr)
{
    constexpr int NB = 16 / R, M16 = (1 << LM) >> 4;
    syw();
#pragma unroll
    for (int u = 0; u < NB; ++u)
#pragma unroll
        for (int r = 0; r < R; ++r) st(fs_dst<LM, LNS, R>(jj, u, r), v[u + r * NB]);
    syr();
#pragma unroll
    for (int q = 0; q < 16; ++q) v[q] = ld(jj + q * M16);
}

// Length-2^LM transform of the line this thread shares with M/16 - 1 others: v[q] = x[jj + q M/16] in, X[jj + q M/16] out.
template <int LM, bool INV, typename St, typename Ld, typename SyW, typename SyR>
__device__ __forceinline__ void fft16(cplx (&v)[16], const cplx *__restrict__ W, int jj, St st, Ld ld, SyW syw, SyR syr)
{
    static_assert(LM >= 5 && LM <= 9, "32 <= M <= 512");
    constexpr int NS16 = LM / 4, REM = LM % 4;
    fs_core<LM, 0, 16, INV>(v, W, jj);
    fs_exchange<LM, 0, 16>(v, jj, st, ld, syw, syr);
    if constexpr (NS16 == 1) {                       // M = 32, 64, 128: 16 x {2, 4, 8}
        fs_core<LM, 4, (1 << REM), INV>(v, W, jj);
    } else {                                         // M = 256, 512: 16 x 16 (x 2)
        fs_core<LM, 4, 16, INV>(v, W, jj);
        if constexpr (REM != 0) {
            fs_exchange<LM, 4, 16>(v, jj, st, ld, syw, syr);
            fs_core<LM, 8, (1 << REM), INV>(v, W, jj);
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
// y transforms: spec[g][kz][x][.] for kz < M/2 (the Nyquist plane kz = M/2 is never used: the k-space pass zeroes it),
// in place.  M/16 threads of one warp per line, YF_THREADS / (M/16) lines per CTA.
// ------------------------------------------------------------------------------------------------------------
#define YF_THREADS 128
template <int LM> struct YfTraits {
    static constexpr int M = 1 << LM, M16 = M >> 4, LPC = YF_THREADS / M16;
    static constexpr int PITCH = (M + (M >> 4) + 1) | 1;             // skewed positions of M values, odd
    static constexpr size_t SMEM = (size_t)(LPC * PITCH + M) * 16;
};

template <int LM, bool INV>
__global__ void __launch_bounds__(YF_THREADS, 4) k_yfft(double2 *__restrict__ spec, const double2 *__restrict__ Wtab, int ngrids)
{
    using TR = YfTraits<LM>;
    constexpr int M = TR::M, M16 = TR::M16, Nh = M / 2, Zc = Nh + 1;
    extern __shared__ __align__(16) unsigned char yf_smem[];
    cplx *L = reinterpret_cast<cplx *>(yf_smem), *W = L + TR::LPC * TR::PITCH;
    const int tid = threadIdx.x;
    for (int q = tid; q < M; q += YF_THREADS) { const double2 w = Wtab[q]; W[q] = { w.x, w.y }; }
    __syncthreads();
    const int line = tid / M16, jj = tid - line * M16;
    const size_t per = (size_t)Nh * M;                                // lines per grid
    const size_t gl = (size_t)blockIdx.x * TR::LPC + line;
    const bool valid = gl < per * ngrids;
    const size_t g = valid ? gl / per : 0, rem = valid ? gl - g * per : 0;
    double2 *__restrict__ row = spec + (g * Zc * M + rem) * M;
    cplx *ln = L + line * TR::PITCH;
    cplx v[16];
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        const double2 t = valid ? row[jj + q * M16] : make_double2(0.0, 0.0);
        v[q] = { t.x, t.y };
    }
    fft16<LM, INV>(v, W, jj,
                   [&](int pos, cplx val) { ln[xf_sk<4>(pos)] = val; },
                   [&](int pos) { return ln[xf_sk<4>(pos)]; },
                   [] { __syncwarp(); }, [] { __syncwarp(); });
    if (valid) {
#pragma unroll
        for (int q = 0; q < 16; ++q) row[jj + q * M16] = make_double2(v[q].x, v[q].y);
    }
}

// ------------------------------------------------------------------------------------------------------------
// x transforms fused with the k-space pass
// ------------------------------------------------------------------------------------------------------------
#ifndef XM_MINB
#define XM_MINB 2                  // resident CTAs per SM k_xmid is compiled for when a CTA has <= 192 threads (3: spills, slower)
#endif
template <int LM, int YB, bool COMP> struct XmTraits {
    static constexpr int M = 1 << LM, M16 = M >> 4;
    static constexpr int NG = COMP ? 4 : 3;                           // thread groups: H_x, H_y, H_z (, Hs)
    static constexpr int GT = YB * M16;                               // threads per group
    static constexpr int NT = NG * GT;
    static constexpr bool NAMED = (GT % 32) == 0;                     // a group is whole warps: named barriers
    static constexpr int PITCH = M + (M >> 4) + 1;                    // rows (x positions, skewed) per component
    static constexpr size_t SMEM = ((size_t)NG * PITCH * YB + M) * 16 + (size_t)M * 8;
};

// SHEAR: k = (2 pi/L)(jx, jy - gamma jx, jz) in the Green's function, the projector and w = -k^2 u; the Gaussians are
// deconvolved in the FRACTIONAL wave number, so the factor is e^{-k^2/4xi^2} (one exponential per mode) times the separable
// e^{+eta_se kq^2/4xi^2} from the table (then Etab holds that factor).
template <int LM, int YB, bool COMP, bool SHEAR>
__global__ void __launch_bounds__(XmTraits<LM, YB, COMP>::NT, (XmTraits<LM, YB, COMP>::NT <= 192 ? XM_MINB : 1))
k_xmid(SeConst c, const double2 *__restrict__ Hk, const double2 *__restrict__ Hsk, double2 *__restrict__ Gk,
       double2 *__restrict__ Pk, const double2 *__restrict__ Wtab, const double *__restrict__ Etab)
{
    using TR = XmTraits<LM, YB, COMP>;
    constexpr int M = TR::M, M16 = TR::M16, Nh = M / 2, Zc = Nh + 1, GT = TR::GT, PITCH = TR::PITCH;
    extern __shared__ __align__(16) unsigned char xm_smem[];
    cplx *E = reinterpret_cast<cplx *>(xm_smem);                      // [NG][PITCH][YB]
    cplx *W = E + (size_t)TR::NG * PITCH * YB;                        // [M]
    double *ET = reinterpret_cast<double *>(W + M);                   // [M] exp(-(1-eta_se) k_i^2 / 4 xi^2)
    const int tid = threadIdx.x;
    for (int q = tid; q < M; q += TR::NT) { const double2 w = Wtab[q]; W[q] = { w.x, w.y }; ET[q] = Etab[q]; }
    const int y = tid % YB, jj = (tid / YB) % M16, grp = tid / GT;
    constexpr int NYB = M / YB;
    const int kz = blockIdx.x / NYB, iy = (blockIdx.x - kz * NYB) * YB + y;
    const size_t Gc = (size_t)Zc * M * M;
    const size_t off = ((size_t)kz * M) * M + iy;                     // + x * M
    auto group_sync = [&] {
        if constexpr (TR::NAMED) asm volatile("bar.sync %0, %1;" ::"r"(grp + 1), "n"(GT) : "memory");
        else __syncthreads();
    };
    cplx *Eg = E + (size_t)grp * PITCH * YB + y;
    auto st = [&](int pos, cplx val) { Eg[xf_sk<4>(pos) * YB] = val; };
    auto ld = [&](int pos) { return Eg[xf_sk<4>(pos) * YB]; };

    cplx v[16];
    if (kz == Nh) {                                   // Nyquist plane: zeros, nothing is read
        if (grp < 3) {
#pragma unroll
            for (int q = 0; q < 16; ++q) {
                const size_t a = off + (size_t)(jj + q * M16) * M;
                Gk[grp * Gc + a] = make_double2(0.0, 0.0);
                Gk[(3 + grp) * Gc + a] = make_double2(0.0, 0.0);
            }
        } else if (Pk) {
#pragma unroll
            for (int q = 0; q < 16; ++q) Pk[off + (size_t)(jj + q * M16) * M] = make_double2(0.0, 0.0);
        }
        return;
    }
    {
        const double2 *__restrict__ src = grp < 3 ? Hk + grp * Gc : Hsk;
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            const double2 t = src ? src[off + (size_t)(jj + q * M16) * M] : make_double2(0.0, 0.0);
            v[q] = { t.x, t.y };
        }
    }
    __syncthreads();                                  // twiddle and exp tables
    fft16<LM, false>(v, W, jj, st, ld, group_sync, group_sync);

    // ---- exchange of the components, k-space arithmetic ----
    group_sync();                                     // the group's exchange rows are no longer read
#pragma unroll
    for (int q = 0; q < 16; ++q) st(jj + q * M16, v[q]);
    __syncthreads();
    cplx uu[16];
    const int jy = iy < Nh ? iy : iy - M;
    const double ky0 = c.twopiL * jy, kzv = c.twopiL * kz;
    const double eyz = ET[iy] * ET[kz], kyz2 = ky0 * ky0 + kzv * kzv;
    const cplx *E0 = E + y, *E1 = E0 + (size_t)PITCH * YB, *E2 = E1 + (size_t)PITCH * YB, *E3 = E2 + (size_t)PITCH * YB;
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        const int ix = jj + q * M16, ps = xf_sk<4>(ix) * YB;
        const int jx = ix < Nh ? ix : ix - M;
        const double kx = c.twopiL * jx;
        const double ky = SHEAR ? c.twopiL * ((double)jy - c.gamma * (double)jx) : ky0;
        const double k2 = SHEAR ? kx * kx + ky * ky + kzv * kzv : kx * kx + kyz2;
        const bool zero = (ix == 0 && iy == 0 && kz == 0) || ix == Nh || iy == Nh;
        const double inv = zero ? 0.0 : 1.0 / k2;
        const double dec = SHEAR ? exp(-k2 * c.inv4xi2) * (ET[ix] * eyz) : ET[ix] * eyz;
        const cplx h0 = grp == 0 ? v[q] : E0[ps], h1 = grp == 1 ? v[q] : E1[ps], h2 = grp == 2 ? v[q] : E2[ps];
        const double pr = (kx * h0.x + ky * h1.x + kzv * h2.x) * inv, pi = (kx * h0.y + ky * h1.y + kzv * h2.y) * inv;
        cplx r;
        if (grp < 3) {
            const double sc = zero ? 0.0 : c.scale0 * (1.0 + k2 * c.inv4xi2) * dec * inv;
            const double kc = grp == 0 ? kx : (grp == 1 ? ky : kzv);
            r = { sc * (v[q].x - kc * pr), sc * (v[q].y - kc * pi) };
            if (COMP) {                               // -i (x + i y) = y - i x
                const cplx hs = E3[ps];
                const double cs = 0.25 * c.scale0 * dec * inv * kc;
                r.x += cs * hs.y; r.y -= cs * hs.x;
            }
        } else {
            const double cp = zero ? 0.0 : c.scale0 * c.eta0 * dec;   // Delta^3 / V
            r = { cp * pi, -cp * pr };
        }
        uu[q] = r;
        v[q] = r;
    }
    __syncthreads();                                  // every group has read the others' rows
    // ---- inverse transforms: u (and p), then w = -k^2 u ----
    fft16<LM, true>(v, W, jj, st, ld, group_sync, group_sync);
    {
        double2 *__restrict__ dst = grp < 3 ? Gk + grp * Gc : Pk;
        if (dst) {
#pragma unroll
            for (int q = 0; q < 16; ++q) dst[off + (size_t)(jj + q * M16) * M] = make_double2(v[q].x, v[q].y);
        }
    }
    if (COMP && grp == 3 && TR::NAMED) return;        // the fourth group has no second round (its barriers are its own)
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        const int ix = jj + q * M16, jx = ix < Nh ? ix : ix - M;
        const double kx = c.twopiL * jx, kys = c.twopiL * ((double)jy - c.gamma * (double)jx);
        const double k2 = SHEAR ? kx * kx + kys * kys + kzv * kzv : kx * kx + kyz2;
        v[q] = { -k2 * uu[q].x, -k2 * uu[q].y };
    }
    fft16<LM, true>(v, W, jj, st, ld, group_sync, group_sync);
    if (grp < 3) {
        double2 *__restrict__ dst = Gk + (3 + grp) * Gc;
#pragma unroll
        for (int q = 0; q < 16; ++q) dst[off + (size_t)(jj + q * M16) * M] = make_double2(v[q].x, v[q].y);
    }
}
