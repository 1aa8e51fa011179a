// a7: Gaussian gather (Eq. 45 / Eq. 52 by the trapezoidal rule, L280) and a8: epilogue.
//   U_i  = D^3 sum_n gamma(d) (u~ + cF_i w~)
//   Om_i = D^3 sum_n al gamma(d) d x u~
//   E_i  = traceless part of D^3 sum_n al gamma(d) (d q + q d),  q = u~ + cS_i w~,   d = x_n - r_i
// over the same P^3 support as the spreading.
//
// Design: the mirror of the spreading sweep (se_sweep.cuh).  A thread owns one grid column (y,z) and sweeps
// along x with a window of P planes of three grids in registers, so every grid value is read from HBM once
// per segment, in coalesced 64-byte rows.  Two "roles" share the work: role 0 sweeps u~ (grids 0-2), role 1
// sweeps w~ = lap u~ (grids 3-5).  For every particle whose support starts at the window's first plane and
// covers the column, the thread reduces along x,
//     m0[g] = sum_k gx(k) g(p+k),   m1[g] = sum_k gx(k) dx_k g(p+k),
// and weights them with the (y,z) Gaussian: the twelve sums  gyz {m0, m1, dy m0, dz m0}[g]  are all that
// U, Omega and E need.  They are reduced over the warp (reduce-scatter: 18 shuffles for 12 values) and added
// with one fp64 reduction per value into moments[N][24] (caller order); a8 combines them per particle.
#pragma once
#include "se_sweep.cuh"

#define GATHER_SUMS 24             // per particle: role 0 (u~) sums 0..11, role 1 (w~) sums 12..23

// Warp reduce-scatter of v[0..11]: returns in every lane the total of value (lane>>4)*6 + ((lane>>3)&1)*3 + t
// for t = 0,1,2 in out[t].
__device__ __forceinline__ void warp_reduce12(const double (&v)[12], int lane, double (&out)[3])
{
    const bool hi16 = (lane & 16) != 0, hi8 = (lane & 8) != 0;
    double a[6];
#pragma unroll
    for (int i = 0; i < 6; ++i) {
        const double keep = hi16 ? v[i + 6] : v[i], send = hi16 ? v[i] : v[i + 6];
        a[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
    }
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        const double keep = hi8 ? a[i + 3] : a[i], send = hi8 ? a[i] : a[i + 3];
        double t = keep + __shfl_xor_sync(0xffffffffu, send, 8);
        t += __shfl_xor_sync(0xffffffffu, t, 4);
        t += __shfl_xor_sync(0xffffffffu, t, 2);
        t += __shfl_xor_sync(0xffffffffu, t, 1);
        out[i] = t;
    }
}

template <int P>
__device__ __forceinline__ void gather_hit(const SeConst &c, const double *__restrict__ rec, int y, int z, bool active,
                                           const double (&win)[P][3], int role, int lane, double *__restrict__ moments)
{
    const int M = c.M;
    const int2 yz = *reinterpret_cast<const int2 *>(rec);
    int ry = y - yz.x, rz = z - yz.y;
    ry += ry < 0 ? M : 0;
    rz += rz < 0 ? M : 0;
    const bool hit = active && ry < P && rz < P;
    if (!__any_sync(0xffffffffu, hit)) return;
    double v[12];
#pragma unroll
    for (int i = 0; i < 12; ++i) v[i] = 0.0;
    if (hit) {
        const double Delta = c.Delta;
        // two partial sums per moment (even / odd planes) keep the FP64 pipe busy with few resident warps
        double m0[2][3] = { { 0.0, 0.0, 0.0 }, { 0.0, 0.0, 0.0 } }, m1[2][3] = { { 0.0, 0.0, 0.0 }, { 0.0, 0.0, 0.0 } };
        const double *__restrict__ X0 = rec + SE_REC_HDR, *__restrict__ X1 = rec + SE_REC_HDR + 3 * P;
#pragma unroll
        for (int k = 0; k < P; ++k) {
            const double gx = X0[k], gxd = X1[k];
#pragma unroll
            for (int g = 0; g < 3; ++g) {
                m0[k & 1][g] = fma(gx, win[k][g], m0[k & 1][g]);
                m1[k & 1][g] = fma(gxd, win[k][g], m1[k & 1][g]);
            }
        }
        const double dy = rec[REC_D0 + 1] + ry * Delta, dz = rec[REC_D0 + 2] + rz * Delta;
        const double gyz = rec[SE_REC_HDR + P + ry] * rec[SE_REC_HDR + 2 * P + rz];
        const double wy = gyz * dy, wz = gyz * dz;
#pragma unroll
        for (int g = 0; g < 3; ++g) {
            const double s0 = m0[0][g] + m0[1][g], s1 = m1[0][g] + m1[1][g];
            v[g] = gyz * s0;
            v[3 + g] = gyz * s1;
            v[6 + g] = wy * s0;
            v[9 + g] = wz * s0;
        }
    }
    double tot[3];
    warp_reduce12(v, lane, tot);
    const int orig = reinterpret_cast<const int2 *>(rec)[1].y;
    const int t = lane & 7;
    if (t < 3) {
        const int q = (lane >> 4) * 6 + ((lane >> 3) & 1) * 3;
        atomicAdd(moments + (size_t)orig * GATHER_SUMS + role * 12 + q + t, t == 0 ? tot[0] : (t == 1 ? tot[1] : tot[2]));
    }
}

// Grid: nseg * 2 roles * npatch warps.  Segment s handles the particles whose support starts in planes
// [s*seg_len, (s+1)*seg_len) and reads planes up to P-1 beyond.
template <int P>
__global__ void __launch_bounds__(SWEEP_WARPS * 32, SWEEP_MIN_BLOCKS) k_gather(SeConst c, const double *__restrict__ recs,
                                                              const int *__restrict__ start_s, const double *__restrict__ Gr,
                                                              double *__restrict__ moments)
{
    extern __shared__ __align__(16) unsigned char sweep_smem[];
    const int lane = threadIdx.x & 31, wl = threadIdx.x >> 5;
    const int wid = blockIdx.x * SWEEP_WARPS + wl;
    const int npatch = c.NBY * c.NBZ;
    const int sr = wid / npatch, patch = wid - sr * npatch;
    if (sr >= 2 * c.nseg) return;
    const int seg = sr >> 1, role = sr & 1;
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
    const int seg_start = seg * c.seg_len, seg_end = min(seg_start + c.seg_len, M);
    const size_t G = (size_t)M * M * M, MM = (size_t)M * M;
    const double *__restrict__ g0 = Gr + (size_t)(3 * role) * G + (active ? (size_t)y * M + z : 0);
    auto plane = [&](int q) { return (size_t)(q >= M ? q - M : q) * MM; };

    int p = seg_start;
    SweepList cur = sweep_scan(sweep_load(rg, start_s, p * npatch, lane), lane);
    sweep_stage(cur, recs, stride, smem_u32(slot0), bar0, lane);
    int2 raw = sweep_load(rg, start_s, min(p + 1, seg_end - 1) * npatch, lane);

    double win[P][3], nx[3];
#pragma unroll
    for (int k = 0; k < P - 1; ++k) {
        const size_t o = plane(p + k);
#pragma unroll
        for (int g = 0; g < 3; ++g) win[k][g] = active ? g0[g * G + o] : 0.0;
    }
    {
        const size_t o = plane(p + P - 1);
#pragma unroll
        for (int g = 0; g < 3; ++g) nx[g] = active ? g0[g * G + o] : 0.0;
    }
    unsigned parity = 0;
    for (int buf = 0; p < seg_end; ++p, buf ^= 1) {
#pragma unroll
        for (int g = 0; g < 3; ++g) win[P - 1][g] = nx[g];
        SweepList nxt;
        nxt.js = 0; nxt.cnt = 0; nxt.off = 0; nxt.n = 0;
        if (p + 1 < seg_end) {
            nxt = sweep_scan(raw, lane);
            sweep_stage(nxt, recs, stride, smem_u32(buf ? slot0 : slot1), buf ? bar0 : bar1, lane);
            raw = sweep_load(rg, start_s, min(p + 2, seg_end - 1) * npatch, lane);
            const size_t o = plane(p + P);                    // last plane of the next window
#pragma unroll
            for (int g = 0; g < 3; ++g) nx[g] = active ? g0[g * G + o] : 0.0;
        }
        if (cur.n > 0) {
            mbar_wait(buf ? bar1 : bar0, (parity >> buf) & 1u);
            parity ^= 1u << buf;
            const double *__restrict__ sl = buf ? slot1 : slot0;
            const int ns = min(cur.n, SWEEP_CAP);
            for (int ci = 0; ci < ns; ++ci) gather_hit<P>(c, sl + (size_t)ci * stride, y, z, active, win, role, lane, moments);
            for (int ci = SWEEP_CAP; ci < cur.n; ++ci) {
                const int j = sweep_overflow_index(cur, ci);
                gather_hit<P>(c, recs + (size_t)j * stride, y, z, active, win, role, lane, moments);
            }
            __syncwarp();
        }
#pragma unroll
        for (int k = 0; k < P - 1; ++k) { win[k][0] = win[k + 1][0]; win[k][1] = win[k + 1][1]; win[k][2] = win[k + 1][2]; }
        cur = nxt;
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
                           const double *__restrict__ out_real, const double *__restrict__ moments,
                           double *__restrict__ U, double *__restrict__ W, double *__restrict__ E)
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
        const double *orl = out_real + 11 * (size_t)i;
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
}
