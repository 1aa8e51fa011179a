// Shared definitions of the CUDA path (sm_100a).  No code here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define SE_PMAX 24                 // largest supported Gaussian support per axis
#define SE_TILE_Y 4                // spreading patch: 4 (y) x 8 (z) grid columns per warp
#define SE_TILE_Z 8
#define SE_REC_HDR 24              // doubles before the per-axis Gaussian tables in a particle record

// Constants of one plan, passed by value to every kernel.
struct SeConst {
    int N, M, P;
    int ncr;                       // real-space cells per axis (1 = all pairs)
    int NBY, NBZ;                  // spreading tile bins per plane: ceil(M/4), ceil(M/8)
    int rec_stride;                // doubles per spreading record
    int grec_stride;               // doubles per gather record
    int nseg, seg_len;             // sweep segments of the spreading kernel
    double L, MoverL, Delta, alpha, gnorm, eta_se;
    double xi, rc2, eta0, hr;      // hr = real-space cell edge L/ncr
    // real-space pair constants: q = 2 xi/sqrt(pi), powers of xi^2, k0 = 1/(8 pi eta0)
    double q, x2, x4, x6, x8, x10, x12, k0;
    // k-space: scale0 = Delta^3/(eta0 V), inv4xi2 = 1/(4 xi^2), dec = (1 - eta_se)/(4 xi^2), twopiL = 2 pi/L
    double scale0, inv4xi2, dec, twopiL;
    double D3;                     // Delta^3 (gather quadrature weight)
    // sheared (Lees-Edwards) lattice a1 = (L,0,0), a2 = (gamma L, L, 0), a3 = (0,0,L):
    double gamma, invL;            // strain (0 = cubic box: every kernel then takes its original path); 1/L
};

// Position of a particle on the grid axis d.  Cubic box: the wrapped coordinate x - L floor(x/L) (returned in *xw) times M/L.
// Sheared lattice: the wrapped FRACTIONAL coordinate t = A^{-1} r = ((x - gamma y)/L, y/L, z/L), t - floor(t) (returned in
// *xw, times L), times M -- evaluated without fused multiply-adds, in the order the oracle uses, so that both sides choose
// the same support for a particle that sits on a grid plane.
__device__ __forceinline__ double se_grid_coord(const SeConst &c, const double *__restrict__ pos3, int d, double *xw)
{
    if (c.gamma == 0.0) {
        const double x = pos3[d];
        *xw = x - c.L * floor(x / c.L);
        return *xw * c.MoverL;
    }
    const double t = d == 0 ? __dmul_rn(__dsub_rn(pos3[0], __dmul_rn(c.gamma, pos3[1])), c.invL) : __dmul_rn(pos3[d], c.invL);
    const double tw = t - floor(t);
    *xw = tw * c.L;
    return __dmul_rn(tw, (double)c.M);
}

// Minimum image of a separation (r_c <= L/2: at most one image lies within r_c, and it is this one).  Sheared lattice: the
// y and z images by rounding, then the x image given the shift gamma L of the chosen y image.
__device__ __forceinline__ void se_min_image(const SeConst &c, double &dx, double &dy, double &dz)
{
    const double n1 = rint(dy * c.invL);
    dy -= c.L * n1;
    if (c.gamma != 0.0) dx -= c.gamma * c.L * n1;
    dx -= c.L * rint(dx * c.invL);
    dz -= c.L * rint(dz * c.invL);
}

// Spreading record (AoS, rec_stride doubles, 16-byte aligned), in spreading-tile order:
//   [0]  int2 (y0w, z0w)   wrapped first support index along y, z
//   [1]  int2 (x0w, orig)  wrapped first support plane along x (the sweep axis), caller index
//   [2..4]   d0x, d0y, d0z   offset of the first support point from the particle, (n0 - u) Delta
//   [5..8]   f0, f1, s0, s1  size polynomials: 1-6 al cF, 4 al^2 cF, 2 al (1-10 al cS), 8 al^3 cS
//   [9..11] F  [12..14] T  [15..20] S (xx,xy,xz,yy,yz,zz)
//   [21] cF = a^2/6  [22] cS = a^2/10  [23] pressure moment s (a9; 0 without)
//   [24..24+P) gx * (al/pi)^{3/2}   [24+P..24+2P) gy   [24+2P..24+3P) gz     per-axis Gaussians
#define REC_D0 2
#define REC_POLY 5
#define REC_F 9
#define REC_T 12
#define REC_S 15
#define REC_CF 21
#define REC_CS 22
#define REC_SP 23
__host__ __device__ inline int se_rec_stride(int P) { return (SE_REC_HDR + 3 * P + 1) & ~1; }

// Gather record (grec_stride doubles, 16-byte aligned), in gather order (tile major, starting plane minor):
//   [0] int2 (y0w, z0w)  [1] int2 (x0w, orig)  [2] d0y  [3] d0z
//   [4 .. 4+PP) gy, [4+PP .. 4+2PP) gz, zero beyond P (PP = P rounded up to a multiple of 8)
//   [4+2PP .. 4+2PP+2P)  (gx, gx dx)(k) interleaved, gx with the factor (al/pi)^{3/2}
__host__ __device__ inline int se_grec_pp(int P) { return (P + 7) & ~7; }
__host__ __device__ inline int se_grec_stride(int P) { return 4 + 2 * se_grec_pp(P) + 2 * P; }

__host__ __device__ inline int se_support_start(double u, int P)
{
    // exactly P points per axis; even P: centred between grid points, odd P: centred on the nearest
    return (P & 1) ? (int)floor(u + 0.5) - (P - 1) / 2 : (int)floor(u) - P / 2 + 1;
}

__device__ __forceinline__ int se_mod(int a, int m)
{
    int r = a % m;
    return r < 0 ? r + m : r;
}
