"""ORACLE -- TEST INFRASTRUCTURE ONLY (ctypes wrapper around ``se_oracle.c``).

Plain fp64 CPU implementation of the SEASD far-field mobility product written from PAPER.md
(Wang & Brady, arXiv 1506.08481).  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package.  It shares no code with, and never
imports, ``paper_1506_08481_b200`` (the CUDA path).

* :func:`o1_apply`  -- O1, the definition: direct Ewald sum (tiny N).  Eq. 13-17, 19-23, 24-37.
* :func:`o2_apply`  -- O2, the algorithm step by step: cell-list real-space sum (Sec. 3.3) + Spectral
  Ewald hybrid wave-space sum (Sec. 3.1-3.2) + self and one-body terms.  The CUDA path is held to this.
* :func:`o2_real_targets` -- O2's real-space sum for selected particles by brute force over all j.

Parity pins (tests/test_oracle_pins.py): Eq. 37 printed coefficients; the radial chain of Eq. 22 against
symbolic differentiation; Hasimoto's periodic-array constant (N=1); independence of the splitting
parameter xi; symmetry and positive definiteness of the assembled grand mobility; free-space
Rotne-Prager / rotlet / stresslet / source limits (Eq. 18, 26, 29); self terms against quadrature;
O2 -> O1 spectral convergence in P (Eq. 79).  No function here is "parity unpinned".
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libse_oracle.so")

PART_REAL, PART_WAVE, PART_SELF, PART_ONEBODY = 1, 2, 4, 8
PART_ALL = 15


def build(force: bool = False) -> str:
    """Compile se_oracle.c (gcc -O2 -fopenmp) into libse_oracle.so; returns its path."""
    src = os.path.join(_HERE, "se_oracle.c")
    if force or not os.path.exists(_LIB_PATH) or os.path.getmtime(_LIB_PATH) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-std=c11", "-shared", "-fPIC", "-o", _LIB_PATH, src, "-lm"])
    return _LIB_PATH


_lib = None
_D, _I64, _INT, _U, _P = ctypes.c_double, ctypes.c_int64, ctypes.c_int, ctypes.c_uint, ctypes.c_void_p


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        L.o1_apply.restype = _INT
        L.o1_apply.argtypes = [_I64, _D, _P, _P, _D, _D, _INT, _INT, _U, _P, _P, _P, _P, _P, _P, _P, _P]
        L.o2_apply.restype = _INT
        L.o2_apply.argtypes = [_I64, _D, _P, _P, _D, _D, _INT, _INT, _D, _D, _U, _P, _P, _P, _P, _P, _P, _P, _P, _P, _P]
        L.o1_apply_sheared.restype = _INT
        L.o1_apply_sheared.argtypes = [_I64, _D, _D, _P, _P, _D, _D, _INT, _INT, _U, _P, _P, _P, _P, _P, _P, _P, _P]
        L.o2_apply_sheared.restype = _INT
        L.o2_apply_sheared.argtypes = [_I64, _D, _D, _P, _P, _D, _D, _INT, _INT, _D, _D, _U, _P, _P, _P, _P, _P, _P, _P, _P, _P, _P]
        L.o2_apply_variant.restype = _INT
        L.o2_apply_variant.argtypes = [_INT, _I64, _D, _P, _P, _D, _D, _INT, _INT, _D, _D, _U, _P, _P, _P, _P, _P, _P, _P, _P]
        L.o2_apply_variant_sheared.restype = _INT
        L.o2_apply_variant_sheared.argtypes = [_INT, _I64, _D, _D, _P, _P, _D, _D, _INT, _INT, _D, _D, _U, _P, _P, _P, _P, _P, _P, _P, _P]
        L.o2_real_targets.restype = _INT
        L.o2_real_targets.argtypes = [_I64, _D, _P, _P, _D, _D, _D, _P, _P, _P, _P, _I64, _P, _P, _P, _P, _P]
        L.oracle_radial.restype = _D
        L.oracle_radial.argtypes = [_INT, _INT, _D, _D]
        L.oracle_self_coeffs.restype = None
        L.oracle_self_coeffs.argtypes = [_D, _D, _D, _P]
        L.oracle_se_constants.restype = None
        L.oracle_se_constants.argtypes = [_D, _D, _INT, _INT, _D, _P]
        _lib = L
    return _lib


def num_threads() -> int:
    """Threads the OpenMP loops of the oracle will use (OMP_NUM_THREADS or all cores)."""
    v = os.environ.get("OMP_NUM_THREADS")
    return int(v) if v else (os.cpu_count() or 1)


def _c(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None:
        assert a.shape == shape, (a.shape, shape)
    return a


def _ptr(a):
    return None if a is None else a.ctypes.data


def o1_apply(pos, radii, L, xi, F, T, S, s=None, eta0=1.0, nimg=3, kmax=12, parts=PART_ALL):
    """Direct Ewald sum.  Returns (U[N,3], Omega[N,3], E[N,5], s_out[N])."""
    N = len(radii)
    pos, radii, F, T, S = _c(pos, (N, 3)), _c(radii, (N,)), _c(F, (N, 3)), _c(T, (N, 3)), _c(S, (N, 5))
    s_in = None if s is None else _c(s, (N,))
    U, W, E, so = np.zeros((N, 3)), np.zeros((N, 3)), np.zeros((N, 5)), np.zeros(N)
    rc = lib().o1_apply(N, L, _ptr(pos), _ptr(radii), xi, eta0, nimg, kmax, parts,
                        _ptr(F), _ptr(T), _ptr(S), _ptr(s_in), _ptr(U), _ptr(W), _ptr(E), _ptr(so))
    if rc:
        raise RuntimeError(f"o1_apply status {rc}")
    return U, W, E, so


def o1_matrix(pos, radii, L, xi, eta0=1.0, nimg=3, kmax=12, parts=PART_ALL):
    """Assembled grand mobility in the stored basis, [12N,12N]: rows (U3, Omega3, E5, s) per particle,
    columns (F3, T3, S5, s) per particle, by applying O1 to unit vectors."""
    N = len(radii)
    A = np.zeros((12 * N, 12 * N))
    for j in range(N):
        for c in range(12):
            F, T, S, s = np.zeros((N, 3)), np.zeros((N, 3)), np.zeros((N, 5)), np.zeros(N)
            if c < 3:
                F[j, c] = 1.0
            elif c < 6:
                T[j, c - 3] = 1.0
            elif c < 11:
                S[j, c - 6] = 1.0
            else:
                s[j] = 1.0
            U, W, E, so = o1_apply(pos, radii, L, xi, F, T, S, s, eta0, nimg, kmax, parts)
            A[:, 12 * j + c] = np.concatenate([U, W, E, so[:, None]], axis=1).reshape(-1)
    return A


def o2_apply(pos, radii, L, xi, rc, M, P, F, T, S, s=None, m=None, eta0=1.0, parts=PART_ALL,
             want_grids=False):
    """Step-by-step Spectral Ewald product.  Returns dict(U, Omega, E, s_out[, gridH, gridOut])."""
    N = len(radii)
    pos, radii, F, T, S = _c(pos, (N, 3)), _c(radii, (N,)), _c(F, (N, 3)), _c(T, (N, 3)), _c(S, (N, 5))
    s_in = None if s is None else _c(s, (N,))
    if m is None:
        m = float(np.sqrt(np.pi * P))
    U, W, E = np.zeros((N, 3)), np.zeros((N, 3)), np.zeros((N, 5))
    so = None if s is None else np.zeros(N)
    gH = gO = None
    if want_grids:
        gH = np.zeros((4 if s is not None else 3, M, M, M))
        gO = np.zeros((7 if s is not None else 6, M, M, M))
    rcode = lib().o2_apply(N, L, _ptr(pos), _ptr(radii), xi, rc, M, P, m, eta0, parts,
                           _ptr(F), _ptr(T), _ptr(S), _ptr(s_in), _ptr(U), _ptr(W), _ptr(E), _ptr(so),
                           _ptr(gH), _ptr(gO))
    if rcode:
        raise RuntimeError(f"o2_apply status {rcode}")
    out = dict(U=U, Omega=W, E=E, s_out=so)
    if want_grids:
        out["gridH"], out["gridOut"] = gH, gO
    return out


def o1_apply_sheared(pos, radii, L, gamma, xi, F, T, S, s=None, eta0=1.0, nimg=3, kmax=12, parts=PART_ALL):
    """Direct Ewald sum on the sheared lattice a1 = (L,0,0), a2 = (gamma L, L, 0), a3 = (0,0,L).  Returns (U, Omega, E, s_out)."""
    N = len(radii)
    pos, radii, F, T, S = _c(pos, (N, 3)), _c(radii, (N,)), _c(F, (N, 3)), _c(T, (N, 3)), _c(S, (N, 5))
    s_in = None if s is None else _c(s, (N,))
    U, W, E, so = np.zeros((N, 3)), np.zeros((N, 3)), np.zeros((N, 5)), np.zeros(N)
    rc = lib().o1_apply_sheared(N, L, gamma, _ptr(pos), _ptr(radii), xi, eta0, nimg, kmax, parts,
                                _ptr(F), _ptr(T), _ptr(S), _ptr(s_in), _ptr(U), _ptr(W), _ptr(E), _ptr(so))
    if rc:
        raise RuntimeError(f"o1_apply_sheared status {rc}")
    return U, W, E, so


def o1_matrix_sheared(pos, radii, L, gamma, xi, eta0=1.0, nimg=3, kmax=12, parts=PART_ALL):
    """Assembled [11N, 11N] grand mobility (stored basis, no pressure row/column) on the sheared lattice."""
    N = len(radii)
    A = np.zeros((11 * N, 11 * N))
    for j in range(N):
        for c in range(11):
            F, T, S = np.zeros((N, 3)), np.zeros((N, 3)), np.zeros((N, 5))
            if c < 3:
                F[j, c] = 1.0
            elif c < 6:
                T[j, c - 3] = 1.0
            else:
                S[j, c - 6] = 1.0
            U, W, E, _ = o1_apply_sheared(pos, radii, L, gamma, xi, F, T, S, None, eta0, nimg, kmax, parts)
            A[:, 11 * j + c] = np.concatenate([U, W, E], axis=1).reshape(-1)
    return A


def o2_apply_sheared(pos, radii, L, gamma, xi, rc, M, P, F, T, S, s=None, m=None, eta0=1.0, parts=PART_ALL, want_grids=False):
    """Step-by-step Spectral Ewald product on the sheared lattice.  Returns dict(U, Omega, E, s_out[, gridH, gridOut])."""
    N = len(radii)
    pos, radii, F, T, S = _c(pos, (N, 3)), _c(radii, (N,)), _c(F, (N, 3)), _c(T, (N, 3)), _c(S, (N, 5))
    s_in = None if s is None else _c(s, (N,))
    if m is None:
        m = float(np.sqrt(np.pi * P))
    U, W, E = np.zeros((N, 3)), np.zeros((N, 3)), np.zeros((N, 5))
    so = None if s is None else np.zeros(N)
    gH = gO = None
    if want_grids:
        gH = np.zeros((4 if s is not None else 3, M, M, M))
        gO = np.zeros((7 if s is not None else 6, M, M, M))
    rcode = lib().o2_apply_sheared(N, L, gamma, _ptr(pos), _ptr(radii), xi, rc, M, P, m, eta0, parts,
                                   _ptr(F), _ptr(T), _ptr(S), _ptr(s_in), _ptr(U), _ptr(W), _ptr(E), _ptr(so), _ptr(gH), _ptr(gO))
    if rcode:
        raise RuntimeError(f"o2_apply_sheared status {rcode}")
    out = dict(U=U, Omega=W, E=E, s_out=so)
    if want_grids:
        out["gridH"], out["gridOut"] = gH, gO
    return out


VARIANT_HYBRID, VARIANT_REAL, VARIANT_WAVE = 0, 1, 2


def o2_apply_variant(variant, pos, radii, L, xi, rc, M, P, F, T, S, s=None, m=None, eta0=1.0, parts=PART_ALL):
    """Spectral Ewald product with the particle size brought in the real-space way (variant 1) or the
    wave-space way (variant 2, Eq. 49-52); variant 0 is o2_apply (hybrid).  Returns dict(U, Omega, E, s_out)."""
    if variant == VARIANT_HYBRID:
        return o2_apply(pos, radii, L, xi, rc, M, P, F, T, S, s, m=m, eta0=eta0, parts=parts)
    N = len(radii)
    pos, radii, F, T, S = _c(pos, (N, 3)), _c(radii, (N,)), _c(F, (N, 3)), _c(T, (N, 3)), _c(S, (N, 5))
    s_in = None if s is None else _c(s, (N,))
    if m is None:
        m = float(np.sqrt(np.pi * P))
    U, W, E = np.zeros((N, 3)), np.zeros((N, 3)), np.zeros((N, 5))
    so = None if s is None else np.zeros(N)
    rcode = lib().o2_apply_variant(variant, N, L, _ptr(pos), _ptr(radii), xi, rc, M, P, m, eta0, parts,
                                   _ptr(F), _ptr(T), _ptr(S), _ptr(s_in), _ptr(U), _ptr(W), _ptr(E), _ptr(so))
    if rcode:
        raise RuntimeError(f"o2_apply_variant status {rcode}")
    return dict(U=U, Omega=W, E=E, s_out=so)


def o2_apply_variant_sheared(variant, pos, radii, L, gamma, xi, rc, M, P, F, T, S, s=None, m=None, eta0=1.0, parts=PART_ALL):
    """The real-space (1) or wave-space (2) size variant on the sheared lattice; variant 0 is o2_apply_sheared."""
    if variant == VARIANT_HYBRID:
        return o2_apply_sheared(pos, radii, L, gamma, xi, rc, M, P, F, T, S, s, m=m, eta0=eta0, parts=parts)
    N = len(radii)
    pos, radii, F, T, S = _c(pos, (N, 3)), _c(radii, (N,)), _c(F, (N, 3)), _c(T, (N, 3)), _c(S, (N, 5))
    s_in = None if s is None else _c(s, (N,))
    if m is None:
        m = float(np.sqrt(np.pi * P))
    U, W, E = np.zeros((N, 3)), np.zeros((N, 3)), np.zeros((N, 5))
    so = None if s is None else np.zeros(N)
    rcode = lib().o2_apply_variant_sheared(variant, N, L, gamma, _ptr(pos), _ptr(radii), xi, rc, M, P, m, eta0, parts,
                                           _ptr(F), _ptr(T), _ptr(S), _ptr(s_in), _ptr(U), _ptr(W), _ptr(E), _ptr(so))
    if rcode:
        raise RuntimeError(f"o2_apply_variant_sheared status {rcode}")
    return dict(U=U, Omega=W, E=E, s_out=so)


def o2_real_targets(pos, radii, L, xi, rc, F, T, S, targets, s=None, eta0=1.0):
    """Real-space part of O2 for the particle indices in ``targets`` (brute force over all j)."""
    N = len(radii)
    pos, radii, F, T, S = _c(pos, (N, 3)), _c(radii, (N,)), _c(F, (N, 3)), _c(T, (N, 3)), _c(S, (N, 5))
    s_in = None if s is None else _c(s, (N,))
    tgt = np.ascontiguousarray(targets, dtype=np.int64)
    n = tgt.size
    U, W, E, so = np.zeros((n, 3)), np.zeros((n, 3)), np.zeros((n, 5)), np.zeros(n)
    rcode = lib().o2_real_targets(N, L, _ptr(pos), _ptr(radii), xi, rc, eta0, _ptr(F), _ptr(T), _ptr(S), _ptr(s_in),
                                  n, _ptr(tgt), _ptr(U), _ptr(W), _ptr(E), _ptr(so))
    if rcode:
        raise RuntimeError(f"o2_real_targets status {rcode}")
    return U, W, E, so


def radial(fam: int, order: int, xi: float, r: float) -> float:
    """((1/r)d/dr)^order of family fam (0 Phi, 1 lap Phi, 2 lap^2 Phi, 3 lap^3 Phi, 4 erfc(xi r)/r,
    5 lap of it) at separation r -- the mechanically generated radial chain of Eq. 22."""
    return float(lib().oracle_radial(fam, order, xi, r))


def self_coeffs(a: float, xi: float, eta0: float = 1.0):
    out = np.zeros(3)
    lib().oracle_self_coeffs(a, xi, eta0, _ptr(out))
    return out


def se_constants(L, xi, M, P, m=None):
    """(Delta, eta_se, alpha, gnorm) of O2 step 1."""
    if m is None:
        m = float(np.sqrt(np.pi * P))
    out = np.zeros(4)
    lib().oracle_se_constants(L, xi, M, P, m, _ptr(out))
    return out
