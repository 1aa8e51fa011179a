"""Seeded synthetic workloads for the SEASD far-field mobility product.

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA path
(``paper_1506_08481_b200/``).  It contains input generators and the parameter recipe of
DESIGN.md §"Input recipe" and none of the method's arithmetic.

The five configurations are the ones listed in BASELINE.json ``configs`` (c1..c5).  They stand in for
the paper's workloads -- random mono/bidisperse hard-sphere suspensions at volume fractions up to 0.45
(PAPER.md L491, L552); the paper's own equilibrated configurations are not available, no public data
set is involved.

RNG: NumPy ``Generator(PCG64)`` seeded from ``SeedSequence([150608481, c])`` and spawned into three
child streams (radii, positions, moments).  Positions come from a compiled seeded RSA generator
(``rsa.c``; its 64-bit seed is drawn from the positions stream) or, for c3 whose volume fraction RSA
cannot reach, from a randomly thinned and jittered FCC lattice.
"""
from __future__ import annotations

import ctypes
import math
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "librsa.so")
_BASE_SEED = 150608481
EPS_TRUNC = 1.0e-8  # truncation level of the balanced (xi, r_c) rule


def build(force: bool = False) -> str:
    """Compile rsa.c into librsa.so (gcc); returns the library path."""
    src = os.path.join(_HERE, "rsa.c")
    if force or not os.path.exists(_LIB_PATH) or os.path.getmtime(_LIB_PATH) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-shared", "-fPIC", "-o", _LIB_PATH, src, "-lm"])
    return _LIB_PATH


_lib = None


def _rsa_lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.rsa_generate.restype = ctypes.c_int
        _lib.rsa_generate.argtypes = [
            ctypes.c_int64, ctypes.c_double, ctypes.c_void_p, ctypes.c_uint64, ctypes.c_int64,
            ctypes.c_void_p, ctypes.c_void_p,
        ]
    return _lib


def rsa_positions(radii: np.ndarray, L: float, seed: int, max_attempts: int = 2_000_000) -> np.ndarray:
    """Random sequential addition in insertion order = descending radius; returns pos in the
    ORIGINAL order of ``radii``."""
    radii = np.ascontiguousarray(radii, dtype=np.float64)
    order = np.argsort(-radii, kind="stable")
    r_sorted = np.ascontiguousarray(radii[order])
    pos_sorted = np.empty((radii.size, 3), dtype=np.float64)
    attempts = ctypes.c_int64(0)
    rc = _rsa_lib().rsa_generate(radii.size, float(L), r_sorted.ctypes.data, ctypes.c_uint64(seed),
                                 max_attempts, pos_sorted.ctypes.data, ctypes.byref(attempts))
    if rc != 0:
        raise RuntimeError(f"RSA failed (status {rc}) at N={radii.size}, L={L}")
    pos = np.empty_like(pos_sorted)
    pos[order] = pos_sorted
    return pos


def fcc_jittered_positions(N: int, L: float, a: float, rng: np.random.Generator) -> np.ndarray:
    """Dense monodisperse stand-in (c3): smallest FCC lattice with >= N sites, keep a seeded random
    subset of N, displace each by a uniform vector in a ball small enough to forbid overlap."""
    n = 1
    while 4 * n ** 3 < N:
        n += 1
    alat = L / n
    nn = alat / math.sqrt(2.0)
    if nn <= 2.0 * a:
        raise ValueError("FCC lattice too dense for non-overlapping spheres")
    base = np.array([[0, 0, 0], [0.5, 0.5, 0], [0.5, 0, 0.5], [0, 0.5, 0.5]], dtype=np.float64)
    g = np.stack(np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij"), axis=-1).reshape(-1, 1, 3)
    sites = ((g + base[None, :, :]) * alat).reshape(-1, 3)
    keep = rng.permutation(sites.shape[0])[:N]
    pos = sites[keep]
    rmax = 0.999 * (nn - 2.0 * a) / 2.0
    v = rng.standard_normal((N, 3))
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    rad = rmax * rng.random(N) ** (1.0 / 3.0)
    pos = pos + v * rad[:, None]
    return np.mod(pos, L)


@dataclass
class Workload:
    """One seeded problem instance: geometry, SE parameters and moments (all float64, host)."""
    name: str
    N: int
    L: float
    radii: np.ndarray
    pos: np.ndarray
    F: np.ndarray
    T: np.ndarray
    S: np.ndarray          # [N,5] = (xx, xy, xz, yy, yz); zz = -(xx+yy)
    xi: float
    rc: float
    M: int
    P: int
    m: float
    eta0: float = 1.0
    phi: float = 0.0
    meta: dict = field(default_factory=dict)


# name: (N, M, P, phi, radii recipe, position recipe, fixed r_c or None)
CONFIGS = {
    "c1": dict(N=100, M=32, P=8, phi=0.10, radii="mono", positions="rsa", rc_fixed=3.0),
    "c2": dict(N=1000, M=64, P=10, phi=0.30, radii="bi_1_2", positions="rsa", rc_fixed=None),
    "c3": dict(N=10_000, M=128, P=12, phi=0.45, radii="mono", positions="fcc", rc_fixed=None),
    "c4": dict(N=100_000, M=256, P=12, phi=0.40, radii="bi_1_4", positions="rsa", rc_fixed=None),
    "c5": dict(N=1_000_000, M=512, P=12, phi=0.30, radii="lognormal", positions="rsa", rc_fixed=None),
}


def make_radii(recipe: str, N: int, rng: np.random.Generator) -> np.ndarray:
    if recipe == "mono":
        return np.ones(N)
    if recipe == "bi_1_2":       # equal species volume fractions: N1*1^3 = N2*2^3
        n_large = int(round(N / 9.0))
        return np.concatenate([np.ones(N - n_large), 2.0 * np.ones(n_large)])
    if recipe == "bi_1_4":       # phi_large = phi_small: N_small = 64 N_large
        n_large = int(N / 65.0)
        return np.concatenate([np.ones(N - n_large), 4.0 * np.ones(n_large)])
    if recipe == "lognormal":    # median 1, sigma_ln 0.25, clipped to [0.5, 2]
        return np.clip(np.exp(0.25 * rng.standard_normal(N)), 0.5, 2.0)
    raise ValueError(recipe)


def box_edge(radii: np.ndarray, phi: float) -> float:
    return float((np.sum(4.0 * math.pi * radii ** 3 / 3.0) / phi) ** (1.0 / 3.0))


def resolve_split(L: float, M: int, rc_fixed: float | None = None, eps: float = EPS_TRUNC):
    """Balanced Ewald parameters: exp(-xi^2 r_c^2) = exp(-k_N^2 / 4 xi^2) = eps with k_N = pi M / L,
    unless r_c is fixed (c1), in which case xi balances the two exponents for that r_c."""
    kN = math.pi * M / L
    if rc_fixed is None:
        s = math.sqrt(math.log(1.0 / eps))
        xi = kN / (2.0 * s)
        rc = s / xi
    else:
        rc = float(rc_fixed)
        xi = math.sqrt(kN / (2.0 * rc))
    return xi, rc


def make_moments(N: int, rng: np.random.Generator, unit_norm: bool = False):
    """F, T i.i.d. N(0,1); S: five stored components i.i.d. N(0,1), zz implied (traceless).
    unit_norm=True rescales each particle's F, T, S to unit norm."""
    F = rng.standard_normal((N, 3))
    T = rng.standard_normal((N, 3))
    S = rng.standard_normal((N, 5))
    if unit_norm:
        F /= np.linalg.norm(F, axis=1, keepdims=True)
        T /= np.linalg.norm(T, axis=1, keepdims=True)
        szz = -(S[:, 0] + S[:, 3])
        nrm = np.sqrt(S[:, 0] ** 2 + S[:, 3] ** 2 + szz ** 2 + 2 * (S[:, 1] ** 2 + S[:, 2] ** 2 + S[:, 4] ** 2))
        S /= nrm[:, None]
    return F, T, S


def make_workload(name: str, N: int | None = None, M: int | None = None, P: int | None = None) -> Workload:
    """Build config ``name`` (c1..c5).  N/M/P overrides give reduced versions of the same recipe
    (same composition, volume fraction and parameter rule) for parity tests the oracle finishes fast."""
    spec = dict(CONFIGS[name])
    if N is not None:
        spec["N"] = int(N)
    if M is not None:
        spec["M"] = int(M)
    if P is not None:
        spec["P"] = int(P)
    c = int(name[1:])
    ss = np.random.SeedSequence([_BASE_SEED, c])
    rng_radii, rng_pos, rng_mom = (np.random.Generator(np.random.PCG64(s)) for s in ss.spawn(3))

    Np = spec["N"]
    radii = make_radii(spec["radii"], Np, rng_radii)
    L = box_edge(radii, spec["phi"])
    if spec["positions"] == "rsa":
        seed = int(rng_pos.integers(0, 2 ** 63 - 1))
        pos = rsa_positions(radii, L, seed)
    else:
        pos = fcc_jittered_positions(Np, L, 1.0, rng_pos)
    # caller order is a seeded shuffle so that particle index carries no size/insert-order structure
    perm = rng_pos.permutation(Np)
    radii = np.ascontiguousarray(radii[perm])
    pos = np.ascontiguousarray(pos[perm])
    F, T, S = make_moments(Np, rng_mom)
    xi, rc = resolve_split(L, spec["M"], spec["rc_fixed"])
    rc = min(rc, 0.5 * L)
    Pp = spec["P"]
    return Workload(name=name, N=Np, L=L, radii=radii, pos=pos, F=F, T=T, S=S, xi=xi, rc=rc,
                    M=spec["M"], P=Pp, m=math.sqrt(math.pi * Pp), eta0=1.0, phi=spec["phi"],
                    meta=dict(radii=spec["radii"], positions=spec["positions"]))


def make_accuracy_system(seed: int = 78, N: int = 50, phi: float = 0.05, lam: float = 2.0, x2: float = 0.3):
    """The paper's accuracy test system: random bidisperse hard spheres, N=50,
    phi=0.05, size ratio 2, number fraction of large spheres 0.3, unit-norm F, T, S."""
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([_BASE_SEED, 1000 + seed])))
    n2 = int(round(x2 * N))
    radii = np.concatenate([np.ones(N - n2), lam * np.ones(n2)])
    L = box_edge(radii, phi)
    pos = rsa_positions(radii, L, int(rng.integers(0, 2 ** 63 - 1)))
    perm = rng.permutation(N)
    radii, pos = np.ascontiguousarray(radii[perm]), np.ascontiguousarray(pos[perm])
    F, T, S = make_moments(N, rng, unit_norm=True)
    return dict(N=N, L=L, radii=radii, pos=pos, F=F, T=T, S=S)


def random_small_system(seed: int, N: int, L: float, amin: float = 0.6, amax: float = 1.5):
    """Tiny polydisperse non-overlapping system for the direct-Ewald pins."""
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([_BASE_SEED, 2000 + seed])))
    radii = amin + (amax - amin) * rng.random(N)
    pos = rsa_positions(radii, L, int(rng.integers(0, 2 ** 63 - 1)))
    F, T, S = make_moments(N, rng)
    s = rng.standard_normal(N)
    return dict(N=N, L=L, radii=radii, pos=pos, F=F, T=T, S=S, s=s)


def shard_range(n_units: int, rank: int, world: int) -> range:
    """Contiguous block partition of ``n_units`` independent products over ``world`` ranks
    (replicas-only multi-GPU).  Sizes differ by at most one."""
    base, rem = divmod(n_units, world)
    lo = rank * base + min(rank, rem)
    return range(lo, lo + base + (1 if rank < rem else 0))


def make_uniform_system(seed: int, N: int, phi: float, M: int, P: int, rc_over_L: float) -> Workload:
    """Monodisperse (a = 1) RSA suspension with the real-space cutoff given as a fraction of the box edge --
    parity cases that reach the dense branches of the real-space kernel (many candidates per cell; all pairs)."""
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([_BASE_SEED, 3000 + seed])))
    radii = np.ones(N)
    L = box_edge(radii, phi)
    pos = rsa_positions(radii, L, int(rng.integers(0, 2 ** 63 - 1)))
    F, T, S = make_moments(N, rng)
    xi, _ = resolve_split(L, M)
    return Workload(name=f"uniform{seed}", N=N, L=L, radii=radii, pos=pos, F=F, T=T, S=S, xi=xi, rc=rc_over_L * L,
                    M=M, P=P, m=math.sqrt(math.pi * P), eta0=1.0, phi=phi, meta=dict(radii="mono", positions="rsa"))


def make_clustered_system(seed: int, N: int, n_cluster: int, L: float, M: int, P: int, rc: float) -> Workload:
    """Polydisperse point cloud (overlaps allowed: the formulas are regular for r > 0) in which ``n_cluster`` particles
    sit inside ONE grid cell column of 1 x 4 x 8 grid spacings, so that their P^3 supports all start in the same
    plane-thin tile bin -- the degenerate case of the particle<->grid kernels (bin overflow, one dense tile).  The
    cluster members keep a minimum mutual distance of 0.05 so that the pair terms stay well conditioned."""
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([_BASE_SEED, 4000 + seed])))
    radii = 0.6 + 0.9 * rng.random(N)
    pos = L * rng.random((N, 3))
    D = L / M
    # support origin n0 = floor(x / D) - P/2 + 1 (even P): choose the cell column so that n0_y is a multiple of 4 and
    # n0_z a multiple of 8, the bin edges of the spreading sort
    assert P % 2 == 0
    corner = np.array([M // 2 + 1, 4 * (M // 8) + P // 2 - 1, 8 * (M // 16) + P // 2 - 1], dtype=np.float64) * D
    ext = np.array([0.98 * D, 3.98 * D, 7.98 * D])
    pts = []
    while len(pts) < n_cluster:
        c = corner + 0.01 * D + ext * rng.random(3)
        if all(np.linalg.norm(c - q) >= 0.05 for q in pts):
            pts.append(c)
    pos[:n_cluster] = np.array(pts)
    perm = rng.permutation(N)
    radii, pos = np.ascontiguousarray(radii[perm]), np.ascontiguousarray(pos[perm])
    F, T, S = make_moments(N, rng)
    xi, _ = resolve_split(L, M)
    return Workload(name=f"cluster{seed}", N=N, L=L, radii=radii, pos=pos, F=F, T=T, S=S, xi=xi, rc=rc,
                    M=M, P=P, m=math.sqrt(math.pi * P), eta0=1.0, phi=0.0, meta=dict(radii="uniform[0.6,1.5]", positions="clustered"))
