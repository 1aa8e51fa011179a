"""ctypes binding of include/se_mobility.h -- same names, argument marshalling only."""
from __future__ import annotations

import ctypes
import os
import re

import numpy as np

from . import build as _build

SE_SKIP_REAL, SE_SKIP_WAVE, SE_SKIP_SELF, SE_SKIP_ONEBODY, SE_TIMING, SE_CUFFT3D = 0x1, 0x2, 0x4, 0x8, 0x10, 0x40
SE_OPT_REAL_OVERLAP, SE_OPT_REAL_CTAS, SE_OPT_XY_PATH, SE_OPT_YZ_FUSED, SE_OPT_GRAPH, SE_OPT_PAIR_CACHE = 0, 1, 2, 3, 4, 5
SE_OPT_SIZE_VARIANT, SE_OPT_GRID_FP32 = 6, 7
SE_VARIANT_HYBRID, SE_VARIANT_REAL, SE_VARIANT_WAVE = 0, 1, 2
SE_NUM_STAGES = 8
STAGE_NAMES = ("sort", "real", "spread", "fft_fwd", "kspace", "fft_inv", "gather", "epilogue")
_STATUS = {0: "SE_OK", 1: "SE_ERR_INVALID_ARG", 2: "SE_ERR_UNSUPPORTED", 3: "SE_ERR_ALLOC", 4: "SE_ERR_CUDA",
           5: "SE_ERR_CUFFT"}

_HEADER = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "se_mobility.h")


class SeError(RuntimeError):
    def __init__(self, status: int, where: str, detail: str = ""):
        self.status = status
        super().__init__(f"{where}: {_STATUS.get(status, status)} {detail}".strip())


def declared_symbols() -> list[str]:
    """Names of the functions include/se_mobility.h declares."""
    text = open(_HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b((?:se_|far_mobility_)\w+)\s*\(", text)))


_lib = None


def load_library(build_if_missing: bool = True):
    """dlopen libse_mobility.so (building it with nvcc if sources are newer); fails loudly."""
    global _lib
    if _lib is not None:
        return _lib
    if build_if_missing and _build.needs_build():
        _build.build()
    if not os.path.exists(_build.LIB_PATH):
        raise ImportError(f"{_build.LIB_PATH} is missing: run `python -m paper_1506_08481_b200.build`")
    L = ctypes.CDLL(_build.LIB_PATH)
    D, I64, INT, U, P, SZ = ctypes.c_double, ctypes.c_int64, ctypes.c_int, ctypes.c_uint, ctypes.c_void_p, ctypes.c_size_t
    L.se_plan_create.restype = INT
    L.se_plan_create.argtypes = [ctypes.POINTER(P), I64, D, P, D, D, INT, INT, D]
    L.se_plan_set_shape.restype = INT
    L.se_plan_set_shape.argtypes = [P, D]
    L.se_plan_set_strain.restype = INT
    L.se_plan_set_strain.argtypes = [P, D]
    L.se_plan_set_tuning.restype = INT
    L.se_plan_set_tuning.argtypes = [P, INT, INT]
    L.se_plan_set_option.restype = INT
    L.se_plan_set_option.argtypes = [P, INT, INT]
    L.se_plan_set_positions.restype = INT
    L.se_plan_set_positions.argtypes = [P, P, P]
    L.se_plan_set_flags.restype = INT
    L.se_plan_set_flags.argtypes = [P, U]
    L.far_mobility_apply.restype = INT
    L.far_mobility_apply.argtypes = [P] * 9
    L.far_mobility_apply_batch.restype = INT
    L.far_mobility_apply_batch.argtypes = [P, P, INT, P, P, P, P, P, P, P]
    L.far_mobility_apply_compressible.restype = INT
    L.far_mobility_apply_compressible.argtypes = [P] * 11
    L.se_self_image_blocks.restype = INT
    L.se_self_image_blocks.argtypes = [P, P, P]
    L.far_mobility_apply_host.restype = INT
    L.far_mobility_apply_host.argtypes = [P] * 9
    L.far_mobility_apply_host_async.restype = INT
    L.far_mobility_apply_host_async.argtypes = [P] * 9
    L.se_plan_copy_grids.restype = INT
    L.se_plan_copy_grids.argtypes = [P, INT, P]
    L.se_plan_debug_stop.restype = INT
    L.se_plan_debug_stop.argtypes = [P, INT]
    L.se_plan_get_timings.restype = INT
    L.se_plan_get_timings.argtypes = [P, P]
    L.se_plan_last_launch_count.restype = INT
    L.se_plan_last_launch_count.argtypes = [P]
    L.se_plan_workspace_bytes.restype = SZ
    L.se_plan_workspace_bytes.argtypes = [P]
    L.se_plan_get_constants.restype = INT
    L.se_plan_get_constants.argtypes = [P, P]
    L.se_last_error.restype = ctypes.c_char_p
    L.se_last_error.argtypes = [P]
    L.se_plan_destroy.restype = INT
    L.se_plan_destroy.argtypes = [P]
    L.se_measure_fp64_peak.restype = INT
    L.se_measure_fp64_peak.argtypes = [P, P]
    L.se_version.restype = ctypes.c_char_p
    L.se_version.argtypes = []
    L.far_mobility_real_noalloc.restype = INT
    L.far_mobility_real_noalloc.argtypes = [I64, D, D, D, D] + [P] * 9 + [ctypes.c_char_p, SZ]
    _lib = L
    return L


SE_NOALLOC_MAX_N = 8192


def real_noalloc(L, xi, rc, pos, radii, F, T, S, U, Omega, E, eta0=1.0, stream=None):
    """far_mobility_real_noalloc: the real-space pair sum on CUDA float64 tensors, no plan and no allocation (the scratch is a
    static device array inside the library, N <= SE_NOALLOC_MAX_N; calls that overlap on the GPU race)."""
    import torch
    N = int(radii.numel())
    sp = (torch.cuda.current_stream() if stream is None else stream).cuda_stream
    buf = ctypes.create_string_buffer(256)
    st = load_library().far_mobility_real_noalloc(N, float(L), float(xi), float(rc), float(eta0), _dptr(pos, 3 * N, "pos"),
                                                  _dptr(radii, N, "radii"), _dptr(F, 3 * N, "F"), _dptr(T, 3 * N, "T"),
                                                  _dptr(S, 5 * N, "S"), _dptr(U, 3 * N, "U"), _dptr(Omega, 3 * N, "Omega"),
                                                  _dptr(E, 5 * N, "E"), sp, buf, 256)
    if st != 0:
        raise SeError(st, "far_mobility_real_noalloc", buf.value.decode())


def version() -> str:
    return load_library().se_version().decode()


def measure_fp64_peak(stream=None) -> float:
    """se_measure_fp64_peak: sustained independent-DFMA rate of the current device in TFLOP/s."""
    import torch
    sp = (torch.cuda.current_stream() if stream is None else stream).cuda_stream
    out = ctypes.c_double(0.0)
    st = load_library().se_measure_fp64_peak(ctypes.byref(out), sp)
    if st != 0:
        raise SeError(st, "se_measure_fp64_peak")
    return float(out.value)


def _dptr(t, n, name):
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous() or t.numel() != n:
        raise ValueError(f"{name}: expected a contiguous CUDA float64 tensor with {n} elements")
    return t.data_ptr()


def _hptr(a, n, name):
    if not isinstance(a, np.ndarray) or a.dtype != np.float64 or not a.flags.c_contiguous or a.size != n:
        raise ValueError(f"{name}: expected a C-contiguous float64 numpy array with {n} elements")
    return a.ctypes.data


class SePlan:
    """se_plan_create / far_mobility_apply / se_plan_destroy with the header's argument meaning."""

    def __init__(self, N, L, radii, xi, r_c, M, P, eta0=1.0):
        self._lib = load_library()
        self._h = ctypes.c_void_p()
        rad = np.ascontiguousarray(radii, dtype=np.float64)
        if rad.size != N:
            raise ValueError("radii must have N entries")
        st = self._lib.se_plan_create(ctypes.byref(self._h), int(N), float(L), rad.ctypes.data, float(xi), float(r_c),
                                      int(M), int(P), float(eta0))
        if st != 0:
            self._h = ctypes.c_void_p()
            raise SeError(st, "se_plan_create")
        self.N, self.L, self.M, self.P = int(N), float(L), int(M), int(P)

    # -- helpers --
    def _check(self, st, where):
        if st != 0:
            raise SeError(st, where, self._lib.se_last_error(self._h).decode())

    def set_shape(self, m):
        self._check(self._lib.se_plan_set_shape(self._h, float(m)), "se_plan_set_shape")

    def set_strain(self, gamma):
        """se_plan_set_strain: Lees-Edwards strain of the lattice, a2 = (gamma L, L, 0)."""
        self._check(self._lib.se_plan_set_strain(self._h, float(gamma)), "se_plan_set_strain")

    def set_tuning(self, spread_segments=0, gather_segments=0):
        self._check(self._lib.se_plan_set_tuning(self._h, int(spread_segments), int(gather_segments)), "se_plan_set_tuning")

    def set_option(self, key, value):
        self._check(self._lib.se_plan_set_option(self._h, int(key), int(value)), "se_plan_set_option")

    def set_flags(self, flags):
        self._check(self._lib.se_plan_set_flags(self._h, int(flags)), "se_plan_set_flags")

    def set_positions(self, pos, stream=None):
        """se_plan_set_positions: run a1 once for ``pos`` (CUDA float64 [N,3]); later applies may pass pos=None."""
        import torch
        sp = (torch.cuda.current_stream() if stream is None else stream).cuda_stream
        ptr = None if pos is None else _dptr(pos, 3 * self.N, "pos")
        self._check(self._lib.se_plan_set_positions(self._h, ptr, sp), "se_plan_set_positions")

    def debug_stop(self, stage):
        self._check(self._lib.se_plan_debug_stop(self._h, int(stage)), "se_plan_debug_stop")

    def apply(self, pos, F, T, S, U, Omega, E, stream=None):
        """far_mobility_apply on CUDA float64 tensors; enqueues on ``stream`` (default: torch's current)."""
        import torch
        N = self.N
        sp = (torch.cuda.current_stream() if stream is None else stream).cuda_stream
        st = self._lib.far_mobility_apply(self._h, None if pos is None else _dptr(pos, 3 * N, "pos"), _dptr(F, 3 * N, "F"), _dptr(T, 3 * N, "T"),
                                          _dptr(S, 5 * N, "S"), _dptr(U, 3 * N, "U"), _dptr(Omega, 3 * N, "Omega"),
                                          _dptr(E, 5 * N, "E"), sp)
        self._check(st, "far_mobility_apply")

    def apply_batch(self, pos, F, T, S, U, Omega, E, stream=None):
        """far_mobility_apply_batch: F, T, U, Omega are CUDA float64 [nrhs, N, 3], S and E [nrhs, N, 5]; pos [N, 3] or None."""
        import torch
        N, nrhs = self.N, int(F.shape[0])
        sp = (torch.cuda.current_stream() if stream is None else stream).cuda_stream
        st = self._lib.far_mobility_apply_batch(
            self._h, None if pos is None else _dptr(pos, 3 * N, "pos"), nrhs, _dptr(F, 3 * N * nrhs, "F"), _dptr(T, 3 * N * nrhs, "T"),
            _dptr(S, 5 * N * nrhs, "S"), _dptr(U, 3 * N * nrhs, "U"), _dptr(Omega, 3 * N * nrhs, "Omega"), _dptr(E, 5 * N * nrhs, "E"), sp)
        self._check(st, "far_mobility_apply_batch")

    def apply_compressible(self, pos, F, T, S, s_in, U, Omega, E, s_out, stream=None):
        """far_mobility_apply_compressible; ``s_in`` / ``s_out`` are CUDA float64 tensors of N entries or None."""
        import torch
        N = self.N
        sp = (torch.cuda.current_stream() if stream is None else stream).cuda_stream
        st = self._lib.far_mobility_apply_compressible(
            self._h, None if pos is None else _dptr(pos, 3 * N, "pos"), _dptr(F, 3 * N, "F"), _dptr(T, 3 * N, "T"), _dptr(S, 5 * N, "S"),
            None if s_in is None else _dptr(s_in, N, "s_in"), _dptr(U, 3 * N, "U"), _dptr(Omega, 3 * N, "Omega"),
            _dptr(E, 5 * N, "E"), None if s_out is None else _dptr(s_out, N, "s_out"), sp)
        self._check(st, "far_mobility_apply_compressible")

    def self_image_blocks(self, out, stream=None):
        """se_self_image_blocks: ``out`` is a CUDA float64 tensor [N, 11, 11], overwritten."""
        import torch
        sp = (torch.cuda.current_stream() if stream is None else stream).cuda_stream
        self._check(self._lib.se_self_image_blocks(self._h, _dptr(out, 121 * self.N, "out"), sp), "se_self_image_blocks")

    def apply_raw(self, pos, F, T, S, U, Omega, E, stream_ptr=0):
        """far_mobility_apply on raw device addresses (ints); used to test NULL handling."""
        return self._lib.far_mobility_apply(self._h, pos, F, T, S, U, Omega, E, stream_ptr)

    def apply_host(self, pos, F, T, S, U, Omega, E, stream=None):
        """far_mobility_apply_host on numpy float64 arrays (copies in, computes, copies out, synchronises)."""
        import torch
        N = self.N
        sp = (torch.cuda.current_stream() if stream is None else stream).cuda_stream
        st = self._lib.far_mobility_apply_host(self._h, _hptr(pos, 3 * N, "pos"), _hptr(F, 3 * N, "F"), _hptr(T, 3 * N, "T"),
                                               _hptr(S, 5 * N, "S"), _hptr(U, 3 * N, "U"), _hptr(Omega, 3 * N, "Omega"),
                                               _hptr(E, 5 * N, "E"), sp)
        self._check(st, "far_mobility_apply_host")

    def apply_host_async(self, pos, F, T, S, U, Omega, E, stream=None):
        """far_mobility_apply_host_async on (pinned) numpy float64 arrays: enqueues copies and product, does not synchronise."""
        import torch
        N = self.N
        sp = (torch.cuda.current_stream() if stream is None else stream).cuda_stream
        st = self._lib.far_mobility_apply_host_async(self._h, _hptr(pos, 3 * N, "pos"), _hptr(F, 3 * N, "F"), _hptr(T, 3 * N, "T"),
                                                     _hptr(S, 5 * N, "S"), _hptr(U, 3 * N, "U"), _hptr(Omega, 3 * N, "Omega"),
                                                     _hptr(E, 5 * N, "E"), sp)
        self._check(st, "far_mobility_apply_host_async")

    def copy_grids(self, which):
        out = np.empty(({0: 3, 1: 6, 2: 1}[which], self.M, self.M, self.M))
        self._check(self._lib.se_plan_copy_grids(self._h, int(which), out.ctypes.data), "se_plan_copy_grids")
        return out

    def timings(self):
        ms = np.zeros(SE_NUM_STAGES)
        self._check(self._lib.se_plan_get_timings(self._h, ms.ctypes.data), "se_plan_get_timings")
        return dict(zip(STAGE_NAMES, ms.tolist()))

    def last_launch_count(self):
        return int(self._lib.se_plan_last_launch_count(self._h))

    def workspace_bytes(self):
        return int(self._lib.se_plan_workspace_bytes(self._h))

    def constants(self):
        out = np.zeros(7)
        self._check(self._lib.se_plan_get_constants(self._h, out.ctypes.data), "se_plan_get_constants")
        return dict(Delta=out[0], eta_se=out[1], alpha=out[2], m=out[3], real_cells=int(out[4]), spread_segments=int(out[5]),
                    gather_segments=int(out[6]))

    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h:
            self._lib.se_plan_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
