"""ctypes binding of libpsd.so: same names as include/psd.h, argument marshalling only.

Every step of the path (tet generation, census, binning, clip, accumulate, flush) runs in the
CUDA kernels behind the C ABI; torch is used here only to hold device memory and streams.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import _build

F32, F64 = 0, 1
OPT_WEIGHT_MODE, OPT_KERNEL, OPT_COUNTERS, OPT_CHUNK, OPT_CHORD_AXIS, OPT_REFINE_SUBBLOCK, OPT_CLASS_SMALL_CELLS, OPT_PATCH_RESTRICT, OPT_PAIR_RECORDS, OPT_ROWS_FP32, OPT_FACE_SHARING = 0, 1, 2, 3, 4, 5, 6, 7, 8, 9, 10
SUBBLOCK_UNIT = 1 << 20
RULE_LITERAL_TOP_DOWN, RULE_BOTTOM_UP_LEVEL_MEAN = 0, 1

# every symbol include/psd.h declares (tests check the library exports exactly these)
EXPORTS = ("psd_create", "psd_destroy", "psd_build_tets", "psd_deposit_uniform",
           "psd_refine_patches", "psd_deposit_patches", "psd_deposit_uniform_host",
           "psd_deposit_patches_host",
           "psd_get_stats", "psd_get_tile_counts", "psd_get_tile_class_counts", "psd_set_option", "psd_sync", "psd_last_error", "psd_launch_count",
           "psd_version", "psd_deposit_uniform_static")


class PsdError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libpsd error {code}: {msg}")
        self.code = code


class PsdPatch(C.Structure):
    _fields_ = [("level", C.c_int32), ("ox", C.c_int32), ("oy", C.c_int32), ("oz", C.c_int32)]


class PsdStats(C.Structure):
    _fields_ = [
        ("n_tets", C.c_int64), ("n_tiles", C.c_int64), ("n_pairs", C.c_int64),
        ("n_work_items", C.c_int64), ("sum_cells", C.c_int64), ("max_cells", C.c_int64), ("max_extent", C.c_int64),
        ("n_inverted", C.c_int64), ("n_degenerate", C.c_int64), ("n_unwrap_suspect", C.c_int64),
        ("n_nonfinite", C.c_int64),
        ("hist_tet", C.c_uint64 * 64), ("hist_pair", C.c_uint64 * 64),
        ("n_face_jobs", C.c_int64), ("n_face_clips", C.c_int64), ("n_plane_evals", C.c_int64),
        ("n_cells_written", C.c_int64), ("n_restricted_patches", C.c_int64), ("n_general_clips", C.c_int64), ("shared_faces", C.c_int64), ("n_rows_missed", C.c_int64),
        ("tile_counts_dev", C.c_void_p),
        ("ms_census", C.c_float), ("ms_scan", C.c_float), ("ms_scatter", C.c_float),
        ("ms_deposit", C.c_float), ("ms_total", C.c_float),
    ]

    def as_dict(self) -> dict:
        d = {}
        for name, _ in self._fields_:
            v = getattr(self, name)
            d[name] = list(v) if hasattr(v, "__len__") else v
        return d


_lib = None


def lib() -> C.CDLL:
    """Load (building it first if the sources are newer) the in-tree libpsd.so."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if _build.is_stale():
        path = _build.build()
    if not os.path.exists(path):
        raise ImportError("libpsd.so is missing and could not be built; there is no CPU fallback")
    L = C.CDLL(path)
    vp, i, d, i64 = C.c_void_p, C.c_int, C.c_double, C.c_int64
    L.psd_create.argtypes = [C.POINTER(vp), i, vp]
    L.psd_destroy.argtypes = [vp]
    L.psd_destroy.restype = None
    L.psd_build_tets.argtypes = [vp, vp, i, i, i, d, d]
    L.psd_deposit_uniform.argtypes = [vp, i, vp, i]
    L.psd_refine_patches.argtypes = [vp, i, i, i, d, i, C.POINTER(PsdPatch), i64,
                                     C.POINTER(i64), C.POINTER(C.c_uint64)]
    L.psd_deposit_patches.argtypes = [vp, C.POINTER(PsdPatch), i64, i, i, vp, i]
    L.psd_deposit_uniform_host.argtypes = [vp, vp, i, i, i, d, d, i, vp]
    L.psd_deposit_patches_host.argtypes = [vp, vp, i, i, i, d, d, i, i, i, d, i, C.POINTER(PsdPatch), i64,
                                           C.POINTER(i64), vp]
    L.psd_get_stats.argtypes = [vp, C.POINTER(PsdStats)]
    L.psd_get_tile_counts.argtypes = [vp, C.POINTER(C.c_uint32), i64]
    L.psd_get_tile_class_counts.argtypes = [vp, C.POINTER(C.c_uint32), i64]
    L.psd_set_option.argtypes = [vp, i, d]
    L.psd_sync.argtypes = [vp]
    L.psd_last_error.argtypes = [vp]
    L.psd_last_error.restype = C.c_char_p
    L.psd_launch_count.argtypes = [vp]
    L.psd_launch_count.restype = i64
    L.psd_version.argtypes = []
    L.psd_version.restype = C.c_char_p
    L.psd_deposit_uniform_static.argtypes = [i, vp, vp, i, i, i, d, d, i, vp, C.POINTER(i64), C.c_char_p, i]
    _lib = L
    return L


def version() -> str:
    return lib().psd_version().decode()


def _pos_meta(pos):
    """(dtype code, stride, N) of a torch tensor or numpy array shaped (..., 3|4) with N^3 rows."""
    name = str(pos.dtype)
    if name.endswith("float32"):
        dt = F32
    elif name.endswith("float64"):
        dt = F64
    else:
        raise TypeError("positions must be float32 or float64")
    stride = int(pos.shape[-1])
    n3 = int(np.prod(pos.shape[:-1]))
    N = round(n3 ** (1.0 / 3.0))
    if N * N * N != n3 or stride not in (3, 4):
        raise ValueError("positions must hold N^3 particles of 3 or 4 components")
    return dt, stride, N


STATIC_MAX_N, STATIC_MAX_G, STATIC_MAX_PAIRS = 64, 128, 4 << 20


def psd_deposit_uniform_static(pos_dev, G: int, grid_dev, L: float = 1.0, total_mass: float = 1.0,
                               device: int = 0, stream=None) -> int:
    """include/psd.h psd_deposit_uniform_static: the deposit that allocates nothing (no context, all
    scratch in the library's static device array).  `grid_dev` is the caller's; returns n_pairs."""
    import torch
    if not pos_dev.is_cuda or not pos_dev.is_contiguous():
        raise ValueError("pos_dev must be a contiguous CUDA tensor")
    if (not grid_dev.is_cuda or grid_dev.dtype != torch.float64 or grid_dev.numel() != G ** 3
            or not grid_dev.is_contiguous()):
        raise ValueError("grid_dev must be a contiguous CUDA float64 tensor of G^3 elements")
    dt, stride, N = _pos_meta(pos_dev)
    st = stream if stream is not None else torch.cuda.current_stream(device)
    err = C.create_string_buffer(256)
    n_pairs = C.c_int64(0)
    rc = lib().psd_deposit_uniform_static(int(device), C.c_void_p(st.cuda_stream), pos_dev.data_ptr(), dt, stride, N,
                                          L, total_mass, G, grid_dev.data_ptr(), C.byref(n_pairs), err, 256)
    if rc:
        raise PsdError(rc, err.value.decode())
    return n_pairs.value


class Context:
    """One psd_ctx.  Methods carry the names of the C entry points they call."""

    def __init__(self, device: int = 0, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("libpsd needs a CUDA device (no CPU fallback)")
        self._torch = torch
        self._L = lib()
        self._h = C.c_void_p()
        self.device = int(device)
        torch.cuda.init()
        with torch.cuda.device(self.device):
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            rc = self._L.psd_create(C.byref(self._h), self.device, C.c_void_p(self.stream.cuda_stream))
        if rc:
            raise PsdError(rc, "psd_create failed")
        self._pos = None  # keeps the borrowed positions alive

    def close(self):
        if getattr(self, "_h", None):
            self._L.psd_destroy(self._h)
            self._h = C.c_void_p()
            self._pos = None

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def _ck(self, rc: int):
        if rc:
            raise PsdError(rc, self._L.psd_last_error(self._h).decode())

    # ---- include/psd.h entry points -------------------------------------------------------
    def psd_build_tets(self, pos_dev, L: float = 1.0, total_mass: float = 1.0):
        if not pos_dev.is_cuda or not pos_dev.is_contiguous():
            raise ValueError("pos_dev must be a contiguous CUDA tensor")
        dt, stride, N = _pos_meta(pos_dev)
        self._pos = pos_dev
        self._ck(self._L.psd_build_tets(self._h, pos_dev.data_ptr(), dt, stride, N, L, total_mass))
        return N

    def psd_deposit_uniform(self, G: int, grid_dev=None, accumulate: bool = False):
        t = self._torch
        if grid_dev is None:
            grid_dev = t.empty((G, G, G), dtype=t.float64, device=f"cuda:{self.device}")
        if (not grid_dev.is_cuda or grid_dev.dtype != t.float64 or grid_dev.numel() != G ** 3
                or not grid_dev.is_contiguous()):
            raise ValueError("grid_dev must be a contiguous CUDA float64 tensor of G^3 elements")
        self._ck(self._L.psd_deposit_uniform(self._h, G, grid_dev.data_ptr(), int(accumulate)))
        return grid_dev

    def psd_refine_patches(self, base_G: int, P: int, max_level: int, factor: float,
                           rule: int = RULE_BOTTOM_UP_LEVEL_MEAN, want_counts: bool = False):
        nl = max_level + 1
        sizes = [((base_G << l) // P) ** 3 for l in range(nl)]
        cap = sum(sizes)
        out = (PsdPatch * cap)()
        n = C.c_int64(0)
        counts = np.zeros(sum(sizes), dtype=np.uint64) if want_counts else None
        cp = counts.ctypes.data_as(C.POINTER(C.c_uint64)) if want_counts else None
        self._ck(self._L.psd_refine_patches(self._h, base_G, P, max_level, factor, rule, out, cap,
                                            C.byref(n), cp))
        arr = np.frombuffer(out, dtype=np.int32).reshape(cap, 4)[: n.value].copy()
        if want_counts:
            per_level, o = [], 0
            for l, s in enumerate(sizes):
                npos = (base_G << l) // P
                per_level.append(counts[o:o + s].reshape(npos, npos, npos))
                o += s
            return arr, per_level
        return arr

    def psd_deposit_patches(self, patches, P: int, base_G: int, mass_dev=None,
                            accumulate: bool = False):
        t = self._torch
        pa = np.ascontiguousarray(patches, dtype=np.int32).reshape(-1, 4)
        n = pa.shape[0]
        if mass_dev is None:
            mass_dev = t.empty((n, P, P, P), dtype=t.float64, device=f"cuda:{self.device}")
        if (not mass_dev.is_cuda or mass_dev.dtype != t.float64 or mass_dev.numel() != n * P ** 3
                or not mass_dev.is_contiguous()):
            raise ValueError("mass_dev must be a contiguous CUDA float64 tensor of n*P^3 elements")
        self._ck(self._L.psd_deposit_patches(self._h, pa.ctypes.data_as(C.POINTER(PsdPatch)), n, P,
                                             base_G, mass_dev.data_ptr(), int(accumulate)))
        return mass_dev

    @staticmethod
    def _host_ptr(a, what: str, dtype_name: str | None = None, numel: int | None = None) -> int:
        """Address of a C-contiguous HOST array (torch CPU tensor or numpy array), validated: the
        library writes / reads it with raw copies, so a wrong dtype or size would corrupt memory."""
        is_torch = hasattr(a, "data_ptr")
        if is_torch:
            if a.is_cuda:
                raise ValueError(f"{what} must be a host (CPU) tensor")
            contiguous, n = a.is_contiguous(), a.numel()
        elif isinstance(a, np.ndarray):
            contiguous, n = a.flags.c_contiguous, a.size
        else:
            raise TypeError(f"{what} must be a torch CPU tensor or a numpy array")
        if not contiguous:
            raise ValueError(f"{what} must be C-contiguous")
        if dtype_name is not None and not str(a.dtype).endswith(dtype_name):
            raise ValueError(f"{what} must be {dtype_name}, not {a.dtype}")
        if numel is not None and n != numel:
            raise ValueError(f"{what} must hold {numel} elements, not {n}")
        if not is_torch and not a.flags.writeable and dtype_name is not None:
            raise ValueError(f"{what} must be writeable")
        return a.data_ptr() if is_torch else a.ctypes.data

    def psd_deposit_uniform_host(self, pos_host, G: int, grid_host, L: float = 1.0,
                                 total_mass: float = 1.0):
        """pos_host / grid_host: host (ideally pinned) torch tensors or numpy arrays."""
        dt, stride, N = _pos_meta(pos_host)
        pp = self._host_ptr(pos_host, "pos_host")
        gp = self._host_ptr(grid_host, "grid_host", "float64", int(G) ** 3)
        self._ck(self._L.psd_deposit_uniform_host(self._h, pp, dt, stride, N, L, total_mass, G, gp))
        return grid_host

    def psd_deposit_patches_host(self, pos_host, base_G: int, P: int, max_level: int, factor: float,
                                 mass_host, rule: int = RULE_BOTTOM_UP_LEVEL_MEAN, L: float = 1.0,
                                 total_mass: float = 1.0):
        """Host-buffer patch deposit: returns the (n, 4) int32 patch list; the masses of patch q
        are mass_host.reshape(-1, P, P, P)[q].  mass_host: float64 host buffer whose capacity
        (elements // P^3) bounds the number of patches."""
        dt, stride, N = _pos_meta(pos_host)
        pp = self._host_ptr(pos_host, "pos_host")
        mp = self._host_ptr(mass_host, "mass_host", "float64")
        n_el = mass_host.numel() if hasattr(mass_host, "numel") else mass_host.size
        cap = int(n_el) // (P ** 3)
        if cap < 1:
            raise ValueError("mass_host has no room for a single patch")
        out = (PsdPatch * cap)()
        n = C.c_int64(0)
        self._ck(self._L.psd_deposit_patches_host(self._h, pp, dt, stride, N, L, total_mass, base_G, P,
                                                  max_level, factor, rule, out, cap, C.byref(n), mp))
        return np.frombuffer(out, dtype=np.int32).reshape(cap, 4)[: n.value].copy()

    def psd_get_stats(self) -> PsdStats:
        s = PsdStats()
        self._ck(self._L.psd_get_stats(self._h, C.byref(s)))
        return s

    def psd_set_option(self, key: int, value: float):
        self._ck(self._L.psd_set_option(self._h, key, float(value)))

    def psd_sync(self):
        self._ck(self._L.psd_sync(self._h))

    def psd_launch_count(self) -> int:
        return int(self._L.psd_launch_count(self._h))

    def psd_get_tile_class_counts(self) -> np.ndarray:
        """(n_tiles, 2) uint32: pairs of each tile by size class (small, large)."""
        n = int(self.psd_get_stats().n_tiles)
        out = np.zeros((max(n, 1), 2), dtype=np.uint32)
        self._ck(self._L.psd_get_tile_class_counts(self._h, out.ctypes.data_as(C.POINTER(C.c_uint32)), 2 * n))
        return out[:n]

    def psd_get_tile_counts(self) -> np.ndarray:
        n = int(self.psd_get_stats().n_tiles)
        out = np.zeros(max(n, 1), dtype=np.uint32)
        self._ck(self._L.psd_get_tile_counts(self._h, out.ctypes.data_as(C.POINTER(C.c_uint32)), n))
        return out[:n]
