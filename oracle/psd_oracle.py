"""ctypes front end of the CPU oracle (oracle/psd_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
import this.  It never imports paper_1612_09491_b200 (the CUDA path) and the CUDA path
never imports it.  Two builds of the same C source: `double` (the timed baseline) and
`gold` (__float128 geometry, tiny inputs only).

Citations are PAPER.md:LINE of /root/reference/PAPER.md (arXiv:1612.09491).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import sys

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "psd_oracle.c")
_LIBS = {"double": os.path.join(_HERE, "libpsd_oracle.so"),
         "gold": os.path.join(_HERE, "libpsd_oracle_gold.so"),
         "single": os.path.join(_HERE, "libpsd_oracle_single.so")}

F32, F64 = 0, 1
MODE_MASS, MODE_SIGNED = 0, 1
TILE = 8


def build(force: bool = False) -> None:
    """Compile both oracle builds with gcc (plain C, OpenMP, no FMA contraction)."""
    for kind, lib in _LIBS.items():
        if not force and os.path.exists(lib) and os.path.getmtime(lib) >= os.path.getmtime(_SRC):
            continue
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
               "-Wall", "-Wextra", _SRC, "-o", lib + ".tmp"]
        if kind == "gold":
            cmd += ["-DPSDO_GOLD", "-lquadmath"]
        if kind == "single":
            cmd += ["-DPSDO_SINGLE", "-Wno-maybe-uninitialized"]
        cmd += ["-lm"]
        subprocess.run(cmd, check=True)
        os.replace(lib + ".tmp", lib)


class _Patch(C.Structure):
    _fields_ = [("level", C.c_int32), ("ox", C.c_int32), ("oy", C.c_int32), ("oz", C.c_int32)]


_loaded: dict[str, C.CDLL] = {}


def _lib(kind: str = "double") -> C.CDLL:
    if kind not in _loaded:
        build()
        lib = C.CDLL(_LIBS[kind])
        vp, i, d, i64p = C.c_void_p, C.c_int, C.c_double, C.POINTER(C.c_int64)
        dp = C.POINTER(C.c_double)
        lib.psdo_deposit_uniform.argtypes = [vp, i, i, i, d, d, i, dp, i, i64p]
        lib.psdo_deposit_window.argtypes = [vp, i, i, i, d, d, i, i64p, i64p, dp, i, i64p]
        lib.psdo_deposit_uniform_range.argtypes = [vp, i, i, i, d, d, i, dp, i, C.c_int64,
                                                   C.c_int64, i64p]
        lib.psdo_census.argtypes = [vp, i, i, i, d, i, i, C.POINTER(C.c_uint32),
                                    C.POINTER(C.c_uint64), C.POINTER(C.c_uint64), i64p]
        lib.psdo_tet_box_volume.argtypes = [dp, dp, d]
        lib.psdo_tet_box_volume.restype = d
        lib.psdo_tet_aabox_volume.argtypes = [dp, dp, dp]
        lib.psdo_tet_aabox_volume.restype = d
        lib.psdo_tet_deposit_box.argtypes = [dp, i64p, i64p, dp, dp]
        lib.psdo_build_tet.argtypes = [vp, i, i, i, d, i, i, i, i, i, dp, dp, i64p]
        lib.psdo_kuhn_table.argtypes = [C.POINTER(C.c_int)]
        lib.psdo_deposit_patches.argtypes = [vp, i, i, i, d, d, i, i, C.POINTER(_Patch),
                                             C.c_int64, dp, i]
        lib.psdo_patch_counts.argtypes = [vp, i, i, i, d, i, i, i, C.POINTER(C.c_uint64)]
        _loaded[kind] = lib
    return _loaded[kind]


def _pos_args(pos: np.ndarray):
    """pos: (N,N,N,3|4) or (N^3,3|4) float32/float64, C-contiguous."""
    if pos.dtype == np.float32:
        dt = F32
    elif pos.dtype == np.float64:
        dt = F64
    else:
        raise TypeError("positions must be float32 or float64")
    if not pos.flags.c_contiguous:
        raise ValueError("positions must be C-contiguous")
    stride = pos.shape[-1]
    n3 = pos.size // stride
    N = round(n3 ** (1.0 / 3.0))
    if N * N * N != n3 or stride not in (3, 4):
        raise ValueError("positions must hold N^3 particles of 3 or 4 components")
    return pos.ctypes.data_as(C.c_void_p), dt, stride, N


def _dp(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _i64p(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_int64))


STAT_KEYS = ("n_tets", "n_candidates", "n_nonzero", "n_degenerate", "n_inverted")


def deposit_uniform(pos, L: float, M: float, G: int, mode: int = MODE_MASS, kind: str = "double"):
    """mass[c] = sum_T m vol(T n C_c)/|V_T| on the periodic G^3 grid."""
    p, dt, stride, N = _pos_args(pos)
    grid = np.empty((G, G, G), dtype=np.float64)
    stats = np.zeros(8, dtype=np.int64)
    rc = _lib(kind).psdo_deposit_uniform(p, dt, stride, N, L, M, G, _dp(grid), mode, _i64p(stats))
    if rc:
        raise ValueError("psdo_deposit_uniform: invalid argument")
    return grid, dict(zip(STAT_KEYS, stats[:5].tolist()))


def deposit_window(pos, L, M, G, win_lo, win_n, mode: int = MODE_MASS, kind: str = "double"):
    """As deposit_uniform but only the cells win_lo <= c < win_lo+win_n (wrapped) are kept."""
    p, dt, stride, N = _pos_args(pos)
    lo = np.asarray(win_lo, dtype=np.int64)
    n = np.asarray(win_n, dtype=np.int64)
    out = np.empty(tuple(int(x) for x in n), dtype=np.float64)
    stats = np.zeros(8, dtype=np.int64)
    rc = _lib(kind).psdo_deposit_window(p, dt, stride, N, L, M, G, _i64p(lo), _i64p(n), _dp(out),
                                        mode, _i64p(stats))
    if rc:
        raise ValueError("psdo_deposit_window: invalid argument")
    return out


def deposit_uniform_range(pos, L, M, G, cell_begin: int, cell_end: int, grid=None,
                          mode: int = MODE_MASS):
    """Deposit only the tets of Lagrangian cells [cell_begin, cell_end) (bounded timing sample)."""
    p, dt, stride, N = _pos_args(pos)
    if grid is None:
        grid = np.zeros((G, G, G), dtype=np.float64)
    stats = np.zeros(8, dtype=np.int64)
    rc = _lib().psdo_deposit_uniform_range(p, dt, stride, N, L, M, G, _dp(grid), mode,
                                           cell_begin, cell_end, _i64p(stats))
    if rc:
        raise ValueError("psdo_deposit_uniform_range: invalid argument")
    return grid, dict(zip(STAT_KEYS, stats[:5].tolist()))


def census(pos, L: float, G: int, tile: int = TILE):
    """O5 counters: per-tile tet counts, size-class histograms (bit-exact vs the GPU)."""
    p, dt, stride, N = _pos_args(pos)
    nt = G // tile
    tc = np.zeros(nt * nt * nt, dtype=np.uint32)
    ht = np.zeros(64, dtype=np.uint64)
    hp = np.zeros(64, dtype=np.uint64)
    sc = np.zeros(8, dtype=np.int64)
    rc = _lib().psdo_census(p, dt, stride, N, L, G, tile,
                            tc.ctypes.data_as(C.POINTER(C.c_uint32)),
                            ht.ctypes.data_as(C.POINTER(C.c_uint64)),
                            hp.ctypes.data_as(C.POINTER(C.c_uint64)), _i64p(sc))
    if rc:
        raise ValueError("psdo_census: invalid argument")
    return {"tile_counts": tc, "hist_tet": ht, "hist_pair": hp, "n_tets": int(sc[0]),
            "n_pairs": int(sc[1]), "sum_cells": int(sc[2]), "max_cells": int(sc[3]),
            "n_inverted": int(sc[4])}


def census_classes(pos, L: float, G: int, tile: int = TILE, small_max: int = 8, win_lo=None, win_n=None):
    """The census at full size (OpenMP over Lagrangian slabs), per tile split by the a3 size class
    of the pair, optionally only for a window of tiles (wrapped tile coordinates)."""
    p, dt, stride, N = _pos_args(pos)
    nt = G // tile
    wl = np.asarray(win_lo if win_lo is not None else (0, 0, 0), dtype=np.int64)
    wn = np.asarray(win_n if win_n is not None else (nt, nt, nt), dtype=np.int64)
    shape = tuple(int(x) for x in wn)
    cs = np.zeros(shape, dtype=np.uint32)
    cl = np.zeros(shape, dtype=np.uint32)
    ht = np.zeros(64, dtype=np.uint64)
    hp = np.zeros(64, dtype=np.uint64)
    sc = np.zeros(8, dtype=np.int64)
    lib = _lib()
    u32p, u64p = C.POINTER(C.c_uint32), C.POINTER(C.c_uint64)
    lib.psdo_census_classes.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_double, C.c_int, C.c_int,
                                        C.c_int64, C.POINTER(C.c_int64), C.POINTER(C.c_int64), u32p, u32p,
                                        u64p, u64p, C.POINTER(C.c_int64)]
    windowed = win_lo is not None
    rc = lib.psdo_census_classes(p, dt, stride, N, L, G, tile, small_max,
                                 _i64p(wl) if windowed else None, _i64p(wn) if windowed else None,
                                 cs.ctypes.data_as(u32p), cl.ctypes.data_as(u32p),
                                 ht.ctypes.data_as(u64p), hp.ctypes.data_as(u64p), _i64p(sc))
    if rc:
        raise ValueError(f"psdo_census_classes: rc={rc}")
    return {"counts_small": cs, "counts_large": cl, "hist_tet": ht, "hist_pair": hp, "n_tets": int(sc[0]),
            "n_pairs": int(sc[1]), "sum_cells": int(sc[2]), "max_cells": int(sc[3]), "n_inverted": int(sc[4])}


def deposit_windows(pos, L, M, G, windows, mode: int = MODE_MASS):
    """Several windows [(lo, n), ...] of the grid in one pass over the tets (see deposit_window)."""
    p, dt, stride, N = _pos_args(pos)
    K = len(windows)
    lo = np.array([w[0] for w in windows], dtype=np.int64).reshape(K, 3)
    n = np.array([w[1] for w in windows], dtype=np.int64).reshape(K, 3)
    sizes = [int(np.prod(r)) for r in n]
    out = np.empty(sum(sizes), dtype=np.float64)
    lib = _lib()
    lib.psdo_deposit_windows.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_int,
                                         C.c_int, C.POINTER(C.c_int64), C.POINTER(C.c_int64),
                                         C.POINTER(C.c_double), C.c_int]
    rc = lib.psdo_deposit_windows(p, dt, stride, N, L, M, G, K, _i64p(lo), _i64p(n), _dp(out), mode)
    if rc:
        raise ValueError("psdo_deposit_windows: invalid argument")
    res, o = [], 0
    for r, sz in zip(n, sizes):
        res.append(out[o:o + sz].reshape(tuple(int(x) for x in r)))
        o += sz
    return res


def extreme_tets(pos, L: float, G: int, min_cells: int = 8):
    """The tet with the largest cell range and the thinnest one (smallest |det| / AABB volume):
    where the full-size parity tests aim their windows."""
    p, dt, stride, N = _pos_args(pos)
    out = np.zeros(16, dtype=np.int64)
    thin = C.c_double(0.0)
    lib = _lib()
    lib.psdo_extreme_tets.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_double, C.c_int, C.c_int64,
                                      C.POINTER(C.c_int64), C.POINTER(C.c_double)]
    rc = lib.psdo_extreme_tets(p, dt, stride, N, L, G, min_cells, _i64p(out), C.byref(thin))
    if rc:
        raise ValueError("psdo_extreme_tets: invalid argument")
    return {"largest": {"tet": tuple(out[0:4].tolist()), "lo": out[4:7].copy(), "n_cells": int(out[7])},
            "thinnest": {"tet": tuple(out[8:12].tolist()), "lo": out[12:15].copy(), "ratio": thin.value}}


def tet_box_volume(verts, lo, h: float, kind: str = "double") -> float:
    """vol(T n [lo,lo+h]^3) by iterative plane splitting."""
    v = np.ascontiguousarray(verts, dtype=np.float64).reshape(12)
    l = np.ascontiguousarray(lo, dtype=np.float64).reshape(3)
    return float(_lib(kind).psdo_tet_box_volume(_dp(v), _dp(l), float(h)))


def tet_aabox_volume(verts, lo, hi, kind: str = "double") -> float:
    """vol(T n prod[lo_x,hi_x]) for a general axis-aligned box."""
    v = np.ascontiguousarray(verts, dtype=np.float64).reshape(12)
    l = np.ascontiguousarray(lo, dtype=np.float64).reshape(3)
    h = np.ascontiguousarray(hi, dtype=np.float64).reshape(3)
    return float(_lib(kind).psdo_tet_aabox_volume(_dp(v), _dp(l), _dp(h)))


def tet_deposit_box(verts_grid_units, lo, n, kind: str = "double"):
    """Overlap volumes (cell units) of one tet with each unit cell of an integer box."""
    v = np.ascontiguousarray(verts_grid_units, dtype=np.float64).reshape(12)
    lo = np.asarray(lo, dtype=np.int64)
    n = np.asarray(n, dtype=np.int64)
    out = np.empty(tuple(int(x) for x in n), dtype=np.float64)
    vol = C.c_double(0.0)
    _lib(kind).psdo_tet_deposit_box(_dp(v), _i64p(lo), _i64p(n), _dp(out), C.byref(vol))
    return out, vol.value


def build_tet(pos, L: float, G: int, i: int, j: int, k: int, t: int):
    """Unwrapped vertices (box units), signed det (grid units) and cell range of one tet."""
    p, dt, stride, N = _pos_args(pos)
    verts = np.empty((4, 3), dtype=np.float64)
    det = C.c_double(0.0)
    lohi = np.zeros(6, dtype=np.int64)
    rc = _lib().psdo_build_tet(p, dt, stride, N, L, G, i, j, k, t, _dp(verts), C.byref(det),
                               _i64p(lohi))
    if rc:
        raise ValueError("psdo_build_tet: invalid argument")
    return verts, det.value, lohi[:3].copy(), lohi[3:].copy()


def kuhn_table() -> np.ndarray:
    out = (C.c_int * 24)()
    _lib().psdo_kuhn_table(out)
    return np.array(out[:], dtype=np.int64).reshape(6, 4)


def deposit_patches(pos, L, M, base_G: int, P: int, patches, mode: int = MODE_MASS,
                    kind: str = "double") -> np.ndarray:
    """patches: (n,4) int32 rows {level, ox, oy, oz}; returns (n,P,P,P) masses."""
    p, dt, stride, N = _pos_args(pos)
    pa = np.ascontiguousarray(patches, dtype=np.int32).reshape(-1, 4)
    n = pa.shape[0]
    mass = np.empty((n, P, P, P), dtype=np.float64)
    rc = _lib(kind).psdo_deposit_patches(p, dt, stride, N, L, M, base_G, P,
                                         pa.ctypes.data_as(C.POINTER(_Patch)), n, _dp(mass), mode)
    if rc:
        raise ValueError("psdo_deposit_patches: invalid argument")
    return mass


def deposit_patches_stats(pos, L, M, base_G: int, P: int, patches):
    """deposit_patches plus per-patch counters: (masses, (n,2) int64 [candidate cells, cells with
    non-zero overlap]) -- the method-defined counts bench.py's work model uses."""
    p, dt, stride, N = _pos_args(pos)
    pa = np.ascontiguousarray(patches, dtype=np.int32).reshape(-1, 4)
    n = pa.shape[0]
    mass = np.empty((n, P, P, P), dtype=np.float64)
    st = np.zeros((n, 2), dtype=np.int64)
    lib = _lib()
    lib.psdo_deposit_patches_stats.argtypes = list(lib.psdo_deposit_patches.argtypes) + [C.POINTER(C.c_int64)]
    rc = lib.psdo_deposit_patches_stats(p, dt, stride, N, L, M, base_G, P,
                                        pa.ctypes.data_as(C.POINTER(_Patch)), n, _dp(mass), MODE_MASS,
                                        _i64p(st))
    if rc:
        raise ValueError("psdo_deposit_patches_stats: invalid argument")
    return mass, st


def patch_counts(pos, L, base_G: int, P: int, level: int) -> np.ndarray:
    """#tets whose cell range meets each candidate patch position of `level`."""
    p, dt, stride, N = _pos_args(pos)
    npos = (base_G << level) // P
    cnt = np.zeros((npos, npos, npos), dtype=np.uint64)
    rc = _lib().psdo_patch_counts(p, dt, stride, N, L, base_G, P, level,
                                  cnt.ctypes.data_as(C.POINTER(C.c_uint64)))
    if rc:
        raise ValueError("psdo_patch_counts: invalid argument")
    return cnt


SUBBLOCK_UNIT = 1 << 20  # subblock_counts are in units of 2^-20 tets


def subblock_counts(pos, L, base_G: int, P: int, level: int, B: int = 8) -> np.ndarray:
    """tets over each candidate patch position of `level`, ESTIMATED from the
    bounding boxes of the B^3-cell Lagrangian sub-blocks (uint64, units of 2^-20 tets)."""
    p, dt, stride, N = _pos_args(pos)
    npos = (base_G << level) // P
    cnt = np.zeros((npos, npos, npos), dtype=np.uint64)
    lib = _lib()
    lib.psdo_subblock_counts.restype = C.c_int
    lib.psdo_subblock_counts.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_double, C.c_int,
                                         C.c_int, C.c_int, C.c_int, C.POINTER(C.c_uint64)]
    rc = lib.psdo_subblock_counts(p, dt, stride, N, L, base_G, P, level, B,
                                  cnt.ctypes.data_as(C.POINTER(C.c_uint64)))
    if rc:
        raise ValueError(f"psdo_subblock_counts: rc={rc}")
    return cnt


RULE_LITERAL_TOP_DOWN = 0
RULE_BOTTOM_UP_LEVEL_MEAN = 1


def refine_patches(counts, factor: float, rule: int = RULE_BOTTOM_UP_LEVEL_MEAN) -> np.ndarray:
    """Patch list from per-level candidate counts (reading Q14).

    counts[l] is the dense patch_counts array of level l (l = 0..max_level).
    rule 1 (BOTTOM_UP_LEVEL_MEAN): a candidate at level l >= 1 is *hot* if its count exceeds
    factor x the mean count over all candidate positions of that level.  A level-(l-1) patch
    is refined (all 8 children created) if any child is hot or itself must be refined.
    rule 0 (LITERAL_TOP_DOWN): threshold = factor x mean of the level-0 counts; a patch whose
    count exceeds it is refined, children tested against the same absolute number.
    Level 0 is always complete.  Order: level, then (ox,oy,oz) lexicographic.
    """
    nl = len(counts)
    need = [np.zeros(c.shape, dtype=bool) for c in counts]  # patch exists
    need[0][...] = True
    if rule == RULE_BOTTOM_UP_LEVEL_MEAN:
        hot = [None] * nl
        for l in range(1, nl):
            c = counts[l].astype(np.float64)
            hot[l] = c > factor * c.mean()
        refine = [np.zeros(c.shape, dtype=bool) for c in counts]  # patch is split into 8
        for l in range(nl - 2, -1, -1):
            child = hot[l + 1] | refine[l + 1]
            n = counts[l].shape[0]
            refine[l] = child.reshape(n, 2, n, 2, n, 2).any(axis=(1, 3, 5))
        for l in range(1, nl):
            par = refine[l - 1] & need[l - 1]
            need[l] = np.repeat(np.repeat(np.repeat(par, 2, 0), 2, 1), 2, 2)
    else:
        thr = factor * counts[0].astype(np.float64).mean()
        for l in range(1, nl):
            par = need[l - 1] & (counts[l - 1].astype(np.float64) > thr)
            need[l] = np.repeat(np.repeat(np.repeat(par, 2, 0), 2, 1), 2, 2)
    rows = []
    for l in range(nl):
        idx = np.argwhere(need[l])
        rows.append(np.concatenate([np.full((idx.shape[0], 1), l), idx], axis=1))
    return np.concatenate(rows, axis=0).astype(np.int32)


def num_threads() -> int:
    return int(_lib().psdo_num_threads())


if __name__ == "__main__":
    build(force="--force" in sys.argv)
    print("built:", ", ".join(_LIBS.values()))
