"""Seeded input generator: Levy graphs + smallest-last colouring (ctypes binding of libxy_levy.so).

Shared by the CUDA harness, bench.py and the tests that drive the oracle; it holds none of the
Monte-Carlo arithmetic (include/xy_levy.h).
"""
import ctypes as C
from dataclasses import dataclass

import numpy as np

from . import _build

_lib = None
_i32p = np.ctypeslib.ndpointer(np.int32, flags="C_CONTIGUOUS")


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build_levy())
        L.xy_levy_build.argtypes = [C.c_int, C.c_double, C.c_int, C.c_uint64, C.c_uint32, C.c_int, C.c_int,
                                    _i32p, _i32p, _i32p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.xy_levy_build.restype = C.c_int
        L.xy_levy_build_fbc.argtypes = L.xy_levy_build.argtypes
        L.xy_levy_build_fbc.restype = C.c_int
        L.xy_levy_build_opt.argtypes = [C.c_int, C.c_int] + L.xy_levy_build.argtypes
        L.xy_levy_build_opt.restype = C.c_int
        L.xy_colour_smallest_last.argtypes = [C.c_int, _i32p, _i32p, _i32p]
        L.xy_colour_smallest_last.restype = C.c_int
        L.xy_colour_reduce.argtypes = [C.c_int, _i32p, _i32p, _i32p, C.c_int, C.c_uint64, C.c_uint32, C.c_int64]
        L.xy_colour_reduce.restype = C.c_int
        L.xy_renumber_colour_major.argtypes = [C.c_int, _i32p, _i32p, _i32p, _i32p, _i32p, _i32p, _i32p]
        L.xy_renumber_colour_major.restype = C.c_int
        L.xy_levy_last_error.restype = C.c_char_p
        _lib = L
    return _lib


class LevyError(RuntimeError):
    pass


@dataclass
class LevyGraphs:
    """S coloured samples in colour-major numbering (all HOST numpy arrays)."""
    L: int
    rho: float
    z: int
    seed: int
    sample_base: int
    row_ptr: np.ndarray      # [S][N+1] int32
    col_idx: np.ndarray      # [S][N*z] int32
    colour: np.ndarray       # [S][N]   int32, non-decreasing per sample
    new_to_old: np.ndarray   # [S][N]   int32 lattice id y*L+x of each site
    n_colours: np.ndarray    # [S]      int32
    n_draws: np.ndarray      # [S]      int64

    @property
    def S(self):
        return self.row_ptr.shape[0]

    @property
    def N(self):
        return self.L * self.L

    def class_ptr(self, s):
        Q = int(self.n_colours[s])
        return np.searchsorted(self.colour[s], np.arange(Q + 1)).astype(np.int32)


def build(L, rho, z, seed, S=1, sample_base=0, n_threads=0, boundary="periodic", reduce_colours=0):
    """reduce_colours = moves per site of the colour-reducing local search after the smallest-last colouring
    (xy_levy_build_opt; 0 = the plain smallest-last colouring that the oracle restates bit for bit)."""
    N = L * L
    row_ptr = np.zeros((S, N + 1), np.int32)
    col_idx = np.zeros((S, N * z), np.int32)
    colour = np.zeros((S, N), np.int32)
    n2o = np.zeros((S, N), np.int32)
    nq = np.zeros(S, np.int32)
    nd = np.zeros(S, np.int64)
    if boundary not in ("periodic", "free"):
        raise ValueError("boundary must be 'periodic' or 'free'")
    out = (row_ptr.reshape(-1), col_idx.reshape(-1), colour.reshape(-1), n2o.ctypes.data, nq.ctypes.data, nd.ctypes.data)
    if reduce_colours:
        rc = lib().xy_levy_build_opt(int(boundary == "free"), int(reduce_colours), L, float(rho), z, seed, sample_base, S,
                                     n_threads, *out)
    else:
        fn = lib().xy_levy_build if boundary == "periodic" else lib().xy_levy_build_fbc
        rc = fn(L, float(rho), z, seed, sample_base, S, n_threads, *out)
    if rc != 0:
        raise LevyError(f"xy_levy_build: {rc}: {lib().xy_levy_last_error().decode()}")
    return LevyGraphs(L, float(rho), z, seed, sample_base, row_ptr, col_idx, colour, n2o, nq, nd)


def colour_smallest_last(row_ptr, col_idx):
    row_ptr = np.ascontiguousarray(row_ptr, np.int32)
    col_idx = np.ascontiguousarray(col_idx, np.int32)
    N = len(row_ptr) - 1
    colour = np.zeros(max(N, 1), np.int32)
    Q = lib().xy_colour_smallest_last(N, row_ptr, col_idx if col_idx.size else np.zeros(1, np.int32), colour)
    if Q < 0:
        raise LevyError(lib().xy_levy_last_error().decode())
    return colour[:N], Q


def colour_reduce(row_ptr, col_idx, colour, target_q, seed, sample=0, max_moves=None):
    """local search for a proper colouring with fewer colours; returns (colour, Q)"""
    row_ptr = np.ascontiguousarray(row_ptr, np.int32)
    col_idx = np.ascontiguousarray(col_idx, np.int32)
    colour = np.array(colour, np.int32, copy=True)
    N = len(row_ptr) - 1
    Q = lib().xy_colour_reduce(N, row_ptr, col_idx if col_idx.size else np.zeros(1, np.int32), colour, target_q, seed, sample,
                               64 * N if max_moves is None else max_moves)
    if Q < 0:
        raise LevyError(lib().xy_levy_last_error().decode())
    return colour, Q


def renumber_colour_major(row_ptr, col_idx, colour):
    row_ptr = np.ascontiguousarray(row_ptr, np.int32)
    col_idx = np.ascontiguousarray(col_idx, np.int32)
    colour = np.ascontiguousarray(colour, np.int32)
    N = len(row_ptr) - 1
    n2o = np.zeros(N, np.int32); rp = np.zeros(N + 1, np.int32)
    ci = np.zeros(max(len(col_idx), 1), np.int32); cn = np.zeros(N, np.int32)
    rc = lib().xy_renumber_colour_major(N, row_ptr, col_idx if col_idx.size else np.zeros(1, np.int32), colour,
                                        n2o, rp, ci, cn)
    if rc != 0:
        raise LevyError(lib().xy_levy_last_error().decode())
    return n2o, rp, ci[: len(col_idx)].copy(), cn
