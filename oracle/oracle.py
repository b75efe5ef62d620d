"""ctypes front-end of the CPU oracle (oracle/xy_oracle.c).

TEST INFRASTRUCTURE, not the product: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs import this.  It imports nothing from the package.
Every function is argument marshalling around the C routine of the same name.
"""
import ctypes as C
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import build_oracle  # noqa: E402

NACC = 8
_lib = None

_i32p = np.ctypeslib.ndpointer(np.int32, flags="C_CONTIGUOUS")
_f32p = np.ctypeslib.ndpointer(np.float32, flags="C_CONTIGUOUS")
_f64p = np.ctypeslib.ndpointer(np.float64, flags="C_CONTIGUOUS")
_u32p = np.ctypeslib.ndpointer(np.uint32, flags="C_CONTIGUOUS")


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build_oracle.build())
        L.orc_philox4x32_10.argtypes = [_u32p, _u32p, _u32p]
        L.orc_philox4x32_10.restype = None
        L.orc_u01.argtypes = [C.c_uint32]
        L.orc_u01.restype = C.c_float
        L.orc_slot_uniforms.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32,
                                        C.c_uint32, C.c_uint32, C.POINTER(C.c_float),
                                        C.POINTER(C.c_float)]
        L.orc_slot_uniforms.restype = None
        L.orc_levy_edges.argtypes = [C.c_int, C.c_double, C.c_int, C.c_uint64, C.c_uint32, _i32p,
                                     C.c_int64]
        L.orc_levy_edges.restype = C.c_int64
        L.orc_levy_edges_fbc.argtypes = L.orc_levy_edges.argtypes
        L.orc_levy_edges_fbc.restype = C.c_int64
        L.orc_csr_from_edges.argtypes = [C.c_int, C.c_int, _i32p, _i32p, _i32p]
        L.orc_csr_from_edges.restype = None
        L.orc_colour_smallest_last.argtypes = [C.c_int, _i32p, _i32p, _i32p]
        L.orc_colour_smallest_last.restype = C.c_int
        L.orc_renumber_colour_major.argtypes = [C.c_int, _i32p, _i32p, _i32p, _i32p, _i32p, _i32p,
                                                _i32p]
        L.orc_renumber_colour_major.restype = None
        L.orc_colouring_is_proper.argtypes = [C.c_int, _i32p, _i32p, _i32p]
        L.orc_colouring_is_proper.restype = C.c_int
        L.orc_geometric_temperatures.argtypes = [C.c_int, C.c_double, C.c_double, _f64p]
        L.orc_geometric_temperatures.restype = None
        L.orc_temperature_params.argtypes = [C.c_int, _f64p, _f32p, _f32p]
        L.orc_temperature_params.restype = None
        L.orc_init_theta.argtypes = [C.c_int, C.c_int, C.c_uint64, C.c_uint32, _f32p]
        L.orc_init_theta.restype = None
        L.orc_metropolis_sites.argtypes = [C.c_int, C.c_int, _i32p, _i32p, _f32p, _i32p, C.c_int,
                                           _f32p, _f32p, C.c_uint64, C.c_uint32, C.c_uint32,
                                           C.c_void_p, C.c_void_p]
        L.orc_metropolis_sites.restype = None
        L.orc_overrelax_sites.argtypes = [C.c_int, C.c_int, _i32p, _i32p, _f32p, _i32p, C.c_int,
                                          C.c_void_p]
        L.orc_overrelax_sites.restype = None
        L.orc_measure.argtypes = [C.c_int, C.c_int, _i32p, _i32p, _f32p, _f64p, _f64p, _f64p]
        L.orc_measure.restype = None
        L.orc_accumulate.argtypes = [C.c_int, C.c_int, _f64p, _f64p, _f64p, _i32p, _f64p]
        L.orc_accumulate.restype = None
        L.orc_pt_swap.argtypes = [C.c_int, _f64p, _f64p, _i32p, _i32p, C.c_uint64, C.c_uint32,
                                  C.c_uint32, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_pt_swap.restype = None
        L.orc_fourier.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, _i32p, _i32p, _f32p, _f64p, _f64p]
        L.orc_fourier.restype = None
        L.orc_xi2.argtypes = [C.c_double, C.c_double, C.c_int, C.c_double]
        L.orc_xi2.restype = C.c_double
        L.orc_random_walk.argtypes = [C.c_int, _i32p, _i32p, C.c_int, _i32p, C.c_int, C.c_uint64, C.c_uint32,
                                      np.ctypeslib.ndpointer(np.int64, flags="C_CONTIGUOUS")]
        L.orc_random_walk.restype = None
        L.orc_run.argtypes = [C.c_int, C.c_int, C.c_int, _i32p, _i32p, _i32p, _f32p, _f64p, _i32p,
                              _i32p, C.c_uint64, C.c_uint32, C.POINTER(C.c_uint32),
                              C.POINTER(C.c_uint32), C.c_int, C.c_int, C.c_int, C.c_int, _f64p,
                              C.c_void_p, C.c_void_p]
        L.orc_run.restype = None
        L.orc_run_order.argtypes = [C.c_int, C.c_int, C.c_int, _i32p, _i32p, _i32p, _f32p, _f64p, _i32p,
                                    _i32p, C.c_uint64, C.c_uint32, C.POINTER(C.c_uint32),
                                    C.POINTER(C.c_uint32), C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, _f64p,
                                    C.c_void_p, C.c_void_p]
        L.orc_run_order.restype = None
        _lib = L
    return _lib


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def philox4x32_10(ctr, key):
    out = np.zeros(4, np.uint32)
    lib().orc_philox4x32_10(np.ascontiguousarray(ctr, np.uint32), np.ascontiguousarray(key, np.uint32), out)
    return out


def u01(x):
    return float(lib().orc_u01(int(x) & 0xFFFFFFFF))


def slot_uniforms(seed, domain, site, sweep, sample, slot):
    a, b = C.c_float(), C.c_float()
    lib().orc_slot_uniforms(seed, domain, site, sweep, sample, slot, C.byref(a), C.byref(b))
    return a.value, b.value


def levy_edges(L, rho, z, seed, sample, max_draws=1 << 40, boundary="periodic"):
    N = L * L
    edges = np.zeros((N * z // 2, 2), np.int32)
    fn = lib().orc_levy_edges if boundary == "periodic" else lib().orc_levy_edges_fbc
    draws = fn(L, float(rho), z, seed, sample, edges, max_draws)
    if draws < 0:
        raise RuntimeError("orc_levy_edges failed")
    return edges, int(draws)


def csr_from_edges(N, edges):
    edges = np.ascontiguousarray(edges, np.int32).reshape(-1, 2)
    row_ptr = np.zeros(N + 1, np.int32)
    col_idx = np.zeros(max(2 * len(edges), 1), np.int32)
    lib().orc_csr_from_edges(N, len(edges), edges if len(edges) else np.zeros((1, 2), np.int32),
                             row_ptr, col_idx)
    return row_ptr, col_idx[: 2 * len(edges)].copy() if len(edges) else np.zeros(0, np.int32)


def _ci(col_idx):
    col_idx = np.ascontiguousarray(col_idx, np.int32)
    return col_idx if col_idx.size else np.zeros(1, np.int32)


def colour_smallest_last(row_ptr, col_idx):
    N = len(row_ptr) - 1
    colour = np.zeros(N, np.int32)
    Q = lib().orc_colour_smallest_last(N, row_ptr, _ci(col_idx), colour)
    return colour, int(Q)


def renumber_colour_major(row_ptr, col_idx, colour):
    N = len(row_ptr) - 1
    new_to_old = np.zeros(N, np.int32)
    rp = np.zeros(N + 1, np.int32)
    ci = np.zeros(max(len(col_idx), 1), np.int32)
    cn = np.zeros(N, np.int32)
    lib().orc_renumber_colour_major(N, row_ptr, _ci(col_idx), colour, new_to_old, rp, ci, cn)
    return new_to_old, rp, ci[: len(col_idx)].copy(), cn


def colouring_is_proper(row_ptr, col_idx, colour):
    return bool(lib().orc_colouring_is_proper(len(row_ptr) - 1, row_ptr, _ci(col_idx),
                                              np.ascontiguousarray(colour, np.int32)))


def class_ptr_from_colour(colour):
    """colour must be non-decreasing (colour-major numbering); returns class_ptr[Q+1]."""
    colour = np.asarray(colour)
    assert np.all(np.diff(colour) >= 0)
    Q = int(colour.max()) + 1 if len(colour) else 0
    return np.searchsorted(colour, np.arange(Q + 1)).astype(np.int32)


def geometric_temperatures(R, Tmin, Tmax):
    T = np.zeros(R, np.float64)
    lib().orc_geometric_temperatures(R, Tmin, Tmax, T)
    return T


def temperature_params(T):
    T = np.ascontiguousarray(T, np.float64)
    b = np.zeros(len(T), np.float32)
    w = np.zeros(len(T), np.float32)
    lib().orc_temperature_params(len(T), T, b, w)
    return b, w


def init_theta(N, R, seed, sample):
    th = np.zeros((N, R), np.float32)
    lib().orc_init_theta(N, R, seed, sample, th)
    return th


def metropolis_sites(row_ptr, col_idx, theta, sites, beta_slot, w_slot, seed, sweep, sample,
                     want_margin=False):
    """In-place on theta [N][R].  Returns (margin, accepted) arrays [len(sites)][R] or (None, None)."""
    N, R = theta.shape
    sites = np.ascontiguousarray(sites, np.int32)
    margin = np.zeros((len(sites), R), np.float64) if want_margin else None
    acc = np.zeros((len(sites), R), np.uint8) if want_margin else None
    lib().orc_metropolis_sites(N, R, row_ptr, _ci(col_idx), theta, sites if len(sites) else np.zeros(1, np.int32),
                               len(sites), np.ascontiguousarray(beta_slot, np.float32),
                               np.ascontiguousarray(w_slot, np.float32), seed, sweep, sample,
                               _ptr(margin), _ptr(acc))
    return margin, acc


def overrelax_sites(row_ptr, col_idx, theta, sites, want_hnorm=False):
    N, R = theta.shape
    sites = np.ascontiguousarray(sites, np.int32)
    hn = np.zeros((len(sites), R), np.float64) if want_hnorm else None
    lib().orc_overrelax_sites(N, R, row_ptr, _ci(col_idx), theta, sites if len(sites) else np.zeros(1, np.int32),
                              len(sites), _ptr(hn))
    return hn


def measure(row_ptr, col_idx, theta):
    N, R = theta.shape
    E = np.zeros(R); Mx = np.zeros(R); My = np.zeros(R)
    lib().orc_measure(N, R, row_ptr, _ci(col_idx), theta, E, Mx, My)
    return E, Mx, My


def fourier(Lx, Ly, x, y, theta):
    """G1, G2 [R]: |sum_i S_i exp(i k r_i)|^2 / N at k = (2 pi/Lx, 0) and (0, 2 pi/Ly)."""
    N, R = theta.shape
    G1 = np.zeros(R); G2 = np.zeros(R)
    lib().orc_fourier(N, R, Lx, Ly, np.ascontiguousarray(x, np.int32), np.ascontiguousarray(y, np.int32), theta, G1, G2)
    return G1, G2


def xi2(chi0, chik, L, psi=2.0):
    return float(lib().orc_xi2(float(chi0), float(chik), int(L), float(psi)))


def random_walk(row_ptr, col_idx, start, n_steps, seed, sample=0):
    """hist [n_steps+1] int64: visits of the origin at time t, summed over the walkers."""
    start = np.ascontiguousarray(start, np.int32)
    hist = np.zeros(n_steps + 1, np.int64)
    lib().orc_random_walk(len(row_ptr) - 1, np.ascontiguousarray(row_ptr, np.int32), _ci(col_idx), len(start), start,
                          n_steps, seed, sample, hist)
    return hist


def accumulate(N, E, Mx, My, temp_of_slot, acc):
    lib().orc_accumulate(N, len(E), E, Mx, My, np.ascontiguousarray(temp_of_slot, np.int32), acc)


def pt_swap(T, E_slot, slot_of_temp, temp_of_slot, seed, round_, sample, decisions_in=None):
    """In-place on the two label arrays.  Returns (decisions[R], margin[R]) for attempted pairs."""
    R = len(T)
    dec = np.zeros(R, np.uint8)
    mar = np.full(R, np.inf, np.float64)
    din = None if decisions_in is None else np.ascontiguousarray(decisions_in, np.uint8)
    lib().orc_pt_swap(R, np.ascontiguousarray(T, np.float64), np.ascontiguousarray(E_slot, np.float64),
                      slot_of_temp, temp_of_slot, seed, round_, sample, _ptr(din), _ptr(dec), _ptr(mar))
    return dec, mar


class Chain:
    """State of one sample's PT ensemble driven by orc_run."""

    def __init__(self, row_ptr, col_idx, class_ptr, T, seed, sample=0, theta=None):
        self.row_ptr = np.ascontiguousarray(row_ptr, np.int32)
        self.col_idx = _ci(col_idx)
        self.class_ptr = np.ascontiguousarray(class_ptr, np.int32)
        self.N = len(self.row_ptr) - 1
        self.Q = len(self.class_ptr) - 1
        self.T = np.ascontiguousarray(T, np.float64)
        self.R = len(self.T)
        self.seed, self.sample = seed, sample
        self.theta = init_theta(self.N, self.R, seed, sample) if theta is None else np.ascontiguousarray(theta, np.float32)
        self.temp_of_slot = np.arange(self.R, dtype=np.int32)
        self.slot_of_temp = np.arange(self.R, dtype=np.int32)
        self.sweep = C.c_uint32(0)
        self.round = C.c_uint32(0)
        self.acc = np.zeros((self.R, NACC), np.float64)
        self.swap_attempts = np.zeros(max(self.R - 1, 1), np.int64)
        self.swap_accepts = np.zeros(max(self.R - 1, 1), np.int64)

    def run(self, n_cycles, sweeps_per_swap=10, or_per_sweep=1, measure_every=1, order=0):
        lib().orc_run_order(self.N, self.R, self.Q, self.row_ptr, self.col_idx, self.class_ptr,
                            self.theta, self.T, self.temp_of_slot, self.slot_of_temp, self.seed,
                            self.sample, C.byref(self.sweep), C.byref(self.round), n_cycles,
                            sweeps_per_swap, or_per_sweep, measure_every, order, self.acc,
                            _ptr(self.swap_attempts), _ptr(self.swap_accepts))

    def reset_acc(self):
        self.acc[:] = 0.0
