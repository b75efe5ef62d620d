"""Thin Python binding of the C ABI in include/xy_b200.h: same names, argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind libxy_b200.so.  PyTorch is used for device
memory (the theta tensor) and the CUDA stream, nothing else.  There is no CPU fallback: if the library
cannot be built or loaded, or no CUDA device is present, the calls raise.
"""
import ctypes as C

import numpy as np

from . import _build

XY_OK, XY_EINVAL, XY_ENOMEM, XY_ECUDA, XY_EGRAPH, XY_ESTATE = 0, -1, -2, -3, -4, -5
XY_NACC = 8
_CODES = {XY_EINVAL: "XY_EINVAL", XY_ENOMEM: "XY_ENOMEM", XY_ECUDA: "XY_ECUDA", XY_EGRAPH: "XY_EGRAPH",
          XY_ESTATE: "XY_ESTATE"}

# every symbol include/xy_b200.h declares (tests/test_abi_symbols.py checks the header against this list)
SYMBOLS = {
    "xy_last_error": (C.c_char_p, []),
    "xy_abi_version": (C.c_int, []),
    "xy_graph_load": (C.c_int, [C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(C.c_void_p)]),
    "xy_graph_free": (C.c_int, [C.c_void_p]),
    "xy_graph_set_coords": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p]),
    "xy_measure_fourier": (C.c_int, [C.c_void_p, C.c_void_p]),
    "xy_read_fourier_accumulators": (C.c_int, [C.c_void_p, C.c_void_p]),
    "xy_random_walk": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_uint64, C.c_uint32, C.c_void_p, C.c_void_p]),
    "xy_random_walk_kernel_us": (C.c_int, [C.POINTER(C.c_double)]),
    "xy_random_walk_static": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_uint64, C.c_uint32, C.c_void_p, C.c_void_p]),
    "xy_set_path": (C.c_int, [C.c_void_p, C.c_int]),
    "xy_get_path": (C.c_int, [C.c_void_p, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_int)]),
    "xy_get_schedule": (C.c_int, [C.c_void_p, C.POINTER(C.c_int), C.POINTER(C.c_int64)]),
    "xy_graph_info": (C.c_int, [C.c_void_p, C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int64),
                                C.POINTER(C.c_int), C.POINTER(C.c_int)]),
    "xy_pt_create": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint32, C.c_void_p,
                               C.c_void_p, C.POINTER(C.c_void_p)]),
    "xy_pt_destroy": (C.c_int, [C.c_void_p]),
    "xy_sweep": (C.c_int, [C.c_void_p, C.c_int]),
    "xy_sweep_acceptance": (C.c_int, [C.c_void_p, C.c_void_p]),
    "xy_overrelax": (C.c_int, [C.c_void_p, C.c_int]),
    "xy_pt_swap": (C.c_int, [C.c_void_p]),
    "xy_measure": (C.c_int, [C.c_void_p, C.c_void_p]),
    "xy_run": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int]),
    "xy_run_sweeps": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_int]),
    "xy_set_schedule": (C.c_int, [C.c_void_p, C.c_int]),
    "xy_set_tuning": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int]),
    "xy_metropolis_colour": (C.c_int, [C.c_void_p, C.c_int, C.c_uint32]),
    "xy_overrelax_colour": (C.c_int, [C.c_void_p, C.c_int]),
    "xy_metor_colour": (C.c_int, [C.c_void_p, C.c_int, C.c_uint32]),
    "xy_set_order": (C.c_int, [C.c_void_p, C.c_int]),
    "xy_get_theta": (C.c_int, [C.c_void_p, C.c_void_p]),
    "xy_set_theta": (C.c_int, [C.c_void_p, C.c_void_p]),
    "xy_set_theta_async": (C.c_int, [C.c_void_p, C.c_void_p]),
    "xy_get_labels": (C.c_int, [C.c_void_p, C.c_void_p]),
    "xy_set_labels": (C.c_int, [C.c_void_p, C.c_void_p]),
    "xy_get_energy": (C.c_int, [C.c_void_p, C.c_void_p]),
    "xy_swap_with_decisions": (C.c_int, [C.c_void_p, C.c_void_p]),
    "xy_read_accumulators": (C.c_int, [C.c_void_p, C.c_void_p]),
    "xy_reset_accumulators": (C.c_int, [C.c_void_p]),
    "xy_get_counters": (C.c_int, [C.c_void_p, C.POINTER(C.c_uint32), C.POINTER(C.c_uint32), C.c_void_p, C.c_void_p]),
    "xy_set_counters": (C.c_int, [C.c_void_p, C.c_uint32, C.c_uint32]),
    "xy_theta_device": (C.c_int, [C.c_void_p, C.POINTER(C.c_void_p)]),
    "xy_launch_count": (C.c_int, [C.c_void_p, C.POINTER(C.c_int64)]),
    "xy_synchronize": (C.c_int, [C.c_void_p]),
    "xy_l2_bandwidth": (C.c_int, [C.c_size_t, C.c_int, C.c_int, C.c_void_p, C.POINTER(C.c_double)]),
}

_lib = None


class XYError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{_CODES.get(code, code)}: {msg}")
        self.code = code


def lib():
    """Load (building if stale) libxy_b200.so.  Raises if nvcc or the build fails: there is no fallback."""
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build_xy())
        for name, (res, args) in SYMBOLS.items():
            f = getattr(L, name)
            f.restype, f.argtypes = res, args
        _lib = L
    return _lib


def _check(rc):
    if rc != XY_OK:
        raise XYError(rc, lib().xy_last_error().decode())


def _host(a, dtype):
    a = np.ascontiguousarray(a, dtype)
    return a, a.ctypes.data_as(C.c_void_p)


def xy_last_error():
    return lib().xy_last_error().decode()


def xy_abi_version():
    return lib().xy_abi_version()


def xy_graph_load(row_ptr, col_idx, colour, stream=None):
    """row_ptr [S][N+1], col_idx [S][nnz] (or concatenated 1-D), colour [S][N] host int32 -> graph handle."""
    row_ptr = np.ascontiguousarray(row_ptr, np.int32)
    colour = np.ascontiguousarray(colour, np.int32)
    if row_ptr.ndim == 1:
        row_ptr, colour = row_ptr[None, :], colour.reshape(1, -1)
    S, N = colour.shape
    col = np.ascontiguousarray(col_idx, np.int32).reshape(-1)
    out = C.c_void_p()
    _check(lib().xy_graph_load(S, N, row_ptr.ctypes.data_as(C.c_void_p),
                               col.ctypes.data_as(C.c_void_p) if col.size else None,
                               colour.ctypes.data_as(C.c_void_p), stream, C.byref(out)))
    return out


def xy_graph_free(g):
    _check(lib().xy_graph_free(g))


def xy_graph_info(g):
    S, N, q, d = C.c_int(), C.c_int(), C.c_int(), C.c_int()
    nnz = C.c_int64()
    _check(lib().xy_graph_info(g, C.byref(S), C.byref(N), C.byref(nnz), C.byref(q), C.byref(d)))
    return dict(S=S.value, N=N.value, nnz_total=nnz.value, q_max=q.value, max_degree=d.value)


def xy_graph_set_coords(g, Lx, Ly, x, y):
    x, xp = _host(x, np.int32)
    y, yp = _host(y, np.int32)
    _check(lib().xy_graph_set_coords(g, Lx, Ly, xp, yp))


def xy_measure_fourier(pt, shape=None):
    """shape = (S, R) to get (G1, G2) of this configuration back as a host array [S][R][2] by temperature."""
    if shape is None:
        _check(lib().xy_measure_fourier(pt, None))
        return None
    out = np.zeros((*shape, 2), np.float64)
    _check(lib().xy_measure_fourier(pt, out.ctypes.data_as(C.c_void_p)))
    return out


def xy_read_fourier_accumulators(pt, shape):
    out = np.empty((*shape, 3), np.float64)
    _check(lib().xy_read_fourier_accumulators(pt, out.ctypes.data_as(C.c_void_p)))
    return out


def xy_random_walk(g, start, n_steps, seed, sample_base=0, stream=None):
    """start [S][n_walkers] host int32 -> hist [S][n_steps+1] int64 (visits of the origin at time t)."""
    start, sp = _host(start, np.int32)
    if start.ndim == 1:
        start = start[None, :]
    hist = np.zeros((start.shape[0], n_steps + 1), np.int64)
    _check(lib().xy_random_walk(g, start.shape[1], sp, n_steps, seed, sample_base, stream, hist.ctypes.data_as(C.c_void_p)))
    return hist


XY_WALK_STATIC_ENTRIES = 65536


def xy_random_walk_static(g, n_walkers, start_dev, n_steps, seed, hist_dev, sample_base=0, stream=None):
    """the walk without any allocation: start_dev / hist_dev = device addresses (int) of caller-owned buffers
    [S][n_walkers] int32 and [S][n_steps+1] int64; S * (n_steps + 1) <= XY_WALK_STATIC_ENTRIES."""
    _check(lib().xy_random_walk_static(g, n_walkers, start_dev, n_steps, seed, sample_base, stream, hist_dev))


def xy_random_walk_kernel_us():
    out = C.c_double()
    _check(lib().xy_random_walk_kernel_us(C.byref(out)))
    return out.value


def xy_set_path(pt, path):
    _check(lib().xy_set_path(pt, path))


def xy_get_path(pt, or_per_sweep=1):
    """(path xy_run would take: 1 = launch per colour class, 2 = cluster per sample; CTAs per cluster)"""
    p, c = C.c_int(), C.c_int()
    _check(lib().xy_get_path(pt, or_per_sweep, C.byref(p), C.byref(c)))
    return p.value, c.value


def xy_get_schedule(pt):
    """(samples per launch group, bytes one group keeps live)"""
    g, b = C.c_int(), C.c_int64()
    _check(lib().xy_get_schedule(pt, C.byref(g), C.byref(b)))
    return g.value, b.value


def xy_pt_create(g, T, seed, width=None, sample_base=0, theta_dev=None, stream=None):
    """theta_dev: device address (int) of a caller-owned [S][N][R] fp32 buffer, e.g. tensor.data_ptr()."""
    T, Tp = _host(T, np.float64)
    wp = None
    if width is not None:
        width, wp = _host(width, np.float64)
    out = C.c_void_p()
    _check(lib().xy_pt_create(g, len(T), Tp, wp, seed, sample_base, theta_dev, stream, C.byref(out)))
    return out


def xy_pt_destroy(pt):
    _check(lib().xy_pt_destroy(pt))


def xy_sweep(pt, n_sweeps=1):
    _check(lib().xy_sweep(pt, n_sweeps))


def xy_sweep_acceptance(pt, shape):
    """one Metropolis sweep + the fraction of accepted proposals [S][R] by temperature; shape = (S, R)"""
    out = np.zeros(shape, np.float64)
    _check(lib().xy_sweep_acceptance(pt, out.ctypes.data_as(C.c_void_p)))
    return out


def xy_overrelax(pt, n_sweeps=1):
    _check(lib().xy_overrelax(pt, n_sweeps))


def xy_pt_swap(pt):
    _check(lib().xy_pt_swap(pt))


def xy_measure(pt, shape=None):
    """shape = (S, R) to get this measurement back as a host array [S][R][3] (E, Mx, My) by temperature."""
    if shape is None:
        _check(lib().xy_measure(pt, None))
        return None
    out = np.zeros((*shape, 3), np.float64)
    _check(lib().xy_measure(pt, out.ctypes.data_as(C.c_void_p)))
    return out


def xy_run(pt, n_cycles, sweeps_per_swap=10, or_per_sweep=1, measure_every=1):
    _check(lib().xy_run(pt, n_cycles, sweeps_per_swap, or_per_sweep, measure_every))


def xy_run_sweeps(pt, n_blocks, sweeps_per_block=10, or_per_sweep=1):
    _check(lib().xy_run_sweeps(pt, n_blocks, sweeps_per_block, or_per_sweep))


def xy_set_schedule(pt, samples_per_group):
    _check(lib().xy_set_schedule(pt, samples_per_group))


def xy_set_tuning(pt, balance=1, pdl=1, l2_persist=1, fuse_measure=1, cta_shape=0):
    _check(lib().xy_set_tuning(pt, balance, pdl, l2_persist, fuse_measure, cta_shape))


def xy_metropolis_colour(pt, colour, sweep):
    _check(lib().xy_metropolis_colour(pt, colour, sweep))


def xy_metor_colour(pt, colour, sweep):
    _check(lib().xy_metor_colour(pt, colour, sweep))


def xy_set_order(pt, order):
    _check(lib().xy_set_order(pt, order))


def xy_overrelax_colour(pt, colour):
    _check(lib().xy_overrelax_colour(pt, colour))


def xy_get_theta(pt, shape, out=None):
    out = np.empty(shape, np.float32) if out is None else out
    _check(lib().xy_get_theta(pt, out.ctypes.data_as(C.c_void_p)))
    return out


def xy_set_theta(pt, theta):
    theta, p = _host(theta, np.float32)
    _check(lib().xy_set_theta(pt, p))


def xy_set_theta_async(pt, theta_pinned):
    """theta_pinned: C-contiguous float32 numpy view of PINNED host memory; the caller keeps it alive and unchanged
    until xy_synchronize."""
    if theta_pinned.dtype != np.float32 or not theta_pinned.flags["C_CONTIGUOUS"]:
        raise ValueError("theta_pinned must be a C-contiguous float32 array")
    _check(lib().xy_set_theta_async(pt, theta_pinned.ctypes.data_as(C.c_void_p)))


def xy_get_labels(pt, shape):
    out = np.empty(shape, np.int32)
    _check(lib().xy_get_labels(pt, out.ctypes.data_as(C.c_void_p)))
    return out


def xy_set_labels(pt, temp_of_slot):
    a, p = _host(temp_of_slot, np.int32)
    _check(lib().xy_set_labels(pt, p))


def xy_get_energy(pt, shape):
    out = np.empty(shape, np.float64)
    _check(lib().xy_get_energy(pt, out.ctypes.data_as(C.c_void_p)))
    return out


def xy_swap_with_decisions(pt, accept):
    a, p = _host(accept, np.uint8)
    _check(lib().xy_swap_with_decisions(pt, p))


def xy_read_accumulators(pt, shape):
    out = np.empty((*shape, XY_NACC), np.float64)
    _check(lib().xy_read_accumulators(pt, out.ctypes.data_as(C.c_void_p)))
    return out


def xy_reset_accumulators(pt):
    _check(lib().xy_reset_accumulators(pt))


def xy_get_counters(pt, shape):
    sw, rd = C.c_uint32(), C.c_uint32()
    att = np.empty(shape, np.int64)
    acc = np.empty(shape, np.int64)
    _check(lib().xy_get_counters(pt, C.byref(sw), C.byref(rd), att.ctypes.data_as(C.c_void_p),
                                 acc.ctypes.data_as(C.c_void_p)))
    return sw.value, rd.value, att, acc


def xy_set_counters(pt, sweep, round_):
    _check(lib().xy_set_counters(pt, sweep, round_))


def xy_theta_device(pt):
    p = C.c_void_p()
    _check(lib().xy_theta_device(pt, C.byref(p)))
    return p.value


def xy_launch_count(pt):
    n = C.c_int64()
    _check(lib().xy_launch_count(pt, C.byref(n)))
    return n.value


def xy_synchronize(pt):
    _check(lib().xy_synchronize(pt))


def xy_l2_bandwidth(nbytes=32 << 20, mode=0, repeats=5, stream=None):
    """GB/s of the L2 read microbenchmark (mode 0 linear stream, 1 random 256-byte rows)."""
    out = C.c_double()
    _check(lib().xy_l2_bandwidth(nbytes, mode, repeats, stream, C.byref(out)))
    return out.value


class Ensemble:
    """Convenience owner of one graph + PT handle; theta lives in a torch tensor on its own torch stream.
    Still marshalling only: every method forwards to the xy_* call of the same name."""

    def __init__(self, row_ptr, col_idx, colour, T, seed, width=None, sample_base=0, device="cuda:0"):
        import torch
        if not torch.cuda.is_available():
            raise XYError(XY_ECUDA, "no CUDA device: this library has no CPU fallback")
        self.torch = torch
        self.device = torch.device(device)
        colour = np.ascontiguousarray(colour, np.int32)
        if colour.ndim == 1:
            colour = colour[None, :]
        self.S, self.N = colour.shape
        self.T = np.ascontiguousarray(T, np.float64)
        self.R = len(self.T)
        with torch.cuda.device(self.device):
            self.stream = torch.cuda.Stream()
            self.theta = torch.empty((self.S, self.N, self.R), dtype=torch.float32, device=self.device)
            self.graph = xy_graph_load(row_ptr, col_idx, colour, self.stream.cuda_stream)
            self.pt = xy_pt_create(self.graph, self.T, seed, width, sample_base, self.theta.data_ptr(),
                                   self.stream.cuda_stream)

    def close(self):
        if getattr(self, "pt", None) is not None:
            xy_pt_destroy(self.pt)
            xy_graph_free(self.graph)
            self.pt = self.graph = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # forwarding
    def sweep(self, n=1): xy_sweep(self.pt, n)
    def sweep_acceptance(self): return xy_sweep_acceptance(self.pt, (self.S, self.R))
    def overrelax(self, n=1): xy_overrelax(self.pt, n)
    def pt_swap(self): xy_pt_swap(self.pt)
    def measure(self, want=False): return xy_measure(self.pt, (self.S, self.R) if want else None)
    def set_coords(self, Lx, Ly, x, y): xy_graph_set_coords(self.graph, Lx, Ly, x, y)
    def measure_fourier(self, want=False): return xy_measure_fourier(self.pt, (self.S, self.R) if want else None)
    def read_fourier_accumulators(self): return xy_read_fourier_accumulators(self.pt, (self.S, self.R))
    def run(self, n_cycles, sweeps_per_swap=10, or_per_sweep=1, measure_every=1):
        xy_run(self.pt, n_cycles, sweeps_per_swap, or_per_sweep, measure_every)
    def run_sweeps(self, n_blocks, sweeps_per_block=10, or_per_sweep=1):
        xy_run_sweeps(self.pt, n_blocks, sweeps_per_block, or_per_sweep)
    def set_schedule(self, g): xy_set_schedule(self.pt, g)
    def get_schedule(self): return xy_get_schedule(self.pt)
    def set_path(self, path): xy_set_path(self.pt, path)
    def get_path(self, or_per_sweep=1): return xy_get_path(self.pt, or_per_sweep)

    def path_name(self, or_per_sweep=1):
        p, c = self.get_path(or_per_sweep)
        return (f"k_cycle: one {c}-CTA cluster per sample, whole cycles per launch" if p == 2
                else "k_phase: one launch per colour class (captured graph, PDL edges)")
    def set_tuning(self, balance=1, pdl=1, l2_persist=1, fuse_measure=1, cta_shape=0):
        xy_set_tuning(self.pt, balance, pdl, l2_persist, fuse_measure, cta_shape)
    def metropolis_colour(self, c, sweep): xy_metropolis_colour(self.pt, c, sweep)
    def overrelax_colour(self, c): xy_overrelax_colour(self.pt, c)
    def metor_colour(self, c, sweep): xy_metor_colour(self.pt, c, sweep)
    def set_order(self, order): xy_set_order(self.pt, order)
    def get_theta(self, out=None): return xy_get_theta(self.pt, (self.S, self.N, self.R), out)
    def set_theta(self, th): xy_set_theta(self.pt, th)
    def set_theta_async(self, th_pinned): xy_set_theta_async(self.pt, th_pinned)
    def get_labels(self): return xy_get_labels(self.pt, (self.S, self.R))
    def set_labels(self, lab): xy_set_labels(self.pt, lab)
    def get_energy(self): return xy_get_energy(self.pt, (self.S, self.R))
    def swap_with_decisions(self, acc): xy_swap_with_decisions(self.pt, acc)
    def read_accumulators(self): return xy_read_accumulators(self.pt, (self.S, self.R))
    def reset_accumulators(self): xy_reset_accumulators(self.pt)
    def get_counters(self): return xy_get_counters(self.pt, (self.S, self.R))
    def set_counters(self, sweep, round_): xy_set_counters(self.pt, sweep, round_)
    def launch_count(self): return xy_launch_count(self.pt)
    def synchronize(self): xy_synchronize(self.pt)
