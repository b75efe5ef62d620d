"""Helpers of the -m gpu parity tests: build an Ensemble for a workload and compare single-colour steps
of the CUDA path with the oracle applied to the SAME pre-state (lockstep)."""
import numpy as np

import oracle as O
from paper_1211_3991_b200 import binding as B
from paper_1211_3991_b200 import levy

TWO_PI = 2.0 * np.pi
TOL = 1e-5          # rad, BASELINE.json north_star
BAND = 1e-5         # acceptance-threshold band, BASELINE.json north_star


def circ(a, b):
    d = np.abs(a.astype(np.float64) - b.astype(np.float64)) % TWO_PI
    return np.minimum(d, TWO_PI - d)


def ensemble_from_levy(g, T, seed, sample_base=0, width=None):
    return B.Ensemble(g.row_ptr, g.col_idx, g.colour, T, seed, width=width, sample_base=sample_base)


def ensemble_from_graph(gd, T, seed, S=1, sample_base=0):
    """gd: tests/graphs.py colour_major dict; replicated S times as S samples."""
    rp = np.tile(gd["row_ptr"], (S, 1)); ci = np.tile(gd["col_idx"], (S, 1)); col = np.tile(gd["colour"], (S, 1))
    return B.Ensemble(rp, ci, col, T, seed, sample_base=sample_base)


class _Theta:
    """theta of the ensemble on the host: the whole state (xy_get_theta), or -- for the full-size tests, where the state
    is hundreds of MB -- only the samples asked for, read from the torch tensor the Ensemble owns (device memory is torch's
    job; the stream is synchronised first)."""

    def __init__(self, ens, samples):
        if samples is None:
            self.full, self.part = ens.get_theta(), None
        else:
            ens.synchronize()
            self.full, self.part = None, {s: ens.theta[s].cpu().numpy() for s in samples}

    def __getitem__(self, s):
        return self.full[s] if self.part is None else self.part[s]


def read_theta(ens, samples=None, sparse=False):
    return _Theta(ens, samples if sparse else None)


def slot_params(T, labels_s):
    beta_f, w_f = O.temperature_params(T)
    return beta_f[labels_s], w_f[labels_s]


def lockstep_metropolis(ens, graphs, T, seed, colour, sweep, samples=None, site_subset=None, sample_base=0, rng=None,
                        sparse=False):
    """Run Metropolis on one colour class on the GPU and on the oracle from the same pre-state.
    graphs: list of (row_ptr, col_idx, class_ptr) per sample.  Returns a dict of counts; raises on mismatch."""
    pre = read_theta(ens, samples, sparse)
    labels = ens.get_labels()
    ens.metropolis_colour(colour, sweep)
    post = read_theta(ens, samples, sparse)
    stats = dict(updates=0, near=0, bad=0, maxerr=0.0, accepted=0, disagree_near=0)
    for s in (range(ens.S) if samples is None else samples):
        rp, ci, cp = graphs[s]
        lo, hi = (int(cp[colour]), int(cp[colour + 1])) if colour + 1 < len(cp) else (0, 0)
        # everything outside the class must be untouched, bit for bit
        assert np.array_equal(post[s][:lo], pre[s][:lo]) and np.array_equal(post[s][hi:], pre[s][hi:])
        sites = np.arange(lo, hi, dtype=np.int32)
        if site_subset is not None and len(sites) > site_subset:
            sites = np.sort(rng.choice(sites, site_subset, replace=False)).astype(np.int32)
        if len(sites) == 0:
            continue
        bs, ws = slot_params(T, labels[s])
        ref = pre[s].copy()
        margin, acc = O.metropolis_sites(rp, ci, ref, sites, bs, ws, seed, sweep, sample_base + s, want_margin=True)
        err = circ(post[s][sites], ref[sites])
        near = margin < BAND
        stats["updates"] += err.size
        stats["near"] += int(near.sum())
        stats["accepted"] += int(acc.sum())
        stats["disagree_near"] += int(((err > TOL) & near).sum())
        bad = (err > TOL) & ~near
        stats["bad"] += int(bad.sum())
        if (~near).any():
            stats["maxerr"] = max(stats["maxerr"], float(err[~near].max()))
    return stats


def lockstep_overrelax(ens, graphs, colour, samples=None, site_subset=None, rng=None, sparse=False):
    pre = read_theta(ens, samples, sparse)
    ens.overrelax_colour(colour)
    post = read_theta(ens, samples, sparse)
    stats = dict(updates=0, illcond=0, bad=0, maxerr_scaled=0.0, maxerr_wellcond=0.0)
    for s in (range(ens.S) if samples is None else samples):
        rp, ci, cp = graphs[s]
        lo, hi = (int(cp[colour]), int(cp[colour + 1])) if colour + 1 < len(cp) else (0, 0)
        assert np.array_equal(post[s][:lo], pre[s][:lo]) and np.array_equal(post[s][hi:], pre[s][hi:])
        sites = np.arange(lo, hi, dtype=np.int32)
        if site_subset is not None and len(sites) > site_subset:
            sites = np.sort(rng.choice(sites, site_subset, replace=False)).astype(np.int32)
        if len(sites) == 0:
            continue
        ref = pre[s].copy()
        hn = O.overrelax_sites(rp, ci, ref, sites, want_hnorm=True)
        err = circ(post[s][sites], ref[sites])
        scaled = err * np.minimum(1.0, hn)
        stats["updates"] += err.size
        stats["illcond"] += int(((err > TOL) & (scaled <= TOL)).sum())     # pass only through the |h| factor (R7)
        stats["bad"] += int((scaled > TOL).sum())
        stats["maxerr_scaled"] = max(stats["maxerr_scaled"], float(scaled.max()))
        well = hn >= 1.0
        if well.any():
            stats["maxerr_wellcond"] = max(stats["maxerr_wellcond"], float(err[well].max()))
    return stats


def graphs_of_levy(g):
    return [(g.row_ptr[s], g.col_idx[s], g.class_ptr(s)) for s in range(g.S)]


def lockstep_metor(ens, graphs, T, seed, colour, sweep, samples=None, site_subset=None, sample_base=0, rng=None,
                   sparse=False):
    """interleaved order: Metropolis then over-relaxation of one colour class in one launch, against the oracle's
    two calls from the same pre-state.  Sites whose Metropolis decision is near threshold (R6) are excluded and
    counted; the rest must satisfy the |h|-weighted over-relaxation bar (R7)."""
    pre = read_theta(ens, samples, sparse)
    labels = ens.get_labels()
    ens.metor_colour(colour, sweep)
    post = read_theta(ens, samples, sparse)
    stats = dict(updates=0, near=0, bad=0, illcond=0, accepted=0)
    for s in (range(ens.S) if samples is None else samples):
        rp, ci, cp = graphs[s]
        lo, hi = (int(cp[colour]), int(cp[colour + 1])) if colour + 1 < len(cp) else (0, 0)
        assert np.array_equal(post[s][:lo], pre[s][:lo]) and np.array_equal(post[s][hi:], pre[s][hi:])
        sites = np.arange(lo, hi, dtype=np.int32)
        if site_subset is not None and len(sites) > site_subset:
            sites = np.sort(rng.choice(sites, site_subset, replace=False)).astype(np.int32)
        if len(sites) == 0:
            continue
        bs, ws = slot_params(T, labels[s])
        ref = pre[s].copy()
        margin, acc = O.metropolis_sites(rp, ci, ref, sites, bs, ws, seed, sweep, sample_base + s, want_margin=True)
        hn = O.overrelax_sites(rp, ci, ref, sites, want_hnorm=True)
        err = circ(post[s][sites], ref[sites])
        scaled = err * np.minimum(1.0, hn)
        near = margin < BAND
        stats["updates"] += err.size
        stats["near"] += int(near.sum())
        stats["accepted"] += int(acc.sum())
        stats["illcond"] += int(((err > TOL) & (scaled <= TOL) & ~near).sum())
        stats["bad"] += int(((scaled > TOL) & ~near).sum())
    return stats
