"""The PT-cycle protocol written out with the oracle's single-step primitives, so that a test can
watch the decision margins while it runs.  tests/test_oracle_equilibrium.py checks that this loop is bit-identical to
orc_run_order (the oracle's own loop), so it adds no second definition of the protocol -- only visibility."""
import numpy as np

import oracle as O


def run_with_margins(rp, ci, cp, T, seed, n_cycles, sps, orps, me, order=0, sample=0, mutate=None, theta0=None):
    """Returns a list (one entry per cycle) of dict(theta, temp_of_slot, acc, min_margin, min_swap_margin): the state after
    the cycle and the smallest Metropolis / swap decision margin seen SO FAR.  mutate = "or_first_last_colour" runs a
    deliberately wrong order (over-relaxation before Metropolis on the last colour) for the tests' own sensitivity check.
    theta0 [N][R]: the initial angles (default: the library's Philox initialisation)."""
    N, R, Q = len(rp) - 1, len(T), len(cp) - 1
    th = O.init_theta(N, R, seed, sample) if theta0 is None else np.array(theta0, np.float32, copy=True)
    tos = np.arange(R, dtype=np.int32)
    sot = np.arange(R, dtype=np.int32)
    acc = np.zeros((R, O.NACC))
    beta_f, w_f = O.temperature_params(T)
    sites = [np.arange(cp[c], cp[c + 1], dtype=np.int32) for c in range(Q)]
    sweep = rnd = 0
    mm = ms = np.inf
    out = []

    def met(c):
        nonlocal mm
        if len(sites[c]) == 0:
            return
        m, _ = O.metropolis_sites(rp, ci, th, sites[c], beta_f[tos], w_f[tos], seed, sweep, sample, want_margin=True)
        mm = min(mm, float(m.min()))

    for _ in range(n_cycles):
        for _k in range(sps):
            sweep += 1
            if order == 0:
                if mutate == "or_first_last_colour":
                    for c in range(Q - 1):
                        met(c)
                    O.overrelax_sites(rp, ci, th, sites[Q - 1])
                    met(Q - 1)
                    for c in range(Q - 1):
                        O.overrelax_sites(rp, ci, th, sites[c])
                else:
                    for c in range(Q):
                        met(c)
                    for _o in range(orps):
                        for c in range(Q):
                            O.overrelax_sites(rp, ci, th, sites[c])
            else:
                for c in range(Q):
                    met(c)
                    O.overrelax_sites(rp, ci, th, sites[c])
            if me > 0 and sweep % me == 0:
                E, Mx, My = O.measure(rp, ci, th)
                O.accumulate(N, E, Mx, My, tos, acc)
        E, _, _ = O.measure(rp, ci, th)
        _, mar = O.pt_swap(T, E, sot, tos, seed, rnd, sample)
        rnd += 1
        ms = min(ms, float(mar.min()))
        out.append(dict(theta=th.copy(), temp_of_slot=tos.copy(), acc=acc.copy(), min_margin=mm, min_swap_margin=ms))
    return out
