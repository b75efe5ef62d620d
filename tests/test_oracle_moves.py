"""Pins for the oracle's single-step rules: measure, Metropolis, over-relaxation, PT swap
(SURVEY.md 8(c) P7-P9).  Each test would fail on a dropped term, a wrong sign or a transposed index."""
import numpy as np
import pytest

import graphs as G
import oracle as O

SEED = 0xC0FFEE
TWO_PI = 2 * np.pi


def _levy(L=8, rho=3.5, z=6, sample=0):
    edges, _ = O.levy_edges(L, rho, z, 0x12113991, sample)
    return G.colour_major(L * L, [tuple(e) for e in edges])


def circ(a, b):
    d = np.abs(a.astype(np.float64) - b.astype(np.float64)) % TWO_PI
    return np.minimum(d, TWO_PI - d)


def test_measure_matches_dense_definition():
    g = _levy()
    th = O.init_theta(g["N"], 5, SEED, 0)
    E, Mx, My = O.measure(g["row_ptr"], g["col_idx"], th)
    E2, Mx2, My2 = G.dense_energy_magnetisation(g["N"], g["edges"], th)
    assert np.allclose(E, E2, rtol=0, atol=1e-10) and np.allclose(Mx, Mx2, atol=1e-10) and np.allclose(My, My2, atol=1e-10)
    # aligned spins: E = -E_b, |M| = N
    th[:] = 1.234
    E, Mx, My = O.measure(g["row_ptr"], g["col_idx"], th)
    assert np.allclose(E, -len(g["edges"])) and np.allclose(np.hypot(Mx, My), g["N"])


def test_measure_two_site_signs():
    rp, ci = G.csr_from_edges(2, [(0, 1)])
    th = np.array([[0.0, 0.0, 0.5], [np.pi, np.pi / 2, 0.5]], np.float32)
    E, Mx, My = O.measure(rp, ci, th)
    assert np.allclose(E, [1.0, 0.0, -1.0], atol=1e-6)          # antiparallel +1, orthogonal 0, parallel -1
    assert np.allclose(Mx, [0.0, 1.0, 2 * np.cos(0.5)], atol=1e-6) and np.allclose(My, [0.0, 1.0, 2 * np.sin(0.5)], atol=1e-6)


def test_metropolis_delta_e_is_total_energy_difference():
    """for every accepted single-site move, exp(-beta dE) with dE = E(after)-E(before) from orc_measure
    reproduces the recorded acceptance margin; rejected moves leave theta bit-identical; accepted moves
    equal wrap(fp32(theta + w(u1-1/2)))."""
    g = _levy()
    R = 6
    T = O.geometric_temperatures(R, 0.7, 3.0)
    beta, w = O.temperature_params(T)
    th = O.init_theta(g["N"], R, SEED, 0)
    n_acc = n_rej = 0
    for site in [0, 5, 17, 40, 63]:
        before = th.copy()
        E0, _, _ = O.measure(g["row_ptr"], g["col_idx"], before)
        margin, acc = O.metropolis_sites(g["row_ptr"], g["col_idx"], th, [site], beta, w, SEED, 3, 0, want_margin=True)
        assert np.array_equal(np.delete(th, site, 0), np.delete(before, site, 0))     # only that site moved
        for r in range(R):
            u1, u2 = O.slot_uniforms(SEED, 1, site, 3, 0, r)
            prop = np.float32(before[site, r] + np.float32(w[r] * np.float32(np.float32(u1) - np.float32(0.5))))
            trial = before.copy(); trial[site, r] = prop
            E1, _, _ = O.measure(g["row_ptr"], g["col_idx"], trial)
            p = np.exp(-float(beta[r]) * (E1[r] - E0[r]))
            assert abs(margin[0, r] - abs(u2 - min(1.0, p))) < 1e-9
            assert bool(acc[0, r]) == (u2 < p)
            if acc[0, r]:
                wrapped = prop - np.float32(6.2831855) if prop >= np.float32(6.2831855) else (prop + np.float32(6.2831855) if prop < 0 else prop)
                assert th[site, r] == np.float32(wrapped)
                n_acc += 1
            else:
                assert th[site, r] == before[site, r]
                n_rej += 1
    assert n_acc > 3 and n_rej > 3


def test_metropolis_beta_zero_accepts_everything_and_isolated_site():
    g = _levy()
    R = 4
    th = O.init_theta(g["N"], R, SEED, 0)
    sites = np.arange(g["class_ptr"][0], g["class_ptr"][1], dtype=np.int32)
    _, acc = O.metropolis_sites(g["row_ptr"], g["col_idx"], th, sites, np.zeros(R, np.float32),
                                np.full(R, 6.2831855, np.float32), SEED, 1, 0, want_margin=True)
    assert acc.all()
    # isolated site (degree 0): dE = 0, always accepted (DESIGN R3)
    rp = np.array([0, 0, 1, 2], np.int32); ci = np.array([2, 1], np.int32)
    th = O.init_theta(3, R, SEED, 0)
    _, acc = O.metropolis_sites(rp, ci, th, [0], np.full(R, 5.0, np.float32), np.ones(R, np.float32), SEED, 1, 0, True)
    assert acc.all()


def test_metropolis_wrap_keeps_range():
    g = _levy()
    R = 4
    T = np.array([2.0, 3.0, 4.0, 50.0]); beta, w = O.temperature_params(T)
    assert np.allclose(w, 2 * np.pi, rtol=1e-6)                     # w = 2 pi min(1, T/2)
    th = O.init_theta(g["N"], R, SEED, 0)
    allsites = np.arange(g["N"], dtype=np.int32)
    for sweep in range(1, 30):
        for c in range(len(g["class_ptr"]) - 1):
            O.metropolis_sites(g["row_ptr"], g["col_idx"], th, allsites[g["class_ptr"][c]:g["class_ptr"][c + 1]], beta, w, SEED, sweep, 0)
        assert th.min() >= 0.0 and th.max() <= np.float32(6.2831855)


def test_proposal_width_rule():
    T = np.array([0.5, 1.0, 1.999, 2.0, 3.7])
    beta, w = O.temperature_params(T)
    assert np.array_equal(beta, (1.0 / T).astype(np.float32))
    assert np.array_equal(w, (2 * np.pi * np.minimum(1.0, T / 2)).astype(np.float32))
    Tg = O.geometric_temperatures(8, 1.0, 4.0)
    assert np.allclose(Tg, 1.0 * 4.0 ** (np.arange(8) / 7), rtol=1e-15) and Tg[0] == 1.0 and abs(Tg[-1] - 4.0) < 1e-14


def test_overrelax_conserves_energy_is_involution_and_reflects():
    g = _levy()
    R = 5
    th = O.init_theta(g["N"], R, SEED, 0)
    allsites = np.arange(g["N"], dtype=np.int32)
    E0, _, _ = O.measure(g["row_ptr"], g["col_idx"], th)
    moved = 0.0
    for c in range(len(g["class_ptr"]) - 1):
        cls = allsites[g["class_ptr"][c]:g["class_ptr"][c + 1]]
        before = th.copy()
        hn = O.overrelax_sites(g["row_ptr"], g["col_idx"], th, cls, want_hnorm=True)
        moved += circ(th, before).sum()
        # reflection about the local field: (theta' + theta)/2 == phi (mod pi)
        th64 = before.astype(np.float64)
        for k, i in enumerate(cls[:10]):
            nb = g["col_idx"][g["row_ptr"][i]:g["row_ptr"][i + 1]]
            hx = np.cos(th64[nb]).sum(0); hy = np.sin(th64[nb]).sum(0)
            assert np.allclose(hn[k], np.hypot(hx, hy), atol=1e-12)
            phi = np.arctan2(hy, hx)
            resid = np.angle(np.exp(1j * (th[i].astype(np.float64) + th64[i] - 2 * phi)))
            assert np.all(np.abs(resid) < 1e-6 / np.minimum(1.0, np.maximum(hn[k], 1e-3)))
        # involution: a second reflection of the same class restores the angles
        again = th.copy()
        O.overrelax_sites(g["row_ptr"], g["col_idx"], again, cls)
        assert circ(again, before).max() < 2e-6
    E1, _, _ = O.measure(g["row_ptr"], g["col_idx"], th)
    assert moved > 10.0
    assert np.all(np.abs(E1 - E0) < 1e-6 * g["N"])


def test_overrelax_degree_zero_is_noop_and_two_site_value():
    rp = np.array([0, 0, 1, 2], np.int32); ci = np.array([2, 1], np.int32)
    th = np.array([[1.0], [0.3], [2.0]], np.float32)
    O.overrelax_sites(rp, ci, th, [0])
    assert th[0, 0] == np.float32(1.0)
    O.overrelax_sites(rp, ci, th, [1])                       # h along theta_2 = 2.0 -> theta' = 4.0 - 0.3
    assert abs(th[1, 0] - 3.7) < 1e-6
    th = np.array([[0.1], [6.0], [0.2]], np.float32)
    O.overrelax_sites(rp, ci, th, [1])                       # 0.4 - 6.0 + 2 pi
    assert abs(th[1, 0] - (0.4 - 6.0 + TWO_PI)) < 1e-6


def test_pt_swap_rule_and_permutation():
    R = 6
    T = O.geometric_temperatures(R, 1.0, 4.0)
    rng = np.random.default_rng(5)
    sot = np.arange(R, dtype=np.int32); tos = np.arange(R, dtype=np.int32)
    acc_count = np.zeros(R); att = np.zeros(R); p_sum = np.zeros(R)
    for rnd in range(4000):
        E = rng.normal(0, 3, R)
        before = sot.copy()
        dec, mar = O.pt_swap(T, E, sot, tos, SEED, rnd, 2)
        for t in range(rnd & 1, R - 1, 2):
            a, b = before[t], before[t + 1]
            p = min(1.0, np.exp((1 / T[t] - 1 / T[t + 1]) * (E[a] - E[b])))
            x = O.philox4x32_10([t, rnd, 2 << 16, 2], [SEED & 0xFFFFFFFF, SEED >> 32])
            u = O.u01(x[0])
            assert bool(dec[t]) == (u < np.exp((1 / T[t] - 1 / T[t + 1]) * (E[a] - E[b])))
            assert abs(mar[t] - abs(u - p)) < 1e-12
            att[t] += 1; acc_count[t] += dec[t]; p_sum[t] += p
            if dec[t]:
                assert sot[t] == b and sot[t + 1] == a
            else:
                assert sot[t] == a and sot[t + 1] == b
        for t in range(1 - (rnd & 1), R - 1, 2):                # untouched pairs of the other parity
            pass
        assert np.array_equal(sot[tos], np.arange(R)) and np.array_equal(tos[sot], np.arange(R))
    # acceptance frequency == mean of min(1, exp(dbeta dE)) (north_star PT pin)
    for t in range(R - 1):
        assert att[t] == 2000
        assert abs(acc_count[t] - p_sum[t]) < 5 * np.sqrt(att[t] * 0.25)


def test_pt_swap_lower_energy_moves_to_colder_always():
    # slot a at the colder T has the higher energy: (beta_t - beta_t+1)(E_a - E_b) > 0 -> always accept
    T = np.array([1.0, 2.0]); sot = np.array([0, 1], np.int32); tos = np.array([0, 1], np.int32)
    dec, _ = O.pt_swap(T, np.array([5.0, -5.0]), sot, tos, SEED, 0, 0)
    assert dec[0] == 1 and list(sot) == [1, 0] and list(tos) == [1, 0]
    # forced decisions path
    dec, _ = O.pt_swap(T, np.array([5.0, -5.0]), sot, tos, SEED, 2, 0, decisions_in=np.array([0, 0], np.uint8))
    assert dec[0] == 0 and list(sot) == [1, 0]
    # odd round with R=2 attempts nothing
    dec, mar = O.pt_swap(T, np.array([5.0, -5.0]), sot, tos, SEED, 1, 0)
    assert not dec.any() and np.isinf(mar).all()


def test_accumulate_files_under_temperature():
    acc = np.zeros((3, O.NACC))
    O.accumulate(4, np.array([1.0, 2.0, 3.0]), np.array([4.0, 0.0, 2.0]), np.array([0.0, 2.0, 0.0]),
                 np.array([2, 0, 1], np.int32), acc)
    assert list(acc[:, 1]) == [2.0, 3.0, 1.0] and list(acc[:, 2]) == [4.0, 9.0, 1.0]
    assert np.allclose(acc[:, 3], [0.5, 0.5, 1.0]) and np.allclose(acc[:, 4], [0.25, 0.25, 1.0]) and np.allclose(acc[:, 5], [0.0625, 0.0625, 1.0])
    assert np.allclose(acc[:, 6], [0.0, 0.5, 1.0]) and np.allclose(acc[:, 7], [0.5, 0.0, 0.0]) and np.all(acc[:, 0] == 1)
