"""-m gpu physics validation on the paper's own benchmark limit:
the rho = 0 Levy graph is the Erdos-Renyi graph, where the XY model has a mean-field transition at
the analytic T_c = 1.9361 for z = 4.  The Binder cumulants (Eq. 15, graph-averaged over 32 samples) of
two sizes must cross there.  This exercises the whole CUDA path (builder, coloured Metropolis + over-relaxation,
parallel tempering, fused measurement, accumulators) against a number the paper prints."""
import numpy as np
import pytest

import stats as S
from paper_1211_3991_b200 import binding as B
from paper_1211_3991_b200 import levy, workloads

pytestmark = pytest.mark.gpu
def paper_value(name):
    import os
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")):
        f = line.split()
        if f and f[0] == name:
            return float(f[1])
    raise KeyError(name)


TC_ER_Z4 = paper_value("tc_erdos_renyi_z4")          # 1.9361


def binder(L, T, order):
    g = levy.build(L, 0.0, 4, workloads.BASE_SEED, S=32)
    ens = B.Ensemble(g.row_ptr, g.col_idx, g.colour, T, 0x7C0000 + L)
    ens.set_order(order)
    ens.run(1000, 10, 1, 1)
    ens.reset_accumulators()
    ens.run(2000, 10, 1, 1)
    acc = ens.read_accumulators()
    ens.close()
    m = acc / acc[..., :1]
    return m[..., S.M4_].mean(0) / (m[..., S.M2_] ** 2).mean(0) - 1.0      # Eq. 15 (DESIGN R14, literal reading)


@pytest.mark.parametrize("order", [0, 1])
def test_erdos_renyi_z4_binder_crossing_at_the_analytic_tc(order):
    T = np.linspace(1.70, 2.20, 32)
    u = {L: binder(L, T, order) for L in (32, 64, 128)}
    for L in u:                                                   # ordered side -> 0, disordered side -> 1 (R14)
        assert u[L][0] < 0.1 and u[L][-1] > 0.85
    cross = {}
    for a, b in ((32, 64), (64, 128)):
        d = u[a] - u[b]
        k = np.where(np.sign(d[:-1]) != np.sign(d[1:]))[0]
        k = k[np.argmin(np.abs(T[k] - TC_ER_Z4))]
        cross[(a, b)] = T[k] + (T[k + 1] - T[k]) * d[k] / (d[k] - d[k + 1])
    print(f"\nER z=4 Binder crossings (order {order}): {cross}  analytic T_c = {TC_ER_Z4}")
    assert abs(cross[(64, 128)] - TC_ER_Z4) < 0.03
    assert abs(cross[(32, 64)] - TC_ER_Z4) < 0.06
    assert abs(cross[(64, 128)] - TC_ER_Z4) <= abs(cross[(32, 64)] - TC_ER_Z4) + 0.01     # converging with size


TC_SQUARE = paper_value("tc_square_lattice")         # 0.8929
ETA_KT = paper_value("eta_kt_at_tc")                 # 1/4,    PAPER.md:278 Eq. 27
R_KT = paper_value("r_kt_log")                       # 1/16


def test_square_lattice_kt_susceptibility_exponent_at_the_paper_tc():
    """The paper's own benchmark of its algorithm: on the 2D square lattice (the rho = infinity
    limit, z = 4, two colours) the susceptibility at T_c = 0.8929 scales as chi ~ L^(2 - eta) with
    eta = 1/4 (Eq. 27); eta(T), "numerically interpolating Eq. (27) at different temperatures", grows with T, passes 1/4
    at T_c (the paper's independent estimate T_c = 0.894(5)), and chi stops growing with L in the vortex phase.
    chi = N <m^2> (item (3): <m>^2 is negligible).  L = 32, 64, 128 (the largest is the lattice of the
    paper's Table III); 16 independent copies of each lattice.  Coarse check (R22): the leading power law is
    fitted; Eq. 27's factor (ln L)^(-2r), whose sign differs between the paper (r = 1/16) and the KT literature it cites
    (r = -1/16) and which shifts eta by -+0.03 at these sizes, is reported beside it, not asserted."""
    T = np.sort(np.append(np.linspace(0.70, 1.30, 15), TC_SQUARE))
    k_c = int(np.where(T == TC_SQUARE)[0][0])
    sizes = (32, 64, 128)
    lnchi, err = {}, {}
    for L in sizes:
        w = workloads.square_lattice(L, len(T), T[0], T[-1], 16)
        g = levy.build(w.L, w.rho, w.z, w.seed, S=1)
        assert int(g.n_colours[0]) == 2 and np.all(np.diff(g.row_ptr[0]) == 4)
        ens = B.Ensemble(np.tile(g.row_ptr, (w.S, 1)), np.tile(g.col_idx, (w.S, 1)), np.tile(g.colour, (w.S, 1)), T, 0x2D0000 + L)
        ens.run(2000, 10, 1, 1)
        blocks = []
        for _ in range(20):
            ens.reset_accumulators()
            ens.run(300, 10, 1, 1)
            blocks.append(ens.read_accumulators().sum(0))             # pool the 16 copies of the same lattice
        ens.close()
        est, sig = S.jackknife(np.array(blocks), lambda m: np.log(L * L * m[..., S.M2_]))
        lnchi[L], err[L] = est, sig
    x = np.log(np.array(sizes, np.float64))

    def eta_of(r):              # Eq. 27: ln chi + 2 r ln ln L = (2 - eta) ln L + const
        y = np.array([lnchi[L] + 2 * r * np.log(np.log(L)) for L in sizes])
        return 2.0 - ((x - x.mean())[:, None] * (y - y.mean(0))).sum(0) / ((x - x.mean()) ** 2).sum()

    eta = eta_of(0.0)
    print("\nsquare lattice: T        " + " ".join(f"{t:6.3f}" for t in T))
    print("                eta(T)   " + " ".join(f"{e:6.3f}" for e in eta))
    print(f"eta at the paper's T_c = {TC_SQUARE}: {eta[k_c]:.4f} (paper / KT theory: {ETA_KT}); with Eq. 27's log factor, r = +1/16: "
          f"{eta_of(R_KT)[k_c]:.4f}, r = -1/16: {eta_of(-R_KT)[k_c]:.4f}; max jackknife sigma of ln chi {max(e.max() for e in err.values()):.1e}")
    assert abs(eta[k_c] - ETA_KT) < 0.03
    assert np.all(np.diff(eta) > -0.05) and np.all(np.diff(eta[k_c - 1:k_c + 5]) > 0)      # eta grows with T (noise 0.02 below T_c; 2 = saturation)
    assert eta[0] < 0.20 and eta[-1] > 1.0               # spin-wave phase below, saturating chi above
    # the temperature at which eta = 1/4 (the paper's "independent estimate" T_c = 0.894(5))
    k = int(np.where((eta[:-1] < ETA_KT) & (eta[1:] >= ETA_KT))[0][0])
    t_eta = T[k] + (T[k + 1] - T[k]) * (ETA_KT - eta[k]) / (eta[k + 1] - eta[k])
    print(f"T(eta = 1/4) = {t_eta:.4f}")
    assert abs(t_eta - TC_SQUARE) < 0.03
