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
