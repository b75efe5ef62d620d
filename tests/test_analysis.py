"""Host-side analysis helpers (paper_1211_3991_b200/analysis.py): the observables of Eq. 13-18 from accumulators,
checked on accumulators built from explicit samples; and (gpu) the paper's exponentially growing windows."""
import numpy as np
import pytest

import oracle as O
from paper_1211_3991_b200 import analysis as A


def test_observables_from_explicit_samples():
    rng = np.random.default_rng(0)
    N, R, n = 50, 3, 400
    T = np.array([0.8, 1.3, 2.1])
    E = rng.normal(-60, 5, (n, R)); mx = rng.normal(0.3, 0.1, (n, R)); my = rng.normal(-0.1, 0.1, (n, R))
    g1 = rng.random((n, R)) + 0.5; g2 = rng.random((n, R)) + 0.5
    m2 = mx ** 2 + my ** 2
    acc = np.stack([np.full(R, n), E.sum(0), (E ** 2).sum(0), np.sqrt(m2).sum(0), m2.sum(0), (m2 ** 2).sum(0), mx.sum(0), my.sum(0)], axis=-1)
    acc_k = np.stack([np.full(R, n), g1.sum(0), g2.sum(0)], axis=-1)
    o = A.observables(acc, N, T, acc_k, L=16, psi=2.0)
    assert np.allclose(o["e"], E.mean(0) / N) and np.allclose(o["c"], E.var(0) / (N * T ** 2))
    assert np.allclose(o["absm"], np.sqrt(m2).mean(0)) and np.allclose(o["u4"], (m2 ** 2).mean(0) / m2.mean(0) ** 2 - 1)
    assert np.allclose(o["chi"], N * (m2.mean(0) - mx.mean(0) ** 2 - my.mean(0) ** 2))
    chik = 0.5 * (g1.mean(0) + g2.mean(0))
    assert np.allclose(o["chik"], chik) and np.allclose(o["chi0"], N * m2.mean(0))
    for r in range(R):                                            # Eq. 17 against the oracle's formula
        assert abs(o["xi2"][r] - O.xi2(N * m2.mean(0)[r], chik[r], 16, 2.0)) < 1e-12
    accS = np.stack([acc, acc * 1.0, acc])                        # three identical "samples"
    assert np.allclose(A.binder_graph_average(accS), o["u4"])


@pytest.mark.gpu
def test_log_windows_on_gpu_are_consistent_once_equilibrated():
    import gpu_util as U
    from paper_1211_3991_b200 import levy, workloads
    w = workloads.CONFIGS[0]
    g = levy.build(w.L, w.rho, w.z, w.seed, S=4)
    ens = U.ensemble_from_levy(g, w.temperatures(), 0x106)
    lat = g.new_to_old
    ens.set_coords(w.L, w.L, (lat % w.L).astype(np.int32), (lat // w.L).astype(np.int32))
    win = A.run_log_windows(ens, 4, 9, fourier=True)
    assert [x["cycles"] for x in win] == [16, 32, 64, 128, 256, 512]
    for x in win:
        assert np.all(x["acc"][..., 0] == x["cycles"] * 10) and np.all(x["acc_k"][..., 0] == x["cycles"])
    ok, worst = A.windows_consistent(win, w.N, w.temperatures(), rtol=0.03, atol=5e-3)
    assert ok, worst
    o = A.observables(win[-1]["acc"], w.N, w.temperatures(), win[-1]["acc_k"], L=w.L)
    assert np.all(np.diff(o["e"].mean(0)) > 0)                    # energy rises with temperature
    assert o["absm"].mean(0)[0] > 0.7 and o["absm"].mean(0)[-1] < 0.2
    assert np.all(o["xi2"] > 0) and o["xi2"].mean(0)[0] > o["xi2"].mean(0)[-1]     # longer correlations when ordered
    ens.close()
