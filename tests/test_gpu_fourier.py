"""-m gpu tests of the structure factor at k_min / second-moment correlation length row (
PAPER.md:183-190): the CUDA path (xy_measure_fourier through the C ABI) against the oracle on the same
configurations, element by element; accumulators by temperature; and against exact physics (ring C(r), beta = 0)."""
import numpy as np
import pytest

import closed_forms as CF
import graphs as G
import gpu_util as U
import oracle as O
from paper_1211_3991_b200 import binding as B
from paper_1211_3991_b200 import levy, workloads

pytestmark = pytest.mark.gpu
SEED = 0xF0C1E5B2


def levy_coords(g):
    return (g.new_to_old % g.L).astype(np.int32), (g.new_to_old // g.L).astype(np.int32)


@pytest.mark.parametrize("L,R,S", [(16, 8, 2), (16, 64, 2), (24, 32, 1), (12, 3, 2), (20, 128, 1), (33, 16, 1), (16, 2, 2), (40, 4, 1)])
def test_fourier_matches_oracle(L, R, S):
    g = levy.build(L, 3.5, 6, workloads.BASE_SEED, S=S)
    T = O.geometric_temperatures(R, 1.0, 4.0)
    ens = U.ensemble_from_levy(g, T, SEED)
    with pytest.raises(B.XYError) as e:
        ens.measure_fourier()
    assert e.value.code == B.XY_ESTATE                       # coordinates not set yet
    x, y = levy_coords(g)
    ens.set_coords(L, L, x, y)
    ens.run(2, 5, 1, 1)                                       # labels get permuted
    lab = ens.get_labels()
    out = ens.measure_fourier(want=True)
    th = ens.get_theta()
    for s in range(S):
        G1, G2 = O.fourier(L, L, x[s], y[s], th[s])
        # fast sincos (3.6e-7 abs) on N terms with random signs + 2^-23 quantisation: |dF| <~ 1e-6 sqrt(N); G = |F|^2/N
        tol = 2e-5 * (1.0 + np.maximum(G1, G2))
        assert np.all(np.abs(out[s, lab[s], 0] - G1) <= tol), np.abs(out[s, lab[s], 0] - G1).max()
        assert np.all(np.abs(out[s, lab[s], 1] - G2) <= tol)
    acc = ens.read_fourier_accumulators()
    assert np.all(acc[..., 0] == 1) and np.allclose(acc[..., 1:], out, rtol=1e-12, atol=0)
    out2 = ens.measure_fourier(want=True)
    assert np.array_equal(out, out2)                          # exact integer sums: bit-reproducible
    assert np.allclose(ens.read_fourier_accumulators()[..., 1:], 2 * out, rtol=1e-12)
    ens.reset_accumulators()
    assert np.all(ens.read_fourier_accumulators() == 0)
    with pytest.raises(B.XYError):
        ens.set_coords(L, L, x + L, y)                        # out of range
    ens.close()


@pytest.mark.parametrize("L,R", [(24, 8), (40, 32), (24, 64), (20, 128), (33, 16)])
def test_fourier_bulk_copy_and_cp_async_flavours_give_the_same_bits(L, R):
    """k_fourier2 fills its ring with the TMA engine (cp.async.bulk) when theta is 16-byte aligned and with per-lane
    cp.async copies otherwise: the same rows in the same order, so G1, G2 must be bit-identical -- and equal the oracle's."""
    import torch
    g = levy.build(L, 3.5, 6, workloads.BASE_SEED, S=2)
    T = O.geometric_temperatures(R, 1.0, 4.0)
    x, y = levy_coords(g)
    S, N = g.colour.shape
    rng = np.random.default_rng(L * 1000 + R)
    th = (rng.random((S, N, R)) * 6.28).astype(np.float32)
    outs = []
    for shift in (0, 2):                                     # floats: 0 = 16-byte aligned (bulk copies), 2 = 8 mod 16 (cp.async)
        stream = torch.cuda.Stream()
        buf = torch.empty(S * N * R + 4, dtype=torch.float32, device="cuda:0")
        ptr = buf.data_ptr() + 4 * shift
        assert buf.data_ptr() % 16 == 0
        graph = B.xy_graph_load(g.row_ptr, g.col_idx, g.colour, stream.cuda_stream)
        pt = B.xy_pt_create(graph, T, SEED, None, 0, ptr, stream.cuda_stream)
        B.xy_graph_set_coords(graph, L, L, x, y)
        B.xy_set_theta(pt, th)
        outs.append(B.xy_measure_fourier(pt, (S, R)))
        B.xy_pt_destroy(pt)
        B.xy_graph_free(graph)
    assert np.array_equal(outs[0], outs[1])
    for s in range(S):
        G1, G2 = O.fourier(L, L, x[s], y[s], th[s])
        assert np.all(np.abs(outs[0][s, :, 0] - G1) <= 2e-5 * (1.0 + G1)) and np.all(np.abs(outs[0][s, :, 1] - G2) <= 2e-5 * (1.0 + G2))


def test_fourier_closed_form_configurations_on_gpu():
    L = 16
    g = levy.build(L, 3.5, 6, workloads.BASE_SEED, S=1)
    x, y = levy_coords(g)
    ens = U.ensemble_from_levy(g, np.array([1.0, 2.0]), SEED)
    ens.set_coords(L, L, x, y)
    th = np.zeros((1, L * L, 2), np.float32)
    th[0, :, 0] = 2 * np.pi * x[0] / L                        # plane wave along x: G1 = N/2, G2 = 0
    th[0, :, 1] = 1.25                                        # aligned: both vanish
    ens.set_theta(th)
    out = ens.measure_fourier(want=True)[0]
    assert abs(out[0, 0] - L * L / 2) < 1e-3 and abs(out[0, 1]) < 1e-4
    assert abs(out[1, 0]) < 1e-4 and abs(out[1, 1]) < 1e-4
    ens.close()


def test_gpu_ring_structure_factor_and_xi2():
    """equilibrium on the periodic ring: <G(k)> at k = 2 pi/N and 4 pi/N against the exact C(r); xi_2 from the
    accumulators against the value the exact chi(0), chi(k) give."""
    N = 16
    T = np.array([0.5, 1.0, 2.0])
    gd = G.colour_major(N, G.ring_edges(N))
    S = 8
    ens = U.ensemble_from_graph(gd, T, SEED, S=S)
    x = np.tile(gd["new_to_old"].astype(np.int32), (S, 1))
    ens.set_coords(N, N, x, (2 * x) % N)
    ens.run(30, 10, 1, 1)
    ens.reset_accumulators()
    blocks = []
    prev = np.zeros((S, len(T), 3))
    for _ in range(30):
        for _ in range(40):
            ens.run(1, 10, 1, 1)
            ens.measure_fourier()
        cur = ens.read_fourier_accumulators()
        blocks.append((cur - prev).sum(0))                    # pool the 8 independent copies of the ring
        prev = cur
    blocks = np.array(blocks)
    mean = blocks[..., 1:] / blocks[..., :1]
    m, sg = mean.mean(0), mean.std(0, ddof=1) / np.sqrt(len(mean))
    for t, temp in enumerate(T):
        for col, kidx in ((0, 1), (1, 2)):
            exact = CF.ring_structure_factor(N, 1 / temp, kidx)
            assert abs(m[t, col] - exact) < 4.5 * sg[t, col], (temp, kidx, m[t, col], exact, sg[t, col])
            assert sg[t, col] < 0.03 * exact
    acc = ens.read_accumulators().sum(0)
    chi0 = N * acc[:, 4] / acc[:, 0]
    for t, temp in enumerate(T):
        exact0 = CF.ring_structure_factor(N, 1 / temp, 0)
        exact1 = CF.ring_structure_factor(N, 1 / temp, 1)
        assert abs(chi0[t] - exact0) < 0.03 * exact0
        if exact0 / exact1 - 1.0 > 0.5:      # xi_2 amplifies the relative error of chi(0)/chi(k) - 1: check it where that is O(1)
            assert abs(O.xi2(chi0[t], m[t, 0], N, 2.0) - O.xi2(exact0, exact1, N, 2.0)) < 0.08 * O.xi2(exact0, exact1, N, 2.0)
    ens.close()


def test_gpu_beta_zero_structure_factor_is_one():
    L = 8
    g = levy.build(L, 3.5, 6, workloads.BASE_SEED, S=16)
    x, y = levy_coords(g)
    ens = U.ensemble_from_levy(g, np.array([np.inf, np.inf]), SEED)
    ens.set_coords(L, L, x, y)
    ens.run(3, 10, 1, 1)
    vals = []
    for _ in range(200):
        ens.run(1, 5, 1, 0)
        vals.append(ens.measure_fourier(want=True))
    vals = np.array(vals).reshape(200, -1)
    m, sg = vals.mean(), vals.mean(1).std(ddof=1) / np.sqrt(200)
    assert abs(m - 1.0) < 4.5 * sg and sg < 0.01


def test_fourier_full_size_config4_sampled_slots():
    """BASELINE config 4 at full size: G1, G2 of every slot of two samples against the oracle."""
    w = workloads.CONFIGS[4]
    g = levy.build(w.L, w.rho, w.z, w.seed, S=w.S)
    x, y = levy_coords(g)
    ens = U.ensemble_from_levy(g, w.temperatures(), SEED)
    ens.set_coords(w.L, w.L, x, y)
    ens.run(1, 10, 1, 1)
    lab = ens.get_labels()
    out = ens.measure_fourier(want=True)
    for s in (0, 5):
        th = ens.get_theta()[s]
        G1, G2 = O.fourier(w.L, w.L, x[s], y[s], th)
        tol = 2e-5 * (1.0 + np.maximum(G1, G2))
        assert np.all(np.abs(out[s, lab[s], 0] - G1) <= tol) and np.all(np.abs(out[s, lab[s], 1] - G2) <= tol)
    ens.close()
