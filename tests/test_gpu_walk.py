"""-m gpu tests of the random-walk self-return histogram (App. A):
integer work, so the CUDA path (xy_random_walk through the C ABI) must equal the oracle BIT FOR BIT on the same
seeded inputs -- small graphs, Levy graphs with isolated sites, BASELINE config 4's graph at full size; plus the
exact square-lattice return probability and spectral dimension on the GPU alone."""
import numpy as np
import pytest
from scipy.special import comb

import graphs as G
import oracle as O
from paper_1211_3991_b200 import binding as B
from paper_1211_3991_b200 import levy, workloads

pytestmark = pytest.mark.gpu
SEED = 0x3A1CB200


def starts_like_the_paper(g, n_walkers, rng):
    """App. A: rho > 4: the centre of the lattice; rho <= 4: random sites of degree > 2."""
    out = np.zeros((g.S, n_walkers), np.int32)
    for s in range(g.S):
        if g.rho > 4:
            out[s] = int(np.where(g.new_to_old[s] == (g.L // 2) * g.L + g.L // 2)[0][0])
        else:
            deg = np.diff(g.row_ptr[s])
            out[s] = rng.choice(np.where(deg > 2)[0], n_walkers)
    return out


@pytest.mark.parametrize("L,rho,S,W,steps", [(16, 3.5, 3, 1000, 37), (12, 4.5, 2, 257, 64), (24, 2.5, 1, 5000, 200), (8, 3.0, 2, 1, 5),
                                             (16, 3.5, 1, 300, 0)])
def test_walk_bit_exact_small(L, rho, S, W, steps):
    g = levy.build(L, rho, 6, workloads.BASE_SEED, S=S, sample_base=2)
    gh = B.xy_graph_load(g.row_ptr, g.col_idx, g.colour)
    rng = np.random.default_rng(5)
    st = starts_like_the_paper(g, W, rng)
    st[:, 0] = [int(np.argmin(np.diff(g.row_ptr[s]))) for s in range(S)]      # a lowest-degree (possibly isolated) origin too
    h = B.xy_random_walk(gh, st, steps, SEED, sample_base=2)
    for s in range(S):
        assert np.array_equal(h[s], O.random_walk(g.row_ptr[s], g.col_idx[s], st[s], steps, SEED, 2 + s)), s
    assert np.all(h[:, 0] == W)
    with pytest.raises(B.XYError):
        B.xy_random_walk(gh, st + L * L, steps, SEED)
    with pytest.raises(B.XYError):
        B.xy_random_walk(gh, st, 20000, SEED)
    B.xy_graph_free(gh)


def test_walk_square_lattice_closed_form_and_spectral_dimension():
    L, W = 64, 400_000
    gd = G.colour_major(L * L, G.square_lattice_edges(L))
    gh = B.xy_graph_load(gd["row_ptr"], gd["col_idx"], gd["colour"])
    origin = int(np.where(gd["new_to_old"] == (L // 2) * L + L // 2)[0][0])
    h = B.xy_random_walk(gh, np.full((1, W), origin, np.int32), 48, SEED)[0]
    B.xy_graph_free(gh)
    ex = np.array([(comb(t, t // 2) / 2.0 ** t) ** 2 if t % 2 == 0 else 0.0 for t in range(49)])
    assert np.all(h[1::2] == 0)
    sig = np.sqrt(np.maximum(ex * (1 - ex), 1e-12) / W)
    assert np.all(np.abs(h / W - ex) <= 4.5 * sig + 1e-12)
    t = np.arange(8, 49, 2)
    slope = np.polyfit(np.log(t), np.log(h[t] / W), 1)[0]
    assert abs(-2 * slope - 2.0) < 0.1, slope                   # Eq. 11: dbar = 2


def test_walk_full_size_config4_graph_bit_exact():
    """the paper's protocol (4e4 walkers per graph) on BASELINE config 4's L = 512 graphs: every sample bit-exact."""
    w = workloads.CONFIGS[4]
    g = levy.build(w.L, w.rho, w.z, w.seed, S=2)
    gh = B.xy_graph_load(g.row_ptr, g.col_idx, g.colour)
    st = starts_like_the_paper(g, 40_000, np.random.default_rng(9))
    h = B.xy_random_walk(gh, st, 256, SEED)
    B.xy_graph_free(gh)
    for s in range(2):
        assert np.array_equal(h[s], O.random_walk(g.row_ptr[s], g.col_idx[s], st[s], 256, SEED, s))
    assert h[:, 2].min() > 0                                      # some walkers are back after two steps
