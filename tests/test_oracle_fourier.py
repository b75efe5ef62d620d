"""Pins of the oracle's structure factor at k_min and second-moment correlation length (
PAPER.md:183-190 Eq. 17-18): numpy's FFT on the lattice field, configurations with closed forms, the
Ornstein-Zernike identity that defines xi_2, beta = 0, and the exact C(r) of the periodic ring."""
import numpy as np

import closed_forms as CF
import graphs as G
import oracle as O
import stats as S

SEED = 0xF0C1E5


def lattice_coords(L):
    i = np.arange(L * L, dtype=np.int32)
    return i % L, i // L


def test_fourier_matches_numpy_fft_on_a_random_configuration():
    L, R = 12, 3
    rng = np.random.default_rng(1)
    th = (rng.random((L * L, R)) * 2 * np.pi).astype(np.float32)
    perm = rng.permutation(L * L)                      # site numbering is arbitrary (colour-major in the product)
    x, y = lattice_coords(L)
    G1, G2 = O.fourier(L, L, x[perm], y[perm], th)
    for r in range(R):
        field = np.zeros((L, L), np.complex128)       # [y][x], complex spin cos + i sin would mix components: do both
        c = np.zeros((L, L)); s = np.zeros((L, L))
        c[y[perm], x[perm]] = np.cos(th[:, r].astype(np.float64)); s[y[perm], x[perm]] = np.sin(th[:, r].astype(np.float64))
        Fc, Fs = np.fft.fft2(c), np.fft.fft2(s)
        # numpy's FFT uses exp(-i k r); |F|^2 is the same for +k and -k of a real field
        assert abs(G1[r] - (abs(Fc[0, 1]) ** 2 + abs(Fs[0, 1]) ** 2) / L ** 2) < 1e-9
        assert abs(G2[r] - (abs(Fc[1, 0]) ** 2 + abs(Fs[1, 0]) ** 2) / L ** 2) < 1e-9


def test_fourier_closed_form_configurations():
    L = 8
    N = L * L
    x, y = lattice_coords(L)
    # aligned spins: the k != 0 modes vanish (sum of the roots of unity)
    th = np.full((N, 2), 1.2345, np.float32)
    G1, G2 = O.fourier(L, L, x, y, th)
    assert np.all(np.abs(G1) < 1e-9) and np.all(np.abs(G2) < 1e-9)
    # plane wave theta = 2 pi x / L: S = (cos kx, sin kx) -> F_c(k1) = N/2, F_s(k1) = i N/2 -> G1 = N/2; G2 = 0
    th = np.stack([2 * np.pi * x / L, 2 * np.pi * y / L], axis=1).astype(np.float32)
    G1, G2 = O.fourier(L, L, x, y, th)
    assert abs(G1[0] - N / 2) < 1e-4 and abs(G2[0]) < 1e-4          # fp32 angles: 1e-7 relative
    assert abs(G2[1] - N / 2) < 1e-4 and abs(G1[1]) < 1e-4
    # a single flipped spin in an aligned background: F(k) = -2 S exp(i k r0) -> G = 4 / N
    th = np.zeros((N, 1), np.float32); th[19, 0] = np.float32(np.pi)
    G1, G2 = O.fourier(L, L, x, y, th)
    assert abs(G1[0] - 4 / N) < 1e-6 and abs(G2[0] - 4 / N) < 1e-6


def test_xi2_is_the_ornstein_zernike_length():
    """Eq. 17 with psi = 2 inverts chi(k) = chi(0) / (1 + xi^2 4 sin^2(k/2)) exactly."""
    for L in (16, 64, 384):
        for xi in (0.5, 3.0, 40.0):
            chi0 = 7.0
            chik = chi0 / (1 + xi ** 2 * 4 * np.sin(np.pi / L) ** 2)
            assert abs(O.xi2(chi0, chik, L, 2.0) - xi) < 1e-9 * xi
    # psi = rho - d in the long-range regime
    assert abs(O.xi2(3.0, 1.0, 32, 1.5) - 2.0 ** (1 / 1.5) / (2 * np.sin(np.pi / 32))) < 1e-12


def fourier_blocks(g, T, coords, n_blocks, cycles_per_block, burn):
    Lx, Ly, x, y = coords
    ch = O.Chain(g["row_ptr"], g["col_idx"], g["class_ptr"], T, SEED)
    ch.run(burn, 10, 1, 0)
    out = []
    for _ in range(n_blocks):
        acc = np.zeros((len(T), 2))
        for _ in range(cycles_per_block):
            ch.run(1, 10, 1, 0)
            G1, G2 = O.fourier(Lx, Ly, x, y, ch.theta)
            acc[ch.temp_of_slot, 0] += G1; acc[ch.temp_of_slot, 1] += G2
        out.append(acc / cycles_per_block)
    return np.array(out)


def mean_sigma(blocks):
    return blocks.mean(0), blocks.std(0, ddof=1) / np.sqrt(len(blocks))


def test_ring_structure_factor_closed_form():
    """Metropolis + OR + PT on the periodic ring: <G(k)> at k = 2 pi / N and 4 pi / N against the exact C(r)."""
    N = 16
    T = np.array([0.5, 1.0, 2.0])
    g = G.colour_major(N, G.ring_edges(N))
    x = g["new_to_old"].astype(np.int32)
    # second "direction": the same ring with doubled momentum (y = 2 x mod N, Ly = N) -> k_index 2
    y = ((2 * x) % N).astype(np.int32)
    blocks = fourier_blocks(g, T, (N, N, x, y), 30, 60, 30)
    m, sg = mean_sigma(blocks)
    for t, temp in enumerate(T):
        for col, kidx in ((0, 1), (1, 2)):
            exact = CF.ring_structure_factor(N, 1 / temp, kidx)
            assert abs(m[t, col] - exact) < 4.5 * sg[t, col], (temp, kidx, m[t, col], exact, sg[t, col])
            assert sg[t, col] < 0.05 * exact


def test_beta_zero_structure_factor_is_one():
    """independent unit spins: <|sum_i S_i e^{ikr}|^2> = N for every k, so <G> = 1."""
    L = 8
    edges, _ = O.levy_edges(L, 3.5, 6, 0x12113991, 0)
    g = G.colour_major(L * L, [tuple(e) for e in edges])
    lat = g["new_to_old"]
    blocks = fourier_blocks(g, np.array([np.inf, np.inf]), (L, L, (lat % L).astype(np.int32), (lat // L).astype(np.int32)), 30, 30, 3)
    m, sg = mean_sigma(blocks)
    assert np.all(np.abs(m - 1.0) < 4.5 * sg) and np.all(sg < 0.05)
