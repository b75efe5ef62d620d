"""Block / jackknife statistics used by the equilibrium tests (R13)."""
import numpy as np

# accumulator columns (same order on both sides: n, E, E^2, |m|, m^2, m^4, Mx/N, My/N)
N_, E_, E2_, AM_, M2_, M4_, MX_, MY_ = range(8)


def block_means(blocks):
    """blocks: array [B][..., 8] of accumulator *increments*; returns per-block means [B][..., 8]."""
    blocks = np.asarray(blocks, np.float64)
    return blocks / blocks[..., N_:N_ + 1]


def jackknife(blocks, fn):
    """delete-one jackknife of fn(mean accumulators) over blocks; returns (estimate, sigma)."""
    blocks = np.asarray(blocks, np.float64)
    B = blocks.shape[0]
    tot = blocks.sum(0)
    full = fn(tot / tot[..., N_:N_ + 1])
    loo = np.array([fn((tot - blocks[b]) / (tot - blocks[b])[..., N_:N_ + 1]) for b in range(B)])
    sigma = np.sqrt((B - 1) / B * ((loo - loo.mean(0)) ** 2).sum(0))
    return full, sigma


def obs_energy(N):
    return lambda m: m[..., E_] / N


def obs_absm():
    return lambda m: m[..., AM_]


def obs_m2():
    return lambda m: m[..., M2_]


def obs_m4():
    return lambda m: m[..., M4_]


def obs_u4():
    return lambda m: m[..., M4_] / m[..., M2_] ** 2 - 1.0          # Eq. 15 per sample (DESIGN R14)


def obs_var_e():
    return lambda m: m[..., E2_] - m[..., E_] ** 2


def specific_heat_estimators(blocks, T, N):
    """Eq. 13: c = (<E^2> - <E>^2) / (N T^2) = (1/N) d<E>/dT.  blocks [B][R][8] accumulator increments
    by temperature (pooled over samples of one graph, or one sample).  Returns, for the interior temperatures,
    (c_fluct, sigma, c_deriv, sigma): delete-one jackknife; the derivative is the 3-point Lagrange formula on the
    (non-uniform) ladder."""
    T = np.asarray(T, np.float64)

    def deriv(m):
        e = m[..., E_] / N
        h0, h1 = T[1:-1] - T[:-2], T[2:] - T[1:-1]
        return (-h1 / (h0 * (h0 + h1)) * e[..., :-2] + (h1 - h0) / (h0 * h1) * e[..., 1:-1]
                + h0 / (h1 * (h0 + h1)) * e[..., 2:])

    def fluct(m):
        return ((m[..., E2_] - m[..., E_] ** 2) / (N * T ** 2))[..., 1:-1]

    cf, sf = jackknife(blocks, fluct)
    cd, sd = jackknife(blocks, deriv)
    return cf, sf, cd, sd
