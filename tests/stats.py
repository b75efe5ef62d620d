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
