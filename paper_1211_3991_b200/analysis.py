"""Host-side arithmetic on the fp64 accumulators the library fills (PAPER.md:167-190 Eq. 13-18; :233 the paper's
time-averaging policy).  Nothing here touches the device state or the Monte-Carlo arithmetic: the device produces the
sums (xy_read_accumulators, xy_read_fourier_accumulators), this module turns them into the paper's observables and
drives the exponentially growing measurement windows.
"""
import numpy as np

# accumulator columns (include/xy_b200.h XY_NACC): n, E, E^2, |m|, m^2, m^4, Mx/N, My/N
N_, E_, E2_, AM_, M2_, M4_, MX_, MY_ = range(8)


def observables(acc, N, T, acc_k=None, L=None, psi=2.0):
    """acc [..., R, 8] accumulators by temperature (any leading sample axes), T [R].  Returns a dict of arrays [..., R]:
    e = <E>/N, c = (<E^2>-<E>^2)/(N T^2) (Eq. 13), absm = <|m|>, chi = N (<m^2> - |<m>|^2) (Eq. 14, vector <m>),
    u4 = <m^4>/<m^2>^2 - 1 (Eq. 15 per sample), and with acc_k [..., R, 3] (n, sum G1, sum G2) and L: chik = the
    average of the two orientations of chi(k_min), chi0 = N <m^2>, xi2 (Eq. 17 with exponent 1/psi)."""
    acc = np.asarray(acc, np.float64)
    T = np.asarray(T, np.float64)
    m = acc / acc[..., N_:N_ + 1]
    out = {
        "n": acc[..., N_],
        "e": m[..., E_] / N,
        "c": (m[..., E2_] - m[..., E_] ** 2) / (N * T ** 2),
        "absm": m[..., AM_],
        "m2": m[..., M2_],
        "chi": N * (m[..., M2_] - m[..., MX_] ** 2 - m[..., MY_] ** 2),
        "u4": m[..., M4_] / m[..., M2_] ** 2 - 1.0,
    }
    if acc_k is not None:
        acc_k = np.asarray(acc_k, np.float64)
        chik = 0.5 * (acc_k[..., 1] + acc_k[..., 2]) / acc_k[..., 0]
        chi0 = N * m[..., M2_]
        out["chik"] = chik
        out["chi0"] = chi0
        if L is not None:
            ratio = np.maximum(chi0 / chik - 1.0, 0.0)
            out["xi2"] = ratio ** (1.0 / psi) / (2.0 * np.sin(np.pi / L))
    return out


def binder_graph_average(acc):
    """Eq. 15 with the overlines read literally (DESIGN R14): mean over samples of <m^4> over mean of <m^2>^2, minus 1.
    acc [S, R, 8] -> [R]."""
    acc = np.asarray(acc, np.float64)
    m = acc / acc[..., N_:N_ + 1]
    return m[..., M4_].mean(0) / (m[..., M2_] ** 2).mean(0) - 1.0


def run_log_windows(ens, k_first, k_last, sweeps_per_swap=10, or_per_sweep=1, measure_every=1, fourier=False):
    """The paper's time averaging: averages over exponentially increasing windows.  Time is counted in
    PT cycles (sweeps_per_swap sweeps + one swap round): window k covers cycles (2^k, 2^(k+1)].  Runs the ensemble
    from its current state: first 2^k_first cycles without keeping their measurements, then windows k_first..k_last,
    each with freshly cleared accumulators.  With fourier=True the structure factor is measured once per cycle
    (the graph's coordinates must have been set).  Returns a list of dicts {k, cycles, acc [S,R,8], acc_k or None}."""
    ens.run(2 ** k_first, sweeps_per_swap, or_per_sweep, measure_every)
    windows = []
    for k in range(k_first, k_last + 1):
        ens.reset_accumulators()
        n = 2 ** k
        if fourier:
            for _ in range(n):
                ens.run(1, sweeps_per_swap, or_per_sweep, measure_every)
                ens.measure_fourier()
        else:
            ens.run(n, sweeps_per_swap, or_per_sweep, measure_every)
        windows.append({"k": k, "cycles": n, "acc": ens.read_accumulators(),
                        "acc_k": ens.read_fourier_accumulators() if fourier else None})
    return windows


def windows_consistent(windows, N, T, keys=("e", "absm"), rtol=0.02, atol=2e-3):
    """The paper's equilibration check: the observables of the last two windows agree.  Returns (ok, worst) where worst
    is the largest |difference| / (atol + rtol |value|) over the keys, samples and temperatures."""
    a = observables(windows[-2]["acc"], N, T)
    b = observables(windows[-1]["acc"], N, T)
    worst = 0.0
    for key in keys:
        worst = max(worst, float(np.max(np.abs(a[key] - b[key]) / (atol + rtol * np.abs(b[key])))))
    return worst <= 1.0, worst
