"""The five BASELINE.json configs (and the L-scan of config 3) as seeded synthetic workloads.

The paper's runs draw random Levy graphs (rho in {0, 5/3, ..., 14/3, inf}, L = 16..384, z = 4,
PAPER.md:233); no dataset is involved.  These recipes stand in for them with BASELINE.json's shapes
(z = 6), built by the shared builder (levy.py) from base seed 0x12113991.
"""
from dataclasses import dataclass, replace

import numpy as np

BASE_SEED = 0x12113991
# moves per site of the colour-reducing local search that bench.py applies after the smallest-last colouring
# (levy.build(reduce_colours=...), include/xy_levy.h xy_levy_build_opt): the fifth colour class shrinks from ~1.4 % of
# the sites to a few dozen.  The parity tests run both colourings; the oracle goldens use the plain one.
REDUCE_COLOURS = 8


@dataclass(frozen=True)
class Workload:
    name: str
    L: int
    rho: float
    z: int
    R: int
    T_min: float
    T_max: float
    S: int
    sweeps: int
    sweeps_per_swap: int = 10
    or_per_sweep: int = 1
    measure_every: int = 1
    seed: int = BASE_SEED

    @property
    def N(self):
        return self.L * self.L

    def temperatures(self):
        """geometric grid, fp64 (R15)."""
        if self.R == 1:
            return np.array([self.T_min])
        k = np.arange(self.R, dtype=np.float64)
        return self.T_min * (self.T_max / self.T_min) ** (k / (self.R - 1))

    def updates_per_sweep(self):
        """one Metropolis + one OR update of every spin of every replica and sample."""
        return (1 + self.or_per_sweep) * self.N * self.R * self.S

    def bytes_per_update(self):
        """own angle + z indices / R + z gathered angles + write-back."""
        return 4.0 + 4.0 * self.z / self.R + 4.0 * self.z + 4.0

    def scaled(self, **kw):
        return replace(self, **kw)


CONFIGS = {
    0: Workload("config0_L16_rho3.5_R8_S1", 16, 3.5, 6, 8, 1.0, 4.0, 1, 10_000),
    1: Workload("config1_L64_rho2.5_R16_S32", 64, 2.5, 6, 16, 1.5, 4.0, 32, 20_000),
    2: Workload("config2_L128_rho3.5_R32_S64", 128, 3.5, 6, 32, 1.5, 4.0, 64, 10_000),
    3: Workload("config3_L256_rho4.5_R32_S16", 256, 4.5, 6, 32, 1.0, 3.5, 16, 5_000),
    4: Workload("config4_L512_rho3.0_R64_S8", 512, 3.0, 6, 64, 1.5, 4.0, 8, 2_000),
}


def lscan(L):
    """config 3's throughput scan: L in {32, 64, 128, 256} at 512 replica-samples (R=32 x S=16)."""
    return CONFIGS[3].scaled(name=f"config3b_L{L}_rho4.5_R32_S16", L=L)


def square_lattice(L, R, T_min, T_max, S, name=None):
    """rho -> infinity at z = 4 is the periodic square lattice, Q = 2 colours: the paper's KT
    benchmark and, with L = 128, the shape of its timing experiment (Table III, PAPER.md:474-494:
    square lattice, N = 2^14, PBC).  Built by the shared builder with rho = 100 (every other bond has weight <= 2^-50)."""
    return Workload(name or f"square_L{L}_z4_R{R}_S{S}", L, 100.0, 4, R, T_min, T_max, S, 0)
