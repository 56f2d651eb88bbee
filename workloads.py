"""Seeded synthetic workloads (BASELINE.json `configs`).

These stand in for the paper's HITRAN / HITEMP H2O line lists,
whose files are not available here.  This module holds NO arithmetic of the method: it only draws
random line records and names the run parameters.  Both the CPU oracle (`oracle/`) and the CUDA
path (`paper_1503_03806_b200/`) are fed from here; neither imports the other.

Recipe (all float64, `numpy.random.Generator(PCG64(seed))`, seed = config index):
draw order is the nu0 block, then the log10(S) block, then the g0 block, then (config 4) the E''
block.  The drawn list is then ordered by line centre, as HITRAN/HITEMP files are
(wavenumber-ordered); `sorted_by_nu0=False` returns the raw draw order instead.
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np

BAR_PER_ATM = 1.01325          # 1 atm = 1.01325 bar  (PAPER.md:41/187 prints the inverse; reading G4)
MASS_AMU = 18.0                # every config: m = 18 amu


@dataclass
class Workload:
    name: str
    seed: int
    nu0: np.ndarray            # [n] line centres, cm^-1
    S: np.ndarray              # [n] line strength, cm/molecule (at T, or at 296 K when E_low is given)
    gamma0: np.ndarray         # [n] Lorentz HWHM at 296 K and 1 atm, cm^-1/atm
    E_low: np.ndarray | None   # [n] lower-state energy, cm^-1 (config 4) or None
    T: list                    # temperatures, K
    P_atm: list                # pressures, atm
    nu_min: float
    nu_max: float
    dnu: float
    cutoff: float
    bin_width: float | None    # k-distribution bin width, cm^-1 (None: no k-distribution asked)
    n_g: int = 20
    mass_amu: float = MASS_AMU
    q_ratio: object = None     # callable T -> Q(296)/Q(T) (config 4) or None
    extra: dict = field(default_factory=dict)

    @property
    def n_lines(self) -> int:
        return int(self.nu0.shape[0])

    @property
    def n_points(self) -> int:
        return int(round((self.nu_max - self.nu_min) / self.dnu))

    def tp_pairs(self):
        return [(t, p) for t in self.T for p in self.P_atm]


def _order(sorted_by_nu0, nu0, *cols):
    if not sorted_by_nu0:
        return (nu0,) + cols
    idx = np.argsort(nu0, kind="stable")
    return (np.ascontiguousarray(nu0[idx]),) + tuple(None if c is None else np.ascontiguousarray(c[idx]) for c in cols)


def _uniform_S(rng, n, lo, hi):
    return 10.0 ** rng.uniform(lo, hi, n)


def _normal_S(rng, n, mean, sd, lo, hi):
    return 10.0 ** np.clip(rng.normal(mean, sd, n), lo, hi)


def config(k: int, n_lines: int | None = None, sorted_by_nu0: bool = True) -> Workload:
    """Config `k` of BASELINE.json.  `n_lines` overrides the line count (scaled-down test cases keep
    every distribution and run parameter of the config)."""
    rng = np.random.Generator(np.random.PCG64(k))
    if k == 0:
        n = n_lines or 1000
        nu0 = rng.uniform(0.0, 3000.0, n)
        S = _uniform_S(rng, n, -27.0, -19.0)
        g0 = rng.uniform(0.02, 0.1, n)
        nu0, S, g0 = _order(sorted_by_nu0, nu0, S, g0)
        return Workload("cfg0_1e3_lines", 0, nu0, S, g0, None, [1500.0], [1.0], 0.0, 3000.0, 0.01, 25.0, 10.0)
    if k == 1:
        n = n_lines or 100_000
        nu0 = rng.uniform(0.0, 30000.0, n)
        S = _uniform_S(rng, n, -27.0, -19.0)
        g0 = rng.uniform(0.02, 0.1, n)
        nu0, S, g0 = _order(sorted_by_nu0, nu0, S, g0)
        return Workload("cfg1_1e5_lines", 1, nu0, S, g0, None, [1500.0], [1.0], 0.0, 30000.0, 0.01, 100.0, 10.0)
    if k == 2:
        n = n_lines or 1_000_000
        nu0 = rng.uniform(0.0, 30000.0, n)
        S = _normal_S(rng, n, -24.0, 2.0, -32.0, -18.0)
        g0 = rng.uniform(0.02, 0.1, n)
        nu0, S, g0 = _order(sorted_by_nu0, nu0, S, g0)
        P = [p / BAR_PER_ATM for p in (1e-5, 1e-3, 1e-1, 1.0, 10.0, 100.0)]
        return Workload("cfg2_1e6_lines_Psweep", 2, nu0, S, g0, None, [1000.0], P, 0.0, 30000.0, 0.01, 100.0, None)
    if k == 3:
        n = n_lines or 100_000_000
        # density proportional to (30000 - nu): rising linearly toward low wavenumber
        nu0 = 30000.0 * (1.0 - np.sqrt(1.0 - rng.random(n)))
        S = _normal_S(rng, n, -28.0, 3.0, -40.0, -18.0)
        g0 = rng.uniform(0.02, 0.1, n)
        nu0, S, g0 = _order(sorted_by_nu0, nu0, S, g0)
        return Workload("cfg3_1e8_lines", 3, nu0, S, g0, None, [2500.0], [1.0 / BAR_PER_ATM], 0.0, 30000.0, 0.01, 25.0, 100.0)
    if k == 4:
        n = n_lines or 1_000_000
        nu0 = rng.uniform(0.0, 30000.0, n)
        S = _normal_S(rng, n, -24.0, 2.0, -32.0, -18.0)
        g0 = rng.uniform(0.02, 0.1, n)
        E = rng.uniform(0.0, 20000.0, n)
        nu0, S, g0, E = _order(sorted_by_nu0, nu0, S, g0, E)
        T = [float(t) for t in np.logspace(np.log10(500.0), np.log10(3000.0), 20)]
        P = [float(p) / BAR_PER_ATM for p in np.logspace(-4.0, 2.0, 10)]
        # Q(T) = 0.1 T^1.5  =>  Q(296)/Q(T) = (296/T)^1.5 ; this is workload data, not method arithmetic
        return Workload("cfg4_TP_table", 4, nu0, S, g0, E, T, P, 0.0, 30000.0, 0.01, 100.0, 10.0,
                        q_ratio=lambda t: (296.0 / t) ** 1.5)
    raise ValueError(f"no such config: {k}")


def small(seed: int, n_lines: int, nu_max: float, cutoff: float, dnu: float = 0.01, T: float = 1500.0,
          P_atm: float = 1.0, bin_width: float | None = 10.0, with_E: bool = False,
          logS=(-27.0, -19.0), sorted_by_nu0: bool = True) -> Workload:
    """Small ad-hoc case with config-0 distributions, for unit and edge-case tests."""
    rng = np.random.Generator(np.random.PCG64(seed))
    nu0 = rng.uniform(0.0, nu_max, n_lines)
    S = _uniform_S(rng, n_lines, *logS)
    g0 = rng.uniform(0.02, 0.1, n_lines)
    E = rng.uniform(0.0, 20000.0, n_lines) if with_E else None
    nu0, S, g0, E = _order(sorted_by_nu0, nu0, S, g0, E)
    return Workload(f"small_s{seed}_n{n_lines}", seed, nu0, S, g0, E, [T], [P_atm], 0.0, nu_max, dnu, cutoff, bin_width,
                    q_ratio=(lambda t: (296.0 / t) ** 1.5) if with_E else None)
