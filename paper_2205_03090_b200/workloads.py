"""Seeded synthetic workloads for the batched SRK two-phase flash (BASELINE.json configs 1-4 and the paper's own
three case studies).

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the method's
arithmetic: only component tables, a counter-based random number generator and the sampling recipes
(uniform P, T; Dirichlet z).  The paper's own case studies are synthetic by construction
(Latin-hypercube + Dirichlet sampling, section 2.4); these recipes keep the same
shapes and value distributions with plain seeded i.i.d. draws.

Counter-based RNG: the k-th uniform of mixture n under seed s is

    u = ((mix64(s + 0x9E3779B97F4A7C15 * (64 n + k + 1)) >> 11) + 0.5) * 2**-53

with mix64 the SplitMix64 finaliser, so 0 < u < 1 strictly and any prefix of a config is
reproducible.  k = 0 -> T, k = 1 -> P, k >= 2 -> composition draws.

Config 5 (warm start near the phase boundary) needs oracle labels to build its inputs and therefore
lives with the tests (tests/config5.py), not here.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)

SEEDS = {1: 2205030901, 2: 2205030902, 3: 2205030903, 4: 2205030904, 5: 2205030905}


def mix64(x: np.ndarray) -> np.ndarray:
    """SplitMix64 finaliser on uint64 arrays (wrap-around arithmetic)."""
    x = np.asarray(x, dtype=np.uint64)
    with np.errstate(over="ignore"):
        x = (x ^ (x >> np.uint64(30))) * _M1
        x = (x ^ (x >> np.uint64(27))) * _M2
        x = x ^ (x >> np.uint64(31))
    return x


def uniform(seed: int, n: np.ndarray, k: int) -> np.ndarray:
    """k-th uniform in (0, 1) of mixtures ``n`` (int array) under ``seed``."""
    n = np.asarray(n, dtype=np.uint64)
    with np.errstate(over="ignore"):
        ctr = np.uint64(seed) + _GOLDEN * (np.uint64(64) * n + np.uint64(k + 1))
    bits = mix64(ctr) >> np.uint64(11)
    return (bits.astype(np.float64) + 0.5) * (2.0 ** -53)


def normal(seed: int, n: np.ndarray, k: int) -> np.ndarray:
    """Standard normal from uniforms k and k+1 (Box-Muller, cosine branch)."""
    u1 = uniform(seed, n, k)
    u2 = uniform(seed, n, k + 1)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)


# ----------------------------------------------------------------------------------------------
# Component data (BASELINE.json configs; Tc in K, Pc in bar, acentric factor)
# ----------------------------------------------------------------------------------------------
_COMP = {
    "C1": (190.56, 45.99, 0.011),
    "C2": (305.32, 48.72, 0.099),
    "C3": (369.83, 42.48, 0.152),
    "nC4": (425.12, 37.96, 0.200),
    "nC5": (469.7, 33.70, 0.252),
    "nC6": (507.6, 30.25, 0.301),
    "nC7": (540.2, 27.40, 0.350),
    "nC10": (617.7, 21.10, 0.490),
    "CO2": (304.13, 73.77, 0.225),
    "N2": (126.2, 33.98, 0.037),
}

HC8 = ["C1", "C2", "C3", "nC4", "nC5", "nC6", "nC7", "nC10"]


@dataclass
class System:
    """Component constants of one mixture family (what ptflash_create takes)."""

    names: list
    Tc: np.ndarray
    Pc: np.ndarray
    omega: np.ndarray
    kij: np.ndarray  # [nc, nc] symmetric, zero diagonal

    @property
    def nc(self) -> int:
        return len(self.names)


def make_system(names, kij_pairs=None) -> System:
    nc = len(names)
    Tc = np.array([_COMP[c][0] for c in names], dtype=np.float64)
    Pc = np.array([_COMP[c][1] for c in names], dtype=np.float64)
    om = np.array([_COMP[c][2] for c in names], dtype=np.float64)
    kij = np.zeros((nc, nc), dtype=np.float64)
    for (a, b), v in (kij_pairs or {}).items():
        i, j = names.index(a), names.index(b)
        kij[i, j] = kij[j, i] = v
    return System(list(names), Tc, Pc, om, kij)


def system_binary() -> System:
    """Config 1: methane / n-decane, kij = 0."""
    return make_system(["C1", "nC10"])


def system_hc8() -> System:
    """Config 2: eight n-alkanes, kij = 0."""
    return make_system(HC8)


def system_co2_10() -> System:
    """Configs 3-5: the eight hydrocarbons + CO2 + N2; CO2-HC 0.12, N2-HC 0.10, CO2-N2 -0.02."""
    names = HC8 + ["CO2", "N2"]
    pairs = {}
    for hc in HC8:
        pairs[(hc, "CO2")] = 0.12
        pairs[(hc, "N2")] = 0.10
    pairs[("CO2", "N2")] = -0.02
    return make_system(names, pairs)


@dataclass
class Workload:
    """One batch of flash problems: component-major SoA, exactly the layout the C ABI takes."""

    name: str
    system: System
    P: np.ndarray  # [N] bar
    T: np.ndarray  # [N] K
    z: np.ndarray  # [nc, N], columns sum to 1
    meta: dict = field(default_factory=dict)

    @property
    def N(self) -> int:
        return int(self.P.shape[0])


def _dirichlet1(seed, n, nc, k0=2):
    """Dirichlet(1,...,1): normalised exponentials e_i = -ln u."""
    e = np.stack([-np.log(uniform(seed, n, k0 + i)) for i in range(nc)])
    return e / e.sum(axis=0, keepdims=True)


def _dirichlet_half(seed, n, nc, k0=2):
    """Dirichlet(1/2,...,1/2): Gamma(1/2) = normal^2 / 2, then normalise."""
    g = np.stack([0.5 * normal(seed, n, k0 + 2 * i) ** 2 for i in range(nc)])
    return g / g.sum(axis=0, keepdims=True)


def config1(N: int = 1000, seed: int = SEEDS[1], offset: int = 0) -> Workload:
    """Binary C1/nC10: T ~ U[250,550] K, P ~ U[1,150] bar, z_C1 ~ U[0.01,0.99]."""
    n = np.arange(offset, offset + N)
    T = 250.0 + 300.0 * uniform(seed, n, 0)
    P = 1.0 + 149.0 * uniform(seed, n, 1)
    z1 = 0.01 + 0.98 * uniform(seed, n, 2)
    z = np.stack([z1, 1.0 - z1])
    return Workload("config1_binary_c1_nc10", system_binary(), P, T, np.ascontiguousarray(z),
                    {"seed": seed, "offset": offset})


def config2(N: int = 1_000_000, seed: int = SEEDS[2], offset: int = 0) -> Workload:
    """8-component hydrocarbons: z ~ Dirichlet(1), T ~ U[200,600] K, P ~ U[1,200] bar."""
    n = np.arange(offset, offset + N)
    T = 200.0 + 400.0 * uniform(seed, n, 0)
    P = 1.0 + 199.0 * uniform(seed, n, 1)
    z = _dirichlet1(seed, n, 8)
    return Workload("config2_hc8", system_hc8(), P, T, np.ascontiguousarray(z),
                    {"seed": seed, "offset": offset})


def config3(N: int = 1_000_000, seed: int = SEEDS[3], offset: int = 0) -> Workload:
    """10-component CO2-rich: z = 0.6 Dirichlet(1) + 0.4 e_CO2, T ~ U[220,500] K, P ~ U[5,300] bar."""
    n = np.arange(offset, offset + N)
    T = 220.0 + 280.0 * uniform(seed, n, 0)
    P = 5.0 + 295.0 * uniform(seed, n, 1)
    d = _dirichlet1(seed, n, 10)
    z = 0.6 * d
    z[8] += 0.4
    z = z / z.sum(axis=0, keepdims=True)
    return Workload("config3_co2_rich_10", system_co2_10(), P, T, np.ascontiguousarray(z),
                    {"seed": seed, "offset": offset})


def config4(N: int = 1 << 20, seed: int = SEEDS[4], offset: int = 0) -> Workload:
    """Scaling sweep: 10-component system, z ~ Dirichlet(1/2) (whole composition law), P, T as config 3."""
    n = np.arange(offset, offset + N)
    T = 220.0 + 280.0 * uniform(seed, n, 0)
    P = 5.0 + 295.0 * uniform(seed, n, 1)
    z = _dirichlet_half(seed, n, 10)
    return Workload("config4_scaling_dir_half_10", system_co2_10(), P, T, np.ascontiguousarray(z),
                    {"seed": seed, "offset": offset})


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4}


# ----------------------------------------------------------------------------------------------
# The paper's own case studies (section 2.3-2.4)
# ----------------------------------------------------------------------------------------------
# Table 1: Tc in K, Pc in MPa (so P is in MPa for these workloads), acentric factor
_PAPER_COMP = {
    "CH4": (190.55, 4.6, 0.0111),
    "C2H6": (305.43, 4.875, 0.097),
    "C3H8": (369.82, 4.268, 0.1536),
    "nC4H10": (425.16, 3.796, 0.2008),
    "nC5H12": (467.15, 3.3332, 0.2635),
    "C6H14": (507.4, 2.9688, 0.296),
    "C7H16+": (604.5, 2.622, 0.3565),
    "CO2": (304.19, 7.382, 0.225),
    "N2": (126.25, 3.3944, 0.039),
}
PAPER9 = list(_PAPER_COMP)
# Table 2: compositional ranges (low, high) of the four reservoir-fluid types, component order of Table 1
PAPER_FLUID_RANGES = {
    "wet_gas": [(0.80, 1.00), (0.02, 0.07), (0, 0.03), (0, 0.02), (0, 0.02), (0, 0.02), (0, 0.01), (0, 0.02), (0, 0.005)],
    "gas_condensate": [(0.60, 0.80), (0.05, 0.10), (0, 0.04), (0, 0.03), (0, 0.02), (0, 0.02), (0.05, 0.10), (0, 0.035), (0, 0.005)],
    "volatile_oil": [(0.50, 0.70), (0.06, 0.10), (0, 0.045), (0, 0.03), (0, 0.02), (0, 0.02), (0.10, 0.30), (0, 0.02), (0, 0.005)],
    "black_oil": [(0.20, 0.40), (0.03, 0.06), (0, 0.015), (0, 0.015), (0, 0.01), (0, 0.02), (0.45, 0.65), (0, 0.001), (0, 0.005)],
}
# Table 3: Dirichlet concentration parameters (alpha_1 CH4, alpha_2 C2H6, alpha_7 C7+; 1 for the others)
PAPER_FLUID_ALPHA = {"wet_gas": (100.0, 5.0, 1.0), "gas_condensate": (40.0, 5.0, 5.0), "volatile_oil": (55.0, 8.0, 20.0),
                     "black_oil": (25.0, 4.0, 40.0)}
PAPER_FLUIDS = list(PAPER_FLUID_RANGES)
# Table D.6: one typical composition per fluid type (Fig. 3a), component order of Table 1
PAPER_TYPICAL = {
    "wet_gas": [0.9246, 0.0318, 0.0101, 0.0052, 0.0021, 0.0014, 0.0082, 0.0141, 0.0025],
    "gas_condensate": [0.7319, 0.078, 0.0355, 0.0216, 0.0132, 0.0109, 0.0821, 0.0237, 0.0031],
    "volatile_oil": [0.576, 0.0735, 0.0421, 0.0281, 0.0148, 0.0192, 0.2257, 0.0182, 0.0024],
    "black_oil": [0.336, 0.0401, 0.0101, 0.0115, 0.0065, 0.018, 0.574, 0.0007, 0.0031],
}
SEEDS.update({"paper2": 2205030912, "paper4": 2205030914, "paper9": 2205030919})


def make_paper_system(names, kij_pairs=None) -> System:
    nc = len(names)
    Tc = np.array([_PAPER_COMP[c][0] for c in names], dtype=np.float64)
    Pc = np.array([_PAPER_COMP[c][1] for c in names], dtype=np.float64)
    om = np.array([_PAPER_COMP[c][2] for c in names], dtype=np.float64)
    kij = np.zeros((nc, nc), dtype=np.float64)
    for (a, b), v in (kij_pairs or {}).items():
        i, j = names.index(a), names.index(b)
        kij[i, j] = kij[j, i] = v
    return System(list(names), Tc, Pc, om, kij)


def system_paper9() -> System:
    """All nine components of Table 1; the only non-zero BIP is CH4-CO2 = 0.0882."""
    return make_paper_system(PAPER9, {("CH4", "CO2"): 0.0882})


def paper2(N: int = 1_000_000, seed: int = SEEDS["paper2"], offset: int = 0) -> Workload:
    """First case study: CH4 / C6H14, P ~ U[0.1,10] MPa, T ~ U[200,500] K, z ~ Dirichlet(1) (whole simplex)."""
    n = np.arange(offset, offset + N)
    T = 200.0 + 300.0 * uniform(seed, n, 0)
    P = 0.1 + 9.9 * uniform(seed, n, 1)
    z = _dirichlet1(seed, n, 2)
    return Workload("paper2_ch4_c6", make_paper_system(["CH4", "C6H14"]), P, T, np.ascontiguousarray(z),
                    {"seed": seed, "offset": offset, "P_unit": "MPa"})


def paper4(N: int = 1_000_000, seed: int = SEEDS["paper4"], offset: int = 0) -> Workload:
    """Second case study: CH4, C2H6, C3H8, n-C4H10, same P, T ranges, z ~ Dirichlet(1)."""
    n = np.arange(offset, offset + N)
    T = 200.0 + 300.0 * uniform(seed, n, 0)
    P = 0.1 + 9.9 * uniform(seed, n, 1)
    z = _dirichlet1(seed, n, 4)
    return Workload("paper4_c1_c4", make_paper_system(["CH4", "C2H6", "C3H8", "nC4H10"]), P, T, np.ascontiguousarray(z),
                    {"seed": seed, "offset": offset, "P_unit": "MPa"})


_PAPER9_CHUNK = 1 << 18   # proposals per rejection round: fixed, so that the accepted sequence does not depend on N


def _paper9_fluid(kind: str, count: int, seed: int) -> np.ndarray:
    """`count` compositions [9, count] of one fluid type: z ~ Dirichlet(alpha of Table 3) (eq. 9) kept only
    inside the ranges of Table 2.  Gamma variates come from a Philox stream keyed by (seed, type) instead of the paper's
    Latin-hypercube + quantile transform (same law, plain i.i.d. draws).  The six alpha = 1 components other than CH4,
    C2H6, C7+ are drawn as their sum, Gamma(6), times a Dirichlet(1) split, so that a proposal failing the three
    range tests with narrow windows is rejected before the other six numbers are drawn (same joint law)."""
    a1, a2, a7 = PAPER_FLUID_ALPHA[kind]
    lo = np.array([r[0] for r in PAPER_FLUID_RANGES[kind]])[:, None]
    hi = np.array([r[1] for r in PAPER_FLUID_RANGES[kind]])[:, None]
    rng = np.random.Generator(np.random.Philox(key=[seed, PAPER_FLUIDS.index(kind)]))
    rng_rest = np.random.Generator(np.random.Philox(key=[seed, 16 + PAPER_FLUIDS.index(kind)]))   # consumed by survivors only
    big, rest = [0, 1, 6], [2, 3, 4, 5, 7, 8]
    out, have, proposed = [], 0, 0
    while have < count:
        m = _PAPER9_CHUNK
        g = np.stack([rng.standard_gamma(a1, m), rng.standard_gamma(a2, m), rng.standard_gamma(a7, m)])
        G6 = rng.standard_gamma(6.0, m)
        proposed += m
        tot = g.sum(axis=0) + G6
        zb = g / tot
        keep = np.nonzero(np.all((zb >= lo[big]) & (zb <= hi[big]), axis=0))[0]
        e = rng_rest.standard_exponential((6, keep.size))
        zr = e / e.sum(axis=0) * (G6[keep] / tot[keep])
        ok = np.all((zr >= lo[rest]) & (zr <= hi[rest]), axis=0)
        z = np.empty((9, int(ok.sum())))
        z[big] = zb[:, keep[ok]]
        z[rest] = zr[:, ok]
        out.append(z)
        have += z.shape[1]
    z = np.concatenate(out, axis=1)[:, :count]
    return z / z.sum(axis=0, keepdims=True), have / proposed


def paper9(N: int = 1_000_000, seed: int = SEEDS["paper9"], offset: int = 0) -> Workload:
    """Third case study (Tables 1-3): nine components, P ~ U[5,25] MPa, T ~ U[200,600] K, the four fluid types
    equally represented (mixture n is of type n mod 4: wet gas, gas condensate, volatile oil, black oil)."""
    n = np.arange(offset, offset + N)
    T = 200.0 + 400.0 * uniform(seed, n, 0)
    P = 5.0 + 20.0 * uniform(seed, n, 1)
    z = np.empty((9, N))
    accept = {}
    for t, kind in enumerate(PAPER_FLUIDS):
        idx = np.nonzero(n % 4 == t)[0]
        if idx.size == 0:
            continue
        first = (int(n[idx[0]]) - t) // 4            # ordinal of the first requested mixture within its type
        zz, accept[kind] = _paper9_fluid(kind, first + idx.size, seed)
        z[:, idx] = zz[:, first:first + idx.size]
    return Workload("paper9_reservoir_fluids", system_paper9(), P, T, np.ascontiguousarray(z),
                    {"seed": seed, "offset": offset, "P_unit": "MPa", "acceptance": accept, "fluid_of": "n mod 4"})


CONFIGS.update({"paper2": paper2, "paper4": paper4, "paper9": paper9})
