"""Seeded, synthetic input descriptions shared by the tests, bench.py, the oracle wrapper and the
CUDA binding.  This module holds INPUTS ONLY -- species tables, trap parameters, tolerances, launch
descriptors and seeded explicit initial conditions -- and none of the method's arithmetic (no
right-hand side, no integrator, no generator of directions/phases: the oracle and the CUDA path each
implement their own Philox / grid generator from the recipe in DESIGN.md).  It imports neither
``oracle`` nor ``paper_2509_15117_b200``.

The five workloads are BASELINE.json ``configs[0..4]``; they stand in for the paper's own runs
(Fig. 1 / Fig. 4 of arXiv 2509.15117), whose inputs were never published.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import Dict, List

import numpy as np

# --- unit conversions (CODATA 2022 values; inputs to both sides) ---------------------------------
AU_TIME_S = 2.4188843265864e-17          # 1 a.u. of time in seconds
OMEGA_RF_AU = 2.0 * math.pi * 2.0e6 * AU_TIME_S   # Omega_rf = 2 pi * 2 MHz (BASELINE.json configs[0])

# species: mass in u, static dipole polarisability in a.u. (BASELINE.json configs[0], [2])
M_YB174_U = 173.94
ATOMS: Dict[str, Dict[str, float]] = {
    "Li7": {"m_u": 7.016, "alpha": 164.1},
    "Na23": {"m_u": 22.990, "alpha": 162.7},
    "K39": {"m_u": 38.964, "alpha": 290.0},
    "Rb87": {"m_u": 86.909, "alpha": 319.2},
    "Cs133": {"m_u": 132.905, "alpha": 401.0},
}

MODE_EXPLICIT, MODE_GRID, MODE_PHILOX, MODE_THERMAL = 0, 1, 2, 3


@dataclass(frozen=True)
class Params:
    """Physical + numerical parameters of one cell (what ia_create takes)."""
    m_ion_u: float = M_YB174_U
    m_atom_u: float = ATOMS["Rb87"]["m_u"]
    alpha_au: float = ATOMS["Rb87"]["alpha"]
    a: tuple = (-0.0005, -0.0005, 0.001)
    q: tuple = (0.1, -0.1, 0.0)
    omega_rf_au: float = OMEGA_RF_AU
    De_K: float = 1.0
    r0_a0: float = 5000.0
    rtol: float = 1e-10
    atol: float = 1e-12
    t_max_rf: float = 1.0e4
    h_max_rf: float = 0.25
    r_coll_a0: float = 500.0
    max_steps: int = 2 ** 31

    def with_atom(self, name: str) -> "Params":
        return replace(self, m_atom_u=ATOMS[name]["m_u"], alpha_au=ATOMS[name]["alpha"])


@dataclass(frozen=True)
class Launch:
    """Initial-condition description of one launch (what ia_run takes)."""
    mode: int = MODE_GRID
    n: int = 0
    n_theta: int = 0
    n_phi: int = 0
    domain: int = 0            # 0 octant, 1 full sphere
    phase_mode: int = 0        # 0 fixed phase0, 1 uniform from Philox
    phase0: float = 0.0
    E_min_uK: float = 1.0
    E_max_uK: float = 1.0
    seed: int = 0
    cell: int = 0
    first_index: int = 0
    path: int = 0              # 0 production kernel pair, 1 bulk kernel only, 2 cooperative kernel only
    T_atom_uK: float = 0.0     # THERMAL: bath temperature
    T_ion_uK: float = 0.0      # THERMAL: ion temperature (the paper's thermal runs use 10 uK)


@dataclass(frozen=True)
class Cell:
    name: str
    params: Params
    launch: Launch


DEFAULT_SEED = 0x2509_15117_B200 & 0xFFFFFFFFFFFFFFFF


def config0() -> Cell:
    """Yb+ + 7Li, E = 10 uK, 32x32 octant grid, phase 0, t_max 2000 T_rf (BASELINE.json configs[0])."""
    p = replace(Params().with_atom("Li7"), t_max_rf=2000.0)
    return Cell("config0_YbLi_10uK_32x32", p,
                Launch(mode=MODE_GRID, n=32 * 32, n_theta=32, n_phi=32, E_min_uK=10.0, E_max_uK=10.0))


def config1(n_side: int = 512) -> Cell:
    """Yb+ + 87Rb fractal angle map, E = 1.5 uK, n_side x n_side octant grid (configs[1])."""
    p = Params().with_atom("Rb87")
    return Cell(f"config1_YbRb_1.5uK_{n_side}x{n_side}", p,
                Launch(mode=MODE_GRID, n=n_side * n_side, n_theta=n_side, n_phi=n_side,
                       E_min_uK=1.5, E_max_uK=1.5))


SPECIES_ORDER = ["Li7", "Na23", "K39", "Rb87", "Cs133"]
ENERGIES_UK = [1.0, 3.0, 10.0, 30.0, 100.0]


def config2(n_per_cell: int = 2 ** 20, seed: int = DEFAULT_SEED) -> List[Cell]:
    """Species x energy sweep, 25 cells, Philox(seed, cell = 5*species + energy, index) (configs[2])."""
    cells = []
    for si, sp in enumerate(SPECIES_ORDER):
        for ei, E in enumerate(ENERGIES_UK):
            cells.append(Cell(f"config2_{sp}_{E:g}uK", Params().with_atom(sp),
                              Launch(mode=MODE_PHILOX, n=n_per_cell, domain=0, phase_mode=1,
                                     E_min_uK=E, E_max_uK=E, seed=seed, cell=5 * si + ei)))
    return cells


DE_SWEEP_K = [0.1, 1.0, 10.0, 100.0]
QX_SWEEP = [0.05, 0.1, 0.2, 0.3, 0.4]


def config3(n_per_cell: int = 2 ** 22, seed: int = DEFAULT_SEED) -> List[Cell]:
    """Yb+ + 87Rb at 3 uK, D_e x q_x sweep, 20 cells (configs[3])."""
    cells = []
    for di, De in enumerate(DE_SWEEP_K):
        for qi, qx in enumerate(QX_SWEEP):
            p = replace(Params().with_atom("Rb87"), De_K=De, q=(qx, -qx, 0.0))
            cells.append(Cell(f"config3_De{De:g}K_q{qx:g}", p,
                              Launch(mode=MODE_PHILOX, n=n_per_cell, domain=0, phase_mode=1,
                                     E_min_uK=3.0, E_max_uK=3.0, seed=seed, cell=100 + 5 * di + qi)))
    return cells


def config4(n_total: int = 300_000_000, batch: int = 2 ** 24, seed: int = DEFAULT_SEED) -> List[Cell]:
    """Throughput ensemble: Yb+ + 87Rb, E log-uniform in [1,100] uK, full sphere, uniform phase,
    streamed in batches of one Philox stream (configs[4])."""
    cells = []
    first = 0
    p = Params().with_atom("Rb87")
    while first < n_total:
        n = min(batch, n_total - first)
        cells.append(Cell(f"config4_batch{len(cells)}", p,
                          Launch(mode=MODE_PHILOX, n=n, domain=1, phase_mode=1, E_min_uK=1.0,
                                 E_max_uK=100.0, seed=seed, cell=200, first_index=first)))
        first += n
    return cells


THERMAL_T_UK = [1.0, 3.0, 10.0, 30.0, 100.0]


def thermal(atom: str = "Rb87", T_atom_uK: float = 1.0, De_K: float = 1.0, n: int = 2 ** 20,
            seed: int = DEFAULT_SEED) -> Cell:
    """One bar of the paper's Fig. 3: thermal run of Yb+ with
    `atom` at bath temperature T, ion at 10 uK, atom uniform on the r0 sphere with Maxwell-Boltzmann velocity
    (v_r < 0 enforced), uniform rf phase.  Philox cell = 300 + 25*[De = 100 K] + 5*species + temperature index
    (or 399 for a temperature off the list)."""
    si = SPECIES_ORDER.index(atom)
    ti = THERMAL_T_UK.index(T_atom_uK) if T_atom_uK in THERMAL_T_UK else None
    cell = 399 if ti is None else 300 + (25 if De_K >= 50.0 else 0) + 5 * si + ti
    p = replace(Params().with_atom(atom), De_K=De_K)
    return Cell(f"thermal_{atom}_{T_atom_uK:g}uK_De{De_K:g}K", p,
                Launch(mode=MODE_THERMAL, n=n, domain=1, phase_mode=1, seed=seed, cell=cell,
                       T_atom_uK=T_atom_uK, T_ion_uK=10.0))


def fig4(atom: str = "Rb87", E_uK: float = 10.0, n: int = 10_000, phase_mode: int = 1, phase0: float = 0.0,
         r0_a0: float = 20_000.0, seed: int = DEFAULT_SEED) -> Cell:
    """One point of the paper's Fig. 4: head-on collisions of `atom` with
    Yb+ at one collision energy from the sphere r0 = 20 000 a0, D_e = 1 K, directions uniform on the octant, rf phase
    uniformly random (phase_mode 1, the figure) or fixed at phase0 (phase_mode 0: the oscillation of about +-0.1 in
    the probability that PAPER.md:68 describes).  Philox cell = 400 + species."""
    p = replace(Params().with_atom(atom), r0_a0=r0_a0)
    return Cell(f"fig4_{atom}_{E_uK:g}uK_r0{r0_a0:g}" + ("" if phase_mode else f"_phase{phase0:.3f}"), p,
                Launch(mode=MODE_PHILOX, n=n, domain=0, phase_mode=phase_mode, phase0=phase0, E_min_uK=E_uK,
                       E_max_uK=E_uK, seed=seed, cell=400 + SPECIES_ORDER.index(atom)))


def subgrid_indices(n_side: int, every: int) -> np.ndarray:
    """Local indices of the (every x every)-decimated sub-grid of an n_side x n_side grid launch."""
    ii = np.arange(every // 2, n_side, every, dtype=np.uint64)
    return (ii[:, None] * np.uint64(n_side) + ii[None, :]).reshape(-1)


# --- seeded explicit initial conditions (numbers only; no physics beyond placing the particles) ---

def impact_ic(b_a0: float, r0_a0: float, v0_au: float) -> np.ndarray:
    """Ion at rest at the origin; atom on the r0 sphere at impact parameter b, moving along +x."""
    y = np.zeros(12)
    y[3] = -math.sqrt(r0_a0 ** 2 - b_a0 ** 2)
    y[4] = b_a0
    y[9] = v0_au
    return y


def random_states(n: int, seed: int, r_lo: float = 55.0, r_hi: float = 4000.0) -> np.ndarray:
    """n seeded 12-vectors spanning far field to short range, for one-step-map parity tests:
    ion within ~200 a0 of the centre, separation log-uniform in [r_lo, r_hi], velocities ~1e-8..1e-6."""
    rng = np.random.default_rng(seed)
    y = np.zeros((n, 12))
    y[:, 0:3] = rng.normal(0.0, 100.0, (n, 3))
    r = np.exp(rng.uniform(math.log(r_lo), math.log(r_hi), n))
    dirs = rng.normal(size=(n, 3))
    dirs /= np.linalg.norm(dirs, axis=1, keepdims=True)
    y[:, 3:6] = y[:, 0:3] + r[:, None] * dirs
    y[:, 6:9] = rng.normal(0.0, 3e-8, (n, 3))
    y[:, 9:12] = rng.normal(0.0, 2e-7, (n, 3))
    return y
