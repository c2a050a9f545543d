"""The five BASELINE.json configurations as seeded synthetic problems (inputs only).

make_config(i) returns a Problem for config i (1-based, as in BASELINE.json `configs`);
`scale` < 1 returns a down-scaled twin from the same generator (fewer pins / smaller domain at the
same triangle size and ray spacing) for CPU-affordable tests.  Seeds: 20260701 + i.
"""
from dataclasses import dataclass, field
import numpy as np

from .mesh import Mesh, pin_cell_mesh, square_lattice_mesh, hex_core_mesh, delaunay_mesh
from .xs import CrossSections, make_xs
from .quadrature import tabuchi_yamamoto

BC_VACUUM = 0
BC_REFLECTIVE = 1
N_CONFIGS = 5
_SEED0 = 20260701


@dataclass
class Problem:
    name: str
    mesh: Mesh
    xs: CrossSections
    n_azim: int                 # directions over [0, 2*pi)
    spacing: float              # desired ray spacing, cm
    polar_sin: np.ndarray       # [P]
    polar_weight: np.ndarray    # [P]
    bc: tuple                   # (left, right, bottom, top) in {BC_VACUUM, BC_REFLECTIVE}
    n_iters: int                # fixed power-iteration count used for k_eff parity
    notes: str = ""
    extra: dict = field(default_factory=dict)

    @property
    def n_groups(self):
        return self.xs.n_groups

    @property
    def n_polar(self):
        return int(len(self.polar_sin))


def _guide_tubes(rng, n, count):
    pos = rng.choice(n * n, size=min(count, n * n // 4), replace=False)
    m = np.zeros((n, n), dtype=bool)
    m.ravel()[pos] = True
    return m


def make_config(index: int, scale: float = 1.0) -> Problem:
    if not 1 <= index <= N_CONFIGS:
        raise ValueError("config index must be 1..5")
    seed = _SEED0 + index
    rng = np.random.default_rng(seed)
    if index == 1:
        mesh = pin_cell_mesh(1.26, 0.54, seed=seed)
        xs = make_xs(2, [True, False, False], seed, sigt_range=(0.2, 1.5), c_range=(0.3, 0.89),
                     n_up=0, chi_first_only=True)
        s, w = tabuchi_yamamoto(2)
        return Problem("cfg1_pin_cell", mesh, xs, 8, 0.1, s, w, (1, 1, 1, 1), 50,
                       "single square pin cell, 64 FSRs, 2 groups, reflective x4")
    if index == 2:
        n = max(3, int(round(17 * np.sqrt(scale))))
        fuel = ((np.add.outer(np.arange(n) // 5, np.arange(n) // 5) + int(rng.integers(0, 4))) % 4).astype(np.int64)
        gt = _guide_tubes(rng, n, 25)
        pinmat = np.where(gt, 4, fuel)
        mesh = square_lattice_mesh(pinmat, 1.26, 0.54, moderator=5)
        xs = make_xs(7, [True, True, True, True, False, False], seed, sigt_range=(0.2, 1.5),
                     c_range=(0.4, 0.95), n_up=3)
        s, w = tabuchi_yamamoto(3)
        return Problem("cfg2_assembly17", mesh, xs, 32, 0.05, s, w, (1, 1, 1, 1), 20,
                       f"{n}x{n} pin assembly, 24 FSRs per pin, 7 groups, reflective x4")
    if index == 3:
        n = max(3, int(round(17 * np.sqrt(scale))))
        pinmat = np.zeros((2 * n, 2 * n), dtype=np.int64)
        for ay in range(2):
            for ax in range(2):
                ii, jj = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
                edge = np.minimum(np.minimum(ii, n - 1 - ii), np.minimum(jj, n - 1 - jj))
                if (ax + ay) % 2 == 0:
                    blk = np.zeros((n, n), dtype=np.int64)                  # UO2-like: one fuel type
                else:
                    blk = np.where(edge == 0, 1, np.where(edge <= 2, 2, 3))   # MOX-like: three zones
                gt = _guide_tubes(rng, n, 25)
                blk = np.where(gt, 4, blk)
                pinmat[ay * n:(ay + 1) * n, ax * n:(ax + 1) * n] = blk
        band_cells = max(1, int(round(6 * np.sqrt(scale))))
        band_w = 1.19 * band_cells
        mesh = square_lattice_mesh(pinmat, 1.26, 0.54, moderator=5, band_cells=band_cells,
                                   band_width=band_w, band_material=5)
        xs = make_xs(7, [True, True, True, True, False, False], seed, sigt_range=(0.2, 1.5),
                     c_range=(0.4, 0.95), n_up=3)
        s, w = tabuchi_yamamoto(3)
        return Problem("cfg3_quarter_core", mesh, xs, 64, 0.02, s, w, (1, 0, 1, 0), 20,
                       "2x2 assemblies + water band on +x/+y; reflective left/bottom, vacuum right/top")
    if index == 4:
        rings = max(2, int(round(9 * np.sqrt(scale))))
        mesh = hex_core_mesh(0.9, rings, seed=seed)
        xs = make_xs(33, [True] * 7 + [False, False], seed, sigt_range=(0.1, 0.6), c_range=(0.5, 0.93),
                     n_up=4, down_decay=0.7, up_frac=0.02, chi_groups=14)
        s, w = tabuchi_yamamoto(3)
        return Problem("cfg4_hex_fast", mesh, xs, 48, 0.03, s, w, (0, 0, 0, 0), 20,
                       "7 hex assemblies on one hex lattice + duct/coolant filler; vacuum x4")
    # index == 5
    n_side = max(8, int(round(707 * np.sqrt(scale))))
    L = 100.0 * n_side / 707.0
    mesh = delaunay_mesh(L, L, n_side, seed=seed, n_materials=8)
    xs = make_xs(51, [True, False, True, False, True, False, False, True], seed, sigt_range=(0.2, 1.2),
                 c_range=(0.4, 0.93), n_up=6, down_decay=0.75, chi_groups=17)
    s, w = tabuchi_yamamoto(3)
    return Problem("cfg5_stress", mesh, xs, 64, 0.01, s, w, (1, 0, 1, 0), 20,
                   f"Delaunay stress mesh {L:.1f} cm square; reflective left/bottom, vacuum right/top")
