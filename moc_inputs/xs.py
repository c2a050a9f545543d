"""Seeded synthetic multigroup cross sections (problem INPUTS).

Layouts follow the C ABI (include/nd.h): sigma_t [M][G], sigma_s [M][G_to][G_from]
(row = destination group g, column = source group g', i.e. Sigma_{s,g'->g} of PAPER.md Eq. (1)),
nu_sigma_f [M][G], chi [M][G].  Values are drawn, never benchmark values.
"""
from dataclasses import dataclass
import numpy as np


@dataclass
class CrossSections:
    sigma_t: np.ndarray     # [M][G]
    sigma_s: np.ndarray     # [M][G][G]  [m][g_to][g_from]
    nu_sigma_f: np.ndarray  # [M][G]
    chi: np.ndarray         # [M][G]

    @property
    def n_materials(self) -> int:
        return int(self.sigma_t.shape[0])

    @property
    def n_groups(self) -> int:
        return int(self.sigma_t.shape[1])


def _one_material(rng, G, sigt_range, c_range, fissile, eta_range, n_up, down_decay, up_frac, chi_groups):
    sigt = rng.uniform(sigt_range[0], sigt_range[1], size=G)
    c = rng.uniform(c_range[0], c_range[1], size=G)
    S = np.zeros((G, G))
    for gp in range(G):                      # source group g'
        w = np.zeros(G)
        w[gp] = 1.0                          # in-group
        nd = G - 1 - gp
        if nd > 0:                           # dense downscatter g > g', geometrically decaying, seeded
            w[gp + 1:] = rng.uniform(0.2, 1.0, size=nd) * down_decay ** np.arange(nd) * rng.uniform(0.3, 1.2)
        if n_up > 0 and gp >= G - n_up:      # sparse upscatter only among the last n_up groups
            for g in range(G - n_up, gp):
                if rng.random() < 0.6:
                    w[g] = up_frac * rng.uniform(0.2, 1.0)
        S[:, gp] = w / w.sum() * c[gp] * sigt[gp]
    siga = sigt - S.sum(axis=0)
    if fissile:
        eta = rng.uniform(eta_range[0], eta_range[1], size=G)
        nusf = eta * siga
        chi = np.zeros(G)
        ng = max(1, min(G, chi_groups))
        chi[:ng] = rng.uniform(0.3, 1.0, size=ng) * np.exp(-0.35 * np.arange(ng))
        chi /= chi.sum()
    else:
        nusf = np.zeros(G)
        chi = np.zeros(G)
    return sigt, S, nusf, chi


def make_xs(n_groups, fissile_mask, seed, sigt_range=(0.2, 1.5), c_range=(0.3, 0.89), eta_range=(1.2, 2.0),
            n_up=0, down_decay=0.5, up_frac=0.05, chi_groups=None, chi_first_only=False) -> CrossSections:
    """Draw one XS set.  fissile_mask[m] says whether material m has nuSigma_f > 0."""
    rng = np.random.default_rng(seed)
    G = int(n_groups)
    M = len(fissile_mask)
    if chi_groups is None:
        chi_groups = max(1, G // 3)
    st = np.zeros((M, G))
    ss = np.zeros((M, G, G))
    nf = np.zeros((M, G))
    ch = np.zeros((M, G))
    for m in range(M):
        st[m], ss[m], nf[m], ch[m] = _one_material(rng, G, sigt_range, c_range, bool(fissile_mask[m]),
                                                   eta_range, n_up, down_decay, up_frac, chi_groups)
        if chi_first_only and fissile_mask[m]:
            ch[m] = 0.0
            ch[m, 0] = 1.0
    return CrossSections(st, ss, nf, ch)


def homogeneous_xs(n_groups, seed, **kw) -> CrossSections:
    """A single fissile material (closed-form infinite-medium tests)."""
    return make_xs(n_groups, [True], seed, **kw)
