"""Shared helpers of the GPU parity tests: build the same seeded problem for the oracle (its own tracer) and for the
CUDA path (the library's tracer), and the error norms of DESIGN.md ("Tolerances")."""
import numpy as np

import oracle
import paper_2607_01591_b200 as nd
from moc_inputs import make_config

PHI_RTOL = 1e-4      # BASELINE.json north_star: per-sweep FSR scalar flux max rel err <= 1e-4
K_PCM = 5.0          # k_eff within 5 pcm
PSI_ATOL_REL = 2e-5  # boundary flux: diagnostic bound, relative to max |psi| (FP32 chain of <= ~2000 steps)


def phi_rel_err(phi_gpu, phi_orc):
    """Reading 18: max over (r,g) of |phi_gpu-phi_orc| / max(|phi_orc|, 1e-6*max|phi_orc|)."""
    phi_gpu, phi_orc = np.asarray(phi_gpu, np.float64), np.asarray(phi_orc, np.float64)
    den = np.maximum(np.abs(phi_orc), 1e-6 * np.abs(phi_orc).max())
    return float((np.abs(phi_gpu - phi_orc) / den).max())


_POWER_CACHE = {}


class Pair:
    """One seeded problem, set up on both sides independently."""

    def __init__(self, prob, **options):
        self.prob = prob
        m = prob.mesh
        self.o_tr = oracle.generate_tracks(m.xy, m.tri, m.W, m.H, prob.bc, prob.n_azim, prob.spacing)
        self.g_tr = nd.nd_tracks_generate(m.xy, m.tri, m.W, m.H, prob.bc, prob.n_azim, prob.spacing)
        self.gpu = nd.nd_problem_create(prob.xs, prob.polar_sin, prob.polar_weight, m.material, self.g_tr, **options)
        self.R, self.G, self.P, self.T = m.n_regions, prob.n_groups, prob.n_polar, self.o_tr.n_tracks

    def oracle_sweep(self, Q, psi_in):
        p, t = self.prob, self.o_tr
        return oracle.sweep(p.mesh.material, p.xs.sigma_t, p.polar_sin, p.polar_weight, t.seg_offset, t.seg_region,
                            t.seg_length, t.track_weight, t.link, t.volume, Q, psi_in)

    def oracle_power(self, n_iters, state=None, cache_key=None):
        """O-8 on the oracle; results are cached per (problem, n_iters) so kernel variants share one oracle run."""
        key = (self.prob.name, self.R, self.T, n_iters, cache_key)
        if state is None and key in _POWER_CACHE:
            return _POWER_CACHE[key]
        p, t = self.prob, self.o_tr
        out = oracle.power_iteration(p.mesh.material, p.xs.sigma_t, p.xs.sigma_s, p.xs.nu_sigma_f, p.xs.chi,
                                     p.polar_sin, p.polar_weight, t.seg_offset, t.seg_region, t.seg_length,
                                     t.track_weight, t.link, t.volume, n_iters, state=state)
        if state is None:
            _POWER_CACHE[key] = out
        return out

    def close(self):
        self.gpu.destroy()
        self.g_tr.destroy()


def make_pair(index, scale=1.0, **options):
    return Pair(make_config(index, scale=scale), **options)


def seeded_sweep_inputs(pair, seed):
    """Random positive Q and boundary psi (FP32-representable so both sides start from identical values)."""
    rng = np.random.default_rng(seed)
    Q = rng.uniform(0.05, 1.0, size=(pair.R, pair.G))
    psi = rng.uniform(0.0, 2.0, size=(pair.T, 2, pair.P, pair.G)).astype(np.float32)
    return Q, psi
