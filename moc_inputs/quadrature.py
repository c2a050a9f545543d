"""Polar quadrature constants (problem INPUTS, not method arithmetic).

The paper states no quadrature (§II.A gives only Eq. (4)-(5));
BASELINE.json's configs name the Tabuchi-Yamamoto sets.  The constants below
are the published optimal 2- and 3-point sets (sin(theta_p), weight over the
upper hemisphere, weights sum to 1).  Parity does not depend on them: both the
oracle and the CUDA path read these same arrays.  tests/test_inputs.py checks
them against what the mathematics fixes (sum w = 1, sum w sin = pi/4 to
quadrature accuracy, Bickley Ki3 reproduction).
"""
import numpy as np

_TY = {
    1: ([0.798184], [1.0]),
    2: ([0.363900, 0.899900], [0.212854, 0.787146]),
    3: ([0.166648, 0.537707, 0.932954], [0.046233, 0.283619, 0.670148]),
}


def tabuchi_yamamoto(n_polar: int):
    """Return (sin_theta[P], weight[P]) float64; weights renormalised to sum exactly ~1."""
    if n_polar not in _TY:
        raise ValueError(f"no Tabuchi-Yamamoto set for P={n_polar}")
    s, w = _TY[n_polar]
    s = np.asarray(s, dtype=np.float64)
    w = np.asarray(w, dtype=np.float64)
    w = w / w.sum()
    return s.copy(), w
