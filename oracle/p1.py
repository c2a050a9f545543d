"""ctypes front-end of oracle/moc_oracle_p1.c -- TEST INFRASTRUCTURE, FP64.

SURVEY 8(f) NEXT-4: the oracle's sweep with a linearly anisotropic (P_1) scattering source, Eq. (2) of
arxiv/paper_2607_01591 truncated at l = 1; readings P-1..P-6 in the C file's header and DESIGN.md 8e.
Nothing here is shared with, or imported by, the CUDA path.
"""
import ctypes as C

import numpy as np

from . import _dp, _f64, _i32, _i64, lib


def track_directions(ends):
    """Unit vector from the start point to the end point of every track, [T][2] (P-2)."""
    e = _f64(ends).reshape(-1, 4)
    u = e[:, 2:] - e[:, :2]
    return np.ascontiguousarray(u / np.sqrt((u * u).sum(1))[:, None])


def moments(n_regions, seg_offset, seg_region, seg_length, track_weight, track_dir):
    """P-5: Mxx, Mxy, Myy [R]."""
    so, sr, sl, tw, td = _i64(seg_offset), _i32(seg_region), _f64(seg_length), _f64(track_weight), _f64(track_dir)
    out = [np.empty(n_regions) for _ in range(3)]
    rc = lib().orc_p1_moments(C.c_int(n_regions), C.c_int(len(tw)), _dp(so), _dp(sr), _dp(sl), _dp(tw), _dp(td), *[_dp(a) for a in out])
    if rc != 0:
        raise RuntimeError(f"orc_p1_moments failed with code {rc}")
    return out


def source(region_material, sigma_s0, sigma_s1, nu_sigma_f, chi, phi, Jx, Jy, k):
    """P-1.  Returns Q0, Q1x, Q1y [R][G]."""
    rm, s0, s1, nf, ch = _i32(region_material), _f64(sigma_s0), _f64(sigma_s1), _f64(nu_sigma_f), _f64(chi)
    R, (M, G) = len(rm), nf.shape
    phi, Jx, Jy = (_f64(a).reshape(R, G) for a in (phi, Jx, Jy))
    out = [np.empty((R, G)) for _ in range(3)]
    rc = lib().orc_p1_source(C.c_int(R), C.c_int(M), C.c_int(G), _dp(rm), _dp(s0), _dp(s1), _dp(nf), _dp(ch), _dp(phi), _dp(Jx),
                             _dp(Jy), C.c_double(k), *[_dp(a) for a in out])
    if rc != 0:
        raise RuntimeError(f"orc_p1_source failed with code {rc}")
    return out


def sweep(region_material, sigma_t, polar_sin, polar_weight, seg_offset, seg_region, seg_length, track_weight, track_dir, link,
          volume, Q0, Q1x, Q1y, psi_in, n_threads=0):
    """P-2..P-5.  Returns (phi, Jx, Jy [R][G], psi_next [T][2][P][G], tallies [3][R][G])."""
    rm, st, ps, pw = _i32(region_material), _f64(sigma_t), _f64(polar_sin), _f64(polar_weight)
    so, sr, sl, tw, td, lk, vol = (_i64(seg_offset), _i32(seg_region), _f64(seg_length), _f64(track_weight), _f64(track_dir),
                                   _i32(link), _f64(volume))
    R, (M, G), P, T = len(rm), st.shape, len(ps), len(tw)
    Q0, Q1x, Q1y = (_f64(a).reshape(R, G) for a in (Q0, Q1x, Q1y))
    psi_in = _f64(psi_in).reshape(T, 2, P, G)
    Mxx, Mxy, Myy = moments(R, so, sr, sl, tw, td)
    phi, Jx, Jy, psi_next, tally = np.empty((R, G)), np.empty((R, G)), np.empty((R, G)), np.empty((T, 2, P, G)), np.empty((3, R, G))
    rc = lib().orc_p1_sweep(C.c_int(R), C.c_int(M), C.c_int(G), C.c_int(P), C.c_int(T), _dp(rm), _dp(st), _dp(ps), _dp(pw), _dp(so),
                            _dp(sr), _dp(sl), _dp(tw), _dp(td), _dp(lk), _dp(vol), _dp(Mxx), _dp(Mxy), _dp(Myy), _dp(Q0), _dp(Q1x),
                            _dp(Q1y), _dp(psi_in), _dp(phi), _dp(Jx), _dp(Jy), _dp(psi_next), _dp(tally), C.c_int(n_threads))
    if rc != 0:
        raise RuntimeError(f"orc_p1_sweep failed with code {rc}")
    return phi, Jx, Jy, psi_next, tally


def power_iteration(region_material, sigma_t, sigma_s0, sigma_s1, nu_sigma_f, chi, polar_sin, polar_weight, seg_offset, seg_region,
                    seg_length, track_weight, track_dir, link, volume, n_iters, state=None, n_threads=0):
    """P-6.  Returns (k, phi, Jx, Jy, psi, k_history).  state = (k, phi, Jx, Jy, psi) resumes."""
    rm, st, s0, s1, nf, ch = (_i32(region_material), _f64(sigma_t), _f64(sigma_s0), _f64(sigma_s1), _f64(nu_sigma_f), _f64(chi))
    ps, pw = _f64(polar_sin), _f64(polar_weight)
    so, sr, sl, tw, td, lk, vol = (_i64(seg_offset), _i32(seg_region), _f64(seg_length), _f64(track_weight), _f64(track_dir),
                                   _i32(link), _f64(volume))
    R, (M, G), P, T = len(rm), st.shape, len(ps), len(tw)
    if state is None:
        k, resume = C.c_double(1.0), 0
        phi, Jx, Jy, psi = np.empty((R, G)), np.empty((R, G)), np.empty((R, G)), np.empty((T, 2, P, G))
    else:
        k, resume = C.c_double(state[0]), 1
        phi, Jx, Jy = (_f64(a).reshape(R, G).copy() for a in state[1:4])
        psi = _f64(state[4]).reshape(T, 2, P, G).copy()
    hist = np.empty(max(n_iters, 1))
    rc = lib().orc_p1_power_iteration(C.c_int(R), C.c_int(M), C.c_int(G), C.c_int(P), C.c_int(T), _dp(rm), _dp(st), _dp(s0), _dp(s1),
                                      _dp(nf), _dp(ch), _dp(ps), _dp(pw), _dp(so), _dp(sr), _dp(sl), _dp(tw), _dp(td), _dp(lk),
                                      _dp(vol), C.c_int(n_iters), C.c_int(resume), C.byref(k), _dp(phi), _dp(Jx), _dp(Jy), _dp(psi),
                                      _dp(hist), C.c_int(n_threads))
    if rc != 0:
        raise RuntimeError(f"orc_p1_power_iteration failed with code {rc}")
    return k.value, phi, Jx, Jy, psi, hist[:n_iters]
