"""ctypes front-end of the FP64 CPU oracle (oracle/moc_oracle.c).

TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this package; the product (paper_2607_01591_b200) never does.
The oracle follows arxiv/paper_2607_01591 Eq. (1), (3)-(5) and the readings in
DESIGN.md; see the C file's header for the passage-by-passage map and its pins.
"""
import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "moc_oracle.c")
_SRC_P1 = os.path.join(_HERE, "moc_oracle_p1.c")          # NEXT-4: the same sweep with a P_1 scattering source
_LIB = os.path.join(_HERE, "libmoc_oracle.so")
CFLAGS = ["-O2", "-std=c11", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC"]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no -ffast-math, no -march) and return the .so path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_P1)):
        subprocess.check_call(["gcc", *CFLAGS, _SRC, _SRC_P1, "-o", _LIB, "-lm"])
    return _LIB


_lib = None


def _dp(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_fission_rate.restype = C.c_double
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _i64(a):
    return np.ascontiguousarray(a, dtype=np.int64)


@dataclass
class Tracks:
    seg_offset: np.ndarray    # [T+1] int64
    seg_region: np.ndarray    # [S] int32
    seg_length: np.ndarray    # [S] float64
    track_weight: np.ndarray  # [T] float64  omega_a * delta_a
    link: np.ndarray          # [T][2] int32
    track_azim: np.ndarray    # [T] int32
    ends: np.ndarray          # [T][4] float64 x0,y0,x1,y1
    keys: np.ndarray          # [T][4] int32 start side, start slot, end side, end slot
    volume: np.ndarray        # [R] float64 track-estimated areas
    azim_phi: np.ndarray      # [N_a/2]
    azim_weight: np.ndarray   # [N_a/2] per direction
    azim_spacing: np.ndarray  # [N_a/2]
    azim_nx: np.ndarray
    azim_ny: np.ndarray

    @property
    def n_tracks(self):
        return int(len(self.track_weight))

    @property
    def n_segs(self):
        return int(len(self.seg_region))


def generate_tracks(xy, tri, W, H, bc, n_azim, spacing, n_threads=0) -> Tracks:
    """O-2..O-5: cyclic track laydown, links, half-edge ray walk, track-estimated areas."""
    L = lib()
    xy, tri = _f64(xy), _i32(tri)
    bc = _i32(bc)
    h = C.c_void_p()
    rc = L.orc_tracks_generate(C.c_int(len(xy)), C.c_int(len(tri)), _dp(xy), _dp(tri), C.c_double(W), C.c_double(H),
                               _dp(bc), C.c_int(n_azim), C.c_double(spacing), C.c_int(n_threads), C.byref(h))
    if rc != 0:
        raise RuntimeError(f"orc_tracks_generate failed with code {rc}")
    try:
        T, S, NH = C.c_int(), C.c_int64(), C.c_int()
        L.orc_tracks_dims(h, C.byref(T), C.byref(S), C.byref(NH))
        T, S, NH = T.value, S.value, NH.value
        out = Tracks(np.empty(T + 1, np.int64), np.empty(S, np.int32), np.empty(S, np.float64),
                     np.empty(T, np.float64), np.empty((T, 2), np.int32), np.empty(T, np.int32),
                     np.empty((T, 4), np.float64), np.empty((T, 4), np.int32), np.empty(len(tri), np.float64),
                     np.empty(NH, np.float64), np.empty(NH, np.float64), np.empty(NH, np.float64),
                     np.empty(NH, np.int32), np.empty(NH, np.int32))
        L.orc_tracks_copy(h, _dp(out.seg_offset), _dp(out.seg_region), _dp(out.seg_length), _dp(out.track_weight),
                          _dp(out.link), _dp(out.track_azim), _dp(out.ends), _dp(out.keys), _dp(out.volume),
                          _dp(out.azim_phi), _dp(out.azim_weight), _dp(out.azim_spacing), _dp(out.azim_nx),
                          _dp(out.azim_ny))
    finally:
        L.orc_tracks_free(h)
    return out


def track_volumes(n_regions, seg_offset, seg_region, seg_length, track_weight):
    vol = np.empty(n_regions, np.float64)
    so, sr, sl, tw = _i64(seg_offset), _i32(seg_region), _f64(seg_length), _f64(track_weight)
    rc = lib().orc_track_volumes(C.c_int(n_regions), C.c_int(len(tw)), _dp(so), _dp(sr), _dp(sl), _dp(tw), _dp(vol))
    if rc != 0:
        raise RuntimeError(f"orc_track_volumes failed with code {rc}")
    return vol


def sweep(region_material, sigma_t, polar_sin, polar_weight, seg_offset, seg_region, seg_length, track_weight,
          link, volume, Q, psi_in, n_threads=0):
    """O-6.  Returns (phi [R][G], psi_next [T][2][P][G], tally [R][G])."""
    rm, st = _i32(region_material), _f64(sigma_t)
    ps, pw = _f64(polar_sin), _f64(polar_weight)
    so, sr, sl, tw, lk, vol = _i64(seg_offset), _i32(seg_region), _f64(seg_length), _f64(track_weight), _i32(link), _f64(volume)
    R, (M, G), P, T = len(rm), st.shape, len(ps), len(tw)
    Q = _f64(Q).reshape(R, G)
    psi_in = _f64(psi_in).reshape(T, 2, P, G)
    phi, psi_next, tally = np.empty((R, G)), np.empty((T, 2, P, G)), np.empty((R, G))
    rc = lib().orc_sweep(C.c_int(R), C.c_int(M), C.c_int(G), C.c_int(P), C.c_int(T), _dp(rm), _dp(st), _dp(ps), _dp(pw),
                         _dp(so), _dp(sr), _dp(sl), _dp(tw), _dp(lk), _dp(vol), _dp(Q), _dp(psi_in), _dp(phi),
                         _dp(psi_next), _dp(tally), C.c_int(n_threads))
    if rc != 0:
        raise RuntimeError(f"orc_sweep failed with code {rc}")
    return phi, psi_next, tally


def source(region_material, sigma_s, nu_sigma_f, chi, phi, k):
    """O-7.  Returns Q [R][G] (per steradian)."""
    rm, ss, nf, ch = _i32(region_material), _f64(sigma_s), _f64(nu_sigma_f), _f64(chi)
    R, (M, G) = len(rm), nf.shape
    phi = _f64(phi).reshape(R, G)
    Q = np.empty((R, G))
    rc = lib().orc_source(C.c_int(R), C.c_int(M), C.c_int(G), _dp(rm), _dp(ss), _dp(nf), _dp(ch), _dp(phi),
                          C.c_double(k), _dp(Q))
    if rc != 0:
        raise RuntimeError(f"orc_source failed with code {rc}")
    return Q


def fission_rate(region_material, nu_sigma_f, volume, phi):
    rm, nf, vol = _i32(region_material), _f64(nu_sigma_f), _f64(volume)
    R, G = len(rm), nf.shape[1]
    phi = _f64(phi).reshape(R, G)
    return float(lib().orc_fission_rate(C.c_int(R), C.c_int(G), _dp(rm), _dp(nf), _dp(vol), _dp(phi)))


def power_iteration(region_material, sigma_t, sigma_s, nu_sigma_f, chi, polar_sin, polar_weight, seg_offset,
                    seg_region, seg_length, track_weight, link, volume, n_iters, state=None, n_threads=0):
    """O-8.  Returns (k, phi [R][G], psi [T][2][P][G], k_history[n_iters]).  state=(k,phi,psi) resumes."""
    rm, st, ss, nf, ch = _i32(region_material), _f64(sigma_t), _f64(sigma_s), _f64(nu_sigma_f), _f64(chi)
    ps, pw = _f64(polar_sin), _f64(polar_weight)
    so, sr, sl, tw, lk, vol = _i64(seg_offset), _i32(seg_region), _f64(seg_length), _f64(track_weight), _i32(link), _f64(volume)
    R, (M, G), P, T = len(rm), st.shape, len(ps), len(tw)
    if state is None:
        k, phi, psi, resume = C.c_double(1.0), np.empty((R, G)), np.empty((T, 2, P, G)), 0
    else:
        k, phi, psi, resume = C.c_double(state[0]), _f64(state[1]).reshape(R, G).copy(), _f64(state[2]).reshape(T, 2, P, G).copy(), 1
    hist = np.empty(max(n_iters, 1))
    rc = lib().orc_power_iteration(C.c_int(R), C.c_int(M), C.c_int(G), C.c_int(P), C.c_int(T), _dp(rm), _dp(st), _dp(ss),
                                   _dp(nf), _dp(ch), _dp(ps), _dp(pw), _dp(so), _dp(sr), _dp(sl), _dp(tw), _dp(lk),
                                   _dp(vol), C.c_int(n_iters), C.c_int(resume), C.byref(k), _dp(phi), _dp(psi),
                                   _dp(hist), C.c_int(n_threads))
    if rc != 0:
        raise RuntimeError(f"orc_power_iteration failed with code {rc}")
    return k.value, phi, psi, hist[:n_iters]
