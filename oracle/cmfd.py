"""CMFD acceleration of the oracle's power iteration -- TEST INFRASTRUCTURE, FP64, dense.

Algorithm 1 of arxiv/paper_2607_01591 names the steps -- "Perform MOC on the fine mesh", "Solve CMFD
on the coarse mesh", update the fine-mesh flux -- and gives no formula; PAPER.md:129 states the purpose ("enforce global
neutron balance consistency").  The reading used here is the textbook CMFD and is listed in DESIGN.md section 8d
(C-1..C-9); every function below cites its item.  Nothing here is shared with, or imported by, the CUDA path.

Pins (tests/test_oracle_cmfd.py): per-cell telescoping balance of the tallied currents (C-3); the accelerated iteration
converges to the SAME k and flux as the plain O-8 iteration (the CMFD correction vanishes at the fixed point) in several
times fewer sweeps; the homogeneous reflective medium reaches the closed-form k_inf in a handful of sweeps; the coarse
operator returns the tallied currents exactly at the collapsed flux; the coarse eigen-solve against numpy's dense
eigen-decomposition.
"""
import ctypes as C

import numpy as np

from . import _dp, _f64, _i32, _i64, fission_rate, lib, source, sweep


def coarse_surfaces(seg_offset, seg_region, cell, link=None):
    """C-2: the interior surfaces = sorted unique pairs (lo < hi) of coarse cells that consecutive segments of some
    track join, plus the pairs a reflective hand-over joins (exit cell of a chain, entry cell of link[chain]).
    Returns (pair_lo, pair_hi) int32."""
    so, sr, cell = _i64(seg_offset), _i32(seg_region), _i32(cell)
    c = cell[sr]
    same_track = np.ones(len(sr), bool)
    same_track[so[1:-1][so[1:-1] < len(sr)]] = False          # segment k starts a new track: no pair (k-1, k)
    a, b = c[:-1], c[1:]
    keep = same_track[1:] & (a != b)
    lo, hi = np.minimum(a[keep], b[keep]), np.maximum(a[keep], b[keep])
    if link is not None:
        lk = _i32(link).reshape(-1)                               # chain 2t+d -> receiving chain or -1
        nonempty = so[1:] > so[:-1]
        first, last = sr[np.minimum(so[:-1], len(sr) - 1)], sr[np.maximum(so[1:] - 1, 0)]
        exit_cell = np.stack([cell[last], cell[first]], 1).reshape(-1)      # chain (t,0) exits in the last region
        entry_cell = np.stack([cell[first], cell[last]], 1).reshape(-1)
        ok = (lk >= 0) & np.repeat(nonempty, 2)
        a2, b2 = exit_cell[ok], entry_cell[lk[ok]]
        d = a2 != b2
        lo = np.concatenate([lo, np.minimum(a2[d], b2[d])])
        hi = np.concatenate([hi, np.maximum(a2[d], b2[d])])
    pairs = np.unique(np.stack([lo, hi], 1), axis=0) if len(lo) else np.zeros((0, 2), np.int32)
    return np.ascontiguousarray(pairs[:, 0], np.int32), np.ascontiguousarray(pairs[:, 1], np.int32)


def sweep_currents(region_material, sigma_t, polar_sin, polar_weight, seg_offset, seg_region, seg_length, track_weight,
                   link, Q, psi_in, cell, n_cells, pair_lo, pair_hi):
    """C-3 (O-9 of moc_oracle.c): net currents of the sweep that O-6 performs with the same Q and psi_in.
    Returns J_surf [n_pairs][G] (positive from lo to hi), J_vac [n_cells][G], J_ref [n_cells][G] (outward)."""
    rm, st = _i32(region_material), _f64(sigma_t)
    ps, pw = _f64(polar_sin), _f64(polar_weight)
    so, sr, sl, tw, lk = _i64(seg_offset), _i32(seg_region), _f64(seg_length), _f64(track_weight), _i32(link)
    R, (M, G), P, T = len(rm), st.shape, len(ps), len(tw)
    Q, psi_in, cell = _f64(Q).reshape(R, G), _f64(psi_in).reshape(T, 2, P, G), _i32(cell)
    lo, hi = _i32(pair_lo), _i32(pair_hi)
    Js, Jv, Jr = np.empty((len(lo), G)), np.empty((n_cells, G)), np.empty((n_cells, G))
    rc = lib().orc_sweep_currents(C.c_int(R), C.c_int(M), C.c_int(G), C.c_int(P), C.c_int(T), _dp(rm), _dp(st), _dp(ps),
                                  _dp(pw), _dp(so), _dp(sr), _dp(sl), _dp(tw), _dp(lk), _dp(Q), _dp(psi_in),
                                  C.c_int(n_cells), _dp(cell), C.c_int(len(lo)), _dp(lo), _dp(hi), _dp(Js), _dp(Jv), _dp(Jr))
    if rc != 0:
        raise RuntimeError(f"orc_sweep_currents failed with code {rc}")
    return Js, Jv, Jr


def collapse(region_material, sigma_t, sigma_s, nu_sigma_f, chi, volume, phi, cell, n_cells):
    """C-4: flux-volume weighted coarse constants.  Returns dict V [C], Phi [C][G], sigt [C][G], sigs [C][g][g'] (from g'
    into g, as in O-7), nusf [C][G], chi [C][G] (fission-emission weighted)."""
    rm, vol, cell = _i32(region_material), _f64(volume), _i32(cell)
    st, ss, nf, ch = _f64(sigma_t), _f64(sigma_s), _f64(nu_sigma_f), _f64(chi)
    G = st.shape[1]
    phi = _f64(phi).reshape(len(rm), G)
    V = np.zeros(n_cells)
    PhiV = np.zeros((n_cells, G))
    stPhi, nfPhi = np.zeros((n_cells, G)), np.zeros((n_cells, G))
    ssPhi = np.zeros((n_cells, G, G))
    chF, F = np.zeros((n_cells, G)), np.zeros(n_cells)
    for r in range(len(rm)):                                  # plain loop: small cases only
        c, m, a = cell[r], rm[r], vol[r]
        V[c] += a
        PhiV[c] += a * phi[r]
        stPhi[c] += a * st[m] * phi[r]
        nfPhi[c] += a * nf[m] * phi[r]
        ssPhi[c] += a * ss[m] * phi[r][None, :]               # [g][g'] * phi[g']
        f = a * float(nf[m] @ phi[r])
        chF[c] += ch[m] * f
        F[c] += f
    with np.errstate(divide="ignore", invalid="ignore"):
        Phi = PhiV / V[:, None]
        out = dict(V=V, Phi=Phi, sigt=stPhi / PhiV, nusf=nfPhi / PhiV, sigs=ssPhi / PhiV[:, None, :],
                   chi=np.where(F[:, None] > 0, chF / np.where(F > 0, F, 1.0)[:, None], 0.0))
    return out


def coarse_operators(co, pair_lo, pair_hi, coupling, J_surf, J_vac):
    """C-5..C-7: dense loss-minus-scatter matrix A and fission matrix B of the coarse eigenproblem A Phi = (1/k) B Phi,
    unknowns ordered [cell][group]; also returns (Dhat, Dtil) [n_pairs][G] and alpha [C][G]."""
    V, Phi, sigt, sigs, nusf, chi = co["V"], co["Phi"], co["sigt"], co["sigs"], co["nusf"], co["chi"]
    NC, G = Phi.shape
    D = 1.0 / (3.0 * sigt)                                                        # C-5
    lo, hi = np.asarray(pair_lo), np.asarray(pair_hi)
    Dhat = 2.0 * D[lo] * D[hi] / (D[lo] + D[hi]) * np.asarray(coupling, float)[:, None]
    Dtil = -(J_surf + Dhat * (Phi[hi] - Phi[lo])) / (Phi[hi] + Phi[lo])           # C-6
    alpha = J_vac / Phi                                                           # vacuum ends: J = alpha * Phi
    A = np.zeros((NC * G, NC * G))
    B = np.zeros((NC * G, NC * G))
    for c in range(NC):                                                           # C-7, removal, scattering, fission
        for g in range(G):
            i = c * G + g
            A[i, i] += sigt[c, g] * V[c] + alpha[c, g]
            for gp in range(G):
                A[i, c * G + gp] -= sigs[c, g, gp] * V[c]
                B[i, c * G + gp] += chi[c, g] * nusf[c, gp] * V[c]
    for s in range(len(lo)):                                                      # net current lo -> hi
        for g in range(G):
            i, j = lo[s] * G + g, hi[s] * G + g
            out_lo, in_hi = Dhat[s, g] - Dtil[s, g], Dhat[s, g] + Dtil[s, g]      # J = out_lo*Phi_lo - in_hi*Phi_hi
            A[i, i] += out_lo; A[i, j] -= in_hi
            A[j, j] += in_hi;  A[j, i] -= out_lo
    return A, B, Dhat, Dtil, alpha


def coarse_eigen(A, B, Phi0, k0, tol=1e-13, max_outer=100000):
    """C-8: dominant eigenpair of A Phi = (1/k) B Phi by power iteration with an exact (dense) inner solve, started
    from the collapsed flux; Phi is returned with the fission production of Phi0."""
    x = Phi0.reshape(-1).copy()
    k = float(k0)
    P0 = float(np.sum(B @ x))
    lu = np.linalg.inv(A)
    for _ in range(max_outer):
        f = B @ x
        y = lu @ (f / k)
        k_new = k * float(np.sum(B @ y)) / float(np.sum(f))
        y *= P0 / float(np.sum(B @ y))
        done = abs(k_new - k) < tol * abs(k_new) and np.max(np.abs(y - x)) < 1e-11 * np.max(np.abs(y))
        x, k = y, k_new
        if done:
            break
    return k, x.reshape(Phi0.shape)


def power_iteration_cmfd(region_material, sigma_t, sigma_s, nu_sigma_f, chi, polar_sin, polar_weight, seg_offset,
                         seg_region, seg_length, track_weight, link, volume, cell, n_cells, coupling_of_pair, n_iters,
                         state=None, accelerate=True, tol_k=0.0):
    """O-8 with the CMFD step C-1..C-9 after every sweep (accelerate=False: the same loop without it, i.e. O-8).
    coupling_of_pair(lo, hi) -> A_s / d_s per interior surface (C-5).  Returns (k, phi, psi, k_history)."""
    rm, st = _i32(region_material), _f64(sigma_t)
    R, (M, G), P, T = len(rm), st.shape, len(polar_sin), len(track_weight)
    so, sr = _i64(seg_offset), _i32(seg_region)
    cell = _i32(cell)
    lo, hi = coarse_surfaces(so, sr, cell, link)
    coupling = np.asarray(coupling_of_pair(lo, hi), float)
    first = np.where(so[1:] > so[:-1], sr[np.minimum(so[:-1], len(sr) - 1)], 0)
    last = np.where(so[1:] > so[:-1], sr[np.maximum(so[1:] - 1, 0)], 0)
    entry_cell = np.stack([cell[first], cell[last]], 1)       # C-9: cell where direction d of track t enters
    if state is None:
        k, phi, psi = 1.0, np.ones((R, G)), np.zeros((T, 2, P, G))
    else:
        k, phi, psi = float(state[0]), _f64(state[1]).reshape(R, G).copy(), _f64(state[2]).reshape(T, 2, P, G).copy()
    hist = []
    for _ in range(n_iters):
        F_old = fission_rate(rm, nu_sigma_f, volume, phi)
        phi, psi = phi / F_old, psi / F_old
        Q = source(rm, sigma_s, nu_sigma_f, chi, phi, k)
        phi_new, psi_next, _ = sweep(rm, st, polar_sin, polar_weight, so, sr, seg_length, track_weight, link, volume, Q, psi)
        k_new = k * fission_rate(rm, nu_sigma_f, volume, phi_new)
        if accelerate:
            Js, Jv, _ = sweep_currents(rm, st, polar_sin, polar_weight, so, sr, seg_length, track_weight, link, Q, psi,
                                       cell, n_cells, lo, hi)
            co = collapse(rm, st, sigma_s, nu_sigma_f, chi, volume, phi_new, cell, n_cells)
            A, B, _, _, _ = coarse_operators(co, lo, hi, coupling, Js, Jv)
            k_new, Phi_new = coarse_eigen(A, B, co["Phi"], k_new)
            ratio = Phi_new / co["Phi"]                        # C-9: prolongation of phi and of the boundary flux
            phi_new = phi_new * ratio[cell]
            psi_next = psi_next * ratio[entry_cell][:, :, None, :]
        dk = abs(k_new - k)
        k, phi, psi = k_new, phi_new, psi_next
        hist.append(k)
        if tol_k > 0.0 and dk < tol_k:
            break
    return k, phi, psi, np.array(hist)
