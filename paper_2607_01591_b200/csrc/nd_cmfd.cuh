// nd_cmfd.cuh -- NEXT-3 (CMFD, Algorithm 1), step C-3 of DESIGN.md 8d: the net currents of one sweep
// through the surfaces of a coarse mesh.  First CUDA step of that row: the simple (atomic) sweep with crossings tallied.
//   k_reduced_q       q = (float)(Q / Sigma_t), the reduced source the sweep kernels read
//   k_link_forward    inverts the gather-form link table: fwd[src[e]] = e  (exit of chain src[e] feeds entry e)
//   k_entry_cell      coarse cell of the first region of every chain (t, d)
//   k_sweep_currents  Eq. (5) per (track, direction, polar, group) as in k_sweep_atomic; instead of the
//                     region tally it adds +-w psi at every change of coarse cell (C-3) and the end terms of C-3
//   k_cmfd_accumulate C-4: Psi[c][m][g] = sum over the regions r of cell c with material m of A~_r phi[r][g], V[c]
//   k_cmfd_constants  C-4: the flux-volume weighted coarse constants from Psi (every sum over regions is a sum over m)
//   k_cmfd_prolong_*  C-9: phi[r][g] *= ratio[cell[r]][g]; boundary psi of chain (t, d) *= ratio[cell it enters][g]
//   k_coarse_*        C-5..C-8: dense coarse operator A (removal - scatter + alpha + Dhat -+ Dtil couplings), its inverse by
//                     in-place Gauss-Jordan (no pivoting: A is a diagonally dominant M-matrix-like operator), and the
//                     power iteration A Phi = (1/k) B Phi with B = chi (nuSigma_f V)^T applied cell by cell
#pragma once
#include "nd_kernels.cuh"

namespace ndk {

__global__ void __launch_bounds__(256) k_reduced_q(const double* __restrict__ Q, const int32_t* __restrict__ reg_mat,
                                                   const double* __restrict__ sigt, float* __restrict__ q, int64_t R,
                                                   int G, int Gs)
{
    const int64_t n = R * Gs;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t r = i / Gs;
        const int g = (int)(i - r * Gs);
        q[i] = g < G ? (float)(Q[r * G + g] / sigt[(size_t)reg_mat[r] * G + g]) : 0.f;
    }
}

__global__ void __launch_bounds__(256) k_link_forward(const int32_t* __restrict__ src, int32_t* __restrict__ fwd,
                                                      int64_t n_entries)
{
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n_entries; e += (int64_t)gridDim.x * blockDim.x)
        if (src[e] >= 0) fwd[src[e]] = (int32_t)e;
}

__global__ void __launch_bounds__(256) k_entry_cell(const uint32_t* __restrict__ seg_rm, const int64_t* __restrict__ trk_off,
                                                    const int32_t* __restrict__ cell, int32_t* __restrict__ entry_cell,
                                                    int64_t n_entries)
{
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n_entries; e += (int64_t)gridDim.x * blockDim.x) {
        const int64_t t = e >> 1;
        const int64_t k0 = trk_off[t], k1 = trk_off[t + 1];
        // the padding records at the end of a run repeat its last region, so k1 - 1 is the entry of direction 1
        entry_cell[e] = k1 == k0 ? -1 : cell[rm_region(seg_rm[(e & 1) ? k1 - 1 : k0])];
    }
}

struct CurrentParams {
    SweepParams sw;                        // stream, q, Sigma_t, psi_in, polar tables (tally and psi_out are not touched)
    const int32_t* __restrict__ cell;      // [R] coarse cell of a region
    const int32_t* __restrict__ link_fwd;  // [2T] entry that the exit of chain e feeds, -1 = vacuum
    const int32_t* __restrict__ entry_cell;// [2T]
    const int64_t* __restrict__ pair_key;  // [n_pairs] sorted lo * n_cells + hi
    const int32_t* __restrict__ pair_idx;  // [n_pairs] the caller's index of the sorted key
    double* __restrict__ J_surf;           // [n_pairs][G], positive from lo to hi
    double* __restrict__ J_vac;            // [n_cells][G]
    double* __restrict__ J_ref;            // [n_cells][G]
    int* __restrict__ missing;             // set when a crossing joins a pair that is not listed
    int n_pairs, n_cells;
    int lanes_per_chain;                   // power of two, min(32, >= G)
};

__device__ __forceinline__ int find_surface(const CurrentParams& cp, int a, int b)
{
    const int64_t key = (int64_t)(a < b ? a : b) * cp.n_cells + (a < b ? b : a);
    int l = 0, h = cp.n_pairs - 1;
    while (l <= h) {
        const int m = (l + h) >> 1;
        const int64_t v = cp.pair_key[m];
        if (v < key) l = m + 1;
        else if (v > key) h = m - 1;
        else return cp.pair_idx[m];
    }
    return -1;
}

// One chain (track, direction) per group of lanes_per_chain lanes, lanes over groups (the layout of k_sweep_atomic, with
// 32 / lanes_per_chain chains to a warp when G <= 16).  The cell of a segment and the surface search are uniform within
// a chain's lanes; the kernel uses no warp-wide primitive, so chains of different lengths may share a warp.
// NG = groups a lane carries through one walk (2 when G > 32: the walk of a chain is then done once for 64 groups).
template <int P, int EXPM, int NG>
__global__ void __launch_bounds__(256) k_sweep_currents(const CurrentParams cp)
{
    const SweepParams& prm = cp.sw;
    const int lpc = cp.lanes_per_chain;              // 32 / lpc chains share a warp when G <= 16
    const int lane = threadIdx.x % lpc;
    const int chains_per_block = blockDim.x / lpc;
    const int64_t n_chains = 2 * (int64_t)prm.T;
    const float inv_f = (float)(1.0 / *prm.scale_div);
    for (int64_t chain = (int64_t)blockIdx.x * chains_per_block + threadIdx.x / lpc; chain < n_chains;
         chain += (int64_t)gridDim.x * chains_per_block) {
        const int t = (int)(chain >> 1), dir = (int)(chain & 1);
        const int64_t k0 = prm.trk_off[t], k1 = prm.trk_off[t + 1];
        if (k1 == k0) continue;
        const float wt = prm.trk_w[t];
        const int32_t lk = cp.link_fwd[chain];
        const int32_t c2 = lk >= 0 ? cp.entry_cell[lk] : -1;
        for (int g0 = lane; g0 < prm.G; g0 += lpc * NG) {
            float psi[NG][P];
            int g[NG];
            bool act[NG];
#pragma unroll
            for (int j = 0; j < NG; ++j) {
                act[j] = g0 + j * lpc < prm.G;
                g[j] = act[j] ? g0 + j * lpc : g0;   // an idle slot repeats group g0 and adds nothing
#pragma unroll
                for (int p = 0; p < P; ++p) psi[j][p] = prm.psi_in[(chain * P + p) * prm.Gs + g[j]] * inv_f;
            }
            int c_prev = -1;
            for (int64_t i = 0; i < k1 - k0; ++i) {
                const int64_t k = dir == 0 ? k0 + i : k1 - 1 - i;
                const uint32_t rm = prm.seg_rm[k];
                const float s = prm.seg_len[k];
                const uint32_t r = rm_region(rm);
                const int c = cp.cell[r];
                if (c_prev >= 0 && c != c_prev) {
                    const int sidx = find_surface(cp, c_prev, c);
                    if (sidx < 0) {
                        *cp.missing = 1;
                    } else {
#pragma unroll
                        for (int j = 0; j < NG; ++j) {
                            float cur = 0.f;
#pragma unroll
                            for (int p = 0; p < P; ++p) cur = fmaf(prm.wp[p], psi[j][p], cur);
                            const double jj = (double)wt * (double)cur;
                            if (act[j]) atomicAdd(&cp.J_surf[(size_t)sidx * prm.G + g[j]], c_prev < c ? jj : -jj);
                        }
                    }
                }
#pragma unroll
                for (int j = 0; j < NG; ++j) {
                    const float st = prm.sigt[rm_material(rm) * prm.Gs + g[j]];
                    const float qv = prm.q[(size_t)r * prm.Gs + g[j]];
                    attenuate<P, EXPM>(psi[j], qv, st * s, prm);
                }
                c_prev = c;
            }
            // chain end (C-3): what leaves minus what the opposite direction brings in at this end
            const int sidx2 = lk >= 0 && c2 != c_prev ? (c2 >= 0 ? find_surface(cp, c_prev, c2) : -1) : -2;
            if (sidx2 == -1) *cp.missing = 1;
#pragma unroll
            for (int j = 0; j < NG; ++j) {
                if (!act[j]) continue;
                float out = 0.f, net = 0.f;
#pragma unroll
                for (int p = 0; p < P; ++p) {
                    const float back = prm.psi_in[((chain ^ 1) * P + p) * prm.Gs + g[j]] * inv_f;
                    out = fmaf(prm.wp[p], psi[j][p], out);
                    net = fmaf(prm.wp[p], psi[j][p] - back, net);
                }
                double* J = lk < 0 ? cp.J_vac : cp.J_ref;
                atomicAdd(&J[(size_t)c_prev * prm.G + g[j]], (double)wt * (double)net);
                if (sidx2 >= 0) {   // reflective hand-over into another coarse cell: a surface crossing
                    const double jj = (double)wt * (double)out;
                    atomicAdd(&cp.J_surf[(size_t)sidx2 * prm.G + g[j]], c_prev < c2 ? jj : -jj);
                    atomicAdd(&cp.J_ref[(size_t)c_prev * prm.G + g[j]], -jj);
                    atomicAdd(&cp.J_ref[(size_t)c2 * prm.G + g[j]], jj);
                }
            }
        }
    }
}

// ---- C-4, pass 1: thread per (r, g) ----
__global__ void __launch_bounds__(256) k_cmfd_accumulate(const double* __restrict__ phi, const double* __restrict__ vol,
                                                         const int32_t* __restrict__ reg_mat, const int32_t* __restrict__ cell,
                                                         double* __restrict__ Psi, double* __restrict__ V, int64_t R, int G, int M)
{
    const int64_t n = R * G;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t r = i / G;
        const int g = (int)(i - r * G);
        const int c = cell[r];
        const double a = vol[r];
        atomicAdd(&Psi[((size_t)c * M + reg_mat[r]) * G + g], a * phi[i]);
        if (g == 0) atomicAdd(&V[c], a);
    }
}

// ---- C-4, pass 2: thread per (c, g).  out = [Phi | sigt | nusf | chi] each [C][G], then sigs [C][g][g'] ----
__global__ void __launch_bounds__(128) k_cmfd_constants(const double* __restrict__ Psi, const double* __restrict__ V,
                                                        const double* __restrict__ sigt, const double* __restrict__ sigsT,
                                                        const double* __restrict__ nusf, const double* __restrict__ chi,
                                                        double* __restrict__ out, int C, int G, int M)
{
    const int64_t n = (int64_t)C * G;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int c = (int)(i / G), g = (int)(i - (int64_t)c * G);
        const double* psi_c = Psi + (size_t)c * M * G;
        double phiV = 0.0, stPhi = 0.0, nfPhi = 0.0, chF = 0.0, F = 0.0;
        for (int m = 0; m < M; ++m) {
            const double x = psi_c[(size_t)m * G + g];
            phiV += x;
            stPhi += sigt[(size_t)m * G + g] * x;
            nfPhi += nusf[(size_t)m * G + g] * x;
            double f = 0.0;                                   // fission emission of material m in cell c
            for (int gp = 0; gp < G; ++gp) f += nusf[(size_t)m * G + gp] * psi_c[(size_t)m * G + gp];
            chF += chi[(size_t)m * G + g] * f;
            F += f;
        }
        out[i] = phiV / V[c];
        out[n + i] = stPhi / phiV;
        out[2 * n + i] = nfPhi / phiV;
        out[3 * n + i] = F > 0.0 ? chF / F : 0.0;
        double* sigs = out + 4 * n + (size_t)i * G;           // row g of cell c: from g' into g
        for (int gp = 0; gp < G; ++gp) {
            double ss = 0.0, pv = 0.0;
            for (int m = 0; m < M; ++m) {
                const double x = psi_c[(size_t)m * G + gp];
                ss += sigsT[((size_t)m * G + gp) * G + g] * x;
                pv += x;
            }
            sigs[gp] = ss / pv;
        }
    }
}

// ---- C-9 ----
__global__ void __launch_bounds__(256) k_cmfd_prolong_phi(double* __restrict__ phi, const int32_t* __restrict__ cell,
                                                          const double* __restrict__ ratio, int64_t R, int G)
{
    const int64_t n = R * G;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t r = i / G;
        phi[i] *= ratio[(size_t)cell[r] * G + (i - r * G)];
    }
}

// psi [2T][P][Gs] FP32; entry_region[e] = first region of chain e (-1: empty track)
__global__ void __launch_bounds__(256) k_cmfd_prolong_psi(float* __restrict__ psi, const int32_t* __restrict__ entry_region,
                                                          const int32_t* __restrict__ cell, const double* __restrict__ ratio,
                                                          int64_t n_entries, int P, int G, int Gs)
{
    const int64_t PG = (int64_t)P * Gs, n = n_entries * PG;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t e = i / PG;
        const int g = (int)((i - e * PG) % Gs);
        const int32_t r = entry_region[e];
        if (r >= 0 && g < G) psi[i] = (float)((double)psi[i] * ratio[(size_t)cell[r] * G + g]);
    }
}

// ---- C-5..C-7: the dense coarse operator, unknowns ordered [cell][group], n = C G ----
struct CoarseParams {
    const double* __restrict__ V;      // [C]
    const double* __restrict__ Phi;    // [C][G]
    const double* __restrict__ sigt;   // [C][G]
    const double* __restrict__ sigs;   // [C][g][g']
    const double* __restrict__ nusf;   // [C][G]
    const double* __restrict__ chi;    // [C][G]
    const double* __restrict__ J_vac;  // [C][G]
    const int32_t* __restrict__ lo;    // [S]
    const int32_t* __restrict__ hi;    // [S]
    const double* __restrict__ coupling; // [S] A_s / d_s
    const double* __restrict__ J_surf; // [S][G]
    double* __restrict__ A;            // [n][n], zeroed by the caller
    int C, G, S;
};

__global__ void __launch_bounds__(256) k_coarse_cell_blocks(const CoarseParams cp)
{
    const int G = cp.G;
    const int64_t n = (int64_t)cp.C * G, total = n * G;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t row = i / G;                 // c G + g
        const int gp = (int)(i - row * G);
        const int c = (int)(row / G), g = (int)(row - (int64_t)c * G);
        double v = -cp.sigs[i] * cp.V[c];
        if (gp == g) v += cp.sigt[row] * cp.V[c] + cp.J_vac[row] / cp.Phi[row];   // removal + vacuum ends (alpha, C-6)
        cp.A[row * n + (int64_t)c * G + gp] = v;
    }
}

__global__ void __launch_bounds__(256) k_coarse_surfaces(const CoarseParams cp)
{
    const int G = cp.G;
    const int64_t n = (int64_t)cp.C * G, total = (int64_t)cp.S * G;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
        const int s = (int)(i / G), g = (int)(i - (int64_t)s * G);
        const int64_t a = (int64_t)cp.lo[s] * G + g, b = (int64_t)cp.hi[s] * G + g;
        const double Da = 1.0 / (3.0 * cp.sigt[a]), Db = 1.0 / (3.0 * cp.sigt[b]);                 // C-5
        const double Dhat = 2.0 * Da * Db / (Da + Db) * cp.coupling[s];
        const double Dtil = -(cp.J_surf[i] + Dhat * (cp.Phi[b] - cp.Phi[a])) / (cp.Phi[b] + cp.Phi[a]);   // C-6
        const double out_lo = Dhat - Dtil, in_hi = Dhat + Dtil;                                     // J = out_lo Phi_lo - in_hi Phi_hi
        atomicAdd(&cp.A[a * n + a], out_lo);
        atomicAdd(&cp.A[a * n + b], -in_hi);
        atomicAdd(&cp.A[b * n + b], in_hi);
        atomicAdd(&cp.A[b * n + a], -out_lo);
    }
}

// ---- in-place Gauss-Jordan inverse, pivot p: (1) save column p and the scaled pivot row, (2) rank-1 update ----
__global__ void __launch_bounds__(256) k_gj_prepare(const double* __restrict__ A, double* __restrict__ col,
                                                    double* __restrict__ row, int64_t n, int64_t p)
{
    const double inv = 1.0 / A[p * n + p];
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        col[i] = A[i * n + p];
        row[i] = i == p ? inv : A[p * n + i] * inv;
    }
}

__global__ void __launch_bounds__(256) k_gj_update(double* __restrict__ A, const double* __restrict__ col,
                                                   const double* __restrict__ row, int64_t n, int64_t p)
{
    const int64_t total = n * n;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < total; k += (int64_t)gridDim.x * blockDim.x) {
        const int64_t i = k / n, j = k - i * n;
        A[k] = i == p ? row[j] : (j == p ? 0.0 : A[k]) - col[i] * row[j];
    }
}

// ---- C-8: f = B x, with B[(c,g),(c,g')] = chi[c][g] nuSigma_f[c][g'] V[c] ----
__global__ void __launch_bounds__(256) k_coarse_fission(const double* __restrict__ x, const double* __restrict__ V,
                                                        const double* __restrict__ nusf, const double* __restrict__ chi,
                                                        double* __restrict__ f, int C, int G, const int* __restrict__ done)
{
    if (done && *done) return;
    const int64_t n = (int64_t)C * G;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int c = (int)(i / G);
        double e = 0.0;
        for (int gp = 0; gp < G; ++gp) e += nusf[(size_t)c * G + gp] * x[(size_t)c * G + gp];
        f[i] = chi[i] * V[c] * e;
    }
}

// y = Ainv f, one warp per row
__global__ void __launch_bounds__(256) k_coarse_matvec(const double* __restrict__ Ainv, const double* __restrict__ f,
                                                       double* __restrict__ y, int64_t n, const int* __restrict__ done)
{
    if (*done) return;
    const int lane = threadIdx.x & 31;
    for (int64_t r = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5; r < n; r += ((int64_t)gridDim.x * blockDim.x) >> 5) {
        double acc = 0.0;
        for (int64_t j = lane; j < n; j += 32) acc += Ainv[r * n + j] * f[j];
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
        if (lane == 0) y[r] = acc;
    }
}

// One block.  With y' = Ainv f (= k times the oracle's y): k_new = sum(B y') / sum(f); x_new = y' P0 / sum(B y');
// converged when |k_new - k| < tol |k_new| and max |x_new - x| < 1e-11 max |x_new| (the oracle's test).
// state: [0] k, [1] P0 (sum B x0; set by the first call when init != 0).
__global__ void __launch_bounds__(1024) k_coarse_update(double* __restrict__ x, const double* __restrict__ y,
                                                        const double* __restrict__ f, const double* __restrict__ V, const double* __restrict__ nusf,
                                                        const double* __restrict__ chi, double* __restrict__ state,
                                                        int* __restrict__ done, int* __restrict__ iters, int C, int G,
                                                        double tol, int init)
{
    __shared__ double scratch[32];
    __shared__ double bc[2];                        // block_sum / block_max leave their result in thread 0 only
    if (*done) return;
    const int64_t n = (int64_t)C * G;
    double sf = 0.0;
    for (int64_t i = threadIdx.x; i < n; i += blockDim.x) sf += f[i];
    sf = block_sum(sf, scratch);
    if (init) {                                     // P0 = sum(B x0) = sum(f) of the first product
        if (threadIdx.x == 0) state[1] = sf;
        return;
    }
    double sby = 0.0;
    for (int64_t i = threadIdx.x; i < n; i += blockDim.x) {
        const int c = (int)(i / G);
        double e = 0.0;
        for (int gp = 0; gp < G; ++gp) e += nusf[(size_t)c * G + gp] * y[(size_t)c * G + gp];
        sby += chi[i] * V[c] * e;
    }
    sby = block_sum(sby, scratch);
    if (threadIdx.x == 0) { bc[0] = sf; bc[1] = sby; }
    __syncthreads();
    sf = bc[0]; sby = bc[1];
    const double k_old = state[0], k_new = sby / sf, scale = state[1] / sby;
    double dmax = 0.0, ymax = 0.0;
    for (int64_t i = threadIdx.x; i < n; i += blockDim.x) {
        const double v = y[i] * scale;
        dmax = fmax(dmax, fabs(v - x[i]));
        ymax = fmax(ymax, fabs(v));
        x[i] = v;
    }
    dmax = block_max(dmax, scratch);
    ymax = block_max(ymax, scratch);
    __syncthreads();                                // every thread has read state[0] before it is replaced
    if (threadIdx.x == 0) {
        state[0] = k_new;
        ++*iters;
        if (fabs(k_new - k_old) < tol * fabs(k_new) && dmax < 1e-11 * ymax) *done = 1;
    }
}

} // namespace ndk
