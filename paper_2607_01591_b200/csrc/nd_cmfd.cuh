// nd_cmfd.cuh -- NEXT-3 (CMFD, Algorithm 1), the device side of steps C-3..C-9 of DESIGN.md 8d.
// The surface crossings of C-3 are tallied inside the sweep kernel (nd_sweep_swath.cuh, CUR = 1); here:
//   k_link_forward     inverts the gather-form link table: fwd[src[e]] = e  (exit of chain src[e] feeds entry e)
//   k_end_currents     C-3, the chain ends: J_vac / J_ref and the reflective hand-over into another coarse cell
//   k_cmfd_accumulate  C-4: Psi[c][m][g] = sum over the regions r of cell c with material m of A~_r phi[r][g], V[c]
//   k_cmfd_constants   C-4: the flux-volume weighted coarse constants from Psi (every sum over regions is a sum over m)
//   k_coarse_solve     C-5..C-8: ONE cooperative kernel: Dhat / Dtil per surface, the G x G diagonal block of every cell
//                      inverted with partial pivoting, and the dominant eigenpair of A Phi = (1/k) B Phi by fission-source
//                      iteration with block-Jacobi inner sweeps; no host interaction until it has converged
//   k_cmfd_prolong_*   C-9: phi[r][g] *= ratio[cell[r]][g]; boundary psi of chain (t, d) *= ratio[cell it enters][g]
#pragma once
#include <cooperative_groups.h>

#include "nd_kernels.cuh"

namespace ndk {

__global__ void __launch_bounds__(256) k_link_forward(const int32_t* __restrict__ src, int32_t* __restrict__ fwd,
                                                      int64_t n_entries)
{
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n_entries; e += (int64_t)gridDim.x * blockDim.x)
        if (src[e] >= 0) fwd[src[e]] = (int32_t)e;
}

// Sorted surface keys lo * n_cells + hi -> the caller's surface index; -1 if the pair is not a listed surface.
__device__ __forceinline__ int find_surface(const int64_t* __restrict__ pair_key, const int32_t* __restrict__ pair_idx, int n_pairs,
                                            int n_cells, int a, int b)
{
    const int64_t key = (int64_t)(a < b ? a : b) * n_cells + (a < b ? b : a);
    int l = 0, h = n_pairs - 1;
    while (l <= h) {
        const int m = (l + h) >> 1;
        const int64_t v = pair_key[m];
        if (v < key) l = m + 1;
        else if (v > key) h = m - 1;
        else return pair_idx[m];
    }
    return -1;
}

// ---- C-3, chain ends (run between the sweep and the link swap).  Thread per (chain e = 2t+d, group g).
// At the exit of chain e: w (psi_exit - psi_in of the opposite direction at this end) into J_vac[cell of the end] at a vacuum end,
// J_ref at a reflective one; a hand-over into another cell c2 also adds +-w psi_exit to that surface and moves w psi_exit
// from J_ref[c] to J_ref[c2].  entry_cell[e] = coarse cell of the first region of chain e (-1: empty track): chain e ends where
// chain e^1 begins. ----
struct EndCurrentParams {
    const float* __restrict__ psi_in;       // [2T][P][Gs] what entered (used as psi_in / F)
    const float* __restrict__ psi_out;      // [2T][P][Gs] what left
    const float* __restrict__ trk_w;        // [T]
    const int32_t* __restrict__ link_fwd;   // [2T] entry fed by the exit of chain e, -1 = vacuum
    const int32_t* __restrict__ entry_cell; // [2T]
    const int64_t* __restrict__ pair_key;   // [n_pairs] sorted
    const int32_t* __restrict__ pair_idx;   // [n_pairs]
    const double* __restrict__ scale_div;
    double* __restrict__ J_surf;            // [n_pairs][G]   } of replica 0; a block adds into replica blockIdx.x % J_replicas
    double* __restrict__ J_vac;             // [n_cells][G]   } (J_stride doubles apart): few addresses, many chains
    double* __restrict__ J_ref;             // [n_cells][G]   }
    long long J_stride;
    int J_replicas;
    int* __restrict__ missing;              // set when a hand-over joins two cells that are not a listed surface
    int64_t n_entries;
    int P, G, Gs, n_pairs, n_cells;
    float wp[kMaxPolar];
};

__global__ void __launch_bounds__(256) k_end_currents(const EndCurrentParams ep)
{
    const int64_t n = ep.n_entries * ep.G;
    const double inv_f = 1.0 / *ep.scale_div;
    const size_t rep = (size_t)(blockIdx.x % ep.J_replicas) * ep.J_stride;
    double* const J_surf = ep.J_surf + rep;
    double* const J_vac = ep.J_vac + rep;
    double* const J_ref = ep.J_ref + rep;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t e = i / ep.G;
        const int g = (int)(i - e * ep.G);
        const int c = ep.entry_cell[e ^ 1];
        if (c < 0) continue;                                   // empty track
        const double wt = (double)ep.trk_w[e >> 1];
        double out = 0.0, back = 0.0;
        for (int p = 0; p < ep.P; ++p) {
            out += (double)ep.wp[p] * (double)ep.psi_out[(e * ep.P + p) * ep.Gs + g];
            back += (double)ep.wp[p] * (double)ep.psi_in[((e ^ 1) * ep.P + p) * ep.Gs + g] * inv_f;
        }
        out *= wt; back *= wt;
        const int32_t lk = ep.link_fwd[e];
        atomicAdd((lk < 0 ? J_vac : J_ref) + (size_t)c * ep.G + g, out - back);
        if (lk >= 0) {
            const int c2 = ep.entry_cell[lk];
            if (c2 >= 0 && c2 != c) {
                const int s = find_surface(ep.pair_key, ep.pair_idx, ep.n_pairs, ep.n_cells, c, c2);
                if (s < 0) { *ep.missing = 1; continue; }
                atomicAdd(J_surf + (size_t)s * ep.G + g, c < c2 ? out : -out);
                atomicAdd(J_ref + (size_t)c * ep.G + g, -out);
                atomicAdd(J_ref + (size_t)c2 * ep.G + g, out);
            }
        }
    }
}

// replica 0 += replicas 1 .. K-1 (fixed order: deterministic given the replicas)
__global__ void __launch_bounds__(256) k_cmfd_reduce_replicas(double* __restrict__ J, long long stride, int K, long long n)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        double s = J[i];
        for (int k = 1; k < K; ++k) s += J[(size_t)k * stride + i];
        J[i] = s;
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

// ---- C-9.  ratio[c][g] = 1 + relax (Phi_new / Phi_old - 1) when the coarse solve succeeded (state[ST_OK] != 0), else 1:
// the prolongation of a failed solve leaves the plain iteration's state untouched. ----
enum { ST_K = 0, ST_P0 = 1, ST_SBY = 2, ST_SAY = 3, ST_DMAX = 4, ST_XMAX = 5, ST_OK = 6, ST_ITERS = 7, ST_KPREV = 8, ST_DONE = 9, ST_COUNT = 16 };

__global__ void __launch_bounds__(256) k_cmfd_ratio(const double* __restrict__ Phi_new, const double* __restrict__ Phi,
                                                    const double* __restrict__ state, double relax, double* __restrict__ ratio,
                                                    double* __restrict__ k_state /* the problem's k, or NULL */, int64_t n)
{
    const bool ok = state[ST_OK] != 0.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        ratio[i] = ok ? 1.0 + relax * (Phi_new[i] / Phi[i] - 1.0) : 1.0;
    if (k_state && ok && blockIdx.x == 0 && threadIdx.x == 0) *k_state = state[ST_K];
}

__global__ void __launch_bounds__(256) k_cmfd_prolong_phi(double* __restrict__ phi, const int32_t* __restrict__ cell,
                                                          const double* __restrict__ ratio, int64_t R, int G)
{
    const int64_t n = R * G;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t r = i / G;
        phi[i] *= ratio[(size_t)cell[r] * G + (i - r * G)];
    }
}

// psi [2T][P][Gs] FP32; entry_cell[e] = coarse cell of the first region of chain e (-1: empty track)
__global__ void __launch_bounds__(256) k_cmfd_prolong_psi(float* __restrict__ psi, const int32_t* __restrict__ entry_cell,
                                                          const double* __restrict__ ratio, int64_t n_entries, int P, int G, int Gs)
{
    const int64_t PG = (int64_t)P * Gs, n = n_entries * PG;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t e = i / PG;
        const int g = (int)((i - e * PG) % Gs);
        const int32_t c = entry_cell[e];
        if (c >= 0 && g < G) psi[i] = (float)((double)psi[i] * ratio[(size_t)c * G + g]);
    }
}

// ---- C-5..C-8 in one cooperative kernel ----
// Unknowns x[c][g].  Per surface s = (lo, hi) and group: D = 1 / (3 Sigma_t), Dhat = 2 D_lo D_hi / (D_lo + D_hi) coupling_s,
// Dtil = -(J_s + Dhat (Phi_hi - Phi_lo)) / (Phi_hi + Phi_lo); net current lo -> hi = out_lo x_lo - in_hi x_hi with
// out_lo = Dhat - Dtil, in_hi = Dhat + Dtil.  Loss operator A = M (G x G block per cell: removal + alpha + its surfaces' out-flow
// on the diagonal, minus in-scatter) - N (what flows in from the neighbours); fission operator B = chi V nuSigma_f^T per cell.
// Iteration: f = B x / k;  y <- M^-1 (f + N y), `inner` block-Jacobi sweeps from y = x;  k = sum(B y) / sum(A y) (the global
// balance; the coupling terms cancel in the sum);  x = y P0 / sum(B y).  The eigenpair is a fixed point for any `inner`.
struct CoarseSolveParams {
    const double* __restrict__ V;        // [C]
    const double* __restrict__ Phi;      // [C][G] collapsed flux (start vector, and the flux Dtil / alpha are formed with)
    const double* __restrict__ sigt;     // [C][G]
    const double* __restrict__ sigs;     // [C][g][g']
    const double* __restrict__ nusf;     // [C][G]
    const double* __restrict__ chi;      // [C][G]
    const double* __restrict__ J_surf;   // [S][G]
    const double* __restrict__ J_vac;    // [C][G]
    const int32_t* __restrict__ lo;      // [S]
    const int32_t* __restrict__ hi;      // [S]
    const double* __restrict__ coupling; // [S]
    const int32_t* __restrict__ adj_off; // [C+1]
    const int32_t* __restrict__ adj_ent; // [2S] surface << 1 | (1 if the cell is the surface's hi side)
    double* __restrict__ out_lo;         // [S][G] scratch
    double* __restrict__ in_hi;          // [S][G] scratch
    double* __restrict__ Mw;             // [C][G][G] scratch: the block, destroyed by the elimination
    double* __restrict__ Minv;           // [C][G][G]
    double* __restrict__ x;              // [C][G] result (Phi_new, normalised to the fission production of Phi)
    double* __restrict__ y;              // [C][G] scratch
    double* __restrict__ y2;             // [C][G] scratch
    double* __restrict__ f;              // [C][G] scratch
    double* __restrict__ state;          // [ST_COUNT]
    const double* __restrict__ k0;       // start eigenvalue (device scalar)
    int C, G, S, max_outer, inner;
    int single_block;                    // 1: launched as ONE thread block (small systems): block barriers instead of grid syncs
    double tol_k, tol_x;
    double rel_tol;                      // > 0: also stop once max |dx| has fallen to rel_tol x its value in the first iteration
};

__device__ __forceinline__ double warp_sum(double v)
{
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_max(double v)
{
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ void atomic_max_pos(double* addr, double v)   // v >= 0: the bit pattern is monotone
{
    atomicMax(reinterpret_cast<unsigned long long*>(addr), (unsigned long long)__double_as_longlong(v));
}

struct GridOrBlockSync {            // grid-wide barrier of a cooperative launch, or the block barrier of a one-block launch
    cooperative_groups::grid_group g;
    bool single;
    __device__ __forceinline__ void sync() { if (single) __syncthreads(); else g.sync(); }
};

__global__ void __launch_bounds__(1024) k_coarse_solve(const CoarseSolveParams cp)
{
    namespace cg = cooperative_groups;
    GridOrBlockSync grid{cg::this_grid(), cp.single_block != 0};
    const int C = cp.C, G = cp.G, S = cp.S, tid = threadIdx.x, nthr = blockDim.x;
    const int64_t n = (int64_t)C * G, gtid = (int64_t)blockIdx.x * nthr + tid, gn = (int64_t)gridDim.x * nthr;
    const int lane = tid & 31;

    // ---- phase 0: surface coefficients, state ----
    for (int64_t i = gtid; i < (int64_t)S * G; i += gn) {
        const int s = (int)(i / G), g = (int)(i - (int64_t)s * G);
        const int64_t a = (int64_t)cp.lo[s] * G + g, b = (int64_t)cp.hi[s] * G + g;
        const double Da = 1.0 / (3.0 * cp.sigt[a]), Db = 1.0 / (3.0 * cp.sigt[b]);
        const double Dhat = 2.0 * Da * Db / (Da + Db) * cp.coupling[s];
        const double Dtil = -(cp.J_surf[i] + Dhat * (cp.Phi[b] - cp.Phi[a])) / (cp.Phi[b] + cp.Phi[a]);
        cp.out_lo[i] = Dhat - Dtil;
        cp.in_hi[i] = Dhat + Dtil;
    }
    if (gtid == 0) {
        for (int i = 0; i < ST_COUNT; ++i) cp.state[i] = 0.0;
        cp.state[ST_K] = *cp.k0;
    }
    grid.sync();

    // ---- phase 1: M_c and its inverse: Gauss-Jordan with partial pivoting on [M | I], a WARP per cell, lanes over the columns.
    // At pivot k only the columns j > k of M (and every column of I) are updated, so a lane touches its own columns alone and
    // reads column k, which nobody writes at this step: one __syncwarp per pivot is all the ordering the elimination needs. ----
    {
        const int wpb = nthr >> 5;
        for (int c = blockIdx.x * wpb + (tid >> 5); c < C; c += gridDim.x * wpb) {
            double* M = cp.Mw + (size_t)c * G * G;
            double* Inv = cp.Minv + (size_t)c * G * G;
            for (int i = lane; i < G * G; i += 32) {
                const int g = i / G, gp = i - g * G;
                double v = -cp.sigs[(size_t)c * G * G + i] * cp.V[c];
                if (g == gp) {
                    v += cp.sigt[(size_t)c * G + g] * cp.V[c] + cp.J_vac[(size_t)c * G + g] / cp.Phi[(size_t)c * G + g];
                    for (int a = cp.adj_off[c]; a < cp.adj_off[c + 1]; ++a) {
                        const int ent = cp.adj_ent[a], s = ent >> 1;
                        v += (ent & 1) ? cp.in_hi[(size_t)s * G + g] : cp.out_lo[(size_t)s * G + g];
                    }
                }
                M[i] = v;
                Inv[i] = g == gp ? 1.0 : 0.0;
            }
            __syncwarp();
            for (int k = 0; k < G; ++k) {
                double best = -1.0;                          // pivot: the largest |M[r][k]|, r >= k, lowest row on ties
                int br = k;
                for (int r = k + lane; r < G; r += 32) {
                    const double a = fabs(M[r * G + k]);
                    if (a > best) { best = a; br = r; }
                }
                for (int o = 16; o > 0; o >>= 1) {
                    const double ob = __shfl_xor_sync(0xffffffffu, best, o);
                    const int orow = __shfl_xor_sync(0xffffffffu, br, o);
                    if (ob > best || (ob == best && orow < br)) { best = ob; br = orow; }
                }
                const double pivot = M[br * G + k];          // read before any lane swaps the rows
                __syncwarp();
                const double inv_p = 1.0 / pivot;
                for (int j = lane; j < 2 * G; j += 32) {     // this lane's columns: j < G in M (only j > k live), j >= G in I
                    if (j <= k) continue;
                    double* A = j < G ? M : Inv;
                    const int col = j < G ? j : j - G;
                    double pk = A[br * G + col];             // swap rows k and br, scale the pivot row
                    if (br != k) { A[br * G + col] = A[k * G + col]; }
                    pk *= inv_p;
                    A[k * G + col] = pk;
                }
                if (br != k && lane == 0) {                  // column k itself travels with its rows (read as factors below)
                    const double t = M[br * G + k]; M[br * G + k] = M[k * G + k]; M[k * G + k] = t;
                }
                __syncwarp();
                for (int j = lane; j < 2 * G; j += 32) {
                    if (j <= k) continue;
                    double* A = j < G ? M : Inv;
                    const int col = j < G ? j : j - G;
                    const double pk = A[k * G + col];
                    for (int r = 0; r < G; ++r)
                        if (r != k) A[r * G + col] -= M[r * G + k] * pk;
                }
                __syncwarp();
            }
        }
    }
    // start vector and its fission production P0
    {
        double part = 0.0;
        for (int64_t i = gtid; i < n; i += gn) {
            const int c = (int)(i / G);
            cp.x[i] = cp.Phi[i];
            double e = 0.0;
            for (int gp = 0; gp < G; ++gp) e += cp.nusf[(size_t)c * G + gp] * cp.Phi[(size_t)c * G + gp];
            part += cp.chi[i] * cp.V[c] * e;
        }
        part = warp_sum(part);
        if (lane == 0 && part != 0.0) atomicAdd(cp.state + ST_P0, part);
    }
    grid.sync();

    // y_new = Minv (f + N y_old) for every (cell, group); thread per unknown, the right-hand side of a cell is recomputed by
    // each of its G threads' inner products (G^2 work per cell, no shared staging: cells are spread over the whole grid)
    auto jacobi = [&](const double* __restrict__ yo, double* __restrict__ yn) {
        for (int64_t i = gtid; i < n; i += gn) {
            const int c = (int)(i / G), g = (int)(i - (int64_t)c * G);
            const double* Inv = cp.Minv + (size_t)c * G * G + (size_t)g * G;
            double acc = 0.0;
            for (int gp = 0; gp < G; ++gp) {
                double rhs = cp.f[(size_t)c * G + gp];
                for (int a = cp.adj_off[c]; a < cp.adj_off[c + 1]; ++a) {
                    const int ent = cp.adj_ent[a], s = ent >> 1;
                    rhs += (ent & 1) ? cp.out_lo[(size_t)s * G + gp] * yo[(size_t)cp.lo[s] * G + gp]
                                     : cp.in_hi[(size_t)s * G + gp] * yo[(size_t)cp.hi[s] * G + gp];
                }
                acc += Inv[gp] * rhs;
            }
            yn[i] = acc;
        }
    };

    int it = 0;
    bool done = false;
    double d_first = -1.0;
    for (; it < cp.max_outer && !done; ++it) {
        const double k = cp.state[ST_K];
        for (int64_t i = gtid; i < n; i += gn) {             // f = B x / k
            const int c = (int)(i / G);
            double e = 0.0;
            for (int gp = 0; gp < G; ++gp) e += cp.nusf[(size_t)c * G + gp] * cp.x[(size_t)c * G + gp];
            cp.f[i] = cp.chi[i] * cp.V[c] * e / k;
        }
        if (gtid == 0) { cp.state[ST_SBY] = 0.0; cp.state[ST_SAY] = 0.0; cp.state[ST_DMAX] = 0.0; cp.state[ST_XMAX] = 0.0; }
        grid.sync();
        const double* yo = cp.x;
        double* yn = cp.y;
        for (int s = 0; s < cp.inner; ++s) {
            jacobi(yo, yn);
            grid.sync();
            yo = yn;
            yn = yn == cp.y ? cp.y2 : cp.y;
        }
        {   // sums of B y and A y over all unknowns (the coupling terms cancel in the sum of A y)
            double sby = 0.0, say = 0.0;
            for (int64_t i = gtid; i < n; i += gn) {
                const int c = (int)(i / G), g = (int)(i - (int64_t)c * G);
                double e = 0.0, sc = 0.0;
                for (int gp = 0; gp < G; ++gp) {
                    e += cp.nusf[(size_t)c * G + gp] * yo[(size_t)c * G + gp];
                    sc += cp.sigs[((size_t)c * G + g) * G + gp] * yo[(size_t)c * G + gp];
                }
                sby += cp.chi[i] * cp.V[c] * e;
                say += (cp.sigt[i] * cp.V[c] + cp.J_vac[i] / cp.Phi[i]) * yo[i] - cp.V[c] * sc;
            }
            sby = warp_sum(sby); say = warp_sum(say);
            if (lane == 0) { atomicAdd(cp.state + ST_SBY, sby); atomicAdd(cp.state + ST_SAY, say); }
        }
        grid.sync();
        const double sby = cp.state[ST_SBY], say = cp.state[ST_SAY];
        const double k_new = sby / say, scale = cp.state[ST_P0] / sby;
        {
            double dmax = 0.0, xmax = 0.0;
            for (int64_t i = gtid; i < n; i += gn) {
                const double v = yo[i] * scale;
                dmax = fmax(dmax, fabs(v - cp.x[i]));
                xmax = fmax(xmax, fabs(v));
                cp.x[i] = v;
            }
            dmax = warp_max(dmax); xmax = warp_max(xmax);
            if (lane == 0) { atomic_max_pos(cp.state + ST_DMAX, dmax); atomic_max_pos(cp.state + ST_XMAX, xmax); }
        }
        grid.sync();
        const double dmax_it = cp.state[ST_DMAX];
        if (d_first < 0.0) d_first = dmax_it;
        done = (fabs(k_new - k) < cp.tol_k * fabs(k_new) && dmax_it < cp.tol_x * cp.state[ST_XMAX]) ||
               (cp.rel_tol > 0.0 && it > 0 && dmax_it <= cp.rel_tol * d_first);
        grid.sync();                                         // everybody has read the state of this iteration
        if (gtid == 0) { cp.state[ST_KPREV] = k; cp.state[ST_K] = k_new; }
        grid.sync();
    }
    // success = converged to a positive eigenvalue with a positive flux
    {
        double xmin = 1.0;
        for (int64_t i = gtid; i < n; i += gn) xmin = fmin(xmin, cp.x[i] > 0.0 ? 1.0 : 0.0);
        xmin = -warp_max(-xmin);
        if (lane == 0 && xmin == 0.0) atomicAdd(cp.state + ST_DONE, 1.0);   // counts warps that saw a non-positive flux
    }
    grid.sync();
    if (gtid == 0) {
        cp.state[ST_ITERS] = (double)it;
        cp.state[ST_OK] = (done && cp.state[ST_K] > 0.0 && cp.state[ST_DONE] == 0.0) ? 1.0 : 0.0;
        cp.state[ST_DONE] = done ? 1.0 : 0.0;
    }
}

} // namespace ndk
