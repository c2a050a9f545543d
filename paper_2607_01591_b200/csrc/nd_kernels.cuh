// nd_kernels.cuh -- device kernels of the planar-MOC hot path (sm_100a).  Rows A2..A6 of DESIGN.md.
//   k_source_tiled  A5  scatter + fission source (Eq. (1)/(3) RHS), reduced source q, tally reset
//   k_sweep_atomic  A2  Eq. (5) per (track, direction, polar, group); FP64 global atomics per segment
//   k_link_swap     A3  boundary angular flux through the link table (compressed psi: track ends only)
//   k_finalise      A4  phi = 4 pi Q/Sigma_t + tally/(Sigma_t A~) + partial fission-rate sums
//   k_reduce_*      A6  fission rate, k_eff update
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ndk {

constexpr int kMaxPolar = 4;
constexpr int kPartialStride = 4;   // doubles per block in the partial-sum arrays of the reductions
constexpr double kFourPi = 12.566370614359172953850573533118;

// Segment stream record (SoA): seg_rm[k] = region | material << 24 ; seg_len[k] = FP32 projected length.
__host__ __device__ inline uint32_t pack_rm(uint32_t region, uint32_t material) { return region | (material << 24); }
__device__ __forceinline__ uint32_t rm_region(uint32_t rm) { return rm & 0x00ffffffu; }
__device__ __forceinline__ uint32_t rm_material(uint32_t rm) { return rm >> 24; }

struct SweepParams {
    // segment stream
    const uint32_t* __restrict__ seg_rm;
    const float* __restrict__ seg_len;
    const int64_t* __restrict__ trk_off;   // [T+1] padded offsets (multiples of 4)
    const float* __restrict__ trk_w;       // [T] 4 pi omega_a delta_a
    // region / material data
    const float* __restrict__ q;           // [R][Gs] reduced source Q/Sigma_t
    const float* __restrict__ sigt;        // [M][Gs]
    double* __restrict__ tally;            // [R][Gs]
    // boundary flux
    const float* __restrict__ psi_in;      // [T][2][P][Gs]
    float* __restrict__ psi_out;           // [T][2][P][Gs]
    const double* __restrict__ scale_div;  // device scalar F: psi_in is used as psi_in / F
    int T, G, Gs;
    float c[kMaxPolar];                    // -log2(e)/sin(theta_p)      (ND_EXP_FAST)
    float inv_sin[kMaxPolar];              // 1/sin(theta_p)             (ND_EXP_EXPM1)
    float wp[kMaxPolar];                   // polar_weight*polar_sin
};

__device__ __forceinline__ float ex2_approx(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// One Eq.-(5) step for P polar chains of one (track, direction, group): returns sum_p wp*Delta_p.
template <int P, int EXPM>
__device__ __forceinline__ float attenuate(float (&psi)[P], float qv, float st_s, const SweepParams& prm)
{
    float acc = 0.f;
#pragma unroll
    for (int p = 0; p < P; ++p) {
        const float d = psi[p] - qv;
        float delta;
        if (EXPM == 0) {
            const float a = ex2_approx(st_s * prm.c[p]);   // exp(-tau)
            delta = fmaf(-d, a, d);                         // d*(1-a)
        } else {
            delta = d * (-expm1f(-st_s * prm.inv_sin[p]));
        }
        psi[p] -= delta;
        acc = fmaf(prm.wp[p], delta, acc);
    }
    return acc;
}

// ---- A2, baseline: one warp per (track, direction); lanes over groups; FP64 atomics per (segment, group) ----
template <int P, int EXPM>
__global__ void __launch_bounds__(256) k_sweep_atomic(const SweepParams prm)
{
    const int lane = threadIdx.x & 31;
    const int warps_per_block = blockDim.x >> 5;
    const int64_t n_pairs = 2 * (int64_t)prm.T;
    const float inv_f = (float)(1.0 / *prm.scale_div);
    for (int64_t pair = (int64_t)blockIdx.x * warps_per_block + (threadIdx.x >> 5); pair < n_pairs;
         pair += (int64_t)gridDim.x * warps_per_block) {
        const int t = (int)(pair >> 1), dir = (int)(pair & 1);
        const int64_t k0 = prm.trk_off[t], k1 = prm.trk_off[t + 1];
        const float wt = prm.trk_w[t];
        for (int g = lane; g < prm.G; g += 32) {
            float psi[P];
#pragma unroll
            for (int p = 0; p < P; ++p) psi[p] = prm.psi_in[(pair * P + p) * prm.Gs + g] * inv_f;
            for (int64_t i = 0; i < k1 - k0; ++i) {
                const int64_t k = dir == 0 ? k0 + i : k1 - 1 - i;
                const uint32_t rm = prm.seg_rm[k];
                const float s = prm.seg_len[k];
                const uint32_t r = rm_region(rm);
                const float st = prm.sigt[rm_material(rm) * prm.Gs + g];
                const float qv = prm.q[(size_t)r * prm.Gs + g];
                const float acc = attenuate<P, EXPM>(psi, qv, st * s, prm);
                if (s > 0.f) atomicAdd(&prm.tally[(size_t)r * prm.Gs + g], (double)(wt * acc));
            }
#pragma unroll
            for (int p = 0; p < P; ++p) prm.psi_out[(pair * P + p) * prm.Gs + g] = psi[p];
        }
    }
}

// ---- A3: psi_next[e] = src[e] >= 0 ? psi_out[src[e]] : 0  for every entry e = 2t+d (gather form) ----
__global__ void __launch_bounds__(256) k_link_swap(const float* __restrict__ psi_out, float* __restrict__ psi_next,
                                                   const int32_t* __restrict__ src, int64_t n_entries, int PG)
{
    // one 16-byte piece per thread and step (PG is a multiple of 4); (e, j) advance with i: no division per element
    const int PG4 = PG >> 2;
    const int64_t n = n_entries * PG4, stride = (int64_t)gridDim.x * blockDim.x;
    const int64_t de = stride / PG4;
    const int dj = (int)(stride - de * PG4);
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int64_t e = i / PG4;
    int j = (int)(i - e * PG4);
    const float4* __restrict__ in4 = reinterpret_cast<const float4*>(psi_out);
    float4* __restrict__ out4 = reinterpret_cast<float4*>(psi_next);
    for (; i < n; i += stride, e += de, j += dj) {
        if (j >= PG4) { j -= PG4; ++e; }
        const int32_t s = src[e];
        out4[i] = s >= 0 ? in4[(int64_t)s * PG4 + j] : make_float4(0.f, 0.f, 0.f, 0.f);
    }
}

// ---- A5: source (k_source_tiled below).
// Q[r][g] = (1/4pi) ( sum_g' Ss[m][g][g'] phi[r][g']/F + chi[m][g]/k * sum_g' nSf[m][g'] phi[r][g']/F )
// Also writes q = (float)(Q/Sigma_t) and zeroes the tally row.  sigsT is [m][g_from][g_to].
struct SourceParams {
    const double* __restrict__ phi;      // [R][G]
    const int32_t* __restrict__ reg_mat; // [R]
    const double* __restrict__ sigt;     // [M][G]
    const double* __restrict__ sigsT;    // [M][G_from][G_to]
    const double* __restrict__ nusf;     // [M][G]
    const double* __restrict__ chi;      // [M][G]
    const double* __restrict__ k_ptr;    // device scalar k (or NULL: use k_val)
    const double* __restrict__ f_ptr;    // device scalar F (or NULL: 1)
    double k_val;
    double* __restrict__ Q;              // [R][G]
    float* __restrict__ q;               // [R][Gs] or NULL
    double* __restrict__ tally;          // [R][Gs] or NULL
    int R, G, Gs;
};

// ---- A5, tiled: regions are visited in material-grouped CHUNKS (host-built: src_region is a permutation of the
// regions, chunk = (first, count, material)), so one thread block works with ONE scattering matrix at a time.
// The fission sum nuSigma_f . phi is formed once per region (warp shuffle), not once per destination group.
struct SourceChunkParams {
    SourceParams base;
    const int32_t* __restrict__ src_region;   // [R] regions grouped by material
    const int4* __restrict__ chunks;          // (first index into src_region, count, material, -)
    int n_chunks, chunk_regions;              // chunk_regions = nsub * kSrcTile (max count)
};

// q = Q/Sigma_t and tally = 0 for a caller-supplied Q (fixed-source nd_transport_sweep)
__global__ void __launch_bounds__(256) k_reduced_source(const double* __restrict__ Q, const int32_t* __restrict__ reg_mat,
                                                        const double* __restrict__ sigt, float* __restrict__ q,
                                                        double* __restrict__ tally, int64_t R, int G, int Gs)
{
    const int64_t n = R * Gs;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t r = i / Gs;
        const int g = (int)(i - r * Gs);
        tally[i] = 0.0;
        q[i] = g < G ? (float)(Q[r * G + g] / sigt[(size_t)reg_mat[r] * G + g]) : 0.f;
    }
}

// Thread (sub, pair): kSrcTile regions x 2 destination groups in registers; per PAIR of source groups four Sigma_s loads and
// kSrcTile 16-byte shared-memory loads of phi feed 4 * kSrcTile FP64 FMAs (0.375 loads per FMA; with 4 regions x 1 group per
// thread it was 1.25, and the kernel's time was the LSU's, not the FP64 pipe's).  phi rows are padded to an even
// number of doubles in shared memory; an odd G repeats the last group in the pad lane (zero phi, nothing stored).  Every
// accumulator adds its terms in the order of the source groups.
// SS_SMEM: the chunk's scattering matrix is staged in shared memory ([G][Gp] doubles, reloaded only when the material
// changes between two chunks of a block), so the inner loop waits on no global load; used when it fits beside the phi tile.
constexpr int kSrcTile = 8;
__device__ __forceinline__ void src_cp_async_8(double* smem_dst, const double* gmem_src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((uint32_t)__cvta_generic_to_shared(smem_dst)), "l"(gmem_src) : "memory");
}
// The phi tile is DOUBLE-BUFFERED: the rows of the block's next chunk are gathered by 8-byte cp.async (a phi row starts on an
// 8-byte boundary only) while the current chunk is computed, so the gather's latency is off the path.  phi / F is applied to
// the results (the source is linear in phi), not to the staged values.
template <bool SS_SMEM>
__global__ void __launch_bounds__(256, 2) k_source_tiled(const SourceChunkParams cp)
{
    extern __shared__ __align__(16) double s_src2[];   // phi [2][chunk_regions][Gp], fis [chunk_regions], (Sigma_s^T [G][Gp])
    const SourceParams& prm = cp.base;
    const int G = prm.G, CR = cp.chunk_regions, np = (G + 1) >> 1, Gp = 2 * np;
    double* s_fis = s_src2 + 2 * (size_t)CR * Gp;
    double* s_ss = s_fis + ((CR + 1) & ~1);            // 16-byte aligned
    int m_loaded = -1;
    const int nsub = CR / kSrcTile;            // <= blockDim.x / np, capped by the host so that the phi tiles fit
    const int sub = threadIdx.x / np, pr = threadIdx.x - sub * np;
    const int g0 = 2 * pr, g1 = g0 + 1 < G ? g0 + 1 : g0;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    const double inv_f = prm.f_ptr ? 1.0 / *prm.f_ptr : 1.0;
    const double inv_k = 1.0 / (prm.k_ptr ? *prm.k_ptr : prm.k_val);
    const double scale = inv_f / kFourPi;
    if (Gp > G)   // the pad column of both buffers: never written by the copies
        for (int i = threadIdx.x; i < 2 * CR; i += blockDim.x) s_src2[(size_t)i * Gp + G] = 0.0;
    auto gather = [&](int c, int buf) {   // rows of chunk c -> buffer buf: a warp per row and a lane per group (wide rows)
        const int4 ch = cp.chunks[c];
        double* dst = s_src2 + (size_t)buf * CR * Gp;
        if (G >= 24) {
            for (int lr = warp; lr < ch.y; lr += nwarp) {
                const double* src = prm.phi + (size_t)cp.src_region[ch.x + lr] * G;
                for (int g = lane; g < G; g += 32) src_cp_async_8(dst + (size_t)lr * Gp + g, src + g);
            }
        } else {   // narrow rows: a thread per element
            for (int i = threadIdx.x; i < ch.y * G; i += blockDim.x) {
                const int lr = i / G, g = i - lr * G;
                src_cp_async_8(dst + (size_t)lr * Gp + g, prm.phi + (size_t)cp.src_region[ch.x + lr] * G + g);
            }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    int buf = 0;
    if ((int)blockIdx.x < cp.n_chunks) gather(blockIdx.x, 0);
    for (int c = blockIdx.x; c < cp.n_chunks; c += gridDim.x, buf ^= 1) {
        const int4 ch = cp.chunks[c];
        const int first = ch.x, cnt = ch.y, m = ch.z;
        const double* s_phi = s_src2 + (size_t)buf * CR * Gp;
        const int c_next = c + gridDim.x;
        if (c_next < cp.n_chunks) {   // the other buffer is free: every thread is past the previous chunk (barrier below)
            gather(c_next, buf ^ 1);
            asm volatile("cp.async.wait_group 1;" ::: "memory");
        } else {
            asm volatile("cp.async.wait_group 0;" ::: "memory");
        }
        if (SS_SMEM && m != m_loaded) {   // rows gp of Sigma_s^T, padded to Gp (the pad column repeats the last group)
            const double* src = prm.sigsT + (size_t)m * G * G;
            for (int i = threadIdx.x; i < G * Gp; i += blockDim.x) {
                const int gp = i / Gp, g = i - gp * Gp;
                s_ss[i] = src[(size_t)gp * G + (g < G ? g : G - 1)];
            }
            m_loaded = m;
        }
        __syncthreads();
        const double* nf = prm.nusf + (size_t)m * G;
        for (int lr = warp; lr < cnt; lr += nwarp) {   // fission sum of region lr
            double f = 0.0;
            for (int gp = lane; gp < G; gp += 32) f += nf[gp] * s_phi[lr * Gp + gp];
            for (int o = 16; o > 0; o >>= 1) f += __shfl_xor_sync(0xffffffffu, f, o);
            if (lane == 0) s_fis[lr] = f;
        }
        __syncthreads();
        if (sub < nsub) {
            const double* ss = prm.sigsT + (size_t)m * G * G;
            double acc0[kSrcTile], acc1[kSrcTile];
            const double* ph[kSrcTile];
#pragma unroll
            for (int i = 0; i < kSrcTile; ++i) {
                acc0[i] = 0.0; acc1[i] = 0.0;
                const int lr = sub + i * nsub;
                ph[i] = s_phi + (size_t)(lr < cnt ? lr : 0) * Gp;
            }
            for (int gp = 0; gp < Gp; gp += 2) {
                const int gq = gp + 1 < G ? gp + 1 : gp;       // pad lane of an odd G: phi = 0 there
                double a00, a01, a10, a11;
                if (SS_SMEM) {
                    const double2 u = *reinterpret_cast<const double2*>(s_ss + (size_t)gp * Gp + g0);
                    const double2 w = *reinterpret_cast<const double2*>(s_ss + (size_t)gq * Gp + g0);
                    a00 = u.x; a01 = u.y; a10 = w.x; a11 = w.y;
                } else {
                    a00 = ss[(size_t)gp * G + g0]; a01 = ss[(size_t)gp * G + g1];
                    a10 = ss[(size_t)gq * G + g0]; a11 = ss[(size_t)gq * G + g1];
                }
#pragma unroll
                for (int i = 0; i < kSrcTile; ++i) {
                    const double2 v = *reinterpret_cast<const double2*>(ph[i] + gp);
                    acc0[i] = fma(a00, v.x, acc0[i]); acc1[i] = fma(a01, v.x, acc1[i]);
                    acc0[i] = fma(a10, v.y, acc0[i]); acc1[i] = fma(a11, v.y, acc1[i]);
                }
            }
            const double chi0 = prm.chi[(size_t)m * G + g0] * inv_k, chi1 = prm.chi[(size_t)m * G + g1] * inv_k;
            const double st0 = prm.sigt[(size_t)m * G + g0], st1 = prm.sigt[(size_t)m * G + g1];
            const bool two = g0 + 1 < G;
#pragma unroll
            for (int i = 0; i < kSrcTile; ++i) {
                const int lr = sub + i * nsub;
                if (lr < cnt) {
                    const int64_t r = cp.src_region[first + lr];
                    const double Q0 = (acc0[i] + chi0 * s_fis[lr]) * scale, Q1 = (acc1[i] + chi1 * s_fis[lr]) * scale;
                    prm.Q[r * G + g0] = Q0;
                    if (two) prm.Q[r * G + g1] = Q1;
                    // q and tally rows are padded to Gs (a multiple of 4): the pair (g0, g0 + 1) is always inside the row
                    if (prm.q) *reinterpret_cast<float2*>(prm.q + r * prm.Gs + g0) = make_float2((float)(Q0 / st0), two ? (float)(Q1 / st1) : 0.f);
                    if (prm.tally) *reinterpret_cast<double2*>(prm.tally + r * prm.Gs + g0) = make_double2(0.0, 0.0);
                }
            }
        }
        __syncthreads();   // the buffer just computed from is the target of the next iteration's gather
    }
}

// ---- block-wide FP64 sum / max (deterministic tree) ----
__device__ __forceinline__ double block_sum(double v, double* scratch)
{
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) scratch[w] = v;
    __syncthreads();
    if (w == 0) {
        v = lane < (blockDim.x >> 5) ? scratch[lane] : 0.0;
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    }
    return v; // valid in thread 0
}
__device__ __forceinline__ double block_max(double v, double* scratch)
{
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_down_sync(0xffffffffu, v, o));
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) scratch[w] = v;
    __syncthreads();
    if (w == 0) {
        v = lane < (blockDim.x >> 5) ? scratch[lane] : 0.0;
        for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_down_sync(0xffffffffu, v, o));
    }
    return v;
}

// ---- A4 + first stage of A6 ----
// phi_new[r][g] = 4 pi Q/Sigma_t + (A~_r > 0 ? tally/(Sigma_t A~_r) : 0)
// partial[4*b+0] = sum over the block's elements of A~_r nuSigma_f phi_new          (fission rate)
// partial[4*b+1] = max |phi_new - phi_old/F|   partial[4*b+2] = max |phi_new|       (only if phi_old != NULL)
// partial[4*b+3] = sum of the tally (what the chains of the sweep lost, by the telescoping identity)
struct FinaliseParams {
    const double* __restrict__ Q;        // [R][G]
    const double* __restrict__ tally;    // [R][Gs]
    const int32_t* __restrict__ reg_mat;
    const double* __restrict__ sigt;     // [M][G]
    const double* __restrict__ nusf;     // [M][G]
    const double* __restrict__ vol;      // [R]
    const double* __restrict__ phi_old;  // [R][G] or NULL
    const double* __restrict__ f_ptr;    // scalar F for phi_old normalisation (or NULL)
    double* __restrict__ phi_new;        // [R][G]
    double* __restrict__ partial;        // [gridDim.x][kPartialStride]
    int64_t R;
    int G, Gs;
};

// TAB: Sigma_t and nu Sigma_f of all materials are staged in shared memory (M G <= kFinTab entries each), which takes two
// global loads out of the chain that hangs on the region's material id.
constexpr int kFinTab = 2048;
template <bool TAB>
__global__ void __launch_bounds__(256) k_finalise(const FinaliseParams prm, int MG)
{
    __shared__ double scratch[32];
    __shared__ double s_st[TAB ? kFinTab : 1], s_nf[TAB ? kFinTab : 1];
    if (TAB) {
        for (int i = threadIdx.x; i < MG; i += blockDim.x) { s_st[i] = prm.sigt[i]; s_nf[i] = prm.nusf[i]; }
        __syncthreads();
    }
    const int64_t n = prm.R * prm.G;
    const double inv_f = (prm.phi_old && prm.f_ptr) ? 1.0 / *prm.f_ptr : 1.0;
    double fsum = 0.0, dmax = 0.0, pmax = 0.0, tsum = 0.0;
    // (r, g) of element i advance with i: no 64-bit division per element
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const int64_t dr = stride / prm.G;
    const int dg = (int)(stride - dr * prm.G);
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int64_t r = i / prm.G;
    int g = (int)(i - r * prm.G);
    for (; i < n; i += stride, r += dr, g += dg) {
        if (g >= prm.G) { g -= prm.G; ++r; }
        const int m = prm.reg_mat[r];
        const double st = TAB ? s_st[m * prm.G + g] : prm.sigt[(size_t)m * prm.G + g];
        const double a = prm.vol[r];
        const double tl = prm.tally[r * prm.Gs + g];
        tsum += tl;
        double phi = kFourPi * prm.Q[i] / st;
        if (a > 0.0) phi += tl / (st * a);
        prm.phi_new[i] = phi;
        fsum += a * (TAB ? s_nf[m * prm.G + g] : prm.nusf[(size_t)m * prm.G + g]) * phi;
        if (prm.phi_old) {
            dmax = fmax(dmax, fabs(phi - prm.phi_old[i] * inv_f));
            pmax = fmax(pmax, fabs(phi));
        }
    }
    fsum = block_sum(fsum, scratch);
    dmax = block_max(dmax, scratch);
    pmax = block_max(pmax, scratch);
    tsum = block_sum(tsum, scratch);
    if (threadIdx.x == 0) {
        prm.partial[kPartialStride * blockIdx.x + 0] = fsum;
        prm.partial[kPartialStride * blockIdx.x + 1] = dmax;
        prm.partial[kPartialStride * blockIdx.x + 2] = pmax;
        prm.partial[kPartialStride * blockIdx.x + 3] = tsum;
    }
}

// ---- A6, boundary side of the balance: over every chain e = 2t+d of ONE sweep (run between the sweep and the link swap)
//   partial[4*b+0] = sum w_{t,p} psi_in / F      what entered through the track ends (0 at vacuum ends)
//   partial[4*b+1] = sum w_{t,p} psi_out         what left through them
//   partial[4*b+2] = the part of [1] that left through VACUUM ends: the leakage
__global__ void __launch_bounds__(256) k_boundary_balance(const float* __restrict__ psi_in, const float* __restrict__ psi_out,
                                                          const float* __restrict__ trk_w, const uint8_t* __restrict__ exit_vacuum,
                                                          const double* __restrict__ scale_div, double* __restrict__ partial,
                                                          int64_t n_entries, int P, int G, int Gs, float wp0, float wp1, float wp2,
                                                          float wp3)
{
    __shared__ double scratch[32];
    const float wp[kMaxPolar] = {wp0, wp1, wp2, wp3};
    const int PG = P * Gs;
    const int64_t n = n_entries * PG;
    const double inv_f = 1.0 / *scale_div;
    double s_in = 0.0, s_out = 0.0, s_leak = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t e = i / PG;
        const int j = (int)(i - e * PG), p = j / Gs, g = j - p * Gs;
        if (g >= G) continue;
        const double w = (double)trk_w[e >> 1] * (double)wp[p];
        const double o = w * (double)psi_out[i];
        s_in += w * (double)psi_in[i] * inv_f;
        s_out += o;
        if (exit_vacuum[e]) s_leak += o;
    }
    s_in = block_sum(s_in, scratch);
    s_out = block_sum(s_out, scratch);
    s_leak = block_sum(s_leak, scratch);
    if (threadIdx.x == 0) {
        partial[kPartialStride * blockIdx.x + 0] = s_in;
        partial[kPartialStride * blockIdx.x + 1] = s_out;
        partial[kPartialStride * blockIdx.x + 2] = s_leak;
        partial[kPartialStride * blockIdx.x + 3] = 0.0;
    }
}

// fission rate of an arbitrary phi: partial[4*b] = sum A~ nuSigma_f phi
__global__ void __launch_bounds__(256) k_fission_partial(const double* __restrict__ phi, const int32_t* __restrict__ reg_mat,
                                                         const double* __restrict__ nusf, const double* __restrict__ vol,
                                                         double* __restrict__ partial, int64_t R, int G)
{
    __shared__ double scratch[32];
    const int64_t n = R * G;
    double fsum = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t r = i / G;
        const int g = (int)(i - r * G);
        fsum += vol[r] * nusf[(size_t)reg_mat[r] * G + g] * phi[i];
    }
    fsum = block_sum(fsum, scratch);
    if (threadIdx.x == 0) {
        partial[kPartialStride * blockIdx.x] = fsum;
        partial[kPartialStride * blockIdx.x + 1] = partial[kPartialStride * blockIdx.x + 2] = partial[kPartialStride * blockIdx.x + 3] = 0.0;
    }
}

// ---- A6 second stage (one block): scalars[] layout below.  mode 0: F <- sum (no k update).
//      mode 1 (power iteration): F_new = sum; k_prev = k; k <- k*F_new; F <- F_new; dphi = max/max ----
enum { SC_K = 0, SC_F = 1, SC_KPREV = 2, SC_DPHI = 3, SC_ONE = 4, SC_COUNT = 8 };

constexpr int kStatsStride = 6;   // doubles per iteration record: k, F, dk, dphi, leakage, balance residual

__global__ void __launch_bounds__(256) k_reduce_final(const double* __restrict__ partial, int n_partial,
                                                      double* __restrict__ scalars, int mode,
                                                      double* __restrict__ stats_slot /* kStatsStride doubles or NULL */,
                                                      const double* __restrict__ partial_b /* k_boundary_balance's, or NULL */,
                                                      int n_partial_b)
{
    __shared__ double scratch[32];
    double fsum = 0.0, dmax = 0.0, pmax = 0.0, tsum = 0.0, s_in = 0.0, s_out = 0.0, s_leak = 0.0;
    for (int i = threadIdx.x; i < n_partial; i += blockDim.x) {
        fsum += partial[kPartialStride * i];
        dmax = fmax(dmax, partial[kPartialStride * i + 1]);
        pmax = fmax(pmax, partial[kPartialStride * i + 2]);
        tsum += partial[kPartialStride * i + 3];
    }
    if (partial_b)
        for (int i = threadIdx.x; i < n_partial_b; i += blockDim.x) {
            s_in += partial_b[kPartialStride * i];
            s_out += partial_b[kPartialStride * i + 1];
            s_leak += partial_b[kPartialStride * i + 2];
        }
    fsum = block_sum(fsum, scratch);
    dmax = block_max(dmax, scratch);
    pmax = block_max(pmax, scratch);
    tsum = block_sum(tsum, scratch);
    s_in = block_sum(s_in, scratch);
    s_out = block_sum(s_out, scratch);
    s_leak = block_sum(s_leak, scratch);
    if (threadIdx.x == 0) {
        if (mode == 1) {
            const double k_prev = scalars[SC_K];
            const double k_new = k_prev * fsum;
            scalars[SC_KPREV] = k_prev;
            scalars[SC_K] = k_new;
            scalars[SC_DPHI] = pmax > 0.0 ? dmax / pmax : 0.0;
            if (stats_slot) {
                stats_slot[0] = k_new; stats_slot[1] = fsum; stats_slot[2] = k_new - k_prev; stats_slot[3] = scalars[SC_DPHI];
                // telescoping identity of the sweep: sum of the tallies = what entered - what left through the track ends
                const double den = fabs(s_in) + fabs(s_out);
                stats_slot[4] = partial_b ? s_leak : 0.0;
                stats_slot[5] = partial_b && den > 0.0 ? (s_in - s_out - tsum) / den : 0.0;
            }
        }
        scalars[SC_F] = fsum;
    }
}

__global__ void k_fill_f64(double* __restrict__ p, double v, int64_t n)
{
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) p[i] = v;
}
__global__ void k_fill_f32(float* __restrict__ p, float v, int64_t n)
{
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) p[i] = v;
}
// compact [R][Gs] -> [R][G]
__global__ void k_unpad_f64(const double* __restrict__ src, double* __restrict__ dst, int64_t R, int G, int Gs)
{
    const int64_t n = R * G;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t r = i / G;
        dst[i] = src[r * Gs + (i - r * G)];
    }
}

} // namespace ndk
