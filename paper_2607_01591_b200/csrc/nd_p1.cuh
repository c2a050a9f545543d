// nd_p1.cuh -- NEXT-4: the transport sweep with a linearly anisotropic (P_1) scattering source, the l = 1
// truncation of the Legendre expansion Eq. (2) of the paper inside Eq. (5).  Readings P-1..P-6
// of DESIGN.md 8e.  First correct kernels on the same segment data (the paper: the solvers "share the ray tracing and segment
// data structures"): the simple one-warp-per-chain sweep over the SoA stream with three FP64 tallies.
//   k_p1_moment_source  Q1x, Q1y = (1/4pi) Sigma_s1 J / F and their reduced FP32 rows; zeroes the two moment tallies
//   k_sweep_p1          Eq. (5) with q(Omega) = q0 + 3 (Omega_x q1x + Omega_y q1y) for the chain's own direction; tallies
//                       w D, w Omega_x D, w Omega_y D
//   k_p1_currents       J = [ 4 pi 3 c2 (M Q1) + tally ] / (Sigma_t A~)   (phi is finalised by k_finalise, as in O-6)
#pragma once
#include "nd_kernels.cuh"

namespace ndk {

struct P1SweepParams {
    SweepParams sw;                         // stream, q = q0, Sigma_t, tally = tally0, psi_in / psi_out, polar tables
    const float* __restrict__ q1x;          // [R][Gs] Q1x / Sigma_t
    const float* __restrict__ q1y;          // [R][Gs]
    const float* __restrict__ trk_dir;      // [T][2] unit vector from the start to the end point of a track
    double* __restrict__ tally_x;           // [R][Gs]
    double* __restrict__ tally_y;           // [R][Gs]
    float sin_t[kMaxPolar];                 // sin(theta_p)
};

// One warp per (track, direction), lanes over groups, P polar chains per lane (the layout of k_sweep_atomic).
template <int P>
__global__ void __launch_bounds__(256) k_sweep_p1(const P1SweepParams pp)
{
    const SweepParams& prm = pp.sw;
    const int lane = threadIdx.x & 31;
    const int warps_per_block = blockDim.x >> 5;
    const int64_t n_pairs = 2 * (int64_t)prm.T;
    const float inv_f = (float)(1.0 / *prm.scale_div);
    for (int64_t pair = (int64_t)blockIdx.x * warps_per_block + (threadIdx.x >> 5); pair < n_pairs;
         pair += (int64_t)gridDim.x * warps_per_block) {
        const int t = (int)(pair >> 1), dir = (int)(pair & 1);
        const int64_t k0 = prm.trk_off[t], k1 = prm.trk_off[t + 1];
        const float wt = prm.trk_w[t];
        const float sgn = dir == 0 ? 1.f : -1.f;
        const float ux = sgn * pp.trk_dir[2 * t], uy = sgn * pp.trk_dir[2 * t + 1];    // P-2: direction of travel
        for (int g = lane; g < prm.G; g += 32) {
            float psi[P];
#pragma unroll
            for (int p = 0; p < P; ++p) psi[p] = prm.psi_in[(pair * P + p) * prm.Gs + g] * inv_f;
            for (int64_t i = 0; i < k1 - k0; ++i) {
                const int64_t k = dir == 0 ? k0 + i : k1 - 1 - i;
                const uint32_t rm = prm.seg_rm[k];
                const float s = prm.seg_len[k];
                const uint32_t r = rm_region(rm);
                const float st_s = prm.sigt[rm_material(rm) * prm.Gs + g] * s;
                const size_t at = (size_t)r * prm.Gs + g;
                const float q0 = prm.q[at];
                const float qm = 3.f * (ux * pp.q1x[at] + uy * pp.q1y[at]);   // 3 (u . q1): times sin(theta_p) below
                float a0 = 0.f, a1 = 0.f;
#pragma unroll
                for (int p = 0; p < P; ++p) {
                    const float d = psi[p] - fmaf(pp.sin_t[p], qm, q0);           // P-1, P-3
                    const float a = ex2_approx(st_s * prm.c[p]);
                    const float delta = fmaf(-d, a, d);
                    psi[p] -= delta;
                    a0 = fmaf(prm.wp[p], delta, a0);                             // P-4: sum_p w_p D and sum_p w_p sin(theta_p) D
                    a1 = fmaf(prm.wp[p] * pp.sin_t[p], delta, a1);
                }
                if (s > 0.f) {
                    atomicAdd(&prm.tally[at], (double)(wt * a0));
                    atomicAdd(&pp.tally_x[at], (double)(wt * ux * a1));
                    atomicAdd(&pp.tally_y[at], (double)(wt * uy * a1));
                }
            }
#pragma unroll
            for (int p = 0; p < P; ++p) prm.psi_out[(pair * P + p) * prm.Gs + g] = psi[p];
        }
    }
}

// P-1: Q1[r][g] = (1/4pi) sum_g' Ss1[m][g][g'] J[r][g'] / F for both components; q1 = (float)(Q1 / Sigma_t); moment tallies zeroed.
// s1T is [m][g_from][g_to].  f_ptr may be NULL (F = 1).
__global__ void __launch_bounds__(256) k_p1_moment_source(const double* __restrict__ Jx, const double* __restrict__ Jy,
                                                          const int32_t* __restrict__ reg_mat, const double* __restrict__ sigt,
                                                          const double* __restrict__ s1T, const double* __restrict__ f_ptr,
                                                          double* __restrict__ Q1x, double* __restrict__ Q1y, float* __restrict__ q1x,
                                                          float* __restrict__ q1y, double* __restrict__ tally_x,
                                                          double* __restrict__ tally_y, int64_t R, int G, int Gs)
{
    const int64_t n = R * Gs;
    const double inv_f = f_ptr ? 1.0 / *f_ptr : 1.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t r = i / Gs;
        const int g = (int)(i - r * Gs);
        if (tally_x) { tally_x[i] = 0.0; tally_y[i] = 0.0; }
        if (g >= G) { if (q1x) { q1x[i] = 0.f; q1y[i] = 0.f; } continue; }
        const int m = reg_mat[r];
        const double* s1 = s1T + (size_t)m * G * G + g;
        double sx = 0.0, sy = 0.0;
        for (int gp = 0; gp < G; ++gp) {
            const double a = s1[(size_t)gp * G];
            sx = fma(a, Jx[r * G + gp], sx);
            sy = fma(a, Jy[r * G + gp], sy);
        }
        sx *= inv_f / kFourPi; sy *= inv_f / kFourPi;
        if (Q1x) { Q1x[r * G + g] = sx; Q1y[r * G + g] = sy; }
        if (q1x) {
            const double st = sigt[(size_t)m * G + g];
            q1x[i] = (float)(sx / st); q1y[i] = (float)(sy / st);
        }
    }
}

// reduced rows of caller-supplied moment sources (fixed-source nd_p1_transport_sweep)
__global__ void __launch_bounds__(256) k_p1_reduced_moments(const double* __restrict__ Q1x, const double* __restrict__ Q1y,
                                                            const int32_t* __restrict__ reg_mat, const double* __restrict__ sigt,
                                                            float* __restrict__ q1x, float* __restrict__ q1y, double* __restrict__ tally_x,
                                                            double* __restrict__ tally_y, int64_t R, int G, int Gs)
{
    const int64_t n = R * Gs;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t r = i / Gs;
        const int g = (int)(i - r * Gs);
        tally_x[i] = 0.0; tally_y[i] = 0.0;
        const double st = g < G ? sigt[(size_t)reg_mat[r] * G + g] : 1.0;
        q1x[i] = g < G ? (float)(Q1x[r * G + g] / st) : 0.f;
        q1y[i] = g < G ? (float)(Q1y[r * G + g] / st) : 0.f;
    }
}

// P-5: J = [ 4 pi 3 c2 (M Q1) + tally ] / (Sigma_t A~);  A~ = 0: J = 0
__global__ void __launch_bounds__(256) k_p1_currents(const double* __restrict__ Q1x, const double* __restrict__ Q1y,
                                                     const double* __restrict__ tally_x, const double* __restrict__ tally_y,
                                                     const int32_t* __restrict__ reg_mat, const double* __restrict__ sigt,
                                                     const double* __restrict__ vol, const double* __restrict__ Mxx,
                                                     const double* __restrict__ Mxy, const double* __restrict__ Myy, double c2,
                                                     double* __restrict__ Jx, double* __restrict__ Jy, int64_t R, int G, int Gs)
{
    const int64_t n = R * G;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t r = i / G;
        const int g = (int)(i - r * G);
        const double a = vol[r];
        double jx = 0.0, jy = 0.0;
        if (a > 0.0) {
            const double den = sigt[(size_t)reg_mat[r] * G + g] * a, f = kFourPi * 3.0 * c2;
            jx = (f * (Mxx[r] * Q1x[i] + Mxy[r] * Q1y[i]) + tally_x[r * Gs + g]) / den;
            jy = (f * (Mxy[r] * Q1x[i] + Myy[r] * Q1y[i]) + tally_y[r * Gs + g]) / den;
        }
        Jx[i] = jx; Jy[i] = jy;
    }
}

} // namespace ndk
