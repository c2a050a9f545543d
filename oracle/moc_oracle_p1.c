/*
 * oracle/moc_oracle_p1.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * the planar-MOC sweep of moc_oracle.c with a LINEARLY ANISOTROPIC (P_1) scattering source, the
 * L = 1 truncation of the Legendre expansion Eq. (2) of arxiv/paper_2607_01591 inside Eq. (1)/(3)
 * and Eq. (4)-(5).  Plain FP64, step by step, no blocking; shares no code with the
 * CUDA path.  The paper prints Eq. (2) and nothing about how the planar solver carries the moments; the reading is
 * (P-1..P-6):
 *   P-1  Sigma_s(Omega'.Omega) = (1/4pi) [ Sigma_s0 + 3 Sigma_s1 (Omega'.Omega) ]   (Eq. (2), l = 0, 1), so the angular source
 *        per steradian of group g in region r for the direction Omega is
 *            Q(Omega) = Q0 + 3 (Omega_x Q1x + Omega_y Q1y),
 *            Q0  = (1/4pi) ( sum_g' Ss0[g][g'] phi_g' + chi_g/k sum_g' nuSf_g' phi_g' ),
 *            Q1x = (1/4pi) sum_g' Ss1[g][g'] Jx_g'      (Q1y alike),   J = integral of Omega psi dOmega.
 *   P-2  2-D extruded geometry: J_z = 0 by the up/down symmetry, the polar quadrature of the upper hemisphere stands for
 *        both; Omega_xy = sin(theta_p) (u_x, u_y) with u the unit vector of the direction of travel: from the start
 *        point of the track to its end point for d = 0, reversed for d = 1.
 *   P-3  Eq. (5) with q = Q(Omega)/Sigma_t for the chain's own direction:  D = (psi - Q(Omega)/Sigma_t)(1 - exp(-tau)).
 *   P-4  tallies: tally0 += w D,  tallyx += w Omega_x D,  tallyy += w Omega_y D,   w = w_{t,p} of O-5.
 *   P-5  finalise.  With l = s / sin(theta) the 3-D length of a segment, Eq. (4) integrated over it gives
 *        Sigma_t psi_bar l = Q(Omega) l + D, and the region averages are sums of w l psi_bar (w l = 4 pi omega_a omega_p delta_a s):
 *            phi A~ Sigma_t = sum w l Q(Omega) + tally0:  the odd part of Q cancels between d = 0 and d = 1, so
 *            phi = 4 pi Q0 / Sigma_t + tally0 / (Sigma_t A~)                                   (as O-6)
 *            Jx A~ Sigma_t = sum w l Omega_x Q(Omega) + tallyx:  now the EVEN part cancels and the odd part doubles:
 *            Jx = [ 4 pi 3 c2 (Mxx Q1x + Mxy Q1y) + tallyx ] / (Sigma_t A~),   c2 = sum_p omega_p sin^2(theta_p),
 *            Mab[r] = sum over the segments k of region r of 2 omega_a delta_a s_k u_a u_b   (Mxx + Myy = A~).
 *        A~ = 0: phi = 4 pi Q0 / Sigma_t, J = 0.
 *   P-6  power iteration as O-8 with J = 0 at the start; phi, J and the boundary flux are divided by F_old.
 *
 * Pins (tests/test_oracle_p1.py): Sigma_s1 = 0 reproduces orc_sweep / orc_power_iteration; the infinite medium keeps its
 * closed-form k_inf and J = 0 whatever Sigma_s1 is; one sweep of a uniform anisotropic source in a vacuum rectangle against
 * a Monte-Carlo integration of the integral transport equation (phi, Jx, Jy: the factor 3, the direction cosines, the
 * moment weights and Mab); Mxx + Myy = A~; a diffusive bare rectangle has the eigenvalue of its transport-corrected
 * isotropic twin (Sigma_tr = Sigma_t - Sigma_s1) and not that of the uncorrected one.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_OK 0
#define ORC_ERR_ARG 1
#define ORC_ERR_MEM 4

static const double P1_PI = 3.14159265358979323846;

/* P-5: Mxx, Mxy, Myy [R] from the segments; track_dir [T][2] = unit vector from the start to the end point of a track */
int orc_p1_moments(int R, int T, const int64_t *seg_offset, const int *seg_region, const double *seg_length,
                   const double *track_weight, const double *track_dir, double *Mxx, double *Mxy, double *Myy)
{
    if (!seg_offset || !seg_region || !seg_length || !track_weight || !track_dir || !Mxx || !Mxy || !Myy || R < 1 || T < 1)
        return ORC_ERR_ARG;
    for (int r = 0; r < R; ++r) Mxx[r] = Mxy[r] = Myy[r] = 0.0;
    for (int t = 0; t < T; ++t) {
        double ux = track_dir[2 * t], uy = track_dir[2 * t + 1];
        for (int64_t k = seg_offset[t]; k < seg_offset[t + 1]; ++k) {
            double a = 2.0 * track_weight[t] * seg_length[k];
            int r = seg_region[k];
            Mxx[r] += a * ux * ux;
            Mxy[r] += a * ux * uy;
            Myy[r] += a * uy * uy;
        }
    }
    return ORC_OK;
}

/* P-1: Q0 as O-7; Q1x, Q1y from the currents.  sigma_s1 [M][g][g'] (from g' into g) */
int orc_p1_source(int R, int M, int G, const int *region_material, const double *sigma_s0, const double *sigma_s1,
                  const double *nu_sigma_f, const double *chi, const double *phi, const double *Jx, const double *Jy, double k,
                  double *Q0, double *Q1x, double *Q1y)
{
    if (!region_material || !sigma_s0 || !sigma_s1 || !nu_sigma_f || !chi || !phi || !Jx || !Jy || !Q0 || !Q1x || !Q1y || !(k > 0.0))
        return ORC_ERR_ARG;
    (void)M;
    for (int r = 0; r < R; ++r) {
        int m = region_material[r];
        double fis = 0.0;
        for (int gp = 0; gp < G; ++gp) fis += nu_sigma_f[(size_t)m * G + gp] * phi[(size_t)r * G + gp];
        for (int g = 0; g < G; ++g) {
            double s0 = 0.0, sx = 0.0, sy = 0.0;
            for (int gp = 0; gp < G; ++gp) {
                s0 += sigma_s0[((size_t)m * G + g) * G + gp] * phi[(size_t)r * G + gp];
                sx += sigma_s1[((size_t)m * G + g) * G + gp] * Jx[(size_t)r * G + gp];
                sy += sigma_s1[((size_t)m * G + g) * G + gp] * Jy[(size_t)r * G + gp];
            }
            Q0[(size_t)r * G + g] = (s0 + chi[(size_t)m * G + g] / k * fis) / (4.0 * P1_PI);
            Q1x[(size_t)r * G + g] = sx / (4.0 * P1_PI);
            Q1y[(size_t)r * G + g] = sy / (4.0 * P1_PI);
        }
    }
    return ORC_OK;
}

/* P-2..P-5: one sweep.  Outputs phi, Jx, Jy [R][G], psi_next [T][2][P][G]; tallies (may be NULL) [3][R][G]. */
int orc_p1_sweep(int R, int M, int G, int P, int T, const int *region_material, const double *sigma_t, const double *polar_sin,
                 const double *polar_weight, const int64_t *seg_offset, const int *seg_region, const double *seg_length,
                 const double *track_weight, const double *track_dir, const int *link, const double *volume, const double *Mxx,
                 const double *Mxy, const double *Myy, const double *Q0, const double *Q1x, const double *Q1y,
                 const double *psi_in, double *phi_out, double *Jx_out, double *Jy_out, double *psi_next, double *tally_out,
                 int n_threads)
{
    if (!region_material || !sigma_t || !polar_sin || !polar_weight || !seg_offset || !seg_region || !seg_length || !track_weight ||
        !track_dir || !link || !volume || !Mxx || !Mxy || !Myy || !Q0 || !Q1x || !Q1y || !psi_in || !phi_out || !Jx_out || !Jy_out ||
        !psi_next || R < 1 || M < 1 || G < 1 || P < 1 || T < 1)
        return ORC_ERR_ARG;
    size_t RG = (size_t)R * (size_t)G, PG = (size_t)P * (size_t)G;
    int nth = 1;
#ifdef _OPENMP
    nth = n_threads > 0 ? n_threads : omp_get_max_threads();
#endif
    double *priv = (double *)calloc(3 * RG * (size_t)nth, sizeof(double));
    if (!priv) return ORC_ERR_MEM;
    memset(psi_next, 0, sizeof(double) * (size_t)T * 2 * PG);
#pragma omp parallel num_threads(nth)
    {
        int me = 0;
#ifdef _OPENMP
        me = omp_get_thread_num();
#endif
        double *t0 = priv + 3 * RG * (size_t)me, *tx = t0 + RG, *ty = tx + RG;
#pragma omp for schedule(dynamic, 16)
        for (int t = 0; t < T; ++t) {
            int64_t k0 = seg_offset[t], k1 = seg_offset[t + 1];
            for (int d = 0; d < 2; ++d) {
                double sgn = d == 0 ? 1.0 : -1.0;
                for (int p = 0; p < P; ++p) {
                    double w = 4.0 * P1_PI * track_weight[t] * polar_weight[p] * polar_sin[p];
                    double ox = sgn * polar_sin[p] * track_dir[2 * t], oy = sgn * polar_sin[p] * track_dir[2 * t + 1]; /* P-2 */
                    for (int g = 0; g < G; ++g) {
                        double psi = psi_in[((size_t)t * 2 + d) * PG + (size_t)p * G + g];
                        for (int64_t q = 0; q < k1 - k0; ++q) {
                            int64_t k = d == 0 ? k0 + q : k1 - 1 - q;
                            int r = seg_region[k];
                            size_t i = (size_t)r * G + g;
                            double st = sigma_t[(size_t)region_material[r] * G + g];
                            double tau = st * seg_length[k] / polar_sin[p];
                            double Qdir = Q0[i] + 3.0 * (ox * Q1x[i] + oy * Q1y[i]);                /* P-1 */
                            double D = (psi - Qdir / st) * (-expm1(-tau));                          /* P-3 */
                            psi -= D;
                            t0[i] += w * D;                                                          /* P-4 */
                            tx[i] += w * ox * D;
                            ty[i] += w * oy * D;
                        }
                        int lk = link[2 * t + d];
                        if (lk >= 0) psi_next[(size_t)lk * PG + (size_t)p * G + g] = psi;
                    }
                }
            }
        }
    }
    for (int th = 1; th < nth; ++th) /* fixed-order reduction */
        for (size_t i = 0; i < 3 * RG; ++i) priv[i] += priv[3 * RG * (size_t)th + i];
    double c2 = 0.0;
    for (int p = 0; p < P; ++p) c2 += polar_weight[p] * polar_sin[p] * polar_sin[p];
    for (int r = 0; r < R; ++r)
        for (int g = 0; g < G; ++g) {                                                               /* P-5 */
            size_t i = (size_t)r * G + g;
            double st = sigma_t[(size_t)region_material[r] * G + g];
            double phi = 4.0 * P1_PI * Q0[i] / st, jx = 0.0, jy = 0.0;
            if (volume[r] > 0.0) {
                phi += priv[i] / (st * volume[r]);
                jx = (4.0 * P1_PI * 3.0 * c2 * (Mxx[r] * Q1x[i] + Mxy[r] * Q1y[i]) + priv[RG + i]) / (st * volume[r]);
                jy = (4.0 * P1_PI * 3.0 * c2 * (Mxy[r] * Q1x[i] + Myy[r] * Q1y[i]) + priv[2 * RG + i]) / (st * volume[r]);
            }
            phi_out[i] = phi; Jx_out[i] = jx; Jy_out[i] = jy;
        }
    if (tally_out) memcpy(tally_out, priv, sizeof(double) * 3 * RG);
    free(priv);
    return ORC_OK;
}

/* P-6.  phi_io, Jx_io, Jy_io [R][G], psi_io [T][2][P][G]: starting state if resume != 0, else initialised here. */
int orc_p1_power_iteration(int R, int M, int G, int P, int T, const int *region_material, const double *sigma_t,
                           const double *sigma_s0, const double *sigma_s1, const double *nu_sigma_f, const double *chi,
                           const double *polar_sin, const double *polar_weight, const int64_t *seg_offset, const int *seg_region,
                           const double *seg_length, const double *track_weight, const double *track_dir, const int *link,
                           const double *volume, int n_iters, int resume, double *k_io, double *phi_io, double *Jx_io,
                           double *Jy_io, double *psi_io, double *k_history, int n_threads)
{
    if (!k_io || !phi_io || !Jx_io || !Jy_io || !psi_io || n_iters < 0 || !nu_sigma_f || !volume) return ORC_ERR_ARG;
    size_t RG = (size_t)R * G, NPSI = (size_t)T * 2 * P * G;
    double *buf = (double *)malloc(sizeof(double) * (6 * RG + 3 * (size_t)R));
    double *psi_next = (double *)malloc(sizeof(double) * NPSI);
    if (!buf || !psi_next) { free(buf); free(psi_next); return ORC_ERR_MEM; }
    double *Q0 = buf, *Q1x = Q0 + RG, *Q1y = Q1x + RG, *phi_new = Q1y + RG, *Jx_new = phi_new + RG, *Jy_new = Jx_new + RG;
    double *Mxx = Jy_new + RG, *Mxy = Mxx + R, *Myy = Mxy + R;
    int rc = orc_p1_moments(R, T, seg_offset, seg_region, seg_length, track_weight, track_dir, Mxx, Mxy, Myy);
    double k = resume ? *k_io : 1.0;
    if (!resume) {
        for (size_t i = 0; i < RG; ++i) { phi_io[i] = 1.0; Jx_io[i] = 0.0; Jy_io[i] = 0.0; }
        for (size_t i = 0; i < NPSI; ++i) psi_io[i] = 0.0;
    }
    for (int it = 0; it < n_iters && rc == ORC_OK; ++it) {
        double F_old = 0.0;
        for (int r = 0; r < R; ++r) {
            double f = 0.0;
            for (int g = 0; g < G; ++g) f += nu_sigma_f[(size_t)region_material[r] * G + g] * phi_io[(size_t)r * G + g];
            F_old += volume[r] * f;
        }
        if (!(F_old > 0.0)) { rc = ORC_ERR_ARG; break; }
        for (size_t i = 0; i < RG; ++i) { phi_io[i] /= F_old; Jx_io[i] /= F_old; Jy_io[i] /= F_old; }
        for (size_t i = 0; i < NPSI; ++i) psi_io[i] /= F_old;
        rc = orc_p1_source(R, M, G, region_material, sigma_s0, sigma_s1, nu_sigma_f, chi, phi_io, Jx_io, Jy_io, k, Q0, Q1x, Q1y);
        if (rc != ORC_OK) break;
        rc = orc_p1_sweep(R, M, G, P, T, region_material, sigma_t, polar_sin, polar_weight, seg_offset, seg_region, seg_length,
                          track_weight, track_dir, link, volume, Mxx, Mxy, Myy, Q0, Q1x, Q1y, psi_io, phi_new, Jx_new, Jy_new,
                          psi_next, NULL, n_threads);
        if (rc != ORC_OK) break;
        double F_new = 0.0;
        for (int r = 0; r < R; ++r) {
            double f = 0.0;
            for (int g = 0; g < G; ++g) f += nu_sigma_f[(size_t)region_material[r] * G + g] * phi_new[(size_t)r * G + g];
            F_new += volume[r] * f;
        }
        k = k * F_new;
        memcpy(phi_io, phi_new, sizeof(double) * RG);
        memcpy(Jx_io, Jx_new, sizeof(double) * RG);
        memcpy(Jy_io, Jy_new, sizeof(double) * RG);
        memcpy(psi_io, psi_next, sizeof(double) * NPSI);
        if (k_history) k_history[it] = k;
    }
    *k_io = k;
    free(buf); free(psi_next);
    return rc;
}
