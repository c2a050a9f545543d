/*
 * oracle/moc_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, FP64 CPU statement of the planar Method-of-Characteristics hot path of
 * arxiv/paper_2607_01591 (NuDEAL), written from the paper step by step.  It exists only to check the
 * CUDA path (tests/, __graft_entry__.smoke(), bench.py's cpu_baseline / --impl reference leg).  It
 * shares no code, header, table or helper with paper_2607_01591_b200/ and must never be linked,
 * imported or called by it.
 *
 * Passages followed (line numbers of /root/reference/PAPER.md):
 *   Eq. (1)  PAPER.md:45-51   multigroup eigen-equation: scattering + chi/k * fission source
 *   Eq. (3)  PAPER.md:57-61   element-wise form (one element = one flat-source region)
 *   Eq. (4)  PAPER.md:67      characteristic ODE
 *   Eq. (5)  PAPER.md:71      flat-source segment solution psi(s) = psi(0)e^{-St s} + q/St (1-e^{-St s})
 *   PAPER.md:73               scalar flux = angular integration over all discrete directions
 *   PAPER.md:169-174          half-edge mesh, modular rays on the bounding box of the whole domain,
 *                             ray-mesh intersection computed once
 *   PAPER.md:31,176           Jacobi sweeping in energy
 * The paper is silent on quadrature, track laydown, volumes, boundary update order, the k update and
 * the initial guess; the readings used here are the ones listed in DESIGN.md "Readings" (R-T, R-W,
 * O-5..O-8) and nothing else.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): single-track attenuation closed form; telescoping and
 * particle-balance invariants; infinite-medium k_inf closed form; pure-absorber flux; the vacuum
 * rectangle worked example against an escape-probability Monte Carlo and an independent per-track
 * closed form; brute-force triangle clipping for the ray walker; laydown integer invariants.
 * O-9 (coarse-mesh net currents for CMFD, with oracle/cmfd.py; tests/test_oracle_cmfd.py): exact per-cell balance of
 * the tallied currents, exact coarse balance at the collapsed flux, closed-form k_inf in one step, unchanged fixed point.
 * "parity unpinned": heterogeneous eigenvalues of configs 1-5 have no external truth.
 *
 * Build: gcc -O2 -std=c11 -ffp-contract=off -fopenmp -shared -fPIC  (no -ffast-math, no -march).
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
#define ORC_ERR_MESH 2
#define ORC_ERR_WALK 3
#define ORC_ERR_MEM 4

static const double ORC_PI = 3.14159265358979323846;

/* ------------------------------------------------------------------------------------------------
 * O-2  Track laydown (rule R-T): integer-indexed cyclic tracks on the bounding rectangle.
 * ---------------------------------------------------------------------------------------------- */
typedef struct {
    int nx, ny;          /* tracks starting on the bottom side / on the left (Q1) or right (Q2) side */
    double dx, dy, h;    /* slot widths and sqrt(dx^2+dy^2) */
    double ux, uy;       /* unit forward direction, uy > 0 */
    double delta;        /* effective spacing dx*dy/h */
    double phi;          /* effective angle atan2(dy,dx) of the first-quadrant partner (weights only) */
    double omega;        /* azimuthal weight per direction, sum over N_a directions = 1 */
    int first;           /* global id of track 0 of this angle */
    int quadrant2;       /* 0: u = (+dx,+dy)/h ; 1: u = (-dx,+dy)/h */
} orc_angle;

struct orc_tracks {
    int n_azim, n_half, n_tracks, n_regions;
    int64_t n_segs;
    orc_angle *ang;       /* [n_half] */
    int *track_azim;      /* [T] track-angle index j */
    double *track_weight; /* [T] omega_a * delta_a */
    double *ends;         /* [T][4] x0,y0,x1,y1 */
    int *key;             /* [T][4] start side, start slot, end side, end slot */
    int *link;            /* [T][2] */
    int64_t *seg_offset;  /* [T+1] */
    int *seg_region;      /* [S] */
    double *seg_length;   /* [S] */
    double *volume;       /* [R] track-estimated areas */
};
typedef struct orc_tracks orc_tracks;

enum { SIDE_LEFT = 0, SIDE_RIGHT = 1, SIDE_BOTTOM = 2, SIDE_TOP = 3 };

static void side_point(int side, int slot, const orc_angle *a, double W, double H, double *x, double *y)
{
    /* end points come from the half-integer slot, never from marching */
    switch (side) {
    case SIDE_LEFT:   *x = 0.0; *y = ((double)slot + 0.5) * a->dy; break;
    case SIDE_RIGHT:  *x = W;   *y = ((double)slot + 0.5) * a->dy; break;
    case SIDE_BOTTOM: *x = ((double)slot + 0.5) * a->dx; *y = 0.0; break;
    default:          *x = ((double)slot + 0.5) * a->dx; *y = H;   break;
    }
}

static int laydown(orc_tracks *tr, double W, double H, int n_azim, double spacing, const int *bc)
{
    int nq = n_azim / 4, nh = n_azim / 2;
    tr->n_azim = n_azim;
    tr->n_half = nh;
    tr->ang = (orc_angle *)calloc((size_t)nh, sizeof(orc_angle));
    if (!tr->ang) return ORC_ERR_MEM;
    for (int a = 0; a < nq; ++a) {
        double phi_des = (2.0 * ORC_PI / (double)n_azim) * ((double)a + 0.5);
        orc_angle *q = &tr->ang[a];
        q->nx = (int)floor((W / spacing) * sin(phi_des)) + 1;
        q->ny = (int)floor((H / spacing) * cos(phi_des)) + 1;
        q->dx = W / (double)q->nx;
        q->dy = H / (double)q->ny;
        q->h = sqrt(q->dx * q->dx + q->dy * q->dy);
        q->ux = q->dx / q->h;
        q->uy = q->dy / q->h;
        q->delta = q->dx * q->dy / q->h;
        q->phi = atan2(q->dy, q->dx);
        q->quadrant2 = 0;
    }
    for (int a = 1; a < nq; ++a)
        if (!(tr->ang[a].phi > tr->ang[a - 1].phi)) return ORC_ERR_ARG; /* effective angles must increase */
    for (int a = 0; a < nq; ++a) {
        double b_lo = (a == 0) ? 0.0 : 0.5 * (tr->ang[a - 1].phi + tr->ang[a].phi);
        double b_hi = (a == nq - 1) ? 0.5 * ORC_PI : 0.5 * (tr->ang[a].phi + tr->ang[a + 1].phi);
        tr->ang[a].omega = (b_hi - b_lo) / (2.0 * ORC_PI);
    }
    for (int j = nq; j < nh; ++j) { /* complement angles: mirror of a = nh-1-j */
        tr->ang[j] = tr->ang[nh - 1 - j];
        tr->ang[j].ux = -tr->ang[j].ux;
        tr->ang[j].quadrant2 = 1;
    }
    int T = 0;
    for (int j = 0; j < nh; ++j) { tr->ang[j].first = T; T += tr->ang[j].nx + tr->ang[j].ny; }
    tr->n_tracks = T;
    tr->track_azim = (int *)malloc(sizeof(int) * (size_t)T);
    tr->track_weight = (double *)malloc(sizeof(double) * (size_t)T);
    tr->ends = (double *)malloc(sizeof(double) * 4 * (size_t)T);
    tr->key = (int *)malloc(sizeof(int) * 4 * (size_t)T);
    tr->link = (int *)malloc(sizeof(int) * 2 * (size_t)T);
    if (!tr->track_azim || !tr->track_weight || !tr->ends || !tr->key || !tr->link) return ORC_ERR_MEM;

    for (int j = 0; j < nh; ++j) {
        const orc_angle *a = &tr->ang[j];
        int nx = a->nx, ny = a->ny;
        for (int i = 0; i < nx + ny; ++i) {
            int t = a->first + i;
            int s_side, s_slot, e_side, e_slot;
            if (!a->quadrant2) {
                if (i < nx) { /* from bottom slot i */
                    s_side = SIDE_BOTTOM; s_slot = i;
                    int jp = nx - i - 1;
                    if (jp <= ny - 1) { e_side = SIDE_RIGHT; e_slot = jp; }
                    else              { e_side = SIDE_TOP;   e_slot = i + ny; }
                } else {      /* from left slot jl */
                    int jl = i - nx;
                    s_side = SIDE_LEFT; s_slot = jl;
                    int k = ny - jl - 1;
                    if (k <= nx - 1) { e_side = SIDE_TOP;   e_slot = k; }
                    else             { e_side = SIDE_RIGHT; e_slot = jl + nx; }
                }
            } else {
                if (i < nx) { /* from bottom slot i, heading up-left */
                    s_side = SIDE_BOTTOM; s_slot = i;
                    if (i <= ny - 1) { e_side = SIDE_LEFT; e_slot = i; }
                    else             { e_side = SIDE_TOP;  e_slot = i - ny; }
                } else {      /* from right slot jr */
                    int jr = i - nx;
                    s_side = SIDE_RIGHT; s_slot = jr;
                    int k = nx - ny + jr;
                    if (k >= 0) { e_side = SIDE_TOP;  e_slot = k; }
                    else        { e_side = SIDE_LEFT; e_slot = jr + nx; }
                }
            }
            tr->key[4 * t + 0] = s_side; tr->key[4 * t + 1] = s_slot;
            tr->key[4 * t + 2] = e_side; tr->key[4 * t + 3] = e_slot;
            side_point(s_side, s_slot, a, W, H, &tr->ends[4 * t + 0], &tr->ends[4 * t + 1]);
            side_point(e_side, e_slot, a, W, H, &tr->ends[4 * t + 2], &tr->ends[4 * t + 3]);
            tr->track_azim[t] = j;
            tr->track_weight[t] = a->omega * a->delta;
        }
    }
    /* O-3 links: reflection maps angle j to nh-1-j; the partner is the track of that angle with the
     * same (side, slot) key; key is its start -> enter forward (d'=0); its end -> enter backward. */
    for (int j = 0; j < nh; ++j) {
        const orc_angle *a = &tr->ang[j];
        const orc_angle *c = &tr->ang[nh - 1 - j];
        int n = a->nx + a->ny; /* same for the complement */
        int nslot = (a->nx > a->ny ? a->nx : a->ny);
        int *start_of = (int *)malloc(sizeof(int) * 4 * (size_t)nslot);
        int *end_of = (int *)malloc(sizeof(int) * 4 * (size_t)nslot);
        if (!start_of || !end_of) return ORC_ERR_MEM;
        for (int q = 0; q < 4 * nslot; ++q) { start_of[q] = -1; end_of[q] = -1; }
        for (int i = 0; i < n; ++i) {
            int t = c->first + i;
            start_of[tr->key[4 * t + 0] * nslot + tr->key[4 * t + 1]] = t;
            end_of[tr->key[4 * t + 2] * nslot + tr->key[4 * t + 3]] = t;
        }
        for (int i = 0; i < n; ++i) {
            int t = a->first + i;
            for (int d = 0; d < 2; ++d) {
                int side = d == 0 ? tr->key[4 * t + 2] : tr->key[4 * t + 0];
                int slot = d == 0 ? tr->key[4 * t + 3] : tr->key[4 * t + 1];
                int lk = -1;
                if (bc[side] != 0) {
                    int ts = start_of[side * nslot + slot], te = end_of[side * nslot + slot];
                    if (ts >= 0) lk = 2 * ts + 0;
                    else if (te >= 0) lk = 2 * te + 1;
                    else { free(start_of); free(end_of); return ORC_ERR_ARG; }
                }
                tr->link[2 * t + d] = lk;
            }
        }
        free(start_of);
        free(end_of);
    }
    return ORC_OK;
}

/* ------------------------------------------------------------------------------------------------
 * Half-edge connectivity: local edge e of triangle t runs v_e -> v_{(e+1)%3};
 * nbr[3t+e] = triangle across that edge or -1 on the boundary.
 * ---------------------------------------------------------------------------------------------- */
typedef struct { int a, b, t, e; } edge_rec;

static int edge_cmp(const void *p, const void *q)
{
    const edge_rec *x = (const edge_rec *)p, *y = (const edge_rec *)q;
    if (x->a != y->a) return x->a < y->a ? -1 : 1;
    if (x->b != y->b) return x->b < y->b ? -1 : 1;
    return 0;
}

typedef struct { double lo, hi; int t; } bedge;

static int bedge_cmp(const void *p, const void *q)
{
    const bedge *x = (const bedge *)p, *y = (const bedge *)q;
    if (x->lo != y->lo) return x->lo < y->lo ? -1 : 1;
    return 0;
}

typedef struct {
    int nR;
    const double *xy;
    const int *tri;
    int *nbr;
    bedge *side[4];
    int n_side[4];
} heds;

static void heds_free(heds *m)
{
    free(m->nbr);
    for (int s = 0; s < 4; ++s) free(m->side[s]);
}

static int heds_build(heds *m, int nV, int nR, const double *xy, const int *tri, double W, double H)
{
    memset(m, 0, sizeof(*m));
    m->nR = nR; m->xy = xy; m->tri = tri;
    size_t nE = 3 * (size_t)nR;
    edge_rec *er = (edge_rec *)malloc(sizeof(edge_rec) * nE);
    m->nbr = (int *)malloc(sizeof(int) * nE);
    if (!er || !m->nbr) { free(er); return ORC_ERR_MEM; }
    for (int t = 0; t < nR; ++t)
        for (int e = 0; e < 3; ++e) {
            int v0 = tri[3 * t + e], v1 = tri[3 * t + (e + 1) % 3];
            if (v0 < 0 || v0 >= nV || v1 < 0 || v1 >= nV || v0 == v1) { free(er); return ORC_ERR_MESH; }
            edge_rec *r = &er[3 * (size_t)t + e];
            r->a = v0 < v1 ? v0 : v1; r->b = v0 < v1 ? v1 : v0; r->t = t; r->e = e;
            m->nbr[3 * (size_t)t + e] = -1;
        }
    qsort(er, nE, sizeof(edge_rec), edge_cmp);
    int nb[4] = {0, 0, 0, 0};
    for (size_t i = 0; i < nE;) {
        size_t k = i + 1;
        while (k < nE && er[k].a == er[i].a && er[k].b == er[i].b) ++k;
        if (k - i == 2) {
            m->nbr[3 * (size_t)er[i].t + er[i].e] = er[i + 1].t;
            m->nbr[3 * (size_t)er[i + 1].t + er[i + 1].e] = er[i].t;
        } else if (k - i != 1) { free(er); return ORC_ERR_MESH; }
        i = k;
    }
    /* boundary half-edges per side, sorted by along-side coordinate */
    for (int pass = 0; pass < 2; ++pass) {
        int cnt[4] = {0, 0, 0, 0};
        for (size_t i = 0; i < nE; ++i) {
            int t = er[i].t, e = er[i].e;
            if (m->nbr[3 * (size_t)t + e] >= 0) continue;
            const double *pa = &xy[2 * er[i].a], *pb = &xy[2 * er[i].b];
            int s; double c0, c1;
            if (pa[0] == 0.0 && pb[0] == 0.0)      { s = SIDE_LEFT;   c0 = pa[1]; c1 = pb[1]; }
            else if (pa[0] == W && pb[0] == W)     { s = SIDE_RIGHT;  c0 = pa[1]; c1 = pb[1]; }
            else if (pa[1] == 0.0 && pb[1] == 0.0) { s = SIDE_BOTTOM; c0 = pa[0]; c1 = pb[0]; }
            else if (pa[1] == H && pb[1] == H)     { s = SIDE_TOP;    c0 = pa[0]; c1 = pb[0]; }
            else { free(er); return ORC_ERR_MESH; }
            if (pass == 1) {
                bedge *b = &m->side[s][cnt[s]];
                b->lo = c0 < c1 ? c0 : c1; b->hi = c0 < c1 ? c1 : c0; b->t = t;
            }
            ++cnt[s];
        }
        if (pass == 0)
            for (int s = 0; s < 4; ++s) {
                nb[s] = cnt[s];
                m->n_side[s] = cnt[s];
                m->side[s] = (bedge *)malloc(sizeof(bedge) * (size_t)(cnt[s] > 0 ? cnt[s] : 1));
                if (!m->side[s]) { free(er); return ORC_ERR_MEM; }
            }
    }
    (void)nb;
    free(er);
    for (int s = 0; s < 4; ++s) {
        if (m->n_side[s] == 0) return ORC_ERR_MESH;
        qsort(m->side[s], (size_t)m->n_side[s], sizeof(bedge), bedge_cmp);
    }
    return ORC_OK;
}

/* start triangle: the boundary half-edge on `side` whose half-open interval [lo,hi) contains c
 * (the last edge of the side is closed) */
static int start_triangle(const heds *m, int side, double c)
{
    const bedge *b = m->side[side];
    int n = m->n_side[side], lo = 0, hi = n - 1;
    while (lo < hi) { /* largest index with b[idx].lo <= c */
        int mid = (lo + hi + 1) / 2;
        if (b[mid].lo <= c) lo = mid; else hi = mid - 1;
    }
    return b[lo].t;
}

/* ------------------------------------------------------------------------------------------------
 * O-4  Ray walk (rule R-W).  Canonical-edge lambda measured from the track origin; exit edge = the
 * candidate (u.n > 0, strict) with the smallest lambda, tie -> lower local edge index; segments
 * with s <= 0 are skipped, the walk continues.  If out_region == NULL only counts.
 * ---------------------------------------------------------------------------------------------- */
static int64_t walk_track(const heds *m, int start_side, double x0, double y0, double ux, double uy,
                          int *out_region, double *out_length, double *lambda_last)
{
    const double *xy = m->xy;
    const int *tri = m->tri;
    double c = (start_side == SIDE_BOTTOM || start_side == SIDE_TOP) ? x0 : y0;
    int t = start_triangle(m, start_side, c);
    double lam_in = 0.0;
    int64_t n = 0, steps = 0, max_steps = 4 * (int64_t)m->nR + 16;
    for (;;) {
        int best = -1;
        double best_lam = 0.0;
        for (int e = 0; e < 3; ++e) {
            int v0 = tri[3 * t + e], v1 = tri[3 * t + (e + 1) % 3];
            double ex = xy[2 * v1] - xy[2 * v0], ey = xy[2 * v1 + 1] - xy[2 * v0 + 1];
            double test = ux * ey - uy * ex; /* u . outward normal of the CCW edge */
            if (test > 0.0) {
                int a = v0 < v1 ? v0 : v1, b = v0 < v1 ? v1 : v0;
                double Ex = xy[2 * b] - xy[2 * a], Ey = xy[2 * b + 1] - xy[2 * a + 1];
                double den = ux * Ey - uy * Ex;
                double num = (xy[2 * a] - x0) * Ey - (xy[2 * a + 1] - y0) * Ex;
                double lam = num / den;
                if (best < 0 || lam < best_lam) { best = e; best_lam = lam; }
            }
        }
        if (best < 0) return -1;
        double s = best_lam - lam_in;
        if (s > 0.0) {
            if (out_region) { out_region[n] = t; out_length[n] = s; }
            ++n;
        }
        lam_in = best_lam;
        int nt = m->nbr[3 * (size_t)t + best];
        if (nt < 0) break;
        t = nt;
        if (++steps > max_steps) return -1;
    }
    if (lambda_last) *lambda_last = lam_in;
    return n;
}

void orc_tracks_free(orc_tracks *tr)
{
    if (!tr) return;
    free(tr->ang); free(tr->track_azim); free(tr->track_weight); free(tr->ends); free(tr->key);
    free(tr->link); free(tr->seg_offset); free(tr->seg_region); free(tr->seg_length); free(tr->volume);
    free(tr);
}

/* bc[4] = left,right,bottom,top ; 0 vacuum, 1 reflective */
int orc_tracks_generate(int nV, int nR, const double *xy, const int *tri, double W, double H, const int *bc,
                        int n_azim, double spacing, int n_threads, orc_tracks **out)
{
    if (!xy || !tri || !bc || !out || nV < 3 || nR < 1 || !(W > 0.0) || !(H > 0.0) || !(spacing > 0.0) ||
        n_azim < 4 || n_azim % 4 != 0)
        return ORC_ERR_ARG;
    orc_tracks *tr = (orc_tracks *)calloc(1, sizeof(orc_tracks));
    if (!tr) return ORC_ERR_MEM;
    tr->n_regions = nR;
    int rc = laydown(tr, W, H, n_azim, spacing, bc);
    if (rc != ORC_OK) { orc_tracks_free(tr); return rc; }
    heds m;
    rc = heds_build(&m, nV, nR, xy, tri, W, H);
    if (rc != ORC_OK) { heds_free(&m); orc_tracks_free(tr); return rc; }
    int T = tr->n_tracks;
    tr->seg_offset = (int64_t *)calloc((size_t)T + 1, sizeof(int64_t));
    if (!tr->seg_offset) { heds_free(&m); orc_tracks_free(tr); return ORC_ERR_MEM; }
    int bad = 0;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
    /* pass 1: count, pass 2: fill (the walk is deterministic, both passes take identical steps) */
#pragma omp parallel for schedule(dynamic, 64) reduction(| : bad)
    for (int t = 0; t < T; ++t) {
        const orc_angle *a = &tr->ang[tr->track_azim[t]];
        int64_t n = walk_track(&m, tr->key[4 * t], tr->ends[4 * t], tr->ends[4 * t + 1], a->ux, a->uy, NULL, NULL, NULL);
        if (n < 0) { bad |= 1; n = 0; }
        tr->seg_offset[t + 1] = n;
    }
    if (bad) { heds_free(&m); orc_tracks_free(tr); return ORC_ERR_WALK; }
    for (int t = 0; t < T; ++t) tr->seg_offset[t + 1] += tr->seg_offset[t];
    tr->n_segs = tr->seg_offset[T];
    tr->seg_region = (int *)malloc(sizeof(int) * (size_t)(tr->n_segs > 0 ? tr->n_segs : 1));
    tr->seg_length = (double *)malloc(sizeof(double) * (size_t)(tr->n_segs > 0 ? tr->n_segs : 1));
    tr->volume = (double *)calloc((size_t)nR, sizeof(double));
    if (!tr->seg_region || !tr->seg_length || !tr->volume) { heds_free(&m); orc_tracks_free(tr); return ORC_ERR_MEM; }
#pragma omp parallel for schedule(dynamic, 64)
    for (int t = 0; t < T; ++t) {
        const orc_angle *a = &tr->ang[tr->track_azim[t]];
        int64_t o = tr->seg_offset[t];
        walk_track(&m, tr->key[4 * t], tr->ends[4 * t], tr->ends[4 * t + 1], a->ux, a->uy,
                   tr->seg_region + o, tr->seg_length + o, NULL);
    }
    heds_free(&m);
    /* O-5 track-estimated areas: A~_r = sum over segments in r of 2 * omega_a * delta_a * s */
    for (int t = 0; t < T; ++t)
        for (int64_t k = tr->seg_offset[t]; k < tr->seg_offset[t + 1]; ++k)
            tr->volume[tr->seg_region[k]] += 2.0 * tr->track_weight[t] * tr->seg_length[k];
    *out = tr;
    return ORC_OK;
}

void orc_tracks_dims(const orc_tracks *tr, int *n_tracks, int64_t *n_segs, int *n_half)
{
    if (n_tracks) *n_tracks = tr->n_tracks;
    if (n_segs) *n_segs = tr->n_segs;
    if (n_half) *n_half = tr->n_half;
}

/* copies out; any destination may be NULL */
void orc_tracks_copy(const orc_tracks *tr, int64_t *seg_offset, int *seg_region, double *seg_length,
                     double *track_weight, int *link, int *track_azim, double *ends, int *keys, double *volume,
                     double *azim_phi, double *azim_weight, double *azim_spacing, int *azim_nx, int *azim_ny)
{
    size_t T = (size_t)tr->n_tracks, S = (size_t)tr->n_segs;
    if (seg_offset) memcpy(seg_offset, tr->seg_offset, sizeof(int64_t) * (T + 1));
    if (seg_region) memcpy(seg_region, tr->seg_region, sizeof(int) * S);
    if (seg_length) memcpy(seg_length, tr->seg_length, sizeof(double) * S);
    if (track_weight) memcpy(track_weight, tr->track_weight, sizeof(double) * T);
    if (link) memcpy(link, tr->link, sizeof(int) * 2 * T);
    if (track_azim) memcpy(track_azim, tr->track_azim, sizeof(int) * T);
    if (ends) memcpy(ends, tr->ends, sizeof(double) * 4 * T);
    if (keys) memcpy(keys, tr->key, sizeof(int) * 4 * T);
    if (volume) memcpy(volume, tr->volume, sizeof(double) * (size_t)tr->n_regions);
    for (int j = 0; j < tr->n_half; ++j) {
        if (azim_phi) azim_phi[j] = tr->ang[j].quadrant2 ? ORC_PI - tr->ang[j].phi : tr->ang[j].phi;
        if (azim_weight) azim_weight[j] = tr->ang[j].omega;
        if (azim_spacing) azim_spacing[j] = tr->ang[j].delta;
        if (azim_nx) azim_nx[j] = tr->ang[j].nx;
        if (azim_ny) azim_ny[j] = tr->ang[j].ny;
    }
}

/* O-5 for caller-supplied tracks */
int orc_track_volumes(int R, int T, const int64_t *seg_offset, const int *seg_region, const double *seg_length,
                      const double *track_weight, double *volume)
{
    if (!seg_offset || !seg_region || !seg_length || !track_weight || !volume) return ORC_ERR_ARG;
    for (int r = 0; r < R; ++r) volume[r] = 0.0;
    for (int t = 0; t < T; ++t)
        for (int64_t k = seg_offset[t]; k < seg_offset[t + 1]; ++k) {
            if (seg_region[k] < 0 || seg_region[k] >= R) return ORC_ERR_ARG;
            volume[seg_region[k]] += 2.0 * track_weight[t] * seg_length[k];
        }
    return ORC_OK;
}

/* ------------------------------------------------------------------------------------------------
 * O-6  Transport sweep.  For every track t, direction d, polar p, group g:
 *        psi <- psi_in[t][d][p][g]
 *        for each segment (forward order for d=0, reverse for d=1), Eq. (5) PAPER.md:71 with the 3-D
 *        path s / sin(theta_p):
 *            tau = Sigma_t[m(r)][g] * s / sin(theta_p)
 *            D   = (psi - Q[r][g]/Sigma_t) * (1 - exp(-tau))            [ = psi_in - psi_out of Eq. (5) ]
 *            psi <- psi - D ;  tally[r][g] += w_{t,p} * D ,   w_{t,p} = 4 pi * track_weight[t] * w_p * sin(theta_p)
 *        psi_next[link[t][d]] = psi  (reflective) ; vacuum ends keep psi_next = 0.
 *      Jacobi (double-buffered) boundary update: every chain reads the previous sweep's psi_in.
 *      Finalise:  phi[r][g] = 4 pi Q/Sigma_t + tally/(Sigma_t * A~_r)   (tally term 0 if A~_r = 0).
 * ---------------------------------------------------------------------------------------------- */
int orc_sweep(int R, int M, int G, int P, int T, const int *region_material, const double *sigma_t,
              const double *polar_sin, const double *polar_weight, const int64_t *seg_offset, const int *seg_region,
              const double *seg_length, const double *track_weight, const int *link, const double *volume,
              const double *Q, const double *psi_in, double *phi_out, double *psi_next, double *tally_out,
              int n_threads)
{
    if (!region_material || !sigma_t || !polar_sin || !polar_weight || !seg_offset || !seg_region || !seg_length ||
        !track_weight || !link || !volume || !Q || !psi_in || !phi_out || !psi_next || R < 1 || M < 1 || G < 1 ||
        P < 1 || T < 1)
        return ORC_ERR_ARG;
    size_t RG = (size_t)R * (size_t)G, PG = (size_t)P * (size_t)G;
    int nth = 1;
#ifdef _OPENMP
    nth = n_threads > 0 ? n_threads : omp_get_max_threads();
#endif
    double *priv = (double *)calloc(RG * (size_t)nth, sizeof(double));
    if (!priv) return ORC_ERR_MEM;
    memset(psi_next, 0, sizeof(double) * (size_t)T * 2 * PG);
#pragma omp parallel num_threads(nth)
    {
        int me = 0;
#ifdef _OPENMP
        me = omp_get_thread_num();
#endif
        double *tally = priv + RG * (size_t)me;
#pragma omp for schedule(dynamic, 16)
        for (int t = 0; t < T; ++t) {
            int64_t k0 = seg_offset[t], k1 = seg_offset[t + 1];
            for (int d = 0; d < 2; ++d)
                for (int p = 0; p < P; ++p) {
                    double w = 4.0 * ORC_PI * track_weight[t] * polar_weight[p] * polar_sin[p];
                    for (int g = 0; g < G; ++g) {
                        double psi = psi_in[((size_t)t * 2 + d) * PG + (size_t)p * G + g];
                        for (int64_t q = 0; q < k1 - k0; ++q) {
                            int64_t k = d == 0 ? k0 + q : k1 - 1 - q;
                            int r = seg_region[k];
                            double st = sigma_t[(size_t)region_material[r] * G + g];
                            double tau = st * seg_length[k] / polar_sin[p];
                            double D = (psi - Q[(size_t)r * G + g] / st) * (-expm1(-tau));
                            psi -= D;
                            tally[(size_t)r * G + g] += w * D;
                        }
                        int lk = link[2 * t + d];
                        if (lk >= 0) psi_next[(size_t)lk * PG + (size_t)p * G + g] = psi;
                    }
                }
        }
    }
    for (int th = 1; th < nth; ++th) /* fixed-order reduction */
        for (size_t i = 0; i < RG; ++i) priv[i] += priv[RG * (size_t)th + i];
    for (int r = 0; r < R; ++r)
        for (int g = 0; g < G; ++g) {
            size_t i = (size_t)r * G + g;
            double st = sigma_t[(size_t)region_material[r] * G + g];
            double phi = 4.0 * ORC_PI * Q[i] / st;
            if (volume[r] > 0.0) phi += priv[i] / (st * volume[r]);
            phi_out[i] = phi;
            if (tally_out) tally_out[i] = priv[i];
        }
    free(priv);
    return ORC_OK;
}

/* O-7  Source, RHS of Eq. (1)/(3) divided by 4 pi (angular source per steradian), all groups from the
 * previous iterate (Jacobi in energy): Q[r][g] = (1/4pi) ( sum_g' Ss[m][g][g'] phi[r][g'] + chi[m][g]/k sum_g' nSf[m][g'] phi[r][g'] ) */
int orc_source(int R, int M, int G, const int *region_material, const double *sigma_s, const double *nu_sigma_f,
               const double *chi, const double *phi, double k, double *Q)
{
    if (!region_material || !sigma_s || !nu_sigma_f || !chi || !phi || !Q || !(k > 0.0)) return ORC_ERR_ARG;
    (void)M;
    for (int r = 0; r < R; ++r) {
        int m = region_material[r];
        double fis = 0.0;
        for (int gp = 0; gp < G; ++gp) fis += nu_sigma_f[(size_t)m * G + gp] * phi[(size_t)r * G + gp];
        for (int g = 0; g < G; ++g) {
            double sc = 0.0;
            for (int gp = 0; gp < G; ++gp) sc += sigma_s[((size_t)m * G + g) * G + gp] * phi[(size_t)r * G + gp];
            Q[(size_t)r * G + g] = (sc + chi[(size_t)m * G + g] / k * fis) / (4.0 * ORC_PI);
        }
    }
    return ORC_OK;
}

/* F = sum_r A~_r sum_g nuSigma_f phi  (fission production, Eq. (1)) */
double orc_fission_rate(int R, int G, const int *region_material, const double *nu_sigma_f, const double *volume,
                        const double *phi)
{
    double F = 0.0;
    for (int r = 0; r < R; ++r) {
        double f = 0.0;
        for (int g = 0; g < G; ++g) f += nu_sigma_f[(size_t)region_material[r] * G + g] * phi[(size_t)r * G + g];
        F += volume[r] * f;
    }
    return F;
}

/* O-8  Canonical power iteration.  phi=1, psi_in=0, k=1; each iteration: F_old; scale phi and psi_in by
 * 1/F_old; Q from O-7 with current k; sweep; F_new; k <- k*F_new; phi <- phi_new; psi_in <- psi_next.
 * phi_io / psi_io: if `resume` != 0 they hold the starting state, else they are initialised here.
 * k_history (may be NULL) receives k after every iteration. */
int orc_power_iteration(int R, int M, int G, int P, int T, const int *region_material, const double *sigma_t,
                        const double *sigma_s, const double *nu_sigma_f, const double *chi, const double *polar_sin,
                        const double *polar_weight, const int64_t *seg_offset, const int *seg_region,
                        const double *seg_length, const double *track_weight, const int *link, const double *volume,
                        int n_iters, int resume, double *k_io, double *phi_io, double *psi_io, double *k_history,
                        int n_threads)
{
    if (!k_io || !phi_io || !psi_io || n_iters < 0) return ORC_ERR_ARG;
    size_t RG = (size_t)R * G, NPSI = (size_t)T * 2 * P * G;
    double *Q = (double *)malloc(sizeof(double) * RG);
    double *phi_new = (double *)malloc(sizeof(double) * RG);
    double *psi_next = (double *)malloc(sizeof(double) * NPSI);
    if (!Q || !phi_new || !psi_next) { free(Q); free(phi_new); free(psi_next); return ORC_ERR_MEM; }
    double k = resume ? *k_io : 1.0;
    if (!resume) {
        for (size_t i = 0; i < RG; ++i) phi_io[i] = 1.0;
        for (size_t i = 0; i < NPSI; ++i) psi_io[i] = 0.0;
    }
    int rc = ORC_OK;
    for (int it = 0; it < n_iters; ++it) {
        double F_old = orc_fission_rate(R, G, region_material, nu_sigma_f, volume, phi_io);
        if (!(F_old > 0.0)) { rc = ORC_ERR_ARG; break; }
        for (size_t i = 0; i < RG; ++i) phi_io[i] /= F_old;
        for (size_t i = 0; i < NPSI; ++i) psi_io[i] /= F_old;
        rc = orc_source(R, M, G, region_material, sigma_s, nu_sigma_f, chi, phi_io, k, Q);
        if (rc != ORC_OK) break;
        rc = orc_sweep(R, M, G, P, T, region_material, sigma_t, polar_sin, polar_weight, seg_offset, seg_region,
                       seg_length, track_weight, link, volume, Q, psi_io, phi_new, psi_next, NULL, n_threads);
        if (rc != ORC_OK) break;
        double F_new = orc_fission_rate(R, G, region_material, nu_sigma_f, volume, phi_new);
        k = k * F_new;
        memcpy(phi_io, phi_new, sizeof(double) * RG);
        memcpy(psi_io, psi_next, sizeof(double) * NPSI);
        if (k_history) k_history[it] = k;
    }
    *k_io = k;
    free(Q); free(phi_new); free(psi_next);
    return rc;
}

/* ------------------------------------------------------------------------------------------------
 * O-9  Net currents of a sweep on a coarse mesh (CMFD, Algorithm 1 line 5 "Solve CMFD on the coarse
 *      mesh"; the paper gives no formula -- DESIGN.md section 8d states the reading).
 *      cell[r] maps every region to a coarse cell.  The walk is the one of O-6 (same psi_in, same Q, same
 *      w_{t,p}); wherever a chain steps from a region of cell C into a region of another cell C' the
 *      weighted angular flux crosses the interior surface {C, C'}:
 *            J_surf[s][g] += sgn * w_{t,p} * psi ,   s = index of (min(C,C'), max(C,C')) in the sorted
 *                                                    pair list,  sgn = +1 if C < C' else -1
 *      and at the exit end of a chain (track t, direction d) in cell C, with psi_in' the flux that
 *      enters the opposite direction at that same end:
 *            J_end[C][g] += w_{t,p} * (psi_exit - psi_in')       into J_vac if that end is a vacuum end
 *                                                                (link[t][d] < 0), else into J_ref.
 *      A reflective end hands psi_exit to the chain link[t][d]; if that chain ENTERS in another cell C' (the two tracks
 *      meet at a mesh vertex on the boundary and rule R-W puts them into different triangles) the hand-over is a
 *      crossing of the surface {C, C'} like any other:  J_surf += sgn * w * psi_exit,  J_ref[C] -= w * psi_exit,
 *      J_ref[C'] += w * psi_exit -- so J_ref holds only what vanishes when the boundary flux has converged.
 *      Exact consequence (telescoping, checked in tests): for every cell and group
 *            sum_{r in C} tally[r][g] + sum_{s=(C,.)} J_surf - sum_{s=(.,C)} J_surf + J_vac[C] + J_ref[C] = 0.
 *      pair_lo/pair_hi: the n_pairs interior surfaces, sorted by (lo, hi), lo < hi.
 * ---------------------------------------------------------------------------------------------- */
static int64_t find_pair(int n, const int *lo, const int *hi, int a, int b)
{
    int64_t l = 0, h = n - 1;
    while (l <= h) {
        int64_t m = (l + h) / 2;
        if (lo[m] < a || (lo[m] == a && hi[m] < b)) l = m + 1;
        else if (lo[m] > a || hi[m] > b) h = m - 1;
        else return m;
    }
    return -1;
}

int orc_sweep_currents(int R, int M, int G, int P, int T, const int *region_material, const double *sigma_t,
                       const double *polar_sin, const double *polar_weight, const int64_t *seg_offset,
                       const int *seg_region, const double *seg_length, const double *track_weight, const int *link,
                       const double *Q, const double *psi_in, int n_cells, const int *cell, int n_pairs,
                       const int *pair_lo, const int *pair_hi, double *J_surf, double *J_vac, double *J_ref)
{
    if (!region_material || !sigma_t || !polar_sin || !polar_weight || !seg_offset || !seg_region || !seg_length ||
        !track_weight || !link || !Q || !psi_in || !cell || !J_surf || !J_vac || !J_ref || R < 1 || M < 1 || G < 1 ||
        P < 1 || T < 1 || n_cells < 1 || n_pairs < 0 || (n_pairs > 0 && (!pair_lo || !pair_hi)))
        return ORC_ERR_ARG;
    size_t PG = (size_t)P * (size_t)G;
    memset(J_surf, 0, sizeof(double) * (size_t)n_pairs * G);
    memset(J_vac, 0, sizeof(double) * (size_t)n_cells * G);
    memset(J_ref, 0, sizeof(double) * (size_t)n_cells * G);
    for (int t = 0; t < T; ++t) {
        int64_t k0 = seg_offset[t], k1 = seg_offset[t + 1];
        if (k1 == k0) continue;
        for (int d = 0; d < 2; ++d)
            for (int p = 0; p < P; ++p) {
                double w = 4.0 * ORC_PI * track_weight[t] * polar_weight[p] * polar_sin[p];
                for (int g = 0; g < G; ++g) {
                    double psi = psi_in[((size_t)t * 2 + d) * PG + (size_t)p * G + g];
                    int c_prev = -1;
                    for (int64_t q = 0; q < k1 - k0; ++q) {
                        int64_t k = d == 0 ? k0 + q : k1 - 1 - q;
                        int r = seg_region[k];
                        int c = cell[r];
                        if (c < 0 || c >= n_cells) return ORC_ERR_ARG;
                        if (c_prev >= 0 && c != c_prev) {
                            int a = c_prev < c ? c_prev : c, b = c_prev < c ? c : c_prev;
                            int64_t s = find_pair(n_pairs, pair_lo, pair_hi, a, b);
                            if (s < 0) return ORC_ERR_ARG;
                            J_surf[(size_t)s * G + g] += (c_prev < c ? 1.0 : -1.0) * w * psi;
                        }
                        double st = sigma_t[(size_t)region_material[r] * G + g];
                        double tau = st * seg_length[k] / polar_sin[p];
                        psi -= (psi - Q[(size_t)r * G + g] / st) * (-expm1(-tau));
                        c_prev = c;
                    }
                    double back = psi_in[((size_t)t * 2 + (1 - d)) * PG + (size_t)p * G + g];
                    int lk = link[2 * t + d];
                    double *J = lk < 0 ? J_vac : J_ref;
                    J[(size_t)c_prev * G + g] += w * (psi - back);
                    if (lk >= 0) {
                        int t2 = lk / 2, d2 = lk % 2;
                        if (t2 >= T || seg_offset[t2 + 1] == seg_offset[t2]) return ORC_ERR_ARG;
                        int c2 = cell[seg_region[d2 == 0 ? seg_offset[t2] : seg_offset[t2 + 1] - 1]];
                        if (c2 != c_prev) {
                            int a = c_prev < c2 ? c_prev : c2, b = c_prev < c2 ? c2 : c_prev;
                            int64_t s = find_pair(n_pairs, pair_lo, pair_hi, a, b);
                            if (s < 0) return ORC_ERR_ARG;
                            J_surf[(size_t)s * G + g] += (c_prev < c2 ? 1.0 : -1.0) * w * psi;
                            J_ref[(size_t)c_prev * G + g] -= w * psi;
                            J_ref[(size_t)c2 * G + g] += w * psi;
                        }
                    }
                }
            }
    }
    return ORC_OK;
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
