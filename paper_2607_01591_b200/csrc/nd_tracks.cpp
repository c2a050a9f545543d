// nd_tracks.cpp -- host preprocessing of the planar-MOC hot path (row A0 of DESIGN.md):
// cyclic track laydown on the bounding rectangle (rule R-T), reflective/vacuum links
// (O-3), ray-mesh intersection by walking a half-edge mesh (rule R-W) and the
// track-estimated region areas (O-5).
//
// Written independently of oracle/ (no shared code); only the *rules* are shared, and they fix the
// FP64 expression trees so that two implementations agree bit for bit:
//   - geometry uses only + - * / sqrt in FP64, compiled with -ffp-contract=off (no FMA fusion);
//   - an edge's intersection parameter is always computed from the TRACK ORIGIN with the edge taken
//     in canonical orientation (lower vertex id first);
//   - sin/cos appear only inside the integer track counts, atan2 only in the weights.
// Compile with:  g++ -O2 -ffp-contract=off -fopenmp   (never -ffast-math / -march=native)
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <new>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

#include "nd.h"
#include "nd_internal.h"
#include "nd_tracks_internal.h"

namespace {

constexpr double kPi = 3.14159265358979323846;

enum Side : int { kLeft = 0, kRight = 1, kBottom = 2, kTop = 3 };

using AngleSet = NdAngleSet;

struct EndKey { int side, slot; };

// Where a track of angle `a` with in-angle index i starts and ends (integer rule R-T).
inline void track_keys(const AngleSet& a, int i, EndKey& s, EndKey& e)
{
    const int nx = a.nx, ny = a.ny;
    if (!a.mirrored) {
        if (i < nx) {
            s = {kBottom, i};
            const int r = nx - 1 - i;                 // slot on the right side, if it gets there
            e = (r < ny) ? EndKey{kRight, r} : EndKey{kTop, i + ny};
        } else {
            const int l = i - nx;
            s = {kLeft, l};
            const int k = ny - 1 - l;
            e = (k < nx) ? EndKey{kTop, k} : EndKey{kRight, l + nx};
        }
    } else {
        if (i < nx) {
            s = {kBottom, i};
            e = (i < ny) ? EndKey{kLeft, i} : EndKey{kTop, i - ny};
        } else {
            const int r = i - nx;
            s = {kRight, r};
            const int k = nx - ny + r;
            e = (k >= 0) ? EndKey{kTop, k} : EndKey{kLeft, r + nx};
        }
    }
}

inline void key_point(const EndKey& k, const AngleSet& a, double W, double H, double* p)
{
    const double c = (static_cast<double>(k.slot) + 0.5) * ((k.side == kLeft || k.side == kRight) ? a.dy : a.dx);
    switch (k.side) {
    case kLeft:   p[0] = 0.0; p[1] = c; break;
    case kRight:  p[0] = W;   p[1] = c; break;
    case kBottom: p[0] = c;   p[1] = 0.0; break;
    default:      p[0] = c;   p[1] = H; break;
    }
}

// ---- half-edge mesh ------------------------------------------------------------------------------
// Half-edge h = 3*t + e runs from tri[3t+e] to tri[3t+(e+1)%3]; twin[h] = opposite half-edge or -1.
struct HalfEdgeMesh {
    int nV = 0, nT = 0;
    const double* xy = nullptr;
    const int32_t* tri = nullptr;
    std::vector<int32_t> twin;
    // canonical edge data per half-edge: origin = lower-id vertex, E = higher - lower
    std::vector<double> ax, ay, Ex, Ey;
    // CCW edge vector of the owning triangle (for the outward-normal test)
    std::vector<double> ex, ey;
    // boundary half-edges per side sorted by their lower along-side coordinate
    std::vector<double> side_lo[4];
    std::vector<int32_t> side_tri[4];
};

nd_status build_mesh(HalfEdgeMesh& m, const nd_mesh_desc* d)
{
    m.nV = d->n_vertices; m.nT = d->n_triangles; m.xy = d->xy; m.tri = d->tri;
    const size_t nH = 3 * static_cast<size_t>(m.nT);
    m.twin.assign(nH, -1);
    m.ax.resize(nH); m.ay.resize(nH); m.Ex.resize(nH); m.Ey.resize(nH); m.ex.resize(nH); m.ey.resize(nH);
    // bucket half-edges by their lower vertex id (counting sort), then pair inside each bucket
    std::vector<int64_t> head(static_cast<size_t>(m.nV) + 1, 0);
    for (int t = 0; t < m.nT; ++t)
        for (int e = 0; e < 3; ++e) {
            const int v0 = m.tri[3 * t + e], v1 = m.tri[3 * t + (e + 1) % 3];
            if (v0 < 0 || v1 < 0 || v0 >= m.nV || v1 >= m.nV || v0 == v1) return ND_ERR_MESH;
            ++head[static_cast<size_t>(std::min(v0, v1)) + 1];
        }
    for (int v = 0; v < m.nV; ++v) head[v + 1] += head[v];
    std::vector<int32_t> bucket(nH);
    {
        std::vector<int64_t> fill(head.begin(), head.end() - 1);
        for (size_t h = 0; h < nH; ++h) {
            const int t = static_cast<int>(h / 3), e = static_cast<int>(h % 3);
            const int v0 = m.tri[3 * t + e], v1 = m.tri[3 * t + (e + 1) % 3];
            bucket[fill[std::min(v0, v1)]++] = static_cast<int32_t>(h);
        }
    }
    auto hi_vertex = [&](int32_t h) {
        const int t = h / 3, e = h % 3;
        return std::max(m.tri[3 * t + e], m.tri[3 * t + (e + 1) % 3]);
    };
    for (int v = 0; v < m.nV; ++v) {
        const int64_t b0 = head[v], b1 = head[v + 1];
        for (int64_t i = b0; i < b1; ++i) {
            const int32_t h = bucket[i];
            if (m.twin[h] >= 0) continue;
            int matches = 0;
            for (int64_t k = i + 1; k < b1; ++k) {
                const int32_t g = bucket[k];
                if (hi_vertex(g) == hi_vertex(h)) {
                    if (matches++ > 0 || m.twin[g] >= 0) return ND_ERR_MESH; // edge shared by > 2 triangles
                    // opposite orientation required for a conforming CCW mesh
                    if (m.tri[3 * (g / 3) + g % 3] == m.tri[3 * (h / 3) + h % 3]) return ND_ERR_MESH;
                    m.twin[h] = g; m.twin[g] = h;
                }
            }
        }
    }
    for (size_t h = 0; h < nH; ++h) {
        const int t = static_cast<int>(h / 3), e = static_cast<int>(h % 3);
        const int v0 = m.tri[3 * t + e], v1 = m.tri[3 * t + (e + 1) % 3];
        const int a = std::min(v0, v1), b = std::max(v0, v1);
        m.ax[h] = m.xy[2 * a]; m.ay[h] = m.xy[2 * a + 1];
        m.Ex[h] = m.xy[2 * b] - m.xy[2 * a];
        m.Ey[h] = m.xy[2 * b + 1] - m.xy[2 * a + 1];
        m.ex[h] = m.xy[2 * v1] - m.xy[2 * v0];
        m.ey[h] = m.xy[2 * v1 + 1] - m.xy[2 * v0 + 1];
    }
    // boundary half-edges must lie on one of the four sides
    struct BE { double lo; int32_t t; };
    std::vector<BE> be[4];
    for (size_t h = 0; h < nH; ++h) {
        if (m.twin[h] >= 0) continue;
        const int t = static_cast<int>(h / 3), e = static_cast<int>(h % 3);
        const double* p = &m.xy[2 * m.tri[3 * t + e]];
        const double* q = &m.xy[2 * m.tri[3 * t + (e + 1) % 3]];
        int s;
        double c0, c1;
        if (p[0] == 0.0 && q[0] == 0.0)        { s = kLeft;   c0 = p[1]; c1 = q[1]; }
        else if (p[0] == d->W && q[0] == d->W) { s = kRight;  c0 = p[1]; c1 = q[1]; }
        else if (p[1] == 0.0 && q[1] == 0.0)   { s = kBottom; c0 = p[0]; c1 = q[0]; }
        else if (p[1] == d->H && q[1] == d->H) { s = kTop;    c0 = p[0]; c1 = q[0]; }
        else return ND_ERR_MESH;
        be[s].push_back({std::min(c0, c1), static_cast<int32_t>(t)});
    }
    for (int s = 0; s < 4; ++s) {
        if (be[s].empty()) return ND_ERR_MESH;
        std::sort(be[s].begin(), be[s].end(), [](const BE& x, const BE& y) { return x.lo < y.lo; });
        m.side_lo[s].resize(be[s].size());
        m.side_tri[s].resize(be[s].size());
        for (size_t i = 0; i < be[s].size(); ++i) { m.side_lo[s][i] = be[s][i].lo; m.side_tri[s][i] = be[s][i].t; }
    }
    return ND_OK;
}

// Start triangle: the boundary edge on `side` whose interval [lo, next lo) holds c (last one closed).
inline int first_triangle(const HalfEdgeMesh& m, int side, double c)
{
    const std::vector<double>& lo = m.side_lo[side];
    auto it = std::upper_bound(lo.begin(), lo.end(), c); // first lo > c
    size_t idx = (it == lo.begin()) ? 0 : static_cast<size_t>(it - lo.begin()) - 1;
    return m.side_tri[side][idx];
}

// Walk one track.  Emits (triangle, chord) for chords > 0.  Returns the count, or -1 on failure.
template <bool kStore>
int64_t walk(const HalfEdgeMesh& m, int start_side, double x0, double y0, double ux, double uy, int32_t* reg, double* len)
{
    int t = first_triangle(m, start_side, (start_side == kBottom || start_side == kTop) ? x0 : y0);
    double lam_prev = 0.0;
    int64_t count = 0;
    const int64_t guard = 4 * static_cast<int64_t>(m.nT) + 16;
    for (int64_t step = 0; step <= guard; ++step) {
        int exit_e = -1;
        double lam_exit = 0.0;
        for (int e = 0; e < 3; ++e) {
            const size_t h = 3 * static_cast<size_t>(t) + e;
            const double facing = ux * m.ey[h] - uy * m.ex[h];     // u . outward normal of the CCW edge
            if (!(facing > 0.0)) continue;                          // parallel and entry edges never qualify
            const double den = ux * m.Ey[h] - uy * m.Ex[h];
            const double num = (m.ax[h] - x0) * m.Ey[h] - (m.ay[h] - y0) * m.Ex[h];
            const double lam = num / den;
            if (exit_e < 0 || lam < lam_exit) { exit_e = e; lam_exit = lam; }   // ties keep the lower edge
        }
        if (exit_e < 0) return -1;
        const double chord = lam_exit - lam_prev;
        if (chord > 0.0) {
            if (kStore) { reg[count] = t; len[count] = chord; }
            ++count;
        }
        lam_prev = lam_exit;
        const int32_t tw = m.twin[3 * static_cast<size_t>(t) + exit_e];
        if (tw < 0) return count;
        t = tw / 3;
    }
    return -1;
}

} // namespace

namespace {

// Laydown (R-T), links (O-3) and the half-edge mesh; on success *out owns the tracks (no segments yet).
nd_status prepare_impl(const nd_mesh_desc* mesh, int32_t n_azim, double spacing, nd_tracks** out, HalfEdgeMesh& hm,
                       std::vector<EndKey>& kstart)
{
    if (!mesh || !out || !mesh->xy || !mesh->tri) return nd_fail(ND_ERR_NULL, "nd_tracks_generate: NULL argument");
    if (mesh->n_vertices < 3 || mesh->n_triangles < 1 || !(mesh->W > 0.0) || !(mesh->H > 0.0) || !(spacing > 0.0) ||
        n_azim < 4 || n_azim % 4 != 0)
        return nd_fail(ND_ERR_INVALID, "nd_tracks_generate: need V>=3, R>=1, W,H,spacing>0, n_azim a positive multiple of 4");
    for (int s = 0; s < 4; ++s)
        if (mesh->bc[s] != ND_BC_VACUUM && mesh->bc[s] != ND_BC_REFLECTIVE)
            return nd_fail(ND_ERR_INVALID, "nd_tracks_generate: bc must be ND_BC_VACUUM or ND_BC_REFLECTIVE");
    nd_tracks* tr = nullptr;
    try {
        tr = new nd_tracks();
        const double W = mesh->W, H = mesh->H;
        const int nq = n_azim / 4, nh = n_azim / 2;
        tr->n_azim = n_azim; tr->n_half = nh; tr->n_regions = mesh->n_triangles;
        tr->angles.resize(nh);
        // ---- R-T: integer track counts from the desired angle, everything else from dx, dy ----
        for (int a = 0; a < nq; ++a) {
            AngleSet& A = tr->angles[a];
            const double phi_des = (2.0 * kPi / static_cast<double>(n_azim)) * (static_cast<double>(a) + 0.5);
            A.nx = static_cast<int>(std::floor((W / spacing) * std::sin(phi_des))) + 1;
            A.ny = static_cast<int>(std::floor((H / spacing) * std::cos(phi_des))) + 1;
            A.dx = W / static_cast<double>(A.nx);
            A.dy = H / static_cast<double>(A.ny);
            const double h = std::sqrt(A.dx * A.dx + A.dy * A.dy);
            A.ux = A.dx / h;
            A.uy = A.dy / h;
            A.delta = A.dx * A.dy / h;
            A.phi = std::atan2(A.dy, A.dx);
        }
        for (int a = 1; a < nq; ++a)
            if (!(tr->angles[a].phi > tr->angles[a - 1].phi)) {
                delete tr;
                return nd_fail(ND_ERR_INVALID, "nd_tracks_generate: spacing too coarse, effective angles are not increasing");
            }
        for (int a = 0; a < nq; ++a) {
            const double lo = (a == 0) ? 0.0 : 0.5 * (tr->angles[a - 1].phi + tr->angles[a].phi);
            const double hi = (a == nq - 1) ? 0.5 * kPi : 0.5 * (tr->angles[a].phi + tr->angles[a + 1].phi);
            tr->angles[a].omega = (hi - lo) / (2.0 * kPi);
        }
        for (int j = nq; j < nh; ++j) {
            tr->angles[j] = tr->angles[nh - 1 - j];
            tr->angles[j].ux = -tr->angles[j].ux;
            tr->angles[j].mirrored = true;
        }
        int T = 0;
        for (int j = 0; j < nh; ++j) { tr->angles[j].first = T; T += tr->angles[j].nx + tr->angles[j].ny; }
        tr->n_tracks = T;
        tr->track_weight.resize(T); tr->track_azim.resize(T); tr->ends.resize(4 * static_cast<size_t>(T));
        tr->link.assign(2 * static_cast<size_t>(T), -1);
        kstart.assign(T, EndKey{0, 0});
        std::vector<EndKey> kend(T);
        for (int j = 0; j < nh; ++j) {
            const AngleSet& A = tr->angles[j];
            for (int i = 0; i < A.nx + A.ny; ++i) {
                const int t = A.first + i;
                track_keys(A, i, kstart[t], kend[t]);
                key_point(kstart[t], A, W, H, &tr->ends[4 * static_cast<size_t>(t)]);
                key_point(kend[t], A, W, H, &tr->ends[4 * static_cast<size_t>(t) + 2]);
                tr->track_azim[t] = j;
                tr->track_weight[t] = A.omega * A.delta;
            }
        }
        // ---- O-3: an outgoing end with key K on a reflective side enters the complement-angle track with key K ----
        for (int j = 0; j < nh; ++j) {
            const AngleSet& A = tr->angles[j];
            const AngleSet& C = tr->angles[nh - 1 - j];
            const int n = A.nx + A.ny, span = std::max(A.nx, A.ny);
            std::vector<int32_t> enter(4 * static_cast<size_t>(span), -1); // (side,slot) -> 2*t'+d'
            for (int i = 0; i < n; ++i) {
                const int t = C.first + i;
                // a key that is some complement track's start wins over one that is an end (they never coincide)
                int32_t& se = enter[static_cast<size_t>(kend[t].side) * span + kend[t].slot];
                if (se < 0) se = 2 * t + 1;
                enter[static_cast<size_t>(kstart[t].side) * span + kstart[t].slot] = 2 * t + 0;
            }
            for (int i = 0; i < n; ++i) {
                const int t = A.first + i;
                const EndKey out_key[2] = {kend[t], kstart[t]};
                for (int d = 0; d < 2; ++d) {
                    if (mesh->bc[out_key[d].side] == ND_BC_VACUUM) continue;
                    const int32_t v = enter[static_cast<size_t>(out_key[d].side) * span + out_key[d].slot];
                    if (v < 0) { delete tr; return nd_fail(ND_ERR_INVALID, "nd_tracks_generate: unmatched cyclic track end"); }
                    tr->link[2 * static_cast<size_t>(t) + d] = v;
                }
            }
        }
        nd_status rc = build_mesh(hm, mesh);
        if (rc != ND_OK) { delete tr; return nd_fail(rc, "nd_tracks_generate: mesh is not a conforming CCW triangulation of [0,W]x[0,H]"); }
    } catch (const std::bad_alloc&) {
        delete tr;
        return nd_fail(ND_ERR_NOMEM, "nd_tracks_generate: out of host memory");
    }
    *out = tr;
    return ND_OK;
}

} // namespace

nd_status nd_tracks_prepare(const nd_mesh_desc* mesh, int32_t n_azim, double spacing, nd_tracks** out, NdWalkInput* walk_in)
{
    if (!walk_in) return nd_fail(ND_ERR_NULL, "nd_tracks_prepare: NULL argument");
    HalfEdgeMesh hm;
    std::vector<EndKey> kstart;
    nd_tracks* tr = nullptr;
    nd_status rc = prepare_impl(mesh, n_azim, spacing, &tr, hm, kstart);
    if (rc != ND_OK) return rc;
    try {
        walk_in->twin = hm.twin;
        walk_in->start_tri.resize(static_cast<size_t>(tr->n_tracks));
        for (int t = 0; t < tr->n_tracks; ++t) {
            const double x0 = tr->ends[4 * static_cast<size_t>(t)], y0 = tr->ends[4 * static_cast<size_t>(t) + 1];
            const int side = kstart[t].side;
            walk_in->start_tri[t] = first_triangle(hm, side, (side == kBottom || side == kTop) ? x0 : y0);
        }
    } catch (const std::bad_alloc&) {
        delete tr;
        return nd_fail(ND_ERR_NOMEM, "nd_tracks_prepare: out of host memory");
    }
    *out = tr;
    return ND_OK;
}

nd_status nd_tracks_finish(nd_tracks* tr, bool volumes_from_segments)
{
    if (!tr) return nd_fail(ND_ERR_NULL, "nd_tracks_finish: NULL argument");
    try {
        const int T = tr->n_tracks, nh = tr->n_half;
        // ---- O-5: track-estimated areas, summed in canonical (track, segment) order ----
        if (volumes_from_segments) tr->volume.assign(static_cast<size_t>(tr->n_regions), 0.0);
        for (int t = 0; t < T && volumes_from_segments; ++t) {
            const double w2 = 2.0 * tr->track_weight[t];
            for (int64_t k = tr->seg_offset[t]; k < tr->seg_offset[static_cast<size_t>(t) + 1]; ++k)
                tr->volume[tr->seg_region[k]] += w2 * tr->seg_length[k];
        }
        tr->global_id.resize(static_cast<size_t>(T));
        for (int t = 0; t < T; ++t) tr->global_id[t] = t;
        tr->azim_phi.resize(nh); tr->azim_weight.resize(nh); tr->azim_spacing.resize(nh);
        for (int j = 0; j < nh; ++j) {
            tr->azim_phi[j] = tr->angles[j].mirrored ? kPi - tr->angles[j].phi : tr->angles[j].phi;
            tr->azim_weight[j] = tr->angles[j].omega;
            tr->azim_spacing[j] = tr->angles[j].delta;
        }
    } catch (const std::bad_alloc&) {
        return nd_fail(ND_ERR_NOMEM, "nd_tracks_finish: out of host memory");
    }
    return ND_OK;
}

extern "C" nd_status nd_tracks_generate(const nd_mesh_desc* mesh, int32_t n_azim, double spacing, int32_t n_threads,
                                        nd_tracks** out)
{
    if (!out) return nd_fail(ND_ERR_NULL, "nd_tracks_generate: NULL argument");
    HalfEdgeMesh hm;
    std::vector<EndKey> kstart;
    nd_tracks* tr = nullptr;
    nd_status rc = prepare_impl(mesh, n_azim, spacing, &tr, hm, kstart);
    if (rc != ND_OK) return rc;
    try {
        const int T = tr->n_tracks;
        // ---- R-W: walk every track through the half-edge mesh (count pass, then fill pass) ----
#ifdef _OPENMP
        const int nth = n_threads > 0 ? n_threads : omp_get_max_threads();
#else
        const int nth = 1;
        (void)n_threads;
#endif
        tr->seg_offset.assign(static_cast<size_t>(T) + 1, 0);
        int failed = 0;
#pragma omp parallel for schedule(dynamic, 64) num_threads(nth) reduction(+ : failed)
        for (int t = 0; t < T; ++t) {
            const AngleSet& A = tr->angles[tr->track_azim[t]];
            const int64_t n = walk<false>(hm, kstart[t].side, tr->ends[4 * static_cast<size_t>(t)],
                                          tr->ends[4 * static_cast<size_t>(t) + 1], A.ux, A.uy, nullptr, nullptr);
            if (n < 0) ++failed; else tr->seg_offset[static_cast<size_t>(t) + 1] = n;
        }
        if (failed) { delete tr; return nd_fail(ND_ERR_MESH, "nd_tracks_generate: ray walk left the mesh"); }
        for (int t = 0; t < T; ++t) tr->seg_offset[static_cast<size_t>(t) + 1] += tr->seg_offset[t];
        tr->n_segments = tr->seg_offset[T];
        tr->seg_region.resize(static_cast<size_t>(tr->n_segments));
        tr->seg_length.resize(static_cast<size_t>(tr->n_segments));
#pragma omp parallel for schedule(dynamic, 64) num_threads(nth)
        for (int t = 0; t < T; ++t) {
            const AngleSet& A = tr->angles[tr->track_azim[t]];
            const int64_t o = tr->seg_offset[t];
            walk<true>(hm, kstart[t].side, tr->ends[4 * static_cast<size_t>(t)], tr->ends[4 * static_cast<size_t>(t) + 1],
                       A.ux, A.uy, tr->seg_region.data() + o, tr->seg_length.data() + o);
        }
    } catch (const std::bad_alloc&) {
        delete tr;
        return nd_fail(ND_ERR_NOMEM, "nd_tracks_generate: out of host memory");
    }
    rc = nd_tracks_finish(tr);
    if (rc != ND_OK) { delete tr; return rc; }
    *out = tr;
    return ND_OK;
}

extern "C" nd_status nd_tracks_view(const nd_tracks* tr, nd_tracks_view_t* v)
{
    if (!tr || !v) return nd_fail(ND_ERR_NULL, "nd_tracks_view: NULL argument");
    v->n_tracks = tr->n_tracks; v->n_regions = tr->n_regions; v->n_segments = tr->n_segments; v->n_half = tr->n_half;
    v->track_seg_offset = tr->seg_offset.data();
    v->seg_region = tr->host_segments ? tr->seg_region.data() : nullptr;
    v->seg_length = tr->host_segments ? tr->seg_length.data() : nullptr;
    v->seg_region_device = tr->d_seg_region;
    v->seg_length_device = tr->d_seg_length;
    v->track_weight = tr->track_weight.data();
    v->link = tr->link.data();
    v->track_azim = tr->track_azim.data();
    v->track_ends = tr->ends.data();
    v->track_volume = tr->volume.data();
    v->azim_phi = tr->azim_phi.data();
    v->azim_weight = tr->azim_weight.data();
    v->azim_spacing = tr->azim_spacing.data();
    v->track_global = tr->global_id.data();
    return ND_OK;
}

// NEXT-2: the tracks of one shard of an angle-pair partition.  A reflective link joins a track of angle j
// to one of its complement N_a/2-1-j (O-3), so a shard that owns whole pairs {j, N_a/2-1-j} never exchanges boundary flux.
extern "C" nd_status nd_tracks_shard(const nd_tracks* full, int32_t n_shards, int32_t shard, nd_tracks** out)
{
    if (!full || !out) return nd_fail(ND_ERR_NULL, "nd_tracks_shard: NULL argument");
    const int nh = full->n_half, np = nh / 2, T = full->n_tracks;
    if (n_shards < 1 || shard < 0 || shard >= n_shards) return nd_fail(ND_ERR_INVALID, "nd_tracks_shard: need 0 <= shard < n_shards");
    if (nh < 2 || nh % 2 != 0 || (int)full->angles.size() != nh) return nd_fail(ND_ERR_STATE, "nd_tracks_shard: not a cyclic laydown");
    if (n_shards > np) return nd_fail(ND_ERR_INVALID, "nd_tracks_shard: more shards than angle pairs (N_a / 4)");
    if ((int)full->global_id.size() != T) return nd_fail(ND_ERR_STATE, "nd_tracks_shard: incomplete tracks object");
    if (!full->host_segments) return nd_fail(ND_ERR_STATE, "nd_tracks_shard: device-resident tracks, call nd_tracks_materialise first");
    for (int t = 0; t < T; ++t)
        if (full->global_id[t] != t) return nd_fail(ND_ERR_STATE, "nd_tracks_shard: the input is already a shard");
    nd_tracks* tr = nullptr;
    try {
        // ---- segments per angle pair, pairs dealt to the shards longest first (deterministic) ----
        std::vector<int64_t> seg_of_angle(static_cast<size_t>(nh), 0);
        for (int t = 0; t < T; ++t) seg_of_angle[full->track_azim[t]] += full->seg_offset[static_cast<size_t>(t) + 1] - full->seg_offset[t];
        std::vector<int> order(static_cast<size_t>(np));
        std::vector<int64_t> w(static_cast<size_t>(np));
        for (int j = 0; j < np; ++j) { order[j] = j; w[j] = seg_of_angle[j] + seg_of_angle[nh - 1 - j]; }
        std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return w[a] > w[b]; });
        std::vector<int64_t> load(static_cast<size_t>(n_shards), 0);
        std::vector<int> owner(static_cast<size_t>(nh), -1);
        for (int i = 0; i < np; ++i) {
            int best = 0;
            for (int s = 1; s < n_shards; ++s)
                if (load[s] < load[best]) best = s;
            load[best] += w[order[i]];
            owner[order[i]] = owner[nh - 1 - order[i]] = best;
        }
        // ---- copy the shard's tracks in canonical order ----
        tr = new nd_tracks();
        tr->n_azim = full->n_azim; tr->n_half = nh; tr->n_regions = full->n_regions;
        tr->angles = full->angles;
        tr->azim_phi = full->azim_phi; tr->azim_weight = full->azim_weight; tr->azim_spacing = full->azim_spacing;
        tr->volume = full->volume;                       // the areas A~_r of the WHOLE laydown: every shard divides by them
        std::vector<int32_t> local(static_cast<size_t>(T), -1);
        int n = 0;
        int64_t S = 0;
        for (int t = 0; t < T; ++t)
            if (owner[full->track_azim[t]] == shard) {
                local[t] = n++;
                S += full->seg_offset[static_cast<size_t>(t) + 1] - full->seg_offset[t];
            }
        tr->n_tracks = n; tr->n_segments = S;
        tr->seg_offset.assign(static_cast<size_t>(n) + 1, 0);
        tr->seg_region.resize(static_cast<size_t>(S));
        tr->seg_length.resize(static_cast<size_t>(S));
        tr->track_weight.resize(static_cast<size_t>(n)); tr->track_azim.resize(static_cast<size_t>(n));
        tr->link.resize(2 * static_cast<size_t>(n)); tr->ends.resize(4 * static_cast<size_t>(n));
        tr->global_id.resize(static_cast<size_t>(n));
        int64_t o = 0;
        for (int t = 0; t < T; ++t) {
            const int lt = local[t];
            if (lt < 0) continue;
            const int64_t k0 = full->seg_offset[t], k1 = full->seg_offset[static_cast<size_t>(t) + 1];
            tr->seg_offset[lt] = o;
            for (int64_t k = k0; k < k1; ++k, ++o) { tr->seg_region[o] = full->seg_region[k]; tr->seg_length[o] = full->seg_length[k]; }
            tr->track_weight[lt] = full->track_weight[t];
            tr->track_azim[lt] = full->track_azim[t];
            tr->global_id[lt] = t;
            for (int c = 0; c < 4; ++c) tr->ends[4 * static_cast<size_t>(lt) + c] = full->ends[4 * static_cast<size_t>(t) + c];
            for (int d = 0; d < 2; ++d) {
                const int32_t lk = full->link[2 * static_cast<size_t>(t) + d];
                if (lk < 0) { tr->link[2 * static_cast<size_t>(lt) + d] = -1; continue; }
                const int32_t l2 = local[lk >> 1];
                if (l2 < 0) { delete tr; return nd_fail(ND_ERR_STATE, "nd_tracks_shard: a link leaves its angle pair"); }
                tr->link[2 * static_cast<size_t>(lt) + d] = 2 * l2 + (lk & 1);
            }
        }
        tr->seg_offset[n] = o;
    } catch (const std::bad_alloc&) {
        delete tr;
        return nd_fail(ND_ERR_NOMEM, "nd_tracks_shard: out of host memory");
    }
    *out = tr;
    return ND_OK;
}

extern "C" nd_status nd_tracks_destroy(nd_tracks* tr)
{
    delete tr;
    return ND_OK;
}

void nd_touch_pages(void* p, size_t bytes)
{
    volatile unsigned char* b = static_cast<volatile unsigned char*>(p);
    const int64_t n_pages = (int64_t)((bytes + 4095) / 4096);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n_pages; ++i) b[(size_t)i * 4096] = 0;
}
