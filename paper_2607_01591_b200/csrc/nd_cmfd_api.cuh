// nd_cmfd_api.cuh -- NEXT-3: the CMFD plan (include/nd.h "nd_cmfd_*"), included by nd_api.cu behind the problem's internals.
// Algorithm 1 of the paper ("Perform MOC on the fine mesh", "Solve CMFD on the coarse mesh", update of the
// fine-mesh flux) with the reading C-1..C-9 of DESIGN.md 8d.  A plan binds a coarse mesh to one problem: its cell map, surface
// list, crossing lists and every coarse array live in ONE caller-owned device workspace, the currents of C-3 are tallied by
// the sweep kernel itself, and an accelerated iteration launches kernels only -- no allocation, no host arithmetic, no stream
// synchronisation between its steps.

struct nd_cmfd {
    nd_problem* p = nullptr;
    int C = 0, S = 0;                       // coarse cells, interior surfaces
    nd_cmfd_options opt{};
    // device arrays (all inside the caller's workspace)
    int32_t* cell = nullptr;                // [R]
    int32_t* entry_cell = nullptr;          // [2T] coarse cell in which chain (t, d) begins, -1 = empty track
    int32_t* link_fwd = nullptr;            // [2T]
    int32_t* lo = nullptr; int32_t* hi = nullptr;               // [S]
    int64_t* pair_key = nullptr; int32_t* pair_idx = nullptr;   // [S] sorted keys lo * C + hi and the caller's index
    int32_t* adj_off = nullptr; int32_t* adj_ent = nullptr;     // [C+1], [2S]
    double* coupling = nullptr;             // [S]
    double* J = nullptr;                    // J_surf [S][G] | J_vac [C][G] | J_ref [C][G]
    double* Psi = nullptr; double* V = nullptr;                 // [C][M][G], [C]
    double* co = nullptr;                   // Phi | sigt | nusf | chi [C][G] each, then sigs [C][G][G]
    double* out_lo = nullptr; double* in_hi = nullptr;          // [S][G]
    double* Mw = nullptr; double* Minv = nullptr;               // [C][G][G]
    double* x = nullptr; double* y = nullptr; double* y2 = nullptr; double* f = nullptr; double* ratio = nullptr;   // [C][G]
    double* state = nullptr;                // [ST_COUNT] of the coarse solve, then k0 at [ST_COUNT]
    double* stats = nullptr;                // [kCmfdMaxStats][4]: k after the sweep, coarse k, coarse iterations, solve ok
    double* Qtmp = nullptr;                 // [R][G] (nd_cmfd_sweep keeps no caller array)
    int* flags = nullptr;                   // [0] a hand-over joined two cells that are not a listed surface
    uint8_t* xblob = nullptr; uint32_t* xoff = nullptr;         // crossing lists of every tile
    int64_t n_crossings = 0;
    int coop_grid = 1;
    int J_replicas = 1;                     // copies of J the sweep's blocks spread their atomics over; summed into copy 0
    int64_t J_stride = 0;                   // doubles per copy
};

namespace {

constexpr int kCmfdMaxStats = 1024;

struct CmfdLayout {
    size_t cell, entry_cell, link_fwd, lo, hi, pair_key, pair_idx, adj_off, adj_ent, coupling, J, Psi, V, co, out_lo, in_hi, Mw, Minv, x, y,
        y2, f, ratio, state, stats, Qtmp, flags, xoff, xblob, total;
};

// copies of the current arrays: 64, fewer when a copy is large (then the atomics are spread over many lines anyway)
inline int64_t cmfd_J_stride(const Dims& d, int C, int S) { return ((int64_t)S * d.G + 2 * (int64_t)C * d.G + 31) / 32 * 32; }
inline int cmfd_J_replicas(const Dims& d, int C, int S)
{
    const int64_t bytes = 8 * cmfd_J_stride(d, C, S);
    return (int)std::max<int64_t>(1, std::min<int64_t>(64, ((int64_t)64 << 20) / std::max<int64_t>(bytes, 1)));
}

CmfdLayout cmfd_layout(const Dims& d, int C, int S, int64_t n_tiles, size_t xblob_bytes)
{
    CmfdLayout L{};
    size_t c = 0;
    const size_t CG = (size_t)C * d.G, SG = (size_t)S * d.G;
    L.cell = bump(c, sizeof(int32_t) * (size_t)d.R);
    L.entry_cell = bump(c, sizeof(int32_t) * 2 * (size_t)d.T);
    L.link_fwd = bump(c, sizeof(int32_t) * 2 * (size_t)d.T);
    L.lo = bump(c, sizeof(int32_t) * ((size_t)S + 1));
    L.hi = bump(c, sizeof(int32_t) * ((size_t)S + 1));
    L.pair_key = bump(c, sizeof(int64_t) * ((size_t)S + 1));
    L.pair_idx = bump(c, sizeof(int32_t) * ((size_t)S + 1));
    L.adj_off = bump(c, sizeof(int32_t) * ((size_t)C + 1));
    L.adj_ent = bump(c, sizeof(int32_t) * (2 * (size_t)S + 1));
    L.coupling = bump(c, sizeof(double) * ((size_t)S + 1));
    L.J = bump(c, sizeof(double) * (size_t)cmfd_J_stride(d, C, S) * cmfd_J_replicas(d, C, S));
    L.Psi = bump(c, sizeof(double) * CG * d.M);
    L.V = bump(c, sizeof(double) * (size_t)C);
    L.co = bump(c, sizeof(double) * (4 * CG + CG * d.G));
    L.out_lo = bump(c, sizeof(double) * (SG + 1));
    L.in_hi = bump(c, sizeof(double) * (SG + 1));
    L.Mw = bump(c, sizeof(double) * CG * d.G);
    L.Minv = bump(c, sizeof(double) * CG * d.G);
    L.x = bump(c, sizeof(double) * CG);
    L.y = bump(c, sizeof(double) * CG);
    L.y2 = bump(c, sizeof(double) * CG);
    L.f = bump(c, sizeof(double) * CG);
    L.ratio = bump(c, sizeof(double) * CG);
    L.state = bump(c, sizeof(double) * (ndk::ST_COUNT + 8));
    L.stats = bump(c, sizeof(double) * 4 * kCmfdMaxStats);
    L.Qtmp = bump(c, sizeof(double) * (size_t)d.R * d.G);
    L.flags = bump(c, 256);
    L.xoff = bump(c, sizeof(uint32_t) * ((size_t)n_tiles + 1));
    L.xblob = bump(c, xblob_bytes + 16);
    L.total = c;
    return L;
}

// Host: the crossing list of every tile (C-3).  A crossing = two consecutive segments of a track in different coarse cells;
// it belongs to the tile that holds the first of the two (in forward order).  Entry: { surface << 1 | sign bit (1: the forward
// direction runs from the higher to the lower cell id), slot | position inside the slot's run << 16 }.
// count_only: only sizes are computed (nd_cmfd_workspace_bytes).
nd_status cmfd_build_crossings(const nd_problem* p, const nd_problem_desc* desc, int C, const int32_t* cell, int S,
                               const std::vector<int64_t>& key_sorted, const std::vector<int32_t>& idx_sorted, bool count_only,
                               std::vector<uint32_t>* xoff, std::vector<uint8_t>* xblob, int64_t* n_crossings, uint64_t* blob16)
{
    const int NT = p->sc.sp.NT;
    const int64_t n_sw = (int64_t)p->h_swath_tile0.size() - 1, n_tiles = p->n_tiles;
    const int64_t* off = desc->track_seg_offset;
    std::vector<uint32_t> cnt((size_t)n_tiles + 1, 0);      // crossings per tile
    int missing = 0;
    for (int pass = 0; pass < (count_only ? 1 : 2); ++pass) {
        if (pass == 1) {
            // offsets in 16-byte units: 8-byte header + 8 bytes per crossing, rounded up
            xoff->assign((size_t)n_tiles + 1, 0);
            uint64_t o = 0;
            for (int64_t ti = 0; ti < n_tiles; ++ti) {
                (*xoff)[(size_t)ti] = (uint32_t)o;
                o += (8 * (1 + (uint64_t)cnt[(size_t)ti]) + 15) / 16;
                if (o >= 0xffffffffull) return nd_fail(ND_ERR_RANGE, "nd_cmfd_create: crossing lists exceed 64 GiB");
            }
            (*xoff)[(size_t)n_tiles] = (uint32_t)o;
            xblob->assign((size_t)o * 16, 0);
        }
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : missing)
        for (int64_t sw = 0; sw < n_sw; ++sw) {
            const int32_t* trk = &p->h_swath_track[(size_t)sw * NT];
            std::vector<int64_t> cur((size_t)NT, 0);
            for (int b = 0; b < NT; ++b) cur[b] = trk[b] >= 0 ? off[trk[b]] : 0;
            for (int64_t ti = p->h_swath_tile0[(size_t)sw]; ti < p->h_swath_tile0[(size_t)sw + 1]; ++ti) {
                const uint16_t* ss = &p->h_slot_start[(size_t)ti * (NT + 1)];
                uint32_t n = 0;
                uint32_t* out = pass == 1 ? reinterpret_cast<uint32_t*>(xblob->data() + (size_t)(*xoff)[(size_t)ti] * 16) : nullptr;
                for (int b = 0; b < NT; ++b) {
                    const int c_b = ss[b + 1] - ss[b];
                    if (trk[b] < 0 || c_b == 0) continue;
                    const int64_t k_end = off[trk[b] + 1];
                    for (int j = 0; j < c_b; ++j) {
                        const int64_t k = cur[b] + j;
                        if (k + 1 >= k_end) break;
                        const int32_t a = cell[desc->seg_region[k]], bb = cell[desc->seg_region[k + 1]];
                        if (a == bb) continue;
                        if (pass == 1) {
                            const int64_t key = (int64_t)std::min(a, bb) * C + std::max(a, bb);
                            const auto it = std::lower_bound(key_sorted.begin(), key_sorted.end(), key);
                            if (it == key_sorted.end() || *it != key) { ++missing; continue; }
                            const uint32_t s = (uint32_t)idx_sorted[(size_t)(it - key_sorted.begin())];
                            out[2 * (1 + n)] = (s << 1) | (a > bb ? 1u : 0u);
                            out[2 * (1 + n) + 1] = (uint32_t)b | ((uint32_t)j << 16);
                        }
                        ++n;
                    }
                    cur[b] += c_b;
                }
                if (pass == 0) cnt[(size_t)ti] = n;
                else out[0] = n;
            }
        }
        if (missing) return nd_fail(ND_ERR_INVALID, "nd_cmfd_create: a track crosses between two coarse cells that are not a listed surface");
    }
    int64_t total = 0;
    uint64_t o16 = 0;
    for (int64_t ti = 0; ti < n_tiles; ++ti) {
        total += cnt[(size_t)ti];
        o16 += (8 * (1 + (uint64_t)cnt[(size_t)ti]) + 15) / 16;
    }
    *n_crossings = total;
    *blob16 = o16;
    (void)S;
    return ND_OK;
}

nd_status cmfd_check_inputs(const nd_problem* p, const nd_problem_desc* desc, int32_t n_cells, const int32_t* cell, int32_t n_pairs,
                            const int32_t* pair_lo, const int32_t* pair_hi, const char* who)
{
    auto fail = [who](nd_status s, const char* m) { return nd_fail(s, (std::string(who) + ": " + m).c_str()); };
    if (!p || !desc || !cell) return fail(ND_ERR_NULL, "NULL argument");
    if (n_pairs > 0 && (!pair_lo || !pair_hi)) return fail(ND_ERR_NULL, "pair_lo / pair_hi are NULL");
    if (n_cells < 1 || n_pairs < 0) return fail(ND_ERR_INVALID, "n_cells must be >= 1 and n_pairs >= 0");
    if (p->sweep_kernel != ND_SWEEP_SWATH || p->h_slot_start.empty())
        return fail(ND_ERR_STATE, "needs a problem created with the swath sweep kernel and nd_options.cmfd_stream = 1 "
                                  "(the sweep kernel tallies the currents; its shared memory is laid out for that at creation)");
    if (p->opt.exp_mode != ND_EXP_FAST) return fail(ND_ERR_STATE, "the current tally is built for exp_mode = ND_EXP_FAST");
    const Dims& d = p->d;
    if (!desc->track_seg_offset || !desc->seg_region) return fail(ND_ERR_NULL, "a descriptor array is NULL");
    if (desc->n_tracks != d.T || desc->n_regions != d.R || desc->track_seg_offset[d.T] != d.S)
        return fail(ND_ERR_INVALID, "the descriptor is not the one the problem was created from");
    for (int64_t r = 0; r < d.R; ++r)
        if (cell[r] < 0 || cell[r] >= n_cells) return fail(ND_ERR_RANGE, "cell[r] out of [0, n_cells)");
    for (int32_t s = 0; s < n_pairs; ++s)
        if (pair_lo[s] < 0 || pair_hi[s] >= n_cells || pair_lo[s] >= pair_hi[s]) return fail(ND_ERR_RANGE, "a surface needs 0 <= lo < hi < n_cells");
    return ND_OK;
}

nd_status cmfd_sorted_keys(int32_t n_cells, int32_t n_pairs, const int32_t* pair_lo, const int32_t* pair_hi,
                           std::vector<int64_t>* key, std::vector<int32_t>* idx)
{
    std::vector<std::pair<int64_t, int32_t>> keyed;
    keyed.reserve((size_t)n_pairs);
    for (int32_t s = 0; s < n_pairs; ++s) keyed.emplace_back((int64_t)pair_lo[s] * n_cells + pair_hi[s], s);
    std::sort(keyed.begin(), keyed.end());
    key->resize((size_t)n_pairs);
    idx->resize((size_t)n_pairs);
    for (int32_t s = 0; s < n_pairs; ++s) {
        if (s > 0 && keyed[s].first == keyed[s - 1].first) return nd_fail(ND_ERR_INVALID, "nd_cmfd: a surface is listed twice");
        (*key)[s] = keyed[s].first;
        (*idx)[s] = keyed[s].second;
    }
    return ND_OK;
}

void cmfd_fill_sweep_params(const nd_cmfd* c, ndk::SwathParams* prm)
{
    prm->xblob = c->xblob;
    prm->xoff = c->xoff;
    prm->J_surf = c->J;
    prm->J_stride = c->J_stride;
    prm->J_replicas = c->J_replicas;
}

nd_status cmfd_end_currents(nd_cmfd* c, const double* scale_div, cudaStream_t st)
{
    nd_problem* p = c->p;
    const Dims& d = p->d;
    ndk::EndCurrentParams ep{};
    ep.psi_in = p->psi_in; ep.psi_out = p->psi_out; ep.trk_w = p->trk_w; ep.link_fwd = c->link_fwd; ep.entry_cell = c->entry_cell;
    ep.pair_key = c->pair_key; ep.pair_idx = c->pair_idx; ep.scale_div = scale_div;
    ep.J_surf = c->J; ep.J_vac = c->J + (size_t)c->S * d.G; ep.J_ref = ep.J_vac + (size_t)c->C * d.G; ep.missing = c->flags;
    ep.J_stride = c->J_stride; ep.J_replicas = c->J_replicas;
    ep.n_entries = 2 * (int64_t)d.T; ep.P = d.P; ep.G = d.G; ep.Gs = d.Gs; ep.n_pairs = c->S; ep.n_cells = c->C;
    for (int i = 0; i < ndk::kMaxPolar; ++i) ep.wp[i] = p->wp[i];
    ndk::k_end_currents<<<grid_for(ep.n_entries * d.G, 256, 8 * p->n_sm), 256, 0, st>>>(ep);
    ND_LAUNCH_CHECK(p);
    if (c->J_replicas > 1) {
        const int64_t n = (int64_t)c->S * d.G + 2 * (int64_t)c->C * d.G;
        ndk::k_cmfd_reduce_replicas<<<grid_for(n, 256, 4 * p->n_sm), 256, 0, st>>>(c->J, c->J_stride, c->J_replicas, n);
        ND_LAUNCH_CHECK(p);
    }
    return ND_OK;
}

} // namespace

extern "C" nd_status nd_cmfd_workspace_bytes(const nd_problem* p, const nd_problem_desc* desc, int32_t n_cells,
                                             const int32_t* cell, int32_t n_pairs, size_t* device_bytes)
{
    if (!device_bytes) return nd_fail(ND_ERR_NULL, "nd_cmfd_workspace_bytes: device_bytes is NULL");
    nd_status rc = cmfd_check_inputs(p, desc, n_cells, cell, 0, nullptr, nullptr, "nd_cmfd_workspace_bytes");
    if (rc != ND_OK) return rc;
    if (n_pairs < 0) return nd_fail(ND_ERR_INVALID, "nd_cmfd_workspace_bytes: n_pairs must be >= 0");
    try {
        std::vector<uint32_t> xoff;
        std::vector<uint8_t> xblob;
        int64_t nx = 0;
        uint64_t blob16 = 0;
        rc = cmfd_build_crossings(p, desc, n_cells, cell, n_pairs, {}, {}, true, &xoff, &xblob, &nx, &blob16);
        if (rc != ND_OK) return rc;
        *device_bytes = cmfd_layout(p->d, n_cells, n_pairs, p->n_tiles, (size_t)blob16 * 16).total;
    } catch (const std::bad_alloc&) {
        return nd_fail(ND_ERR_NOMEM, "nd_cmfd_workspace_bytes: out of host memory");
    }
    return ND_OK;
}

extern "C" nd_status nd_cmfd_create(nd_problem* p, const nd_problem_desc* desc, int32_t n_cells, const int32_t* cell,
                                    int32_t n_pairs, const int32_t* pair_lo, const int32_t* pair_hi, const double* coupling,
                                    const nd_cmfd_options* opts, void* device_workspace, size_t device_bytes, void* cuda_stream,
                                    nd_cmfd** out)
{
    if (!out || !device_workspace) return nd_fail(ND_ERR_NULL, "nd_cmfd_create: NULL argument");
    nd_status rc = cmfd_check_inputs(p, desc, n_cells, cell, n_pairs, pair_lo, pair_hi, "nd_cmfd_create");
    if (rc != ND_OK) return rc;
    if (n_pairs > 0 && !coupling) return nd_fail(ND_ERR_NULL, "nd_cmfd_create: coupling is NULL");
    if (!desc->link) return nd_fail(ND_ERR_NULL, "nd_cmfd_create: desc->link is NULL");
    nd_cmfd_options opt{};
    if (opts) opt = *opts;
    if (!(opt.tol > 0.0)) opt.tol = 1e-12;
    if (opt.max_outer <= 0) opt.max_outer = 20000;
    if (opt.inner_sweeps <= 0) opt.inner_sweeps = 4;
    if (!(opt.relax > 0.0)) opt.relax = 1.0;
    if (opt.relax > 1.0) return nd_fail(ND_ERR_INVALID, "nd_cmfd_create: relax must lie in (0, 1]");
    if (!(opt.rel_tol >= 0.0) || opt.rel_tol >= 1.0) return nd_fail(ND_ERR_INVALID, "nd_cmfd_create: rel_tol must lie in [0, 1)");
    for (int i = 0; i < 2; ++i)
        if (opt.reserved[i] != 0) return nd_fail(ND_ERR_INVALID, "nd_cmfd_options.reserved must be zero");
    for (int32_t s = 0; s < n_pairs; ++s)
        if (!(coupling[s] >= 0.0) || !std::isfinite(coupling[s])) return nd_fail(ND_ERR_INVALID, "nd_cmfd_create: coupling must be finite and >= 0");
    if (reinterpret_cast<uintptr_t>(device_workspace) % kAlign != 0) return nd_fail(ND_ERR_WORKSPACE, "nd_cmfd_create: workspace must be 256-byte aligned");
    const Dims& d = p->d;
    cudaStream_t st = as_stream(cuda_stream);
    nd_cmfd* c = nullptr;
    try {
        std::vector<int64_t> key;
        std::vector<int32_t> idx;
        rc = cmfd_sorted_keys(n_cells, n_pairs, pair_lo, pair_hi, &key, &idx);
        if (rc != ND_OK) return rc;
        std::vector<uint32_t> xoff;
        std::vector<uint8_t> xblob;
        int64_t nx = 0;
        uint64_t blob16 = 0;
        rc = cmfd_build_crossings(p, desc, n_cells, cell, n_pairs, key, idx, false, &xoff, &xblob, &nx, &blob16);
        if (rc != ND_OK) return rc;
        const CmfdLayout L = cmfd_layout(d, n_cells, n_pairs, p->n_tiles, xblob.size());
        if (device_bytes < L.total) return nd_fail(ND_ERR_WORKSPACE, "nd_cmfd_create: workspace smaller than nd_cmfd_workspace_bytes");
        // entry cells and the hand-over surfaces (C-2 (b)): every linked pair of chains must join a listed surface or one cell
        std::vector<int32_t> h_entry(2 * (size_t)d.T);
        for (size_t e = 0; e < h_entry.size(); ++e) h_entry[e] = p->h_entry_region[e] >= 0 ? cell[p->h_entry_region[e]] : -1;
        for (int64_t e = 0; e < 2 * (int64_t)d.T; ++e) {
            const int32_t lk = desc->link[e];
            if (lk < 0) continue;
            if (lk >= 2 * d.T) return nd_fail(ND_ERR_RANGE, "nd_cmfd_create: link out of range");
            const int32_t a = h_entry[(size_t)(e ^ 1)], b = h_entry[(size_t)lk];
            if (a < 0 || b < 0 || a == b) continue;
            const int64_t k = (int64_t)std::min(a, b) * n_cells + std::max(a, b);
            if (!std::binary_search(key.begin(), key.end(), k))
                return nd_fail(ND_ERR_INVALID, "nd_cmfd_create: a reflective hand-over joins two coarse cells that are not a listed surface");
        }
        // adjacency of the coarse cells (deterministic gather in the coarse solve)
        std::vector<int32_t> adj_off((size_t)n_cells + 1, 0), adj_ent(2 * (size_t)n_pairs + 1, 0);
        for (int32_t s = 0; s < n_pairs; ++s) { ++adj_off[(size_t)pair_lo[s] + 1]; ++adj_off[(size_t)pair_hi[s] + 1]; }
        for (int32_t i = 0; i < n_cells; ++i) adj_off[(size_t)i + 1] += adj_off[(size_t)i];
        {
            std::vector<int32_t> fill(adj_off.begin(), adj_off.end() - 1);
            for (int32_t s = 0; s < n_pairs; ++s) {
                adj_ent[(size_t)fill[(size_t)pair_lo[s]]++] = s << 1;
                adj_ent[(size_t)fill[(size_t)pair_hi[s]]++] = (s << 1) | 1;
            }
        }
        c = new nd_cmfd();
        c->p = p; c->C = n_cells; c->S = n_pairs; c->opt = opt; c->n_crossings = nx;
        c->J_stride = cmfd_J_stride(d, n_cells, n_pairs); c->J_replicas = cmfd_J_replicas(d, n_cells, n_pairs);
        char* ws = static_cast<char*>(device_workspace);
        c->cell = (int32_t*)(ws + L.cell); c->entry_cell = (int32_t*)(ws + L.entry_cell); c->link_fwd = (int32_t*)(ws + L.link_fwd);
        c->lo = (int32_t*)(ws + L.lo); c->hi = (int32_t*)(ws + L.hi); c->pair_key = (int64_t*)(ws + L.pair_key);
        c->pair_idx = (int32_t*)(ws + L.pair_idx); c->adj_off = (int32_t*)(ws + L.adj_off); c->adj_ent = (int32_t*)(ws + L.adj_ent);
        c->coupling = (double*)(ws + L.coupling); c->J = (double*)(ws + L.J); c->Psi = (double*)(ws + L.Psi); c->V = (double*)(ws + L.V);
        c->co = (double*)(ws + L.co); c->out_lo = (double*)(ws + L.out_lo); c->in_hi = (double*)(ws + L.in_hi);
        c->Mw = (double*)(ws + L.Mw); c->Minv = (double*)(ws + L.Minv); c->x = (double*)(ws + L.x); c->y = (double*)(ws + L.y);
        c->y2 = (double*)(ws + L.y2); c->f = (double*)(ws + L.f); c->ratio = (double*)(ws + L.ratio); c->state = (double*)(ws + L.state);
        c->stats = (double*)(ws + L.stats); c->Qtmp = (double*)(ws + L.Qtmp); c->flags = (int*)(ws + L.flags);
        c->xoff = (uint32_t*)(ws + L.xoff); c->xblob = (uint8_t*)(ws + L.xblob);
        auto up = [&](void* dst, const void* src, size_t bytes) {
            return bytes ? cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, st) : cudaSuccess;
        };
        cudaError_t ce = cudaMemsetAsync(ws, 0, L.xoff, st);
        if (ce == cudaSuccess) ce = up(c->cell, cell, sizeof(int32_t) * (size_t)d.R);
        if (ce == cudaSuccess) ce = up(c->entry_cell, h_entry.data(), sizeof(int32_t) * h_entry.size());
        if (ce == cudaSuccess) ce = up(c->lo, pair_lo, sizeof(int32_t) * (size_t)n_pairs);
        if (ce == cudaSuccess) ce = up(c->hi, pair_hi, sizeof(int32_t) * (size_t)n_pairs);
        if (ce == cudaSuccess) ce = up(c->pair_key, key.data(), sizeof(int64_t) * key.size());
        if (ce == cudaSuccess) ce = up(c->pair_idx, idx.data(), sizeof(int32_t) * idx.size());
        if (ce == cudaSuccess) ce = up(c->adj_off, adj_off.data(), sizeof(int32_t) * adj_off.size());
        if (ce == cudaSuccess) ce = up(c->adj_ent, adj_ent.data(), sizeof(int32_t) * 2 * (size_t)n_pairs);
        if (ce == cudaSuccess) ce = up(c->coupling, coupling, sizeof(double) * (size_t)n_pairs);
        if (ce == cudaSuccess) ce = up(c->xoff, xoff.data(), sizeof(uint32_t) * xoff.size());
        if (ce == cudaSuccess) ce = up(c->xblob, xblob.data(), xblob.size());
        if (ce == cudaSuccess) ce = cudaMemsetAsync(c->link_fwd, 0xff, sizeof(int32_t) * 2 * (size_t)d.T, st);
        if (ce == cudaSuccess) {
            ndk::k_link_forward<<<grid_for(2 * (int64_t)d.T, 256, 8 * p->n_sm), 256, 0, st>>>(p->link_src, c->link_fwd, 2 * (int64_t)d.T);
            ce = cudaGetLastError();
        }
        // the coarse solve is a cooperative kernel: every block must be resident
        int per_sm = 0;
        if (ce == cudaSuccess) ce = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ndk::k_coarse_solve, 256, 0);
        if (ce == cudaSuccess) ce = cudaStreamSynchronize(st);      // the host arrays above go out of scope
        if (ce != cudaSuccess) { delete c; return nd_fail(ND_ERR_CUDA, cudaGetErrorString(ce)); }
        // Small systems run as ONE block of 1024 threads (a block barrier costs ~0.1 us, a grid-wide one 2-3 us, and an outer
        // iteration has seven of them); larger ones as a cooperative grid of 256-thread blocks (measured at 11,200 unknowns:
        // one block is latency-starved, 0.6 ms per outer iteration).
        const int64_t want = ((int64_t)n_cells * d.G + 255) / 256;
        c->coop_grid = (int64_t)n_cells * d.G <= 2048     // two unknowns per thread: everything stays in the SM's L1
                           ? 1
                           : (int)std::max<int64_t>(2, std::min<int64_t>({want, (int64_t)n_cells, (int64_t)p->n_sm * std::max(1, per_sm)}));
    } catch (const std::bad_alloc&) {
        delete c;
        return nd_fail(ND_ERR_NOMEM, "nd_cmfd_create: out of host memory");
    }
    *out = c;
    return ND_OK;
}

extern "C" nd_status nd_cmfd_destroy(nd_cmfd* c)
{
    if (c && c->p && c->p->cmfd_sweep == c) c->p->cmfd_sweep = nullptr;
    delete c;
    return ND_OK;
}

namespace {

// C-4 into the plan's arrays
nd_status cmfd_collapse(nd_cmfd* c, const double* phi, cudaStream_t st)
{
    nd_problem* p = c->p;
    const Dims& d = p->d;
    const size_t CG = (size_t)c->C * d.G;
    ND_CUDA(cudaMemsetAsync(c->Psi, 0, sizeof(double) * CG * d.M, st));
    ND_CUDA(cudaMemsetAsync(c->V, 0, sizeof(double) * (size_t)c->C, st));
    ndk::k_cmfd_accumulate<<<grid_for((int64_t)d.R * d.G, 256, 8 * p->n_sm), 256, 0, st>>>(phi, p->vol, p->reg_mat, c->cell, c->Psi, c->V, d.R, d.G, d.M);
    ND_LAUNCH_CHECK(p);
    ndk::k_cmfd_constants<<<grid_for((int64_t)CG, 128, 8 * p->n_sm), 128, 0, st>>>(c->Psi, c->V, p->sigt, p->sigsT, p->nusf, p->chi, c->co, c->C, d.G, d.M);
    ND_LAUNCH_CHECK(p);
    return ND_OK;
}

// C-5..C-8: one cooperative launch; k0 is read from the device scalar *d_k0, the result stays in c->x / c->state
nd_status cmfd_solve(nd_cmfd* c, const double* d_k0, cudaStream_t st)
{
    nd_problem* p = c->p;
    const Dims& d = p->d;
    const size_t CG = (size_t)c->C * d.G;
    ndk::CoarseSolveParams cp{};
    cp.V = c->V; cp.Phi = c->co; cp.sigt = c->co + CG; cp.nusf = c->co + 2 * CG; cp.chi = c->co + 3 * CG; cp.sigs = c->co + 4 * CG;
    cp.J_surf = c->J; cp.J_vac = c->J + (size_t)c->S * d.G; cp.lo = c->lo; cp.hi = c->hi; cp.coupling = c->coupling;
    cp.adj_off = c->adj_off; cp.adj_ent = c->adj_ent; cp.out_lo = c->out_lo; cp.in_hi = c->in_hi; cp.Mw = c->Mw; cp.Minv = c->Minv;
    cp.x = c->x; cp.y = c->y; cp.y2 = c->y2; cp.f = c->f; cp.state = c->state; cp.k0 = d_k0;
    cp.C = c->C; cp.G = d.G; cp.S = c->S; cp.max_outer = c->opt.max_outer; cp.inner = c->opt.inner_sweeps;
    cp.tol_k = c->opt.tol; cp.tol_x = 100.0 * c->opt.tol; cp.rel_tol = c->opt.rel_tol;
    cp.single_block = c->coop_grid == 1;
    if (cp.single_block) {
        ndk::k_coarse_solve<<<1, 1024, 0, st>>>(cp);
        ND_CUDA(cudaGetLastError());
    } else {
        void* args[] = {&cp};
        ND_CUDA(cudaLaunchCooperativeKernel((const void*)ndk::k_coarse_solve, dim3(c->coop_grid), dim3(256), args, 0, st));
    }
    ++p->kernels_launched;
    return ND_OK;
}

// C-9 with the ratio of the last coarse solve (1 everywhere if that solve failed); sets the state's k and fission rate
nd_status cmfd_prolong(nd_cmfd* c, cudaStream_t st)
{
    nd_problem* p = c->p;
    const Dims& d = p->d;
    const int64_t CG = (int64_t)c->C * d.G, nE = 2 * (int64_t)d.T;
    ndk::k_cmfd_ratio<<<grid_for(CG, 256, 8 * p->n_sm), 256, 0, st>>>(c->x, c->co, c->state, c->opt.relax, c->ratio, p->scalars + ndk::SC_K, CG);
    ND_LAUNCH_CHECK(p);
    ndk::k_cmfd_prolong_phi<<<grid_for((int64_t)d.R * d.G, 256, 8 * p->n_sm), 256, 0, st>>>(p->phi_cur, c->cell, c->ratio, d.R, d.G);
    ND_LAUNCH_CHECK(p);
    ndk::k_cmfd_prolong_psi<<<grid_for(nE * d.P * d.Gs, 256, 8 * p->n_sm), 256, 0, st>>>(p->psi_in, c->entry_cell, c->ratio, nE, d.P, d.G, d.Gs);
    ND_LAUNCH_CHECK(p);
    return launch_fission_rate(p, p->phi_cur, nullptr, st);   // the state's F belongs to its flux
}

nd_status cmfd_zero_currents(nd_cmfd* c, cudaStream_t st)
{
    const Dims& d = c->p->d;
    (void)d;
    ND_CUDA(cudaMemsetAsync(c->J, 0, sizeof(double) * (size_t)c->J_stride * c->J_replicas, st));
    return ND_OK;
}

} // namespace

// C-3 with a caller-supplied source: nd_transport_sweep whose sweep kernel also tallies the coarse-mesh currents.
extern "C" nd_status nd_cmfd_sweep(nd_cmfd* c, const double* d_Q, double* d_phi_out, void* cuda_stream)
{
    if (!c || !d_Q || !d_phi_out) return nd_fail(ND_ERR_NULL, "nd_cmfd_sweep: NULL argument");
    cudaStream_t st = as_stream(cuda_stream);
    nd_status rc = cmfd_zero_currents(c, st);
    if (rc != ND_OK) return rc;
    c->p->cmfd_sweep = c;
    rc = nd_transport_sweep(c->p, d_Q, d_phi_out, cuda_stream);
    c->p->cmfd_sweep = nullptr;
    return rc;
}

extern "C" nd_status nd_cmfd_currents_get(nd_cmfd* c, double* J_surf, double* J_vac, double* J_ref, void* cuda_stream)
{
    if (!c || !J_vac || !J_ref || (c->S > 0 && !J_surf)) return nd_fail(ND_ERR_NULL, "nd_cmfd_currents_get: NULL argument");
    cudaStream_t st = as_stream(cuda_stream);
    const Dims& d = c->p->d;
    const size_t SG = (size_t)c->S * d.G, CG = (size_t)c->C * d.G;
    int flag = 0;
    if (SG) ND_CUDA(cudaMemcpyAsync(J_surf, c->J, sizeof(double) * SG, cudaMemcpyDeviceToHost, st));
    ND_CUDA(cudaMemcpyAsync(J_vac, c->J + SG, sizeof(double) * CG, cudaMemcpyDeviceToHost, st));
    ND_CUDA(cudaMemcpyAsync(J_ref, c->J + SG + CG, sizeof(double) * CG, cudaMemcpyDeviceToHost, st));
    ND_CUDA(cudaMemcpyAsync(&flag, c->flags, sizeof(int), cudaMemcpyDeviceToHost, st));
    ND_CUDA(cudaStreamSynchronize(st));
    if (flag) return nd_fail(ND_ERR_STATE, "nd_cmfd: a reflective hand-over joined two coarse cells that are not a listed surface");
    return ND_OK;
}

extern "C" nd_status nd_cmfd_collapse(nd_cmfd* c, const double* d_phi_or_null, void* cuda_stream)
{
    if (!c) return nd_fail(ND_ERR_NULL, "nd_cmfd_collapse: NULL plan");
    return cmfd_collapse(c, d_phi_or_null ? d_phi_or_null : c->p->phi_cur, as_stream(cuda_stream));
}

extern "C" nd_status nd_cmfd_coarse_get(nd_cmfd* c, double* V, double* Phi, double* sigma_t, double* sigma_s, double* nu_sigma_f,
                                        double* chi, void* cuda_stream)
{
    if (!c || !V || !Phi || !sigma_t || !sigma_s || !nu_sigma_f || !chi) return nd_fail(ND_ERR_NULL, "nd_cmfd_coarse_get: NULL argument");
    cudaStream_t st = as_stream(cuda_stream);
    const size_t CG = (size_t)c->C * c->p->d.G, G = (size_t)c->p->d.G;
    ND_CUDA(cudaMemcpyAsync(V, c->V, sizeof(double) * (size_t)c->C, cudaMemcpyDeviceToHost, st));
    ND_CUDA(cudaMemcpyAsync(Phi, c->co, sizeof(double) * CG, cudaMemcpyDeviceToHost, st));
    ND_CUDA(cudaMemcpyAsync(sigma_t, c->co + CG, sizeof(double) * CG, cudaMemcpyDeviceToHost, st));
    ND_CUDA(cudaMemcpyAsync(nu_sigma_f, c->co + 2 * CG, sizeof(double) * CG, cudaMemcpyDeviceToHost, st));
    ND_CUDA(cudaMemcpyAsync(chi, c->co + 3 * CG, sizeof(double) * CG, cudaMemcpyDeviceToHost, st));
    ND_CUDA(cudaMemcpyAsync(sigma_s, c->co + 4 * CG, sizeof(double) * CG * G, cudaMemcpyDeviceToHost, st));
    ND_CUDA(cudaStreamSynchronize(st));
    return ND_OK;
}

extern "C" nd_status nd_cmfd_coarse_set(nd_cmfd* c, const double* V, const double* Phi, const double* sigma_t, const double* sigma_s,
                                        const double* nu_sigma_f, const double* chi, const double* J_surf, const double* J_vac,
                                        void* cuda_stream)
{
    if (!c || !V || !Phi || !sigma_t || !sigma_s || !nu_sigma_f || !chi || !J_vac || (c->S > 0 && !J_surf))
        return nd_fail(ND_ERR_NULL, "nd_cmfd_coarse_set: NULL argument");
    cudaStream_t st = as_stream(cuda_stream);
    const size_t G = (size_t)c->p->d.G, CG = (size_t)c->C * G, SG = (size_t)c->S * G;
    ND_CUDA(cudaMemcpyAsync(c->V, V, sizeof(double) * (size_t)c->C, cudaMemcpyHostToDevice, st));
    ND_CUDA(cudaMemcpyAsync(c->co, Phi, sizeof(double) * CG, cudaMemcpyHostToDevice, st));
    ND_CUDA(cudaMemcpyAsync(c->co + CG, sigma_t, sizeof(double) * CG, cudaMemcpyHostToDevice, st));
    ND_CUDA(cudaMemcpyAsync(c->co + 2 * CG, nu_sigma_f, sizeof(double) * CG, cudaMemcpyHostToDevice, st));
    ND_CUDA(cudaMemcpyAsync(c->co + 3 * CG, chi, sizeof(double) * CG, cudaMemcpyHostToDevice, st));
    ND_CUDA(cudaMemcpyAsync(c->co + 4 * CG, sigma_s, sizeof(double) * CG * G, cudaMemcpyHostToDevice, st));
    if (SG) ND_CUDA(cudaMemcpyAsync(c->J, J_surf, sizeof(double) * SG, cudaMemcpyHostToDevice, st));
    ND_CUDA(cudaMemcpyAsync(c->J + SG, J_vac, sizeof(double) * CG, cudaMemcpyHostToDevice, st));
    ND_CUDA(cudaStreamSynchronize(st));
    return ND_OK;
}

extern "C" nd_status nd_cmfd_solve(nd_cmfd* c, double k0, double* k_out, double* Phi_new, int32_t* iters_done, void* cuda_stream)
{
    if (!c || !k_out) return nd_fail(ND_ERR_NULL, "nd_cmfd_solve: NULL argument");
    if (!(k0 > 0.0)) return nd_fail(ND_ERR_INVALID, "nd_cmfd_solve: k0 must be > 0");
    cudaStream_t st = as_stream(cuda_stream);
    const size_t CG = (size_t)c->C * c->p->d.G;
    double* d_k0 = c->state + ndk::ST_COUNT;
    ND_CUDA(cudaMemcpyAsync(d_k0, &k0, sizeof(double), cudaMemcpyHostToDevice, st));
    ND_CUDA(cudaStreamSynchronize(st));                       // k0 is a stack variable
    nd_status rc = cmfd_solve(c, d_k0, st);
    if (rc != ND_OK) return rc;
    double h[ndk::ST_COUNT];
    ND_CUDA(cudaMemcpyAsync(h, c->state, sizeof h, cudaMemcpyDeviceToHost, st));
    if (Phi_new) ND_CUDA(cudaMemcpyAsync(Phi_new, c->x, sizeof(double) * CG, cudaMemcpyDeviceToHost, st));
    ND_CUDA(cudaStreamSynchronize(st));
    *k_out = h[ndk::ST_K];
    if (iters_done) *iters_done = (int32_t)h[ndk::ST_ITERS];
    if (h[ndk::ST_DONE] == 0.0) return nd_fail(ND_ERR_NOT_CONVERGED, "nd_cmfd_solve: max_outer reached (outputs are written)");
    if (h[ndk::ST_OK] == 0.0) return nd_fail(ND_ERR_INVALID, "nd_cmfd_solve: the coarse eigenpair is not positive (outputs are written)");
    return ND_OK;
}

extern "C" nd_status nd_cmfd_prolong(nd_cmfd* c, void* cuda_stream)
{
    if (!c) return nd_fail(ND_ERR_NULL, "nd_cmfd_prolong: NULL plan");
    return cmfd_prolong(c, as_stream(cuda_stream));
}

// Algorithm 1 on the problem's own state: O-8's iteration with C-3 inside its sweep, then C-4..C-9.
extern "C" nd_status nd_cmfd_iteration(nd_cmfd* c, int32_t n_iters, double* k_eff_out, nd_cmfd_stats* stats, void* cuda_stream)
{
    if (!c || !k_eff_out) return nd_fail(ND_ERR_NULL, "nd_cmfd_iteration: NULL argument");
    if (n_iters < 0) return nd_fail(ND_ERR_INVALID, "nd_cmfd_iteration: n_iters must be >= 0");
    nd_problem* p = c->p;
    const Dims& d = p->d;
    cudaStream_t st = as_stream(cuda_stream);
    ndk::SourceParams sp{};
    sp.reg_mat = p->reg_mat; sp.sigt = p->sigt; sp.sigsT = p->sigsT; sp.nusf = p->nusf; sp.chi = p->chi;
    sp.k_ptr = p->scalars + ndk::SC_K; sp.f_ptr = p->scalars + ndk::SC_F; sp.k_val = 1.0;
    sp.Q = p->Q; sp.q = p->q; sp.tally = p->tally; sp.R = d.R; sp.G = d.G; sp.Gs = d.Gs;
    std::vector<double> hs;
    int delivered = 0;
    auto deliver = [&](int upto) -> nd_status {
        const int n = upto - delivered;
        if (n <= 0 || !stats) { delivered = upto; return ND_OK; }
        hs.resize(4 * (size_t)n);
        ND_CUDA(cudaMemcpyAsync(hs.data(), c->stats, sizeof(double) * hs.size(), cudaMemcpyDeviceToHost, st));
        ND_CUDA(cudaStreamSynchronize(st));
        for (int i = 0; i < n; ++i) {
            nd_cmfd_stats& o = stats[delivered + i];
            o.k_sweep = hs[4 * i]; o.k_eff = hs[4 * i + 1]; o.coarse_iters = (int32_t)hs[4 * i + 2]; o.coarse_ok = (int32_t)hs[4 * i + 3];
        }
        delivered = upto;
        return ND_OK;
    };
    for (int it = 0; it < n_iters; ++it) {
        // ---- O-8: source, sweep (+ C-3), flux, k ----
        sp.phi = p->phi_cur;
        nd_status rc = launch_source(p, sp, st);
        if (rc != ND_OK) return rc;
        rc = cmfd_zero_currents(c, st);
        if (rc != ND_OK) return rc;
        p->cmfd_sweep = c;
        rc = launch_sweep(p, p->scalars + ndk::SC_F, st);
        p->cmfd_sweep = nullptr;
        if (rc != ND_OK) return rc;
        int grid = 0;
        rc = launch_finalise(p, p->Q, p->phi_cur, p->scalars + ndk::SC_F, p->phi_new, &grid, st);
        if (rc != ND_OK) return rc;
        ndk::k_reduce_final<<<1, 256, 0, st>>>(p->partial, grid, p->scalars, 1, nullptr, nullptr, 0);
        ND_LAUNCH_CHECK(p);
        std::swap(p->phi_cur, p->phi_new);
        double* slot = c->stats + 4 * (size_t)((it - delivered) % kCmfdMaxStats);
        ND_CUDA(cudaMemcpyAsync(slot, p->scalars + ndk::SC_K, sizeof(double), cudaMemcpyDeviceToDevice, st));   // k after the sweep
        // ---- C-4 .. C-9 ----
        rc = cmfd_collapse(c, p->phi_cur, st);
        if (rc != ND_OK) return rc;
        rc = cmfd_solve(c, p->scalars + ndk::SC_K, st);
        if (rc != ND_OK) return rc;
        rc = cmfd_prolong(c, st);
        if (rc != ND_OK) return rc;
        ND_CUDA(cudaMemcpyAsync(slot + 1, p->scalars + ndk::SC_K, sizeof(double), cudaMemcpyDeviceToDevice, st));
        ND_CUDA(cudaMemcpyAsync(slot + 2, c->state + ndk::ST_ITERS, sizeof(double), cudaMemcpyDeviceToDevice, st));
        ND_CUDA(cudaMemcpyAsync(slot + 3, c->state + ndk::ST_OK, sizeof(double), cudaMemcpyDeviceToDevice, st));
        if (it + 1 - delivered == kCmfdMaxStats) {
            rc = deliver(it + 1);
            if (rc != ND_OK) return rc;
        }
    }
    nd_status rc = deliver(n_iters);
    if (rc != ND_OK) return rc;
    double hk = 0.0;
    int flag = 0;
    ND_CUDA(cudaMemcpyAsync(&hk, p->scalars + ndk::SC_K, sizeof(double), cudaMemcpyDeviceToHost, st));
    ND_CUDA(cudaMemcpyAsync(&flag, c->flags, sizeof(int), cudaMemcpyDeviceToHost, st));
    ND_CUDA(cudaStreamSynchronize(st));
    *k_eff_out = hk;
    if (flag) return nd_fail(ND_ERR_STATE, "nd_cmfd: a reflective hand-over joined two coarse cells that are not a listed surface");
    return ND_OK;
}
