// nd_p1_api.cuh -- NEXT-4: the P_1-scattering plan (include/nd.h "nd_p1_*"), included by nd_api.cu behind the problem's internals.

struct nd_p1 {
    nd_problem* p = nullptr;
    double c2 = 0.0;                        // sum_p omega_p sin^2(theta_p)
    float sin_t[ndk::kMaxPolar]{};
    // device arrays in the caller's workspace
    double* s1T = nullptr;                  // [M][G_from][G_to]
    float* trk_dir = nullptr;               // [T][2]
    double* Mxx = nullptr; double* Mxy = nullptr; double* Myy = nullptr;   // [R]
    float* q1x = nullptr; float* q1y = nullptr;                            // [R][Gs]
    double* tally_x = nullptr; double* tally_y = nullptr;                  // [R][Gs]
    double* Q1x = nullptr; double* Q1y = nullptr;                          // [R][G]
    double* Jx = nullptr; double* Jy = nullptr;                            // [R][G] state
    double* khist = nullptr;                // [kP1MaxHist]
};

namespace {

constexpr int kP1MaxHist = 4096;

struct P1Layout { size_t s1T, trk_dir, Mxx, Mxy, Myy, q1x, q1y, tally_x, tally_y, Q1x, Q1y, Jx, Jy, khist, total; };

P1Layout p1_layout(const Dims& d)
{
    P1Layout L{};
    size_t c = 0;
    const size_t RG = (size_t)d.R * d.G, RGs = (size_t)d.R * d.Gs;
    L.s1T = bump(c, sizeof(double) * (size_t)d.M * d.G * d.G);
    L.trk_dir = bump(c, sizeof(float) * 2 * (size_t)d.T);
    L.Mxx = bump(c, sizeof(double) * (size_t)d.R);
    L.Mxy = bump(c, sizeof(double) * (size_t)d.R);
    L.Myy = bump(c, sizeof(double) * (size_t)d.R);
    L.q1x = bump(c, sizeof(float) * RGs);
    L.q1y = bump(c, sizeof(float) * RGs);
    L.tally_x = bump(c, sizeof(double) * RGs);
    L.tally_y = bump(c, sizeof(double) * RGs);
    L.Q1x = bump(c, sizeof(double) * RG);
    L.Q1y = bump(c, sizeof(double) * RG);
    L.Jx = bump(c, sizeof(double) * RG);
    L.Jy = bump(c, sizeof(double) * RG);
    L.khist = bump(c, sizeof(double) * kP1MaxHist);
    L.total = c;
    return L;
}

void p1_fill_sweep_params(const nd_p1* c, ndk::SwathParams* prm)
{
    prm->q1x = c->q1x; prm->q1y = c->q1y; prm->trk_dir = c->trk_dir; prm->tally_x = c->tally_x; prm->tally_y = c->tally_y;
    for (int i = 0; i < ndk::kMaxPolar; ++i) prm->sin_t[i] = c->sin_t[i];
}

// sweep with the reduced sources already in p->q, c->q1x, c->q1y and zeroed tallies; then link swap, phi and J
nd_status p1_sweep_and_finalise(nd_p1* c, const double* Q0, const double* scale_div, const double* phi_old, const double* f_ptr,
                                double* phi_out, double* Jx_out, double* Jy_out, int* grid_out, cudaStream_t st)
{
    nd_problem* p = c->p;
    const Dims& d = p->d;
    ndk::P1SweepParams pp{};
    ndk::SweepParams& prm = pp.sw;
    prm.seg_rm = p->seg_rm; prm.seg_len = p->seg_len; prm.trk_off = p->trk_off; prm.trk_w = p->trk_w;
    prm.q = p->q; prm.sigt = p->sigt_f; prm.tally = p->tally; prm.psi_in = p->psi_in; prm.psi_out = p->psi_out; prm.scale_div = scale_div;
    prm.T = d.T; prm.G = d.G; prm.Gs = d.Gs;
    for (int i = 0; i < ndk::kMaxPolar; ++i) { prm.c[i] = p->c[i]; prm.inv_sin[i] = p->inv_sin[i]; prm.wp[i] = p->wp[i]; pp.sin_t[i] = c->sin_t[i]; }
    pp.q1x = c->q1x; pp.q1y = c->q1y; pp.trk_dir = c->trk_dir; pp.tally_x = c->tally_x; pp.tally_y = c->tally_y;
    if (is_swath(p->sweep_kernel)) {   // the swath kernel with the P_1 source (problem created with nd_options.p1_stream)
        p->p1_sweep = c;
        const nd_status rs = launch_swath(p, scale_div, st);
        p->p1_sweep = nullptr;
        if (rs != ND_OK) return rs;
    } else {
        const int grid = grid_for(2 * (int64_t)d.T * 32, 256, 16 * p->n_sm);
        switch (d.P) {
        case 1: ndk::k_sweep_p1<1><<<grid, 256, 0, st>>>(pp); break;
        case 2: ndk::k_sweep_p1<2><<<grid, 256, 0, st>>>(pp); break;
        case 3: ndk::k_sweep_p1<3><<<grid, 256, 0, st>>>(pp); break;
        default: ndk::k_sweep_p1<4><<<grid, 256, 0, st>>>(pp); break;
        }
        ND_LAUNCH_CHECK(p);
    }
    const int PG = d.P * d.Gs;
    const int64_t n = 2 * (int64_t)d.T * PG;
    ndk::k_link_swap<<<grid_for(n, 256, 8 * p->n_sm), 256, 0, st>>>(p->psi_out, p->psi_in, p->link_src, 2 * (int64_t)d.T, PG);
    ND_LAUNCH_CHECK(p);
    nd_status rc = launch_finalise(p, Q0, phi_old, f_ptr, phi_out, grid_out, st);   // phi as in O-6 (the odd part of Q cancels)
    if (rc != ND_OK) return rc;
    ndk::k_p1_currents<<<grid_for((int64_t)d.R * d.G, 256, 8 * p->n_sm), 256, 0, st>>>(c->Q1x, c->Q1y, c->tally_x, c->tally_y, p->reg_mat,
                                                                                    p->sigt, p->vol, c->Mxx, c->Mxy, c->Myy, c->c2,
                                                                                    Jx_out, Jy_out, d.R, d.G, d.Gs);
    ND_LAUNCH_CHECK(p);
    return ND_OK;
}

} // namespace

extern "C" nd_status nd_p1_workspace_bytes(const nd_problem* p, size_t* device_bytes)
{
    if (!p || !device_bytes) return nd_fail(ND_ERR_NULL, "nd_p1_workspace_bytes: NULL argument");
    *device_bytes = p1_layout(p->d).total;
    return ND_OK;
}

extern "C" nd_status nd_p1_create(nd_problem* p, const nd_problem_desc* desc, const double* sigma_s1, void* device_workspace,
                                  size_t device_bytes, void* cuda_stream, nd_p1** out)
{
    if (!p || !desc || !sigma_s1 || !device_workspace || !out) return nd_fail(ND_ERR_NULL, "nd_p1_create: NULL argument");
    if (!p->has_soa && !(is_swath(p->sweep_kernel) && p->opt.p1_stream))
        return nd_fail(ND_ERR_STATE, "nd_p1_create: needs a problem created with sweep_kernel = ND_SWEEP_ATOMIC (the plain segment "
                                     "stream) or a swath-kernel problem created with nd_options.p1_stream = 1");
    if (p->opt.exp_mode != ND_EXP_FAST) return nd_fail(ND_ERR_STATE, "nd_p1_create: built for exp_mode = ND_EXP_FAST");
    const Dims& d = p->d;
    if (!desc->track_ends || !desc->track_seg_offset || !desc->seg_region || !desc->seg_length || !desc->track_weight || !desc->polar_sin ||
        !desc->polar_weight)
        return nd_fail(ND_ERR_NULL, "nd_p1_create: the descriptor needs track_ends, the segment arrays, track_weight and the polar set");
    if (desc->n_tracks != d.T || desc->n_regions != d.R || desc->n_polar != d.P || desc->track_seg_offset[d.T] != d.S)
        return nd_fail(ND_ERR_INVALID, "nd_p1_create: the descriptor is not the one the problem was created from");
    if (reinterpret_cast<uintptr_t>(device_workspace) % kAlign != 0) return nd_fail(ND_ERR_WORKSPACE, "nd_p1_create: workspace must be 256-byte aligned");
    const P1Layout L = p1_layout(d);
    if (device_bytes < L.total) return nd_fail(ND_ERR_WORKSPACE, "nd_p1_create: workspace smaller than nd_p1_workspace_bytes");
    for (size_t i = 0; i < (size_t)d.M * d.G * d.G; ++i)
        if (!std::isfinite(sigma_s1[i])) return nd_fail(ND_ERR_INVALID, "nd_p1_create: sigma_s1 must be finite");
    cudaStream_t st = as_stream(cuda_stream);
    nd_p1* c = nullptr;
    try {
        std::vector<double> s1T((size_t)d.M * d.G * d.G), Mxx((size_t)d.R, 0.0), Mxy((size_t)d.R, 0.0), Myy((size_t)d.R, 0.0);
        std::vector<float> dir(2 * (size_t)d.T);
        for (int m = 0; m < d.M; ++m)
            for (int g = 0; g < d.G; ++g)
                for (int gp = 0; gp < d.G; ++gp) s1T[((size_t)m * d.G + gp) * d.G + g] = sigma_s1[((size_t)m * d.G + g) * d.G + gp];
        for (int t = 0; t < d.T; ++t) {                       // P-2 and the moment areas Mab of P-5
            const double* e = desc->track_ends + 4 * (size_t)t;
            const double dx = e[2] - e[0], dy = e[3] - e[1], h = std::sqrt(dx * dx + dy * dy);
            if (!(h > 0.0) || !std::isfinite(h)) return nd_fail(ND_ERR_INVALID, "nd_p1_create: a track has no direction (track_ends)");
            const double ux = dx / h, uy = dy / h;
            dir[2 * (size_t)t] = (float)ux; dir[2 * (size_t)t + 1] = (float)uy;
            for (int64_t k = desc->track_seg_offset[t]; k < desc->track_seg_offset[t + 1]; ++k) {
                const double a = 2.0 * desc->track_weight[t] * desc->seg_length[k];
                const int32_t r = desc->seg_region[k];
                if (r < 0 || r >= d.R) return nd_fail(ND_ERR_RANGE, "nd_p1_create: seg_region out of range");
                Mxx[(size_t)r] += a * ux * ux; Mxy[(size_t)r] += a * ux * uy; Myy[(size_t)r] += a * uy * uy;
            }
        }
        c = new nd_p1();
        c->p = p;
        for (int i = 0; i < d.P; ++i) {
            c->sin_t[i] = (float)desc->polar_sin[i];
            c->c2 += desc->polar_weight[i] * desc->polar_sin[i] * desc->polar_sin[i];
        }
        char* ws = static_cast<char*>(device_workspace);
        c->s1T = (double*)(ws + L.s1T); c->trk_dir = (float*)(ws + L.trk_dir); c->Mxx = (double*)(ws + L.Mxx); c->Mxy = (double*)(ws + L.Mxy);
        c->Myy = (double*)(ws + L.Myy); c->q1x = (float*)(ws + L.q1x); c->q1y = (float*)(ws + L.q1y); c->tally_x = (double*)(ws + L.tally_x);
        c->tally_y = (double*)(ws + L.tally_y); c->Q1x = (double*)(ws + L.Q1x); c->Q1y = (double*)(ws + L.Q1y); c->Jx = (double*)(ws + L.Jx);
        c->Jy = (double*)(ws + L.Jy); c->khist = (double*)(ws + L.khist);
        cudaError_t ce = cudaMemsetAsync(ws, 0, L.total, st);
        if (ce == cudaSuccess) ce = cudaMemcpyAsync(c->s1T, s1T.data(), sizeof(double) * s1T.size(), cudaMemcpyHostToDevice, st);
        if (ce == cudaSuccess) ce = cudaMemcpyAsync(c->trk_dir, dir.data(), sizeof(float) * dir.size(), cudaMemcpyHostToDevice, st);
        if (ce == cudaSuccess) ce = cudaMemcpyAsync(c->Mxx, Mxx.data(), sizeof(double) * Mxx.size(), cudaMemcpyHostToDevice, st);
        if (ce == cudaSuccess) ce = cudaMemcpyAsync(c->Mxy, Mxy.data(), sizeof(double) * Mxy.size(), cudaMemcpyHostToDevice, st);
        if (ce == cudaSuccess) ce = cudaMemcpyAsync(c->Myy, Myy.data(), sizeof(double) * Myy.size(), cudaMemcpyHostToDevice, st);
        if (ce == cudaSuccess) ce = cudaStreamSynchronize(st);
        if (ce != cudaSuccess) { delete c; return nd_fail(ND_ERR_CUDA, cudaGetErrorString(ce)); }
    } catch (const std::bad_alloc&) {
        delete c;
        return nd_fail(ND_ERR_NOMEM, "nd_p1_create: out of host memory");
    }
    *out = c;
    return ND_OK;
}

extern "C" nd_status nd_p1_destroy(nd_p1* c)
{
    delete c;
    return ND_OK;
}

extern "C" nd_status nd_p1_transport_sweep(nd_p1* c, const double* d_Q0, const double* d_Q1x, const double* d_Q1y, double* d_phi_out,
                                           double* d_Jx_out, double* d_Jy_out, void* cuda_stream)
{
    if (!c || !d_Q0 || !d_Q1x || !d_Q1y || !d_phi_out || !d_Jx_out || !d_Jy_out) return nd_fail(ND_ERR_NULL, "nd_p1_transport_sweep: NULL argument");
    nd_problem* p = c->p;
    const Dims& d = p->d;
    cudaStream_t st = as_stream(cuda_stream);
    const int64_t n = (int64_t)d.R * d.Gs;
    ndk::k_reduced_source<<<grid_for(n, 256, 8 * p->n_sm), 256, 0, st>>>(d_Q0, p->reg_mat, p->sigt, p->q, p->tally, d.R, d.G, d.Gs);
    ND_LAUNCH_CHECK(p);
    ndk::k_p1_reduced_moments<<<grid_for(n, 256, 8 * p->n_sm), 256, 0, st>>>(d_Q1x, d_Q1y, p->reg_mat, p->sigt, c->q1x, c->q1y, c->tally_x,
                                                                             c->tally_y, d.R, d.G, d.Gs);
    ND_LAUNCH_CHECK(p);
    const size_t bytes = sizeof(double) * (size_t)d.R * d.G;
    ND_CUDA(cudaMemcpyAsync(c->Q1x, d_Q1x, bytes, cudaMemcpyDeviceToDevice, st));
    ND_CUDA(cudaMemcpyAsync(c->Q1y, d_Q1y, bytes, cudaMemcpyDeviceToDevice, st));
    int grid = 0;
    return p1_sweep_and_finalise(c, d_Q0, p->scalars + ndk::SC_ONE, nullptr, nullptr, d_phi_out, d_Jx_out, d_Jy_out, &grid, st);
}

extern "C" nd_status nd_p1_source_update(nd_p1* c, const double* d_phi, const double* d_Jx, const double* d_Jy, double k_eff,
                                         double* d_Q0_out, double* d_Q1x_out, double* d_Q1y_out, void* cuda_stream)
{
    if (!c || !d_phi || !d_Jx || !d_Jy || !d_Q0_out || !d_Q1x_out || !d_Q1y_out) return nd_fail(ND_ERR_NULL, "nd_p1_source_update: NULL argument");
    nd_status rc = nd_source_update(c->p, d_phi, k_eff, d_Q0_out, nullptr, cuda_stream);
    if (rc != ND_OK) return rc;
    nd_problem* p = c->p;
    const Dims& d = p->d;
    ndk::k_p1_moment_source<<<grid_for((int64_t)d.R * d.Gs, 256, 8 * p->n_sm), 256, 0, as_stream(cuda_stream)>>>(
        d_Jx, d_Jy, p->reg_mat, p->sigt, c->s1T, nullptr, d_Q1x_out, d_Q1y_out, nullptr, nullptr, nullptr, nullptr, d.R, d.G, d.Gs);
    ND_LAUNCH_CHECK(p);
    return ND_OK;
}

extern "C" nd_status nd_p1_state_reset(nd_p1* c, void* cuda_stream)
{
    if (!c) return nd_fail(ND_ERR_NULL, "nd_p1_state_reset: NULL plan");
    const size_t bytes = sizeof(double) * (size_t)c->p->d.R * c->p->d.G;
    ND_CUDA(cudaMemsetAsync(c->Jx, 0, bytes, as_stream(cuda_stream)));
    ND_CUDA(cudaMemsetAsync(c->Jy, 0, bytes, as_stream(cuda_stream)));
    return reset_state(c->p, as_stream(cuda_stream));
}

// P-6 on the problem's state (phi, boundary psi, k, F) and the plan's currents
extern "C" nd_status nd_p1_power_iteration(nd_p1* c, int32_t n_iters, double* k_eff_out, double* d_phi_out, double* d_Jx_out,
                                           double* d_Jy_out, double* k_history, void* cuda_stream)
{
    if (!c || !k_eff_out) return nd_fail(ND_ERR_NULL, "nd_p1_power_iteration: NULL argument");
    if (n_iters < 0) return nd_fail(ND_ERR_INVALID, "nd_p1_power_iteration: n_iters must be >= 0");
    nd_problem* p = c->p;
    const Dims& d = p->d;
    cudaStream_t st = as_stream(cuda_stream);
    ndk::SourceParams sp{};
    sp.reg_mat = p->reg_mat; sp.sigt = p->sigt; sp.sigsT = p->sigsT; sp.nusf = p->nusf; sp.chi = p->chi;
    sp.k_ptr = p->scalars + ndk::SC_K; sp.f_ptr = p->scalars + ndk::SC_F; sp.k_val = 1.0;
    sp.Q = p->Q; sp.q = p->q; sp.tally = p->tally; sp.R = d.R; sp.G = d.G; sp.Gs = d.Gs;
    int delivered = 0;
    std::vector<double> hs;
    auto deliver = [&](int upto) -> nd_status {
        const int n = upto - delivered;
        if (n > 0 && k_history) {
            hs.resize((size_t)n);
            ND_CUDA(cudaMemcpyAsync(hs.data(), c->khist, sizeof(double) * hs.size(), cudaMemcpyDeviceToHost, st));
            ND_CUDA(cudaStreamSynchronize(st));
            for (int i = 0; i < n; ++i) k_history[delivered + i] = hs[(size_t)i];
        }
        delivered = upto;
        return ND_OK;
    };
    for (int it = 0; it < n_iters; ++it) {
        sp.phi = p->phi_cur;
        nd_status rc = launch_source(p, sp, st);            // Q0, q0, tally0 = 0 (phi / F inside)
        if (rc != ND_OK) return rc;
        ndk::k_p1_moment_source<<<grid_for((int64_t)d.R * d.Gs, 256, 8 * p->n_sm), 256, 0, st>>>(
            c->Jx, c->Jy, p->reg_mat, p->sigt, c->s1T, p->scalars + ndk::SC_F, c->Q1x, c->Q1y, c->q1x, c->q1y, c->tally_x, c->tally_y, d.R, d.G,
            d.Gs);
        ND_LAUNCH_CHECK(p);
        int grid = 0;
        rc = p1_sweep_and_finalise(c, p->Q, p->scalars + ndk::SC_F, p->phi_cur, p->scalars + ndk::SC_F, p->phi_new, c->Jx, c->Jy, &grid, st);
        if (rc != ND_OK) return rc;
        ndk::k_reduce_final<<<1, 256, 0, st>>>(p->partial, grid, p->scalars, 1, nullptr, nullptr, 0);
        ND_LAUNCH_CHECK(p);
        std::swap(p->phi_cur, p->phi_new);
        ND_CUDA(cudaMemcpyAsync(c->khist + (it - delivered) % kP1MaxHist, p->scalars + ndk::SC_K, sizeof(double), cudaMemcpyDeviceToDevice, st));
        if (it + 1 - delivered == kP1MaxHist) {
            rc = deliver(it + 1);
            if (rc != ND_OK) return rc;
        }
    }
    nd_status rc = deliver(n_iters);
    if (rc != ND_OK) return rc;
    double hk = 0.0;
    const size_t bytes = sizeof(double) * (size_t)d.R * d.G;
    ND_CUDA(cudaMemcpyAsync(&hk, p->scalars + ndk::SC_K, sizeof(double), cudaMemcpyDeviceToHost, st));
    if (d_phi_out) ND_CUDA(cudaMemcpyAsync(d_phi_out, p->phi_cur, bytes, cudaMemcpyDeviceToDevice, st));
    if (d_Jx_out) ND_CUDA(cudaMemcpyAsync(d_Jx_out, c->Jx, bytes, cudaMemcpyDeviceToDevice, st));
    if (d_Jy_out) ND_CUDA(cudaMemcpyAsync(d_Jy_out, c->Jy, bytes, cudaMemcpyDeviceToDevice, st));
    ND_CUDA(cudaStreamSynchronize(st));
    *k_eff_out = hk;
    return ND_OK;
}
