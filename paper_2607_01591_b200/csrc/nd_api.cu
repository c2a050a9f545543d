// nd_api.cu -- the C ABI of include/nd.h: validation, device layout, stream packing (row A1), kernel
// launches (rows A2-A6) and the power-iteration driver (row A7).  No CPU fallback anywhere: every compute
// entry point launches CUDA kernels and returns ND_ERR_CUDA if that fails.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include <cuda_runtime.h>
#include <omp.h>

#include "nd.h"
#include "nd_internal.h"
#include "nd_kernels.cuh"
#include "nd_cmfd.cuh"
#include "nd_p1.cuh"
#include "nd_sweep_swath.cuh"
#include "nd_swath.h"
#include "nd_swath_device.h"
#include "nd_setup.cuh"

// ------------------------------------------------------------------------------------------------
// errors
// ------------------------------------------------------------------------------------------------
static thread_local std::string g_last_error;

nd_status nd_fail(nd_status s, const char* msg)
{
    g_last_error = msg ? msg : "";
    return s;
}

#define ND_CUDA(call)                                                                                   \
    do {                                                                                                \
        cudaError_t e_ = (call);                                                                        \
        if (e_ != cudaSuccess) {                                                                        \
            char buf_[512];                                                                             \
            snprintf(buf_, sizeof buf_, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
            return nd_fail(ND_ERR_CUDA, buf_);                                                          \
        }                                                                                               \
    } while (0)

extern "C" const char* nd_status_string(nd_status s)
{
    switch (s) {
    case ND_OK: return "ND_OK";
    case ND_ERR_NULL: return "ND_ERR_NULL";
    case ND_ERR_INVALID: return "ND_ERR_INVALID";
    case ND_ERR_RANGE: return "ND_ERR_RANGE";
    case ND_ERR_WORKSPACE: return "ND_ERR_WORKSPACE";
    case ND_ERR_CUDA: return "ND_ERR_CUDA";
    case ND_ERR_STATE: return "ND_ERR_STATE";
    case ND_ERR_NOT_CONVERGED: return "ND_ERR_NOT_CONVERGED";
    case ND_ERR_MESH: return "ND_ERR_MESH";
    case ND_ERR_NOMEM: return "ND_ERR_NOMEM";
    }
    return "ND_ERR_UNKNOWN";
}
extern "C" const char* nd_last_error(const nd_problem*) { return g_last_error.c_str(); }
extern "C" uint32_t nd_version(void) { return ND_VERSION; }
#ifndef ND_BUILD_ID
#define ND_BUILD_ID "unknown"
#endif
extern "C" const char* nd_build_id(void) { return ND_BUILD_ID; }

// ------------------------------------------------------------------------------------------------
// device layout
// ------------------------------------------------------------------------------------------------
namespace {

constexpr size_t kAlign = 256;
constexpr int kReduceBlocks = 592; // 4 x 148 SMs

struct Dims {
    int R, M, G, P, T, Gs;
    int64_t S, Spad;
};

constexpr int kSmemMax = 227 * 1024;

// Configuration of the swath sweep (ND_SWEEP_SWATH) for a given G; feasible == false -> other kernels only.
struct SwathConfig {
    bool feasible = false;
    NdSwathParams sp{};
    int LPT = 0, warps = 0, ndbuf = 1, blocks_per_sm = 1;
    bool tight = false;                                   // register-capped kernel variant (more than 512 resident threads per SM)
    int head_cap = 0, rec_cap = 0, off_sigt = 0, off_q = 0, off_dbuf = 0, off_head = 0, off_rec = 0, smem_bytes = 0;
    int x_cap = 0, off_x = 0, off_w = 0;                  // nd_options.cmfd_stream: crossing-list ring and the slots' W rows
    int off_q2 = 0, off_dbuf2 = 0;                        // nd_options.p1_stream: second q rows and second delta buffer
    int64_t max_tiles = 0, max_swaths = 0;
    size_t max_blob = 0;
};

inline bool is_swath(int kernel) { return kernel == ND_SWEEP_SWATH; }

SwathConfig make_swath_config_q(const Dims& d, const nd_options& opt, int q_copies)
{
    SwathConfig c;
    c.LPT = d.Gs / 4;
    if (c.LPT > 32) return c;
    const int NC = (c.LPT == 1 || c.LPT == 2 || c.LPT == 4) ? 8 / c.LPT : 1;
    const int row_bytes = 4 * d.Gs, line = NC * row_bytes;
    int NCq = q_copies > 0 ? q_copies : NC;
    if (NCq > NC) NCq = NC;
    while (NC % NCq != 0) --NCq;   // rounded down to a divisor of NC
    const int line_q = NCq * row_bytes;
    if ((int64_t)d.M * line > 64 * 1024) return c;   // the Sigma_t table must leave room for everything else
    int warps = opt.block_warps > 0 ? opt.block_warps : (c.LPT > 8 ? 8 : 4);
    if (warps > 16) warps = 16;
    c.ndbuf = opt.delta_buffers == 2 ? 2 : 1;
    auto pad128 = [](int x) { return (x + 127) / 128 * 128; };
    auto layout = [&](int w, int Kmax, int Lmax) -> bool {   // fills c for (w, Kmax, Lmax); false if the slot count is unusable
        const int NT = w * 32 / c.LPT / NC * NC;               // slots are packed over the lanes of the whole block
        if (NT < 1 || (int64_t)NT * Kmax > 65535) return false;
        if (Lmax < 16) Lmax = 16;
        {   // the kernel's fastdiv works below 2^16: regions x pieces per staged row
            const int per_region = std::max(d.Gs / 2, NC * (d.Gs / 4));
            if (Lmax > 65535 / per_region) Lmax = 65535 / per_region;
        }
        c.sp.NT = NT; c.sp.Kmax = Kmax; c.sp.Lmax = Lmax; c.sp.NC = NC; c.sp.NCq = NCq; c.sp.row_bytes = row_bytes;
        // narrow rows (G <= 16): the flush is cheap, idle slot steps are not -> equal-count tiles while the fronts stay within
        // 16 segments; wide rows: only within 4 segments (the tally re-use rho pays more than level counts), measured in profiles/
        c.sp.lag = opt.tile_lag < 0 ? -1.0 : (opt.tile_lag > 0 ? (double)opt.tile_lag : (row_bytes < 64 ? 16.0 : 4.0));
        c.sp.item_order = opt.item_order;
        c.head_cap = nd_swath_head_capacity(c.sp);
        c.rec_cap = nd_swath_rec_capacity(c.sp);
        c.off_sigt = 128;
        c.off_q = c.off_sigt + pad128(d.M * line);
        c.off_dbuf = c.off_q + pad128(2 * Lmax * line_q);
        c.off_head = c.off_dbuf + pad128(c.ndbuf * (NT * Kmax + 1) * row_bytes);   // + the spare row of the null record
        c.off_rec = c.off_head + pad128(ndk::kSwathHeadBufs * c.head_cap);
        c.smem_bytes = c.off_rec + ndk::kSwathRecBufs * c.rec_cap;
        if (opt.cmfd_stream) {   // CMFD current tally in the sweep kernel: W per slot + a ring of crossing lists
            c.sp.keep_slot_start = true;
            c.x_cap = (8 * (1 + NT * Kmax) + 15) / 16 * 16;
            c.off_w = pad128(c.smem_bytes);
            c.off_x = c.off_w + pad128(NT * row_bytes);
            c.smem_bytes = c.off_x + ndk::kSwathXBufs * c.x_cap;
        }
        if (opt.p1_stream) {     // P_1 sweep in the sweep kernel: qB rows beside the q rows, a second delta buffer
            c.off_q2 = pad128(c.smem_bytes);
            c.off_dbuf2 = c.off_q2 + pad128(2 * Lmax * line_q);
            c.smem_bytes = c.off_dbuf2 + pad128(c.ndbuf * (NT * Kmax + 1) * row_bytes);
        }
        return true;
    };
    // Defaults (measured, profiles/): occupancy beats tile length once a tile holds >= 8 segments per track.  Aim at
    // 3 resident blocks per SM (4 for narrow rows), the longest tile that fits, and a region window sized for the
    // tally re-use the configs show (rho ~ 6.5 wide rows, ~ 8 narrow rows).
    const int target_blocks = row_bytes < 64 ? 4 : 3;
    if (opt.block_warps <= 0) {
        // small problems: fewer tracks per block until there are about two work items (swath, direction) per resident
        // block of a 148-SM part -- the sweep of a small problem is bound by its longest track, not by throughput
        auto slots = [&](int w) { const int n = w * 32 / c.LPT / NC * NC; return n > 0 ? n : 1; };
        while (warps > 1 && 2 * ((int64_t)d.T / slots(warps)) < 2 * 148 * target_blocks) warps /= 2;
    }
    const double rho_est = row_bytes < 64 ? 8.0 : 6.5;
    bool placed = false;
    for (; warps >= 1 && !placed; --warps) {
        const int NT = warps * 32 / c.LPT / NC * NC;
        if (NT < 1) continue;
        if (opt.tile_segments > 0 || opt.window_regions > 0) {   // explicit tile shape: take it if it fits at all
            const int K = opt.tile_segments > 0 ? opt.tile_segments : 16;
            const int Lw = opt.window_regions > 0 ? opt.window_regions : (int)(NT * K / rho_est + 3) / 4 * 4;
            placed = layout(warps, K, Lw) && c.smem_bytes <= kSmemMax;
        } else {
            // longest tile that fits `blocks` per SM; the region window may shrink by up to 8 rows below the estimate
            for (int blocks = target_blocks; blocks >= 1 && !placed; --blocks)
                for (int K = 16; K >= 8 && !placed; --K)
                    for (int cut = 0; cut <= 8 && !placed; cut += 2) {
                        const int Lw = (int)(NT * K / rho_est + 3) / 4 * 4 - cut;
                        placed = layout(warps, K, Lw < 24 ? 24 : Lw) && c.smem_bytes + 1024 <= (kSmemMax + 1024) / blocks;
                    }
        }
        if (placed) break;
    }
    if (!placed) return c;
    c.warps = warps;
    int bps = (kSmemMax + 1024) / (c.smem_bytes + 1024);  // 1 KB per block is reserved by the driver
    if (bps * warps * 32 > 768) bps = 768 / (warps * 32);  // 85 registers per thread at most
    if (bps > 8) bps = 8;
    if (bps < 1) bps = 1;
    if (opt.blocks_per_sm > 0 && opt.blocks_per_sm < bps) bps = opt.blocks_per_sm;
    c.blocks_per_sm = bps;
    if (opt.p1_stream && bps * warps * 32 > 512) bps = std::max(1, 512 / (warps * 32));   // the P_1 loop needs the roomy register budget
    c.tight = bps * warps * 32 > 512 && warps <= 12;
    if (bps * warps * 32 > 512 && !c.tight) c.blocks_per_sm = bps = 512 / (warps * 32) > 0 ? 512 / (warps * 32) : 1;
    c.max_swaths = d.T;
    c.max_tiles = nd_swath_max_tiles(c.sp, d.S, d.T);
    c.max_blob = nd_swath_max_blob(c.sp, d.S, d.T);
    c.feasible = true;
    return c;
}

// q rows: one copy per region unless asked otherwise (measured: config 3 0.628 -> 0.555 ms, config 2 0.079 -> 0.070 ms).
// The register-capped variant of k_sweep_swath is compiled for q rows laid out like the Sigma_t table (NCq = NC, no
// extra registers): if the one-copy layout ends up on the capped variant the configuration is redone with replicated rows.
SwathConfig make_swath_config(const Dims& d, const nd_options& opt)
{
    SwathConfig c = make_swath_config_q(d, opt, opt.q_copies > 0 ? opt.q_copies : 1);
    if (c.feasible && c.tight && c.sp.NCq != c.sp.NC) c = make_swath_config_q(d, opt, 0);
    return c;
}

// Which sweep kernel a descriptor + options select (decided before the workspace is sized).
int select_kernel(const nd_problem_desc* desc, const nd_options& opt, const SwathConfig& sc)
{
    if (is_swath(opt.sweep_kernel) && sc.feasible) return opt.sweep_kernel;
    if (opt.sweep_kernel == ND_SWEEP_AUTO && desc->track_ends && sc.feasible) return ND_SWEEP_SWATH;
    return ND_SWEEP_ATOMIC;
}

struct Layout { // byte offsets into the workspace
    size_t seg_rm, seg_len, trk_off, trk_w, link_src, psi_a, psi_b, q, tally, phi_a, phi_b, Q, reg_mat, vol, sigt, sigsT,
        nusf, chi, sigt_f, scalars, partial, partial_b, exit_vac, stats, src_region, src_chunks, phase, setup, slot_start, blob, tile_chunk, swath_tile0, swath_track, items, counter, total;
    size_t slot_start_bytes;
};

inline size_t bump(size_t& cur, size_t bytes)
{
    const size_t at = cur;
    cur = (cur + bytes + kAlign - 1) / kAlign * kAlign;
    return at;
}

// scratch of nd_problem_create's device passes (nd_problem_desc.seg_on_device): raw offsets, 2 * weights, entry regions, flags
inline size_t setup_scratch_bytes(const Dims& d, const SwathConfig& sc, int kernel)
{
    const size_t T = (size_t)d.T;
    return 4 * kAlign + 8 * (T + 1) + 8 * T + 8 * T + 256 + (is_swath(kernel) ? nd_swath_device_scratch_bytes(d.T, sc.max_swaths) : 0);
}

Layout make_layout(const Dims& d, int max_stats, const SwathConfig& sc, int kernel, bool keep_soa, bool seg_dev)
{
    Layout L{};
    size_t c = 0;
    const size_t RG = (size_t)d.R * d.G, RGs = (size_t)d.R * d.Gs, NPSI = (size_t)d.T * 2 * d.P * d.Gs;
    // the v0 SoA stream is read by the atomic kernel (and the CMFD current tally: nd_options.cmfd_stream); the tiled kernels
    // carry their own chunk stream
    (void)keep_soa;
    const size_t soa = kernel == ND_SWEEP_ATOMIC ? (size_t)d.Spad : 4;
    L.seg_rm = bump(c, sizeof(uint32_t) * soa);
    L.seg_len = bump(c, sizeof(float) * soa);
    L.trk_off = bump(c, sizeof(int64_t) * ((size_t)d.T + 1));
    L.trk_w = bump(c, sizeof(float) * (size_t)d.T);
    L.link_src = bump(c, sizeof(int32_t) * 2 * (size_t)d.T);
    L.psi_a = bump(c, sizeof(float) * NPSI);
    L.psi_b = bump(c, sizeof(float) * NPSI);
    L.q = bump(c, sizeof(float) * RGs);
    L.tally = bump(c, sizeof(double) * RGs);
    L.phi_a = bump(c, sizeof(double) * RG);
    L.phi_b = bump(c, sizeof(double) * RG);
    L.Q = bump(c, sizeof(double) * RG);
    L.reg_mat = bump(c, sizeof(int32_t) * (size_t)d.R);
    L.vol = bump(c, sizeof(double) * (size_t)d.R);
    L.sigt = bump(c, sizeof(double) * (size_t)d.M * d.G);
    L.sigsT = bump(c, sizeof(double) * (size_t)d.M * d.G * d.G);
    L.nusf = bump(c, sizeof(double) * (size_t)d.M * d.G);
    L.chi = bump(c, sizeof(double) * (size_t)d.M * d.G);
    L.sigt_f = bump(c, sizeof(float) * (size_t)d.M * d.Gs);
    L.scalars = bump(c, sizeof(double) * ndk::SC_COUNT);
    L.partial = bump(c, sizeof(double) * ndk::kPartialStride * kReduceBlocks);
    L.partial_b = bump(c, sizeof(double) * ndk::kPartialStride * kReduceBlocks);
    L.exit_vac = bump(c, 2 * (size_t)d.T);
    L.stats = bump(c, sizeof(double) * ndk::kStatsStride * (size_t)max_stats);
    L.phase = bump(c, 256);
    L.src_region = bump(c, sizeof(int32_t) * (size_t)d.R);
    L.src_chunks = bump(c, sizeof(int4) * ((size_t)d.R / 4 + (size_t)d.M + 1));   // chunks hold >= 4 regions except one per material
    if (seg_dev) {
        L.setup = bump(c, setup_scratch_bytes(d, sc, kernel));
        // the CMFD crossing lists are built on the host from every tile's slot_start array: the device builder writes them here
        L.slot_start_bytes = is_swath(kernel) && keep_soa ? 2 * (size_t)sc.max_tiles * (sc.sp.NT + 1) : 0;
        L.slot_start = bump(c, L.slot_start_bytes);
    }
    if (is_swath(kernel)) {
        L.blob = bump(c, sc.max_blob);
        L.tile_chunk = bump(c, sizeof(uint2) * (size_t)sc.max_tiles);
        L.swath_tile0 = bump(c, sizeof(int64_t) * ((size_t)sc.max_swaths + 1));
        L.swath_track = bump(c, sizeof(int32_t) * (size_t)sc.max_swaths * sc.sp.NT);
        L.items = bump(c, sizeof(int4) * (2 * (size_t)sc.max_swaths + 2));
        L.counter = bump(c, 256);
    }
    L.total = c;
    return L;
}

constexpr int kMaxStats = 4096;

nd_status basic_dims(const nd_problem_desc* desc, Dims& d)
{
    if (!desc) return nd_fail(ND_ERR_NULL, "descriptor is NULL");
    if (!desc->track_seg_offset) return nd_fail(ND_ERR_NULL, "track_seg_offset is NULL");
    if (desc->n_regions < 1 || desc->n_materials < 1 || desc->n_groups < 1 || desc->n_polar < 1 || desc->n_tracks < 1)
        return nd_fail(ND_ERR_INVALID, "n_regions, n_materials, n_groups, n_polar, n_tracks must be >= 1");
    if (desc->n_regions > (1 << 24) || desc->n_materials > 256 || desc->n_groups > 256 || desc->n_polar > ndk::kMaxPolar ||
        desc->n_tracks > (1 << 30))
        return nd_fail(ND_ERR_RANGE, "limits: n_regions <= 2^24, n_materials <= 256, n_groups <= 256, n_polar <= 4, n_tracks <= 2^30");
    d.R = desc->n_regions; d.M = desc->n_materials; d.G = desc->n_groups; d.P = desc->n_polar; d.T = desc->n_tracks;
    d.Gs = (d.G + 3) / 4 * 4;
    const int64_t* off = desc->track_seg_offset;
    if (off[0] != 0) return nd_fail(ND_ERR_INVALID, "track_seg_offset[0] must be 0");
    int64_t spad = 0;
    for (int t = 0; t < d.T; ++t) {
        const int64_t n = off[t + 1] - off[t];
        if (n < 0) return nd_fail(ND_ERR_INVALID, "track_seg_offset must be non-decreasing");
        spad += (n + 3) / 4 * 4;
    }
    d.S = off[d.T];
    d.Spad = spad > 0 ? spad : 4;
    return ND_OK;
}

struct EventPair { cudaEvent_t a, b; };

} // namespace

struct nd_problem {
    Dims d{};
    nd_options opt{};
    Layout L{};
    char* ws = nullptr;
    int sweep_kernel = ND_SWEEP_ATOMIC;
    bool has_soa = false;                  // the plain SoA segment stream is on the device (atomic kernel, CMFD currents)
    int n_sm = 148;
    // device pointers into the workspace
    uint32_t* seg_rm; float* seg_len; int64_t* trk_off; float* trk_w; int32_t* link_src;
    float* psi_in; float* psi_out; float* q; double* tally; double* phi_cur; double* phi_new; double* Q;
    int32_t* reg_mat; double* vol; double* sigt; double* sigsT; double* nusf; double* chi; float* sigt_f;
    double* scalars; double* partial; double* partial_b; uint8_t* exit_vac; double* stats;
    int32_t* src_region = nullptr; int4* src_chunks = nullptr;
    int n_src_chunks = 0, src_chunk_regions = 0;
    bool source_attr_set = false;
    // swath sweep
    SwathConfig sc{};
    double lockstep_efficiency = 0.0;
    uint8_t* blob = nullptr; uint2* tile_ref = nullptr; int64_t* swath_tile0 = nullptr; int32_t* swath_track = nullptr;
    int4* items = nullptr; int* counter = nullptr;
    int n_items = 0;
    int64_t n_tiles = 0, n_swaths = 0;
    size_t blob_bytes = 0;
    bool stream_on_device = false;          // the chunk stream was built by nd_build_swaths_device
    double mean_regions_per_tile = 0.0, mean_segments_per_tile = 0.0;
    // host copies
    std::vector<double> h_vol;
    std::vector<int32_t> h_entry_region;   // [2T] first region of chain (t, d), -1 for an empty track (C-9)
    // nd_options.cmfd_stream: what nd_cmfd_create needs to place the coarse-surface crossings into the tiles
    std::vector<int32_t> h_swath_track;    // [n_swaths][NT]
    std::vector<int64_t> h_swath_tile0;    // [n_swaths+1]
    std::vector<uint16_t> h_slot_start;    // [n_tiles][NT+1]
    nd_cmfd* cmfd_sweep = nullptr;         // set while a sweep has to tally the currents of this plan (C-3)
    nd_p1* p1_sweep = nullptr;             // set while the swath kernel sweeps with this plan's P_1 source (nd_options.p1_stream)
    float c[ndk::kMaxPolar]{}, inv_sin[ndk::kMaxPolar]{}, wp[ndk::kMaxPolar]{};
    // profiling
    bool profile = false, phase_profile = false;
    unsigned long long* phase = nullptr;   // [kSwathPhases] device counters of the instrumented swath kernel
    std::vector<EventPair> ev_pool;
    size_t ev_used = 0;
    int64_t kernels_launched = 0;
    // NEXT-2: called on the tally of every sweep before it is turned into a flux (all-reduce over the shards)
    nd_tally_reduce_fn reduce_fn = nullptr;
    void* reduce_user = nullptr;
    // CUDA graph of two power iterations (phi_cur returns to the buffer it started in), see nd_power_iteration
    cudaGraphExec_t iter_graph = nullptr;
    cudaStream_t cap_stream = nullptr;        // capture only; replays run on the caller's stream
    const double* iter_graph_phi = nullptr;   // phi_cur the graph was captured with
    int64_t iter_graph_kernels = 0;           // kernels one replay launches
};

namespace {

void cmfd_fill_sweep_params(const nd_cmfd* c, ndk::SwathParams* prm);   // nd_cmfd_api.cuh
void p1_fill_sweep_params(const nd_p1* c, ndk::SwathParams* prm);       // nd_p1_api.cuh
nd_status cmfd_end_currents(nd_cmfd* c, const double* scale_div, cudaStream_t st);

inline cudaStream_t as_stream(void* s) { return reinterpret_cast<cudaStream_t>(s); }

inline int grid_for(int64_t n, int block, int cap)
{
    int64_t g = (n + block - 1) / block;
    if (g < 1) g = 1;
    return (int)(g > cap ? cap : g);
}

#define ND_LAUNCH_CHECK(p)                                                      \
    do {                                                                        \
        ++(p)->kernels_launched;                                                \
        ND_CUDA(cudaGetLastError());                                            \
    } while (0)

nd_status launch_fill_f64(nd_problem* p, double* ptr, double v, int64_t n, cudaStream_t st)
{
    ndk::k_fill_f64<<<grid_for(n, 256, 4 * p->n_sm), 256, 0, st>>>(ptr, v, n);
    ND_LAUNCH_CHECK(p);
    return ND_OK;
}
nd_status launch_fill_f32(nd_problem* p, float* ptr, float v, int64_t n, cudaStream_t st)
{
    ndk::k_fill_f32<<<grid_for(n, 256, 4 * p->n_sm), 256, 0, st>>>(ptr, v, n);
    ND_LAUNCH_CHECK(p);
    return ND_OK;
}

// F = sum A~ nuSigma_f phi into scalars[SC_F] (and optionally a caller's device scalar)
nd_status launch_fission_rate(nd_problem* p, const double* d_phi, double* d_out, cudaStream_t st)
{
    const Dims& d = p->d;
    const int grid = grid_for((int64_t)d.R * d.G, 256, kReduceBlocks);
    ndk::k_fission_partial<<<grid, 256, 0, st>>>(d_phi, p->reg_mat, p->nusf, p->vol, p->partial, d.R, d.G);
    ND_LAUNCH_CHECK(p);
    ndk::k_reduce_final<<<1, 256, 0, st>>>(p->partial, grid, p->scalars, 0, nullptr, nullptr, 0);
    ND_LAUNCH_CHECK(p);
    if (d_out) ND_CUDA(cudaMemcpyAsync(d_out, p->scalars + ndk::SC_F, sizeof(double), cudaMemcpyDeviceToDevice, st));
    return ND_OK;
}

inline int swath_grid(const nd_problem* p)
{
    const int g = p->n_sm * p->sc.blocks_per_sm;
    return p->n_items < g ? (p->n_items > 0 ? p->n_items : 1) : g;
}

template <int P>
nd_status launch_swath_p(nd_problem* p, const ndk::SwathParams& prm, cudaStream_t st)
{
    const SwathConfig& c = p->sc;
    const bool expm1 = p->opt.exp_mode == ND_EXP_EXPM1;
    const bool tight = c.tight && !expm1;   // the expm1f cross-check path keeps the roomy register budget
    const bool prof = p->phase_profile && !expm1;   // instrumented build: clock64 marks around the phases of a tile
    const bool cur = prm.xblob != nullptr;          // CMFD: the sweep also tallies the coarse-surface currents (fast-exp path only)
    if (prm.q1x != nullptr) {                       // P_1 source (an nd_p1 plan on a problem with nd_options.p1_stream)
        auto k1 = ndk::k_sweep_swath<P, 0, 0, 0, 0, 1>;
        ND_CUDA(cudaFuncSetAttribute(k1, cudaFuncAttributeMaxDynamicSharedMemorySize, c.smem_bytes));
        k1<<<swath_grid(p), 32 * c.warps, c.smem_bytes, st>>>(prm);
        ND_LAUNCH_CHECK(p);
        return ND_OK;
    }
    auto kern = expm1 ? ndk::k_sweep_swath<P, 1, 0, 0>
                : cur ? (tight ? ndk::k_sweep_swath<P, 0, 1, 0, 1> : ndk::k_sweep_swath<P, 0, 0, 0, 1>)
                      : (tight ? (prof ? ndk::k_sweep_swath<P, 0, 1, 1> : ndk::k_sweep_swath<P, 0, 1, 0>)
                               : (prof ? ndk::k_sweep_swath<P, 0, 0, 1> : ndk::k_sweep_swath<P, 0, 0, 0>));
    ND_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, c.smem_bytes));
    kern<<<swath_grid(p), 32 * c.warps, c.smem_bytes, st>>>(prm);
    ND_LAUNCH_CHECK(p);
    return ND_OK;
}

nd_status launch_swath(nd_problem* p, const double* scale_div, cudaStream_t st)
{
    const Dims& d = p->d;
    const SwathConfig& c = p->sc;
    ndk::SwathParams prm{};
    prm.blob = p->blob; prm.tile_ref = p->tile_ref; prm.swath_tile0 = p->swath_tile0; prm.swath_track = p->swath_track;
    prm.items = p->items; prm.counter = p->counter; prm.q = p->q; prm.sigt = p->sigt_f; prm.tally = p->tally; prm.trk_w = p->trk_w;
    prm.psi_in = p->psi_in; prm.psi_out = p->psi_out; prm.scale_div = scale_div;
    prm.n_items = p->n_items; prm.G = d.G; prm.Gs = d.Gs; prm.M = d.M; prm.NT = c.sp.NT; prm.Kmax = c.sp.Kmax; prm.Lmax = c.sp.Lmax;
    prm.LPT = c.LPT; prm.NC = c.sp.NC; prm.NCq = c.sp.NCq > 0 ? c.sp.NCq : c.sp.NC; prm.ndbuf = c.ndbuf; prm.head_cap = c.head_cap; prm.rec_cap = c.rec_cap;
    prm.off_sigt = c.off_sigt; prm.off_q = c.off_q; prm.off_dbuf = c.off_dbuf; prm.off_head = c.off_head; prm.off_rec = c.off_rec;
    for (int i = 0; i < ndk::kMaxPolar; ++i) {
        prm.c[i] = p->c[i]; prm.inv_sin[i] = p->inv_sin[i]; prm.wp[i] = p->wp[i];
        const float ratio = p->c[0] != 0.f ? p->c[i] / p->c[0] : 0.f;   // the kernel's Sigma_t table carries c[0]
        uint32_t bits;
        memcpy(&bits, &ratio, 4);
        prm.c2[i] = (unsigned long long)bits | ((unsigned long long)bits << 32);
    }
    prm.magic_per_row = ndk::fastdiv_magic((uint32_t)((c.sp.NCq > 0 ? c.sp.NCq : c.sp.NC) * (d.Gs / 4)));
    prm.magic_nq = ndk::fastdiv_magic((uint32_t)(d.Gs / 4));
    prm.magic_np = ndk::fastdiv_magic((uint32_t)(d.Gs / 2));
    prm.phase = p->phase;
    prm.x_cap = c.x_cap; prm.off_x = c.off_x; prm.off_w = c.off_w;
    if (p->cmfd_sweep) cmfd_fill_sweep_params(p->cmfd_sweep, &prm);
    prm.off_q2 = c.off_q2; prm.off_dbuf2 = c.off_dbuf2;
    if (p->p1_sweep) p1_fill_sweep_params(p->p1_sweep, &prm);
    ND_CUDA(cudaMemsetAsync(p->counter, 0, sizeof(int), st));
    switch (d.P) {
    case 1: return launch_swath_p<1>(p, prm, st);
    case 2: return launch_swath_p<2>(p, prm, st);
    case 3: return launch_swath_p<3>(p, prm, st);
    default: return launch_swath_p<4>(p, prm, st);
    }
}

template <int P>
nd_status launch_sweep_p(nd_problem* p, const ndk::SweepParams& prm, cudaStream_t st)
{
    const Dims& d = p->d;
    const int block = 256, wpb = block / 32;
    const int64_t pairs = 2 * (int64_t)d.T;
    const int grid = grid_for(pairs * 32, block, 16 * p->n_sm);
    (void)wpb;
    if (p->opt.exp_mode == ND_EXP_EXPM1)
        ndk::k_sweep_atomic<P, 1><<<grid, block, 0, st>>>(prm);
    else
        ndk::k_sweep_atomic<P, 0><<<grid, block, 0, st>>>(prm);
    ND_LAUNCH_CHECK(p);
    return ND_OK;
}

// A5: source update over material-grouped chunks
constexpr size_t kSourceSmemMax = 100 * 1024;

nd_status launch_source(nd_problem* p, const ndk::SourceParams& sp, cudaStream_t st)
{
    const Dims& d = p->d;
    ndk::SourceChunkParams cp{};
    cp.base = sp; cp.src_region = p->src_region; cp.chunks = p->src_chunks; cp.n_chunks = p->n_src_chunks;
    cp.chunk_regions = p->src_chunk_regions;
    const int block = 256;
    const int Gp = (d.G + 1) / 2 * 2;
    const size_t smem = sizeof(double) * (2 * (size_t)p->src_chunk_regions * Gp + ((p->src_chunk_regions + 1) & ~1));
    const int grid = p->n_src_chunks < 8 * p->n_sm ? (p->n_src_chunks > 0 ? p->n_src_chunks : 1) : 8 * p->n_sm;
    // two phi tiles (<= 64 KB + the fission sums, by the cap on the chunk size) and, when it still fits 100 KB, the scattering
    // matrix of the chunk's material beside them (two blocks per SM: the kernel takes 128 registers)
    const size_t smem_ss = smem + sizeof(double) * (size_t)d.G * Gp;
    if (!p->source_attr_set) {   // the attribute belongs to the kernel, not to the problem: every problem sets the same value
        ND_CUDA(cudaFuncSetAttribute(ndk::k_source_tiled<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSourceSmemMax));
        ND_CUDA(cudaFuncSetAttribute(ndk::k_source_tiled<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSourceSmemMax));
        p->source_attr_set = true;
    }
    if (smem_ss <= kSourceSmemMax) {
        ndk::k_source_tiled<true><<<grid, block, smem_ss, st>>>(cp);
    } else {
        ndk::k_source_tiled<false><<<grid, block, smem, st>>>(cp);
    }
    ND_LAUNCH_CHECK(p);
    return ND_OK;
}

// A2 + A3: sweep with the current q/tally, then advance the boundary flux through the link table.  balance: also sum what
// entered and left through the track ends (k_boundary_balance, between the sweep and the swap) into p->partial_b.
nd_status launch_sweep(nd_problem* p, const double* scale_div, cudaStream_t st, bool balance = false)
{
    const Dims& d = p->d;
    ndk::SweepParams prm{};
    prm.seg_rm = p->seg_rm; prm.seg_len = p->seg_len; prm.trk_off = p->trk_off; prm.trk_w = p->trk_w;
    prm.q = p->q; prm.sigt = p->sigt_f; prm.tally = p->tally;
    prm.psi_in = p->psi_in; prm.psi_out = p->psi_out; prm.scale_div = scale_div;
    prm.T = d.T; prm.G = d.G; prm.Gs = d.Gs;
    for (int i = 0; i < ndk::kMaxPolar; ++i) { prm.c[i] = p->c[i]; prm.inv_sin[i] = p->inv_sin[i]; prm.wp[i] = p->wp[i]; }
    EventPair* ev = nullptr;
    if (p->profile) {
        if (p->ev_used == p->ev_pool.size()) {
            EventPair e{};
            ND_CUDA(cudaEventCreate(&e.a));
            ND_CUDA(cudaEventCreate(&e.b));
            p->ev_pool.push_back(e);
        }
        ev = &p->ev_pool[p->ev_used++];
        ND_CUDA(cudaEventRecord(ev->a, st));
    }
    nd_status rc;
    if (is_swath(p->sweep_kernel)) {
        rc = launch_swath(p, scale_div, st);
    } else {
        switch (d.P) {
        case 1: rc = launch_sweep_p<1>(p, prm, st); break;
        case 2: rc = launch_sweep_p<2>(p, prm, st); break;
        case 3: rc = launch_sweep_p<3>(p, prm, st); break;
        default: rc = launch_sweep_p<4>(p, prm, st); break;
        }
    }
    if (rc != ND_OK) return rc;
    if (ev) ND_CUDA(cudaEventRecord(ev->b, st));
    const int PG = d.P * d.Gs;
    const int64_t n = 2 * (int64_t)d.T * PG;
    if (balance) {
        ndk::k_boundary_balance<<<grid_for(n, 256, kReduceBlocks), 256, 0, st>>>(p->psi_in, p->psi_out, p->trk_w, p->exit_vac, scale_div,
                                                                             p->partial_b, 2 * (int64_t)d.T, d.P, d.G, d.Gs, p->wp[0],
                                                                             p->wp[1], p->wp[2], p->wp[3]);
        ND_LAUNCH_CHECK(p);
    }
    if (p->cmfd_sweep) {   // C-3: the chain-end terms need what entered and what left, before the swap overwrites the former
        const nd_status rcc = cmfd_end_currents(p->cmfd_sweep, scale_div, st);
        if (rcc != ND_OK) return rcc;
    }
    ndk::k_link_swap<<<grid_for(n, 256, 8 * p->n_sm), 256, 0, st>>>(p->psi_out, p->psi_in, p->link_src, 2 * (int64_t)d.T, PG);
    ND_LAUNCH_CHECK(p);
    if (p->reduce_fn) {   // NEXT-2: the shards' tallies are summed before any of them forms its flux
        if (p->reduce_fn(p->reduce_user, p->tally, (int64_t)d.R * d.Gs, st) != 0)
            return nd_fail(ND_ERR_STATE, "the tally reducer (nd_tally_reducer_set) reported a failure");
    }
    return ND_OK;
}

nd_status launch_finalise(nd_problem* p, const double* Q, const double* phi_old, const double* f_ptr, double* phi_out,
                          int* grid_out, cudaStream_t st)
{
    const Dims& d = p->d;
    ndk::FinaliseParams fp{};
    fp.Q = Q; fp.tally = p->tally; fp.reg_mat = p->reg_mat; fp.sigt = p->sigt; fp.nusf = p->nusf; fp.vol = p->vol;
    fp.phi_old = phi_old; fp.f_ptr = f_ptr; fp.phi_new = phi_out; fp.partial = p->partial;
    fp.R = d.R; fp.G = d.G; fp.Gs = d.Gs;
    const int grid = grid_for((int64_t)d.R * d.G, 256, kReduceBlocks);
    const int MG = d.M * d.G;
    if (MG <= ndk::kFinTab) ndk::k_finalise<true><<<grid, 256, 0, st>>>(fp, MG);
    else ndk::k_finalise<false><<<grid, 256, 0, st>>>(fp, MG);
    ND_LAUNCH_CHECK(p);
    *grid_out = grid;
    return ND_OK;
}

nd_status reset_state(nd_problem* p, cudaStream_t st)
{
    const Dims& d = p->d;
    nd_status rc;
    if ((rc = launch_fill_f64(p, p->phi_cur, 1.0, (int64_t)d.R * d.G, st)) != ND_OK) return rc;
    if ((rc = launch_fill_f32(p, p->psi_in, 0.f, (int64_t)d.T * 2 * d.P * d.Gs, st)) != ND_OK) return rc;
    const double sc[ndk::SC_COUNT] = {1.0, 0.0, 1.0, 0.0, 1.0, 0.0, 0.0, 0.0};
    ND_CUDA(cudaMemcpyAsync(p->scalars, sc, sizeof sc, cudaMemcpyHostToDevice, st));
    ND_CUDA(cudaStreamSynchronize(st)); // sc is a stack array
    return launch_fission_rate(p, p->phi_cur, nullptr, st);
}

} // namespace

// ------------------------------------------------------------------------------------------------
// create / destroy
// ------------------------------------------------------------------------------------------------
extern "C" nd_status nd_workspace_bytes(const nd_problem_desc* desc, const nd_options* opts, size_t* device_bytes)
{
    if (!device_bytes) return nd_fail(ND_ERR_NULL, "device_bytes is NULL");
    Dims d{};
    nd_status rc = basic_dims(desc, d);
    if (rc != ND_OK) return rc;
    nd_options opt{};
    if (opts) opt = *opts;
    SwathConfig sc;
    if (is_swath(opt.sweep_kernel) || opt.sweep_kernel == ND_SWEEP_AUTO) sc = make_swath_config(d, opt);
    *device_bytes = make_layout(d, kMaxStats, sc, select_kernel(desc, opt, sc), opt.cmfd_stream != 0, desc->seg_on_device != 0).total;
    return ND_OK;
}

extern "C" nd_status nd_problem_create(const nd_problem_desc* desc, const nd_options* opts, void* device_workspace,
                                       size_t device_bytes, void* cuda_stream, nd_problem** out)
{
    if (!desc || !out || !device_workspace) return nd_fail(ND_ERR_NULL, "nd_problem_create: NULL argument");
    if (!desc->region_material || !desc->sigma_t || !desc->sigma_s || !desc->nu_sigma_f || !desc->chi || !desc->polar_sin ||
        !desc->polar_weight || !desc->track_seg_offset || !desc->seg_region || !desc->seg_length || !desc->track_weight ||
        !desc->link)
        return nd_fail(ND_ERR_NULL, "nd_problem_create: a descriptor array is NULL");
    Dims d{};
    nd_status rc = basic_dims(desc, d);
    if (rc != ND_OK) return rc;
    nd_options opt{};
    if (opts) opt = *opts;
    if (opt.item_order < 0 || opt.item_order > 1) return nd_fail(ND_ERR_INVALID, "nd_options.item_order must be 0 or 1");
    for (int i = 0; i < 3; ++i)
        if (opt.reserved[i] != 0) return nd_fail(ND_ERR_INVALID, "nd_options.reserved must be zero");
    if (opt.cmfd_stream < 0 || opt.cmfd_stream > 1) return nd_fail(ND_ERR_INVALID, "nd_options.cmfd_stream must be 0 or 1");
    if (opt.p1_stream < 0 || opt.p1_stream > 1) return nd_fail(ND_ERR_INVALID, "nd_options.p1_stream must be 0 or 1");
    if (opt.p1_stream && opt.cmfd_stream) return nd_fail(ND_ERR_INVALID, "nd_options: p1_stream and cmfd_stream exclude each other");
    if (opt.exp_mode != ND_EXP_FAST && opt.exp_mode != ND_EXP_EXPM1) return nd_fail(ND_ERR_INVALID, "unknown exp_mode");
    if (opt.sweep_kernel != ND_SWEEP_AUTO && opt.sweep_kernel != ND_SWEEP_ATOMIC && opt.sweep_kernel != ND_SWEEP_SWATH)
        return nd_fail(ND_ERR_INVALID, "unknown sweep_kernel");
    if (opt.window_regions < 0 || opt.block_warps < 0 || opt.tile_segments < 0 || opt.delta_buffers < 0 ||
        opt.delta_buffers > 2 || opt.blocks_per_sm < 0 || opt.tile_lag < -1 || opt.q_copies < 0 || opt.graph_mode < 0 || opt.graph_mode > 1)
        return nd_fail(ND_ERR_INVALID, "nd_options: tuning fields must be >= 0 (delta_buffers 0, 1 or 2)");
    if ((desc->track_azim == nullptr) != (desc->track_ends == nullptr))
        return nd_fail(ND_ERR_INVALID, "track_azim and track_ends must both be set or both be NULL");
    SwathConfig sc;
    if (is_swath(opt.sweep_kernel) || opt.sweep_kernel == ND_SWEEP_AUTO) sc = make_swath_config(d, opt);
    const int kernel = select_kernel(desc, opt, sc);
    const bool seg_dev = desc->seg_on_device != 0;
    if (desc->seg_on_device < 0 || desc->seg_on_device > 1 || desc->reserved != 0)
        return nd_fail(ND_ERR_INVALID, "nd_problem_desc.seg_on_device must be 0 or 1, reserved 0");
    if (seg_dev && !desc->track_azim)
        return nd_fail(ND_ERR_INVALID, "device-resident segments need the track geometry (track_azim, track_ends)");
    const Layout L = make_layout(d, kMaxStats, sc, kernel, opt.cmfd_stream != 0, seg_dev);
    if (reinterpret_cast<uintptr_t>(device_workspace) % kAlign != 0) return nd_fail(ND_ERR_WORKSPACE, "workspace must be 256-byte aligned");
    if (device_bytes < L.total) return nd_fail(ND_ERR_WORKSPACE, "workspace smaller than nd_workspace_bytes");

    // ---- validation (host) ----
    for (int r = 0; r < d.R; ++r)
        if (desc->region_material[r] < 0 || desc->region_material[r] >= d.M) return nd_fail(ND_ERR_RANGE, "region_material out of range");
    for (size_t i = 0; i < (size_t)d.M * d.G; ++i) {
        if (!(desc->sigma_t[i] > 0.0) || !std::isfinite(desc->sigma_t[i])) return nd_fail(ND_ERR_INVALID, "sigma_t must be finite and > 0");
        if (!(desc->nu_sigma_f[i] >= 0.0) || !std::isfinite(desc->nu_sigma_f[i])) return nd_fail(ND_ERR_INVALID, "nu_sigma_f must be finite and >= 0");
        if (!(desc->chi[i] >= 0.0) || !std::isfinite(desc->chi[i])) return nd_fail(ND_ERR_INVALID, "chi must be finite and >= 0");
    }
    for (size_t i = 0; i < (size_t)d.M * d.G * d.G; ++i)
        if (!std::isfinite(desc->sigma_s[i])) return nd_fail(ND_ERR_INVALID, "sigma_s must be finite");
    double wsum = 0.0;
    for (int p = 0; p < d.P; ++p) {
        if (!(desc->polar_sin[p] > 0.0) || !(desc->polar_sin[p] <= 1.0)) return nd_fail(ND_ERR_INVALID, "polar_sin must lie in (0,1]");
        if (!(desc->polar_weight[p] > 0.0)) return nd_fail(ND_ERR_INVALID, "polar_weight must be > 0");
        wsum += desc->polar_weight[p];
    }
    if (std::fabs(wsum - 1.0) > 1e-9) return nd_fail(ND_ERR_INVALID, "polar_weight must sum to 1");
    for (int t = 0; t < d.T; ++t)
        if (!(desc->track_weight[t] > 0.0) || !std::isfinite(desc->track_weight[t])) return nd_fail(ND_ERR_INVALID, "track_weight must be finite and > 0");
    if (!seg_dev) {   // 5e8 segments at config 5: all host threads (device-resident segments: k_seg_validate below)
        int bad_region = 0, bad_length = 0;
#pragma omp parallel for schedule(static) reduction(| : bad_region, bad_length)
        for (int64_t k = 0; k < d.S; ++k) {
            bad_region |= desc->seg_region[k] < 0 || desc->seg_region[k] >= d.R;
            bad_length |= !(desc->seg_length[k] > 0.0) || !std::isfinite(desc->seg_length[k]);
        }
        if (bad_region) return nd_fail(ND_ERR_RANGE, "seg_region out of range");
        if (bad_length) return nd_fail(ND_ERR_INVALID, "seg_length must be finite and > 0");
    }
    std::vector<int32_t> link_src;
    std::vector<uint8_t> h_exit_vac;
    nd_problem* p = nullptr;
    std::vector<uint32_t> h_rm;
    std::vector<float> h_len;
    std::vector<int64_t> h_off;
    try {
        link_src.assign(2 * (size_t)d.T, -1);
        h_exit_vac.assign(2 * (size_t)d.T, 0);
        for (int64_t e = 0; e < 2 * (int64_t)d.T; ++e) {
            const int32_t lk = desc->link[e];
            if (lk == -1) { h_exit_vac[(size_t)e] = 1; continue; }
            if (lk < 0 || lk >= 2 * d.T) return nd_fail(ND_ERR_RANGE, "link out of range");
            if (link_src[lk] != -1) return nd_fail(ND_ERR_INVALID, "two track ends link to the same entry");
            link_src[lk] = (int32_t)e;
        }
        p = new nd_problem();
        p->d = d; p->opt = opt; p->L = L; p->ws = static_cast<char*>(device_workspace);
        // ---- A1: pack the segment stream (SoA, every track run padded to a multiple of 4 = 16 bytes) ----
        const bool soa = kernel == ND_SWEEP_ATOMIC;
        p->has_soa = soa;
        h_rm.assign(soa ? (size_t)d.Spad : 4, 0u);
        h_len.assign(soa ? (size_t)d.Spad : 4, 0.f);
        h_off.resize((size_t)d.T + 1);
        p->h_vol.assign((size_t)d.R, 0.0);
        p->h_entry_region.assign(2 * (size_t)d.T, -1);
        int64_t o = 0;
        for (int t = 0; t < d.T; ++t) {                   // padded offsets and the entry regions of both directions
            h_off[t] = o;
            const int64_t k0 = desc->track_seg_offset[t], k1 = desc->track_seg_offset[t + 1];
            if (k1 > k0 && !seg_dev) {
                p->h_entry_region[2 * (size_t)t] = desc->seg_region[k0];
                p->h_entry_region[2 * (size_t)t + 1] = desc->seg_region[k1 - 1];
            }
            o += (k1 - k0 + 3) / 4 * 4;
        }
        h_off[d.T] = o;
        if (soa && !seg_dev) {
#pragma omp parallel for schedule(dynamic, 256)
            for (int t = 0; t < d.T; ++t) {
                int64_t at = h_off[t];
                uint32_t last = 0;
                for (int64_t k = desc->track_seg_offset[t]; k < desc->track_seg_offset[t + 1]; ++k, ++at) {
                    const int32_t r = desc->seg_region[k];
                    last = ndk::pack_rm((uint32_t)r, (uint32_t)desc->region_material[r]);
                    h_rm[at] = last;
                    h_len[at] = (float)desc->seg_length[k];
                }
                for (; at < h_off[t + 1]; ++at) { h_rm[at] = last; h_len[at] = 0.f; }   // zero-length segments are exact no-ops
            }
        }
        if (!desc->region_volume && !seg_dev) {
            // O-5: A~_r = sum 2 omega_a delta_a s.  Small problems: one thread, canonical (track, segment) order.  Large ones:
            // every thread sums a contiguous range of tracks into its own array, the arrays are added in thread order.
            const int nth = d.S > (1 << 22) ? std::max(1, std::min(omp_get_max_threads(), 16)) : 1;
            std::vector<double> part((size_t)d.R * (nth > 1 ? nth : 0), 0.0);
#pragma omp parallel num_threads(nth)
            {
                const int me = omp_get_thread_num();
                double* vol = nth > 1 ? part.data() + (size_t)d.R * me : p->h_vol.data();
                const int t0 = (int)((int64_t)d.T * me / nth), t1 = (int)((int64_t)d.T * (me + 1) / nth);
                for (int t = t0; t < t1; ++t) {
                    const double w2 = 2.0 * desc->track_weight[t];
                    for (int64_t k = desc->track_seg_offset[t]; k < desc->track_seg_offset[t + 1]; ++k)
                        vol[desc->seg_region[k]] += w2 * desc->seg_length[k];
                }
            }
            for (int th = 0; th < (nth > 1 ? nth : 0); ++th)
                for (int r = 0; r < d.R; ++r) p->h_vol[(size_t)r] += part[(size_t)d.R * th + r];
        }
        if (desc->region_volume) {   // a shard of an angle-pair partition: the areas of the whole laydown (nd_tracks_shard)
            for (int r = 0; r < d.R; ++r) {
                if (!(desc->region_volume[r] >= 0.0) || !std::isfinite(desc->region_volume[r])) {
                    delete p;
                    return nd_fail(ND_ERR_INVALID, "region_volume must be finite and >= 0");
                }
                p->h_vol[(size_t)r] = desc->region_volume[r];
            }
        }
    } catch (const std::bad_alloc&) {
        delete p;
        return nd_fail(ND_ERR_NOMEM, "nd_problem_create: out of host memory");
    }
    // ---- A1 (fast path): swath/tile chunk stream of k_sweep_swath ----
    NdSwathSet swaths;
    const bool want_swath = is_swath(kernel);
    const bool tiled = want_swath;
    if (want_swath && !seg_dev) {
        rc = nd_build_swaths(desc, desc->track_azim, desc->track_ends, sc.sp, 0, &swaths);
        if (rc != ND_OK) { delete p; return rc; }
        if (swaths.blob.size() > sc.max_blob || swaths.n_tiles + 1 > sc.max_tiles || swaths.n_swaths > sc.max_swaths ||
            swaths.max_head_bytes > sc.head_cap || swaths.max_rec_bytes > sc.rec_cap) {
            delete p;
            return nd_fail(ND_ERR_WORKSPACE, "internal: swath stream larger than its workspace bound");
        }
    }
    p->sc = sc;
    char* ws = p->ws;
    p->seg_rm = (uint32_t*)(ws + L.seg_rm); p->seg_len = (float*)(ws + L.seg_len); p->trk_off = (int64_t*)(ws + L.trk_off);
    p->trk_w = (float*)(ws + L.trk_w); p->link_src = (int32_t*)(ws + L.link_src);
    p->psi_in = (float*)(ws + L.psi_a); p->psi_out = (float*)(ws + L.psi_b);
    p->q = (float*)(ws + L.q); p->tally = (double*)(ws + L.tally);
    p->phi_cur = (double*)(ws + L.phi_a); p->phi_new = (double*)(ws + L.phi_b); p->Q = (double*)(ws + L.Q);
    p->reg_mat = (int32_t*)(ws + L.reg_mat); p->vol = (double*)(ws + L.vol);
    p->sigt = (double*)(ws + L.sigt); p->sigsT = (double*)(ws + L.sigsT); p->nusf = (double*)(ws + L.nusf);
    p->chi = (double*)(ws + L.chi); p->sigt_f = (float*)(ws + L.sigt_f);
    p->scalars = (double*)(ws + L.scalars); p->partial = (double*)(ws + L.partial); p->stats = (double*)(ws + L.stats);
    p->partial_b = (double*)(ws + L.partial_b); p->exit_vac = (uint8_t*)(ws + L.exit_vac);
    p->phase = (unsigned long long*)(ws + L.phase);
    p->src_region = (int32_t*)(ws + L.src_region); p->src_chunks = (int4*)(ws + L.src_chunks);
    if (tiled) {
        p->blob = (uint8_t*)(ws + L.blob); p->tile_ref = (uint2*)(ws + L.tile_chunk); p->swath_tile0 = (int64_t*)(ws + L.swath_tile0);
        p->swath_track = (int32_t*)(ws + L.swath_track); p->items = (int4*)(ws + L.items); p->counter = (int*)(ws + L.counter);
    }

    cudaStream_t st = as_stream(cuda_stream);
    auto fail = [&](nd_status s) { delete p; return s; };
    int dev = 0;
    cudaError_t ce = cudaGetDevice(&dev);
    if (ce != cudaSuccess) { delete p; return nd_fail(ND_ERR_CUDA, cudaGetErrorString(ce)); }
    cudaDeviceProp prop{};
    ce = cudaGetDeviceProperties(&prop, dev);
    if (ce != cudaSuccess) { delete p; return nd_fail(ND_ERR_CUDA, cudaGetErrorString(ce)); }
    if (prop.major != 10) { delete p; return nd_fail(ND_ERR_CUDA, "libnd_moc.so holds sm_100a kernels only; the current device is not compute capability 10.x"); }
    p->n_sm = prop.multiProcessorCount;

    std::vector<float> h_w((size_t)d.T), h_sigt_f((size_t)d.M * d.Gs, 1.f);
    std::vector<double> h_sigsT((size_t)d.M * d.G * d.G);
    for (int t = 0; t < d.T; ++t) h_w[t] = (float)(ndk::kFourPi * desc->track_weight[t]);
    for (int m = 0; m < d.M; ++m)
        for (int g = 0; g < d.G; ++g) {
            h_sigt_f[(size_t)m * d.Gs + g] = (float)desc->sigma_t[(size_t)m * d.G + g];
            for (int gp = 0; gp < d.G; ++gp)
                h_sigsT[((size_t)m * d.G + gp) * d.G + g] = desc->sigma_s[((size_t)m * d.G + g) * d.G + gp];
        }
    for (int i = 0; i < d.P; ++i) {
        p->c[i] = (float)(-1.4426950408889634074 / desc->polar_sin[i]);
        p->inv_sin[i] = (float)(1.0 / desc->polar_sin[i]);
        p->wp[i] = (float)(desc->polar_weight[i] * desc->polar_sin[i]);
    }
    // A5: regions grouped by material into chunks of nsub * kSrcTile regions (k_source_tiled)
    std::vector<int32_t> h_src_region((size_t)d.R);
    std::vector<int4> h_src_chunks;
    {
        // k_source_tiled: thread = (sub, pair of groups), kSrcTile regions each; at most 64 subs (two phi tiles <= 64 KB)
        const int nsub = std::min(256 / ((d.G + 1) / 2), 64);
        p->src_chunk_regions = nsub * ndk::kSrcTile;
        std::vector<int64_t> count((size_t)d.M + 1, 0);
        for (int r = 0; r < d.R; ++r) ++count[desc->region_material[r] + 1];
        for (int m = 0; m < d.M; ++m) count[m + 1] += count[m];
        std::vector<int64_t> fill(count.begin(), count.end() - 1);
        for (int r = 0; r < d.R; ++r) h_src_region[(size_t)fill[desc->region_material[r]]++] = r;
        for (int m = 0; m < d.M; ++m)
            for (int64_t i = count[m]; i < count[m + 1]; i += p->src_chunk_regions) {
                const int n = (int)std::min<int64_t>(p->src_chunk_regions, count[m + 1] - i);
                h_src_chunks.push_back(make_int4((int)i, n, m, 0));
            }
        p->n_src_chunks = (int)h_src_chunks.size();
    }
    p->sweep_kernel = kernel;

#define ND_CUDA_P(call)                                                                                 \
    do {                                                                                                \
        cudaError_t e_ = (call);                                                                        \
        if (e_ != cudaSuccess) {                                                                        \
            char buf_[512];                                                                             \
            snprintf(buf_, sizeof buf_, "%s failed: %s", #call, cudaGetErrorString(e_));                \
            return fail(nd_fail(ND_ERR_CUDA, buf_));                                                    \
        }                                                                                               \
    } while (0)
    ND_CUDA_P(cudaMemsetAsync(ws, 0, tiled ? L.blob : L.total, st));
    if (want_swath && !seg_dev) {
        static_assert(sizeof(NdSwathItem) == sizeof(int4), "work item layout");
        p->n_items = (int)swaths.items.size();
        p->n_tiles = swaths.n_tiles; p->n_swaths = swaths.n_swaths; p->blob_bytes = swaths.blob.size();
        p->mean_regions_per_tile = swaths.mean_regions_per_tile;
        p->mean_segments_per_tile = swaths.mean_segments_per_tile;
        p->lockstep_efficiency = swaths.lockstep_efficiency;
        if (opt.cmfd_stream) {
            p->h_swath_track = swaths.swath_track;
            p->h_swath_tile0 = swaths.swath_tile0;
            p->h_slot_start.swap(swaths.slot_start);
        }
        ND_CUDA_P(cudaMemcpyAsync(p->blob, swaths.blob.data(), swaths.blob.size(), cudaMemcpyHostToDevice, st));
        static_assert(sizeof(NdSwathTileRef) == sizeof(uint2), "tile reference layout");
        ND_CUDA_P(cudaMemcpyAsync(p->tile_ref, swaths.tile_ref.data(), sizeof(NdSwathTileRef) * swaths.tile_ref.size(), cudaMemcpyHostToDevice, st));
        ND_CUDA_P(cudaMemcpyAsync(p->swath_tile0, swaths.swath_tile0.data(), sizeof(int64_t) * swaths.swath_tile0.size(), cudaMemcpyHostToDevice, st));
        ND_CUDA_P(cudaMemcpyAsync(p->swath_track, swaths.swath_track.data(), sizeof(int32_t) * swaths.swath_track.size(), cudaMemcpyHostToDevice, st));
        ND_CUDA_P(cudaMemcpyAsync(p->items, swaths.items.data(), sizeof(NdSwathItem) * swaths.items.size(), cudaMemcpyHostToDevice, st));
    }
    if (!seg_dev) {
        ND_CUDA_P(cudaMemcpyAsync(p->seg_rm, h_rm.data(), sizeof(uint32_t) * h_rm.size(), cudaMemcpyHostToDevice, st));
        ND_CUDA_P(cudaMemcpyAsync(p->seg_len, h_len.data(), sizeof(float) * h_len.size(), cudaMemcpyHostToDevice, st));
    }
    ND_CUDA_P(cudaMemcpyAsync(p->trk_off, h_off.data(), sizeof(int64_t) * h_off.size(), cudaMemcpyHostToDevice, st));
    ND_CUDA_P(cudaMemcpyAsync(p->trk_w, h_w.data(), sizeof(float) * h_w.size(), cudaMemcpyHostToDevice, st));
    ND_CUDA_P(cudaMemcpyAsync(p->link_src, link_src.data(), sizeof(int32_t) * link_src.size(), cudaMemcpyHostToDevice, st));
    ND_CUDA_P(cudaMemcpyAsync(p->exit_vac, h_exit_vac.data(), h_exit_vac.size(), cudaMemcpyHostToDevice, st));
    ND_CUDA_P(cudaMemcpyAsync(p->reg_mat, desc->region_material, sizeof(int32_t) * (size_t)d.R, cudaMemcpyHostToDevice, st));
    ND_CUDA_P(cudaMemcpyAsync(p->vol, p->h_vol.data(), sizeof(double) * (size_t)d.R, cudaMemcpyHostToDevice, st));
    ND_CUDA_P(cudaMemcpyAsync(p->sigt, desc->sigma_t, sizeof(double) * (size_t)d.M * d.G, cudaMemcpyHostToDevice, st));
    ND_CUDA_P(cudaMemcpyAsync(p->sigsT, h_sigsT.data(), sizeof(double) * h_sigsT.size(), cudaMemcpyHostToDevice, st));
    ND_CUDA_P(cudaMemcpyAsync(p->nusf, desc->nu_sigma_f, sizeof(double) * (size_t)d.M * d.G, cudaMemcpyHostToDevice, st));
    ND_CUDA_P(cudaMemcpyAsync(p->chi, desc->chi, sizeof(double) * (size_t)d.M * d.G, cudaMemcpyHostToDevice, st));
    ND_CUDA_P(cudaMemcpyAsync(p->sigt_f, h_sigt_f.data(), sizeof(float) * h_sigt_f.size(), cudaMemcpyHostToDevice, st));
    ND_CUDA_P(cudaMemcpyAsync(p->src_region, h_src_region.data(), sizeof(int32_t) * h_src_region.size(), cudaMemcpyHostToDevice, st));
    ND_CUDA_P(cudaMemcpyAsync(p->src_chunks, h_src_chunks.data(), sizeof(int4) * h_src_chunks.size(), cudaMemcpyHostToDevice, st));
    if (seg_dev) {
        // ---- the segment passes on the GPU: validation first (everything after it indexes with the region ids) ----
        char* sx = ws + L.setup;
        int* d_flags = (int*)sx; sx += kAlign;
        int64_t* d_off = (int64_t*)sx; sx += (8 * ((size_t)d.T + 1) + kAlign - 1) / kAlign * kAlign;
        double* d_w2 = (double*)sx; sx += (8 * (size_t)d.T + kAlign - 1) / kAlign * kAlign;
        int32_t* d_entry = (int32_t*)sx; sx += (8 * (size_t)d.T + kAlign - 1) / kAlign * kAlign;
        std::vector<double> h_w2((size_t)d.T);
        for (int t = 0; t < d.T; ++t) h_w2[(size_t)t] = 2.0 * desc->track_weight[t];
        ND_CUDA_P(cudaMemcpyAsync(d_off, desc->track_seg_offset, 8 * ((size_t)d.T + 1), cudaMemcpyHostToDevice, st));
        ND_CUDA_P(cudaMemcpyAsync(d_w2, h_w2.data(), 8 * (size_t)d.T, cudaMemcpyHostToDevice, st));
        ndk::k_seg_validate<<<grid_for(d.S, 256, 16 * p->n_sm), 256, 0, st>>>(desc->seg_region, desc->seg_length, d.S, d.R, d_flags);
        ND_CUDA_P(cudaGetLastError());
        int h_flags = 0;
        ND_CUDA_P(cudaMemcpyAsync(&h_flags, d_flags, sizeof(int), cudaMemcpyDeviceToHost, st));
        ND_CUDA_P(cudaStreamSynchronize(st));
        if (h_flags & 1) return fail(nd_fail(ND_ERR_RANGE, "seg_region out of range"));
        if (h_flags & 2) return fail(nd_fail(ND_ERR_INVALID, "seg_length must be finite and > 0"));
        const int tb = (d.T + 127) / 128;
        ndk::k_entry_regions<<<(d.T + 255) / 256, 256, 0, st>>>(d_off, desc->seg_region, d.T, d_entry);
        ND_CUDA_P(cudaGetLastError());
        ND_CUDA_P(cudaMemcpyAsync(p->h_entry_region.data(), d_entry, 8 * (size_t)d.T, cudaMemcpyDeviceToHost, st));
        if (p->has_soa) {
            ndk::k_pack_soa<<<tb, 128, 0, st>>>(d_off, p->trk_off, desc->seg_region, desc->seg_length, p->reg_mat, d.T, p->seg_rm, p->seg_len);
            ND_CUDA_P(cudaGetLastError());
        }
        if (!desc->region_volume) {   // p->vol holds the zeros uploaded above
            ndk::k_track_volume<<<tb, 128, 0, st>>>(d_off, desc->seg_region, desc->seg_length, d_w2, d.T, p->vol);
            ND_CUDA_P(cudaGetLastError());
            ND_CUDA_P(cudaMemcpyAsync(p->h_vol.data(), p->vol, 8 * (size_t)d.R, cudaMemcpyDeviceToHost, st));
        }
        if (want_swath) {
            NdSwathDeviceTargets tg;
            tg.blob = p->blob; tg.blob_cap = sc.max_blob; tg.tile_ref = p->tile_ref; tg.tile_cap = sc.max_tiles;
            tg.swath_tile0 = p->swath_tile0; tg.max_swaths = sc.max_swaths; tg.swath_track = p->swath_track; tg.items = p->items;
            tg.slot_start = L.slot_start_bytes ? (uint16_t*)(ws + L.slot_start) : nullptr; tg.slot_start_cap = L.slot_start_bytes;
            tg.scratch = sx;
            rc = nd_build_swaths_device(desc, p->reg_mat, sc.sp, tg, st, &swaths);
            if (rc != ND_OK) return fail(rc);
            if (swaths.max_head_bytes > sc.head_cap || swaths.max_rec_bytes > sc.rec_cap)
                return fail(nd_fail(ND_ERR_WORKSPACE, "internal: swath stream larger than its workspace bound"));
            p->n_items = (int)swaths.items.size();
            p->n_tiles = swaths.n_tiles; p->n_swaths = swaths.n_swaths; p->blob_bytes = swaths.blob_bytes_device;
            p->stream_on_device = true;
            p->mean_regions_per_tile = swaths.mean_regions_per_tile;
            p->mean_segments_per_tile = swaths.mean_segments_per_tile;
            p->lockstep_efficiency = swaths.lockstep_efficiency;
            if (opt.cmfd_stream) {
                p->h_swath_track = swaths.swath_track;
                p->h_swath_tile0 = swaths.swath_tile0;
                p->h_slot_start.swap(swaths.slot_start);
            }
        }
    }
    ND_CUDA_P(cudaStreamSynchronize(st));
#undef ND_CUDA_P
    rc = reset_state(p, st);
    if (rc != ND_OK) return fail(rc);
    ce = cudaStreamSynchronize(st);
    if (ce != cudaSuccess) { delete p; return nd_fail(ND_ERR_CUDA, cudaGetErrorString(ce)); }
    *out = p;
    return ND_OK;
}

extern "C" nd_status nd_problem_destroy(nd_problem* p)
{
    if (!p) return ND_OK;
    for (auto& e : p->ev_pool) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
    if (p->iter_graph) cudaGraphExecDestroy(p->iter_graph);
    if (p->cap_stream) cudaStreamDestroy(p->cap_stream);
    delete p;
    return ND_OK;
}

// ------------------------------------------------------------------------------------------------
// compute entry points
// ------------------------------------------------------------------------------------------------
extern "C" nd_status nd_transport_sweep(nd_problem* p, const double* d_Q, double* d_phi_out, void* cuda_stream)
{
    if (!p || !d_Q || !d_phi_out) return nd_fail(ND_ERR_NULL, "nd_transport_sweep: NULL argument");
    const Dims& d = p->d;
    cudaStream_t st = as_stream(cuda_stream);
    const int64_t n = (int64_t)d.R * d.Gs;
    ndk::k_reduced_source<<<grid_for(n, 256, 8 * p->n_sm), 256, 0, st>>>(d_Q, p->reg_mat, p->sigt, p->q, p->tally, d.R, d.G, d.Gs);
    ND_LAUNCH_CHECK(p);
    nd_status rc = launch_sweep(p, p->scalars + ndk::SC_ONE, st);
    if (rc != ND_OK) return rc;
    int grid = 0;
    return launch_finalise(p, d_Q, nullptr, nullptr, d_phi_out, &grid, st);
}

extern "C" nd_status nd_source_update(nd_problem* p, const double* d_phi, double k_eff, double* d_Q_out,
                                      double* d_fission_rate_out, void* cuda_stream)
{
    if (!p || !d_phi || !d_Q_out) return nd_fail(ND_ERR_NULL, "nd_source_update: NULL argument");
    if (!(k_eff > 0.0)) return nd_fail(ND_ERR_INVALID, "nd_source_update: k_eff must be > 0");
    const Dims& d = p->d;
    cudaStream_t st = as_stream(cuda_stream);
    ndk::SourceParams sp{};
    sp.phi = d_phi; sp.reg_mat = p->reg_mat; sp.sigt = p->sigt; sp.sigsT = p->sigsT; sp.nusf = p->nusf; sp.chi = p->chi;
    sp.k_ptr = nullptr; sp.f_ptr = nullptr; sp.k_val = k_eff; sp.Q = d_Q_out; sp.q = nullptr; sp.tally = nullptr;
    sp.R = d.R; sp.G = d.G; sp.Gs = d.Gs;
    nd_status rc_src = launch_source(p, sp, st);
    if (rc_src != ND_OK) return rc_src;
    if (d_fission_rate_out) {
        // uses a private scalar slot so the problem's own F (power-iteration state) is not disturbed
        const int grid = grid_for((int64_t)d.R * d.G, 256, kReduceBlocks);
        ndk::k_fission_partial<<<grid, 256, 0, st>>>(d_phi, p->reg_mat, p->nusf, p->vol, p->partial, d.R, d.G);
        ND_LAUNCH_CHECK(p);
        ndk::k_reduce_final<<<1, 256, 0, st>>>(p->partial, grid, p->scalars + 4, 0, nullptr, nullptr, 0); // writes scalars[4+SC_F]
        ND_LAUNCH_CHECK(p);
        ND_CUDA(cudaMemcpyAsync(d_fission_rate_out, p->scalars + 4 + ndk::SC_F, sizeof(double), cudaMemcpyDeviceToDevice, st));
    }
    return ND_OK;
}

extern "C" nd_status nd_power_iteration(nd_problem* p, int32_t max_iters, double tol_k, double tol_phi, double* k_eff_out,
                                        double* d_phi_out, int32_t* iters_done, nd_iter_stats* stats, void* cuda_stream)
{
    if (!p || !k_eff_out) return nd_fail(ND_ERR_NULL, "nd_power_iteration: NULL argument");
    if (max_iters < 0) return nd_fail(ND_ERR_INVALID, "nd_power_iteration: max_iters must be >= 0");
    const Dims& d = p->d;
    cudaStream_t st = as_stream(cuda_stream);
    const bool use_tol = tol_k > 0.0 || tol_phi > 0.0;
    const bool sync_each = use_tol;
    ndk::SourceParams sp{};
    sp.reg_mat = p->reg_mat; sp.sigt = p->sigt; sp.sigsT = p->sigsT; sp.nusf = p->nusf; sp.chi = p->chi;
    sp.k_ptr = p->scalars + ndk::SC_K; sp.f_ptr = p->scalars + ndk::SC_F; sp.k_val = 1.0;
    sp.Q = p->Q; sp.q = p->q; sp.tally = p->tally; sp.R = d.R; sp.G = d.G; sp.Gs = d.Gs;
    int it = 0;
    bool converged = !use_tol;
    auto one_iteration = [&](double* slot, cudaStream_t st) -> nd_status {
        sp.phi = p->phi_cur;
        nd_status rc = launch_source(p, sp, st);
        if (rc != ND_OK) return rc;
        // leakage and the balance residual are only formed for stats, and only when the tally is this problem's own
        const bool balance = slot != nullptr && stats != nullptr && !p->reduce_fn;
        rc = launch_sweep(p, p->scalars + ndk::SC_F, st, balance);
        if (rc != ND_OK) return rc;
        int grid = 0;
        rc = launch_finalise(p, p->Q, p->phi_cur, p->scalars + ndk::SC_F, p->phi_new, &grid, st);
        if (rc != ND_OK) return rc;
        const int grid_b = grid_for(2 * (int64_t)d.T * d.P * d.Gs, 256, kReduceBlocks);
        ndk::k_reduce_final<<<1, 256, 0, st>>>(p->partial, grid, p->scalars, 1, slot, balance ? p->partial_b : nullptr, grid_b);
        ND_LAUNCH_CHECK(p);
        std::swap(p->phi_cur, p->phi_new);
        return ND_OK;
    };
    // Fixed-count calls replay a CUDA graph of TWO iterations (after two, phi_cur is back in the buffer it started in, so
    // one graph serves every pair); an odd iteration and anything with tolerances, stats or profiling is launched plainly.
    const bool graph_ok = !use_tol && !stats && !p->profile && !p->phase_profile && p->opt.graph_mode == 0 && max_iters >= 4 &&
                          !p->reduce_fn;   // a host callback cannot be replayed from a graph
    if (graph_ok) {
        if (p->iter_graph && p->iter_graph_phi != p->phi_cur) {   // an odd number of plain iterations since the capture
            nd_status rc = one_iteration(nullptr, st);
            if (rc != ND_OK) return rc;
            ++it;
        }
        if (!p->iter_graph) {
            const int64_t before = p->kernels_launched;
            const double* phi0 = p->phi_cur;
            cudaGraph_t graph = nullptr;
            // captured on a stream of our own: the caller's may be the legacy default stream, which cannot capture
            if (!p->cap_stream) ND_CUDA(cudaStreamCreateWithFlags(&p->cap_stream, cudaStreamNonBlocking));
            ND_CUDA(cudaStreamBeginCapture(p->cap_stream, cudaStreamCaptureModeRelaxed));
            nd_status rc = one_iteration(nullptr, p->cap_stream);
            if (rc == ND_OK) rc = one_iteration(nullptr, p->cap_stream);
            const cudaError_t ce = cudaStreamEndCapture(p->cap_stream, &graph);
            if (rc != ND_OK || ce != cudaSuccess) {
                if (graph) cudaGraphDestroy(graph);
                if (p->phi_cur != phi0) std::swap(p->phi_cur, p->phi_new);
                return rc != ND_OK ? rc : nd_fail(ND_ERR_CUDA, cudaGetErrorString(ce));
            }
            p->iter_graph_kernels = p->kernels_launched - before;
            p->kernels_launched = before;                          // captured, not launched
            const cudaError_t ci = cudaGraphInstantiate(&p->iter_graph, graph, 0);
            cudaGraphDestroy(graph);
            if (ci != cudaSuccess) { p->iter_graph = nullptr; return nd_fail(ND_ERR_CUDA, cudaGetErrorString(ci)); }
            p->iter_graph_phi = p->phi_cur;                        // == phi0 after two swaps
        }
        for (; it + 2 <= max_iters; it += 2) {
            ND_CUDA(cudaGraphLaunch(p->iter_graph, st));
            p->kernels_launched += p->iter_graph_kernels;
        }
    }
    // Per-iteration records live in a device ring of kMaxStats slots; a full ring (and the last, partial one) is copied to
    // the caller's array, so any iteration count is recorded.  Without stats the convergence test reads slot 0.
    constexpr int SS = ndk::kStatsStride;
    std::vector<double> hs;
    int flushed = 0;   // records already delivered to `stats`
    auto deliver = [&](int upto) -> nd_status {   // stream is synchronised on return
        const int n = upto - flushed;
        if (n <= 0) return ND_OK;
        hs.resize((size_t)SS * n);
        ND_CUDA(cudaMemcpyAsync(hs.data(), p->stats, sizeof(double) * hs.size(), cudaMemcpyDeviceToHost, st));
        ND_CUDA(cudaStreamSynchronize(st));
        for (int i = 0; i < n; ++i) {
            nd_iter_stats& o = stats[flushed + i];
            o.k_eff = hs[SS * i]; o.fission_rate = hs[SS * i + 1]; o.dk = hs[SS * i + 2]; o.dphi_max = hs[SS * i + 3];
            o.leakage = hs[SS * i + 4]; o.balance_residual = hs[SS * i + 5];
        }
        flushed = upto;
        return ND_OK;
    };
    for (; it < max_iters; ++it) {
        double* slot = stats ? p->stats + (size_t)SS * ((it - flushed) % kMaxStats) : (sync_each ? p->stats : nullptr);
        nd_status rc = one_iteration(slot, st);
        if (rc != ND_OK) return rc;
        bool stop = false;
        if (sync_each) {
            double h[4];
            ND_CUDA(cudaMemcpyAsync(h, slot, sizeof h, cudaMemcpyDeviceToHost, st));
            ND_CUDA(cudaStreamSynchronize(st));
            const bool ok_k = !(tol_k > 0.0) || std::fabs(h[2]) < tol_k;
            const bool ok_p = !(tol_phi > 0.0) || h[3] < tol_phi;
            stop = ok_k && ok_p;
        }
        if (stats && (it + 1 - flushed == kMaxStats || stop)) {
            rc = deliver(it + 1);
            if (rc != ND_OK) return rc;
        }
        if (stop) { converged = true; ++it; break; }
    }
    if (stats) {
        const nd_status rc = deliver(it);
        if (rc != ND_OK) return rc;
    }
    double hk[2];
    ND_CUDA(cudaMemcpyAsync(hk, p->scalars, sizeof(double) * 2, cudaMemcpyDeviceToHost, st));
    if (d_phi_out)
        ND_CUDA(cudaMemcpyAsync(d_phi_out, p->phi_cur, sizeof(double) * (size_t)d.R * d.G, cudaMemcpyDeviceToDevice, st));
    ND_CUDA(cudaStreamSynchronize(st));
    *k_eff_out = hk[ndk::SC_K];
    if (iters_done) *iters_done = it;
    if (use_tol && !converged) return nd_fail(ND_ERR_NOT_CONVERGED, "nd_power_iteration: max_iters reached before the tolerances");
    return ND_OK;
}

// ------------------------------------------------------------------------------------------------
// state access
// ------------------------------------------------------------------------------------------------
extern "C" nd_status nd_tally_reducer_set(nd_problem* p, nd_tally_reduce_fn fn, void* user)
{
    if (!p) return nd_fail(ND_ERR_NULL, "nd_tally_reducer_set: NULL problem");
    p->reduce_fn = fn;
    p->reduce_user = user;
    return ND_OK;
}

extern "C" nd_status nd_state_reset(nd_problem* p, void* cuda_stream)
{
    if (!p) return nd_fail(ND_ERR_NULL, "nd_state_reset: NULL problem");
    return reset_state(p, as_stream(cuda_stream));
}

extern "C" nd_status nd_boundary_flux_fill(nd_problem* p, float value, void* cuda_stream)
{
    if (!p) return nd_fail(ND_ERR_NULL, "nd_boundary_flux_fill: NULL problem");
    return launch_fill_f32(p, p->psi_in, value, (int64_t)p->d.T * 2 * p->d.P * p->d.Gs, as_stream(cuda_stream));
}

extern "C" nd_status nd_boundary_flux_get(nd_problem* p, float* host_out, void* cuda_stream)
{
    if (!p || !host_out) return nd_fail(ND_ERR_NULL, "nd_boundary_flux_get: NULL argument");
    cudaStream_t st = as_stream(cuda_stream);
    const Dims& d = p->d;
    const size_t rows = (size_t)d.T * 2 * d.P;
    ND_CUDA(cudaMemcpy2DAsync(host_out, sizeof(float) * d.G, p->psi_in, sizeof(float) * d.Gs, sizeof(float) * d.G, rows, cudaMemcpyDeviceToHost, st));
    ND_CUDA(cudaStreamSynchronize(st));
    return ND_OK;
}

extern "C" nd_status nd_outgoing_flux_get(nd_problem* p, float* host_out, void* cuda_stream)
{
    if (!p || !host_out) return nd_fail(ND_ERR_NULL, "nd_outgoing_flux_get: NULL argument");
    cudaStream_t st = as_stream(cuda_stream);
    const Dims& d = p->d;
    const size_t rows = (size_t)d.T * 2 * d.P;
    ND_CUDA(cudaMemcpy2DAsync(host_out, sizeof(float) * d.G, p->psi_out, sizeof(float) * d.Gs, sizeof(float) * d.G, rows, cudaMemcpyDeviceToHost, st));
    ND_CUDA(cudaStreamSynchronize(st));
    return ND_OK;
}

extern "C" nd_status nd_boundary_flux_set(nd_problem* p, const float* host_in, void* cuda_stream)
{
    if (!p || !host_in) return nd_fail(ND_ERR_NULL, "nd_boundary_flux_set: NULL argument");
    cudaStream_t st = as_stream(cuda_stream);
    const Dims& d = p->d;
    const size_t rows = (size_t)d.T * 2 * d.P;
    ND_CUDA(cudaMemsetAsync(p->psi_in, 0, sizeof(float) * rows * d.Gs, st));
    ND_CUDA(cudaMemcpy2DAsync(p->psi_in, sizeof(float) * d.Gs, host_in, sizeof(float) * d.G, sizeof(float) * d.G, rows, cudaMemcpyHostToDevice, st));
    ND_CUDA(cudaStreamSynchronize(st));
    return ND_OK;
}

extern "C" nd_status nd_flux_get(nd_problem* p, double* d_phi_out, void* cuda_stream)
{
    if (!p || !d_phi_out) return nd_fail(ND_ERR_NULL, "nd_flux_get: NULL argument");
    ND_CUDA(cudaMemcpyAsync(d_phi_out, p->phi_cur, sizeof(double) * (size_t)p->d.R * p->d.G, cudaMemcpyDeviceToDevice, as_stream(cuda_stream)));
    return ND_OK;
}

extern "C" nd_status nd_flux_set(nd_problem* p, const double* d_phi, double k_eff, void* cuda_stream)
{
    if (!p || !d_phi) return nd_fail(ND_ERR_NULL, "nd_flux_set: NULL argument");
    if (!(k_eff > 0.0)) return nd_fail(ND_ERR_INVALID, "nd_flux_set: k_eff must be > 0");
    cudaStream_t st = as_stream(cuda_stream);
    ND_CUDA(cudaMemcpyAsync(p->phi_cur, d_phi, sizeof(double) * (size_t)p->d.R * p->d.G, cudaMemcpyDeviceToDevice, st));
    ND_CUDA(cudaMemcpyAsync(p->scalars + ndk::SC_K, &k_eff, sizeof(double), cudaMemcpyHostToDevice, st));
    ND_CUDA(cudaStreamSynchronize(st));
    return launch_fission_rate(p, p->phi_cur, nullptr, st);
}

extern "C" nd_status nd_track_volume_get(nd_problem* p, double* host_out)
{
    if (!p || !host_out) return nd_fail(ND_ERR_NULL, "nd_track_volume_get: NULL argument");
    memcpy(host_out, p->h_vol.data(), sizeof(double) * p->h_vol.size());
    return ND_OK;
}

extern "C" nd_status nd_tally_get(nd_problem* p, double* d_tally_out, void* cuda_stream)
{
    if (!p || !d_tally_out) return nd_fail(ND_ERR_NULL, "nd_tally_get: NULL argument");
    const Dims& d = p->d;
    cudaStream_t st = as_stream(cuda_stream);
    ndk::k_unpad_f64<<<grid_for((int64_t)d.R * d.G, 256, 8 * p->n_sm), 256, 0, st>>>(p->tally, d_tally_out, d.R, d.G, d.Gs);
    ND_LAUNCH_CHECK(p);
    return ND_OK;
}

#include "nd_cmfd_api.cuh"   // NEXT-3: the CMFD plan (nd_cmfd_*), on the problem's internals above
#include "nd_p1_api.cuh"     // NEXT-4: the P_1-scattering plan (nd_p1_*)

extern "C" nd_status nd_profile_enable(nd_problem* p, int32_t on)
{
    if (!p) return nd_fail(ND_ERR_NULL, "nd_profile_enable: NULL problem");
    p->profile = on != 0;
    p->phase_profile = on == 2 && p->sweep_kernel == ND_SWEEP_SWATH;
    p->ev_used = 0;
    p->kernels_launched = 0;
    if (p->phase_profile) ND_CUDA(cudaMemset(p->phase, 0, sizeof(unsigned long long) * ndk::kSwathPhases));
    return ND_OK;
}

extern "C" nd_status nd_profile_read(nd_problem* p, nd_profile* out)
{
    if (!p || !out) return nd_fail(ND_ERR_NULL, "nd_profile_read: NULL argument");
    double ms = 0.0;
    for (size_t i = 0; i < p->ev_used; ++i) {
        ND_CUDA(cudaEventSynchronize(p->ev_pool[i].b));
        float t = 0.f;
        ND_CUDA(cudaEventElapsedTime(&t, p->ev_pool[i].a, p->ev_pool[i].b));
        ms += t;
    }
    out->sweep_ms = ms;
    out->sweep_launches = (int64_t)p->ev_used;
    out->kernels_launched = p->kernels_launched;
    return ND_OK;
}

extern "C" nd_status nd_sweep_phases_get(nd_problem* p, double* host_out)
{
    if (!p || !host_out) return nd_fail(ND_ERR_NULL, "nd_sweep_phases_get: NULL argument");
    if (!p->phase_profile) return nd_fail(ND_ERR_STATE, "nd_sweep_phases_get: call nd_profile_enable(p, 2) on a swath-kernel problem first");
    unsigned long long h[ndk::kSwathPhases];
    ND_CUDA(cudaDeviceSynchronize());
    ND_CUDA(cudaMemcpy(h, p->phase, sizeof h, cudaMemcpyDeviceToHost));
    double tot = 0.0;
    for (int i = 0; i < ndk::kSwathPhases; ++i) tot += (double)h[i];
    for (int i = 0; i < ndk::kSwathPhases; ++i) host_out[i] = tot > 0.0 ? (double)h[i] / tot : 0.0;
    return ND_OK;
}

extern "C" nd_status nd_problem_stream_view(const nd_problem* p, nd_stream_device_view_t* out)
{
    if (!p || !out) return nd_fail(ND_ERR_NULL, "nd_problem_stream_view: NULL argument");
    if (!is_swath(p->sweep_kernel)) return nd_fail(ND_ERR_STATE, "nd_problem_stream_view: the problem does not run the swath kernel");
    memset(out, 0, sizeof *out);
    out->blob = p->blob; out->blob_bytes = p->blob_bytes; out->tile_ref = reinterpret_cast<const uint32_t*>(p->tile_ref);
    out->swath_tile0 = p->swath_tile0; out->swath_track = p->swath_track; out->items = reinterpret_cast<const int32_t*>(p->items);
    out->n_tiles = p->n_tiles; out->n_swaths = p->n_swaths; out->n_items = p->n_items;
    out->tracks_per_swath = p->sc.sp.NT; out->built_on_device = p->stream_on_device ? 1 : 0;
    return ND_OK;
}

extern "C" nd_status nd_problem_info_get(const nd_problem* p, nd_problem_info* out)
{
    if (!p || !out) return nd_fail(ND_ERR_NULL, "nd_problem_info_get: NULL argument");
    const Dims& d = p->d;
    memset(out, 0, sizeof *out);
    out->n_segments = d.S;
    out->n_segments_padded = d.Spad;
    out->updates_per_sweep = 2 * d.S * d.P * d.G;
    // segment stream once (8 B/segment) + psi in and out (4 B each per chain end)
    // + q read (4 B) and tally write (8 B) per (region, group)
    out->algorithmic_bytes = 8 * d.S + 2 * 4 * (int64_t)d.T * 2 * d.P * d.G + 12 * (int64_t)d.R * d.G;
    out->group_stride = d.Gs;
    out->sweep_kernel = p->sweep_kernel;
    out->n_batches = (int32_t)(p->n_tiles > INT32_MAX ? INT32_MAX : p->n_tiles);
    out->mean_regions_per_tile = p->mean_regions_per_tile;
    out->mean_segments_per_tile = p->mean_segments_per_tile;
    out->lockstep_efficiency = p->lockstep_efficiency;
    if (is_swath(p->sweep_kernel)) {
        out->block_threads = 32 * p->sc.warps; out->smem_bytes = p->sc.smem_bytes; out->grid_blocks = swath_grid(p);
        out->tracks_per_block = p->sc.sp.NT;
    } else {
        out->block_threads = 256;
    }
    return ND_OK;
}
