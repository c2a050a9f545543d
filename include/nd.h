/*
 * nd.h -- C ABI of the B200-native planar Method-of-Characteristics (MOC) hot path of
 * arxiv/paper_2607_01591 (NuDEAL).  One shared library, libnd_moc.so, hand-written CUDA for sm_100a.
 *
 * What the calls compute (line numbers of the paper text PAPER.md; readings R-T, R-W, O-5..O-8 are
 * listed in DESIGN.md because the paper is silent on them):
 *   nd_tracks_generate   cyclic ("modular") rays on the bounding box of the whole domain and the
 *                        ray-mesh intersection through a half-edge structure, done once before the
 *                        solve (section III.A).  HOST code, FP64, bit-exact rules.
 *                        nd_tracks_generate_device runs the ray walk on the GPU, bit-identically.
 *   nd_problem_create    packs the precomputed segment data into the device segment
 *                        stream and uploads cross sections, quadrature weights and the link table.
 *   nd_transport_sweep   Eq. (5) along every track, direction, polar angle and group,
 *                        the angular integration to the scalar flux, and the boundary
 *                        angular-flux exchange through the link table.
 *   nd_source_update     right-hand side of Eq. (1)/(3): scatter + chi/k * fission.
 *   nd_power_iteration   the outer iteration that Eq. (1)'s k_eff implies ("# of
 *                        transport sweeps").
 *
 * Conventions
 *   - No C++ types, no torch types, no exceptions cross this boundary.  Every function returns an
 *     nd_status (ND_OK = 0) except the three string/version getters.  On error, outputs are untouched.
 *   - "HOST" pointers are ordinary host memory, borrowed for the duration of the call and copied.
 *     "DEVICE" pointers are CUDA device memory owned by the caller (e.g. a torch tensor's data_ptr);
 *     the library never allocates device memory: the caller passes one workspace block.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  All device
 *     work is stream-ordered and asynchronous, except where a HOST scalar/array is returned: those
 *     calls synchronise the stream before returning.
 *   - Canonical layouts at the ABI: phi, Q [R][G] row-major FP64; boundary psi [T][2][P][G] FP32,
 *     index [t][d] = the flux ENTERING track t travelling in direction d (0 forward, 1 backward).
 *     Internal device layouts (padding, track order, FP32 copies) are private.
 *   - No CPU fallback exists.  Every compute entry point fails with ND_ERR_CUDA when no device or
 *     no sm_100 kernel image is available.
 */
#ifndef ND_MOC_H
#define ND_MOC_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ND_VERSION 0x00020000u /* major<<16 | minor<<8 | patch */

typedef enum {
    ND_OK = 0,
    ND_ERR_NULL = 1,          /* a required pointer is NULL */
    ND_ERR_INVALID = 2,       /* an argument violates a stated precondition (message in nd_last_error) */
    ND_ERR_RANGE = 3,         /* an index (region, material, link) is out of range, or a size exceeds a limit */
    ND_ERR_WORKSPACE = 4,     /* workspace too small or not 256-byte aligned */
    ND_ERR_CUDA = 5,          /* a CUDA call failed / no usable device */
    ND_ERR_STATE = 6,         /* call not valid in the problem's current state */
    ND_ERR_NOT_CONVERGED = 7, /* nd_power_iteration hit max_iters with tolerances set (outputs ARE written) */
    ND_ERR_MESH = 8,          /* nd_tracks_generate: mesh is not a conforming CCW triangulation of the rectangle */
    ND_ERR_NOMEM = 9          /* host allocation failed */
} nd_status;

enum { ND_BC_VACUUM = 0, ND_BC_REFLECTIVE = 1 };

/* exp_mode: how 1 - exp(-tau) is evaluated in the FP32 sweep */
enum {
    ND_EXP_FAST = 0,    /* ex2.approx (MUFU) on tau*log2(e); abs error of exp <= 2 ulp(1) ~ 2.4e-7   */
    ND_EXP_EXPM1 = 1    /* -expm1f(-tau): ~1 ulp relative in 1-exp(-tau); slow path, used as a cross-check */
};
/* sweep_kernel: which sweep implementation runs (all give the same result up to summation order) */
enum {
    ND_SWEEP_AUTO = 0,      /* the fastest validated kernel for this G,P */
    ND_SWEEP_ATOMIC = 1,    /* warp per (track,direction), lanes over groups, FP64 global atomics per segment */
    ND_SWEEP_SWATH = 3      /* thread block per swath of adjacent tracks, psi in registers along the whole track,
                               per-segment delta rows in shared memory, one FP64 RED per (region, group) per tile.
                               (Values 2 and 4 named two slower round-1 kernels that were removed.) */
};

typedef struct {
    int32_t exp_mode;       /* ND_EXP_*      (default 0) */
    int32_t sweep_kernel;   /* ND_SWEEP_*    (default 0) */
    int32_t window_regions; /* ND_SWEEP_SWATH: max distinct regions per tile; 0 = default */
    int32_t block_warps;    /* ND_SWEEP_SWATH: warps per thread block (tracks per swath = warps * slots per warp); 0 = default */
    int32_t tile_segments;  /* ND_SWEEP_SWATH: max segments of one track per tile; 0 = default */
    int32_t delta_buffers;  /* ND_SWEEP_SWATH: 1 or 2 delta buffers; 0 = default (1).  Two buffers no longer save the barrier
                               before the segment loop (it also guards the chunk ring); kept for experiments */
    int32_t blocks_per_sm;  /* ND_SWEEP_SWATH: resident blocks per SM the grid is sized for; 0 = default */
    int32_t tile_lag;       /* ND_SWEEP_SWATH: drift of the track fronts (in mean segment lengths) under which a tile gives
                               every track the same number of segments; 0 = default, -1 = always cut geometrically */
    int32_t q_copies;       /* ND_SWEEP_SWATH, rows of <= 16 groups: copies of a staged q row per shared-memory line.  The
                               Sigma_t table and the delta rows are interleaved NC = 8 / (lanes per track) slots to a line so
                               that the slots of a warp never meet in a bank; q_copies = NC does the same for the q rows
                               (NC cp.async copies per region and tile), 1 stages one copy per region (adjacent tracks in the
                               same region read it as a broadcast, tracks in different regions may conflict).  0 = default
                               (1); values above NC or not dividing it are rounded down to a divisor of NC.  Configurations that
                               land on the register-capped kernel variant (more than 512 resident threads per SM) always use NC */
    int32_t graph_mode;     /* nd_power_iteration with a fixed iteration count (no tolerances, no per-iteration stats, profiling
                               off) replays a CUDA graph of two iterations instead of launching their kernels one by one:
                               0 = default (on for calls of >= 4 iterations), 1 = never */
    int32_t cmfd_stream;    /* 1: lay the swath kernel's shared memory out for the CMFD current tally (a W row per track and a
                               ring of crossing lists: ~8 KB per block more, so tiles may come out a segment shorter) and keep
                               on the host what nd_cmfd_create needs to place the crossings; 0 = default */
    int32_t item_order;     /* ND_SWEEP_SWATH: order in which thread blocks take the (swath, direction) work items.  0 = default:
                               most expensive first (best load balance; measured fastest at every config); 1 = angle by angle,
                               adjacent swaths consecutively (blocks that run together touch neighbouring regions) */
    int32_t p1_stream;      /* 1: lay the swath kernel's shared memory out for the P_1 sweep of an nd_p1 plan as well (a second q
                               row per region and a second delta row per segment: about twice the tile storage, so tiles come
                               out shorter and the isotropic sweep of this problem somewhat slower); 0 = default */
    int32_t reserved[3];    /* must be 0 */
} nd_options;

/* ------------------------------------------------------------------------------------------------
 * Host preprocessing: track laydown (rule R-T), links (O-3), half-edge ray walk (rule R-W), track
 * volumes (O-5).  Output is bit-exact against the independent oracle (tests/test_abi_and_tracks.py).
 * ---------------------------------------------------------------------------------------------- */
typedef struct {
    int32_t n_vertices, n_triangles;
    const double* xy;       /* HOST [V][2] vertex coordinates, domain is exactly [0,W]x[0,H]            */
    const int32_t* tri;     /* HOST [R][3] counter-clockwise vertex ids; one triangle = one FSR */
    double W, H;            /* bounding rectangle */
    int32_t bc[4];          /* left, right, bottom, top: ND_BC_VACUUM / ND_BC_REFLECTIVE */
} nd_mesh_desc;

typedef struct nd_tracks nd_tracks; /* opaque, HOST memory owned by the library */

/* n_azim: directions over [0,2pi), divisible by 4.  spacing: desired ray spacing (cm).
 * n_threads: host threads for the ray walk (0 = all). */
nd_status nd_tracks_generate(const nd_mesh_desc* mesh, int32_t n_azim, double spacing, int32_t n_threads,
                             nd_tracks** out);

typedef struct {            /* all pointers HOST, owned by the nd_tracks object, valid until nd_tracks_destroy */
    int32_t n_tracks;       /* T */
    int32_t n_regions;      /* R */
    int64_t n_segments;     /* S */
    int32_t n_half;         /* N_a/2 track angles in (0,pi) */
    const int64_t* track_seg_offset; /* [T+1] */
    const int32_t* seg_region;       /* [S] */
    const double* seg_length;        /* [S] 2-D projected lengths, > 0 */
    const double* track_weight;      /* [T] omega_a * delta_a */
    const int32_t* link;             /* [T][2] 2*t'+d' or -1 */
    const int32_t* track_azim;       /* [T] track-angle index j */
    const double* track_ends;        /* [T][4] x0,y0,x1,y1 */
    const double* track_volume;      /* [R] A~_r = sum 2*omega_a*delta_a*s */
    const double* azim_phi;          /* [N_a/2] effective angles */
    const double* azim_weight;       /* [N_a/2] omega_a per direction (sum over N_a directions = 1) */
    const double* azim_spacing;      /* [N_a/2] effective spacing delta_a */
    const int32_t* track_global;     /* [T] id of the track in the unsharded laydown (identity unless made by nd_tracks_shard) */
    const int32_t* seg_region_device;/* DEVICE [S], NULL unless made by nd_tracks_generate_resident (then seg_region and   */
    const double* seg_length_device; /* DEVICE [S]  seg_length above are NULL until nd_tracks_materialise)                */
} nd_tracks_view_t;

/* The same preprocessing with the ray walk (rule R-W, one step per segment: almost all of the work) on the GPU:
 * one thread per track, FP64 round-to-nearest intrinsics only, so the output is bit-identical to nd_tracks_generate's.
 * Laydown, links and the half-edge twins are still built on the host.  The result is the same HOST object.
 *   device_workspace  DEVICE, 256-byte aligned, caller-owned, free to reuse after the call.  It must hold at least
 *                     *min_bytes; every further *bytes_per_segment bytes let one more segment be traced per batch (the
 *                     fill pass runs in as many batches of tracks as the workspace requires).
 * Synchronises the stream before returning.  ND_ERR_WORKSPACE if the workspace is too small for the longest track. */
nd_status nd_tracks_device_workspace_bytes(const nd_mesh_desc* mesh, int32_t n_azim, double spacing, size_t* min_bytes,
                                           size_t* bytes_per_segment);
typedef struct {                /* where the time of nd_tracks_generate_device went (HOST wall clock / CUDA events) */
    double prepare_s;           /* host: laydown, links, half-edge twins, start triangles */
    double count_kernel_ms;     /* device: walk pass 1 (segment counts) */
    double fill_kernel_ms;      /* device: walk pass 2 (segments), summed over the batches */
    double copy_s;              /* device -> host copies of the segment arrays */
    double finish_s;            /* host: track volumes in canonical order */
    double total_s;
    int64_t n_segments;
    int32_t batches, reserved;
} nd_trace_timing;
nd_status nd_tracks_generate_device(const nd_mesh_desc* mesh, int32_t n_azim, double spacing, void* device_workspace,
                                    size_t device_bytes, void* cuda_stream, nd_trace_timing* timing_or_null,
                                    nd_tracks** out);

/* The device tracer with the segments left WHERE THEY ARE: seg_region / seg_length of all S segments stay in
 * `device_workspace` (nd_tracks_view: seg_region_device / seg_length_device; same values, bit for bit, as the host arrays of
 * nd_tracks_generate), and nothing of size S is copied to the host.  Pass them to nd_problem_create with
 * nd_problem_desc.seg_on_device = 1.  The track volumes A~_r are summed on the GPU (FP64 atomics: equal to
 * nd_tracks_generate's to rounding, not bit for bit).  The host arrays of the segments are made on demand by
 * nd_tracks_materialise (what nd_cmfd_surfaces, nd_p1_create and nd_tracks_shard read).
 *   device_workspace  DEVICE, 256-byte aligned, caller-owned; must stay untouched until nd_tracks_destroy or until the
 *                     last use of the device pointers and of nd_tracks_materialise.  It must hold
 *                     *min_bytes (nd_tracks_device_workspace_bytes) - 2^20 * bytes_per_segment + S * bytes_per_segment
 *                     bytes; S is known only after the count pass, so a workspace that is too small gives
 *                     ND_ERR_WORKSPACE with the size that suffices in *required_bytes (call again).
 * Synchronises the stream before returning. */
nd_status nd_tracks_generate_resident(const nd_mesh_desc* mesh, int32_t n_azim, double spacing, void* device_workspace,
                                      size_t device_bytes, void* cuda_stream, nd_trace_timing* timing_or_null,
                                      size_t* required_bytes_or_null, nd_tracks** out);
/* Copies the device-resident segment arrays to host arrays owned by `tracks` (no-op when they exist); nd_tracks_view then
 * returns them.  Synchronises the stream. */
nd_status nd_tracks_materialise(nd_tracks* tracks, void* cuda_stream);

/* NEXT-2 (the paper names multi-GPU as future work): shard `shard` of `n_shards` of an ANGLE-PAIR
 * partition of a cyclic laydown.  A reflective link joins a track of angle j only to one of its complement N_a/2-1-j (O-3),
 * so a shard that owns whole pairs {j, N_a/2-1-j} exchanges no boundary flux; the shards share the additive tally alone
 * (nd_tally_reducer_set).  Pairs are dealt to the shards by segment count, longest first (deterministic).
 * The result is a new HOST object with the shard's tracks in canonical order, ids renumbered, links remapped,
 * track_global = their ids in `full`, and track_volume = the areas A~_r of the WHOLE laydown (pass it to nd_problem_create
 * as nd_problem_desc.region_volume: every shard divides its flux by the full track-estimated area).
 * Errors: ND_ERR_NULL, ND_ERR_INVALID (shard out of range, n_shards > N_a/4), ND_ERR_STATE (`full` is itself a shard). */
nd_status nd_tracks_shard(const nd_tracks* full, int32_t n_shards, int32_t shard, nd_tracks** out);

nd_status nd_tracks_view(const nd_tracks* tracks, nd_tracks_view_t* view);
nd_status nd_tracks_destroy(nd_tracks* tracks);

/* ------------------------------------------------------------------------------------------------
 * Problem: mesh regions, track segments, linked boundary ends, polar quadrature, multigroup XS.
 * ---------------------------------------------------------------------------------------------- */
typedef struct {                    /* all pointers: HOST memory, borrowed for the call only */
    int32_t n_regions, n_materials, n_groups, n_polar, n_tracks;
    const int32_t* region_material; /* [R]  0..M-1 */
    const double* sigma_t;          /* [M][G]  > 0 */
    const double* sigma_s;          /* [M][G_to][G_from]  Sigma_{s,g'->g} at [m][g][g'] */
    const double* nu_sigma_f;       /* [M][G]  >= 0 */
    const double* chi;              /* [M][G]  >= 0 */
    const double* polar_sin;        /* [P]  sin(theta_p) in (0,1] */
    const double* polar_weight;     /* [P]  sums to 1 over the upper hemisphere */
    const int64_t* track_seg_offset;/* [T+1] CSR into the segment arrays, forward order */
    const int32_t* seg_region;      /* [S]  0..R-1 */
    const double* seg_length;       /* [S]  > 0, finite */
    const double* track_weight;     /* [T]  omega_a * delta_a.  The library forms
                                       w[t][p] = 4*pi*track_weight[t]*polar_weight[p]*polar_sin[p]  and
                                       A~[r] = sum over segments in r of 2*track_weight[t]*seg_length     */
    const int32_t* link;            /* [T][2] [t][0]: where the FORWARD outgoing flux goes, [t][1]: BACKWARD.
                                       value 2*t'+d' = enter track t' travelling in direction d'; -1 = vacuum.
                                       Non-negative links must be distinct (each entry is fed at most once). */
    /* Optional track geometry (both NULL or both set; nd_tracks_view provides them).  Used ONLY to order the
       device segment stream (adjacent parallel tracks are batched so that they share flat-source regions);
       results do not depend on it.  Without it ND_SWEEP_AUTO selects the atomic sweep kernel. */
    const int32_t* track_azim;      /* [T] id of the track's angle; tracks with equal id are parallel */
    const double* track_ends;       /* [T][4] x0,y0,x1,y1 (forward direction runs from 0 to 1) */
    /* Optional (NULL = the library forms A~ from this descriptor's own segments): the track-estimated areas A~_r to divide
       by, HOST [R], finite and >= 0.  A shard of an angle-pair partition (nd_tracks_shard) holds a part of the tracks but
       must use the areas of all of them; for unsharded tracks nd_tracks_view's track_volume saves the pass over the segments. */
    const double* region_volume;
    /* 0: seg_region / seg_length are HOST arrays.  1: they are DEVICE arrays (nd_tracks_generate_resident leaves them in
       its workspace; nd_tracks_view: seg_region_device / seg_length_device), borrowed for the call only; every other array
       of the descriptor stays on the host.  The whole of nd_problem_create's work on segments then runs on the GPU: their
       validation, A~_r (when region_volume is NULL; FP64 atomics, so the last bits depend on the order), the atomic
       kernel's SoA stream, and the swath kernel's chunk stream (one thread per swath through the same cutter/encoder as
       the host builder: the two streams are equal byte for byte).  Needs track_azim / track_ends. */
    int32_t seg_on_device;
    int32_t reserved;               /* must be 0 */
} nd_problem_desc;

typedef struct nd_problem nd_problem; /* opaque host object; owns no device memory except what lies in the workspace */
typedef struct nd_cmfd nd_cmfd;       /* a CMFD plan bound to one problem (NEXT-3, below) */

/* Limits: n_regions <= 2^24, n_materials <= 256, n_groups <= 256, n_polar <= 4. */
nd_status nd_workspace_bytes(const nd_problem_desc* desc, const nd_options* opts_or_null, size_t* device_bytes);

/* device_workspace: DEVICE, >= nd_workspace_bytes, 256-byte aligned, caller-owned; must outlive the problem.
 * Validates the descriptor (ranges, monotone offsets, positive lengths and sigma_t, polar weights sum to 1
 * within 1e-9, distinct links), uploads, and sets the state of O-8: phi = 1, boundary psi = 0, k = 1.
 * Synchronises the stream before returning. */
nd_status nd_problem_create(const nd_problem_desc* desc, const nd_options* opts_or_null, void* device_workspace,
                            size_t device_bytes, void* cuda_stream, nd_problem** out);
nd_status nd_problem_destroy(nd_problem* p); /* does not touch the workspace */

/* One transport sweep (O-6) with a caller-supplied isotropic angular source Q (per steradian).
 *   d_Q       DEVICE [R][G] FP64, read
 *   d_phi_out DEVICE [R][G] FP64, written: phi = 4 pi Q/Sigma_t + tally/(Sigma_t A~_r)
 * Reads the problem's current boundary psi (Jacobi: the previous sweep's outgoing fluxes), advances it through
 * the link table (vacuum entries become 0).  FP32 segment arithmetic, FP64 tallies. */
nd_status nd_transport_sweep(nd_problem* p, const double* d_Q, double* d_phi_out, void* cuda_stream);

/* NEXT-2: a problem built from one shard of an angle-pair partition (nd_tracks_shard, with
 * nd_problem_desc.region_volume = the areas of the whole laydown) tallies only its own tracks.  The reducer is called by
 * nd_transport_sweep and by every iteration of nd_power_iteration right after the sweep, before the tally is turned into a
 * flux (O-6 finalise): it must replace d_tally (DEVICE [n_doubles] FP64, the padded [R][Gs] tally) by the SUM over all
 * shards, in stream order on `cuda_stream` (e.g. one NCCL all-reduce).  Everything else -- source, flux, k -- is then
 * computed redundantly and identically by every shard; boundary flux never leaves a shard.  Return 0 on success.
 * fn = NULL removes the reducer.  With a reducer set nd_power_iteration launches its kernels one by one (no CUDA graph),
 * and nd_iter_stats.leakage / balance_residual are reported as 0 (they compare a problem's own boundary flux with its own
 * tally). */
typedef int32_t (*nd_tally_reduce_fn)(void* user, double* d_tally, int64_t n_doubles, void* cuda_stream);
nd_status nd_tally_reducer_set(nd_problem* p, nd_tally_reduce_fn fn, void* user);

/* O-7: Q[r][g] = (1/4pi) ( sum_g' Sigma_s[m][g][g'] phi[r][g'] + chi[m][g]/k * sum_g' nuSigma_f[m][g'] phi[r][g'] ).
 *   d_phi DEVICE [R][G] FP64 read; d_Q_out DEVICE [R][G] FP64 written;
 *   d_fission_rate_out DEVICE FP64 scalar or NULL: F = sum_r A~_r sum_g nuSigma_f phi (of d_phi). */
nd_status nd_source_update(nd_problem* p, const double* d_phi, double k_eff, double* d_Q_out,
                           double* d_fission_rate_out, void* cuda_stream);

/* One record per iteration, HOST.  leakage = sum over the chains that end on a VACUUM side of w_{t,p} psi_exit, all groups
 * (with the state normalised to a fission rate of 1, as O-8 sweeps it).  balance_residual = (in - out - sum of the tallies)
 * / (in + out), in / out = sum of w_{t,p} psi over all track ends entering / leaving: the telescoping identity of Eq. (5)
 * over the whole sweep, zero up to the FP32 rounding of the chains (~1e-7); a tally credited to no region or
 * twice shows up here. */
typedef struct { double k_eff, fission_rate, dk, dphi_max, leakage, balance_residual; } nd_iter_stats;

/* O-8, canonical power iteration from the problem's current state (phi, boundary psi, k).
 *   max_iters >= 0.  tol_k <= 0 and tol_phi <= 0: run exactly max_iters iterations with no host sync inside
 *   the loop.  Otherwise stop when |k - k_prev| < tol_k and max|phi/F - phi_prev|/max(phi) < tol_phi.
 *   k_eff_out HOST; d_phi_out DEVICE [R][G] FP64 or NULL (the un-normalised phi of the last sweep, as in O-8);
 *   iters_done HOST or NULL; stats HOST [max_iters] or NULL: every iteration is recorded (one extra pass over the
 *   boundary flux per iteration for leakage / balance_residual; the host is synchronised once per 4096 iterations). */
nd_status nd_power_iteration(nd_problem* p, int32_t max_iters, double tol_k, double tol_phi, double* k_eff_out,
                             double* d_phi_out, int32_t* iters_done, nd_iter_stats* stats_or_null, void* cuda_stream);

/* State access (checkpoint / resume, tests).  Canonical layouts. */
nd_status nd_state_reset(nd_problem* p, void* cuda_stream);                       /* phi=1, psi=0, k=1 */
nd_status nd_boundary_flux_fill(nd_problem* p, float value, void* cuda_stream);
nd_status nd_boundary_flux_get(nd_problem* p, float* host_out, void* cuda_stream);       /* HOST [T][2][P][G] */
nd_status nd_boundary_flux_set(nd_problem* p, const float* host_in, void* cuda_stream);  /* HOST [T][2][P][G] */
/* The flux LEAVING every track end in the last sweep, [t][d] = exit of track t swept in direction d, before the link
 * table is applied (vacuum exits included): with the entering flux it closes the telescoping balance
 * sum_r tally[r][g] = sum_{t,d,p} w_{t,p} (psi_in - psi_out)[g] at any problem size. */
nd_status nd_outgoing_flux_get(nd_problem* p, float* host_out, void* cuda_stream);       /* HOST [T][2][P][G] */
nd_status nd_flux_get(nd_problem* p, double* d_phi_out, void* cuda_stream);        /* DEVICE [R][G] */
nd_status nd_flux_set(nd_problem* p, const double* d_phi, double k_eff, void* cuda_stream);
nd_status nd_track_volume_get(nd_problem* p, double* host_out);                    /* HOST [R] */
nd_status nd_tally_get(nd_problem* p, double* d_tally_out, void* cuda_stream);     /* DEVICE [R][G], last sweep */

/* NEXT-3 (CMFD, Algorithm 1 "Solve CMFD on the coarse mesh"), step C-2 of DESIGN.md 8d: the interior
 * surfaces of a coarse mesh = the unordered pairs of coarse cells (lo < hi) that two consecutive segments of some track
 * join, plus the pairs a reflective hand-over joins (the cell in which chain (t, d) ends and the cell in which the chain
 * link[t][d] begins).  HOST code, integers only, no GPU.  Uses desc->n_regions, n_tracks, track_seg_offset, seg_region, link.
 *   cell         HOST [R], 0 <= cell[r] < n_cells (C-1: any map of regions to coarse cells)
 *   capacity     entries pair_lo / pair_hi can hold; 0 = size query (pair_lo / pair_hi may be NULL)
 *   n_pairs_out  HOST, written: the number of surfaces
 *   pair_lo/hi   HOST [capacity], written when capacity >= *n_pairs_out, sorted by (lo, hi): what nd_cmfd_create takes
 *                as its surface list
 * Errors: ND_ERR_NULL, ND_ERR_INVALID (sizes; capacity > 0 but too small: *n_pairs_out is still written), ND_ERR_RANGE,
 * ND_ERR_NOMEM. */
nd_status nd_cmfd_surfaces(const nd_problem_desc* desc, int32_t n_cells, const int32_t* cell, int32_t capacity,
                           int32_t* n_pairs_out, int32_t* pair_lo, int32_t* pair_hi);

/* ------------------------------------------------------------------------------------------------
 * NEXT-3: CMFD acceleration, Algorithm 1 of the paper ("Perform MOC on the fine mesh", "Solve CMFD on the
 * coarse mesh", update of the fine-mesh flux; purpose PAPER.md:129).  The paper prints no formula; the reading C-1..C-9 is in
 * DESIGN.md 8d.  A PLAN binds a coarse mesh to one problem.  Everything it needs lives in one caller-owned device workspace;
 * the net currents of C-3 are tallied by the sweep kernel itself (the tracks are walked once), and an accelerated iteration
 * only launches kernels: no allocation, no host arithmetic, no stream synchronisation between its steps.
 * The problem must use the swath sweep kernel, exp_mode = ND_EXP_FAST, and have been created with nd_options.cmfd_stream = 1
 * (its shared-memory layout then holds the per-track W rows and the crossing lists); else ND_ERR_STATE.
 * ---------------------------------------------------------------------------------------------- */
typedef struct {
    double tol;             /* coarse eigen-solve: |dk| < tol |k| and max |dPhi| < 100 tol max |Phi|; 0 = default 1e-12 */
    int32_t max_outer;      /* fission-source iterations of the coarse solve at most; 0 = default 20000 */
    int32_t inner_sweeps;   /* block-Jacobi sweeps per fission-source iteration; 0 = default 4 */
    double relax;           /* C-9 with ratio = 1 + relax (Phi_new / Phi_old - 1), 0 < relax <= 1; 0 = default 1 (undamped).
                               Coarse cells of several mean free paths make the undamped scheme diverge: use
                               cells of at most ~2 mean free paths, or relax ~0.5-0.7 */
    double rel_tol;         /* > 0: the coarse solve also stops once max |dPhi| has fallen to rel_tol x its value in the solve's first
                               iteration.  An inexact coarse solve does not move the fixed point of the accelerated iteration
                               (at the converged fine-mesh flux the collapsed flux IS the coarse eigenvector and the solve
                               stops at once); it trades coarse iterations for a few more sweeps.  0 = default: off */
    int32_t reserved[2];    /* must be 0 */
} nd_cmfd_options;
typedef struct {            /* one per accelerated iteration, HOST */
    double k_sweep;         /* k after the transport sweep (the plain O-8 update) */
    double k_eff;           /* the state's k after the coarse solve and prolongation */
    int32_t coarse_iters;   /* fission-source iterations of the coarse solve */
    int32_t coarse_ok;      /* 1: converged to a positive eigenpair and prolonged; 0: the solve failed and this iteration is a
                               plain one (ratio 1, k = k_sweep) */
} nd_cmfd_stats;

/*   desc            the descriptor the problem was created from (HOST, borrowed): track_seg_offset, seg_region and link are read
 *   cell            HOST [R], 0 <= cell[r] < n_cells (C-1)
 *   pair_lo/hi      HOST [n_pairs], lo < hi, each surface once: nd_cmfd_surfaces gives the list (C-2).  Every pair of cells that
 *                   consecutive segments of a track or a reflective hand-over join must be listed (else ND_ERR_INVALID)
 *   coupling        HOST [n_pairs], A_s / d_s of every surface (C-5), >= 0; 0 = no diffusive coupling (Dtil alone carries it)
 *   device_workspace DEVICE, >= nd_cmfd_workspace_bytes, 256-byte aligned, caller-owned, must outlive the plan
 * nd_cmfd_create synchronises the stream before returning. */
nd_status nd_cmfd_workspace_bytes(const nd_problem* p, const nd_problem_desc* desc, int32_t n_cells, const int32_t* cell,
                                  int32_t n_pairs, size_t* device_bytes);
nd_status nd_cmfd_create(nd_problem* p, const nd_problem_desc* desc, int32_t n_cells, const int32_t* cell, int32_t n_pairs,
                         const int32_t* pair_lo, const int32_t* pair_hi, const double* coupling,
                         const nd_cmfd_options* opts_or_null, void* device_workspace, size_t device_bytes, void* cuda_stream,
                         nd_cmfd** out);
nd_status nd_cmfd_destroy(nd_cmfd* c);

/* Algorithm 1, n_iters accelerated power iterations on the problem's own state: O-8's source, sweep (with C-3 in the sweep
 * kernel), flux and k; then C-4 collapse, C-5..C-8 coarse eigen-solve started from the collapsed flux and the sweep's k, C-9
 * prolongation of phi, of the stored boundary flux and of k.  Stream-ordered; the host is synchronised once, at the end.
 *   k_eff_out HOST; stats HOST [n_iters] or NULL.
 * Errors: ND_ERR_NULL, ND_ERR_INVALID, ND_ERR_CUDA, ND_ERR_STATE (a hand-over between unlisted cells). */
nd_status nd_cmfd_iteration(nd_cmfd* c, int32_t n_iters, double* k_eff_out, nd_cmfd_stats* stats_or_null, void* cuda_stream);

/* The steps one by one (tests, diagnostics).  Device results stay in the plan; the *_get calls copy to HOST and synchronise.
 *   nd_cmfd_sweep        C-3: nd_transport_sweep(d_Q -> d_phi_out) whose sweep kernel also tallies the net currents, integrated
 *                        over each surface with the sweep's own weights w_{t,p} = 4 pi omega_a delta_a w_p sin(theta_p):
 *                        J_surf [n_pairs][G] = sum of +w psi at every crossing lo -> hi, -w psi at hi -> lo;
 *                        J_vac / J_ref [n_cells][G]: at the exit end of every chain (t, d), w (psi_exit - psi_in of the
 *                        opposite direction), into J_vac[cell of the end] at a vacuum end, J_ref at a reflective one; a
 *                        hand-over into another cell c2 also adds w psi_exit to the surface and moves it from J_ref[c] to
 *                        J_ref[c2].  Per cell and group: sum of the sweep's tallies + sum +-J_surf + J_vac + J_ref = 0.
 *   nd_cmfd_collapse     C-4 of d_phi (DEVICE [R][G]; NULL = the problem's current flux): V, Phi = sum A~ phi / V,
 *                        sigma_t, nu_sigma_f = sum A~ Sigma phi / sum A~ phi, sigma_s [c][g][g'] weighted with phi_g',
 *                        chi weighted with the fission emission (0 where there is none).  A cell without regions gives NaN.
 *   nd_cmfd_coarse_set   loads coarse constants and currents from HOST arrays instead (to test the solve alone)
 *   nd_cmfd_solve        C-5..C-8 from the plan's constants and currents: D = 1/(3 Sigma_t), Dhat_s = 2 D_lo D_hi / (D_lo +
 *                        D_hi) coupling_s, Dtil_s = -(J_s + Dhat (Phi_hi - Phi_lo)) / (Phi_hi + Phi_lo), alpha = J_vac / Phi,
 *                        balance sum_s outflow + alpha Phi + Sigma_t V Phi - V sum_g' Sigma_s Phi_g' = (1/k) chi V sum_g'
 *                        nuSigma_f Phi_g'; dominant eigenpair by fission-source iteration with block-Jacobi inner sweeps (G x G
 *                        cell blocks inverted with partial pivoting), in ONE cooperative kernel.  Phi_new [n_cells][G] HOST or
 *                        NULL, normalised to the fission production of Phi.  ND_ERR_NOT_CONVERGED / ND_ERR_INVALID (eigenpair
 *                        not positive): outputs are written.
 *   nd_cmfd_prolong      C-9 with the last solve's Phi_new / Phi (ratio 1 if that solve failed): phi, the stored boundary flux
 *                        of every chain (ratio of the cell it enters), k; the state's fission rate is recomputed. */
nd_status nd_cmfd_sweep(nd_cmfd* c, const double* d_Q, double* d_phi_out, void* cuda_stream);
nd_status nd_cmfd_currents_get(nd_cmfd* c, double* J_surf, double* J_vac, double* J_ref, void* cuda_stream);
nd_status nd_cmfd_collapse(nd_cmfd* c, const double* d_phi_or_null, void* cuda_stream);
nd_status nd_cmfd_coarse_get(nd_cmfd* c, double* V, double* Phi, double* sigma_t, double* sigma_s, double* nu_sigma_f, double* chi,
                             void* cuda_stream);
nd_status nd_cmfd_coarse_set(nd_cmfd* c, const double* V, const double* Phi, const double* sigma_t, const double* sigma_s,
                             const double* nu_sigma_f, const double* chi, const double* J_surf, const double* J_vac,
                             void* cuda_stream);
nd_status nd_cmfd_solve(nd_cmfd* c, double k0, double* k_out, double* Phi_new_or_null, int32_t* iters_done_or_null,
                        void* cuda_stream);
nd_status nd_cmfd_prolong(nd_cmfd* c, void* cuda_stream);

/* ------------------------------------------------------------------------------------------------
 * NEXT-4: a second workload on the same segment data: the transport sweep with a linearly anisotropic (P_1)
 * scattering source, the Legendre expansion Eq. (2) truncated at l = 1.  Readings P-1..P-6, DESIGN.md 8e:
 *   Q(Omega) = Q0 + 3 (Omega_x Q1x + Omega_y Q1y),  Q0 as nd_source_update,  Q1 = (1/4pi) Sigma_s1 J,  J = integral of Omega psi;
 *   Omega_xy = sin(theta_p) x the unit vector of the direction of travel;  Eq. (5) with Q(Omega) of the chain's own direction;
 *   phi = 4 pi Q0/Sigma_t + tally0/(Sigma_t A~);  J = [4 pi 3 c2 (M Q1) + tally_xy] / (Sigma_t A~), c2 = sum_p w_p sin^2(theta_p),
 *   Mab[r] = sum over the segments of r of 2 omega_a delta_a s u_a u_b.
 * Two sweep kernels: on a problem created with sweep_kernel = ND_SWEEP_ATOMIC the one-warp-per-chain sweep over the plain
 * segment stream with three FP64 tallies per segment; on a swath-kernel problem created with nd_options.p1_stream = 1 the
 * swath kernel itself (a second staged source row 3 (u . q1) per region, a second delta row per segment, three tallies per
 * (region, group) of a tile: 2.6 - 5.4 times faster).  Any other problem: ND_ERR_STATE.
 *   desc       the descriptor the problem was created from, WITH track_ends (direction of every track) -- HOST, borrowed
 *   sigma_s1   HOST [M][g][g'] first Legendre moment of the scattering matrix, from g' into g
 * All d_* arrays DEVICE [R][G] FP64.  nd_p1_power_iteration runs O-8 with the P_1 source on the problem's own state (flux,
 * boundary flux, k) and the plan's currents (zero after nd_p1_state_reset / nd_p1_create); k_history HOST [n_iters] or NULL.
 * ---------------------------------------------------------------------------------------------- */
typedef struct nd_p1 nd_p1;
nd_status nd_p1_workspace_bytes(const nd_problem* p, size_t* device_bytes);
nd_status nd_p1_create(nd_problem* p, const nd_problem_desc* desc, const double* sigma_s1, void* device_workspace, size_t device_bytes,
                       void* cuda_stream, nd_p1** out);
nd_status nd_p1_destroy(nd_p1* c);
nd_status nd_p1_transport_sweep(nd_p1* c, const double* d_Q0, const double* d_Q1x, const double* d_Q1y, double* d_phi_out,
                                double* d_Jx_out, double* d_Jy_out, void* cuda_stream);
nd_status nd_p1_source_update(nd_p1* c, const double* d_phi, const double* d_Jx, const double* d_Jy, double k_eff, double* d_Q0_out,
                              double* d_Q1x_out, double* d_Q1y_out, void* cuda_stream);
nd_status nd_p1_state_reset(nd_p1* c, void* cuda_stream);
nd_status nd_p1_power_iteration(nd_p1* c, int32_t n_iters, double* k_eff_out, double* d_phi_out_or_null, double* d_Jx_out_or_null,
                                double* d_Jy_out_or_null, double* k_history_or_null, void* cuda_stream);

/* Device-time accounting.  When enabled, every sweep-kernel launch is bracketed by CUDA events on its own
 * stream; nd_profile_read synchronises and returns the accumulated kernel milliseconds and launch counts
 * since the last nd_profile_enable(p,1).  kernels_launched counts every kernel the library launched. */
typedef struct { double sweep_ms; int64_t sweep_launches; int64_t kernels_launched; } nd_profile;
nd_status nd_profile_enable(nd_problem* p, int32_t on);   /* 0 off, 1 event timing, 2 event timing + the INSTRUMENTED swath kernel */
/* After sweeps run with nd_profile_enable(p, 2): the share of the swath kernel's warp cycles spent in
 * [0] staging issue (chunk TMA, q-row cp.async), [1] waiting at the barrier before the segment loop, [2] the segment loop,
 * [3] waiting for the q rows and at the barrier behind the loop, [4] the tally flush, [5] between tiles (item fetch, psi in /
 * out).  HOST [6], sums to 1.  The instrumented kernel is a separate build (clock64 marks); its timings are not bench values. */
nd_status nd_sweep_phases_get(nd_problem* p, double* host_out);
nd_status nd_profile_read(nd_problem* p, nd_profile* out);

/* Problem facts: padded sizes and the algorithmic byte / update counts DESIGN.md defines. */
typedef struct {
    int64_t n_segments, n_segments_padded;
    int64_t updates_per_sweep;      /* U = 2*S*P*G */
    int64_t algorithmic_bytes;      /* per sweep: stream + psi in/out + q read + tally write */
    int32_t group_stride;           /* padded groups per region row */
    int32_t sweep_kernel;           /* the ND_SWEEP_* actually selected */
    int32_t n_batches;              /* tiles of the tiled sweep kernels */
    int32_t reserved;
    double mean_regions_per_tile;   /* tiled kernels: distinct regions per tile (flush REDs = this x G per tile)  */
    double mean_segments_per_tile;  /* tiled kernels: segments per tile; segments / regions = the tally re-use rho */
    double lockstep_efficiency;     /* ND_SWEEP_SWATH: segments / (track slots x steps), 1 = no idle slot steps   */
    int32_t block_threads, smem_bytes, grid_blocks, tracks_per_block;
} nd_problem_info;
nd_status nd_problem_info_get(const nd_problem* p, nd_problem_info* out);

/* Diagnostics: where the swath kernel's chunk stream lies in the problem's workspace (DEVICE pointers, valid as long as
 * the problem), whichever builder made it -- the host one (host segments) or the device one (seg_on_device).  Tests copy
 * the arrays back and compare the two builders byte for byte.  ND_ERR_STATE unless the problem runs ND_SWEEP_SWATH. */
typedef struct {
    const void* blob;           /* all chunks (format: csrc/nd_swath.h) */
    size_t blob_bytes;
    const uint32_t* tile_ref;   /* [n_tiles + 1][2] chunk offset, head size (16-byte units); last = end sentinel */
    const int64_t* swath_tile0; /* [n_swaths + 1] */
    const int32_t* swath_track; /* [n_swaths][tracks_per_swath] */
    const int32_t* items;       /* [n_items][4] swath, direction, cost, 0 */
    int64_t n_tiles, n_swaths, n_items;
    int32_t tracks_per_swath, built_on_device;
} nd_stream_device_view_t;
nd_status nd_problem_stream_view(const nd_problem* p, nd_stream_device_view_t* out);

/* ------------------------------------------------------------------------------------------------
 * Diagnostics: the swath/tile chunk stream of ND_SWEEP_SWATH (row A1: "segment stream layout"), built on the
 * HOST exactly as nd_problem_create builds it, for inspection by tests.  Chunk format: csrc/nd_swath.h.
 *   tracks_per_swath NT, tile_segments Kmax (per track and tile), window_regions Lmax (distinct regions per
 *   tile), slots_per_line NC (NT % NC == 0), row_bytes = 4 * padded group count (multiple of 16), lag_segments =
 *   allowed drift of the track fronts, in mean segment lengths, under which tiles give every track equal counts
 *   (< 0: always cut geometrically).
 * All view pointers are HOST memory owned by the stream object, valid until nd_swath_stream_destroy.
 * ---------------------------------------------------------------------------------------------- */
typedef struct nd_swath_stream nd_swath_stream;
typedef struct {
    int64_t n_swaths, n_tiles, blob_bytes, n_items;
    const uint8_t* blob;            /* all chunks, 16-byte aligned each */
    const uint32_t* tile_ref;       /* [n_tiles+1][2] chunk offset, size of the chunk's head part; both in 16-byte units */
    const int64_t* swath_tile0;     /* [n_swaths+1] first tile of every swath */
    const int32_t* swath_track;     /* [n_swaths][NT] track id or -1 */
    const int32_t* items;           /* [n_items][4] swath, direction, cost, 0 -- in the order nd_options.item_order selects */
    double mean_regions_per_tile, mean_segments_per_tile, lockstep_efficiency;
    int32_t max_head_bytes, max_rec_bytes;
} nd_swath_stream_view_t;
nd_status nd_swath_stream_build(const nd_problem_desc* desc, int32_t tracks_per_swath, int32_t tile_segments,
                                int32_t window_regions, int32_t slots_per_line, int32_t row_bytes,
                                double lag_segments, int32_t item_order, nd_swath_stream** out);
nd_status nd_swath_stream_view(const nd_swath_stream* s, nd_swath_stream_view_t* view);
nd_status nd_swath_stream_destroy(nd_swath_stream* s);

/* ------------------------------------------------------------------------------------------------
 * Diagnostics: the micro-benchmarks behind the roofline denominators.  One Eq.-(5) update
 * needs one MUFU.EX2, so n_sm x mufu_ex2_per_clk_per_sm x clock bounds the sweep in updates per second.
 *   device_workspace  DEVICE, 256-byte aligned, >= 64 MiB; the HBM-resident RED case needs >= 1 GiB + 1 MiB (else it is
 *                     reported as 0).  Contents are overwritten.
 * Synchronises the stream.  Takes ~0.1 s.  Errors: ND_ERR_NULL, ND_ERR_WORKSPACE, ND_ERR_CUDA.
 * ---------------------------------------------------------------------------------------------- */
typedef struct {
    double mufu_ex2_per_clk_per_sm; /* ex2.approx.ftz.f32 results per clock per SM, 1024 threads x 8 chains per SM, clock64() */
    double mufu_ex2_per_s;          /* the same, whole device, by CUDA events */
    double sm_clock_mhz;            /* SM clock during the run: clock64() ticks per %globaltimer nanosecond */
    double red_f64_l2_per_s;        /* FP64 RED lane-operations per second, random 256-byte rows of a 32 MiB table */
    double red_f64_hbm_per_s;       /* the same on a 1 GiB table (0 if the workspace is too small) */
    int32_t n_sm, reserved;
} nd_microbench_result;
nd_status nd_microbench(void* device_workspace, size_t device_bytes, void* cuda_stream, nd_microbench_result* out);

/* ------------------------------------------------------------------------------------------------
 * Allocation-free fission rate (row A6: F = sum_r A~_r sum_g nuSigma_f[m(r)][g] phi[r][g], the k_eff update of Eq. (1),
 * PAPER.md:48) for callers that can neither call cudaMalloc nor hand over a workspace (CUDA graph capture, serving loops).
 * Its per-block partial sums live in a file-scope __device__ array of the library: 256 KiB that every GPU that loads
 * libnd_moc.so holds until the process exits.  Same quantity as nd_source_update's d_fission_rate_out (which keeps its
 * partial sums in the problem's workspace); the decomposition is fixed (4096 consecutive elements per partial sum), so the
 * result does not depend on the GPU's SM count.
 *   d_phi [R][G], d_region_material [R] (values in 0..M-1: NOT checked), d_nu_sigma_f [M][G], d_volume [R]: DEVICE, inputs;
 *   d_fission_rate_out: DEVICE, one double.  Stream-ordered, asynchronous; calls no allocating routine.
 * LIMIT: n_regions * n_groups <= ND_STATIC_FISSION_MAX_ELEMENTS, else ND_ERR_RANGE (nothing is launched).
 * SHARED STATE: every call on a device uses the same array, which keeps the last call's partial sums.  Nothing has to be
 * cleared (a call reads only what it wrote), but two calls that OVERLAP on the GPU -- different streams, concurrent graph
 * replays -- race on it: order them on one stream or with events.
 * Errors: ND_ERR_NULL, ND_ERR_INVALID (sizes < 1), ND_ERR_RANGE (limit; device ordinal > 63), ND_ERR_CUDA.
 * ---------------------------------------------------------------------------------------------- */
#define ND_STATIC_FISSION_MAX_ELEMENTS (1ll << 27)
nd_status nd_fission_rate_static(int32_t n_regions, int32_t n_groups, const double* d_phi, const int32_t* d_region_material,
                                 const double* d_nu_sigma_f, const double* d_volume, double* d_fission_rate_out,
                                 void* cuda_stream);

const char* nd_status_string(nd_status s);
/* Message of the last call that failed ON THE CALLING THREAD (thread-local storage, valid until that thread's next failing
 * call).  The argument is accepted for symmetry and ignored: errors of calls that have no problem (nd_tracks_generate,
 * nd_problem_create) are reported the same way. */
const char* nd_last_error(const nd_problem* p_or_null);
uint32_t nd_version(void);
const char* nd_build_id(void); /* short hash of the sources this library was built from (paper_2607_01591_b200/_build.py) */

#ifdef __cplusplus
}
#endif
#endif /* ND_MOC_H */
