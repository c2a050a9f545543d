// nd_sweep_swath.cuh -- row A2, the fast path: Eq. (5) with the angular flux of a track held in
// registers from one end of the track to the other, and the region tallies formed in shared memory.
//
// Why this shape (B200 measurements):
//   * one update = 1 MUFU.EX2 + 5 FP32 ops; the MUFU pipe (16/clk/SM) is the roofline.  A realistic inner loop
//     (records, q row, Sigma_t row read from shared memory, one delta row written) sustains 80 % of it with 16 warps/SM.
//   * FP64 global REDs per (segment, group) are 2.4-4x too slow; shared-memory float atomics are CAS loops.
//     Adjacent parallel tracks (0.01-0.05 cm apart) cross the same triangles, so a block that carries NT adjacent
//     tracks sees every region ~rho = 5-10 times per tile.
//
// Mapping
//   * thread block = one SWATH (NT adjacent tracks of one angle) in one direction; persistent blocks pull
//     (swath, direction) items from an atomic counter, most expensive first.
//   * lane group ("slot") = LPT lanes = one track, slots packed over the lanes of the whole block (19 slots of 13 lanes in
//     256 threads for G = 51: 96 % of the lanes carry chains); a lane owns 4 consecutive groups x P polar angles = 4P
//     independent Eq.-(5) chains in registers (ILP hides the MUFU/FMA latency).  psi is read from the boundary
//     array once, at the track's entry, and written once, at its exit.
//   * the swath is processed tile by tile (nd_swath.h).  A tile's chunk arrives by ONE bulk async (TMA) copy,
//     two tiles ahead (ring of three chunk buffers), signalled on an mbarrier; the q rows of its regions are gathered by 16-byte cp.async one
//     tile ahead.  In the segment loop a lane reads the segment record (broadcast), its 16 bytes of the q row and
//     of the Sigma_t row, and STORES sum_p w_p Delta_p into the segment's own row of the delta buffer: no
//     read-modify-write, no atomics (a segment owns its row).
//   * after a block barrier the tile is flushed: per (region, 4 groups) the rows listed in the chunk's CSR are
//     added up in FP32 and leave as FP64 REDs -- one RED per (region, group) per tile instead of one per segment.
//   * narrow rows (G <= 16): NC slots share a 128-byte line (q, Sigma_t and delta rows replicated / interleaved per
//     slot) so that the 8 lanes of a shared-memory phase always hit distinct banks.
#pragma once
#include "nd_kernels.cuh"

#ifndef ND_FLUSH_UNROLL
#define ND_FLUSH_UNROLL 4
#endif

namespace ndk {

constexpr int kFlushUnroll = ND_FLUSH_UNROLL;

struct SwathParams {
    const uint8_t* __restrict__ blob;
    const uint2* __restrict__ tile_ref;        // [n_tiles+1] (chunk offset, head size) in 16-byte units (+ end sentinel)
    const int64_t* __restrict__ swath_tile0;   // [n_swaths+1]
    const int32_t* __restrict__ swath_track;   // [n_swaths][NT]
    const int4* __restrict__ items;            // (swath, dir, cost, -)
    int* __restrict__ counter;
    const float* __restrict__ q;               // [R][Gs]
    const float* __restrict__ sigt;            // [M][Gs]
    double* __restrict__ tally;                // [R][Gs]
    const float* __restrict__ trk_w;
    const float* __restrict__ psi_in;
    float* __restrict__ psi_out;
    const double* __restrict__ scale_div;
    int n_items, G, Gs, M, NT, Kmax, Lmax, LPT, NC, NCq, ndbuf;
    int head_cap, rec_cap;                     // bytes of one head / record staging buffer
    int off_sigt, off_q, off_dbuf, off_head, off_rec;  // shared-memory byte offsets
    float c[kMaxPolar], inv_sin[kMaxPolar], wp[kMaxPolar];
    unsigned long long c2[kMaxPolar];          // {c[p]/c[0], c[p]/c[0]} packed for the FP32x2 path (the Sigma_t table in shared
                                               // memory is pre-multiplied by c[0] = -log2(e)/sin(theta_0) there)
    uint32_t magic_per_row, magic_nq;          // fastdiv constants of NC*Gs/4 and Gs/4
    uint32_t magic_np;                         // fastdiv constant of Gs/2 (group pairs per row: the flush mapping)
    unsigned long long* phase;                 // PROF builds: [kSwathPhases] warp-cycle sums (lane 0 of every warp)
    // CUR builds (CMFD, C-3 of DESIGN.md 8d): the coarse-surface crossings of every tile and the current tally
    const uint8_t* __restrict__ xblob;         // per tile: u32 {count, 0} then count entries {surface << 1 | forward sign bit,
                                               // slot | position << 16}, padded to 16 bytes
    const uint32_t* __restrict__ xoff;         // [n_tiles+1] offsets into xblob, 16-byte units
    double* __restrict__ J_surf;               // [J_replicas][J_stride]: [n_pairs][G] net currents, positive from the lower to the
                                               // higher cell id.  A block adds into replica blockIdx.x % J_replicas: a coarse mesh has
                                               // few surfaces, and FP64 atomics of all blocks on the same few lines serialise in L2
    long long J_stride;
    int J_replicas;
    int x_cap, off_x, off_w;                   // bytes of one crossing buffer; shared-memory offsets of the ring and of W
    // ---- P_1 scattering source (NEXT-4, template flag P1S): q(Omega) = q0 + sin(theta_p) qB with
    // qB = 3 (u . q1) of the item's direction of travel u, staged as a second row per region; a second delta row per segment
    // carries sum_p w_p sin(theta_p) Delta_p, flushed into the two moment tallies times u_x, u_y ----
    const float* __restrict__ q1x;             // [R][Gs] Q1x / Sigma_t (NULL: isotropic source)
    const float* __restrict__ q1y;             // [R][Gs]
    const float* __restrict__ trk_dir;         // [T][2] unit vector from the start to the end point of a track
    double* __restrict__ tally_x;              // [R][Gs]
    double* __restrict__ tally_y;              // [R][Gs]
    float sin_t[kMaxPolar];                    // sin(theta_p)
    int off_q2, off_dbuf2;                     // shared-memory offsets of the qB rows [2][Lmax][line_q] and of the second delta buffer
};

// phases of the instrumented build (nd_profile_enable(p, 2)): where the warps' cycles go
enum { PH_STAGE = 0, PH_WAIT_A, PH_COMPUTE, PH_WAIT_B, PH_FLUSH, PH_ITEM, kSwathPhases };

constexpr int kSwathHeadBufs = 3;   // heads of tiles k, k+1 (its q rows are staged during tile k) and k+2 (in flight)
constexpr int kSwathRecBufs = 2;    // records of tiles k and k+1 (in flight)
constexpr int kSwathXBufs = 2;      // CUR builds: crossing lists of tiles k and k+1 (in flight)

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// 1-D bulk async copy global -> shared through the TMA unit; completion is signalled on the mbarrier.
__device__ __forceinline__ void tma_load_1d(void* smem_dst, const void* gmem_src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(smem_dst)),
                 "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void cp_async_16(uint32_t smem_dst, const void* gmem_src)
{
#ifdef ND_Q_STAGE_CA
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(smem_dst), "l"(gmem_src) : "memory");
#else
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_dst), "l"(gmem_src) : "memory");
#endif
}
__device__ __forceinline__ void cp_async_8(uint32_t smem_dst, const void* gmem_src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_dst), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit_group() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

struct SwathHead {   // decoded chunk head (pointers into the head staging buffer)
    int L, nseg;
    const uint16_t* slot_start;
    const uint2* regions;      // { region id ; first delta row | one past the last << 16 }
};
__device__ __forceinline__ SwathHead decode_head(const unsigned char* hb)
{
    const uint4 h = *reinterpret_cast<const uint4*>(hb);
    SwathHead c;
    c.L = (int)(h.x & 0xffffu); c.nseg = (int)(h.x >> 16);
    c.slot_start = reinterpret_cast<const uint16_t*>(hb + 16);
    c.regions = reinterpret_cast<const uint2*>(hb + 16 * h.y);
    return c;
}

// ---- packed FP32x2 arithmetic (sm_100: FFMA2 / FADD2 / FMUL2 halve the issue slots of the FP32 work) ----
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float lo, float hi) { f32x2 r; asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void upk2(f32x2 v, float& lo, float& hi) { asm("mov.b64 {%0,%1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) { f32x2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) { f32x2 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) { f32x2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b) { f32x2 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }

// x / d for x < 2^16 and d >= 1, with m = fastdiv_magic(d); m == 0 encodes d == 1
__host__ __device__ inline uint32_t fastdiv_magic(uint32_t d) { return d <= 1 ? 0u : (uint32_t)((0x100000000ull + d - 1) / d); }
__device__ __forceinline__ uint32_t fastdiv(uint32_t x, uint32_t m) { return m ? __umulhi(x, m) : x; }

// shared-memory accesses by 32-bit shared-space address (no generic-address conversion in the loop)
__device__ __forceinline__ uint4 lds_u4(uint32_t a)
{
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a));
    return v;
}
__device__ __forceinline__ uint2 lds_u2(uint32_t a)
{
    uint2 v;
    asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ ulonglong2 lds_2x64(uint32_t a)
{
    ulonglong2 v;
    asm volatile("ld.shared.v2.u64 {%0,%1}, [%2];" : "=l"(v.x), "=l"(v.y) : "r"(a));
    return v;
}
__device__ __forceinline__ float4 lds_f4(uint32_t a)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
    return v;
}
__device__ __forceinline__ void sts_2x64(uint32_t a, unsigned long long x, unsigned long long y)
{
    asm volatile("st.shared.v2.u64 [%0], {%1,%2};" ::"r"(a), "l"(x), "l"(y) : "memory");
}
__device__ __forceinline__ void sts_f4(uint32_t a, float x, float y, float z, float w)
{
    asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};" ::"r"(a), "f"(x), "f"(y), "f"(z), "f"(w) : "memory");
}

// One track through one tile: cnt segments starting at the record at shared address rec0 (stepping rstep = +-16 bytes),
// `steps` >= cnt loop trips (slots of a warp run in lock step).  Trips past cnt read the block's NULL RECORD at `null_rec`:
// zero length (exp = 1, Delta = 0: an exact no-op for psi), row offsets 0, and a delta row that no region owns, so the
// loop body carries no predicate.  A record holds the byte offsets of its q row, its Sigma_t row and its delta row: one
// add per access.  Software pipeline: the record of step i+2 and the q / Sigma_t rows of step i+1 are loaded during step i.
template <int P, int EXPM>
__device__ __forceinline__ void segment_loop(float (&psi)[P][4], const float (&wpt)[P], const SwathParams& prm, uint32_t rec0,
                                             int rstep, int cnt, int steps, uint32_t null_rec, uint32_t q_lane,
                                             uint32_t sigt_lane, uint32_t d_lane)
{
    const uint4 r_n = lds_u4(cnt > 0 ? rec0 : null_rec);
    uint4 r_nn = lds_u4(cnt > 1 ? rec0 + rstep : null_rec);
    uint32_t rec_pf = rec0 + 2 * rstep;       // record of step i+2
    uint32_t d_n = r_n.w;
    if (EXPM == 0) {
        f32x2 ps[P][2], w2[P];
#pragma unroll
        for (int p = 0; p < P; ++p) {
            ps[p][0] = pk2(psi[p][0], psi[p][1]);
            ps[p][1] = pk2(psi[p][2], psi[p][3]);
            w2[p] = pk2(wpt[p], wpt[p]);
        }
        ulonglong2 q_n = lds_2x64(q_lane + r_n.y);
        ulonglong2 st_n = lds_2x64(sigt_lane + r_n.z);
        float s_n = __uint_as_float(r_n.x);
        // the 4 P updates of one step and the store of sum_p w_p Delta_p into the segment's delta row
        auto update = [&](const f32x2 (&qa)[2], const f32x2 (&ts)[2], uint32_t d_cur) {
            f32x2 acc[2];
#pragma unroll
            for (int j = 0; j < 2; ++j) {
#pragma unroll
                for (int p = 0; p < P; ++p) {
                    const f32x2 tau = p == 0 ? ts[j] : mul2(ts[j], prm.c2[p]);
                    float t0, t1;
                    upk2(tau, t0, t1);
                    const f32x2 a = pk2(ex2_approx(t0), ex2_approx(t1));
                    const f32x2 d = sub2(ps[p][j], qa[j]);
                    const f32x2 delta = sub2(d, mul2(d, a));      // d*(1-a); contracts to one FFMA2
                    ps[p][j] = sub2(ps[p][j], delta);
                    acc[j] = p == 0 ? mul2(w2[0], delta) : fma2(w2[p], delta, acc[j]);
                }
            }
            sts_2x64(d_lane + d_cur, acc[0], acc[1]);
        };
        // (A peeled last trip without the loads for a step that does not exist measured +-0.1 %: not kept.  Carrying
        // W = sum_p w_p psi_p and storing W_before - W_behind -- two packed operations per (pair, polar angle) instead of
        // three -- measured 1.4 % slower and costs the small Deltas their relative accuracy: not kept.  Carrying the chains as
        // D_p = psi_p - q, D'_p = fma(D_p, a_p, q - q'), sum_p w_p Delta_p = WD - WD' + (q - q') sum_p w_p -- 49.5 instead of 54
        // instructions per step, every parity test green -- measured 5.4 % SLOWER at config 5: the loop is bound by the
        // dependent chains behind each MUFU.EX2, not by its instruction count.  Skipping the Sigma_t load when the material
        // is the one of the previous segment -- 94 % of the segments at config 4, 12 % at config 5 -- measured -0.4 % at
        // config 4, -1.5 % at config 3 and +3.1 % at config 5: not kept.)
        for (int i = 0; i < steps; ++i) {
            const f32x2 s2 = pk2(s_n, s_n);
            const f32x2 qa[2] = {q_n.x, q_n.y};
            const f32x2 ts[2] = {mul2(st_n.x, s2), mul2(st_n.y, s2)};   // Sigma_t * c_0 * s = log2 of the first polar angle's attenuation
            const uint32_t d_cur = d_n;
            const uint4 r_use = r_nn;
            r_nn = lds_u4(i + 2 < cnt ? rec_pf : null_rec);
            rec_pf += rstep;
            q_n = lds_2x64(q_lane + r_use.y);
            st_n = lds_2x64(sigt_lane + r_use.z);
            s_n = __uint_as_float(r_use.x);
            d_n = r_use.w;
            update(qa, ts, d_cur);
        }
#pragma unroll
        for (int p = 0; p < P; ++p) {
            upk2(ps[p][0], psi[p][0], psi[p][1]);
            upk2(ps[p][1], psi[p][2], psi[p][3]);
        }
    } else {
        float4 q_n = lds_f4(q_lane + r_n.y);
        float4 st_n = lds_f4(sigt_lane + r_n.z);
        float s_n = __uint_as_float(r_n.x);
        for (int i = 0; i < steps; ++i) {
            const float sl = s_n;
            const float4 qv = q_n, stv = st_n;
            const uint32_t d_cur = d_n;
            const uint4 r_use = r_nn;
            r_nn = lds_u4(i + 2 < cnt ? rec_pf : null_rec);
            rec_pf += rstep;
            q_n = lds_f4(q_lane + r_use.y);
            st_n = lds_f4(sigt_lane + r_use.z);
            s_n = __uint_as_float(r_use.x);
            d_n = r_use.w;
            const float qa[4] = {qv.x, qv.y, qv.z, qv.w}, sa[4] = {stv.x, stv.y, stv.z, stv.w};
            float a4[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                float acc = 0.f;
#pragma unroll
                for (int p = 0; p < P; ++p) {
                    const float d = psi[p][j] - qa[j];
                    const float delta = d * (-expm1f(-(sa[j] * sl) * prm.inv_sin[p]));
                    psi[p][j] -= delta;
                    acc = fmaf(wpt[p], delta, acc);
                }
                a4[j] = acc;
            }
            sts_f4(d_lane + d_cur, a4[0], a4[1], a4[2], a4[3]);
        }
    }
}

// The same loop with the P_1 source (P1S): the chain of polar angle p sees q0 + sin(theta_p) qB, qB = 3 (u . q1) staged as a
// second row per region at the same offsets, and a second delta row per segment takes sum_p w_p sin(theta_p) Delta_p (P-1..P-4
// of DESIGN.md 8e).  The null record reads row 0 of both buffers with zero length: an exact no-op, as above.
template <int P>
__device__ __forceinline__ void segment_loop_p1(float (&psi)[P][4], const float (&wpt)[P], const SwathParams& prm, uint32_t rec0,
                                                int rstep, int cnt, int steps, uint32_t null_rec, uint32_t q_lane, uint32_t q2_lane,
                                                uint32_t sigt_lane, uint32_t d_lane, uint32_t d2_lane)
{
    const uint4 r_n = lds_u4(cnt > 0 ? rec0 : null_rec);
    uint4 r_nn = lds_u4(cnt > 1 ? rec0 + rstep : null_rec);
    uint32_t rec_pf = rec0 + 2 * rstep;
    uint32_t d_n = r_n.w;
    f32x2 ps[P][2], w2[P], w2s[P], sin2[P];
#pragma unroll
    for (int p = 0; p < P; ++p) {
        ps[p][0] = pk2(psi[p][0], psi[p][1]);
        ps[p][1] = pk2(psi[p][2], psi[p][3]);
        w2[p] = pk2(wpt[p], wpt[p]);
        w2s[p] = pk2(wpt[p] * prm.sin_t[p], wpt[p] * prm.sin_t[p]);
        sin2[p] = pk2(prm.sin_t[p], prm.sin_t[p]);
    }
    ulonglong2 q_n = lds_2x64(q_lane + r_n.y);
    ulonglong2 qb_n = lds_2x64(q2_lane + r_n.y);
    ulonglong2 st_n = lds_2x64(sigt_lane + r_n.z);
    float s_n = __uint_as_float(r_n.x);
    for (int i = 0; i < steps; ++i) {
        const f32x2 s2 = pk2(s_n, s_n);
        const f32x2 qa[2] = {q_n.x, q_n.y}, qb[2] = {qb_n.x, qb_n.y};
        const f32x2 ts[2] = {mul2(st_n.x, s2), mul2(st_n.y, s2)};
        const uint32_t d_cur = d_n;
        const uint4 r_use = r_nn;
        r_nn = lds_u4(i + 2 < cnt ? rec_pf : null_rec);
        rec_pf += rstep;
        q_n = lds_2x64(q_lane + r_use.y);
        qb_n = lds_2x64(q2_lane + r_use.y);
        st_n = lds_2x64(sigt_lane + r_use.z);
        s_n = __uint_as_float(r_use.x);
        d_n = r_use.w;
        f32x2 acc[2], acc1[2];
#pragma unroll
        for (int j = 0; j < 2; ++j) {
#pragma unroll
            for (int p = 0; p < P; ++p) {
                const f32x2 tau = p == 0 ? ts[j] : mul2(ts[j], prm.c2[p]);
                float t0, t1;
                upk2(tau, t0, t1);
                const f32x2 a = pk2(ex2_approx(t0), ex2_approx(t1));
                const f32x2 d = sub2(ps[p][j], fma2(sin2[p], qb[j], qa[j]));
                const f32x2 delta = sub2(d, mul2(d, a));
                ps[p][j] = sub2(ps[p][j], delta);
                acc[j] = p == 0 ? mul2(w2[0], delta) : fma2(w2[p], delta, acc[j]);
                acc1[j] = p == 0 ? mul2(w2s[0], delta) : fma2(w2s[p], delta, acc1[j]);
            }
        }
        sts_2x64(d_lane + d_cur, acc[0], acc[1]);
        sts_2x64(d2_lane + d_cur, acc1[0], acc1[1]);
    }
#pragma unroll
    for (int p = 0; p < P; ++p) {
        upk2(ps[p][0], psi[p][0], psi[p][1]);
        upk2(ps[p][1], psi[p][2], psi[p][3]);
    }
}

// TIGHT = 1 caps the registers at 85 (768 resident threads per SM: three 256-thread or two 384-thread blocks).
// CUR = 1 also tallies the net currents through the surfaces of a coarse mesh (CMFD, C-3 of DESIGN.md 8d) WITHOUT touching the
// segment loop: with W = sum_p w_p psi_p, a delta row is W before its segment minus W behind it, so W at a crossing is W at
// the tile's entry (stored per slot before the loop) minus the delta rows of the slot's segments passed so far.
template <int P, int EXPM, int TIGHT, int PROF, int CUR = 0, int P1S = 0>
__global__ void __launch_bounds__(TIGHT ? 384 : 512, TIGHT ? 2 : 1) k_sweep_swath(const SwathParams prm)
{
    static_assert(!P1S || (EXPM == 0 && TIGHT == 0 && PROF == 0 && CUR == 0), "the P_1 variant exists for the plain fast-exp roomy kernel");
    long long ph[kSwathPhases] = {0, 0, 0, 0, 0, 0};
    long long t_mark = PROF ? clock64() : 0;
    int prof_sink = 0;
    auto mark = [&](int phase) {   // PROF: charge the cycles since the last mark to `phase`
        if (PROF) { const long long now = clock64(); ph[phase] += now - t_mark; t_mark = now; }
    };
    extern __shared__ __align__(128) unsigned char smem_sw[];
    unsigned char* const smem = smem_sw;
    uint64_t* hfull = reinterpret_cast<uint64_t*>(smem);             // [kSwathHeadBufs] head-arrival barriers
    uint64_t* rfull = hfull + kSwathHeadBufs;                        // [kSwathRecBufs] record-arrival barriers
    uint64_t* xfull = reinterpret_cast<uint64_t*>(smem + 96);        // [kSwathXBufs] crossing-list barriers (CUR)
    volatile int* s_item = reinterpret_cast<volatile int*>(smem + 64);
    const uint32_t s_pref = smem_u32(smem + 40);                     // [3] x 8 bytes: prefetched tile references (one thread's)
    uint32_t* s_null = reinterpret_cast<uint32_t*>(smem + 80);       // the null record: { 0.0f, 0, 0, offset of the spare delta row }
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int Gs = prm.Gs, row_bytes = 4 * Gs, line = prm.NC * row_bytes;
    const int line_q = TIGHT ? line : prm.NCq * row_bytes;   // the capped variant is only used with NCq == NC
    unsigned char* sigt_s = smem + prm.off_sigt;
    unsigned char* q_s = smem + prm.off_q;           // [2][Lmax][line_q]
    unsigned char* dbuf_s = smem + prm.off_dbuf;     // [ndbuf][NT * Kmax][row_bytes], rows region-major per tile
    unsigned char* head_s = smem + prm.off_head;     // [kSwathHeadBufs][head_cap]
    unsigned char* rec_s = smem + prm.off_rec;       // [kSwathRecBufs][rec_cap]
    const int q_buf_bytes = prm.Lmax * line_q;
    const int dbuf_bytes = (prm.NT * prm.Kmax + 1) * row_bytes;   // one spare row behind the tile's rows: the null record's
    const int nq = Gs >> 2;                          // 16-byte pieces per row

    if (tid == 0) {
        for (int i = 0; i < kSwathHeadBufs + kSwathRecBufs; ++i) mbar_init(hfull + i, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        s_null[0] = 0u; s_null[1] = 0u; s_null[2] = 0u; s_null[3] = (uint32_t)(prm.NT * prm.Kmax * row_bytes);
        if (CUR) {
            for (int i = 0; i < kSwathXBufs; ++i) mbar_init(xfull + i, 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
    }
    // Sigma_t table, replicated NC times per line; the fast-exp path keeps it pre-multiplied by -log2(e)/sin(theta_0)
    {
        const float pre = EXPM == 0 ? prm.c[0] : 1.f;
        for (int i = tid; i < prm.M * prm.NC * nq; i += nthr) {
            const int m = i / (prm.NC * nq), rem = i - m * (prm.NC * nq), piece = rem % nq;
            float4 v = *reinterpret_cast<const float4*>(prm.sigt + (size_t)m * Gs + piece * 4);
            v.x *= pre; v.y *= pre; v.z *= pre; v.w *= pre;
            *reinterpret_cast<float4*>(sigt_s + (size_t)m * line + rem * 16) = v;
        }
    }
    __syncthreads();

    // ---- slot geometry ----
    // Slots are packed over the lanes of the whole BLOCK (slot = tid / LPT), so a slot may straddle two warps: lanes only
    // share read-only records, and every lane runs its warp's maximum trip count with its own slot's segment count.
    // Lanes beyond the last slot are SHADOWS of the last slot's last lane: same shared-memory addresses (a broadcast,
    // no extra bank conflict), no stores.
    int slot = tid / prm.LPT, ll = tid - slot * prm.LPT;
    const bool lane_ok = slot < prm.NT;
    if (!lane_ok) { slot = prm.NT - 1; ll = prm.LPT - 1; }
    const int sub = slot % prm.NC;                    // position of the slot inside a Sigma_t line
    const uint32_t sigt_lane = smem_u32(sigt_s) + sub * row_bytes + ll * 16;
    const uint32_t null_rec = smem_u32(s_null);
    const int lane_off_q = TIGHT ? sub * row_bytes + ll * 16 : (slot % prm.NCq) * row_bytes + ll * 16;
    const float inv_f = (float)(1.0 / *prm.scale_div);
    const int g0 = ll * 4;
    const int f_np = Gs >> 1;                         // pairs of groups per row: the unit of the flush

    uint32_t seq = 0;   // tiles processed by this block so far: staging buffers and barrier parities follow it
    for (;;) {
        if (tid == 0) *s_item = atomicAdd(prm.counter, 1);
        __syncthreads();
        const int item = *s_item;
        if (item >= prm.n_items) break;
        const int4 it = prm.items[item];
        const int sw = it.x, dir = it.y;
        float ux = 0.f, uy = 0.f;   // P1S: direction of travel of the item (all tracks of a swath share their angle)
        if (P1S) {
            const int t0 = prm.swath_track[(size_t)sw * prm.NT];
            const float sgn = dir == 0 ? 1.f : -1.f;
            ux = sgn * prm.trk_dir[2 * (size_t)t0]; uy = sgn * prm.trk_dir[2 * (size_t)t0 + 1];
        }
        const int64_t tile0 = prm.swath_tile0[sw];
        const int nt = (int)(prm.swath_tile0[sw + 1] - tile0);
        // ---- this slot's track: psi enters the registers ----
        const int t = prm.swath_track[(size_t)sw * prm.NT + slot];
        float psi[P][4], wpt[P];
        size_t psi_at = 0;
#pragma unroll
        for (int p = 0; p < P; ++p) {
            wpt[p] = 0.f;
#pragma unroll
            for (int j = 0; j < 4; ++j) psi[p][j] = 0.f;
        }
        if (t >= 0) {
            psi_at = ((size_t)(2 * t + dir) * P) * Gs + g0;
            const float wt = prm.trk_w[t];
#pragma unroll
            for (int p = 0; p < P; ++p) {
                const float4 v = *reinterpret_cast<const float4*>(prm.psi_in + psi_at + (size_t)p * Gs);
                psi[p][0] = v.x * inv_f; psi[p][1] = v.y * inv_f; psi[p][2] = v.z * inv_f; psi[p][3] = v.w * inv_f;
                wpt[p] = wt * prm.wp[p];
            }
        }
        // ---- prologue: head and records of the first tile and the head of the second in flight, q rows of the first tile ----
        auto tile_index = [&](int k) -> int64_t { return tile0 + (dir ? nt - 1 - k : k); };
        auto issue_head = [&](int k) {   // one thread
            const uint2 ref = prm.tile_ref[tile_index(k)];
            const uint32_t b = (seq + k) % kSwathHeadBufs;
            mbar_expect_tx(hfull + b, ref.y * 16u);
            tma_load_1d(head_s + (size_t)b * prm.head_cap, prm.blob + (size_t)ref.x * 16, ref.y * 16u, hfull + b);
        };
        auto issue_rec = [&](int k) {    // one thread
            const int64_t ti = tile_index(k);
            const uint2 ref = prm.tile_ref[ti];
            const uint32_t bytes = (prm.tile_ref[ti + 1].x - ref.x - ref.y) * 16u;
            const uint32_t b = (seq + k) % kSwathRecBufs;
            mbar_expect_tx(rfull + b, bytes);
            tma_load_1d(rec_s + (size_t)b * prm.rec_cap, prm.blob + ((size_t)ref.x + ref.y) * 16, bytes, rfull + b);
        };
        // The tile references the issuing thread needs at tile k -- of the head of tile k+2 and of the records of tile k+1 --
        // are fetched one tile ahead by three 8-byte cp.async into s_pref (no register lives across the segment loop), so the
        // issuing thread's warp does not enter its loop two dependent global loads behind the others.  Used by the roomy
        // variant (TIGHT = 0; config 3 -1.2 %); the register-capped one measured +-0.2 % and keeps the direct loads.
        auto prefetch_refs = [&](int k) {   // one thread: what tile k will consume
            if (k + 2 < nt) cp_async_8(s_pref, prm.tile_ref + tile_index(k + 2));
            if (k + 1 < nt) {
                const int64_t ti = tile_index(k + 1);
                cp_async_8(s_pref + 8, prm.tile_ref + ti);
                cp_async_8(s_pref + 16, prm.tile_ref + ti + 1);
            }
        };
        auto issue_head_pref = [&](int k) {   // one thread, k = current tile + 2
            const uint2 ref = lds_u2(s_pref);
            const uint32_t b = (seq + k) % kSwathHeadBufs;
            mbar_expect_tx(hfull + b, ref.y * 16u);
            tma_load_1d(head_s + (size_t)b * prm.head_cap, prm.blob + (size_t)ref.x * 16, ref.y * 16u, hfull + b);
        };
        auto issue_rec_pref = [&](int k) {    // one thread, k = current tile + 1
            const uint2 ref = lds_u2(s_pref + 8);
            const uint32_t bytes = (lds_u2(s_pref + 16).x - ref.x - ref.y) * 16u;
            const uint32_t b = (seq + k) % kSwathRecBufs;
            mbar_expect_tx(rfull + b, bytes);
            tma_load_1d(rec_s + (size_t)b * prm.rec_cap, prm.blob + ((size_t)ref.x + ref.y) * 16, bytes, rfull + b);
        };
        auto wait_head = [&](int k) {
            const uint32_t s = seq + k;
            mbar_wait(hfull + (s % kSwathHeadBufs), (s / kSwathHeadBufs) & 1u);
        };
        auto wait_rec = [&](int k) {
            const uint32_t s = seq + k;
            mbar_wait(rfull + (s % kSwathRecBufs), (s / kSwathRecBufs) & 1u);
        };
        auto issue_x = [&](int k) {      // one thread (CUR): the crossing list of tile k
            const int64_t ti = tile_index(k);
            const uint32_t o0 = prm.xoff[ti], bytes = (prm.xoff[ti + 1] - o0) * 16u;
            const uint32_t b = (seq + k) % kSwathXBufs;
            mbar_expect_tx(xfull + b, bytes);
            tma_load_1d(smem + prm.off_x + (size_t)b * prm.x_cap, prm.xblob + (size_t)o0 * 16, bytes, xfull + b);
        };
        auto issue_q_rows = [&](int k) {   // all threads: regions of tile k -> q buffer (seq+k)&1, NCq copies per row
            const uint32_t s = seq + k;
            const unsigned char* hb = head_s + (size_t)(s % kSwathHeadBufs) * prm.head_cap;
            const uint4 h = *reinterpret_cast<const uint4*>(hb);
            const int L = (int)(h.x & 0xffffu);
            const uint2* regions = reinterpret_cast<const uint2*>(hb + 16 * h.y);
            const uint32_t qb = smem_u32(q_s + (size_t)(s & 1u) * q_buf_bytes);
            const int per_row = (TIGHT ? prm.NC : prm.NCq) * nq;
            // (One 1-D bulk copy per region through the TMA unit instead -- no LSU wavefronts, no index arithmetic -- measured
            // 4.8 % SLOWER at config 5 and 6.5 % at config 4: thirty 208-byte bulk copies per tile cost more than 390 cp.async.)
            for (int i = tid; i < L * per_row; i += nthr) {
                const int l = (int)fastdiv((uint32_t)i, prm.magic_per_row), rem = i - l * per_row;
                const int piece = rem - (int)fastdiv((uint32_t)rem, prm.magic_nq) * nq;
                cp_async_16(qb + l * line_q + rem * 16, prm.q + (size_t)regions[l].x * Gs + piece * 4);
                if (P1S) {   // qB = 3 (u . q1): plain loads a tile ahead, stored beside the q0 row (same offsets in the second buffer)
                    const size_t at = (size_t)regions[l].x * Gs + piece * 4;
                    const float4 a = *reinterpret_cast<const float4*>(prm.q1x + at), b = *reinterpret_cast<const float4*>(prm.q1y + at);
                    sts_f4(smem_u32(smem + prm.off_q2) + (s & 1u) * q_buf_bytes + l * line_q + rem * 16, 3.f * fmaf(ux, a.x, uy * b.x),
                           3.f * fmaf(ux, a.y, uy * b.y), 3.f * fmaf(ux, a.z, uy * b.z), 3.f * fmaf(ux, a.w, uy * b.w));
                }
            }
        };
        if (nt > 0) {
            if (tid == 0) {
                issue_head(0);
                issue_rec(0);
                if (nt > 1) issue_head(1);
                if (CUR) issue_x(0);
                if (!TIGHT) prefetch_refs(0);   // lands before the cp_async_wait_all below
            }
            wait_head(0);
            issue_q_rows(0);
            cp_async_commit_group();
            cp_async_wait_all();
        }
        __syncthreads();

        for (int k = 0; k < nt; ++k) {
            mark(PH_ITEM);
            const uint32_t s = seq + k;
            const unsigned char* hb = head_s + (size_t)(s % kSwathHeadBufs) * prm.head_cap;
            // ---- stage ahead: q rows of tile k+1 (its head landed a tile ago) ----
            if (k + 1 < nt) {
                wait_head(k + 1);
                issue_q_rows(k + 1);
            }
            cp_async_commit_group();
            mark(PH_STAGE);
            // Behind this barrier every thread is past the flush of tile k-1: its head buffer takes the head of tile k+2, its
            // record buffer (free since the loop of tile k-1) the records of tile k+1, and its delta rows may be overwritten.
            __syncthreads();
            if (tid == 0) {
                if (!TIGHT) {
                    if (k + 2 < nt) issue_head_pref(k + 2);
                    if (k + 1 < nt) issue_rec_pref(k + 1);
                    if (CUR && k + 1 < nt) issue_x(k + 1);
                    prefetch_refs(k + 1);   // into the slots just read; complete at this thread's cp_async_wait_all behind the loop
                    cp_async_commit_group();
                } else {
                    if (k + 2 < nt) issue_head(k + 2);
                    if (k + 1 < nt) issue_rec(k + 1);
                    if (CUR && k + 1 < nt) issue_x(k + 1);
                }
            }
            wait_rec(k);
            if (PROF) prof_sink += *s_item;        // BAR.SYNC defers its blocking to the next consumer: make one here
            mark(PH_WAIT_A);
            const SwathHead ch = decode_head(hb);
            unsigned char* dbuf = dbuf_s + (size_t)(prm.ndbuf == 1 ? 0u : (s & 1u)) * dbuf_bytes;
            if (CUR) {   // W = sum_p w_p psi_p of this slot at the tile's entry (the previous tile's flush is over: barrier above)
                float wv[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    float a = 0.f;
#pragma unroll
                    for (int p = 0; p < P; ++p) a = fmaf(wpt[p], psi[p][j], a);
                    wv[j] = a;
                }
                sts_f4(smem_u32(smem + prm.off_w) + slot * row_bytes + ll * 16, wv[0], wv[1], wv[2], wv[3]);
            }
            // ---- segment loop of this slot's track through the tile ----
            {
                int s0 = 0, cnt = 0;
                if (t >= 0) { s0 = ch.slot_start[slot]; cnt = ch.slot_start[slot + 1] - s0; }
                const int steps = __reduce_max_sync(0xffffffffu, cnt);
                const uint32_t q_lane = smem_u32(q_s) + (s & 1u) * q_buf_bytes + lane_off_q;
                const uint32_t rec = smem_u32(rec_s) + (s % kSwathRecBufs) * prm.rec_cap;
                // segment j (forward index inside the tile) is visited at step i: j = dir ? cnt-1-i : i.  Shadow lanes carry
                // their slot's chains too and store the same values to the same rows.
                const int j_c = dir ? cnt - 1 : 0;          // segment of the first step
                if (P1S)
                    segment_loop_p1<P>(psi, wpt, prm, rec + 16 * (s0 + j_c), dir ? -16 : 16, cnt, steps, null_rec, q_lane,
                                       q_lane + (uint32_t)(prm.off_q2 - prm.off_q), sigt_lane, smem_u32(dbuf) + ll * 16,
                                       smem_u32(dbuf) + (uint32_t)(prm.off_dbuf2 - prm.off_dbuf) + ll * 16);
                else
                    segment_loop<P, EXPM>(psi, wpt, prm, rec + 16 * (s0 + j_c), dir ? -16 : 16, cnt, steps, null_rec, q_lane, sigt_lane,
                                          smem_u32(dbuf) + ll * 16);
            }
            mark(PH_COMPUTE);
            cp_async_wait_all();   // this thread's q-row copies for tile k+1
            __syncthreads();
            if (PROF) prof_sink += *s_item;
            mark(PH_WAIT_B);
            // ---- flush: one FP64 RED per (region, group) of the tile.  A thread owns a pair of groups of one region, pairs
            // fastest: the lanes of a warp read consecutive 8-byte pieces of the region's contiguous delta rows and their REDs
            // fall on consecutive doubles of the tally row (2-3 lines per instruction); the rows are added with packed FADD2.
            // (Same-box A/B of other mappings, config 5, against 52.7 ms: a unit of (region, 4 groups) with LDS.128 and four REDs
            // 58.9 ms; lanes trading sums by shuffles so that a RED instruction covers 32 consecutive doubles 57.0 ms.  Flushing region by region -- a warp per
            // 32 / LPT regions, 16 bytes per lane, odd rounds dealt in reverse -- is free of bank conflicts and 40 % shorter in
            // instructions, and measured 3.3 % SLOWER at configs 5 and 4: its FP64 REDs fall one per 32-byte sector and
            // instruction instead of two, and the warps of a block no longer reach the next barrier together.  A thread that keeps
            // one pair of groups for the whole kernel and walks the regions nthr / f_np apart -- no division in this loop --
            // measured 0.7 % slower.)
            auto flush_unit = [&](int u) {
                const int l = (int)__umulhi((uint32_t)u, prm.magic_np), gp = u - l * f_np;   // f_np >= 2: the magic is never 0
                const uint2 rg = ch.regions[l];
                const int e0 = (int)(rg.y & 0xffffu), e1 = (int)(rg.y >> 16);
                uint32_t row = smem_u32(dbuf) + e0 * row_bytes + gp * 8;
                f32x2 axy = 0ull;
#pragma unroll kFlushUnroll
                for (int e = e0; e < e1; ++e, row += row_bytes) {
                    f32x2 x;
                    asm volatile("ld.shared.b64 %0, [%1];" : "=l"(x) : "r"(row));
                    axy = add2(axy, x);
                }
                float vx, vy;
                upk2(axy, vx, vy);
                // The tally rows are padded to Gs doubles and nothing reads the pad entries: no bound check, 32-bit index
                // (R Gs <= 2^32).  Without the two branches and the 64-bit index arithmetic: config 5 54.94 -> 52.72 ms.
                double* tp = prm.tally + (uint32_t)(rg.x * (uint32_t)Gs + (uint32_t)(gp * 2));
                atomicAdd(tp, (double)vx);
                atomicAdd(tp + 1, (double)vy);
                if (P1S) {   // the second delta rows: sum_p w_p sin(theta_p) Delta_p, times the direction of travel (P-4)
                    uint32_t row2 = smem_u32(dbuf) + (uint32_t)(prm.off_dbuf2 - prm.off_dbuf) + e0 * row_bytes + gp * 8;
                    f32x2 bxy = 0ull;
                    for (int e = e0; e < e1; ++e, row2 += row_bytes) {
                        f32x2 x;
                        asm volatile("ld.shared.b64 %0, [%1];" : "=l"(x) : "r"(row2));
                        bxy = add2(bxy, x);
                    }
                    float bx, by;
                    upk2(bxy, bx, by);
                    const uint32_t idx = rg.x * (uint32_t)Gs + (uint32_t)(gp * 2);
                    atomicAdd(prm.tally_x + idx, (double)(ux * bx));
                    atomicAdd(prm.tally_x + idx + 1, (double)(ux * by));
                    atomicAdd(prm.tally_y + idx, (double)(uy * bx));
                    atomicAdd(prm.tally_y + idx + 1, (double)(uy * by));
                }
            };
            if (TIGHT) {
                for (int u = tid; u < ch.L * f_np; u += nthr) flush_unit(u);
            } else {
                // The regions are listed by descending row count, so in every pass the low threads hold the long lists: odd
                // passes deal the units in reverse and the warps' sums over the passes come out level.  Worth 2.8 % where the
                // flush is a large share (narrow rows, config 3); with 13 lanes per slot the extra index arithmetic costs
                // more than the balance gains (config 5 +2.8 %), so the register-capped variant keeps the plain order.
                const int f_nu = ch.L * f_np;
                for (int base = 0, odd = 0; base < f_nu; base += nthr, odd ^= 1) {
                    const int u = base + (odd ? nthr - 1 - tid : tid);
                    if (u < f_nu) flush_unit(u);
                }
            }
            if (CUR) {
                // ---- currents: thread -> (crossing, pair of groups).  W at the crossing = W at the slot's entry minus the delta
                // rows of the segments the chain has passed: positions 0..pos forward, pos+1..cnt-1 backward. ----
                mbar_wait(xfull + (s % kSwathXBufs), (s / kSwathXBufs) & 1u);
                const uint2* xl = reinterpret_cast<const uint2*>(smem + prm.off_x + (size_t)(s % kSwathXBufs) * prm.x_cap);
                const int nx = (int)xl[0].x;
                const uint32_t rec_b = smem_u32(rec_s) + (s % kSwathRecBufs) * prm.rec_cap + 12;   // delta offset of record 0
                const uint32_t w_b = smem_u32(smem + prm.off_w);
                for (int u = tid; u < nx * f_np; u += nthr) {
                    const int c = (int)fastdiv((uint32_t)u, prm.magic_np), gp = u - c * f_np;
                    const uint2 xe = xl[1 + c];
                    const int xs = (int)(xe.y & 0xffffu), pos = (int)(xe.y >> 16);
                    const int s0 = ch.slot_start[xs], cnt = ch.slot_start[xs + 1] - s0;
                    const int j0 = dir ? pos + 1 : 0, j1 = dir ? cnt : pos + 1;
                    float wx, wy;
                    asm volatile("ld.shared.v2.f32 {%0,%1}, [%2];" : "=f"(wx), "=f"(wy) : "r"(w_b + xs * row_bytes + gp * 8));
                    for (int j = j0; j < j1; ++j) {
                        uint32_t off;
                        asm volatile("ld.shared.u32 %0, [%1];" : "=r"(off) : "r"(rec_b + 16 * (s0 + j)));
                        float x, y;
                        asm volatile("ld.shared.v2.f32 {%0,%1}, [%2];" : "=f"(x), "=f"(y) : "r"(smem_u32(dbuf) + off + gp * 8));
                        wx -= x; wy -= y;
                    }
                    const bool neg = ((xe.x & 1u) != 0u) != (dir != 0);      // forward sign bit, reversed for the backward chain
                    double* jp = prm.J_surf + (size_t)(blockIdx.x % prm.J_replicas) * prm.J_stride + (size_t)(xe.x >> 1) * prm.G + gp * 2;
                    if (gp * 2 < prm.G) atomicAdd(jp, (double)(neg ? -wx : wx));
                    if (gp * 2 + 1 < prm.G) atomicAdd(jp + 1, (double)(neg ? -wy : wy));
                }
            }
            mark(PH_FLUSH);
        }
        seq += (uint32_t)nt;
        // ---- psi leaves the registers ----
        if (t >= 0 && lane_ok) {
#pragma unroll
            for (int p = 0; p < P; ++p)
                *reinterpret_cast<float4*>(prm.psi_out + psi_at + (size_t)p * Gs) = make_float4(psi[p][0], psi[p][1], psi[p][2], psi[p][3]);
        }
        __syncthreads();   // s_item may be rewritten; the last flush is over before the next item's staging
    }
    if (PROF) {
        mark(PH_ITEM);
        if (prof_sink == 0x7fffffff) prm.phase[kSwathPhases] = 1ull;   // keeps the sink alive
        if ((tid & 31) == 0)
            for (int i = 0; i < kSwathPhases; ++i) atomicAdd(prm.phase + i, (unsigned long long)ph[i]);
    }
}

} // namespace ndk
