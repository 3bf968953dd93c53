// Transport, scoring and statistics kernels (sm_100a).  Tracks live in per-warp pools in shared memory; per
// iteration a warp runs ONE block on up to 32 tracks that are in the state the block serves.
//   electron_kernel : Class II condensed-history steps, d = min[d_vox, d_maxs, d_maxe, d_event]
//                     (PAPER.md:39), Moller / bremsstrahlung hard events, random-hinge MS deflection,
//                     CSDA loss through the range table, dose by red.global.add.f32
//   photon_kernel   : Woodcock flights, Compton / pair / photoelectric
//   atten_kernel    : attenuation-only mode under the fp32 arithmetic contract (R20)
//   finalize_kernel : batch means and standard errors (R17, R18)
#pragma once
#include "mc_device.cuh"
#include "mc_gs.h"

namespace mcb {

constexpr int kThreads = 256;
constexpr unsigned kFull = 0xffffffffu;
constexpr float kInf = 3.0e38f;

// ---- scoring: register accumulation while the target cell is unchanged, then one red ---------------
struct Score {
    float acc;
    uint32_t idx;  // batch * nvox + voxel
    uint32_t n_red;
};
__device__ __forceinline__ void score_flush(Score& s, float* edep) {
    if (s.acc > 0.0f) { atomicAdd(edep + s.idx, s.acc); ++s.n_red; }
    s.acc = 0.0f;
}
__device__ __forceinline__ void score_add(Score& s, float* edep, uint32_t idx, float e) {
    if (idx != s.idx) { score_flush(s, edep); s.idx = idx; }
    s.acc += e;
}

// Warp-aggregated scoring (PAPER.md:74 scores with one atomic per deposit): the lanes that score at the same moment
// are grouped by target cell (match.any); the lowest lane of each group sums the group's energies with shuffles and
// issues ONE red.global.add.f32.  Returns true in the lane that issued it.  Narrow beams put many lanes of a warp on
// the same few cells (config 1: a pencil beam), where the L2 serialises same-address reductions.
__device__ __forceinline__ bool red_add_aggregated(float* edep, uint32_t cell, float e) {
    const unsigned act = __activemask();
    const unsigned grp = __match_any_sync(act, cell);
    const int lane = threadIdx.x & 31, leader = __ffs(grp) - 1;
    float sum = e;
    for (unsigned m = grp & (grp - 1u); m; m &= m - 1u) sum += __shfl_sync(grp, e, __ffs(m) - 1);  // all but the leader
    if (lane == leader) atomicAdd(edep + cell, sum);
    return lane == leader;
}

// ---- geometry helpers --------------------------------------------------------------------------
__device__ __forceinline__ float face_dist(const Geometry& g, float x, float y, float z, float u, float v, float w,
                                           int ix, int iy, int iz, int& ax) {
    float px = fmaf((float)(ix + (u > 0.0f ? 1 : 0)), g.hx, g.ox);
    float py = fmaf((float)(iy + (v > 0.0f ? 1 : 0)), g.hy, g.oy);
    float pz = fmaf((float)(iz + (w > 0.0f ? 1 : 0)), g.hz, g.oz);
    float tx = u != 0.0f ? fmaxf(__fdividef(px - x, u), 0.0f) : kInf;
    float ty = v != 0.0f ? fmaxf(__fdividef(py - y, v), 0.0f) : kInf;
    float tz = w != 0.0f ? fmaxf(__fdividef(pz - z, w), 0.0f) : kInf;
    float best = tx; ax = 0;
    if (ty < best) { best = ty; ax = 1; }
    if (tz < best) { best = tz; ax = 2; }
    return best;
}

__device__ __forceinline__ unsigned long long warp_sum(uint32_t v) {
    unsigned long long s = v;
#pragma unroll
    for (int o = 16; o; o >>= 1) s += __shfl_xor_sync(kFull, s, o);
    return s;
}
__device__ __forceinline__ float warp_sum_f(float v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
    return v;
}
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
    return v;
}
__device__ __forceinline__ void stat_add(unsigned long long* stats, int id, unsigned long long v) {
    if (v) atomicAdd(stats + id, v);
}

// Claim work items for the lanes that want one: returns the item index (valid where `want`).
__device__ __forceinline__ uint32_t claim(uint32_t* head, unsigned want_mask, int lane) {
    int leader = __ffs(want_mask) - 1;
    uint32_t base = 0;
    if (lane == leader) base = atomicAdd(head, (uint32_t)__popc(want_mask));
    base = __shfl_sync(kFull, base, leader);
    return base + __popc(want_mask & ((1u << lane) - 1u));
}

// End of a transport launch: the last CTA to finish empties the consumed input queue and the work counter, so that the
// next launch can be enqueued without the host touching the counters (no launch pushes into its own input queue).
__device__ __forceinline__ void launch_epilogue(const RunParams& P) {
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        if (atomicAdd(P.counters + C_DONE, 1u) == gridDim.x - 1u) {
            P.counters[C_HEAD] = 0u; *P.q_in.count = 0u; P.counters[C_DONE] = 0u;
            __threadfence();
        }
    }
}

// Make a secondary: queue it, or (MC_FLAG_LOCAL_SECONDARIES) score its energy where it is born.
__device__ __forceinline__ void emit(const RunParams& P, const Queue& q, Score& sc, uint32_t cell, const QRec& r,
                                     uint32_t& n_pushed) {
    if (P.flags & 4u) {
        float e = r.E + (((r.tag & 3u) == CODE_POSITRON) ? 2.0f * kMeF : 0.0f);
        score_add(sc, P.edep, cell, e);
        return;
    }
    ++n_pushed;
    push_record(q, P.counters + C_OVERFLOW, r);
}

// =================================================================================================
// electron / positron kernel
//
// A warp executes, per iteration, ONE of three blocks on up to 32 tracks of its pool that are in the state the block
// serves:
//   STEP   one condensed-history step (S4-S6, S8)            — tracks in state L_STEP
//   HARD   hard-event thinning + Moller / bremsstrahlung (S7) — tracks in state L_HARD (pending)
//   REFILL queue pop / source generation (S0, S1)            — slots in state L_IDLE
// Divergent work is deferred until enough tracks of the pool want it (hard_lanes / refill_lanes) or nothing
// else can run, so the rare blocks run with many lanes instead of one or two (profiles/README.md).
// A warp's pool = kSlots x 32 tracks in shared memory, each track kGroups 16-byte groups (one LDS.128 / STS.128 per
// group: 5 loads and 3-4 stores per step); the fields are grouped by how often they change:
//   G0 x y z T | G1 u v w msc | G2 acc d_vox block smax | G3 rho tagk vox idx | G4 hist trk_lo trk_hi -
// (x, y, z = position relative to the low corner of the track's voxel; tagk = batch << 6 | material << 2 | charge code;
// idx = ix | iy << 10 | iz << 20; d_vox = distance to the nearest face along the direction, the only geometric
// quantity carried from step to step.)
// =================================================================================================
// One CTA per SM (the tables are staged once per SM).  kThreadsE = CTA size: 768 (24 warps) when tables + pools fit in
// the 227 KB of shared memory, else 512 or 256 (more materials / finer grids); instantiated in mc_engine.cu.
constexpr int kSlots = 2;       // tracks per lane, parked in shared memory between the blocks that work on them
enum LaneState { L_IDLE = 0, L_STEP = 1, L_HARD = 2, L_DONE = 3 };
constexpr int kGroups = 5;      // 16-byte groups per track
constexpr float kGsTMinF = (float)kGsTMin, kGsTMaxF = (float)kGsTMax;  // Goudsmit-Saunderson table range (mc_gs.h; R27)
enum { SE_STEP = 0, SE_MOLLER, SE_BREMS, SE_SEC_E, SE_SEC_G, SE_HIST, SE_RED, SE_COUNT };

// distances along (u,v,w) to the three faces of the voxel the direction points at; (x,y,z) = position relative to the
// voxel's low corner
__device__ __forceinline__ void face_all(const Geometry& g, float x, float y, float z, float u, float v, float w, float& tx, float& ty,
                                         float& tz) {
    float px = u > 0.0f ? g.hx : 0.0f, py = v > 0.0f ? g.hy : 0.0f, pz = w > 0.0f ? g.hz : 0.0f;
    float a = fmaxf((px - x) * f_rcp(u), 0.0f), b = fmaxf((py - y) * f_rcp(v), 0.0f), c = fmaxf((pz - z) * f_rcp(w), 0.0f);
    tx = fabsf(u) > 1e-20f ? a : kInf;
    ty = fabsf(v) > 1e-20f ? b : kInf;
    tz = fabsf(w) > 1e-20f ? c : kInf;
}

// Table coordinate (node + fraction) of the energy whose residual range is Rt: exact inverse of the piecewise-linear
// (in ln T) range interpolant (R5).  B[lo] = (R[lo], 1 / (R[lo+1] - R[lo]), K1[lo], K1[lo+1] - K1[lo]): node lo
// brackets Rt iff 0 <= (Rt - R[lo]) / (R[lo+1] - R[lo]) < 1.  The search starts at `guess` (callers pass the constant-L
// estimate ex + ln(1 - rho d L/T)/dln, within a fraction of a node): two probes without a branch (the second at the
// neighbour the first one points to, or at the same node), then — rarely — a walk in the same direction.  The walk
// never turns round: a value in the rounding gap between two segments ends it.  `node` returns B[lo] of the result and
// `frac` the fraction inside it (coordinate = lo + frac).
__device__ __forceinline__ float inv_range_coord(const float4* B, float Rt, float guess, int k_cut, int N, float4& node, float& frac) {
    int lo = min(max((int)guess, k_cut), N - 2);
    float4 a = B[lo];
    float f = (Rt - a.x) * a.y;
    const int mv = (f < 0.0f && lo > k_cut) ? -1 : ((f >= 1.0f && lo < N - 2) ? 1 : 0);
    lo += mv;
    a = B[lo];
    f = (Rt - a.x) * a.y;
    if (mv != 0) {  // rarely taken further than the neighbour
        const int stop = mv < 0 ? k_cut : N - 2;
        while ((mv < 0 ? f < 0.0f : f >= 1.0f) && lo != stop) {
            lo += mv;
            a = B[lo];
            f = (Rt - a.x) * a.y;
        }
    }
    node = a;
    frac = fminf(fmaxf(f, 0.0f), 1.0f);
    return (float)lo + frac;
}

struct ELane {
    float x, y, z, T, u, v, w;
    float msc;  // R8b: scattering power travelled but not yet sampled for (< 0: sampled ahead)
    float acc, dvox, smax, rho, ex;
    int vox;
    uint32_t idx, tagk;
    Rng rng;
};

// kMulti: the multi-voxel stepping (flags & 16; R28) instead of one step per voxel.
template <int kThreadsE, bool kMulti>
__global__ void __launch_bounds__(kThreadsE, 1) electron_kernel(const __grid_constant__ RunParams P) {
    extern __shared__ __align__(16) float2 s_tab[];
    // the launch consumes the whole input queue as it stands (no host round trip)
    const uint32_t n_in = *static_cast<const volatile uint32_t*>(P.q_in.count);
    if (n_in + P.n_new == 0u) return;  // nothing to do: an enqueued-ahead launch of a generation that does not exist
    const int ntab = P.n_mat * P.e_stride;
    constexpr int kWarps = kThreadsE / 32;
    uint4* s_trk = reinterpret_cast<uint4*>(s_tab + ntab);                     // [kGroups][kSlots][kThreadsE]
    uint32_t* s_st = reinterpret_cast<uint32_t*>(s_trk + kGroups * kSlots * kThreadsE);  // [kThreadsE]: byte k = state of slot k
    uint32_t* s_asg = s_st + kThreadsE;                                        // [kThreadsE]: per-warp assignment
    double* s_led = reinterpret_cast<double*>(s_asg + kThreadsE);              // [kWarps][2]: e_src, e_esc of the warp
    uint32_t* s_cnt = reinterpret_cast<uint32_t*>(s_led + 2 * kWarps);         // [kWarps][8]: event counters of the warp
    float* s_gs = reinterpret_cast<float*>(s_cnt + 8 * kWarps);                // Goudsmit-Saunderson tables (flags & 8 only)
    const bool gs_ms = P.flags & 8u;
    for (int i = threadIdx.x; i < ntab; i += kThreadsE) s_tab[i] = P.tabE[i];
    if (gs_ms) for (int i = threadIdx.x; i < P.gs_words; i += kThreadsE) s_gs[i] = P.gs[i];
    const int tid = threadIdx.x;
    if (tid < 8 * kWarps) s_cnt[tid] = 0u;
    if (tid < 2 * kWarps) s_led[tid] = 0.0;
    uint32_t st0 = 0u;  // slots beyond kSlots do not exist: L_DONE
#pragma unroll
    for (int k = kSlots; k < 4; ++k) st0 |= (uint32_t)L_DONE << (8 * k);
    s_st[tid] = st0;
    __syncthreads();
    const int lane = tid & 31;
    const unsigned lt_mask = (1u << lane) - 1u;
    const int N = P.N, k_cut = P.k_cut;
    const Geometry& g = P.g;
    const bool no_hard = P.flags & 1u, no_ms = P.flags & 2u, local_sec = P.flags & 4u;
    const int KH = P.hard_lanes, KR = P.refill_lanes;
    constexpr int GS = kSlots * kThreadsE;  // uint4 stride between the groups of a track

    int state = L_IDLE;            // state of the track being worked on (L)
    const int wbase = tid & ~31;   // first thread of this warp: a warp's kSlots x 32 slots form its track pool
    int slot = 0;                  // pool slot of the track being worked on: owner thread * 4 + k
    uint32_t n_step_w = 0u;
    ELane L;
    L.x = L.y = L.z = 0.f; L.u = L.v = 0.f; L.w = 1.f; L.T = 0.f; L.ex = 0.f; L.rho = 1.f; L.dvox = 0.f;
    L.acc = 0.f; L.smax = 0.f; L.msc = 0.f; L.vox = 0; L.idx = 0u; L.tagk = 0u; L.rng = {0, 0, 0, 0};
    auto trk = [&](int s) -> uint4* { return s_trk + (s & 3) * kThreadsE + (s >> 2); };
    auto mat_of = [&]() { return (int)((L.tagk >> 2) & 15u); };
    auto tabA = [&]() { return reinterpret_cast<const float4*>(s_tab + mat_of() * P.e_stride); };
    // what = 0: a new track, every group; 1: after a step or a hard event that stayed in its voxel; 2: after a step
    // that crossed into another voxel.  Identity words (history, track id) never change after birth.
    auto store_slot = [&](int s, int what) {
        uint4* t = trk(s);
        t[0] = make_uint4(__float_as_uint(L.x), __float_as_uint(L.y), __float_as_uint(L.z), __float_as_uint(L.T));
        t[GS] = make_uint4(__float_as_uint(L.u), __float_as_uint(L.v), __float_as_uint(L.w), __float_as_uint(L.msc));
        t[2 * GS] = make_uint4(__float_as_uint(L.acc), __float_as_uint(L.dvox), L.rng.block, __float_as_uint(L.smax));
        if (what != 1) t[3 * GS] = make_uint4(__float_as_uint(L.rho), L.tagk, (uint32_t)L.vox, L.idx);
        if (what == 0) t[4 * GS] = make_uint4(L.rng.hist, L.rng.trk_lo, L.rng.trk_hi, 0u);
    };
    auto load_slot = [&](int s) {
        const uint4* t = trk(s);
        const uint4 a = t[0], b = t[GS], c = t[2 * GS], d = t[3 * GS], e = t[4 * GS];
        L.x = __uint_as_float(a.x); L.y = __uint_as_float(a.y); L.z = __uint_as_float(a.z); L.T = __uint_as_float(a.w);
        L.u = __uint_as_float(b.x); L.v = __uint_as_float(b.y); L.w = __uint_as_float(b.z); L.msc = __uint_as_float(b.w);
        L.acc = __uint_as_float(c.x); L.dvox = __uint_as_float(c.y); L.rng.block = c.z; L.smax = __uint_as_float(c.w);
        L.rho = __uint_as_float(d.x); L.tagk = d.y; L.vox = (int)d.z; L.idx = d.w;
        L.rng.hist = e.x; L.rng.trk_lo = e.y; L.rng.trk_hi = e.z;
        L.ex = fmaf(f_lg2(L.T), P.ex_a, -P.ex_b);  // table coordinate of T (not stored)
    };
    auto park = [&](int what) {  // put the working track back into its pool slot: only live tracks need their data
        if (state == L_STEP || state == L_HARD) store_slot(slot, what);
        reinterpret_cast<volatile uint8_t*>(s_st)[slot] = (uint8_t)state;
    };
    uint32_t* const w_cnt = s_cnt + 8 * (tid >> 5);  // this warp's counters (shared-memory atomics: lanes bump them in divergent code)
    double* const w_led = s_led + 2 * (tid >> 5);
    auto bump = [&](int k) { atomicAdd(w_cnt + k, 1u); };
    auto flush = [&]() {  // one red.global.add.f32 per (track, voxel) visit (S6)
        if (L.acc > 0.0f) {
            const uint32_t cell = (L.tagk >> 6) * (uint32_t)g.nvox + (uint32_t)L.vox;  // n_batches * nvox < 2^32
            if (P.aggregate) { if (red_add_aggregated(P.edep, cell, L.acc)) bump(SE_RED); }
            else { atomicAdd(P.edep + cell, L.acc); bump(SE_RED); }
        }
        L.acc = 0.0f;
    };
    auto qtag = [&](uint32_t code) { return ((L.tagk >> 6) << 2) | code; };  // queue-record tag of a secondary
    auto is_positron = [&]() { return (L.tagk & 3u) == CODE_POSITRON; };
    // a secondary is born where the track stands: world coordinates for the queue record
    auto born_here = [&](QRec& r) {
        r.x = fmaf((float)(L.idx & 1023u), g.hx, g.ox) + L.x; r.y = fmaf((float)((L.idx >> 10) & 1023u), g.hy, g.oy) + L.y;
        r.z = fmaf((float)(L.idx >> 20), g.hz, g.oz) + L.z;
        r.hist = L.rng.hist; r.vox = L.vox;
    };
    auto emit_rec = [&](const Queue& q, const QRec& r, int stat) {
        if (local_sec) { L.acc += r.E + (((r.tag & 3u) == CODE_POSITRON) ? 2.0f * kMeF : 0.0f); return; }
        bump(stat);
        push_record(q, P.counters + C_OVERFLOW, r);
    };
    // end of track (S8): absorb the remaining kinetic energy; a positron annihilates at rest (R9)
    auto terminate = [&]() {
        L.acc += L.T;
        if (is_positron()) {
            uint4 a4 = next_block_rk(L.rng, P);
            float mu = 2.0f * u01f(a4.z) - 1.0f, sn = f_sqrt(fmaxf(1.0f - mu * mu, 0.0f)), ph = kTwoPiF * u01f(a4.w);
            QRec r; born_here(r); r.u = sn * f_cos(ph); r.v = sn * f_sin(ph); r.w = mu; r.E = kMeF;
            r.trk_lo = a4.x; r.trk_hi = a4.y; r.tag = qtag(CODE_PHOTON);
            emit_rec(P.q_p_out, r, SE_SEC_G);
            uint4 b4 = next_block_rk(L.rng, P);
            r.u = -r.u; r.v = -r.v; r.w = -r.w; r.trk_lo = b4.x; r.trk_hi = b4.y;
            emit_rec(P.q_p_out, r, SE_SEC_G);
        }
        flush();
        state = L_IDLE;
    };
    // d_vox of the track where it stands (after a change of direction)
    auto set_dvox = [&]() {
        float tx, ty, tz;
        face_all(g, L.x, L.y, L.z, L.u, L.v, L.w, tx, ty, tz);
        L.dvox = fminf(tx, fminf(ty, tz));
    };

    // The hinge's deflection (S5): multiple-scattering angle for scattering power k1rho * d of the planned step plus what
    // was travelled but not sampled for (R8b), Gaussian model (R7) or Goudsmit-Saunderson (R27); em = table coordinate of
    // the mid-step energy in the tables of material mat_ms, w4 = the step's Philox block (z: polar angle, w: azimuth).
    auto hinge_deflect = [&](float k1rho, float d, float em, int mat_ms, const uint4& w4) {
        // R8b: sample for the planned path plus the path travelled but not yet sampled for; never a negative path
        const float tq = fmaf(k1rho, d, P.ms_carry ? L.msc : 0.0f), t = fmaxf(tq, 0.0f);
        L.msc = tq - t;
        const float am = t < 1e-3f ? t * (1.0f - 0.5f * t) : 1.0f - f_exp(-t);
        if (!gs_ms) {
            if (am > 0.0f) {  // Gaussian on the sphere (R7)
                float omu = -am * kLn2F * f_lg2(1.0f - u01f(w4.z) * (1.0f - f_exp(-2.0f * f_rcp(am))));
                float phi = kTwoPiF * u01f(w4.w);
                rotate_fast(L.u, L.v, L.w, fminf(omu, 2.0f), f_sin(phi), f_cos(phi));
            }
        } else if (t < kGsTMinF) {
            if (P.ms_carry) L.msc += t;  // below the table: not sampled now, carried (R27)
        } else {
            // Goudsmit-Saunderson angle (R27): row by stochastic interpolation (9 low bits of the two
            // words), inverse CDF linear in log2 x inside a quantile interval
            const float2* tl = reinterpret_cast<const float2*>(s_gs + kGsNT * kGsNA * kGsNQ) + mat_ms * P.gs_n8;
            const float e8 = em * 0.125f;
            const int i8 = (int)e8;
            const float2 la = tl[i8];
            const float lnA = fmaf(e8 - (float)i8, la.y, la.x);
            const float tc = fminf(t, kGsTMaxF);
            const float cc = fmaf(f_lg2(tc), kLn2F, 4.0f * f_sqrt(tc));
            int ir = min(max((int)((cc - P.gs_c0) * P.gs_inv_dc), 0), kGsNT - 2);
            const float a0n = P.gs_an[ir], a1n = P.gs_an[ir + 1];
            const float ft = (fminf(am, P.gs_an[kGsNT - 1]) - a0n) * f_rcp(a1n - a0n);
            ir += ((float)(w4.z & 511u) + 0.5f < ft * 512.0f) ? 1 : 0;
            const float al = fminf(fmaxf((lnA - P.gs_lnA0) * P.gs_inv_dA, 0.0f), (float)(kGsNA - 1));
            int jr = min((int)al, kGsNA - 2);
            jr += ((float)(w4.w & 511u) + 0.5f < (al - (float)jr) * 512.0f) ? 1 : 0;
            const float* row = s_gs + (ir * kGsNA + jr) * kGsNQ;
            const float r = u01f(w4.z), s32 = (1.0f - r) * 32.0f;
            int kq;
            float fq;
            if (s32 > 1.0f) { const float r32 = 32.0f * r; kq = (int)r32; fq = r32 - (float)kq; }
            else {
                const int jj = min(126 - (int)(__float_as_uint(s32) >> 23), kGsNQ - 33);
                const float sj = s32 * __uint_as_float((uint32_t)(127 + jj) << 23);  // s 2^jj in (1/2, 1]
                kq = 31 + jj;
                fq = jj < kGsNQ - 33 ? 2.0f - 2.0f * sj : 1.0f - sj;
            }
            const float y0 = row[kq], y1 = row[kq + 1];
            const float xq = kq == 0 ? f_ex2(y1) * fq : f_ex2(fmaf(fq, y1 - y0, y0));
            const float phi = kTwoPiF * u01f(w4.w);
            rotate_fast(L.u, L.v, L.w, fminf(xq, 2.0f), f_sin(phi), f_cos(phi));
        }
            };

    for (;;) {
        // ---- scheduling: count the pool's tracks by state, choose ONE block, hand its tracks to the lanes ------
        // byte k of a lane's state word = state of its slot k; one-hot byte counters summed over the warp (REDUX)
        const uint32_t sw = s_st[tid];
        uint32_t cnt1 = 0u;
#pragma unroll
        for (int k = 0; k < kSlots; ++k) cnt1 += 1u << (8u * ((sw >> (8 * k)) & 3u));
        const uint32_t tot = __reduce_add_sync(kFull, cnt1);
        const int ni = (int)(tot & 0xffu), ns = (int)((tot >> 8) & 0xffu), nh = (int)((tot >> 16) & 0xffu);
        if ((tot & 0xffffffu) == 0u) break;
        // a rare block runs when it can fill a warp (>= KH / KR tracks), or when it has more tracks than STEP
        const bool do_hard = nh >= KH || (nh > ns && nh >= ni);
        const bool do_refill = !do_hard && (ni >= KR || ni > ns);
        const uint32_t cs = do_hard ? (uint32_t)L_HARD : (do_refill ? (uint32_t)L_IDLE : (uint32_t)L_STEP);
        // the r-th track of the chosen state (slot-major, then owner lane) goes to lane r: its owner posts the slot
        int rank = 0;
#pragma unroll
        for (int k = 0; k < kSlots; ++k) {
            const bool mine = ((sw >> (8 * k)) & 0xffu) == cs;
            const unsigned m = __ballot_sync(kFull, mine);
            const int r = rank + __popc(m & lt_mask);
            if (mine && r < 32) s_asg[wbase + r] = (uint32_t)(tid * 4 + k);
            rank += __popc(m);
        }
        __syncwarp();
        const int n_work = min(rank, 32);
        const bool have = lane < n_work;
        slot = have ? (int)s_asg[wbase + lane] : 0;
        __syncwarp();
        if (do_refill) {
            // ---- REFILL: queue first, then new primaries (S0, S1) --------------------------------
            uint32_t item = claim(P.counters + C_HEAD, n_work >= 32 ? kFull : ((1u << n_work) - 1u), lane);
            float e_new = 0.0f, e_out = 0.0f;  // source energy of the new primaries / of those that miss the phantom
            if (have) {
                state = L_IDLE; L.acc = 0.0f; L.msc = 0.0f; L.smax = 0.0f;
                bool ok = false;
                uint32_t qt = 0u;
                int ix = 0, iy = 0, iz = 0;
                if (item < n_in) {
                    QRec r = load_record(P.q_in, item);
                    L.x = r.x; L.y = r.y; L.z = r.z; L.u = r.u; L.v = r.v; L.w = r.w; L.T = r.E;
                    L.rng.hist = r.hist; L.rng.trk_lo = r.trk_lo; L.rng.trk_hi = r.trk_hi; L.rng.block = 0;
                    L.vox = r.vox; qt = r.tag;
                    ix = L.vox % g.nx; int t2 = L.vox / g.nx; iy = t2 % g.ny; iz = t2 / g.ny;
                    ok = true;
                } else if (item < n_in + P.n_new) {
                    unsigned long long h = P.h_first + (item - n_in);
                    L.rng.hist = (uint32_t)h; L.rng.trk_lo = 0; L.rng.trk_hi = 0; L.rng.block = 0;
                    uint4 w4 = next_block_rk(L.rng, P);
                    Primary p = sample_primary<false>(P, w4);
                    uint32_t code = P.beam.particle > 0 ? CODE_POSITRON : CODE_ELECTRON;
                    qt = (batch_of(h, P.n_batches, P.n_total, P.inv_n_total) << 2) | code;
                    float e0 = p.E + (code == CODE_POSITRON ? 2.0f * kMeF : 0.0f);
                    e_new = e0;
                    L.x = p.x; L.y = p.y; L.z = p.z; L.u = p.u; L.v = p.v; L.w = p.w; L.T = p.E;
                    ix = p.ix; iy = p.iy; iz = p.iz; L.vox = ix + g.nx * (iy + g.ny * iz);
                    if (p.inside) ok = true; else e_out = e0;
                } else state = L_DONE;
                if (ok) {
                    uint2 vd = P.vox[L.vox];
                    L.rho = __uint_as_float(vd.x);
                    L.tagk = ((qt >> 2) << 6) | (vd.y << 2) | (qt & 3u);
                    L.idx = (uint32_t)ix | ((uint32_t)iy << 10) | ((uint32_t)iz << 20);
                    // position relative to the voxel's low corner (a particle born on a face may be a rounding error outside)
                    L.x = fminf(fmaxf(L.x - fmaf((float)ix, g.hx, g.ox), 0.0f), g.hx);
                    L.y = fminf(fmaxf(L.y - fmaf((float)iy, g.hy, g.oy), 0.0f), g.hy);
                    L.z = fminf(fmaxf(L.z - fmaf((float)iz, g.hz, g.oz), 0.0f), g.hz);
                    state = L_STEP;
                    if (L.T <= P.e_cut) terminate();  // born at or below the cut-off (pair electrons)
                    else set_dvox();
                }
                park(0);  // L_DONE (nothing left to claim) retires the slot
            }
            __syncwarp();
            // ledger and history count of this refill: one warp-level sum (at most 32 primaries: exact to ~1e-7 in fp32)
            const unsigned m_new = __ballot_sync(kFull, e_new > 0.0f);
            if (m_new) {
                const float s_new = warp_sum_f(e_new), s_out = warp_sum_f(e_out);
                if (lane == 0) { w_led[0] += (double)s_new; w_led[1] += (double)s_out; w_cnt[SE_HIST] += (uint32_t)__popc(m_new); }
                __syncwarp();
            }
            continue;
        }

        if (do_hard) {
            // ---- HARD: thinning against the running-max majorant (R6), then Moller (R10) / bremsstrahlung (R11).
            // The two event types share one code path (Philox blocks, rejection loop, rotation of the secondary,
            // queue push) so that the expensive parts run with all pending lanes, not once per type. -----------
            if (have) {
                load_slot(slot);
                state = L_STEP;
                uint4 h4 = next_block_rk(L.rng, P);
                const float r = u01f(h4.x) * L.smax;
                int i1 = min(max((int)L.ex, 0), N - 2);
                float f1 = L.ex - (float)i1;
                const float4 hd = (tabA() + 2 * N)[i1];  // (S_hard, slope, S_Moller, slope)
                const float SH = fmaf(f1, hd.y, hd.x), SM = fmaf(f1, hd.w, hd.z);
                if (r < SH) {
                    const bool mol = r < SM;
                    const float T0 = L.T;
                    // per-type constants of the rejection sampling:  Moller: a = T0/e_cut, b = (2g-1)/g^2, c = ((g-1)/g)^2, m = g_max
                    //                                              brems : a = lg2(T0/g_cut), b = 1/(T0+mc^2), c = L_scr, m = F_max
                    float ca, cb, cc, cm;
                    const float Et = T0 + kMeF;
                    if (mol) {
                        float tau = T0 * (1.0f / kMeF), gm = tau + 1.0f, ig2 = f_rcp(gm * gm);
                        cb = (2.0f * gm - 1.0f) * ig2; cc = tau * tau * ig2;
                        ca = T0 * f_rcp(P.e_cut);
                        float ec = f_rcp(ca), o = f_rcp(1.0f - ec);
                        cm = fmaxf(1.0f - cb * ec * o + ec * ec * (cc + o * o), 1.0f - cb + 0.25f * (cc + 4.0f));  // max(g(e_c), g(1/2))
                    } else {
                        cb = f_rcp(Et); cc = P.lscr[mat_of()];
                        ca = f_lg2(T0 * f_rcp(P.g_cut));
                        cm = (4.0f / 3.0f) * (fminf(f_ln(2.0f * Et * (Et - P.g_cut) * f_rcp(kMeF * P.g_cut)), cc) - 0.5f);
                    }
                    // one trial: the sampled variable (Moller: eps = W/T0; brems: k) and its acceptance
                    auto trial = [&](uint32_t w0, uint32_t w1, float& val) {
                        const float u0 = u01f(w0), u1 = u01f(w1) * cm;
                        if (mol) {
                            float e = f_rcp(ca - u0 * (ca - 2.0f)), o = f_rcp(1.0f - e);
                            val = e;
                            return u1 <= 1.0f - cb * e * o + e * e * (cc + o * o);
                        }
                        float k = fminf(P.g_cut * f_ex2(ca * u0), T0), Ep = Et - k, rr = Ep * cb;
                        val = k;
                        return u1 <= (1.0f + rr * rr - (2.0f / 3.0f) * rr) * (fminf(f_ln(2.0f * Et * Ep * f_rcp(kMeF * k)), cc) - 0.5f);
                    };
                    float val;
                    for (;;) {
                        uint4 m4 = next_block_rk(L.rng, P);
                        if (trial(m4.x, m4.y, val)) break;
                        if (trial(m4.z, m4.w, val)) break;
                    }
                    const float phi = kTwoPiF * u01f(h4.w);
                    float sphi = f_sin(phi), cphi = f_cos(phi);
                    QRec q; born_here(q); q.u = L.u; q.v = L.v; q.w = L.w;
                    q.trk_lo = h4.y; q.trk_hi = h4.z;
                    float omu_q;  // 1 - cos(polar angle) of the secondary
                    if (mol) {
                        bump(SE_MOLLER);
                        const float W = val * T0, Tp = T0 - W, t2m = T0 + 2.0f * kMeF;
                        const float c1 = f_sqrt(Tp * t2m * f_rcp(T0 * (Tp + 2.0f * kMeF)));
                        omu_q = 1.0f - f_sqrt(W * t2m * f_rcp(T0 * (W + 2.0f * kMeF)));
                        q.E = W; q.tag = qtag(CODE_ELECTRON);
                        rotate_fast(L.u, L.v, L.w, 1.0f - c1, sphi, cphi);
                        set_dvox();
                        sphi = -sphi; cphi = -cphi;  // the delta ray leaves at azimuth phi + pi
                        L.T = Tp;
                    } else {
                        bump(SE_BREMS);
                        const float sh = f_sin(0.5f * kMeF * cb);
                        omu_q = 2.0f * sh * sh;  // polar angle mc^2 / (T0 + mc^2)
                        q.E = val; q.tag = qtag(CODE_PHOTON);
                        L.T = T0 - val;
                    }
                    rotate_fast(q.u, q.v, q.w, omu_q, sphi, cphi);
                    if (local_sec) L.acc += q.E;
                    else {
                        bump(mol ? SE_SEC_E : SE_SEC_G);
                        push_record2(P.q_e_out, P.q_p_out, mol, P.counters + C_OVERFLOW, q);
                    }
                    if (L.T <= P.e_cut) terminate();
                }
                park(1);
            }
            __syncwarp();
            continue;
        }

        n_step_w += (uint32_t)n_work;  // warp-uniform: n_work tracks take a step now
        if (!have) { __syncwarp(); continue; }
        load_slot(slot);
        state = L_STEP;
        if constexpr (kMulti) {
            // ---- STEP, multi-voxel variant (PAPER.md:167 gDPM's stepping; R28): d = min[d_maxs, d_maxe,
            // d_range, d_event] planned from the voxel the step starts in, NOT limited by it.  Both legs of the hinge are
            // walked voxel by voxel: every segment loses energy through the range table of its own material (scored in
            // its own voxel), uses up the sampled mean free paths at rho_i Sigma_max,i(T_start) and adds to the
            // scattering power travelled (R8b).  The step ends early where the mean free paths run out (hard-event
            // candidate), the range does (end of track) or the track leaves the phantom.
            const float4* tA = tabA();
            const int mat0 = mat_of();
            const int i0 = min(max((int)L.ex, 0), N - 2);
            const float f0 = L.ex - (float)i0;
            float4 a0 = tA[i0];
            float2 s0 = reinterpret_cast<const float2*>(tA + 3 * N)[i0];
            const float R0 = fmaf(f0, a0.y, a0.x), L0 = fmaf(f0, a0.w, a0.z);
            float Smax_i = fmaf(f0, s0.y, s0.x);
            const uint4 w4 = next_block_rk(L.rng, P);
            float tau = no_hard ? kInf : -kLn2F * f_lg2(u01f(w4.x));  // mean free paths to the next hard-event candidate
            const float rho0 = L.rho, irho0 = f_rcp(rho0);
            const float d = fminf(fminf(P.d_maxs, P.f_maxe * L.T * irho0 * f_rcp(L0)), fminf(fmaxf(R0, 0.0f) * irho0, tau * irho0 * f_rcp(Smax_i)));
            bool crossed = false;
            if (!(d > 0.0f)) { L.acc += fmaxf(L.T - P.e_cut, 0.0f); L.T = P.e_cut; }  // no residual range left (rounding)
            else {
                // K1 at the mid-step energy, in the start voxel's material; its table coordinate serves every material
                float4 nd;
                float fm = 0.0f, em = L.ex, k1rho0 = 0.0f;
                if (!no_ms) {
                    em = inv_range_coord(tA + N, fmaf(-0.5f * rho0, d, R0), fmaf(f_lg2(fmaf(-0.5f * d, rho0 * L0 * f_rcp(L.T), 1.0f)), P.ex_a, L.ex), k_cut, N, nd, fm);
                    k1rho0 = fmaf(fm, nd.w, nd.z) * rho0;
                }
                const int im = min(max((int)em, 0), N - 2);
                float k1rho_i = k1rho0, q_step = 0.0f, smax_ev = Smax_i;
                float Ri = R0, Li = L0, exc = L.ex;  // residual range, stopping power and table coordinate at the current energy
                int ev = 0;                           // 1: hard-event candidate, 2: end of range, 3: left the phantom
                const float legA = u01f(w4.y) * d;
#pragma unroll 1
                for (int leg = 0; leg < 2 && ev == 0; ++leg) {
                    float len = leg == 0 ? legA : d - legA;
                    if (leg == 1 && !no_ms) {
                        hinge_deflect(k1rho0, d, em, mat0, w4);
                        L.msc = fmaf(-k1rho0, d, L.msc);  // sampled for; the path travelled is added after the walk
                    }
                    float tx, ty, tz;
                    face_all(g, L.x, L.y, L.z, L.u, L.v, L.w, tx, ty, tz);
#pragma unroll 1
                    while (len > 0.0f) {
                        const float rho = L.rho, irho = f_rcp(rho);
                        int ax = 0;
                        float tf = tx;
                        if (ty < tf) { tf = ty; ax = 1; }
                        if (tz < tf) { tf = tz; ax = 2; }
                        float seg = fminf(len, tf);
                        const float l_tau = tau * irho * f_rcp(Smax_i), l_range = fmaxf(Ri, 0.0f) * irho;
                        // "<=" to rounding (of the whole step: what is left in the second leg is a difference): a step planned
                        // up to the event or to the end of the range ends exactly there
                        if (l_tau <= fmaf(1e-5f, d, seg)) { seg = fminf(seg, l_tau); ev = 1; smax_ev = Smax_i; }
                        if (l_range <= fmaf(1e-5f, d, seg)) { seg = fminf(seg, l_range); ev = 2; }
                        L.x = fmaf(seg, L.u, L.x); L.y = fmaf(seg, L.v, L.y); L.z = fmaf(seg, L.w, L.z);
                        tx = fmaxf(tx - seg, 0.0f); ty = fmaxf(ty - seg, 0.0f); tz = fmaxf(tz - seg, 0.0f);
                        float T1 = P.e_cut;
                        if (ev != 2) {
                            float fr;
                            exc = inv_range_coord(tA + N, fmaf(-rho, seg, Ri),
                                                  fmaf(f_lg2(fmaxf(fmaf(-seg, rho * Li * f_rcp(L.T), 1.0f), 1e-3f)), P.ex_a, exc), k_cut, N, nd, fr);
                            T1 = fminf(f_ex2(fmaf(exc, P.t_a, P.t_b)), L.T);
                        }
                        L.acc += L.T - T1;
                        L.T = T1;
                        tau = fmaf(-rho * Smax_i, seg, tau);
                        q_step = fmaf(k1rho_i, seg, q_step);
                        len -= seg;
                        if (ev != 0) break;
                        if (seg >= tf) {
                            // on the face: flush this voxel's deposit, enter the neighbour (as in the per-voxel variant)
                            flush();
                            crossed = true;
                            const bool a0x = ax == 0, a1x = ax == 1, a2x = ax == 2;
                            const float dc = a0x ? L.u : (a1x ? L.v : L.w);
                            const bool up = dc > 0.0f;
                            const float ha = a0x ? g.hx : (a1x ? g.hy : g.hz);
                            const float tnew = ha * f_rcp(fabsf(dc)), xin = up ? 0.0f : ha;
                            L.x = a0x ? xin : L.x; L.y = a1x ? xin : L.y; L.z = a2x ? xin : L.z;
                            tx = a0x ? tnew : tx; ty = a1x ? tnew : ty; tz = a2x ? tnew : tz;
                            const int sh = 10 * ax;
                            const int ia = (int)((L.idx >> sh) & 1023u) + (up ? 1 : -1);
                            const int na = a0x ? g.nx : (a1x ? g.ny : g.nz), stride = a0x ? 1 : (a1x ? g.nx : g.nx * g.ny);
                            if ((unsigned)ia >= (unsigned)na) {
                                atomicAdd(w_led + 1, (double)(L.T + (is_positron() ? 2.0f * kMeF : 0.0f)));
                                state = L_IDLE; ev = 3;
                                break;
                            }
                            L.idx = (L.idx & ~(1023u << sh)) | ((uint32_t)ia << sh);
                            L.vox += up ? stride : -stride;
                            const uint2 vd = P.vox[L.vox];
                            const bool new_mat = vd.y != ((L.tagk >> 2) & 15u);
                            L.rho = __uint_as_float(vd.x); L.tagk = (L.tagk & ~60u) | (vd.y << 2);
                            if (new_mat) {  // the new material's majorant at the step's start energy, its K1 at the mid-step energy
                                tA = tabA();
                                s0 = reinterpret_cast<const float2*>(tA + 3 * N)[i0];
                                Smax_i = fmaf(f0, s0.y, s0.x);
                                const float4 bm = (tA + N)[im];
                                k1rho_i = no_ms ? 0.0f : fmaf(em - (float)im, bm.w, bm.z);
                            }
                            k1rho_i = new_mat ? k1rho_i * L.rho : (no_ms ? 0.0f : k1rho_i * L.rho * irho);
                        }
                        // residual range and stopping power at the current energy in the current material
                        const int ic = min(max((int)exc, 0), N - 2);
                        a0 = tA[ic];
                        Ri = fmaf(exc - (float)ic, a0.y, a0.x); Li = fmaf(exc - (float)ic, a0.w, a0.z);
                    }
                }
                L.msc += q_step;
                if (state == L_STEP && ev == 1 && L.T > P.e_cut) { state = L_HARD; L.smax = smax_ev; }
            }
            if (state == L_STEP && L.T <= P.e_cut) terminate();
            park(crossed ? 2 : 1);
            __syncwarp();
            continue;
        }
        // ---- STEP set-up (S4): d = min[d_vox, d_maxs, d_maxe, d_range, d_event] ------------------------------
        const float4* const tA = tabA();  // [N] (R, slope, L, slope) | [N] inverse-range pack | [N] hard pack | [N] float2 S_max
        const float4* const tB = tA + N;
        int i0 = min(max((int)L.ex, 0), N - 2);
        float f0 = L.ex - (float)i0;
        const float4 a0 = tA[i0];
        const float2 s0 = reinterpret_cast<const float2*>(tA + 3 * N)[i0];
        const float R0 = fmaf(f0, a0.y, a0.x), L0 = fmaf(f0, a0.w, a0.z), Smax = fmaf(f0, s0.y, s0.x);
        uint4 w4 = next_block_rk(L.rng, P);
        const float rho = L.rho, irho = f_rcp(rho);
        const float d_vox = L.dvox;
        float d_lim = P.d_maxs;  // the non-geometric limits
        int lim = 1;
        const float d_maxe = P.f_maxe * L.T * irho * f_rcp(L0);
        const float d_range = fmaxf(R0, 0.0f) * irho;
        if (d_maxe < d_lim) { d_lim = d_maxe; lim = 2; }
        if (d_range < d_lim) { d_lim = d_range; lim = 3; }
        if (!no_hard) {
            float d_event = -kLn2F * f_lg2(u01f(w4.x)) * irho * f_rcp(Smax);
            if (d_event < d_lim) { d_lim = d_event; lim = 4; }
        }
        float d = d_vox;
        if (d_lim < d) d = d_lim; else lim = 0;
        // ---- random hinge (S5; R7, R8) ---------------------------------------------------------------------
        const float legA = u01f(w4.y) * d;
        L.x = fmaf(legA, L.u, L.x); L.y = fmaf(legA, L.v, L.y); L.z = fmaf(legA, L.w, L.z);
        const float xl = rho * L0 * f_rcp(L.T);  // fractional energy loss per unit path at constant L (search guess only)
        const float rd = rho * d;
        float k1rho = 0.0f;
        float4 nd;
        float fm;
        if (!no_ms) {
            const float em = inv_range_coord(tB, fmaf(-0.5f, rd, R0), fmaf(f_lg2(fmaf(-0.5f * d, xl, 1.0f)), P.ex_a, L.ex), k_cut, N, nd, fm);
            k1rho = fmaf(fm, nd.w, nd.z) * rho;  // K1 at the mid-step energy: its node is the one the search ended on
            hinge_deflect(k1rho, d, em, mat_of(), w4);
        }
        float tx, ty, tz;
        face_all(g, L.x, L.y, L.z, L.u, L.v, L.w, tx, ty, tz);
        const float rest = d - legA;
        int ax = 0;
        float tf = tx;
        if (ty < tf) { tf = ty; ax = 1; }
        if (tz < tf) { tf = tz; ax = 2; }
        // R8: a voxel-limited step may run on to the face by up to hinge_overrun of the planned second leg, never
        // beyond the non-geometric limits (removes the tiny catch-up steps after half of the voxel-limited steps)
        const bool cross = tf <= fmaxf(fminf((1.0f + P.hinge_overrun) * rest, d_lim - legA), rest);
        const float legB = cross ? tf : rest;
        L.x = fmaf(legB, L.u, L.x); L.y = fmaf(legB, L.v, L.y); L.z = fmaf(legB, L.w, L.z);
        tx = fmaxf(tx - legB, 0.0f); ty = fmaxf(ty - legB, 0.0f); tz = fmaxf(tz - legB, 0.0f);
        const float d_act = legA + legB;
        L.msc = fmaf(k1rho, d_act - d, L.msc);
        // ---- CSDA loss through the range table (S6; R5) + scoring ------------------------------------------
        float T1;
        if (lim == 3 && !cross) T1 = P.e_cut;
        else {
            const float ex1 = inv_range_coord(tB, fmaf(-rho, d_act, R0), fmaf(f_lg2(fmaxf(fmaf(-d_act, xl, 1.0f), 1e-3f)), P.ex_a, L.ex), k_cut, N, nd, fm);
            T1 = fminf(f_ex2(fmaf(ex1, P.t_a, P.t_b)), L.T);
        }
        L.acc += L.T - T1;
        L.T = T1;
        if (cross) {
            // leave the voxel: flush its deposit, enter the neighbour through the face that was hit (the one the
            // direction points at; R8).  One predicate per axis: selects, not a 3-way branch.
            flush();
            const bool a0x = ax == 0, a1x = ax == 1, a2x = ax == 2;
            const float dc = a0x ? L.u : (a1x ? L.v : L.w);
            const bool up = dc > 0.0f;
            const float ha = a0x ? g.hx : (a1x ? g.hy : g.hz);
            const float tnew = ha * f_rcp(fabsf(dc)), xin = up ? 0.0f : ha;  // local coordinate on the face it enters through
            L.x = a0x ? xin : L.x; L.y = a1x ? xin : L.y; L.z = a2x ? xin : L.z;
            tx = a0x ? tnew : tx; ty = a1x ? tnew : ty; tz = a2x ? tnew : tz;
            const int sh = 10 * ax;
            const int ia = (int)((L.idx >> sh) & 1023u) + (up ? 1 : -1);
            const int na = a0x ? g.nx : (a1x ? g.ny : g.nz), stride = a0x ? 1 : (a1x ? g.nx : g.nx * g.ny);
            if ((unsigned)ia >= (unsigned)na) {
                atomicAdd(w_led + 1, (double)(L.T + (is_positron() ? 2.0f * kMeF : 0.0f)));
                state = L_IDLE;
            } else {
                L.idx = (L.idx & ~(1023u << sh)) | ((uint32_t)ia << sh);
                L.vox += up ? stride : -stride;
                uint2 vd = P.vox[L.vox];
                L.rho = __uint_as_float(vd.x); L.tagk = (L.tagk & ~60u) | (vd.y << 2);
            }
        }
        if (state == L_STEP) {
            if (L.T <= P.e_cut) terminate();
            else if (lim == 4 && !cross) { state = L_HARD; L.smax = Smax; }
        }
        L.dvox = fminf(tx, fminf(ty, tz));
        park(cross ? 2 : 1);
        __syncwarp();
    }
    // ---- exit: the warp's counters and ledger go to the global ones -------------------------------------------------
    __syncwarp();
    const int sid[SE_COUNT] = {S_ESTEP, S_MOLLER, S_BREMS, S_SEC_E, S_SEC_G, S_HIST, S_ATOMICS};
    if (lane < SE_COUNT) stat_add(P.stats, sid[lane], lane == SE_STEP ? (unsigned long long)n_step_w : (unsigned long long)w_cnt[lane]);
    if (lane == 0) {
        if (w_led[0] != 0.0) atomicAdd(P.ledger + LG_SRC, w_led[0]);
        if (w_led[1] != 0.0) atomicAdd(P.ledger + LG_ESC, w_led[1]);
    }
    launch_epilogue(P);
}

// =================================================================================================
// photon kernel: Woodcock tracking (R3), Compton (R4), pair (R12),
// photoelectric absorption (R16).  One Philox block serves two flights.  Same warp scheduling as the electron
// kernel: per iteration a warp runs ONE of  FLY (tracks in L_STEP) / COMPTON (tracks in L_HARD, pending) /
// REFILL (slots in L_IDLE), the rare blocks only when enough tracks want them.  A track is three 16-byte groups
//   G0 x y z E | G1 u v w block | G2 tag hist trk_lo trk_hi   (+ one word: the voxel of a pending Compton event),
// positions in world coordinates (Woodcock flights look the voxel up by position, no boundary computation).
// =================================================================================================
// kThreadsP = CTA size of the photon kernel: 1024 (32 warps), 768 or 512 by what fits (one CTA per SM)
constexpr int kSlotsP = 3;     // tracks per lane in the warp's pool (shared memory)
constexpr int kGroupsP = 3;    // 16-byte groups per track
enum { SP_FLIGHT = 0, SP_FICT, SP_COMPTON, SP_PAIR, SP_PE, SP_SEC_E, SP_HIST, SP_RED, SP_COUNT };

template <int kThreadsP>
__global__ void __launch_bounds__(kThreadsP, 1) photon_kernel(const __grid_constant__ RunParams P) {
    extern __shared__ __align__(16) float2 s_tab[];
    const uint32_t n_in = *static_cast<const volatile uint32_t*>(P.q_in.count);  // as in electron_kernel
    if (n_in + P.n_new == 0u) return;
    const int ntab = (1 + P.n_mat * TP_COUNT) * P.N;
    constexpr int kWarps = kThreadsP / 32;
    constexpr int GS = kSlotsP * kThreadsP;  // uint4 stride between the groups of a track
    uint4* s_trk = reinterpret_cast<uint4*>(s_tab + ((ntab + 1) & ~1));        // [kGroupsP][kSlotsP][kThreadsP]
    uint32_t* s_vox = reinterpret_cast<uint32_t*>(s_trk + kGroupsP * GS);      // [kSlotsP][kThreadsP]: voxel of a pending Compton event
    uint32_t* s_st = s_vox + GS;                                               // [kThreadsP]: byte k = state of slot k
    uint32_t* s_asg = s_st + kThreadsP;                                        // [kThreadsP]: per-warp assignment
    double* s_esc = reinterpret_cast<double*>(s_asg + kThreadsP);              // [kThreadsP]: escaped energy per thread
    double* s_src = s_esc + kThreadsP;                                         // [kWarps]: source energy of the warp
    uint32_t* s_cnt = reinterpret_cast<uint32_t*>(s_src + kWarps);             // [kWarps][8]: event counters of the warp
    for (int i = threadIdx.x; i < ntab; i += kThreadsP) s_tab[i] = P.tabP[i];
    const int tid = threadIdx.x;
    if (tid < 8 * kWarps) s_cnt[tid] = 0u;
    if (tid < kWarps) s_src[tid] = 0.0;
    s_esc[tid] = 0.0;
    uint32_t st0 = 0u;  // slots beyond kSlotsP do not exist: L_DONE
#pragma unroll
    for (int k = kSlotsP; k < 4; ++k) st0 |= (uint32_t)L_DONE << (8 * k);
    s_st[tid] = st0;
    __syncthreads();
    const int lane = tid & 31;
    const unsigned lt_mask = (1u << lane) - 1u;
    const int N = P.N;
    const Geometry& g = P.g;
    const bool local_sec = P.flags & 4u;
    const int KC = P.hard_lanes, KR = P.refill_lanes;
    const float lg_a = kLn2F * P.inv_dlnP, lg_b = P.lnE0P * P.inv_dlnP;  // table coordinate = lg2(E) * lg_a - lg_b
    uint32_t* const w_cnt = s_cnt + 8 * (tid >> 5);

    int state = L_IDLE;  // state of the track being worked on
    const int wbase = tid & ~31;
    int slot = 0;        // pool slot of the track being worked on: owner thread * 4 + k
    float x = 0, y = 0, z = 0, u = 0, v = 0, w = 1, E = 0, lf = 0, maj = 1;
    int li = 0, vox = 0;
    Rng rng = {0, 0, 0, 0};
    uint32_t tag = 0;
    auto trk = [&](int s) -> uint4* { return s_trk + (s & 3) * kThreadsP + (s >> 2); };
    // what = 0: a new track, every group; 1: after flights or a Compton event (identity words unchanged)
    auto store_slot = [&](int s, int what) {
        uint4* t = trk(s);
        t[0] = make_uint4(__float_as_uint(x), __float_as_uint(y), __float_as_uint(z), __float_as_uint(E));
        t[GS] = make_uint4(__float_as_uint(u), __float_as_uint(v), __float_as_uint(w), rng.block);
        if (what == 0) t[2 * GS] = make_uint4(tag, rng.hist, rng.trk_lo, rng.trk_hi);
        if (state == L_HARD) s_vox[(s & 3) * kThreadsP + (s >> 2)] = (uint32_t)vox;
    };
    auto load_slot = [&](int s) {
        const uint4* t = trk(s);
        const uint4 a = t[0], b = t[GS], c = t[2 * GS];
        x = __uint_as_float(a.x); y = __uint_as_float(a.y); z = __uint_as_float(a.z); E = __uint_as_float(a.w);
        u = __uint_as_float(b.x); v = __uint_as_float(b.y); w = __uint_as_float(b.z); rng.block = b.w;
        tag = c.x; rng.hist = c.y; rng.trk_lo = c.z; rng.trk_hi = c.w;
    };
    auto park = [&](int what) {
        if (state == L_STEP || state == L_HARD) store_slot(slot, what);
        reinterpret_cast<volatile uint8_t*>(s_st)[slot] = (uint8_t)state;
    };
    auto bump = [&](int k) { atomicAdd(w_cnt + k, 1u); };
    auto deposit = [&](int vx, float e) {
        const uint32_t cell = (tag >> 2) * (uint32_t)g.nvox + (uint32_t)vx;
        if (P.aggregate) { if (red_add_aggregated(P.edep, cell, e)) bump(SP_RED); }
        else { atomicAdd(P.edep + cell, e); bump(SP_RED); }
    };
    auto set_energy = [&]() {  // table coordinate and majorant of the current energy
        float t = fmaf(f_lg2(E), lg_a, -lg_b);
        li = min(max((int)t, 0), N - 2); lf = t - (float)li;
        maj = lerp(s_tab, li, lf);
    };
    auto emit_e = [&](const QRec& r) {
        if (local_sec) { deposit(r.vox, r.E + (((r.tag & 3u) == CODE_POSITRON) ? 2.0f * kMeF : 0.0f)); return; }
        bump(SP_SEC_E);
        push_record(P.q_e_out, P.counters + C_OVERFLOW, r);
    };

    for (;;) {
        // scheduling as in electron_kernel: one-hot byte counters of the slot states summed over the warp
        const uint32_t sw = s_st[tid];
        uint32_t cnt1 = 0u;
#pragma unroll
        for (int k = 0; k < kSlotsP; ++k) cnt1 += 1u << (8u * ((sw >> (8 * k)) & 3u));
        const uint32_t tot = __reduce_add_sync(kFull, cnt1);
        const int ni = (int)(tot & 0xffu), nf = (int)((tot >> 8) & 0xffu), nc = (int)((tot >> 16) & 0xffu);
        if ((tot & 0xffffffu) == 0u) break;
        const bool do_comp = nc >= KC || (nc > nf && nc >= ni);
        const bool do_refill = !do_comp && (ni >= KR || ni > nf);
        const uint32_t cs = do_comp ? (uint32_t)L_HARD : (do_refill ? (uint32_t)L_IDLE : (uint32_t)L_STEP);
        int rank = 0;
#pragma unroll
        for (int k = 0; k < kSlotsP; ++k) {
            const bool mine = ((sw >> (8 * k)) & 0xffu) == cs;
            const unsigned m = __ballot_sync(kFull, mine);
            const int r = rank + __popc(m & lt_mask);
            if (mine && r < 32) s_asg[wbase + r] = (uint32_t)(tid * 4 + k);
            rank += __popc(m);
        }
        __syncwarp();
        const int n_work = min(rank, 32);
        const bool have = lane < n_work;
        slot = have ? (int)s_asg[wbase + lane] : 0;
        __syncwarp();

        if (do_refill) {
            // ---- REFILL (S0, S1) --------------------------------------------------------------------------------
            uint32_t item = claim(P.counters + C_HEAD, n_work >= 32 ? kFull : ((1u << n_work) - 1u), lane);
            float e_new = 0.0f;  // source energy of a new primary
            if (have) {
                state = L_IDLE;
                bool ok = false;
                if (item < n_in) {
                    QRec r = load_record(P.q_in, item);
                    x = r.x; y = r.y; z = r.z; u = r.u; v = r.v; w = r.w; E = r.E;
                    rng.hist = r.hist; rng.trk_lo = r.trk_lo; rng.trk_hi = r.trk_hi; rng.block = 0;
                    vox = r.vox; tag = r.tag;
                    ok = true;
                } else if (item < n_in + P.n_new) {
                    unsigned long long h = P.h_first + (item - n_in);
                    rng.hist = (uint32_t)h; rng.trk_lo = 0; rng.trk_hi = 0; rng.block = 0;
                    uint4 w4 = next_block_rk(rng, P);
                    Primary p = sample_primary<false>(P, w4);
                    tag = (batch_of(h, P.n_batches, P.n_total, P.inv_n_total) << 2) | CODE_PHOTON;
                    e_new = p.E;
                    x = p.x; y = p.y; z = p.z; u = p.u; v = p.v; w = p.w; E = p.E;
                    vox = p.ix + g.nx * (p.iy + g.ny * p.iz);
                    if (p.inside) ok = true; else s_esc[tid] += (double)p.E;
                } else state = L_DONE;
                if (ok) {
                    if (E < P.g_cut) deposit(vox, E);  // absorbed where it was born
                    else state = L_STEP;
                }
                park(0);
            }
            __syncwarp();
            const unsigned m_new = __ballot_sync(kFull, e_new > 0.0f);
            if (m_new) {  // ledger and history count of this refill: one warp-level sum
                const float s_new = warp_sum_f(e_new);
                if (lane == 0) { s_src[tid >> 5] += (double)s_new; w_cnt[SP_HIST] += (uint32_t)__popc(m_new); }
                __syncwarp();
            }
            continue;
        }

        if (do_comp) {
            // ---- COMPTON: Klein-Nishina by the epsilon decomposition (R4) ----------------------------------------
            if (have) {
                load_slot(slot);
                vox = (int)s_vox[(slot & 3) * kThreadsP + (slot >> 2)];
                bump(SP_COMPTON);
                const float k0 = E * (1.0f / kMeF), e0 = f_rcp(1.0f + 2.0f * k0), e02 = e0 * e0;
                const float a1 = -f_lg2(e0) * kLn2F, a2 = 0.5f * (1.0f - e02), ik0 = f_rcp(k0);
                float eps, tt;
                const float ia2 = f_rcp(a2);
                // one trial from two words: the first picks the branch and, rescaled inside it, samples epsilon (R15)
                auto trial = [&](uint32_t wa, uint32_t wb) {
                    const float r = u01f(wa) * (a1 + a2);
                    eps = r < a1 ? f_ex2(-r * kLog2eF) : f_sqrt(fmaf((1.0f - e02) * ia2, r - a1, e02));
                    tt = (1.0f - eps) * f_rcp(eps) * ik0;
                    const float sin2 = tt * (2.0f - tt);
                    return u01f(wb) <= 1.0f - eps * sin2 * f_rcp(1.0f + eps * eps);
                };
                for (;;) {
                    uint4 c4 = next_block_rk(rng, P);
                    if (trial(c4.x, c4.y)) break;
                    if (trial(c4.z, c4.w)) break;
                }
                uint4 d4 = next_block_rk(rng, P);
                const float E1 = eps * E, Te = E - E1;
                const float u0 = u, v0 = v, w0 = w;
                const float phi = kTwoPiF * u01f(d4.z);
                rotate_fast(u, v, w, tt, f_sin(phi), f_cos(phi));
                float dep = 0.0f;
                if (Te >= P.e_cut || local_sec) {
                    QRec q; q.x = x; q.y = y; q.z = z; q.hist = rng.hist; q.vox = vox;
                    float qx = E * u0 - E1 * u, qy = E * v0 - E1 * v, qz = E * w0 - E1 * w;
                    float inr = f_rsqrt(fmaf(qx, qx, fmaf(qy, qy, qz * qz)));
                    q.u = qx * inr; q.v = qy * inr; q.w = qz * inr;
                    q.E = Te; q.trk_lo = d4.x; q.trk_hi = d4.y; q.tag = (tag & ~3u) | CODE_ELECTRON;
                    emit_e(q);
                } else dep = Te;  // born below the cut-off: absorbed where it is born (R26)
                E = E1;
                if (E < P.g_cut) { dep += E; state = L_IDLE; }
                else state = L_STEP;
                if (dep > 0.0f) deposit(vox, dep);
                park(1);
            }
            __syncwarp();
            continue;
        }

        if (!have) { __syncwarp(); continue; }
        load_slot(slot);
        state = L_STEP;
        set_energy();
        // ---- FLY: up to two Woodcock flights from one Philox block (S2) --------------------------------------------
        uint4 w4 = next_block_rk(rng, P);
        int chan = -1;
        uint32_t n_fl = 0, n_fi = 0;
        const float2* tm = s_tab;
        const float imaj = f_rcp(maj);
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            float sl = -kLn2F * f_lg2(u01f(k ? w4.z : w4.x)) * imaj;
            x = fmaf(sl, u, x); y = fmaf(sl, v, y); z = fmaf(sl, w, z);
            ++n_fl;
            float gx = (x - g.ox) * g.ihx, gy = (y - g.oy) * g.ihy, gz = (z - g.oz) * g.ihz;
            if (!(gx >= 0.0f && gx < (float)g.nx && gy >= 0.0f && gy < (float)g.ny && gz >= 0.0f && gz < (float)g.nz)) {
                s_esc[tid] += (double)E; state = L_IDLE; break;
            }
            vox = (int)gx + g.nx * ((int)gy + g.ny * (int)gz);
            uint2 vd = P.vox[vox];
            float rho = __uint_as_float(vd.x);
            tm = s_tab + (1 + (int)vd.y * TP_COUNT) * N;
            float r = u01f(k ? w4.w : w4.y) * maj;
            float mu = rho * lerp(tm + TP_TOT * N, li, lf);
            if (r > mu) { ++n_fi; continue; }
            float mc = rho * lerp(tm + TP_C * N, li, lf), mp = rho * lerp(tm + TP_PP * N, li, lf);
            chan = r < mc ? 0 : (r < mc + mp ? 1 : 2);
            break;
        }
        {   // flights and fictitious interactions of the lanes that flew: one warp-level sum, one lane books it
            const unsigned act = __activemask();
            const uint32_t both = __reduce_add_sync(act, n_fl | (n_fi << 16));
            if (lane == __ffs(act) - 1) { w_cnt[SP_FLIGHT] += both & 0xffffu; w_cnt[SP_FICT] += both >> 16; }
        }
        if (chan == 0) state = L_HARD;  // Compton: pending
        else if (chan == 2) {           // photoelectric: absorbed locally
            bump(SP_PE);
            deposit(vox, E);
            state = L_IDLE;
        } else if (chan == 1) {  // pair: both along the photon direction, uniform split
            bump(SP_PAIR);
            QRec q; q.x = x; q.y = y; q.z = z; q.hist = rng.hist; q.vox = vox;
            uint4 a4 = next_block_rk(rng, P);
            float Tk = E - 2.0f * kMeF, us = u01f(a4.z);
            q.u = u; q.v = v; q.w = w;
            q.E = us * Tk; q.trk_lo = a4.x; q.trk_hi = a4.y; q.tag = (tag & ~3u) | CODE_ELECTRON;
            emit_e(q);
            uint4 b4 = next_block_rk(rng, P);
            q.E = Tk - q.E; q.trk_lo = b4.x; q.trk_hi = b4.y; q.tag = (tag & ~3u) | CODE_POSITRON;
            emit_e(q);
            state = L_IDLE;
        }
        park(1);
        __syncwarp();
    }
    __syncwarp();
    const int sid[SP_COUNT] = {S_FLIGHT, S_FICT, S_COMPTON, S_PAIR, S_PE, S_SEC_E, S_HIST, S_ATOMICS};
    if (lane < SP_COUNT) stat_add(P.stats, sid[lane], (unsigned long long)w_cnt[lane]);
    const double s_e = warp_sum(s_esc[tid]);
    if (lane == 0) {
        if (s_src[tid >> 5] != 0.0) atomicAdd(P.ledger + LG_SRC, s_src[tid >> 5]);
        if (s_e != 0.0) atomicAdd(P.ledger + LG_ESC, s_e);
    }
    launch_epilogue(P);
}

// =================================================================================================
// attenuation-only mode (R20): primaries only, fp32 arithmetic contract, one thread per
// history.  Output: voxel and channel of the first real interaction.
// =================================================================================================
__global__ void __launch_bounds__(kThreads) atten_kernel(const __grid_constant__ RunParams P, unsigned long long n,
                                                         int32_t* vox_out, uint8_t* chan_out) {
    const Geometry& g = P.g;
    const int N = P.N;
    for (unsigned long long h = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; h < n;
         h += (unsigned long long)gridDim.x * blockDim.x) {
        Rng rng = {(uint32_t)h, 0u, 0u, 0u};
        uint4 w4 = next_block(rng, P.seed_lo, P.seed_hi);
        Primary p = sample_primary(P, w4);
        int32_t vox = -1; uint8_t chan = 255;
        if (p.inside && p.E >= P.g_cut) {
            Lookup l = c_lookup(c_ln(p.E), P.lnE0P, P.inv_dlnP, N);
            float maj = c_lerp(P.tabP, l);
            float x = p.x, y = p.y, z = p.z;
            bool done = false;
            while (!done) {
                w4 = next_block(rng, P.seed_lo, P.seed_hi);
#pragma unroll
                for (int k = 0; k < 2; ++k) {
                    if (done) break;
                    float sl = __fdiv_rn(-c_ln(u01(k ? w4.z : w4.x)), maj);
                    x = __fmaf_rn(sl, p.u, x); y = __fmaf_rn(sl, p.v, y); z = __fmaf_rn(sl, p.w, z);
                    float gx = __fmul_rn(__fsub_rn(x, g.ox), g.ihx), gy = __fmul_rn(__fsub_rn(y, g.oy), g.ihy),
                          gz = __fmul_rn(__fsub_rn(z, g.oz), g.ihz);
                    if (!(gx >= 0.0f && gx < (float)g.nx && gy >= 0.0f && gy < (float)g.ny && gz >= 0.0f && gz < (float)g.nz)) {
                        done = true; break;
                    }
                    int vi = (int)gx + g.nx * ((int)gy + g.ny * (int)gz);
                    uint2 vd = P.vox[vi];
                    float rho = __uint_as_float(vd.x);
                    const float2* tm = P.tabP + (size_t)(1 + (int)vd.y * TP_COUNT) * N;
                    float r = __fmul_rn(u01(k ? w4.w : w4.y), maj);
                    float mu = __fmul_rn(rho, c_lerp(tm + TP_TOT * N, l));
                    if (r <= mu) {
                        float vc = c_lerp(tm + TP_C * N, l), vp = c_lerp(tm + TP_PP * N, l);
                        chan = r < __fmul_rn(rho, vc) ? 0 : (r < __fmul_rn(rho, __fadd_rn(vc, vp)) ? 1 : 2);
                        vox = vi; done = true;
                    }
                }
            }
        }
        vox_out[h] = vox;
        if (chan_out) chan_out[h] = chan;
    }
}

// =================================================================================================
// particle-list source ("phase-space file ... or a user CPU/GPU function"): histories
// [h_first, h_first + n) are the listed particles themselves.  One thread per particle: locate the voxel (floor
// rule, R25), book the source / escaped energy, push a queue record (track id (0,0)) to the queue of its type.
// =================================================================================================
struct ListParticle { float x, y, z, u, v, w, E; int32_t particle; };  // = mc_particle (include/mc.h)
// validation of a device-resident list (a host list is checked on the host): flags |= 1 energy not in (0, e_max],
// 2 direction not a unit vector, 4 unknown particle type
__global__ void __launch_bounds__(kThreads) check_particles_kernel(const ListParticle* __restrict__ list, uint32_t n, float e_max,
                                                                   uint32_t* flags) {
    uint32_t bad = 0u;
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const ListParticle p = list[i];
        if (!(p.E > 0.0f) || !(p.E <= e_max)) bad |= 1u;
        const float nn = p.u * p.u + p.v * p.v + p.w * p.w;
        if (!(fabsf(nn - 1.0f) < 1e-3f)) bad |= 2u;
        if (p.particle < -1 || p.particle > 1) bad |= 4u;
    }
    bad = __reduce_or_sync(kFull, bad);
    if ((threadIdx.x & 31) == 0 && bad) atomicOr(flags, bad);
}

// list[0] is the record of history list_h0 (0 for a whole list, the first history of the wave for a source function's buffer).
__global__ void __launch_bounds__(kThreads) load_particles_kernel(const __grid_constant__ RunParams P, const ListParticle* __restrict__ list,
                                                                  unsigned long long list_h0, uint32_t n) {
    const Geometry& g = P.g;
    double e_src = 0.0, e_esc = 0.0;
    uint32_t n_hist = 0;
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const unsigned long long h = P.h_first + i;
        const ListParticle p = list[h - list_h0];
        const uint32_t code = p.particle == 0 ? CODE_PHOTON : (p.particle > 0 ? CODE_POSITRON : CODE_ELECTRON);
        const float e0 = p.E + (code == CODE_POSITRON ? 2.0f * kMeF : 0.0f);
        e_src += (double)e0; ++n_hist;
        float gx = __fmul_rn(__fsub_rn(p.x, g.ox), g.ihx), gy = __fmul_rn(__fsub_rn(p.y, g.oy), g.ihy), gz = __fmul_rn(__fsub_rn(p.z, g.oz), g.ihz);
        const bool inside = gx >= 0.0f && gx < (float)g.nx && gy >= 0.0f && gy < (float)g.ny && gz >= 0.0f && gz < (float)g.nz;
        if (!inside) { e_esc += (double)e0; continue; }
        QRec r; r.x = p.x; r.y = p.y; r.z = p.z; r.u = p.u; r.v = p.v; r.w = p.w; r.E = p.E;
        r.hist = (uint32_t)h; r.trk_lo = 0u; r.trk_hi = 0u;
        r.vox = (int)gx + g.nx * ((int)gy + g.ny * (int)gz);
        r.tag = (batch_of(h, P.n_batches, P.n_total, P.inv_n_total) << 2) | code;
        push_record2(P.q_e_out, P.q_p_out, code != CODE_PHOTON, P.counters + C_OVERFLOW, r);
    }
    e_src = warp_sum(e_src); e_esc = warp_sum(e_esc);
    unsigned long long nh = warp_sum(n_hist);
    if ((threadIdx.x & 31) == 0) {
        stat_add(P.stats, S_HIST, nh);
        if (e_src != 0.0) atomicAdd(P.ledger + LG_SRC, e_src);
        if (e_esc != 0.0) atomicAdd(P.ledger + LG_ESC, e_esc);
    }
}

// =================================================================================================
// batch statistics (S9; R17, R18): D_b = E_b / (rho V N_b), mean over batches, standard error of the mean
// =================================================================================================
__device__ __forceinline__ double batch_size(unsigned long long n_total, int B, int b) {
    unsigned long long lo = ((unsigned long long)b * n_total + B - 1) / B, hi = ((unsigned long long)(b + 1) * n_total + B - 1) / B;
    return (double)(hi - lo);
}
__global__ void __launch_bounds__(kThreads) finalize_kernel(const float* __restrict__ edep, const uint2* __restrict__ vox, int nvox,
                                                            int B, unsigned long long n_total, double voxel_volume,
                                                            float* __restrict__ dose, float* __restrict__ sigma) {
    extern __shared__ double s_inv_nb[];
    for (int b = threadIdx.x; b < B; b += blockDim.x) s_inv_nb[b] = 1.0 / batch_size(n_total, B, b);
    __syncthreads();
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < nvox; i += gridDim.x * blockDim.x) {
        double inv_mass = 1.0 / ((double)__uint_as_float(vox[i].x) * voxel_volume);
        double mean = 0.0;
        for (int b = 0; b < B; ++b) mean += (double)edep[(size_t)b * nvox + i] * inv_mass * s_inv_nb[b];
        mean /= B;
        double ss = 0.0;
        for (int b = 0; b < B; ++b) { double dlt = (double)edep[(size_t)b * nvox + i] * inv_mass * s_inv_nb[b] - mean; ss += dlt * dlt; }
        dose[i] = (float)mean;
        sigma[i] = B > 1 ? (float)sqrt(ss / ((double)B * (B - 1))) : 0.0f;
    }
}

// Fused exchange + statistics for the sharded job: the per-batch energy of a
// voxel is the SUM over the ranks' grids, read in place — grids[r] may be this device's memory or a peer's, mapped
// through CUDA IPC / peer access, in which case the loads travel over NVLink.  One pass: no all-reduce, no summed copy.
constexpr int kMaxGrids = 16;
struct GridList { const float* g[kMaxGrids]; int n; };
__global__ void __launch_bounds__(kThreads) finalize_multi_kernel(const __grid_constant__ GridList grids, const uint2* __restrict__ vox,
                                                                  int nvox, int v_begin, int v_end, int B, unsigned long long n_total,
                                                                  double voxel_volume, float* __restrict__ dose, float* __restrict__ sigma) {
    extern __shared__ double s_inv_nb[];
    for (int b = threadIdx.x; b < B; b += blockDim.x) s_inv_nb[b] = 1.0 / batch_size(n_total, B, b);
    __syncthreads();
    // voxels [v_begin, v_end): with one slice per rank every grid value crosses NVLink once (reduce-scatter shape)
    for (int i = v_begin + blockIdx.x * blockDim.x + threadIdx.x; i < v_end; i += gridDim.x * blockDim.x) {
        const double inv_mass = 1.0 / ((double)__uint_as_float(vox[i].x) * voxel_volume);
        double mean = 0.0, sq = 0.0;
        for (int b = 0; b < B; ++b) {
            double e = 0.0;
            for (int r = 0; r < grids.n; ++r) e += (double)__ldg(grids.g[r] + (size_t)b * nvox + i);
            const double d = e * inv_mass * s_inv_nb[b];
            mean += d; sq += d * d;
        }
        mean /= B;
        const double ss = fmax(sq - (double)B * mean * mean, 0.0);  // sum of squared deviations from the mean
        dose[i] = (float)mean;
        sigma[i] = B > 1 ? (float)sqrt(ss / ((double)B * (B - 1))) : 0.0f;
    }
}

// total of a float array in fp64 (energy ledger: deposited energy = sum of the batch grids)
__global__ void __launch_bounds__(kThreads) sum_kernel(const float* __restrict__ a, size_t n, double* out) {
    double s = 0.0;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) s += (double)a[i];
    s = warp_sum(s);
    __shared__ double part[kThreads / 32];
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int i = 0; i < kThreads / 32; ++i) t += part[i];
        atomicAdd(out, t);
    }
}

__global__ void philox_test_kernel(const uint32_t* ctr, const uint32_t* key, int n, uint32_t* out) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    uint4 r = philox4x32_10(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], key[2 * i], key[2 * i + 1]);
    out[4 * i] = r.x; out[4 * i + 1] = r.y; out[4 * i + 2] = r.z; out[4 * i + 3] = r.w;
}

// u01f against its defining expression ((w >> 9) + 0.5) * 2^-23 for every 23-bit value, with the 9 discarded bits all
// zero and all one: counts the words whose results differ in any bit.
__global__ void u01_test_kernel(unsigned long long* mismatches) {
    unsigned int bad = 0;
    for (uint32_t m = blockIdx.x * blockDim.x + threadIdx.x; m < (1u << 23); m += gridDim.x * blockDim.x)
        for (uint32_t low = 0; low < 2; ++low) {
            const uint32_t w = (m << 9) | (low ? 0x1ffu : 0u);
            const float ref = __fmaf_rn(__uint2float_rn(w >> 9), 1.1920928955078125e-07f, 5.9604644775390625e-08f);
            if (__float_as_uint(u01f(w)) != __float_as_uint(ref) || __float_as_uint(u01(w)) != __float_as_uint(ref)) ++bad;
        }
    if (bad) atomicAdd(mismatches, (unsigned long long)bad);
}

// L2 reduction micro-benchmark (scoring roofline): every thread issues `per_thread`
// red.global.add.f32 to pseudo-random cells of a window of `n_cells` floats (mode 0), or all lanes of a
// warp to one cell (mode 1).
__global__ void __launch_bounds__(kThreads) red_bench_kernel(float* grid, uint32_t n_cells, int per_thread, int mode) {
    uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t s = (mode == 1 ? (t >> 5) : t) * 2654435761u + 12345u;
    for (int i = 0; i < per_thread; ++i) {
        s = s * 1664525u + 1013904223u;
        uint32_t c = (uint32_t)(((unsigned long long)(s ^ (s >> 15)) * n_cells) >> 32);
        atomicAdd(grid + c, 1.0f);
    }
}

// Issue-rate micro-benchmark (transport roofline): 8 independent FFMA chains per thread,
// `iters` x 64 FFMA each; 1024 threads per CTA keep every scheduler supplied.  Reports thread-instructions / s.
__global__ void __launch_bounds__(1024) issue_bench_kernel(float* out, int iters) {
    float a0 = threadIdx.x * 1e-3f, a1 = a0 + 1.f, a2 = a0 + 2.f, a3 = a0 + 3.f, a4 = a0 + 4.f, a5 = a0 + 5.f, a6 = a0 + 6.f, a7 = a0 + 7.f;
    const float m = 0.999f, c = 1e-3f;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            a0 = fmaf(a0, m, c); a1 = fmaf(a1, m, c); a2 = fmaf(a2, m, c); a3 = fmaf(a3, m, c);
            a4 = fmaf(a4, m, c); a5 = fmaf(a5, m, c); a6 = fmaf(a6, m, c); a7 = fmaf(a7, m, c);
        }
    }
    float r = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
    if (r == 123456.f) out[0] = r;  // never true: keeps the chains alive
}

}  // namespace mcb
