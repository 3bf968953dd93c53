// Transport, scoring and statistics kernels (sm_100a).  One warp lane = one particle track; lanes
// refill themselves from the input queue / the source while the kernel runs.
//   electron_kernel : Class II condensed-history steps, d = min[d_vox, d_maxs, d_maxe, d_event]
//                     (PAPER.md:39), Moller / bremsstrahlung hard events, random-hinge MS deflection,
//                     CSDA loss through the range table, dose by red.global.add.f32
//   photon_kernel   : Woodcock flights, Compton / pair / photoelectric
//   atten_kernel    : attenuation-only mode under the fp32 arithmetic contract (R20)
//   finalize_kernel : batch means and standard errors (R17, R18)
#pragma once
#include "mc_device.cuh"

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

// Table coordinate (node + fraction) of the energy whose residual range is Rt: exact inverse of the
// piecewise-linear (in ln T) range interpolant (R5); search starts at a first-order guess.
__device__ __forceinline__ float inv_range_coord(const float2* R, float Rt, int guess, int k_cut, int N) {
    if (Rt <= 0.0f) return (float)k_cut;
    int lo = min(max(guess, k_cut), N - 2);
    while (lo > k_cut && R[lo].x > Rt) --lo;
    while (lo < N - 2 && R[lo + 1].x <= Rt) ++lo;
    float2 a = R[lo];
    float f = __fdividef(Rt - a.x, a.y);
    return (float)lo + fminf(fmaxf(f, 0.0f), 1.0f);
}

__device__ __forceinline__ unsigned long long warp_sum(uint32_t v) {
    unsigned long long s = v;
#pragma unroll
    for (int o = 16; o; o >>= 1) s += __shfl_xor_sync(kFull, s, o);
    return s;
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
// =================================================================================================
__global__ void __launch_bounds__(kThreads) electron_kernel(const __grid_constant__ RunParams P) {
    extern __shared__ float2 s_tab[];
    {
        const int ntab = P.n_mat * TE_COUNT * P.N;
        for (int i = threadIdx.x; i < ntab; i += blockDim.x) s_tab[i] = P.tabE[i];
    }
    __syncthreads();
    const int lane = threadIdx.x & 31;
    const int N = P.N, k_cut = P.k_cut;
    const Geometry& g = P.g;
    const bool no_hard = P.flags & 1u, no_ms = P.flags & 2u;

    bool active = false, exhausted = false;
    float x = 0, y = 0, z = 0, u = 0, v = 0, w = 1, T = 0, ex = 0, rho = 1;
    int ix = 0, iy = 0, iz = 0, vox = 0;
    const float2* tm = s_tab;  // tables of the current voxel's material
    int mat = 0;
    Rng rng = {0, 0, 0, 0};
    uint32_t tag = 0, cell0 = 0;  // cell0 = batch * nvox
    Score sc = {0.0f, 0u, 0u};
    uint32_t n_step = 0, n_moller = 0, n_brems = 0, n_sec_e = 0, n_sec_g = 0, n_hist = 0;
    double e_src = 0.0, e_esc = 0.0;

    for (;;) {
        // ---- lane refill: queue first, then new primaries ----
        unsigned want = __ballot_sync(kFull, !active && !exhausted);
        unsigned act = __ballot_sync(kFull, active);
        if (want == 0u && act == 0u) break;
        if (want != 0u && (act == 0u || __popc(want) >= P.refill_lanes)) {
            uint32_t item = claim(P.counters + C_HEAD, want, lane);
            if (!active && !exhausted) {
                if (item < P.n_in) {
                    QRec r = load_record(P.q_in, item);
                    x = r.x; y = r.y; z = r.z; u = r.u; v = r.v; w = r.w; T = r.E;
                    rng.hist = r.hist; rng.trk_lo = r.trk_lo; rng.trk_hi = r.trk_hi; rng.block = 0;
                    vox = r.vox; tag = r.tag;
                    ix = vox % g.nx; int t2 = vox / g.nx; iy = t2 % g.ny; iz = t2 / g.ny;
                    active = true;
                } else if (item < P.n_in + P.n_new) {
                    unsigned long long h = P.h_first + (item - P.n_in);
                    rng.hist = (uint32_t)h; rng.trk_lo = 0; rng.trk_hi = 0; rng.block = 0;
                    uint4 w4 = next_block(rng, P.seed_lo, P.seed_hi);
                    Primary p = sample_primary(P, w4);
                    uint32_t code = P.beam.particle > 0 ? CODE_POSITRON : CODE_ELECTRON;
                    tag = (batch_of(h, P.n_batches, P.n_total) << 2) | code;
                    float e0 = p.E + (code == CODE_POSITRON ? 2.0f * kMeF : 0.0f);
                    e_src += (double)e0; ++n_hist;
                    x = p.x; y = p.y; z = p.z; u = p.u; v = p.v; w = p.w; T = p.E;
                    ix = p.ix; iy = p.iy; iz = p.iz; vox = ix + g.nx * (iy + g.ny * iz);
                    if (p.inside) active = true; else e_esc += (double)e0;
                } else exhausted = true;
                if (active) {
                    uint2 vd = P.vox[vox];
                    rho = __uint_as_float(vd.x); mat = (int)vd.y; tm = s_tab + mat * TE_COUNT * N;
                    cell0 = (tag >> 2) * (uint32_t)g.nvox;
                    ex = (__logf(T) - P.lnE0) * P.inv_dln;
                }
            }
            act = __ballot_sync(kFull, active);
            if (act == 0u) continue;
        }
        if (!active) continue;

        // ---- end of track: absorb below the cut-off; a positron annihilates at rest (R9) -----------
        if (T <= P.e_cut) {
            score_add(sc, P.edep, cell0 + vox, T);
            if ((tag & 3u) == CODE_POSITRON) {
                uint4 a4 = next_block(rng, P.seed_lo, P.seed_hi);
                float mu = 2.0f * u01(a4.z) - 1.0f, sn = sqrtf(fmaxf(1.0f - mu * mu, 0.0f)), sp, cp;
                __sincosf(kTwoPiF * u01(a4.w), &sp, &cp);
                QRec r; r.x = x; r.y = y; r.z = z; r.u = sn * cp; r.v = sn * sp; r.w = mu; r.E = kMeF;
                r.hist = rng.hist; r.trk_lo = a4.x; r.trk_hi = a4.y; r.vox = vox; r.tag = (tag & ~3u) | CODE_PHOTON;
                emit(P, P.q_p_out, sc, cell0 + vox, r, n_sec_g);
                uint4 b4 = next_block(rng, P.seed_lo, P.seed_hi);
                r.u = -r.u; r.v = -r.v; r.w = -r.w; r.trk_lo = b4.x; r.trk_hi = b4.y;
                emit(P, P.q_p_out, sc, cell0 + vox, r, n_sec_g);
            }
            active = false;
            continue;
        }

        // ---- step set-up (S4): d = min[d_vox, d_maxs, d_maxe, d_range, d_event] -------------------------
        ++n_step;
        int i0 = min(max((int)ex, 0), N - 2);
        float f0 = ex - (float)i0;
        float R0 = lerp(tm + TE_R * N, i0, f0), L0 = lerp(tm + TE_L * N, i0, f0), Smax = lerp(tm + TE_SMAX * N, i0, f0);
        uint4 w4 = next_block(rng, P.seed_lo, P.seed_hi);
        int ax;
        float d = face_dist(g, x, y, z, u, v, w, ix, iy, iz, ax);
        int lim = 0;
        float rl = rho * L0;
        float d_maxe = __fdividef(P.f_maxe * T, rl);
        float d_range = __fdividef(fmaxf(R0, 0.0f), rho);
        if (P.d_maxs < d) { d = P.d_maxs; lim = 1; }
        if (d_maxe < d) { d = d_maxe; lim = 2; }
        if (d_range < d) { d = d_range; lim = 3; }
        if (!no_hard) {
            float d_event = __fdividef(-__logf(u01(w4.x)), rho * Smax);
            if (d_event < d) { d = d_event; lim = 4; }
        }
        // ---- random hinge (S5; R7, R8) ----------------------------------------------------------------
        float xi = u01(w4.y), legA = xi * d;
        x = fmaf(legA, u, x); y = fmaf(legA, v, y); z = fmaf(legA, w, z);
        // first-order guess of the table-coordinate shift per unit range: d ex / d R = 1 / (T/L * dln) per g/cm^2
        float dex_dR = __fdividef(L0 * P.inv_dln, T);
        float rd = rho * d;
        if (!no_ms) {
            float Rm = fmaf(-0.5f, rd, R0);
            float em = inv_range_coord(tm + TE_R * N, Rm, (int)(ex - 0.5f * rd * dex_dR), k_cut, N);
            int im = min(max((int)em, 0), N - 2);
            float k1 = lerp(tm + TE_K1 * N, im, em - (float)im);
            float t = k1 * rd;
            float am = t < 1e-3f ? t * (1.0f - 0.5f * t) : 1.0f - __expf(-t);
            if (am > 0.0f) {
                float omu = -am * __logf(1.0f - u01(w4.z) * (1.0f - __expf(__fdividef(-2.0f, am))));
                rotate(u, v, w, fminf(omu, 2.0f), kTwoPiF * u01(w4.w));
            }
        }
        float rest = d - legA;
        float tf = face_dist(g, x, y, z, u, v, w, ix, iy, iz, ax);
        bool cross = tf <= rest;
        float legB = cross ? tf : rest;
        x = fmaf(legB, u, x); y = fmaf(legB, v, y); z = fmaf(legB, w, z);
        float d_act = legA + legB;
        // ---- CSDA loss through the range table (S6; R5) + scoring ---------------------------------------
        float T1, ex1;
        if (lim == 3 && !cross) { T1 = P.e_cut; ex1 = (float)k_cut; }
        else {
            float ra = rho * d_act;
            ex1 = inv_range_coord(tm + TE_R * N, fmaf(-rho, d_act, R0), (int)(ex - ra * dex_dR), k_cut, N);
            T1 = fminf(__expf(fmaf(ex1, P.dln, P.lnE0)), T);
        }
        score_add(sc, P.edep, cell0 + vox, T - T1);
        T = T1; ex = ex1;
        if (cross) {
            // move to the neighbour voxel, coordinate snapped to the face (R8)
            int dir;
            if (ax == 0) { dir = u > 0.0f ? 1 : -1; ix += dir; x = fmaf((float)(ix + (dir > 0 ? 0 : 1)), g.hx, g.ox); vox += dir; }
            else if (ax == 1) { dir = v > 0.0f ? 1 : -1; iy += dir; y = fmaf((float)(iy + (dir > 0 ? 0 : 1)), g.hy, g.oy); vox += dir * g.nx; }
            else { dir = w > 0.0f ? 1 : -1; iz += dir; z = fmaf((float)(iz + (dir > 0 ? 0 : 1)), g.hz, g.oz); vox += dir * g.nx * g.ny; }
            if ((unsigned)ix >= (unsigned)g.nx || (unsigned)iy >= (unsigned)g.ny || (unsigned)iz >= (unsigned)g.nz) {
                e_esc += (double)(T + ((tag & 3u) == CODE_POSITRON ? 2.0f * kMeF : 0.0f));
                active = false;
                continue;
            }
            uint2 vd = P.vox[vox];
            rho = __uint_as_float(vd.x);
            if ((int)vd.y != mat) { mat = (int)vd.y; tm = s_tab + mat * TE_COUNT * N; }
            continue;
        }
        if (lim != 4 || T <= P.e_cut) continue;

        // ---- hard-event candidate (S7): thinning against the running-max majorant (R6) -------------------
        uint4 h4 = next_block(rng, P.seed_lo, P.seed_hi);
        float r = u01(h4.x) * Smax;
        int i1 = min(max((int)ex, 0), N - 2);
        float f1 = ex - (float)i1;
        float SH = lerp(tm + TE_SHARD * N, i1, f1);
        if (r >= SH) continue;  // fictitious
        float SM = lerp(tm + TE_SM * N, i1, f1);
        float phi = kTwoPiF * u01(h4.w);
        float T0 = T;
        QRec q; q.x = x; q.y = y; q.z = z; q.u = u; q.v = v; q.w = w; q.hist = rng.hist; q.trk_lo = h4.y; q.trk_hi = h4.z; q.vox = vox;
        if (r < SM) {  // Moller (R10)
            ++n_moller;
            float tau = T0 * (1.0f / kMeF), gm = tau + 1.0f, ig2 = __fdividef(1.0f, gm * gm);
            float qq = (2.0f * gm - 1.0f) * ig2, q1 = tau * tau * ig2;
            float ec = __fdividef(P.e_cut, T0), iec = __fdividef(T0, P.e_cut);
            auto gf = [&](float e) { float o = __fdividef(1.0f, 1.0f - e); return 1.0f - qq * e * o + e * e * (q1 + o * o); };
            float gmax = fmaxf(gf(ec), gf(0.5f)), eps;
            for (;;) {
                uint4 m4 = next_block(rng, P.seed_lo, P.seed_hi);
                eps = __fdividef(1.0f, iec - u01(m4.x) * (iec - 2.0f));
                if (u01(m4.y) * gmax <= gf(eps)) break;
                eps = __fdividef(1.0f, iec - u01(m4.z) * (iec - 2.0f));
                if (u01(m4.w) * gmax <= gf(eps)) break;
            }
            float W = eps * T0, Tp = T0 - W, t2m = T0 + 2.0f * kMeF;
            float c1 = sqrtf(__fdividef(Tp * t2m, T0 * (Tp + 2.0f * kMeF)));
            float c2 = sqrtf(__fdividef(W * t2m, T0 * (W + 2.0f * kMeF)));
            q.E = W; q.tag = (tag & ~3u) | CODE_ELECTRON;
            rotate(q.u, q.v, q.w, 1.0f - c2, phi + 3.14159265358979f);
            rotate(u, v, w, 1.0f - c1, phi);
            T = Tp;
            emit(P, P.q_e_out, sc, cell0 + vox, q, n_sec_e);
        } else {  // bremsstrahlung (R11)
            ++n_brems;
            float Et = T0 + kMeF, lscr = P.lscr[mat], iEt = __fdividef(1.0f, Et);
            auto Ff = [&](float k) {
                float Ep = Et - k, rr = Ep * iEt;
                return (1.0f + rr * rr - (2.0f / 3.0f) * rr) * (fminf(__logf(__fdividef(2.0f * Et * Ep, kMeF * k)), lscr) - 0.5f);
            };
            float Fmax = (4.0f / 3.0f) * (fminf(__logf(__fdividef(2.0f * Et * (Et - P.g_cut), kMeF * P.g_cut)), lscr) - 0.5f);
            float lr = __logf(__fdividef(T0, P.g_cut)), kk;
            for (;;) {
                uint4 m4 = next_block(rng, P.seed_lo, P.seed_hi);
                kk = fminf(P.g_cut * __expf(lr * u01(m4.x)), T0);
                if (u01(m4.y) * Fmax <= Ff(kk)) break;
                kk = fminf(P.g_cut * __expf(lr * u01(m4.z)), T0);
                if (u01(m4.w) * Fmax <= Ff(kk)) break;
            }
            q.E = kk; q.tag = (tag & ~3u) | CODE_PHOTON;
            float sh = __sinf(0.5f * kMeF * iEt);
            rotate(q.u, q.v, q.w, 2.0f * sh * sh, phi);
            T = T0 - kk;
            emit(P, P.q_p_out, sc, cell0 + vox, q, n_sec_g);
        }
        ex = (__logf(fmaxf(T, 1e-30f)) - P.lnE0) * P.inv_dln;
    }
    // ---- warp exit: flush the pending deposit, reduce the counters ---------------------------------------
    score_flush(sc, P.edep);
    unsigned long long s_moller = warp_sum(n_moller), s_brems = warp_sum(n_brems), s_se = warp_sum(n_sec_e),
                       s_sg = warp_sum(n_sec_g), s_red = warp_sum(sc.n_red), s_hist = warp_sum(n_hist),
                       s_step = warp_sum(n_step);
    double s_src = warp_sum(e_src), s_esc = warp_sum(e_esc);
    if (lane == 0) {
        stat_add(P.stats, S_ESTEP, s_step); stat_add(P.stats, S_MOLLER, s_moller); stat_add(P.stats, S_BREMS, s_brems);
        stat_add(P.stats, S_SEC_E, s_se); stat_add(P.stats, S_SEC_G, s_sg); stat_add(P.stats, S_ATOMICS, s_red);
        stat_add(P.stats, S_HIST, s_hist);
        if (s_src != 0.0) atomicAdd(P.ledger + LG_SRC, s_src);
        if (s_esc != 0.0) atomicAdd(P.ledger + LG_ESC, s_esc);
    }
}

// =================================================================================================
// photon kernel: Woodcock tracking (R3), Compton (R4), pair (R12),
// photoelectric absorption (R16).  One Philox block serves two flights.
// =================================================================================================
__global__ void __launch_bounds__(kThreads) photon_kernel(const __grid_constant__ RunParams P) {
    extern __shared__ float2 s_tab[];
    {
        const int ntab = (1 + P.n_mat * TP_COUNT) * P.N;
        for (int i = threadIdx.x; i < ntab; i += blockDim.x) s_tab[i] = P.tabP[i];
    }
    __syncthreads();
    const int lane = threadIdx.x & 31;
    const int N = P.N;
    const Geometry& g = P.g;

    bool active = false, exhausted = false;
    float x = 0, y = 0, z = 0, u = 0, v = 0, w = 1, E = 0, lf = 0, maj = 1;
    int li = 0;
    Rng rng = {0, 0, 0, 0};
    uint32_t tag = 0, cell0 = 0;
    Score sc = {0.0f, 0u, 0u};
    uint32_t n_flight = 0, n_fict = 0, n_compton = 0, n_pair = 0, n_pe = 0, n_sec_e = 0, n_hist = 0;
    double e_src = 0.0, e_esc = 0.0;

    for (;;) {
        unsigned want = __ballot_sync(kFull, !active && !exhausted);
        unsigned act = __ballot_sync(kFull, active);
        if (want == 0u && act == 0u) break;
        if (want != 0u && (act == 0u || __popc(want) >= P.refill_lanes)) {
            uint32_t item = claim(P.counters + C_HEAD, want, lane);
            if (!active && !exhausted) {
                int vox = 0;
                if (item < P.n_in) {
                    QRec r = load_record(P.q_in, item);
                    x = r.x; y = r.y; z = r.z; u = r.u; v = r.v; w = r.w; E = r.E;
                    rng.hist = r.hist; rng.trk_lo = r.trk_lo; rng.trk_hi = r.trk_hi; rng.block = 0;
                    vox = r.vox; tag = r.tag;
                    active = true;
                } else if (item < P.n_in + P.n_new) {
                    unsigned long long h = P.h_first + (item - P.n_in);
                    rng.hist = (uint32_t)h; rng.trk_lo = 0; rng.trk_hi = 0; rng.block = 0;
                    uint4 w4 = next_block(rng, P.seed_lo, P.seed_hi);
                    Primary p = sample_primary(P, w4);
                    tag = (batch_of(h, P.n_batches, P.n_total) << 2) | CODE_PHOTON;
                    e_src += (double)p.E; ++n_hist;
                    x = p.x; y = p.y; z = p.z; u = p.u; v = p.v; w = p.w; E = p.E;
                    vox = p.ix + g.nx * (p.iy + g.ny * p.iz);
                    if (p.inside) active = true; else e_esc += (double)p.E;
                } else exhausted = true;
                if (active) {
                    cell0 = (tag >> 2) * (uint32_t)g.nvox;
                    if (E < P.g_cut) {  // absorbed where it was born
                        score_add(sc, P.edep, cell0 + vox, E);
                        active = false;
                    } else {
                        float t = (__logf(E) - P.lnE0P) * P.inv_dlnP;
                        li = min(max((int)t, 0), N - 2); lf = t - (float)li;
                        maj = lerp(s_tab, li, lf);
                    }
                }
            }
            act = __ballot_sync(kFull, active);
            if (act == 0u) continue;
        }
        if (!active) continue;

        uint4 w4 = next_block(rng, P.seed_lo, P.seed_hi);
        int chan = -1, vox = 0;
        float rho = 0.0f;
        const float2* tm = s_tab;
        float imaj = __fdividef(1.0f, maj);
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            float sl = -__logf(u01(k ? w4.z : w4.x)) * imaj;
            x = fmaf(sl, u, x); y = fmaf(sl, v, y); z = fmaf(sl, w, z);
            ++n_flight;
            float gx = (x - g.ox) * g.ihx, gy = (y - g.oy) * g.ihy, gz = (z - g.oz) * g.ihz;
            if (!(gx >= 0.0f && gx < (float)g.nx && gy >= 0.0f && gy < (float)g.ny && gz >= 0.0f && gz < (float)g.nz)) {
                e_esc += (double)E; active = false; break;
            }
            vox = (int)gx + g.nx * ((int)gy + g.ny * (int)gz);
            uint2 vd = P.vox[vox];
            rho = __uint_as_float(vd.x);
            tm = s_tab + (1 + (int)vd.y * TP_COUNT) * N;
            float r = u01(k ? w4.w : w4.y) * maj;
            float mu = rho * lerp(tm + TP_TOT * N, li, lf);
            if (r > mu) { ++n_fict; continue; }
            float mc = rho * lerp(tm + TP_C * N, li, lf), mp = rho * lerp(tm + TP_PP * N, li, lf);
            chan = r < mc ? 0 : (r < mc + mp ? 1 : 2);
            break;
        }
        if (chan < 0) continue;
        uint32_t cell = cell0 + (uint32_t)vox;
        if (chan == 2) {  // photoelectric: absorbed locally
            ++n_pe;
            score_add(sc, P.edep, cell, E);
            active = false;
            continue;
        }
        QRec q; q.x = x; q.y = y; q.z = z; q.hist = rng.hist; q.vox = vox;
        if (chan == 1) {  // pair: both along the photon direction, uniform split
            ++n_pair;
            uint4 a4 = next_block(rng, P.seed_lo, P.seed_hi);
            float Tk = E - 2.0f * kMeF, us = u01(a4.z);
            q.u = u; q.v = v; q.w = w;
            q.E = us * Tk; q.trk_lo = a4.x; q.trk_hi = a4.y; q.tag = (tag & ~3u) | CODE_ELECTRON;
            emit(P, P.q_e_out, sc, cell, q, n_sec_e);
            uint4 b4 = next_block(rng, P.seed_lo, P.seed_hi);
            q.E = Tk - q.E; q.trk_lo = b4.x; q.trk_hi = b4.y; q.tag = (tag & ~3u) | CODE_POSITRON;
            emit(P, P.q_e_out, sc, cell, q, n_sec_e);
            active = false;
            continue;
        }
        // Compton: Klein-Nishina by the epsilon decomposition (R4)
        ++n_compton;
        float k0 = E * (1.0f / kMeF), e0 = __fdividef(1.0f, 1.0f + 2.0f * k0), e02 = e0 * e0;
        float a1 = -__logf(e0), a2 = 0.5f * (1.0f - e02), ik0 = __fdividef(1.0f, k0);
        float eps, tt;
        for (;;) {
            uint4 c4 = next_block(rng, P.seed_lo, P.seed_hi);
            float u1 = u01(c4.y);
            if (u01(c4.x) * (a1 + a2) < a1) eps = __expf(-a1 * u1);
            else eps = sqrtf(fmaf(1.0f - e02, u1, e02));
            tt = __fdividef(1.0f - eps, eps) * ik0;
            float sin2 = tt * (2.0f - tt);
            if (u01(c4.z) <= 1.0f - __fdividef(eps * sin2, 1.0f + eps * eps)) break;
        }
        uint4 d4 = next_block(rng, P.seed_lo, P.seed_hi);
        float E1 = eps * E, Te = E - E1;
        float u0 = u, v0 = v, w0 = w;
        rotate(u, v, w, tt, kTwoPiF * u01(d4.z));
        if (Te >= P.e_cut || (P.flags & 4u)) {
            float qx = E * u0 - E1 * u, qy = E * v0 - E1 * v, qz = E * w0 - E1 * w;
            float inr = rsqrtf(fmaf(qx, qx, fmaf(qy, qy, qz * qz)));
            q.u = qx * inr; q.v = qy * inr; q.w = qz * inr;
            q.E = Te; q.trk_lo = d4.x; q.trk_hi = d4.y; q.tag = (tag & ~3u) | CODE_ELECTRON;
            emit(P, P.q_e_out, sc, cell, q, n_sec_e);
        } else {
            score_add(sc, P.edep, cell, Te);  // born below the cut-off: absorbed where it is born (R26)
        }
        E = E1;
        if (E < P.g_cut) { score_add(sc, P.edep, cell, E); active = false; continue; }
        float t = (__logf(E) - P.lnE0P) * P.inv_dlnP;
        li = min(max((int)t, 0), N - 2); lf = t - (float)li;
        maj = lerp(s_tab, li, lf);
    }
    score_flush(sc, P.edep);
    unsigned long long s_fl = warp_sum(n_flight), s_fi = warp_sum(n_fict), s_c = warp_sum(n_compton), s_p = warp_sum(n_pair),
                       s_pe = warp_sum(n_pe), s_se = warp_sum(n_sec_e), s_red = warp_sum(sc.n_red), s_hist = warp_sum(n_hist);
    double s_src = warp_sum(e_src), s_esc = warp_sum(e_esc);
    if (lane == 0) {
        stat_add(P.stats, S_FLIGHT, s_fl); stat_add(P.stats, S_FICT, s_fi); stat_add(P.stats, S_COMPTON, s_c);
        stat_add(P.stats, S_PAIR, s_p); stat_add(P.stats, S_PE, s_pe); stat_add(P.stats, S_SEC_E, s_se);
        stat_add(P.stats, S_ATOMICS, s_red); stat_add(P.stats, S_HIST, s_hist);
        if (s_src != 0.0) atomicAdd(P.ledger + LG_SRC, s_src);
        if (s_esc != 0.0) atomicAdd(P.ledger + LG_ESC, s_esc);
    }
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

}  // namespace mcb
