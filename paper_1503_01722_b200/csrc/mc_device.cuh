// Device-side building blocks of the transport kernels (sm_100a).
//   - Philox4x32-10, block-granular streams (R15)
//   - the fp32 arithmetic contract used by source sampling and the photon Woodcock flight
//     (R20): explicit round-to-nearest intrinsics only, never contracted
//   - shared-memory table lookups ((value, slope) pairs, one LDS.64 per lerp)
//   - queue records and warp-aggregated queue push
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace mcb {

constexpr int MAX_MAT = 16;  // the paper's database holds 16 materials
constexpr float kMeF = 0.51099895f;
constexpr float kTwoPiF = 6.28318530717958647692f;

// ---- single-instruction MUFU wrappers (approx, flush-to-zero): the transport kernels' fast math ------------
__device__ __forceinline__ float f_rcp(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float f_lg2(float x) { float r; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float f_ex2(float x) { float r; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float f_sqrt(float x) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float f_rsqrt(float x) { float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float f_sin(float x) { float r; asm("sin.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float f_cos(float x) { float r; asm("cos.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
constexpr float kLn2F = 0.69314718055994530942f;
constexpr float kLog2eF = 1.44269504088896340736f;
__device__ __forceinline__ float f_ln(float x) { return f_lg2(x) * kLn2F; }
__device__ __forceinline__ float f_exp(float x) { return f_ex2(x * kLog2eF); }

// ---- parameters handed to every kernel by value ------------------------------------------------
struct Geometry {
    int nx, ny, nz, nvox;
    float hx, hy, hz, ox, oy, oz, ihx, ihy, ihz;  // ih = 1.0f / h (IEEE fp32 division on the host)
};
struct BeamDev {
    int particle, shape, n_nodes;
    float ex, ey, ez, ax, ay, az, ssd, fx, fy;
    const float* E_nodes;  // device
    const float* pdf_nodes;
    const float* cdf;      // normalised cumulative trapezoid areas (fp64 on the host, rounded)
};
struct QRec {  // 48 bytes = 3 x 16-byte words
    float x, y, z, u;
    float v, w, E; uint32_t hist;
    uint32_t trk_lo, trk_hi; int32_t vox; uint32_t tag;  // tag = (batch << 2) | charge code (0 e-, 1 e+, 2 photon)
};
struct Queue {
    uint4* rec;       // capacity * 3 uint4
    uint32_t* count;  // device counter (tail)
    uint32_t cap;
};
enum Counter { C_HEAD = 0, C_E_A, C_E_B, C_P, C_OVERFLOW, C_DONE, C_FLAGS, C_COUNT };  // C_FLAGS: validation flags of a source function's records;  // C_DONE: CTAs of the running launch that have finished
enum StatId {
    S_ESTEP = 0, S_FLIGHT, S_FICT, S_COMPTON, S_PAIR, S_PE, S_MOLLER, S_BREMS, S_SEC_E, S_SEC_G, S_ATOMICS,
    S_HIST, S_COUNT
};
enum LedgerId { LG_SRC = 0, LG_ESC, LG_DEP, LG_COUNT };
// electron tables per material, node-interleaved so that one 16-byte load serves a look-up (float2 units, N = nodes):
//   [0, 2N)  float4 (R, dR, L, dL)            step start            (d = slope to the next node)
//   [2N, 4N) float4 (R, 1/dR, K1, dK1)        inverse-range probes + K1 at the probed node
//   [4N, 6N) float4 (S_hard, d, S_Moller, d)  hard-event thinning
//   [6N, 7N) float2 (S_max, d)                d_event
constexpr int kETabUnits = 7;  // float2 per node and material; the per-material stride is rounded up to 16 bytes
enum { TP_TOT = 0, TP_C, TP_PP, TP_COUNT };                         // photon tables per material (after mu_maj)
enum { CODE_ELECTRON = 0u, CODE_POSITRON = 1u, CODE_PHOTON = 2u };
struct RunParams {
    Geometry g;
    BeamDev beam;
    const uint2* vox;    // per voxel: (density bits, material index)
    const float2* tabP;  // photon tables, (value, slope): [0] mu_maj, then per material mu_tot, mu_C, mu_pp
    const float2* tabE;  // electron tables per material (layout: kETabUnits above)
    int N, n_mat, k_cut;
    int e_stride;        // float2 per material in tabE
    float lnE0, dln, inv_dln, e_cut, g_cut, d_maxs, f_maxe;
    float lnE0P, inv_dlnP;  // grid of the photon tables (may be user supplied, mc_set_photon_tables)
    float lscr[MAX_MAT];
    uint32_t flags;
    float* edep;  // [n_batches][nvox]
    unsigned long long n_total, h_first;  // job size; first primary history of this launch
    unsigned long long inv_n_total;       // floor(2^64 / n_total), see batch_of
    int n_batches;
    uint32_t seed_lo, seed_hi;
    uint32_t n_new;           // new primaries to generate (the queued particles to consume = *q_in.count, read on the device)
    Queue q_in, q_e_out, q_p_out;
    uint32_t* counters;       // Counter
    unsigned long long* stats;  // StatId
    double* ledger;           // e_src, e_dep, e_esc
    int refill_lanes, aggregate;
    int hard_lanes;           // lanes of a warp that must hold a pending hard event before the warp runs that block
    // table coordinate <-> energy in base 2: ex = lg2(T) * ex_a - ex_b;  T = ex2(ex * t_a + t_b)
    float ex_a, ex_b, t_a, t_b;
    uint32_t seed_rk[10];     // seed_lo + r * 0xBB67AE85: Philox round keys of the second key word
    // Goudsmit-Saunderson angle (flags & 8; R27): quantile table (log2 of 1 - cos theta) followed by the per-material
    // coarse (every 8th node) ln A table as (value, slope) pairs; 1 - exp(-t) at the t-nodes; grid constants
    const float* gs;
    int gs_words, gs_n8;      // floats to stage; coarse ln A entries per material
    float gs_an[16];
    float gs_c0, gs_inv_dc, gs_lnA0, gs_inv_dA;
    float hinge_overrun;      // DESIGN.md R8
    int ms_carry;             // DESIGN.md R8b
};

// ---- Philox4x32-10 -----------------------------------------------------------------------------
struct Rng {
    uint32_t hist, trk_lo, trk_hi, block;
};
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        uint32_t h0 = __umulhi(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
        uint32_t h1 = __umulhi(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
        c0 = h1 ^ c1 ^ k0; c1 = l1; c2 = h0 ^ c3 ^ k1; c3 = l0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return make_uint4(c0, c1, c2, c3);
}
// Same generator with the round keys of the second key word (seed_lo + r * 0xBB67AE85, launch constants) read from
// `rk` instead of being recomputed per block.
__device__ __forceinline__ uint4 philox4x32_10_rk(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, const uint32_t (&rk)[10]) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        uint32_t h0 = __umulhi(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
        uint32_t h1 = __umulhi(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
        c0 = h1 ^ c1 ^ k0; c1 = l1; c2 = h0 ^ c3 ^ rk[r]; c3 = l0;
        k0 += 0x9E3779B9u;
    }
    return make_uint4(c0, c1, c2, c3);
}
__device__ __forceinline__ uint4 next_block(Rng& r, uint32_t seed_lo, uint32_t seed_hi) {
    uint4 w = philox4x32_10(r.block, r.trk_lo, r.trk_hi, seed_hi, r.hist, seed_lo);
    ++r.block;
    return w;
}
__device__ __forceinline__ uint4 next_block_rk(Rng& r, const RunParams& P) {
    uint4 w = philox4x32_10_rk(r.block, r.trk_lo, r.trk_hi, P.seed_hi, r.hist, P.seed_rk);
    ++r.block;
    return w;
}
// u = ((w >> 9) + 0.5) * 2^-23 in (0, 1): exact in fp32
__device__ __forceinline__ float u01(uint32_t w) { return __fmul_rn(__fadd_rn((float)(w >> 9), 0.5f), 1.1920928955078125e-07f); }

// Same value as u01, without the integer-to-float conversion (a quarter-rate XU instruction): one funnel shift puts the 23
// bits under the exponent of 1.0, f = 1 + m 2^-23 in [1, 2), and f - (1 - 2^-24) = (2m + 1) 2^-24 is exact in fp32 (both
// operands and the result are representable, so the subtraction rounds nothing).  Checked for all 2^23 values on the
// device by mc_u01_selftest.
__device__ __forceinline__ float u01f(uint32_t w) { return __fsub_rn(__uint_as_float(__funnelshift_r(w, 0x7fu, 9)), 0.99999994f); }

// ---- fp32 arithmetic contract (R20) -----------------------------------------------------------
__device__ __forceinline__ float c_ln(float x) {
    uint32_t b = __float_as_uint(x);
    int e = (int)(b >> 23) - 127;
    float m = __uint_as_float((b & 0x007fffffu) | 0x3f800000u);
    if (m > 1.41421354f) { m = __fmul_rn(m, 0.5f); e += 1; }
    float f = __fsub_rn(m, 1.0f);
    float s = __fdiv_rn(f, __fadd_rn(2.0f, f));
    float z = __fmul_rn(s, s);
    float p = __fmaf_rn(z, 0.0909090936f, 0.111111112f);
    p = __fmaf_rn(z, p, 0.142857149f);
    p = __fmaf_rn(z, p, 0.2f);
    p = __fmaf_rn(z, p, 0.333333343f);
    p = __fmul_rn(p, z);
    float t = __fadd_rn(s, s);
    float r = __fmaf_rn(t, p, t);
    return __fmaf_rn((float)e, 0.693147182f, r);
}
struct Lookup { int i; float f; };
__device__ __forceinline__ Lookup c_lookup(float lnE, float lnE0, float inv_dln, int N) {
    float x = __fmul_rn(__fsub_rn(lnE, lnE0), inv_dln);
    int i = (int)x;
    i = min(i, N - 2); i = max(i, 0);
    Lookup l; l.i = i; l.f = __fsub_rn(x, (float)i);
    return l;
}
__device__ __forceinline__ float c_lerp(const float2* t, Lookup l) { float2 a = t[l.i]; return __fmaf_rn(l.f, a.y, a.x); }
__device__ __forceinline__ float lerp(const float2* t, int i, float f) { float2 a = t[i]; return fmaf(f, a.y, a.x); }

// ---- queue push with warp aggregation over the currently active lanes ----------------------------
__device__ __forceinline__ void push_record(const Queue& q, uint32_t* overflow, const QRec& r) {
    unsigned m = __activemask();
    int lane = threadIdx.x & 31, leader = __ffs(m) - 1;
    uint32_t base = 0;
    if (lane == leader) base = atomicAdd(q.count, (uint32_t)__popc(m));
    base = __shfl_sync(m, base, leader);
    uint32_t idx = base + __popc(m & ((1u << lane) - 1u));
    if (idx >= q.cap) { atomicExch(overflow, 1u); return; }
    uint4* d = q.rec + 3ull * idx;
    d[0] = make_uint4(__float_as_uint(r.x), __float_as_uint(r.y), __float_as_uint(r.z), __float_as_uint(r.u));
    d[1] = make_uint4(__float_as_uint(r.v), __float_as_uint(r.w), __float_as_uint(r.E), r.hist);
    d[2] = make_uint4(r.trk_lo, r.trk_hi, (uint32_t)r.vox, r.tag);
}
// Push to one of two queues chosen per lane (first ? qa : qb): one pass over the record stores, two aggregated
// tail reservations (one per queue, each over the lanes that chose it).
__device__ __forceinline__ void push_record2(const Queue& qa, const Queue& qb, bool first, uint32_t* overflow, const QRec& r) {
    const unsigned m = __activemask();
    const unsigned ma = __ballot_sync(m, first), mb = m & ~ma;
    const int lane = threadIdx.x & 31;
    uint32_t base_a = 0, base_b = 0;
    if (ma && lane == __ffs(ma) - 1) base_a = atomicAdd(qa.count, (uint32_t)__popc(ma));
    if (mb && lane == __ffs(mb) - 1) base_b = atomicAdd(qb.count, (uint32_t)__popc(mb));
    if (ma) base_a = __shfl_sync(m, base_a, __ffs(ma) - 1);
    if (mb) base_b = __shfl_sync(m, base_b, __ffs(mb) - 1);
    const unsigned mine = first ? ma : mb;
    const uint32_t idx = (first ? base_a : base_b) + __popc(mine & ((1u << lane) - 1u));
    const Queue& q = first ? qa : qb;
    if (idx >= (first ? qa.cap : qb.cap)) { atomicExch(overflow, 1u); return; }
    uint4* d = (first ? qa.rec : qb.rec) + 3ull * idx;
    d[0] = make_uint4(__float_as_uint(r.x), __float_as_uint(r.y), __float_as_uint(r.z), __float_as_uint(r.u));
    d[1] = make_uint4(__float_as_uint(r.v), __float_as_uint(r.w), __float_as_uint(r.E), r.hist);
    d[2] = make_uint4(r.trk_lo, r.trk_hi, (uint32_t)r.vox, r.tag);
    (void)q;
}
__device__ __forceinline__ QRec load_record(const Queue& q, uint32_t idx) {
    const uint4* s = q.rec + 3ull * idx;
    uint4 a = s[0], b = s[1], c = s[2];
    QRec r;
    r.x = __uint_as_float(a.x); r.y = __uint_as_float(a.y); r.z = __uint_as_float(a.z); r.u = __uint_as_float(a.w);
    r.v = __uint_as_float(b.x); r.w = __uint_as_float(b.y); r.E = __uint_as_float(b.z); r.hist = b.w;
    r.trk_lo = c.x; r.trk_hi = c.y; r.vox = (int32_t)c.z; r.tag = c.w;
    return r;
}

// ---- direction rotation (R25) ------------------------------------------------------------------
// Rotate (u,v,w) by polar angle with cos = 1 - omu (omu passed to keep small angles exact) and azimuth phi.
__device__ __forceinline__ void rotate(float& u, float& v, float& w, float omu, float phi) {
    float mu = 1.0f - omu;
    float st = sqrtf(fmaxf(omu * (2.0f - omu), 0.0f));
    float sp, cp;
    __sincosf(phi, &sp, &cp);
    float s2 = fmaf(-w, w, 1.0f);
    float nu, nv, nw;
    if (s2 < 1e-6f) {
        nu = st * cp; nv = st * sp; nw = w >= 0.0f ? mu : -mu;
    } else {
        float is = rsqrtf(s2);
        nu = fmaf(u, mu, st * (u * w * cp - v * sp) * is);
        nv = fmaf(v, mu, st * (v * w * cp + u * sp) * is);
        nw = fmaf(w, mu, -st * s2 * is * cp);
    }
    float n = rsqrtf(fmaf(nu, nu, fmaf(nv, nv, nw * nw)));
    u = nu * n; v = nv * n; w = nw * n;
}

// Same rotation with single-instruction MUFU ops, no divergent branch, first-order renormalisation.
// sphi, cphi: sine and cosine of the azimuth.
__device__ __forceinline__ void rotate_fast(float& u, float& v, float& w, float omu, float sphi, float cphi) {
    float mu = 1.0f - omu;
    float st = f_sqrt(fmaxf(omu * (2.0f - omu), 0.0f));
    float s2 = fmaf(-w, w, 1.0f);
    bool pole = s2 < 1e-6f;
    float is = f_rsqrt(fmaxf(s2, 1e-12f));
    float a = st * cphi * is, b = st * sphi * is;
    float nu = fmaf(u, mu, fmaf(u * w, a, -v * b));
    float nv = fmaf(v, mu, fmaf(v * w, a, u * b));
    float nw = fmaf(w, mu, -s2 * a);
    nu = pole ? st * cphi : nu; nv = pole ? st * sphi : nv; nw = pole ? (w >= 0.0f ? mu : -mu) : nw;
    float n2 = fmaf(nu, nu, fmaf(nv, nv, nw * nw));
    float sc = fmaf(-0.5f, n2, 1.5f);  // 1/sqrt(n2) to first order around 1 (|n2 - 1| ~ 1e-6)
    u = nu * sc; v = nv * sc; w = nw * sc;
}

// ---- source (R13), arithmetic contract ----------------------------------------------------------
struct Primary { float x, y, z, u, v, w, E; bool inside; int ix, iy, iz; };
// kExact = true: the fp32 arithmetic contract (IEEE-rounded division and square root), used by the attenuation-only mode
// where the result must be bit-exact; kExact = false: the same formulas with single MUFU reciprocal / rsqrt for the
// transport kernels (the primary then differs from the contract's in the last bits only).
template <bool kExact = true>
__device__ __forceinline__ Primary sample_primary(const RunParams& P, uint4 w4) {
    const BeamDev& b = P.beam;
    Primary p;
    if (b.n_nodes == 1) p.E = b.E_nodes[0];
    else {
        float u0 = u01(w4.x), u1 = u01(w4.y);
        // j = number of interior nodes cdf[1 .. n-2] that are <= u0 (the cdf is non-decreasing): the bin the linear
        // scan "while (j + 2 < n && u0 >= cdf[j + 1]) ++j" stops in, found by bisection
        int j = 0, hi = b.n_nodes - 2;
        while (j < hi) {
            int mid = (j + hi + 1) >> 1;
            if (u0 >= b.cdf[mid]) j = mid; else hi = mid - 1;
        }
        float p0 = b.pdf_nodes[j], p1 = b.pdf_nodes[j + 1];
        float q = __fmaf_rn(u1, __fsub_rn(__fmul_rn(p1, p1), __fmul_rn(p0, p0)), __fmul_rn(p0, p0));
        float t;
        if (kExact) t = __fdiv_rn(__fmul_rn(u1, __fadd_rn(p0, p1)), __fadd_rn(p0, __fsqrt_rn(q)));
        else t = u1 * (p0 + p1) * f_rcp(p0 + f_sqrt(q));
        p.E = __fmaf_rn(t, __fsub_rn(b.E_nodes[j + 1], b.E_nodes[j]), b.E_nodes[j]);
    }
    if (b.shape == 0) {
        p.x = b.ex; p.y = b.ey; p.z = b.ez; p.u = b.ax; p.v = b.ay; p.w = b.az;
    } else {
        float fx = __fmul_rn(__fsub_rn(u01(w4.z), 0.5f), b.fx), fy = __fmul_rn(__fsub_rn(u01(w4.w), 0.5f), b.fy);
        p.x = __fadd_rn(b.ex, fx); p.y = __fadd_rn(b.ey, fy); p.z = b.ez;
        float n2 = __fmaf_rn(fx, fx, __fmaf_rn(fy, fy, __fmul_rn(b.ssd, b.ssd)));
        if (kExact) {
            float nr = __fsqrt_rn(n2);
            p.u = __fdiv_rn(fx, nr); p.v = __fdiv_rn(fy, nr); p.w = __fdiv_rn(b.ssd, nr);
        } else {
            float inr = f_rsqrt(n2);
            inr = inr * fmaf(-0.5f * n2, inr * inr, 1.5f);  // one Newton step: unit vector to ~1e-7
            p.u = fx * inr; p.v = fy * inr; p.w = b.ssd * inr;
        }
    }
    float gx = __fmul_rn(__fsub_rn(p.x, P.g.ox), P.g.ihx), gy = __fmul_rn(__fsub_rn(p.y, P.g.oy), P.g.ihy),
          gz = __fmul_rn(__fsub_rn(p.z, P.g.oz), P.g.ihz);
    p.inside = gx >= 0.0f && gx < (float)P.g.nx && gy >= 0.0f && gy < (float)P.g.ny && gz >= 0.0f && gz < (float)P.g.nz;
    p.ix = (int)gx; p.iy = (int)gy; p.iz = (int)gz;
    return p;
}

// batch of history h = floor(h * B / N) (R18) without a 64-bit division: inv_n = floor(2^64 / N) gives a quotient that
// is exact or one too small (h * B < 2^63), corrected by one multiply-compare.
__device__ __forceinline__ uint32_t batch_of(unsigned long long h, int n_batches, unsigned long long n_total,
                                             unsigned long long inv_n) {
    const unsigned long long x = h * (unsigned long long)n_batches;
    unsigned long long q = __umul64hi(x, inv_n);
    if (x - q * n_total >= n_total) ++q;
    return (uint32_t)q;
}

}  // namespace mcb
