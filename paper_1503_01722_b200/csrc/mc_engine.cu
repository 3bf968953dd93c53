// C ABI of the engine (include/mc.h): context, table upload, the launch scheduler and the calls.
// Host logic only; every step of the hot path runs in the kernels of mc_kernels.cuh.
#include "../../include/mc.h"
#include "mc_kernels.cuh"
#include "mc_tables.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

using namespace mcb;

struct mc_ctx {
    // phantom (host copies)
    Geometry g{};
    std::vector<uint8_t> h_mat;
    std::vector<float> h_rho;
    // tables (host)
    bool have_tables = false;
    Tables tabs;
    mc_params params{};
    float lnE0P = 0, inv_dlnP = 0;
    std::vector<float> p_maj, p_tot, p_C, p_pp;  // photon tables in use: [N], [n_mat][N] x 3
    // device state (allocated at the first compute call)
    bool dev_ready = false, tables_dirty = true;
    int sm_count = 0;
    cudaStream_t stream = nullptr;
    uint2* d_vox = nullptr;
    float2 *d_tabP = nullptr, *d_tabE = nullptr;
    size_t tabP_cap = 0, tabE_cap = 0;
    ListParticle* d_wave = nullptr;  // one wave of records filled by a user source function (mc_run_source)
    size_t wave_cap = 0;
    float* d_gs = nullptr;  // Goudsmit-Saunderson quantile table + per-material coarse ln A table (flags & MC_FLAG_MS_GS)
    size_t gs_cap = 0, gs_words = 0;
    int gs_n8 = 0;
    uint4* d_q[3] = {nullptr, nullptr, nullptr};  // electron A, electron B, photon
    uint32_t q_cap = 0;
    uint32_t* d_counters = nullptr;
    uint32_t* h_counters = nullptr;  // pinned
    unsigned long long* d_stats = nullptr;
    double* d_ledger = nullptr;
    float* d_edep = nullptr;
    size_t edep_cap = 0;
    float *d_dose = nullptr, *d_sigma = nullptr;
    float* d_beam = nullptr;  // E nodes, pdf nodes, cdf: 3 x kMaxNodes
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
    cudaEvent_t ev_src = nullptr;  // orders the context's stream after a source function's legacy-stream copies
    std::vector<cudaEvent_t> lev;  // event pairs around the transport launches of a run (read after the run's last sync)
    std::vector<char> lev_p;       // launch i was a photon kernel
    // options (M "manually adjusted")
    int64_t wave_size = 1 << 24, queue_factor = 4, blocks_per_sm = 0, refill_lanes = 32, aggregate = -1, hard_lanes = 32, adaptive = 1;
    int64_t electron_threads = 0;  // cap on the electron kernel's CTA size (0 = the largest that fits)
    int64_t plan_ahead = 1;  // enqueue launches ahead of the counters once the secondaries-per-primary ratios are known
    int64_t hinge_overrun_pct = 25, ms_carry = 1;  // readings R8 / R8b; the oracle has the same switches
    mc_stats stats{};
    // secondaries-per-primary ratios measured by the last run, reused when the next run has the same kind of beam
    double beam_key = -1.0, last_m_e = 16.0, last_m_p = 16.0;
    std::string err;
};

namespace {

constexpr int kMaxNodes = 4096;

mc_status fail(mc_ctx* c, mc_status s, const std::string& msg) {
    if (c) c->err = msg;
    return s;
}
#define CU(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess)                                                                     \
            return fail(ctx, e_ == cudaErrorMemoryAllocation ? MC_ERR_OOM : MC_ERR_CUDA,           \
                        std::string(#call) + ": " + cudaGetErrorString(e_));                       \
    } while (0)

int gs_coarse_nodes(int N) { return (N - 1 + 7) / 8 + 1; }  // ln A is kept on every 8th node of the energy grid
size_t e_stride(int N) { return ((size_t)kETabUnits * N + 1) & ~(size_t)1; }  // float2 per material, 16-byte multiple

std::vector<float2> pairs(const float* t, int N) {  // (value, slope to the next node); fp32 subtraction (R20)
    std::vector<float2> o(N);
    for (int i = 0; i < N; ++i) { o[i].x = t[i]; o[i].y = i + 1 < N ? t[i + 1] - t[i] : 0.0f; }
    return o;
}

mc_status ensure_device(mc_ctx* ctx) {
    if (ctx->dev_ready) return MC_OK;
    int n = 0;
    if (cudaGetDeviceCount(&n) != cudaSuccess || n <= 0) {
        cudaGetLastError();
        return fail(ctx, MC_ERR_CUDA, "no CUDA device: this library has no CPU path");
    }
    int dev = 0;
    CU(cudaGetDevice(&dev));
    cudaDeviceProp prop;
    CU(cudaGetDeviceProperties(&prop, dev));
    if (prop.major < 10) return fail(ctx, MC_ERR_CUDA, "built for sm_100a; this device is older");
    ctx->sm_count = prop.multiProcessorCount;
    size_t nvox = ctx->g.nvox;
    std::vector<uint2> pk(nvox);
    for (size_t i = 0; i < nvox; ++i) { memcpy(&pk[i].x, &ctx->h_rho[i], 4); pk[i].y = ctx->h_mat[i]; }
    CU(cudaMalloc(&ctx->d_vox, nvox * sizeof(uint2)));
    CU(cudaMemcpy(ctx->d_vox, pk.data(), nvox * sizeof(uint2), cudaMemcpyHostToDevice));
    CU(cudaMalloc(&ctx->d_counters, C_COUNT * sizeof(uint32_t)));
    CU(cudaMallocHost(&ctx->h_counters, C_COUNT * sizeof(uint32_t)));
    CU(cudaMalloc(&ctx->d_stats, S_COUNT * sizeof(unsigned long long)));
    CU(cudaMalloc(&ctx->d_ledger, LG_COUNT * sizeof(double)));
    CU(cudaMalloc(&ctx->d_dose, nvox * sizeof(float)));
    CU(cudaMalloc(&ctx->d_sigma, nvox * sizeof(float)));
    CU(cudaMalloc(&ctx->d_beam, 3 * kMaxNodes * sizeof(float)));
    for (auto& e : ctx->ev) CU(cudaEventCreate(&e));
    ctx->dev_ready = true;
    return MC_OK;
}

mc_status upload_tables(mc_ctx* ctx) {
    if (!ctx->tables_dirty) return MC_OK;
    const Tables& t = ctx->tabs;
    const int N = t.N, nm = t.n_mat;
    const size_t es = e_stride(N);
    std::vector<float2> P((size_t)(1 + nm * TP_COUNT) * N), E((size_t)nm * es, float2{0.0f, 0.0f});
    auto put = [&](std::vector<float2>& dst, size_t slot, const float* src) {
        std::vector<float2> pr = pairs(src, N);
        std::copy(pr.begin(), pr.end(), dst.begin() + slot * N);
    };
    put(P, 0, ctx->p_maj.data());
    for (int m = 0; m < nm; ++m) {
        put(P, 1 + m * TP_COUNT + TP_TOT, ctx->p_tot.data() + (size_t)m * N);
        put(P, 1 + m * TP_COUNT + TP_C, ctx->p_C.data() + (size_t)m * N);
        put(P, 1 + m * TP_COUNT + TP_PP, ctx->p_pp.data() + (size_t)m * N);
        // electron tables, node-interleaved (mc_device.cuh: kETabUnits)
        const std::vector<float2> R = pairs(t.t[T_RANGE][m].data(), N), Lc = pairs(t.t[T_L][m].data(), N), K1 = pairs(t.t[T_K1][m].data(), N),
                                  SH = pairs(t.t[T_S_HARD][m].data(), N), SM = pairs(t.t[T_S_MOLLER][m].data(), N), SX = pairs(t.t[T_S_MAX][m].data(), N);
        float2* e = E.data() + (size_t)m * es;
        for (int i = 0; i < N; ++i) {
            e[2 * i] = R[i]; e[2 * i + 1] = Lc[i];
            e[2 * N + 2 * i] = float2{R[i].x, R[i].y != 0.0f ? 1.0f / R[i].y : 0.0f}; e[2 * N + 2 * i + 1] = K1[i];
            e[4 * N + 2 * i] = SH[i]; e[4 * N + 2 * i + 1] = SM[i];
            e[6 * N + i] = SX[i];
        }
    }
    if (P.size() > ctx->tabP_cap) { cudaFree(ctx->d_tabP); ctx->d_tabP = nullptr; CU(cudaMalloc(&ctx->d_tabP, P.size() * sizeof(float2))); ctx->tabP_cap = P.size(); }
    if (E.size() > ctx->tabE_cap) { cudaFree(ctx->d_tabE); ctx->d_tabE = nullptr; CU(cudaMalloc(&ctx->d_tabE, E.size() * sizeof(float2))); ctx->tabE_cap = E.size(); }
    CU(cudaMemcpy(ctx->d_tabP, P.data(), P.size() * sizeof(float2), cudaMemcpyHostToDevice));
    CU(cudaMemcpy(ctx->d_tabE, E.data(), E.size() * sizeof(float2), cudaMemcpyHostToDevice));
    if (ctx->params.flags & MC_FLAG_MS_GS) {
        // quantile table as log2 x (one EX2 per sample), then per material ln A on every 8th energy node as (value, slope)
        const GsTable& G = gs_table();
        const int n8 = gs_coarse_nodes(N);
        std::vector<float> buf(G.y.size() + (size_t)nm * n8 * 2);
        for (size_t k = 0; k < G.y.size(); ++k) buf[k] = (float)((double)G.y[k] * 1.4426950408889634);
        for (int m = 0; m < nm; ++m)
            for (int k = 0; k < n8; ++k) {
                const std::vector<float>& la = t.t[T_LNA][m];
                const float v0 = la[std::min(8 * k, N - 1)], v1 = la[std::min(8 * k + 8, N - 1)];
                buf[G.y.size() + 2 * ((size_t)m * n8 + k)] = v0;
                buf[G.y.size() + 2 * ((size_t)m * n8 + k) + 1] = v1 - v0;
            }
        if (buf.size() > ctx->gs_cap) { cudaFree(ctx->d_gs); ctx->d_gs = nullptr; CU(cudaMalloc(&ctx->d_gs, buf.size() * sizeof(float))); ctx->gs_cap = buf.size(); }
        CU(cudaMemcpy(ctx->d_gs, buf.data(), buf.size() * sizeof(float), cudaMemcpyHostToDevice));
        ctx->gs_words = buf.size(); ctx->gs_n8 = n8;
    }
    ctx->tables_dirty = false;
    return MC_OK;
}

// The library's own memory pool for the particle queues, one per device, created on first use (thread-safe: function-local
// statics), never destroyed: freed queues stay in it for the next context.
cudaMemPool_t queue_pool() {
    static std::mutex mu;
    static std::vector<cudaMemPool_t> pools;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    std::lock_guard<std::mutex> lock(mu);
    if ((int)pools.size() <= dev) pools.resize(dev + 1, nullptr);
    if (!pools[dev]) {
        cudaMemPoolProps props{};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t p = nullptr;
        if (cudaMemPoolCreate(&p, &props) != cudaSuccess) { cudaGetLastError(); return nullptr; }
        unsigned long long keep = ~0ull;
        cudaMemPoolSetAttribute(p, cudaMemPoolAttrReleaseThreshold, &keep);
        pools[dev] = p;
    }
    return pools[dev];
}

// shared memory of a transport CTA of T threads: tables + per-thread counters + per-thread energy ledger + track pool
size_t smem_e(const mc_ctx* c, int T) {
    const size_t gs = (c->params.flags & MC_FLAG_MS_GS)
                          ? ((size_t)kGsNT * kGsNA * kGsNQ + 2 * (size_t)c->tabs.n_mat * gs_coarse_nodes(c->tabs.N)) * sizeof(float) : 0;
    return (size_t)c->tabs.n_mat * e_stride(c->tabs.N) * sizeof(float2) + (size_t)kGroups * kSlots * T * sizeof(uint4) +
           2 * (size_t)T * sizeof(uint32_t) + (size_t)(T / 32) * (2 * sizeof(double) + 8 * sizeof(uint32_t)) + gs;
}
size_t smem_p(const mc_ctx* c, int T) {
    const size_t ntab = (size_t)(1 + c->tabs.n_mat * TP_COUNT) * c->tabs.N;
    return ((ntab + 1) & ~(size_t)1) * sizeof(float2) + (size_t)kGroupsP * kSlotsP * T * sizeof(uint4) + (size_t)kSlotsP * T * sizeof(uint32_t) +
           2 * (size_t)T * sizeof(uint32_t) + (size_t)T * sizeof(double) + (size_t)(T / 32) * (sizeof(double) + 8 * sizeof(uint32_t));
}
constexpr size_t kSmemMax = 227 * 1024;  // opt-in dynamic shared memory per CTA on sm_100
using TransportKernel = void (*)(const RunParams);
struct KernelChoice { TransportKernel fn; int threads; size_t smem; };
// the largest CTA whose tables + pools fit (more materials or a finer grid leave less room for the pools)
bool choose_electron_kernel(const mc_ctx* c, KernelChoice& k) {
    constexpr int n = 4;
    const int T[n] = {1024, 768, 512, 256};
    const bool multi = c->params.flags & MC_FLAG_MULTI_VOXEL;
    const TransportKernel fn1[n] = {electron_kernel<1024, false>, electron_kernel<768, false>, electron_kernel<512, false>,
                                    electron_kernel<256, false>};
    const TransportKernel fnm[n] = {electron_kernel<1024, true>, electron_kernel<768, true>, electron_kernel<512, true>,
                                    electron_kernel<256, true>};
    const TransportKernel* fn = multi ? fnm : fn1;
    // the multi-voxel variant needs 80 registers: 768-thread CTAs at most; option "electron_threads" caps the CTA size
    const int cap = c->electron_threads > 0 ? (int)c->electron_threads : (multi ? 768 : 1024);
    for (int i = 0; i < n; ++i)
        if (T[i] <= cap && smem_e(c, T[i]) <= kSmemMax) { k = KernelChoice{fn[i], T[i], smem_e(c, T[i])}; return true; }
    return false;
}
bool choose_photon_kernel(const mc_ctx* c, KernelChoice& k) {
    const int T[3] = {1024, 768, 512};
    const TransportKernel fn[3] = {photon_kernel<1024>, photon_kernel<768>, photon_kernel<512>};
    for (int i = 0; i < 3; ++i)
        if (smem_p(c, T[i]) <= kSmemMax) { k = KernelChoice{fn[i], T[i], smem_p(c, T[i])}; return true; }
    return false;
}

// what the remembered secondaries-per-primary ratios belong to (mc_build_tables, mc_set_photon_tables and mc_set_option
// forget them: cut-offs, tables and scheduling options change the ratios)
// The key covers everything of the beam the ratios depend on: particle, shape, geometry of the field and the whole
// spectrum (FNV-1a over the bytes; 52 bits of it, held exactly in a double; negative values mean "no beam remembered").
double beam_key_of(const mc_ctx*, const mc_beam* b) {
    uint64_t h = 1469598103934665603ull;
    auto eat = [&](const void* p, size_t n) {
        const unsigned char* c = static_cast<const unsigned char*>(p);
        for (size_t i = 0; i < n; ++i) { h ^= c[i]; h *= 1099511628211ull; }
    };
    eat(&b->particle, sizeof b->particle); eat(&b->shape, sizeof b->shape);
    eat(b->entry_cm, sizeof b->entry_cm); eat(b->axis, sizeof b->axis);
    eat(&b->ssd_cm, sizeof b->ssd_cm); eat(b->field_cm, sizeof b->field_cm);
    eat(&b->n_nodes, sizeof b->n_nodes);
    eat(b->E_nodes_MeV, sizeof(float) * (size_t)b->n_nodes);
    if (b->n_nodes > 1) eat(b->pdf_nodes, sizeof(float) * (size_t)b->n_nodes);
    return (double)(h >> 12);
}

mc_status check_beam(mc_ctx* ctx, const mc_beam* b) {
    if (!b) return fail(ctx, MC_ERR_INVALID_ARG, "beam is null");
    if (b->particle < -1 || b->particle > 1) return fail(ctx, MC_ERR_INVALID_ARG, "beam.particle must be -1, 0 or 1");
    if (b->shape != MC_SHAPE_PENCIL && b->shape != MC_SHAPE_POINT_RECT) return fail(ctx, MC_ERR_INVALID_ARG, "beam.shape");
    if (b->n_nodes < 1 || b->n_nodes > kMaxNodes || !b->E_nodes_MeV) return fail(ctx, MC_ERR_INVALID_ARG, "beam.n_nodes / E_nodes_MeV");
    if (b->n_nodes > 1 && !b->pdf_nodes) return fail(ctx, MC_ERR_INVALID_ARG, "beam.pdf_nodes is null");
    float an = std::sqrt(b->axis[0] * b->axis[0] + b->axis[1] * b->axis[1] + b->axis[2] * b->axis[2]);
    if (!(std::fabs(an - 1.0f) < 1e-4f)) return fail(ctx, MC_ERR_INVALID_ARG, "beam.axis must be a unit vector");
    if (b->shape == MC_SHAPE_POINT_RECT) {
        if (!(b->ssd_cm > 0) || !(b->field_cm[0] >= 0) || !(b->field_cm[1] >= 0)) return fail(ctx, MC_ERR_INVALID_ARG, "beam.ssd_cm / field_cm");
        if (!(b->axis[2] > 0.9999f)) return fail(ctx, MC_ERR_INVALID_ARG, "POINT_RECT beams must point along +z");
    }
    double tot = 0;
    for (int i = 0; i < b->n_nodes; ++i) {
        if (!(b->E_nodes_MeV[i] > 0)) return fail(ctx, MC_ERR_INVALID_ARG, "beam energies must be positive");
        if (b->E_nodes_MeV[i] > ctx->params.e_max_MeV) return fail(ctx, MC_ERR_ENERGY_RANGE, "beam energy above e_max_MeV");
        if (i && !(b->E_nodes_MeV[i] > b->E_nodes_MeV[i - 1])) return fail(ctx, MC_ERR_INVALID_ARG, "beam energy nodes must ascend");
        if (b->n_nodes > 1) {
            if (!(b->pdf_nodes[i] >= 0)) return fail(ctx, MC_ERR_INVALID_ARG, "beam pdf must be non-negative");
            if (i) tot += 0.5 * ((double)b->pdf_nodes[i] + b->pdf_nodes[i - 1]) * ((double)b->E_nodes_MeV[i] - b->E_nodes_MeV[i - 1]);
        }
    }
    if (b->n_nodes > 1 && !(tot > 0)) return fail(ctx, MC_ERR_INVALID_ARG, "beam pdf integrates to zero");
    return MC_OK;
}

mc_status upload_beam(mc_ctx* ctx, const mc_beam* b, BeamDev& out) {
    const int n = b->n_nodes;
    std::vector<float> buf(3 * (size_t)kMaxNodes, 0.0f);
    std::vector<double> cd(n, 0.0);
    double tot = 0;
    for (int j = 0; j < n; ++j) {
        buf[j] = b->E_nodes_MeV[j];
        buf[kMaxNodes + j] = n > 1 ? b->pdf_nodes[j] : 1.0f;
        if (j + 1 < n) { tot += 0.5 * ((double)b->pdf_nodes[j] + (double)b->pdf_nodes[j + 1]) * ((double)b->E_nodes_MeV[j + 1] - (double)b->E_nodes_MeV[j]); cd[j + 1] = tot; }
    }
    for (int j = 0; j < n; ++j) buf[2 * kMaxNodes + j] = tot > 0 ? (float)(cd[j] / tot) : 0.0f;
    CU(cudaMemcpyAsync(ctx->d_beam, buf.data(), buf.size() * sizeof(float), cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));  // buf is pageable and local
    out.particle = b->particle; out.shape = b->shape; out.n_nodes = n;
    out.ex = b->entry_cm[0]; out.ey = b->entry_cm[1]; out.ez = b->entry_cm[2];
    out.ax = b->axis[0]; out.ay = b->axis[1]; out.az = b->axis[2];
    out.ssd = b->ssd_cm; out.fx = b->field_cm[0]; out.fy = b->field_cm[1];
    out.E_nodes = ctx->d_beam; out.pdf_nodes = ctx->d_beam + kMaxNodes; out.cdf = ctx->d_beam + 2 * kMaxNodes;
    return MC_OK;
}

void fill_params(const mc_ctx* ctx, RunParams& P) {
    const Tables& t = ctx->tabs;
    P.g = ctx->g;
    P.vox = ctx->d_vox; P.tabP = ctx->d_tabP; P.tabE = ctx->d_tabE;
    P.N = t.N; P.n_mat = t.n_mat; P.k_cut = t.k_cut; P.e_stride = (int)e_stride(t.N);
    P.lnE0 = (float)t.lnE0; P.dln = (float)t.dln; P.inv_dln = (float)(1.0 / t.dln);
    P.lnE0P = ctx->lnE0P; P.inv_dlnP = ctx->inv_dlnP;
    P.e_cut = ctx->params.e_cut_MeV; P.g_cut = ctx->params.g_cut_MeV;
    P.d_maxs = ctx->params.d_maxs_cm; P.f_maxe = ctx->params.f_maxe;
    for (int m = 0; m < MAX_MAT; ++m) P.lscr[m] = m < t.n_mat ? t.lscr[m] : 0.0f;
    P.flags = ctx->params.flags;
    P.counters = ctx->d_counters; P.stats = ctx->d_stats; P.ledger = ctx->d_ledger;
    P.refill_lanes = (int)ctx->refill_lanes; P.aggregate = (int)ctx->aggregate; P.hard_lanes = (int)ctx->hard_lanes;
    const double ln2 = 0.69314718055994530942, log2e = 1.44269504088896340736;
    P.ex_a = (float)(ln2 / t.dln); P.ex_b = (float)(t.lnE0 / t.dln);
    P.t_a = (float)(t.dln * log2e); P.t_b = (float)(t.lnE0 * log2e);
    P.hinge_overrun = 0.01f * (float)ctx->hinge_overrun_pct; P.ms_carry = (int)ctx->ms_carry;
    if (ctx->params.flags & MC_FLAG_MS_GS) {
        const GsTable& G = gs_table();
        P.gs = ctx->d_gs; P.gs_words = (int)ctx->gs_words; P.gs_n8 = ctx->gs_n8;
        for (int i = 0; i < kGsNT; ++i) P.gs_an[i] = G.an[i];
        const double c0 = gs_grid_coordinate(kGsTMin), c1 = gs_grid_coordinate(kGsTMax);
        P.gs_c0 = (float)c0; P.gs_inv_dc = (float)((kGsNT - 1) / (c1 - c0));
        P.gs_lnA0 = (float)std::log(kGsAMin); P.gs_inv_dA = (float)((kGsNA - 1) / std::log(kGsAMax / kGsAMin));
    }
}

}  // namespace

namespace {

// Launch scheduler (workflow Table 1): same-type launches; the queue holding at least one
// full wave goes first, otherwise the group with the most particles (source included).
// Source: a beam (primaries sampled inside the transport kernels) or, with beam == nullptr, a device-resident
// particle list whose entry h is history h (loaded into the queues a wave at a time).
// A user source function (mc_run_source) stands in for the list: it fills one wave of records at a time.
struct SourceFn { mc_source_fn fn = nullptr; void* user = nullptr; };

mc_status transport(mc_ctx* ctx, const mc_beam* beam, const ListParticle* d_list, uint64_t n_total, uint64_t h0, uint64_t h1,
                    uint64_t seed, int n_batches, float* d_edep, SourceFn src = SourceFn()) {
    mc_status st;
    if ((st = ensure_device(ctx)) != MC_OK) return st;
    if ((st = upload_tables(ctx)) != MC_OK) return st;
    const size_t nvox = ctx->g.nvox;
    KernelChoice ke, kp;
    if (!choose_electron_kernel(ctx, ke) || !choose_photon_kernel(ctx, kp))
        return fail(ctx, MC_ERR_INVALID_ARG, "tables do not fit in shared memory: lower n_grid (n_mats * n_grid is too large)");
    const size_t se = ke.smem, sp = kp.smem;
    CU(cudaFuncSetAttribute(ke.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)se));
    CU(cudaFuncSetAttribute(kp.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sp));
    int occ_e = 0, occ_p = 0;
    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_e, ke.fn, ke.threads, se));
    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_p, kp.fn, kp.threads, sp));
    if (occ_e < 1 || occ_p < 1) return fail(ctx, MC_ERR_CUDA, "kernel does not fit on an SM");
    if (ctx->blocks_per_sm > 0) { occ_e = std::min<int>(occ_e, (int)ctx->blocks_per_sm); occ_p = std::min<int>(occ_p, (int)ctx->blocks_per_sm); }

    // queues
    const uint64_t n_run = h1 - h0;
    const uint32_t W = (uint32_t)std::min<uint64_t>((uint64_t)ctx->wave_size, std::max<uint64_t>(n_run, 1024));
    const uint32_t cap = (uint32_t)std::min<uint64_t>((uint64_t)W * (uint64_t)ctx->queue_factor, 0x7fffffffull / 3);
    if (cap > ctx->q_cap) {
        // The queues are gigabytes: they come from a stream-ordered memory pool of the library's own (the device's default
        // pool and its policy are left alone) that keeps freed memory, so that a later context of the same process
        // reuses them instead of paying cudaMalloc / cudaFree of several GB again (measured: 30 - 300 ms per context).
        cudaMemPool_t pool = queue_pool();
        for (auto& q : ctx->d_q) { if (q) cudaFreeAsync(q, ctx->stream); q = nullptr; }
        ctx->q_cap = 0;
        for (auto& q : ctx->d_q) {
            if (pool) CU(cudaMallocFromPoolAsync(&q, (size_t)cap * 3 * sizeof(uint4), pool, ctx->stream));
            else CU(cudaMallocAsync(&q, (size_t)cap * 3 * sizeof(uint4), ctx->stream));
        }
        ctx->q_cap = cap;
    }
    cudaStream_t s = ctx->stream;
    CU(cudaMemsetAsync(d_edep, 0, (size_t)n_batches * nvox * sizeof(float), s));
    CU(cudaMemsetAsync(ctx->d_counters, 0, C_COUNT * sizeof(uint32_t), s));
    CU(cudaMemsetAsync(ctx->d_stats, 0, S_COUNT * sizeof(unsigned long long), s));
    CU(cudaMemsetAsync(ctx->d_ledger, 0, LG_COUNT * sizeof(double), s));

    RunParams P;
    memset(&P, 0, sizeof P);
    fill_params(ctx, P);
    if (beam && (st = upload_beam(ctx, beam, P.beam)) != MC_OK) return st;
    if (ctx->aggregate < 0) {
        // auto: warp-aggregated scoring pays when many lanes of a warp score into the same cell at once, i.e. for beams
        // that enter through a handful of voxel columns (measured: pencil beam 1.7x faster with it, 10x10 and 2x2 cm^2
        // fields 6 % slower, profiles/README.md)
        const double cols = beam && beam->shape == MC_SHAPE_POINT_RECT
                                ? (double)(beam->field_cm[0] / ctx->g.hx) * (double)(beam->field_cm[1] / ctx->g.hy) : (beam ? 1.0 : 1e9);
        P.aggregate = cols < 16.0 ? 1 : 0;
    }
    P.edep = d_edep; P.n_total = n_total; P.n_batches = n_batches;
    P.inv_n_total = n_total > 1 ? (unsigned long long)((((unsigned __int128)1) << 64) / n_total) : ~0ull;
    P.seed_lo = (uint32_t)seed; P.seed_hi = (uint32_t)(seed >> 32);
    for (int r = 0; r < 10; ++r) P.seed_rk[r] = P.seed_lo + (uint32_t)r * 0xBB67AE85u;

    const bool photon_beam = beam && beam->particle == MC_PHOTON;
    uint64_t remaining = n_run, h_next = h0;
    uint32_t cnt_e[2] = {0, 0}, cnt_p = 0;
    int cur = 0;
    mc_stats& S = ctx->stats;
    S = mc_stats{};
    double ms_e = 0, ms_p = 0;
    // secondaries queued per new primary (electron queue, photon queue): measured while running; the first launch of a
    // context is a probe (16 assumed), later runs with the same kind of beam start from the last measurement
    const double key = beam ? beam_key_of(ctx, beam) : -2.0;
    bool have_ratio = key == ctx->beam_key;
    double m_new_e = have_ratio ? ctx->last_m_e : 16.0, m_new_p = have_ratio ? ctx->last_m_p : 16.0;
    // Every transport launch: the kernel reads the size of its input queue on the device, and its last CTA empties that
    // queue and the work counter, so a launch needs nothing from the host but the number of new primaries.
    unsigned long long list_h0 = 0;  // history of d_list[0]
    size_t n_timed = 0;  // event pairs ctx->lev[2i], [2i+1] bracket the launches of this run; lev_p[i] = photon kernel
    auto issue = [&](bool run_p, uint32_t n_new, uint64_t items_hint) -> mc_status {
        P.n_new = n_new; P.h_first = h_next;
        Queue qe_cur{ctx->d_q[cur], ctx->d_counters + C_E_A + cur, ctx->q_cap};
        Queue qe_oth{ctx->d_q[1 - cur], ctx->d_counters + C_E_A + (1 - cur), ctx->q_cap};
        Queue qp{ctx->d_q[2], ctx->d_counters + C_P, ctx->q_cap};
        const int occ = run_p ? occ_p : occ_e, thr = run_p ? kp.threads : ke.threads;
        int grid = (int)std::min<uint64_t>((uint64_t)ctx->sm_count * occ, (items_hint + thr - 1) / thr);
        grid = std::max(grid, 1);
        if (ctx->lev.size() < 2 * (n_timed + 1)) {
            cudaEvent_t a, b;
            CU(cudaEventCreate(&a)); ctx->lev.push_back(a);
            CU(cudaEventCreate(&b)); ctx->lev.push_back(b);
        }
        if (ctx->lev_p.size() < n_timed + 1) ctx->lev_p.resize(n_timed + 1);
        ctx->lev_p[n_timed] = run_p;
        CU(cudaEventRecord(ctx->lev[2 * n_timed], s));
        if (run_p) {
            P.q_in = qp; P.q_e_out = qe_cur; P.q_p_out = qp;
            kp.fn<<<grid, kp.threads, sp, s>>>(P);
        } else {
            P.q_in = qe_cur; P.q_e_out = qe_oth; P.q_p_out = qp;
            ke.fn<<<grid, ke.threads, se, s>>>(P);
            cur = 1 - cur;  // what this launch produced is the next electron launch's input
        }
        CU(cudaGetLastError());
        CU(cudaEventRecord(ctx->lev[2 * n_timed + 1], s));
        ++n_timed;
        ++S.n_kernel_launches;
        remaining -= n_new; h_next += n_new;
        return MC_OK;
    };
    auto read_counters = [&]() -> mc_status {  // the one host <-> device crossing: 24 bytes and a stream synchronisation
        CU(cudaMemcpyAsync(ctx->h_counters, ctx->d_counters, C_COUNT * sizeof(uint32_t), cudaMemcpyDeviceToHost, s));
        CU(cudaStreamSynchronize(s));
        ++S.n_host_syncs;
        if (ctx->h_counters[C_OVERFLOW]) {
            ctx->beam_key = -1.0;  // the remembered ratios admitted too much: probe again next time
            return fail(ctx, MC_ERR_QUEUE_OVERFLOW, "particle queue overflow: lower option wave_size or raise queue_factor");
        }
        if (ctx->h_counters[C_FLAGS] & 1u) return fail(ctx, MC_ERR_ENERGY_RANGE, "source function: particle energy not in (0, e_max_MeV]");
        if (ctx->h_counters[C_FLAGS] & 6u) return fail(ctx, MC_ERR_INVALID_ARG, "source function: directions must be unit vectors and particle types -1, 0 or 1");
        cnt_e[0] = ctx->h_counters[C_E_A]; cnt_e[1] = ctx->h_counters[C_E_B]; cnt_p = ctx->h_counters[C_P];
        return MC_OK;
    };
    // new primaries a launch of the source's type may admit: up to a wave, and no more than the output queues can take
    // at the secondaries-per-primary ratios (R21: a queue must not overflow by admission; overflow is still detected)
    auto admit = [&](bool run_p, double in_e, double in_p) -> uint32_t {
        const double n_in = run_p ? in_p : in_e;
        if (n_in >= W) return 0u;
        const double room_e = (double)ctx->q_cap - (run_p ? in_e : 0.0) - n_in;
        const double room_p = run_p ? 1e30 : (double)ctx->q_cap - in_p - n_in;
        const double fit = ctx->adaptive ? std::max(0.0, std::min(room_e / m_new_e, room_p / m_new_p)) : 1e30;
        uint32_t n_new = (uint32_t)std::min<double>((double)std::min<uint64_t>(remaining, (uint64_t)(W - n_in)), fit);
        if (n_new == 0 && n_in == 0) n_new = (uint32_t)std::min<uint64_t>(remaining, 1024);  // always progress
        return n_new;
    };
    CU(cudaEventRecord(ctx->ev[0], s));
    const bool plan_ahead = beam && ctx->plan_ahead && ctx->adaptive;
    // ---- launches decided one at a time from the counters (Table 1): particle lists, the probe launches of
    // a beam whose secondaries-per-primary ratios are not known yet, and everything when option plan_ahead is 0 --------
    while ((remaining > 0 || cnt_e[cur] > 0 || cnt_p > 0) && !(plan_ahead && have_ratio)) {
        if ((d_list || src.fn) && remaining > 0 && cnt_e[cur] < W && cnt_p < W) {
            // particle-list source: the next wave of listed particles goes straight into the input queues
            const uint32_t n_load = (uint32_t)std::min<uint64_t>(remaining, W);
            if (src.fn) {
                // user source function ("write a CPU/GPU function"): it fills this wave's records — by a kernel of
                // its own on the stream it is given, or by a copy — and the wave is validated like a device-resident list
                if (ctx->wave_cap < n_load) {
                    cudaFree(ctx->d_wave); ctx->d_wave = nullptr; ctx->wave_cap = 0;
                    CU(cudaMalloc(&ctx->d_wave, (size_t)W * sizeof(ListParticle)));
                    ctx->wave_cap = W;
                }
                if (src.fn(src.user, h_next, n_load, reinterpret_cast<mc_particle*>(ctx->d_wave), (void*)s) != 0)
                    return fail(ctx, MC_ERR_INVALID_ARG, "the source function reported a failure");
                if (s != nullptr && s != cudaStreamLegacy) {
                    // A function that filled the wave with a plain cudaMemcpy used the legacy default stream; a copy from
                    // pageable memory may return before its DMA has landed, and a non-blocking context stream is not
                    // ordered after the legacy stream by itself: make it wait for whatever the function left there.
                    if (!ctx->ev_src) CU(cudaEventCreateWithFlags(&ctx->ev_src, cudaEventDisableTiming));
                    CU(cudaEventRecord(ctx->ev_src, cudaStreamLegacy));
                    CU(cudaStreamWaitEvent(s, ctx->ev_src, 0));
                }
                check_particles_kernel<<<std::min<uint32_t>((n_load + kThreads - 1) / kThreads, (uint32_t)ctx->sm_count * 8), kThreads, 0, s>>>(
                    ctx->d_wave, n_load, ctx->params.e_max_MeV, ctx->d_counters + C_FLAGS);
                CU(cudaGetLastError());
                d_list = ctx->d_wave; list_h0 = h_next;  // record h of the job = entry h - h_next of the wave
            }
            P.h_first = h_next; P.n_new = 0;
            P.q_e_out = Queue{ctx->d_q[cur], ctx->d_counters + C_E_A + cur, ctx->q_cap};
            P.q_p_out = Queue{ctx->d_q[2], ctx->d_counters + C_P, ctx->q_cap};
            load_particles_kernel<<<std::min<uint32_t>((n_load + kThreads - 1) / kThreads, (uint32_t)ctx->sm_count * 8), kThreads, 0, s>>>(P, d_list, list_h0, n_load);
            CU(cudaGetLastError());
            ++S.n_kernel_launches;
            if ((st = read_counters()) != MC_OK) return st;
            remaining -= n_load; h_next += n_load;
            continue;
        }
        bool run_p;
        if (cnt_p >= W) run_p = true;
        else if (cnt_e[cur] >= W) run_p = false;
        else {
            const uint64_t src = beam ? remaining : 0;  // a particle list feeds the queues, not the kernels
            uint64_t avail_e = cnt_e[cur] + (photon_beam ? 0 : src), avail_p = cnt_p + (photon_beam ? src : 0);
            run_p = avail_p > avail_e;
        }
        const uint32_t n_in = run_p ? cnt_p : cnt_e[cur];
        const uint32_t n_new = beam && run_p == photon_beam ? admit(run_p, cnt_e[cur], cnt_p) : 0u;
        const uint32_t before_e = cnt_e[cur], before_p = cnt_p;
        const int cur0 = cur;
        if ((st = issue(run_p, n_new, (uint64_t)n_in + n_new)) != MC_OK) return st;
        if ((st = read_counters()) != MC_OK) return st;
        if (n_new >= n_in && n_new >= 1024) {  // a launch dominated by primaries: update the measured ratios
            const double out_e = run_p ? (double)cnt_e[cur0] - before_e : (double)cnt_e[1 - cur0];
            const double out_p = run_p ? 0.0 : (double)cnt_p - before_p;
            const double n_items = (double)n_in + n_new;
            m_new_e = std::max(0.05, 1.5 * out_e / n_items);
            m_new_p = std::max(0.05, 1.5 * out_p / n_items);
            ctx->beam_key = key; ctx->last_m_e = m_new_e; ctx->last_m_p = m_new_p;
            have_ratio = true;
        }
    }
    // ---- launches enqueued ahead (ratios known): the host does not wait between launches.  Per wave: the source's kernel
    // (it also consumes whatever its queue holds), then the other type where its queue fills fastest; after the last wave
    // the cascade is drained by rounds of [photon, electron, electron] launches — a launch whose queue turns out to be
    // empty returns at once — with one read-back per round to see whether anything is left. ---------------------------
    if (remaining > 0 || cnt_e[cur] > 0 || cnt_p > 0) {
        const uint64_t full = ~0ull >> 1;  // size unknown on the host: full grid
        double est_e = cnt_e[cur], est_p = cnt_p;  // upper estimates of what the queues hold
        int wave = 0;
        while (remaining > 0) {
            const uint32_t n_new = admit(photon_beam, est_e, est_p);
            if (n_new == 0) {  // the estimates say the queues are too full: drain one generation and look
                if ((st = issue(!photon_beam, 0, full)) != MC_OK) return st;
                if ((st = issue(photon_beam, 0, full)) != MC_OK) return st;
                if ((st = read_counters()) != MC_OK) return st;
                est_e = cnt_e[cur]; est_p = cnt_p;
                continue;
            }
            if ((st = issue(photon_beam, n_new, full)) != MC_OK) return st;
            if (photon_beam) {
                // a photon wave fills the electron queue: run it now; its own output (delta rays, bremsstrahlung) rides
                // along with the next wave
                est_e += m_new_e * n_new;
                if ((st = issue(false, 0, full)) != MC_OK) return st;
                est_e = 0.15 * est_e; est_p = 0.15 * m_new_e * n_new;
            } else {
                // an electron wave: delta rays go to the next electron launch, photons wait for every second wave
                est_e = m_new_e * n_new; est_p += m_new_p * n_new;
                if ((++wave & 1) == 0 || est_p > 0.5 * ctx->q_cap) {
                    if ((st = issue(true, 0, full)) != MC_OK) return st;
                    est_e += 0.5 * est_p; est_p = 0.0;
                }
            }
        }
        do {
            for (int k = 0; k < 2; ++k) {  // two rounds per read-back: an empty launch costs ~5 us, a read-back ~15 us
                if ((st = issue(true, 0, full)) != MC_OK) return st;
                if ((st = issue(false, 0, full)) != MC_OK) return st;
                if ((st = issue(false, 0, full)) != MC_OK) return st;
            }
            if ((st = read_counters()) != MC_OK) return st;
        } while (cnt_e[0] > 0 || cnt_e[1] > 0 || cnt_p > 0);
    }
    CU(cudaEventRecord(ctx->ev[1], s));
    // ledger: deposited energy is the total of the batch grids
    sum_kernel<<<ctx->sm_count * 4, kThreads, 0, s>>>(d_edep, (size_t)n_batches * nvox, ctx->d_ledger + LG_DEP);
    CU(cudaGetLastError());
    ++S.n_kernel_launches;
    unsigned long long hs[S_COUNT];
    double hl[LG_COUNT];
    CU(cudaMemcpyAsync(hs, ctx->d_stats, sizeof hs, cudaMemcpyDeviceToHost, s));
    CU(cudaMemcpyAsync(hl, ctx->d_ledger, sizeof hl, cudaMemcpyDeviceToHost, s));
    CU(cudaStreamSynchronize(s));
    float ms = 0;
    CU(cudaEventElapsedTime(&ms, ctx->ev[0], ctx->ev[1]));
    for (size_t i = 0; i < n_timed; ++i) {
        float t = 0;
        CU(cudaEventElapsedTime(&t, ctx->lev[2 * i], ctx->lev[2 * i + 1]));
        (ctx->lev_p[i] ? ms_p : ms_e) += t;
    }
    S.n_histories = hs[S_HIST]; S.n_electron_steps = hs[S_ESTEP]; S.n_photon_flights = hs[S_FLIGHT];
    S.n_fictitious = hs[S_FICT]; S.n_compton = hs[S_COMPTON]; S.n_pair = hs[S_PAIR]; S.n_photoelectric = hs[S_PE];
    S.n_moller = hs[S_MOLLER]; S.n_brems = hs[S_BREMS]; S.n_secondary_electrons = hs[S_SEC_E];
    S.n_secondary_photons = hs[S_SEC_G]; S.n_dose_atomics = hs[S_ATOMICS];
    S.e_source_MeV = hl[LG_SRC]; S.e_escaped_MeV = hl[LG_ESC]; S.e_deposited_MeV = hl[LG_DEP];
    S.transport_ms = ms; S.electron_kernel_ms = ms_e; S.photon_kernel_ms = ms_p;
    return MC_OK;
}

// A beam run whose launches were enqueued ahead from REMEMBERED ratios (an earlier run with the same beam) can find
// that they admitted too much; the overflow is detected, nothing is returned, and the run is repeated once with the
// ratios forgotten, i.e. starting with counter-driven probe launches.  An overflow of that second attempt, or of a run
// that was counter-driven to begin with, is the caller's (queue_factor / wave_size too small) and is reported.
mc_status transport_beam(mc_ctx* ctx, const mc_beam* beam, uint64_t n_total, uint64_t h0, uint64_t h1, uint64_t seed, int n_batches,
                         float* d_edep) {
    const bool from_memory = ctx->plan_ahead && ctx->adaptive && ctx->beam_key == beam_key_of(ctx, beam);
    mc_status st = transport(ctx, beam, nullptr, n_total, h0, h1, seed, n_batches, d_edep);
    if (st == MC_ERR_QUEUE_OVERFLOW && from_memory) {
        cudaStreamSynchronize(ctx->stream);
        st = transport(ctx, beam, nullptr, n_total, h0, h1, seed, n_batches, d_edep);  // beam_key was reset: probes first
    }
    return st;
}

mc_status check_run_args(mc_ctx* ctx, const mc_beam* beam, uint64_t n_histories, uint64_t h0, uint64_t h1, int32_t n_batches) {
    if (!ctx) return MC_ERR_INVALID_ARG;
    if (!ctx->have_tables) return fail(ctx, MC_ERR_STATE, "mc_build_tables has not been called");
    mc_status st = check_beam(ctx, beam);
    if (st != MC_OK) return st;
    if (n_histories == 0 || n_histories >= (1ull << 32)) return fail(ctx, MC_ERR_INVALID_ARG, "n_histories must be in [1, 2^32)");
    if (n_batches < 2 || (uint64_t)n_batches > n_histories) return fail(ctx, MC_ERR_INVALID_ARG, "n_batches must be in [2, n_histories]");
    if (h0 > h1 || h1 > n_histories) return fail(ctx, MC_ERR_INVALID_ARG, "history range");
    if ((uint64_t)n_batches * (uint64_t)ctx->g.nvox >= (1ull << 32)) return fail(ctx, MC_ERR_INVALID_ARG, "n_batches * nvox must be < 2^32");
    return MC_OK;
}

mc_status ensure_edep(mc_ctx* ctx, size_t n) {
    if (n <= ctx->edep_cap) return MC_OK;
    cudaFree(ctx->d_edep); ctx->d_edep = nullptr; ctx->edep_cap = 0;
    CU(cudaMalloc(&ctx->d_edep, n * sizeof(float)));
    ctx->edep_cap = n;
    return MC_OK;
}

mc_status finalize_device(mc_ctx* ctx, const float* d_edep, uint64_t n_histories, int n_batches) {
    const int nvox = ctx->g.nvox;
    const double vol = (double)ctx->g.hx * (double)ctx->g.hy * (double)ctx->g.hz;
    int grid = std::min(ctx->sm_count * 8, (nvox + kThreads - 1) / kThreads);
    finalize_kernel<<<grid, kThreads, n_batches * sizeof(double), ctx->stream>>>(d_edep, ctx->d_vox, nvox, n_batches, n_histories, vol,
                                                                                  ctx->d_dose, ctx->d_sigma);
    CU(cudaGetLastError());
    ++ctx->stats.n_kernel_launches;
    return MC_OK;
}

}  // namespace

// =================================================================================================
// C ABI
// =================================================================================================
extern "C" {

mc_status mc_create(const uint8_t* material_idx, const float* density_gcc, const int32_t dims[3], const float voxel_cm[3],
                    const float origin_cm[3], mc_ctx** out) {
    if (!out) return MC_ERR_INVALID_ARG;
    *out = nullptr;
    if (!material_idx || !density_gcc || !dims || !voxel_cm || !origin_cm) return MC_ERR_INVALID_ARG;
    for (int a = 0; a < 3; ++a)
        if (dims[a] <= 0 || dims[a] > 1024 || !(voxel_cm[a] > 0.0f) || !std::isfinite(voxel_cm[a]) || !std::isfinite(origin_cm[a])) return MC_ERR_INVALID_ARG;
    const uint64_t nvox = (uint64_t)dims[0] * (uint64_t)dims[1] * (uint64_t)dims[2];
    if (nvox >= (1ull << 31)) return MC_ERR_INVALID_ARG;
    for (uint64_t i = 0; i < nvox; ++i)
        if (!(density_gcc[i] > 0.0f) || !std::isfinite(density_gcc[i])) return MC_ERR_INVALID_ARG;
    mc_ctx* ctx = new (std::nothrow) mc_ctx();
    if (!ctx) return MC_ERR_OOM;
    Geometry& g = ctx->g;
    g.nx = dims[0]; g.ny = dims[1]; g.nz = dims[2]; g.nvox = (int)nvox;
    g.hx = voxel_cm[0]; g.hy = voxel_cm[1]; g.hz = voxel_cm[2];
    g.ox = origin_cm[0]; g.oy = origin_cm[1]; g.oz = origin_cm[2];
    g.ihx = 1.0f / g.hx; g.ihy = 1.0f / g.hy; g.ihz = 1.0f / g.hz;
    try {
        ctx->h_mat.assign(material_idx, material_idx + nvox);
        ctx->h_rho.assign(density_gcc, density_gcc + nvox);
    } catch (...) { delete ctx; return MC_ERR_OOM; }
    *out = ctx;
    return MC_OK;
}

void mc_destroy(mc_ctx* ctx) {
    if (!ctx) return;
    if (ctx->dev_ready) {
        // every call synchronises the context's stream before it returns, except on some error paths: wait here so that
        // nothing the context enqueued still uses the buffers (the stream may be gone already: then there is nothing to wait for)
        if (cudaStreamSynchronize(ctx->stream) != cudaSuccess) cudaGetLastError();
        cudaFree(ctx->d_vox); cudaFree(ctx->d_tabP); cudaFree(ctx->d_tabE); cudaFree(ctx->d_gs); cudaFree(ctx->d_wave);
        for (auto q : ctx->d_q) if (q) cudaFreeAsync(q, nullptr);  // back to the pool (see transport())
        cudaFree(ctx->d_counters); cudaFreeHost(ctx->h_counters); cudaFree(ctx->d_stats); cudaFree(ctx->d_ledger);
        cudaFree(ctx->d_edep); cudaFree(ctx->d_dose); cudaFree(ctx->d_sigma); cudaFree(ctx->d_beam);
        for (auto e : ctx->ev) if (e) cudaEventDestroy(e);
        if (ctx->ev_src) cudaEventDestroy(ctx->ev_src);
        for (auto e : ctx->lev) cudaEventDestroy(e);
    }
    delete ctx;
}

mc_status mc_build_tables(mc_ctx* ctx, const mc_material* mats, int32_t n_mats, const mc_params* params) {
    if (!ctx) return MC_ERR_INVALID_ARG;
    if (!mats || !params || n_mats <= 0 || n_mats > MAX_MAT) return fail(ctx, MC_ERR_INVALID_ARG, "materials / params (n_mats must be 1..16)");
    if (!(params->d_maxs_cm > 0) || !(params->f_maxe > 0) || !(params->f_maxe <= 1)) return fail(ctx, MC_ERR_INVALID_ARG, "d_maxs_cm must be > 0 and f_maxe in (0, 1]");
    std::vector<double> rho_max(n_mats, 0.0);
    for (size_t i = 0; i < ctx->h_mat.size(); ++i) {
        if (ctx->h_mat[i] >= n_mats) return fail(ctx, MC_ERR_INVALID_ARG, "a voxel's material index is >= n_mats");
        rho_max[ctx->h_mat[i]] = std::max(rho_max[ctx->h_mat[i]], (double)ctx->h_rho[i]);
    }
    std::vector<MaterialSpec> specs(n_mats);
    for (int m = 0; m < n_mats; ++m) {
        const mc_material& s = mats[m];
        if (s.n_elem <= 0 || !s.Z || !s.A || !s.w) return fail(ctx, MC_ERR_INVALID_ARG, "material without elements");
        for (int e = 0; e < s.n_elem; ++e) specs[m].el.push_back(Element{s.Z[e], (double)s.A[e], (double)s.w[e]});
        specs[m].I_eV = s.I_eV; specs[m].rho_nominal = s.rho_nominal;
    }
    TableParams tp{(double)params->e_cut_MeV, (double)params->g_cut_MeV, (double)params->e_max_MeV, params->n_grid};
    Tables t;
    std::string msg = build_tables(specs, tp, rho_max, t);
    if (!msg.empty()) return fail(ctx, MC_ERR_INVALID_ARG, msg);
    ctx->tabs = std::move(t);
    ctx->params = *params;
    const int N = ctx->tabs.N;
    ctx->lnE0P = (float)ctx->tabs.lnE0; ctx->inv_dlnP = (float)(1.0 / ctx->tabs.dln);
    ctx->p_maj = ctx->tabs.mu_maj;
    ctx->p_tot.resize((size_t)n_mats * N); ctx->p_C.resize((size_t)n_mats * N); ctx->p_pp.resize((size_t)n_mats * N);
    for (int m = 0; m < n_mats; ++m) {
        std::copy(ctx->tabs.t[T_MU_TOT][m].begin(), ctx->tabs.t[T_MU_TOT][m].end(), ctx->p_tot.begin() + (size_t)m * N);
        std::copy(ctx->tabs.t[T_MU_C][m].begin(), ctx->tabs.t[T_MU_C][m].end(), ctx->p_C.begin() + (size_t)m * N);
        std::copy(ctx->tabs.t[T_MU_PP][m].begin(), ctx->tabs.t[T_MU_PP][m].end(), ctx->p_pp.begin() + (size_t)m * N);
    }
    ctx->have_tables = true; ctx->tables_dirty = true; ctx->beam_key = -1.0;
    return MC_OK;
}

mc_status mc_export_table(const mc_ctx* cctx, int32_t material, int32_t which, float* out) {
    mc_ctx* ctx = const_cast<mc_ctx*>(cctx);
    if (!ctx || !out) return MC_ERR_INVALID_ARG;
    if (!ctx->have_tables) return fail(ctx, MC_ERR_STATE, "mc_build_tables has not been called");
    const int N = ctx->tabs.N;
    if (which == 9) { std::copy(ctx->p_maj.begin(), ctx->p_maj.end(), out); return MC_OK; }
    if (which < 0 || which > 10 || material < 0 || material >= ctx->tabs.n_mat) return fail(ctx, MC_ERR_INVALID_ARG, "table id / material");
    const float* src;
    if (which == 0) src = ctx->p_tot.data() + (size_t)material * N;
    else if (which == 1) src = ctx->p_C.data() + (size_t)material * N;
    else if (which == 2) src = ctx->p_pp.data() + (size_t)material * N;
    else src = ctx->tabs.t[which == 10 ? (int)T_LNA : which][material].data();  // TableId order matches mc.h for 3..8
    std::copy(src, src + N, out);
    return MC_OK;
}

mc_status mc_export_gs_table(int32_t dims[3], float* t_nodes, float* y) {
    if (!dims) return MC_ERR_INVALID_ARG;
    const GsTable& G = gs_table();
    dims[0] = kGsNT; dims[1] = kGsNA; dims[2] = kGsNQ;
    if (t_nodes) std::copy(G.t, G.t + kGsNT, t_nodes);
    if (y) std::copy(G.y.begin(), G.y.end(), y);
    return MC_OK;
}

mc_status mc_export_grid(const mc_ctx* cctx, double grid[4]) {
    mc_ctx* ctx = const_cast<mc_ctx*>(cctx);
    if (!ctx || !grid) return MC_ERR_INVALID_ARG;
    if (!ctx->have_tables) return fail(ctx, MC_ERR_STATE, "mc_build_tables has not been called");
    grid[0] = ctx->tabs.lnE0; grid[1] = ctx->tabs.dln; grid[2] = ctx->tabs.N; grid[3] = ctx->tabs.k_cut;
    return MC_OK;
}

mc_status mc_set_photon_tables(mc_ctx* ctx, float lnE0, float inv_dln, const float* mu_maj, const float* mu_tot, const float* mu_C,
                               const float* mu_pp) {
    if (!ctx) return MC_ERR_INVALID_ARG;
    if (!ctx->have_tables) return fail(ctx, MC_ERR_STATE, "mc_build_tables has not been called");
    if (!mu_maj || !mu_tot || !mu_C || !mu_pp || !(inv_dln > 0)) return fail(ctx, MC_ERR_INVALID_ARG, "photon tables");
    const size_t N = ctx->tabs.N, nm = ctx->tabs.n_mat;
    ctx->lnE0P = lnE0; ctx->inv_dlnP = inv_dln;
    ctx->p_maj.assign(mu_maj, mu_maj + N);
    ctx->p_tot.assign(mu_tot, mu_tot + nm * N); ctx->p_C.assign(mu_C, mu_C + nm * N); ctx->p_pp.assign(mu_pp, mu_pp + nm * N);
    ctx->tables_dirty = true; ctx->beam_key = -1.0;
    return MC_OK;
}

mc_status mc_run_range(mc_ctx* ctx, const mc_beam* beam, uint64_t n_histories, uint64_t h_begin, uint64_t h_end, uint64_t seed,
                       int32_t n_batches, float* edep_out) {
    mc_status st = check_run_args(ctx, beam, n_histories, h_begin, h_end, n_batches);
    if (st != MC_OK) return st;
    if (!edep_out) return fail(ctx, MC_ERR_INVALID_ARG, "edep_out is null");
    if ((st = ensure_device(ctx)) != MC_OK) return st;
    const size_t n = (size_t)n_batches * ctx->g.nvox;
    if ((st = ensure_edep(ctx, n)) != MC_OK) return st;
    if ((st = transport_beam(ctx, beam, n_histories, h_begin, h_end, seed, n_batches, ctx->d_edep)) != MC_OK) return st;
    if (edep_out != ctx->d_edep) CU(cudaMemcpyAsync(edep_out, ctx->d_edep, n * sizeof(float), cudaMemcpyDefault, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return MC_OK;
}

mc_status mc_finalize(mc_ctx* ctx, const float* edep, uint64_t n_histories, int32_t n_batches, float* dose_out, float* sigma_out) {
    if (!ctx) return MC_ERR_INVALID_ARG;
    if (!edep || !dose_out || !sigma_out || n_batches < 2 || n_histories < (uint64_t)n_batches) return fail(ctx, MC_ERR_INVALID_ARG, "mc_finalize arguments");
    mc_status st;
    if ((st = ensure_device(ctx)) != MC_OK) return st;
    const size_t nvox = ctx->g.nvox, n = (size_t)n_batches * nvox;
    if ((st = ensure_edep(ctx, n)) != MC_OK) return st;
    if (edep != ctx->d_edep) CU(cudaMemcpyAsync(ctx->d_edep, edep, n * sizeof(float), cudaMemcpyDefault, ctx->stream));
    if ((st = finalize_device(ctx, ctx->d_edep, n_histories, n_batches)) != MC_OK) return st;
    CU(cudaMemcpyAsync(dose_out, ctx->d_dose, nvox * sizeof(float), cudaMemcpyDefault, ctx->stream));
    CU(cudaMemcpyAsync(sigma_out, ctx->d_sigma, nvox * sizeof(float), cudaMemcpyDefault, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return MC_OK;
}

mc_status mc_edep_buffer(mc_ctx* ctx, int32_t n_batches, float** out) {
    if (!ctx || !out || n_batches < 1) return MC_ERR_INVALID_ARG;
    mc_status st;
    if ((st = ensure_device(ctx)) != MC_OK) return st;
    if ((st = ensure_edep(ctx, (size_t)n_batches * ctx->g.nvox)) != MC_OK) return st;
    *out = ctx->d_edep;
    return MC_OK;
}

mc_status mc_finalize_multi_range(mc_ctx* ctx, const float* const* edep_grids, int32_t n_grids, uint64_t n_histories, int32_t n_batches,
                                  int64_t v_begin, int64_t v_end, float* dose_out, float* sigma_out) {
    if (!ctx) return MC_ERR_INVALID_ARG;
    if (!edep_grids || n_grids < 1 || n_grids > kMaxGrids || !dose_out || !sigma_out || n_batches < 2 || n_histories < (uint64_t)n_batches)
        return fail(ctx, MC_ERR_INVALID_ARG, "mc_finalize_multi arguments (1 <= n_grids <= 16)");
    if (v_begin < 0 || v_end < v_begin || v_end > (int64_t)ctx->g.nvox) return fail(ctx, MC_ERR_INVALID_ARG, "mc_finalize_multi_range: voxel range");
    mc_status st;
    if ((st = ensure_device(ctx)) != MC_OK) return st;
    GridList gl;
    gl.n = n_grids;
    for (int r = 0; r < kMaxGrids; ++r) gl.g[r] = r < n_grids ? edep_grids[r] : nullptr;
    for (int r = 0; r < n_grids; ++r) if (!gl.g[r]) return fail(ctx, MC_ERR_INVALID_ARG, "mc_finalize_multi: null grid");
    const int nvox = ctx->g.nvox, nv = (int)(v_end - v_begin);
    if (nv == 0) return MC_OK;  // an empty slice (more ranks than voxels)
    const double vol = (double)ctx->g.hx * (double)ctx->g.hy * (double)ctx->g.hz;
    const int grid = std::max(1, std::min(ctx->sm_count * 8, (nv + kThreads - 1) / kThreads));
    finalize_multi_kernel<<<grid, kThreads, n_batches * sizeof(double), ctx->stream>>>(gl, ctx->d_vox, nvox, (int)v_begin, (int)v_end, n_batches,
                                                                                       n_histories, vol, ctx->d_dose, ctx->d_sigma);
    CU(cudaGetLastError());
    ++ctx->stats.n_kernel_launches;
    CU(cudaMemcpyAsync(dose_out, ctx->d_dose + v_begin, (size_t)nv * sizeof(float), cudaMemcpyDefault, ctx->stream));
    CU(cudaMemcpyAsync(sigma_out, ctx->d_sigma + v_begin, (size_t)nv * sizeof(float), cudaMemcpyDefault, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return MC_OK;
}

mc_status mc_finalize_multi(mc_ctx* ctx, const float* const* edep_grids, int32_t n_grids, uint64_t n_histories, int32_t n_batches,
                            float* dose_out, float* sigma_out) {
    if (!ctx) return MC_ERR_INVALID_ARG;
    return mc_finalize_multi_range(ctx, edep_grids, n_grids, n_histories, n_batches, 0, ctx->g.nvox, dose_out, sigma_out);
}

mc_status mc_ipc_get_handle(const void* dev_ptr, uint8_t handle[64]) {
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "cudaIpcMemHandle_t is 64 bytes");
    if (!dev_ptr || !handle) return MC_ERR_INVALID_ARG;
    cudaIpcMemHandle_t h;
    if (cudaIpcGetMemHandle(&h, const_cast<void*>(dev_ptr)) != cudaSuccess) { cudaGetLastError(); return MC_ERR_CUDA; }
    memcpy(handle, &h, 64);
    return MC_OK;
}
mc_status mc_ipc_open_handle(const uint8_t handle[64], void** dev_ptr) {
    if (!handle || !dev_ptr) return MC_ERR_INVALID_ARG;
    cudaIpcMemHandle_t h;
    memcpy(&h, handle, 64);
    if (cudaIpcOpenMemHandle(dev_ptr, h, cudaIpcMemLazyEnablePeerAccess) != cudaSuccess) { cudaGetLastError(); return MC_ERR_CUDA; }
    return MC_OK;
}
mc_status mc_ipc_close_handle(void* dev_ptr) {
    if (!dev_ptr) return MC_ERR_INVALID_ARG;
    if (cudaIpcCloseMemHandle(dev_ptr) != cudaSuccess) { cudaGetLastError(); return MC_ERR_CUDA; }
    return MC_OK;
}

mc_status mc_run(mc_ctx* ctx, const mc_beam* beam, uint64_t n_histories, uint64_t seed, int32_t n_batches, float* dose_out,
                 float* sigma_out) {
    mc_status st = check_run_args(ctx, beam, n_histories, 0, n_histories, n_batches);
    if (st != MC_OK) return st;
    if (!dose_out || !sigma_out) return fail(ctx, MC_ERR_INVALID_ARG, "dose_out / sigma_out is null");
    if ((st = ensure_device(ctx)) != MC_OK) return st;
    const size_t nvox = ctx->g.nvox;
    if ((st = ensure_edep(ctx, (size_t)n_batches * nvox)) != MC_OK) return st;
    if ((st = transport_beam(ctx, beam, n_histories, 0, n_histories, seed, n_batches, ctx->d_edep)) != MC_OK) return st;
    if ((st = finalize_device(ctx, ctx->d_edep, n_histories, n_batches)) != MC_OK) return st;
    CU(cudaMemcpyAsync(dose_out, ctx->d_dose, nvox * sizeof(float), cudaMemcpyDefault, ctx->stream));
    CU(cudaMemcpyAsync(sigma_out, ctx->d_sigma, nvox * sizeof(float), cudaMemcpyDefault, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return MC_OK;
}

mc_status mc_run_particles(mc_ctx* ctx, const mc_particle* particles, uint64_t n, uint64_t seed, int32_t n_batches, float* dose_out,
                           float* sigma_out) {
    if (!ctx) return MC_ERR_INVALID_ARG;
    if (!ctx->have_tables) return fail(ctx, MC_ERR_STATE, "mc_build_tables has not been called");
    if (!particles || !dose_out || !sigma_out) return fail(ctx, MC_ERR_INVALID_ARG, "null pointer");
    if (n == 0 || n >= (1ull << 32)) return fail(ctx, MC_ERR_INVALID_ARG, "n must be in [1, 2^32)");
    if (n_batches < 2 || (uint64_t)n_batches > n) return fail(ctx, MC_ERR_INVALID_ARG, "n_batches must be in [2, n]");
    if ((uint64_t)n_batches * (uint64_t)ctx->g.nvox >= (1ull << 32)) return fail(ctx, MC_ERR_INVALID_ARG, "n_batches * nvox must be < 2^32");
    static_assert(sizeof(mc_particle) == sizeof(ListParticle), "mc_particle layout");
    mc_status st;
    if ((st = ensure_device(ctx)) != MC_OK) return st;
    // the list may be host or device memory: a host list is staged on the device and checked against e_max
    cudaPointerAttributes at;
    const bool on_device = cudaPointerGetAttributes(&at, particles) == cudaSuccess && at.type == cudaMemoryTypeDevice;
    cudaGetLastError();
    const ListParticle* d_list = reinterpret_cast<const ListParticle*>(particles);
    ListParticle* staged = nullptr;
    if (!on_device) {
        for (uint64_t i = 0; i < n; ++i) {
            const mc_particle& q = particles[i];
            // the same three checks, with the same status codes, as check_particles_kernel applies to a device list
            if (!(q.E > 0.0f) || !(q.E <= ctx->params.e_max_MeV)) return fail(ctx, MC_ERR_ENERGY_RANGE, "particle energy not in (0, e_max_MeV]");
            const float nn = q.u * q.u + q.v * q.v + q.w * q.w;
            if (!(std::fabs(nn - 1.0f) < 1e-3f)) return fail(ctx, MC_ERR_INVALID_ARG, "particle directions must be unit vectors");
            if (q.particle < -1 || q.particle > 1) return fail(ctx, MC_ERR_INVALID_ARG, "particle types must be -1, 0 or 1");
        }
        CU(cudaMalloc(&staged, n * sizeof(ListParticle)));
        cudaError_t e = cudaMemcpyAsync(staged, particles, n * sizeof(ListParticle), cudaMemcpyHostToDevice, ctx->stream);
        if (e != cudaSuccess) { cudaFree(staged); return fail(ctx, MC_ERR_CUDA, cudaGetErrorString(e)); }
        d_list = staged;
    }
    const size_t nvox = ctx->g.nvox;
    st = MC_OK;
    if (on_device) {
        // a device-resident list is checked where it is: one pass, one flag word back (bit 0: energy not in (0, e_max],
        // bit 1: direction not a unit vector, bit 2: unknown particle type)
        cudaError_t e = cudaMemsetAsync(ctx->d_counters + C_FLAGS, 0, sizeof(uint32_t), ctx->stream);
        if (e == cudaSuccess) {
            check_particles_kernel<<<std::min<uint64_t>((n + kThreads - 1) / kThreads, (uint64_t)ctx->sm_count * 8), kThreads, 0, ctx->stream>>>(
                d_list, (uint32_t)n, ctx->params.e_max_MeV, ctx->d_counters + C_FLAGS);
            e = cudaGetLastError();
        }
        uint32_t bad = 0;
        if (e == cudaSuccess) e = cudaMemcpyAsync(&bad, ctx->d_counters + C_FLAGS, sizeof bad, cudaMemcpyDeviceToHost, ctx->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
        if (e != cudaSuccess) st = fail(ctx, MC_ERR_CUDA, cudaGetErrorString(e));
        else if (bad & 1u) st = fail(ctx, MC_ERR_ENERGY_RANGE, "particle energy not in (0, e_max_MeV]");
        else if (bad & 6u) st = fail(ctx, MC_ERR_INVALID_ARG, "particle directions must be unit vectors and particle types -1, 0 or 1");
    }
    if (st == MC_OK) st = ensure_edep(ctx, (size_t)n_batches * nvox);
    if (st == MC_OK) st = transport(ctx, nullptr, d_list, n, 0, n, seed, n_batches, ctx->d_edep);
    if (st == MC_OK) st = finalize_device(ctx, ctx->d_edep, n, n_batches);
    if (st == MC_OK) {
        cudaError_t e = cudaMemcpyAsync(dose_out, ctx->d_dose, nvox * sizeof(float), cudaMemcpyDefault, ctx->stream);
        if (e == cudaSuccess) e = cudaMemcpyAsync(sigma_out, ctx->d_sigma, nvox * sizeof(float), cudaMemcpyDefault, ctx->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
        if (e != cudaSuccess) st = fail(ctx, MC_ERR_CUDA, cudaGetErrorString(e));
    } else cudaStreamSynchronize(ctx->stream);
    if (staged) cudaFree(staged);
    return st;
}

mc_status mc_run_source(mc_ctx* ctx, mc_source_fn fn, void* user, uint64_t n, uint64_t seed, int32_t n_batches, float* dose_out,
                        float* sigma_out) {
    if (!ctx) return MC_ERR_INVALID_ARG;
    if (!ctx->have_tables) return fail(ctx, MC_ERR_STATE, "mc_build_tables has not been called");
    if (!fn || !dose_out || !sigma_out) return fail(ctx, MC_ERR_INVALID_ARG, "null pointer");
    if (n == 0 || n >= (1ull << 32)) return fail(ctx, MC_ERR_INVALID_ARG, "n must be in [1, 2^32)");
    if (n_batches < 2 || (uint64_t)n_batches > n) return fail(ctx, MC_ERR_INVALID_ARG, "n_batches must be in [2, n]");
    if ((uint64_t)n_batches * (uint64_t)ctx->g.nvox >= (1ull << 32)) return fail(ctx, MC_ERR_INVALID_ARG, "n_batches * nvox must be < 2^32");
    mc_status st;
    if ((st = ensure_device(ctx)) != MC_OK) return st;
    const size_t nvox = ctx->g.nvox;
    if ((st = ensure_edep(ctx, (size_t)n_batches * nvox)) != MC_OK) return st;
    SourceFn src; src.fn = fn; src.user = user;
    if ((st = transport(ctx, nullptr, nullptr, n, 0, n, seed, n_batches, ctx->d_edep, src)) != MC_OK) { cudaStreamSynchronize(ctx->stream); return st; }
    if ((st = finalize_device(ctx, ctx->d_edep, n, n_batches)) != MC_OK) return st;
    CU(cudaMemcpyAsync(dose_out, ctx->d_dose, nvox * sizeof(float), cudaMemcpyDefault, ctx->stream));
    CU(cudaMemcpyAsync(sigma_out, ctx->d_sigma, nvox * sizeof(float), cudaMemcpyDefault, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return MC_OK;
}

mc_status mc_run_atten(mc_ctx* ctx, const mc_beam* beam, uint64_t n, uint64_t seed, int32_t* voxel_out, uint8_t* channel_out) {
    if (!ctx) return MC_ERR_INVALID_ARG;
    if (!ctx->have_tables) return fail(ctx, MC_ERR_STATE, "mc_build_tables has not been called");
    mc_status st = check_beam(ctx, beam);
    if (st != MC_OK) return st;
    if (beam->particle != MC_PHOTON) return fail(ctx, MC_ERR_INVALID_ARG, "mc_run_atten takes photon beams only");
    if (n >= (1ull << 32)) return fail(ctx, MC_ERR_INVALID_ARG, "n must be < 2^32");
    if (n == 0) return MC_OK;
    if (!voxel_out) return fail(ctx, MC_ERR_INVALID_ARG, "voxel_out is null");
    if ((st = ensure_device(ctx)) != MC_OK) return st;
    if ((st = upload_tables(ctx)) != MC_OK) return st;
    RunParams P;
    memset(&P, 0, sizeof P);
    fill_params(ctx, P);
    if ((st = upload_beam(ctx, beam, P.beam)) != MC_OK) return st;
    P.seed_lo = (uint32_t)seed; P.seed_hi = (uint32_t)(seed >> 32);
    int32_t* d_v = nullptr; uint8_t* d_c = nullptr;
    CU(cudaMalloc(&d_v, n * sizeof(int32_t)));
    if (cudaMalloc(&d_c, n) != cudaSuccess) { cudaFree(d_v); return fail(ctx, MC_ERR_OOM, "cudaMalloc"); }
    const int grid = (int)std::min<uint64_t>((uint64_t)ctx->sm_count * 8, (n + kThreads - 1) / kThreads);
    atten_kernel<<<grid, kThreads, 0, ctx->stream>>>(P, n, d_v, d_c);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemcpyAsync(voxel_out, d_v, n * sizeof(int32_t), cudaMemcpyDefault, ctx->stream);
    if (e == cudaSuccess && channel_out) e = cudaMemcpyAsync(channel_out, d_c, n, cudaMemcpyDefault, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    cudaFree(d_v); cudaFree(d_c);
    if (e != cudaSuccess) return fail(ctx, MC_ERR_CUDA, std::string("mc_run_atten: ") + cudaGetErrorString(e));
    return MC_OK;
}

mc_status mc_philox_selftest(const uint32_t* ctr, const uint32_t* key, int32_t n, uint32_t* out) {
    if (!ctr || !key || !out || n <= 0) return MC_ERR_INVALID_ARG;
    uint32_t *d_c = nullptr, *d_k = nullptr, *d_o = nullptr;
    cudaError_t e = cudaMalloc(&d_c, (size_t)n * 16);
    if (e == cudaSuccess) e = cudaMalloc(&d_k, (size_t)n * 8);
    if (e == cudaSuccess) e = cudaMalloc(&d_o, (size_t)n * 16);
    if (e == cudaSuccess) e = cudaMemcpy(d_c, ctr, (size_t)n * 16, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(d_k, key, (size_t)n * 8, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        philox_test_kernel<<<(n + 127) / 128, 128>>>(d_c, d_k, n, d_o);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpy(out, d_o, (size_t)n * 16, cudaMemcpyDeviceToHost);
    cudaFree(d_c); cudaFree(d_k); cudaFree(d_o);
    if (e != cudaSuccess) { cudaGetLastError(); return MC_ERR_CUDA; }
    return MC_OK;
}

mc_status mc_u01_selftest(uint64_t* n_mismatch) {
    if (!n_mismatch) return MC_ERR_INVALID_ARG;
    unsigned long long* d = nullptr;
    cudaError_t e = cudaMalloc(&d, sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMemset(d, 0, sizeof(unsigned long long));
    if (e == cudaSuccess) {
        u01_test_kernel<<<148 * 8, 256>>>(d);
        e = cudaGetLastError();
    }
    unsigned long long h = ~0ull;
    if (e == cudaSuccess) e = cudaMemcpy(&h, d, sizeof h, cudaMemcpyDeviceToHost);
    cudaFree(d);
    if (e != cudaSuccess) { cudaGetLastError(); return MC_ERR_CUDA; }
    *n_mismatch = h;
    return MC_OK;
}

mc_status mc_bench_red(mc_ctx* ctx, uint32_t n_cells, int32_t per_thread, int32_t mode, int32_t blocks, double* ms_out) {
    if (!ctx || !ms_out || n_cells == 0 || per_thread <= 0 || blocks <= 0 || mode < 0 || mode > 1) return MC_ERR_INVALID_ARG;
    mc_status st;
    if ((st = ensure_device(ctx)) != MC_OK) return st;
    float* d = nullptr;
    CU(cudaMalloc(&d, (size_t)n_cells * sizeof(float)));
    cudaMemsetAsync(d, 0, (size_t)n_cells * sizeof(float), ctx->stream);
    red_bench_kernel<<<blocks, kThreads, 0, ctx->stream>>>(d, n_cells, 1, mode);  // warm-up
    cudaEventRecord(ctx->ev[2], ctx->stream);
    red_bench_kernel<<<blocks, kThreads, 0, ctx->stream>>>(d, n_cells, per_thread, mode);
    cudaEventRecord(ctx->ev[3], ctx->stream);
    cudaError_t e = cudaStreamSynchronize(ctx->stream);
    float ms = 0;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, ctx->ev[2], ctx->ev[3]);
    cudaFree(d);
    if (e != cudaSuccess) return fail(ctx, MC_ERR_CUDA, std::string("mc_bench_red: ") + cudaGetErrorString(e));
    *ms_out = ms;
    return MC_OK;
}

mc_status mc_bench_issue(mc_ctx* ctx, int32_t iters, double* thread_instr_per_s) {
    if (!ctx || !thread_instr_per_s || iters <= 0) return MC_ERR_INVALID_ARG;
    mc_status st;
    if ((st = ensure_device(ctx)) != MC_OK) return st;
    const int blocks = ctx->sm_count * 2;
    issue_bench_kernel<<<blocks, 1024, 0, ctx->stream>>>(ctx->d_dose, 16);  // warm-up
    cudaEventRecord(ctx->ev[2], ctx->stream);
    issue_bench_kernel<<<blocks, 1024, 0, ctx->stream>>>(ctx->d_dose, iters);
    cudaEventRecord(ctx->ev[3], ctx->stream);
    cudaError_t e = cudaStreamSynchronize(ctx->stream);
    float ms = 0;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, ctx->ev[2], ctx->ev[3]);
    if (e != cudaSuccess || !(ms > 0)) return fail(ctx, MC_ERR_CUDA, std::string("mc_bench_issue: ") + cudaGetErrorString(e));
    *thread_instr_per_s = (double)blocks * 1024.0 * (double)iters * 64.0 / (ms * 1e-3);
    return MC_OK;
}

mc_status mc_trim(uint64_t keep_bytes) {
    int n = 0;
    if (cudaGetDeviceCount(&n) != cudaSuccess || n <= 0) { cudaGetLastError(); return MC_ERR_CUDA; }
    cudaMemPool_t pool = queue_pool();
    if (!pool) return MC_ERR_CUDA;
    // queues go back to the pool with cudaFreeAsync: they count as unused once that has executed
    if (cudaDeviceSynchronize() != cudaSuccess || cudaMemPoolTrimTo(pool, (size_t)keep_bytes) != cudaSuccess) { cudaGetLastError(); return MC_ERR_CUDA; }
    return MC_OK;
}

mc_status mc_get_stats(const mc_ctx* ctx, mc_stats* out) {
    if (!ctx || !out) return MC_ERR_INVALID_ARG;
    *out = ctx->stats;
    return MC_OK;
}

mc_status mc_set_stream(mc_ctx* ctx, void* cuda_stream) {
    if (!ctx) return MC_ERR_INVALID_ARG;
    ctx->stream = (cudaStream_t)cuda_stream;
    return MC_OK;
}

mc_status mc_set_option(mc_ctx* ctx, const char* name, int64_t value) {
    if (!ctx || !name) return MC_ERR_INVALID_ARG;
    const std::string n(name);
    if (n == "wave_size") { if (value < 1024 || value > (1ll << 28)) return fail(ctx, MC_ERR_INVALID_ARG, "wave_size in [1024, 2^28]"); ctx->wave_size = value; }
    else if (n == "queue_factor") { if (value < 2 || value > 64) return fail(ctx, MC_ERR_INVALID_ARG, "queue_factor in [2, 64]"); ctx->queue_factor = value; }
    else if (n == "blocks_per_sm") { if (value < 0 || value > 32) return fail(ctx, MC_ERR_INVALID_ARG, "blocks_per_sm in [0, 32]"); ctx->blocks_per_sm = value; }
    else if (n == "refill_lanes") { if (value < 1 || value > 64) return fail(ctx, MC_ERR_INVALID_ARG, "refill_lanes in [1, 64]"); ctx->refill_lanes = value; }
    else if (n == "hard_lanes") { if (value < 1 || value > 64) return fail(ctx, MC_ERR_INVALID_ARG, "hard_lanes in [1, 64]"); ctx->hard_lanes = value; }
    else if (n == "adaptive") { if (value < 0 || value > 1) return fail(ctx, MC_ERR_INVALID_ARG, "adaptive in {0, 1}"); ctx->adaptive = value; }
    else if (n == "aggregate") { if (value < -1 || value > 1) return fail(ctx, MC_ERR_INVALID_ARG, "aggregate in {-1, 0, 1}"); ctx->aggregate = value; }
    else if (n == "hinge_overrun_pct") { if (value < 0 || value > 100) return fail(ctx, MC_ERR_INVALID_ARG, "hinge_overrun_pct in [0, 100]"); ctx->hinge_overrun_pct = value; }
    else if (n == "electron_threads") { if (value != 0 && value != 256 && value != 512 && value != 768 && value != 1024) return fail(ctx, MC_ERR_INVALID_ARG, "electron_threads in {0, 256, 512, 768, 1024}"); ctx->electron_threads = value; }
    else if (n == "plan_ahead") { if (value < 0 || value > 1) return fail(ctx, MC_ERR_INVALID_ARG, "plan_ahead in {0, 1}"); ctx->plan_ahead = value; }
    else if (n == "ms_carry") { if (value < 0 || value > 1) return fail(ctx, MC_ERR_INVALID_ARG, "ms_carry in {0, 1}"); ctx->ms_carry = value; }
    else return fail(ctx, MC_ERR_INVALID_ARG, "unknown option: " + n);
    ctx->beam_key = -1.0;  // scheduling options and readings change the secondaries-per-primary ratios: probe again
    return MC_OK;
}

const char* mc_last_error(const mc_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }
const char* mc_version(void) { return "paper_1503_01722_b200 0.2 (sm_100a)"; }

}  // extern "C"
