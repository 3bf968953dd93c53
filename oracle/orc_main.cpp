// ORACLE — test infrastructure only (parity reference + timed CPU baseline); see orc_physics.h.
// Plain, single-threaded, fp64, one history at a time, depth-first over the history's secondaries.
// Follows PAPER.md:33-39 (§2.1 Physics) step by step, in the readings DESIGN.md lists (R1..R26).
// Build: g++ -O2 -std=c++17 -ffp-contract=off -shared -fPIC (oracle/build.py).
//
// Pins (tests/test_oracle_*.py): Philox known answers; sigma_KN vs numerical integral of the
// differential cross section, Thomson limit, tabulated water values; pair branch continuity and
// asymptote; restricted-L identity L_col + int W dsigma_M = S_col and ESTAR-like water values;
// Moller / brems totals vs independent quadrature; chi-square of the KN, Moller, brems samplers;
// exp(-mu x) attenuation; CSDA range; per-history energy ledger; MS mean cosine; hard-event rate and first-event
// spectrum against the quadrature of Sigma/L; <cos> of the primary after a given energy loss against exp(-int K1/L dT)
// (one voxel and on a 0.25 cm grid: hinge rule R8 + MS carry R8b); rotation at the poles; annihilation isotropy.
// Every sampler is ONE function, called by transport and by the orc_sample_* pin entries alike.
// Sources: beams (R13) and particle lists (R13b, orc_run_particles).  Hinge vs voxel face: readings R8 / R8b (orc_set_option).
// Coupled dose: "parity unpinned" by any external number (no dose value in the paper is
// reproducible here: gDPM, XCOM data and the 6 MV spectrum are missing) — DESIGN.md says so.
#include "orc_physics.h"
#include "orc_gs.h"
#include <cstdint>
#include <cstring>
#include <cstdio>
#include <string>

using namespace orc;

// ------------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al. 2011); R15.
static inline void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// One random stream per particle track: key = (lo32(history), lo32(seed)),
// counter = (block, track_lo, track_hi, hi32(seed)).  Consumption is block-granular: every
// consumer site takes one fresh block and uses its words in a fixed order (R15).
struct Stream {
    uint32_t h, seed_lo, seed_hi, trk_lo, trk_hi, block;
    uint32_t w[4];
    void next() {
        uint32_t c[4] = {block, trk_lo, trk_hi, seed_hi}, k[2] = {h, seed_lo};
        philox4x32_10(c, k, w);
        ++block;
    }
    double u(int i) const { return ((double)(w[i] >> 9) + 0.5) * (1.0 / 8388608.0); }
};

// ------------------------------------------------------------------------------------------------
struct Params { double e_cut, g_cut, e_max; int n_grid; double d_maxs, f_maxe; uint32_t flags; };
enum { F_NO_HARD = 1, F_NO_MS = 2, F_LOCAL_SEC = 4, F_MS_GS = 8, F_MULTI_VOXEL = 16 };
static GsTable g_gs;  // the Goudsmit-Saunderson sampling table (material independent, orc_gs.h), built on first use

struct MatTables {  // all per unit density (cm^2/g, MeV cm^2/g, g/cm^2), one value per grid node
    std::vector<double> mu_tot, mu_C, mu_pp, R, L, S_hard, S_M, S_max, K1;
    std::vector<double> lnA;  // ln of the effective screening parameter (R27): K1 = S_el G_1(A)
};

struct Ctx {
    int nx = 0, ny = 0, nz = 0;
    double h[3], org[3];
    std::vector<uint8_t> mat;
    std::vector<double> rho;
    std::vector<float> rho_f;
    // tables
    bool have_tables = false;
    Params p{};
    std::vector<Material> mats;
    std::vector<MatTables> tab;
    std::vector<double> mu_maj;  // 1/cm
    int N = 0, k_cut = 0;
    double lnE0 = 0, dln = 0;
    // run-time options of the readings (orc_set_option): tests A/B them, the engine has the same switches
    double hinge_overrun = 0.25;  // DESIGN.md R8: the second leg may run on to the face by this fraction of its planned length
    int ms_carry = 1;             // DESIGN.md R8b: the MS path of a step = planned path + (actual - planned) path of the previous steps
    std::string err;
};

static inline double lerp_tab(const Ctx& c, const std::vector<double>& t, double E) {
    double x = (std::log(E) - c.lnE0) / c.dln;
    int i = (int)std::floor(x);
    if (i < 0) i = 0;
    if (i > c.N - 2) i = c.N - 2;
    double f = x - i;
    return t[i] + f * (t[i + 1] - t[i]);
}
// Inverse of the piecewise-linear (in ln T) range interpolant: T with R(T) = Rt (R5).
static inline double inv_range(const Ctx& c, const std::vector<double>& R, double Rt) {
    if (Rt <= 0.0) return c.p.e_cut;
    int lo = c.k_cut, hi = c.N - 1;  // R[lo] = 0 <= Rt
    while (hi - lo > 1) { int mid = (lo + hi) / 2; if (R[mid] <= Rt) lo = mid; else hi = mid; }
    double f = (Rt - R[lo]) / (R[lo + 1] - R[lo]);
    return std::exp(c.lnE0 + (lo + f) * c.dln);
}

// Energy grid: uniform in ln E, N nodes; spacing ln2/n2 so that with e_cut on a node 2*e_cut (the
// Moller threshold, a kink of Sigma_M) is on a node too; origin just below min(e_cut, g_cut).
static bool make_grid(Ctx& c) {
    const Params& p = c.p;
    double Elo = std::min(p.e_cut, p.g_cut);
    c.N = p.n_grid;
    double d0 = std::log(p.e_max / Elo) / (c.N - 1);
    int n2 = (int)std::floor(std::log(2.0) / d0);
    for (; n2 >= 1; --n2) {
        c.dln = std::log(2.0) / n2;
        c.k_cut = (int)std::ceil(std::log(p.e_cut / Elo) / c.dln - 1e-12);
        c.lnE0 = std::log(p.e_cut) - c.k_cut * c.dln;
        if (c.lnE0 + (c.N - 1) * c.dln >= std::log(p.e_max)) return true;
    }
    return false;
}

static void build_tables(Ctx& c) {
    int N = c.N;
    size_t nm = c.mats.size();
    c.tab.assign(nm, MatTables());
    std::vector<double> E(N);
    for (int j = 0; j < N; ++j) E[j] = std::exp(c.lnE0 + j * c.dln);
    E[c.k_cut] = c.p.e_cut;
    for (size_t m = 0; m < nm; ++m) {
        const Material& M = c.mats[m];
        MatTables& t = c.tab[m];
        for (auto* v : {&t.mu_tot, &t.mu_C, &t.mu_pp, &t.R, &t.L, &t.S_hard, &t.S_M, &t.S_max, &t.K1, &t.lnA}) v->assign(N, 0.0);
        for (int j = 0; j < N; ++j) {
            t.mu_C[j] = mu_compton(M, E[j]);
            t.mu_pp[j] = mu_pp(M, E[j]);
            t.mu_tot[j] = t.mu_C[j] + t.mu_pp[j] + mu_pe(M, E[j]);
            t.L[j] = L_total(M, E[j], c.p.e_cut, c.p.g_cut);
            t.S_M[j] = M.ne * moller_sigma(E[j], c.p.e_cut);
            t.S_hard[j] = t.S_M[j] + brems_sigma(M, E[j], c.p.g_cut);
            t.S_max[j] = std::max(t.S_hard[j], j ? t.S_max[j - 1] : 0.0);
            t.K1[j] = K1(M, E[j]);
            t.lnA[j] = std::log(gs_effective_A(t.K1[j], S_el(M, E[j])));
        }
        // range: R(e_cut) = 0, R(T) = int_{e_cut}^{T} dT'/L(T'), Simpson in ln T between nodes
        auto seg = [&](int j) {  // integral from node j to node j+1
            return simpson([&](double x) { double T = std::exp(x); return T / L_total(M, T, c.p.e_cut, c.p.g_cut); },
                           std::log(E[j]), std::log(E[j + 1]), 8);
        };
        t.R[c.k_cut] = 0.0;
        for (int j = c.k_cut; j < N - 1; ++j) t.R[j + 1] = t.R[j] + seg(j);
        for (int j = c.k_cut - 1; j >= 0; --j) t.R[j] = t.R[j + 1] - seg(j);
    }
    // photon majorant: per node, max over voxels of rho_v (mu/rho)_{m_v}  (R3)
    std::vector<double> rmax(nm, 0.0);
    for (size_t v = 0; v < c.mat.size(); ++v) rmax[c.mat[v]] = std::max(rmax[c.mat[v]], c.rho[v]);
    c.mu_maj.assign(N, 0.0);
    for (int j = 0; j < N; ++j)
        for (size_t m = 0; m < nm; ++m) c.mu_maj[j] = std::max(c.mu_maj[j], rmax[m] * c.tab[m].mu_tot[j]);
    c.have_tables = true;
    if (c.p.flags & F_MS_GS) g_gs.build();
}

// ------------------------------------------------------------------------------------------------
// Samplers and kinematics.  ONE function each: the transport code (Run::photon / Run::electron) and the
// orc_sample_* entry points of the chi-square / moment / conservation pins call the same code.
// Rejection loops take a fresh Philox block per two trials (words 0,1 then 2,3; R15).

// rotate direction d by polar cosine mu and azimuth phi (R25: polar-axis branch near +-z)
static void rotate_dir(double d[3], double mu, double phi) {
    double st_ = std::sqrt(std::max(0.0, 1.0 - mu * mu)), cp = std::cos(phi), sp = std::sin(phi);
    double s2 = 1.0 - d[2] * d[2];
    double nx_, ny_, nz_;
    if (s2 < 1e-10) {
        double sg = d[2] >= 0 ? 1.0 : -1.0;
        nx_ = st_ * cp; ny_ = st_ * sp; nz_ = sg * mu;
    } else {
        double s = std::sqrt(s2);
        nx_ = d[0] * mu + st_ * (d[0] * d[2] * cp - d[1] * sp) / s;
        ny_ = d[1] * mu + st_ * (d[1] * d[2] * cp + d[0] * sp) / s;
        nz_ = d[2] * mu - st_ * s * cp;
    }
    double n = std::sqrt(nx_ * nx_ + ny_ * ny_ + nz_ * nz_);
    d[0] = nx_ / n; d[1] = ny_ / n; d[2] = nz_ / n;
}

// Klein-Nishina by the epsilon decomposition (R4): eps = E'/E and tt = 1 - cos(theta).  The first word of a
// trial picks the branch of the decomposition AND, rescaled to (0,1) inside the branch, samples it.
struct KNSample { double eps, tt; };
static KNSample sample_kn(Stream& s, double E) {
    double k0 = E / MEC2, e0 = 1.0 / (1.0 + 2.0 * k0), a1 = std::log(1.0 / e0), a2 = 0.5 * (1.0 - e0 * e0);
    KNSample o;
    for (int k = 2;; ++k) {
        if (k == 2) { s.next(); k = 0; }
        double r = s.u(2 * k) * (a1 + a2);
        if (r < a1) o.eps = std::exp(-r);  // = e0^(r/a1)
        else o.eps = std::sqrt(e0 * e0 + (1.0 - e0 * e0) * (r - a1) / a2);
        o.tt = (1.0 - o.eps) / (k0 * o.eps);
        double sin2 = o.tt * (2.0 - o.tt);
        if (s.u(2 * k + 1) <= 1.0 - o.eps * sin2 / (1.0 + o.eps * o.eps)) break;
    }
    return o;
}
// Compton kinematics: photon direction d rotated in place by (1 - tt, phi); recoil electron direction from
// momentum conservation, E d0 - E' d' normalised.
static void compton_kinematics(double E, const KNSample& kn, double phi, double d[3], double de[3]) {
    double d0[3] = {d[0], d[1], d[2]}, E1 = kn.eps * E, n = 0;
    rotate_dir(d, 1.0 - kn.tt, phi);
    for (int a = 0; a < 3; ++a) { de[a] = E * d0[a] - E1 * d[a]; n += de[a] * de[a]; }
    n = std::sqrt(n);
    for (int a = 0; a < 3; ++a) de[a] /= n;
}
// Moller (R10): eps = W/T0 from the 1/eps^2 proposal on [e_cut/T0, 1/2], rejection g(eps)/max(g(eps_c), g(1/2)).
static double sample_moller(Stream& s, double T0, double e_cut) {
    double tau = T0 / MEC2, g = tau + 1.0, q = (2.0 * g - 1.0) / (g * g), q1 = (g - 1.0) / g;
    q1 *= q1;
    double ec = e_cut / T0;
    auto gf = [&](double e) { return 1.0 - q * e / (1.0 - e) + e * e * (q1 + 1.0 / ((1.0 - e) * (1.0 - e))); };
    double gmax = std::max(gf(ec), gf(0.5)), eps;
    for (int k = 2;; ++k) {
        if (k == 2) { s.next(); k = 0; }
        eps = 1.0 / (1.0 / ec - s.u(2 * k) * (1.0 / ec - 2.0));
        if (s.u(2 * k + 1) * gmax <= gf(eps)) break;
    }
    return eps;
}
// polar cosines of the primary (c1) and of the delta ray (c2) after a Moller event with energy transfer W
static void moller_angles(double T0, double W, double& c1, double& c2) {
    c1 = std::sqrt((T0 - W) * (T0 + 2.0 * MEC2) / (T0 * (T0 - W + 2.0 * MEC2)));
    c2 = std::sqrt(W * (T0 + 2.0 * MEC2) / (T0 * (W + 2.0 * MEC2)));
}
// Bremsstrahlung photon energy (R11): k = g_cut (T0/g_cut)^u, rejection F(k)/F_max.
static double sample_brems(Stream& s, const Material& M, double T0, double g_cut) {
    double Et = T0 + MEC2;
    auto Ff = [&](double k) { double Ep = Et - k, rr = Ep / Et; return (1.0 + rr * rr - 2.0 * rr / 3.0) * (std::min(std::log(2.0 * Et * Ep / (MEC2 * k)), M.Lscr) - 0.5); };
    double Fmax = (4.0 / 3.0) * (std::min(std::log(2.0 * Et * (Et - g_cut) / (MEC2 * g_cut)), M.Lscr) - 0.5), kk;
    for (int k = 2;; ++k) {
        if (k == 2) { s.next(); k = 0; }
        kk = g_cut * std::pow(T0 / g_cut, s.u(2 * k));
        if (s.u(2 * k + 1) * Fmax <= Ff(kk)) break;
    }
    return kk;
}
// Multiple scattering, Gaussian on the sphere (R7): 1 - cos(theta) for strength am = 1 - exp(-K1 rho d), uniform u.
static double sample_ms_omu(double am, double u) { return -am * std::log(1.0 - u * (1.0 - std::exp(-2.0 / am))); }
// Isotropic direction from two uniforms (annihilation photons, R9).
static void iso_direction(double u_mu, double u_phi, double d[3]) {
    double mu = 2.0 * u_mu - 1.0, phi = 2.0 * PI * u_phi, sn = std::sqrt(1.0 - mu * mu);
    d[0] = sn * std::cos(phi); d[1] = sn * std::sin(phi); d[2] = mu;
}

// ------------------------------------------------------------------------------------------------
struct Beam {
    int particle, shape;
    double entry[3], axis[3], ssd, field[2];
    std::vector<double> E, pdf;
    std::vector<double> cdf;  // cumulative trapezoid areas, normalised, size n_nodes (cdf[0]=0)
};

struct Particle {
    int q;  // 0 photon, -1 electron, +1 positron
    double x[3], d[3], E;
    int v[3];
    uint32_t trk_lo, trk_hi;
    uint32_t blk0 = 0;  // first RNG block of the track (1 for primaries: block 0 is the source block)
};

struct Stats {  // doubles so that the Python side can read one flat array
    double e_src, e_dep, e_esc, e_cutdep;  // e_dep includes e_cutdep
    double n_hist, n_flight, n_fict, n_compton, n_pair, n_pe;
    double n_estep, n_moller, n_brems, n_sec_e, n_sec_g, path_e;
    double lim_vox, lim_maxs, lim_maxe, lim_range, lim_event;
    double max_ledger_rel;
};
constexpr int N_STATS = sizeof(Stats) / sizeof(double);
constexpr int N_PROBE = 22;

struct Run {
    const Ctx& c;
    const Beam& b;
    uint64_t seed;
    double* edep;  // current batch grid (MeV)
    Stats& st;
    std::vector<Particle> stack;
    uint32_t hist = 0;
    int32_t first_vox = -1; int first_chan = -1;  // first real interaction of a primary photon
    double* probe = nullptr;  // optional per-history record of the primary electron track (N_PROBE doubles, see orc_run_probe)
    double led_src = 0, led_dep = 0, led_esc = 0;
    Run(const Ctx& c_, const Beam& b_, uint64_t s, Stats& st_) : c(c_), b(b_), seed(s), edep(nullptr), st(st_) {}

    Stream stream(const Particle& p) const { Stream s = stream(p.trk_lo, p.trk_hi); s.block = p.blk0; return s; }
    Stream stream(uint32_t lo, uint32_t hi) const {
        Stream s; s.h = hist; s.seed_lo = (uint32_t)seed; s.seed_hi = (uint32_t)(seed >> 32);
        s.trk_lo = lo; s.trk_hi = hi; s.block = 0; return s;
    }
    int vidx(const int v[3]) const { return v[0] + c.nx * (v[1] + c.ny * v[2]); }
    bool inside(const int v[3]) const { return v[0] >= 0 && v[0] < c.nx && v[1] >= 0 && v[1] < c.ny && v[2] >= 0 && v[2] < c.nz; }
    void deposit(const int v[3], double e, bool cut) {
        edep[vidx(v)] += e; led_dep += e; st.e_dep += e; if (cut) st.e_cutdep += e;
    }
    void escape(double e) { led_esc += e; st.e_esc += e; }
    bool locate(const double x[3], int v[3]) const {  // floor rule (R25)
        const int n[3] = {c.nx, c.ny, c.nz};
        for (int a = 0; a < 3; ++a) {
            double f = (x[a] - c.org[a]) / c.h[a];
            if (f < 0 || f >= n[a]) return false;
            v[a] = (int)f;
        }
        return true;
    }
    // secondary: transported, or deposited where born with F_LOCAL_SEC
    void push(const Particle& p) {
        if (p.q == 0) st.n_sec_g += 1; else st.n_sec_e += 1;
        if (c.p.flags & F_LOCAL_SEC) {
            deposit(p.v, p.E, false);
            if (p.q > 0) deposit(p.v, 2.0 * MEC2, false);  // keeps the ledger closed
            return;
        }
        stack.push_back(p);
    }

    // ---- source (R13): block 0 of track (0,0): w0 bin, w1 in-bin energy, w2 x, w3 y ----------
    bool source(Particle& p) {
        Stream s = stream(0, 0);
        s.next();
        double E;
        size_t nn = b.E.size();
        if (nn == 1) E = b.E[0];
        else {
            double u0 = s.u(0), u1 = s.u(1);
            size_t j = 0;
            while (j + 2 < nn && u0 >= b.cdf[j + 1]) ++j;
            double p0 = b.pdf[j], p1 = b.pdf[j + 1];
            double t = u1 * (p0 + p1) / (p0 + std::sqrt(p0 * p0 + u1 * (p1 * p1 - p0 * p0)));
            E = b.E[j] + t * (b.E[j + 1] - b.E[j]);
        }
        p.q = b.particle; p.E = E; p.trk_lo = 0; p.trk_hi = 0; p.blk0 = 1;
        if (b.shape == 0) {
            for (int a = 0; a < 3; ++a) { p.x[a] = b.entry[a]; p.d[a] = b.axis[a]; }
        } else {
            double fx = (s.u(2) - 0.5) * b.field[0], fy = (s.u(3) - 0.5) * b.field[1];
            p.x[0] = b.entry[0] + fx; p.x[1] = b.entry[1] + fy; p.x[2] = b.entry[2];
            double n = std::sqrt(fx * fx + fy * fy + b.ssd * b.ssd);
            p.d[0] = fx / n; p.d[1] = fy / n; p.d[2] = b.ssd / n;
        }
        led_src += E; st.e_src += E;
        if (!locate(p.x, p.v)) { escape(E + (p.q > 0 ? 2.0 * MEC2 : 0.0)); if (p.q > 0) { led_src += 2 * MEC2; st.e_src += 2 * MEC2; } return false; }
        if (p.q > 0) { led_src += 2.0 * MEC2; st.e_src += 2.0 * MEC2; }  // a positron source carries 2mc^2 of annihilation energy
        return true;
    }

    // ---- photon (R3, R4, R12, R16) --------------------------------------------------
    void photon(Particle p) {
        Stream s = stream(p);
        if (p.E < c.p.g_cut) { deposit(p.v, p.E, true); return; }
        for (;;) {
            double maj = lerp_tab(c, c.mu_maj, p.E);
            s.next();
            int chan = -1;
            for (int k = 0; k < 2 && chan < 0; ++k) {  // one block serves two flights
                double sl = -std::log(s.u(2 * k)) / maj;
                for (int a = 0; a < 3; ++a) p.x[a] += sl * p.d[a];
                st.n_flight += 1;
                if (!locate(p.x, p.v)) { escape(p.E); return; }
                int vi = vidx(p.v);
                const MatTables& t = c.tab[c.mat[vi]];
                double rho = c.rho[vi];
                double r = s.u(2 * k + 1) * maj;
                double mu = rho * lerp_tab(c, t.mu_tot, p.E);
                if (r > mu) { st.n_fict += 1; continue; }
                double mc = rho * lerp_tab(c, t.mu_C, p.E);
                double mp = rho * lerp_tab(c, t.mu_pp, p.E);
                chan = r < mc ? 0 : (r < mc + mp ? 1 : 2);
            }
            if (chan < 0) continue;
            if (p.trk_lo == 0 && p.trk_hi == 0 && first_chan < 0) { first_vox = vidx(p.v); first_chan = chan; }
            if (chan == 2) { st.n_pe += 1; deposit(p.v, p.E, false); return; }  // absorbed locally
            if (chan == 1) {  // pair: both along the photon direction, uniform split
                st.n_pair += 1;
                s.next();
                double Tk = p.E - 2.0 * MEC2, us = s.u(2);
                Particle em = p; em.q = -1; em.blk0 = 0; em.E = us * Tk; em.trk_lo = s.w[0]; em.trk_hi = s.w[1];
                s.next();
                Particle ep = p; ep.q = +1; ep.blk0 = 0; ep.E = (1.0 - us) * Tk; ep.trk_lo = s.w[0]; ep.trk_hi = s.w[1];
                push(em); push(ep);
                return;
            }
            // Compton: Klein-Nishina by the epsilon decomposition (R4)
            st.n_compton += 1;
            KNSample kn = sample_kn(s, p.E);
            s.next();
            double E1 = kn.eps * p.E;
            Particle e = p; e.q = -1; e.blk0 = 0; e.E = p.E - E1; e.trk_lo = s.w[0]; e.trk_hi = s.w[1];
            compton_kinematics(p.E, kn, 2.0 * PI * s.u(2), p.d, e.d);
            push(e);
            p.E = E1;
            if (p.E < c.p.g_cut) { deposit(p.v, p.E, true); return; }
        }
    }

    // distance to the voxel face along d from x inside voxel v; axis of the face in ax
    double face_dist(const double x[3], const double d[3], const int v[3], int& ax) const {
        double best = 1e300; ax = -1;
        for (int a = 0; a < 3; ++a) {
            double t;
            if (d[a] > 0) t = (c.org[a] + (v[a] + 1) * c.h[a] - x[a]) / d[a];
            else if (d[a] < 0) t = (c.org[a] + v[a] * c.h[a] - x[a]) / d[a];
            else continue;
            if (t < 0) t = 0;
            if (t < best) { best = t; ax = a; }
        }
        return best;
    }

    // ---- electron / positron (R2, R5..R11) --------------------------------------
    // ---- electron / positron, multi-voxel steps (gDPM "employed a fixed step algorithm, where an electron
    // can cross multiple voxel boundaries before a hard event occurs"; reading R28) -------------------------
    // The step length d = min[d_maxs, d_maxe, d_range, d_event] is planned from the voxel the step starts in and is NOT
    // limited by the voxel.  The two legs of the random hinge are walked voxel by voxel; every segment loses energy
    // through the range table of its own material (deposited in its own voxel), uses up the sampled number of mean free
    // paths -ln u at rho_i Sigma_max,i(T_start) (Sigma_max is a running maximum, so the value at the step's start energy
    // is a majorant for the whole step in every material: the thinning stays exact without gDPM's cross-section scaling)
    // and adds K1_i(T_mid) rho_i l_i to the scattering power travelled (R8b carries the difference to what the hinge
    // sampled for).  A segment ends the step early where the mean free paths run out (hard-event candidate) or the range
    // does (end of track).
    void electron_multi_voxel(Particle p) {
        Stream s = stream(p);
        const Params& P = c.p;
        const bool primary = probe && p.trk_lo == 0 && p.trk_hi == 0;
        double path = 0, nstep = 0, q_used = 0, q_act = 0, ms_carry = 0;
        auto finish = [&](int reason) {
            if (!primary) return;
            for (int a = 0; a < 3; ++a) { probe[2 + a] = p.x[a]; probe[5 + a] = p.d[a]; }
            probe[8] = path; probe[9] = nstep; probe[10] = p.E; probe[11] = reason; probe[14] = q_used; probe[15] = q_act;
        };
        for (;;) {
            if (p.E <= P.e_cut) {
                finish(0);
                deposit(p.v, p.E, true);
                if (p.q > 0) {  // annihilation at rest (R9)
                    s.next();
                    Particle g = p; g.q = 0; g.blk0 = 0; g.E = MEC2; g.trk_lo = s.w[0]; g.trk_hi = s.w[1];
                    iso_direction(s.u(2), s.u(3), g.d);
                    s.next();
                    Particle g2 = g; g2.trk_lo = s.w[0]; g2.trk_hi = s.w[1];
                    for (int a = 0; a < 3; ++a) g2.d[a] = -g.d[a];
                    push(g); push(g2);
                }
                return;
            }
            const int v0 = vidx(p.v);
            const MatTables& t0 = c.tab[c.mat[v0]];
            const double rho0 = c.rho[v0], T0 = p.E;
            const double R0 = lerp_tab(c, t0.R, T0), L0 = lerp_tab(c, t0.L, T0), Smax0 = lerp_tab(c, t0.S_max, T0);
            s.next();
            double tau = (P.flags & F_NO_HARD) ? 1e300 : -std::log(s.u(0));  // mean free paths to the next hard-event candidate
            double d = std::min(std::min(P.d_maxs, P.f_maxe * T0 / (rho0 * L0)), std::min(std::max(R0, 0.0) / rho0, tau / (rho0 * Smax0)));
            if (!(d > 0.0)) {  // no residual range left above the cut-off (rounding): the track ends here
                deposit(p.v, p.E - P.e_cut, false);
                p.E = P.e_cut;
                continue;
            }
            st.n_estep += 1; nstep += 1;
            const double Tmid = inv_range(c, t0.R, R0 - 0.5 * rho0 * d);
            const double k1rho0 = (P.flags & F_NO_MS) ? 0.0 : lerp_tab(c, t0.K1, Tmid) * rho0;
            double q_step = 0;  // scattering power travelled in this step
            enum { NONE = 0, HARD = 1, STOP = 2, OUT = 3 };
            double Smax_ev = Smax0;
            // walk `len` cm along the direction, voxel by voxel
            auto walk = [&](double len) -> int {
                while (len > 0.0) {
                    const int vi = vidx(p.v);
                    const MatTables& ti = c.tab[c.mat[vi]];
                    const double rho = c.rho[vi];
                    int ax;
                    const double tf = face_dist(p.x, p.d, p.v, ax);
                    const double Smax_i = lerp_tab(c, ti.S_max, T0), Ri = lerp_tab(c, ti.R, p.E);
                    double seg = std::min(len, tf);
                    int ev = NONE;
                    const double l_tau = tau / (rho * Smax_i), l_range = std::max(Ri, 0.0) / rho;
                    // "<=" to rounding (of the whole step: what is left in the second leg is a difference): a step planned up
                    // to the event or to the end of the range ends exactly there
                    if (l_tau <= seg + 1e-9 * d) { seg = std::min(seg, l_tau); ev = HARD; Smax_ev = Smax_i; }
                    if (l_range <= seg + 1e-9 * d) { seg = std::min(seg, l_range); ev = STOP; }
                    for (int a = 0; a < 3; ++a) p.x[a] += seg * p.d[a];
                    const double T1 = ev == STOP ? P.e_cut : inv_range(c, ti.R, Ri - rho * seg);
                    deposit(p.v, p.E - T1, false);
                    p.E = T1;
                    tau -= rho * Smax_i * seg;
                    if (!(P.flags & F_NO_MS)) q_step += lerp_tab(c, ti.K1, Tmid) * rho * seg;
                    st.path_e += seg; path += seg;
                    len -= seg;
                    if (ev != NONE) return ev;
                    if (seg >= tf) {  // on the face: enter the neighbour
                        const int dir = p.d[ax] > 0 ? 1 : -1;
                        p.v[ax] += dir;
                        p.x[ax] = c.org[ax] + (p.v[ax] + (dir > 0 ? 0 : 1)) * c.h[ax];
                        if (!inside(p.v)) return OUT;
                    }
                }
                return NONE;
            };
            const double xi = s.u(1);
            int ev = walk(xi * d);
            if (ev == NONE && (P.flags & F_NO_MS)) ev = walk((1.0 - xi) * d);
            else if (ev == NONE) {
                // the hinge (R7 / R27) with the bookkeeping of R8b
                double tq = k1rho0 * d + (c.ms_carry ? ms_carry : 0.0), tu = std::max(tq, 0.0);
                ms_carry = tq - tu;
                q_used += tu;
                if (P.flags & F_MS_GS) {
                    if (tu < GS_T_MIN) { if (c.ms_carry) ms_carry += tu; q_used -= tu; }
                    else rotate_dir(p.d, 1.0 - gs_sample_omu(g_gs, tu, std::exp(lerp_tab(c, t0.lnA, Tmid)), s.w[2], s.w[3]), 2.0 * PI * s.u(3));
                } else {
                    double am = 1.0 - std::exp(-tu);
                    if (am > 0.0) rotate_dir(p.d, 1.0 - sample_ms_omu(am, s.u(2)), 2.0 * PI * s.u(3));
                }
                ms_carry -= k1rho0 * d;  // what was sampled for beyond the carry; the path travelled is added below
                ev = walk((1.0 - xi) * d);
            }
            ms_carry += q_step; q_act += q_step;
            if (ev == OUT) { finish(1); escape(p.E + (p.q > 0 ? 2.0 * MEC2 : 0.0)); return; }
            if (ev == HARD && p.E > P.e_cut) hard_candidate(p, s, Smax_ev, primary, path);
        }
    }

    void electron(Particle p) {
        if (c.p.flags & F_MULTI_VOXEL) { electron_multi_voxel(p); return; }
        Stream s = stream(p);
        const Params& P = c.p;
        const bool primary = probe && p.trk_lo == 0 && p.trk_hi == 0;  // per-history probe of the primary track (pins)
        double path = 0, nstep = 0, q_used = 0, q_act = 0;
        double ms_carry = 0;  // R8b: scattering power (K1 rho x path) travelled but not yet sampled (< 0: sampled ahead)
        auto finish = [&](int reason) {
            if (!primary) return;
            for (int a = 0; a < 3; ++a) { probe[2 + a] = p.x[a]; probe[5 + a] = p.d[a]; }
            probe[8] = path; probe[9] = nstep; probe[10] = p.E; probe[11] = reason; probe[14] = q_used; probe[15] = q_act;
        };
        for (;;) {
            if (p.E <= P.e_cut) {
                finish(0);
                deposit(p.v, p.E, true);
                if (p.q > 0) {  // annihilation at rest: two back-to-back 0.511 MeV photons (R9)
                    s.next();
                    Particle g = p; g.q = 0; g.blk0 = 0; g.E = MEC2; g.trk_lo = s.w[0]; g.trk_hi = s.w[1];
                    iso_direction(s.u(2), s.u(3), g.d);
                    s.next();
                    Particle g2 = g; g2.trk_lo = s.w[0]; g2.trk_hi = s.w[1];
                    for (int a = 0; a < 3; ++a) g2.d[a] = -g.d[a];
                    if (primary) { for (int a = 0; a < 3; ++a) probe[16 + a] = g.d[a] + g2.d[a]; probe[19] = g.d[2]; }
                    push(g); push(g2);
                }
                return;
            }
            int vi = vidx(p.v);
            const MatTables& t = c.tab[c.mat[vi]];
            double rho = c.rho[vi];
            double T = p.E;
            double R0 = lerp_tab(c, t.R, T), L0 = lerp_tab(c, t.L, T), Smax = lerp_tab(c, t.S_max, T);
            s.next();
            int ax;
            double d_vox = face_dist(p.x, p.d, p.v, ax);
            double d_maxe = P.f_maxe * T / (rho * L0);
            double d_range = std::max(R0, 0.0) / rho;
            double d_event = (P.flags & F_NO_HARD) ? 1e300 : -std::log(s.u(0)) / (rho * Smax);
            double d = d_vox; int lim = 0;
            if (P.d_maxs < d) { d = P.d_maxs; lim = 1; }
            if (d_maxe < d) { d = d_maxe; lim = 2; }
            if (d_range < d) { d = d_range; lim = 3; }
            if (d_event < d) { d = d_event; lim = 4; }
            (&st.lim_vox)[lim] += 1; st.n_estep += 1; nstep += 1;
            // random hinge (R7, R8)
            double xi = s.u(1);
            for (int a = 0; a < 3; ++a) p.x[a] += xi * d * p.d[a];
            double k1rho = 0;
            if (!(P.flags & F_NO_MS)) {
                double Tmid = inv_range(c, t.R, R0 - 0.5 * rho * d);
                k1rho = lerp_tab(c, t.K1, Tmid) * rho;
                // R8b: the angle is sampled for the planned path d plus the path travelled but not yet sampled for
                // (the previous steps ended early at a face or ran on to it); never a negative path
                double tq = k1rho * d + (c.ms_carry ? ms_carry : 0.0);
                double tu = std::max(tq, 0.0);
                ms_carry = tq - tu;
                q_used += tu;
                if (P.flags & F_MS_GS) {
                    // Goudsmit-Saunderson angle (R27): scattering power below the table is not sampled
                    // now but carried (R8b)
                    if (tu < GS_T_MIN) {
                        if (c.ms_carry) ms_carry += tu;
                        q_used -= tu;
                    } else {
                        double A = std::exp(lerp_tab(c, t.lnA, Tmid));
                        rotate_dir(p.d, 1.0 - gs_sample_omu(g_gs, tu, A, s.w[2], s.w[3]), 2.0 * PI * s.u(3));
                    }
                } else {
                    double am = 1.0 - std::exp(-tu);
                    if (am > 0.0) rotate_dir(p.d, 1.0 - sample_ms_omu(am, s.u(2)), 2.0 * PI * s.u(3));
                }
            }
            double rest = (1.0 - xi) * d;
            double tf = face_dist(p.x, p.d, p.v, ax);
            // R8: a step cut short by the voxel (d = d_vox) is meant to end on the face; after the deflection the
            // face may be a little further than planned, so the second leg may run on to it, by at most
            // hinge_overrun of its planned length and never beyond the non-geometric limits.  Without this,
            // about half of the voxel-limited steps stop a hair short of the face and need a tiny extra step.
            double d_lim = std::min(std::min(P.d_maxs, d_maxe), std::min(d_range, d_event));
            double reach = std::min((1.0 + c.hinge_overrun) * rest, d_lim - xi * d);
            bool cross = tf <= std::max(reach, rest);
            double legB = cross ? tf : rest;
            for (int a = 0; a < 3; ++a) p.x[a] += legB * p.d[a];
            double d_act = xi * d + legB;
            st.path_e += d_act; path += d_act;
            ms_carry += k1rho * (d_act - d); q_act += k1rho * d_act;
            // a range-limited step that stayed in the voxel ends exactly at the cut-off
            double T1 = (lim == 3 && !cross) ? P.e_cut : inv_range(c, t.R, R0 - rho * d_act);
            deposit(p.v, T - T1, false);
            p.E = T1;
            if (cross) {
                int dir = p.d[ax] > 0 ? 1 : -1;
                p.v[ax] += dir;
                p.x[ax] = c.org[ax] + (p.v[ax] + (dir > 0 ? 0 : 1)) * c.h[ax];  // snap to the face
                if (!inside(p.v)) { finish(1); escape(p.E + (p.q > 0 ? 2.0 * MEC2 : 0.0)); return; }
                continue;
            }
            if (lim != 4 || p.E <= P.e_cut) continue;
            hard_candidate(p, s, Smax, primary, path);
        }
    }

    // Hard event candidate at the end of a step ("Woodcock again"; R6): thinning against the majorant the
    // distance was sampled with, then Moller (R10) or bremsstrahlung (R11) in the material where the particle stands.
    void hard_candidate(Particle& p, Stream& s, double Smax, bool primary, double path) {
        const Params& P = c.p;
        int vi = vidx(p.v);
        const MatTables& t = c.tab[c.mat[vi]];
        s.next();
        double r = s.u(0) * Smax;
        double SM = lerp_tab(c, t.S_M, p.E), SH = lerp_tab(c, t.S_hard, p.E);
        if (r >= SH) { if (primary && probe[0] == 0) probe[13] += 1; return; }  // fictitious
        uint32_t id_lo = s.w[1], id_hi = s.w[2];
        double phi = 2.0 * PI * s.u(3);
        double T0 = p.E;
        if (primary && probe[0] == 0) { probe[0] = r < SM ? 1 : 2; probe[1] = T0; probe[12] = path; }
        if (r < SM) {  // Moller (R10)
            st.n_moller += 1;
            double W = sample_moller(s, T0, P.e_cut) * T0, c1, c2;
            moller_angles(T0, W, c1, c2);
            Particle e = p; e.q = -1; e.blk0 = 0; e.E = W; e.trk_lo = id_lo; e.trk_hi = id_hi;
            rotate_dir(e.d, c2, phi + PI);
            rotate_dir(p.d, c1, phi);
            p.E = T0 - W;
            push(e);
        } else {  // bremsstrahlung (R11)
            st.n_brems += 1;
            double kk = sample_brems(s, c.mats[c.mat[vi]], T0, P.g_cut);
            Particle g = p; g.q = 0; g.blk0 = 0; g.E = kk; g.trk_lo = id_lo; g.trk_hi = id_hi;
            rotate_dir(g.d, std::cos(MEC2 / (T0 + MEC2)), phi);
            if (primary && probe[21] == 0) {  // instrumentation only: emission angle of the primary's first bremsstrahlung photon
                probe[20] = p.d[0] * g.d[0] + p.d[1] * g.d[1] + p.d[2] * g.d[2]; probe[21] = T0;
            }
            p.E = T0 - kk;
            push(g);
        }
    }

    // History h of a particle-list source ("phase-space file"; R13b): the listed particle is the
    // primary, track id (0,0), stream from block 0; outside the phantom it counts as escaped.
    void history_listed(uint32_t h, int q, const double x[3], const double d[3], double E) {
        hist = h; led_src = led_dep = led_esc = 0; first_vox = -1; first_chan = -1;
        st.n_hist += 1;
        Particle p; p.q = q; p.E = E; p.trk_lo = 0; p.trk_hi = 0; p.blk0 = 0;
        for (int a = 0; a < 3; ++a) { p.x[a] = x[a]; p.d[a] = d[a]; }
        double e0 = E + (q > 0 ? 2.0 * MEC2 : 0.0);
        led_src += e0; st.e_src += e0;
        if (!locate(p.x, p.v)) escape(e0);
        else {
            stack.clear();
            stack.push_back(p);
            while (!stack.empty()) {
                Particle t = stack.back(); stack.pop_back();
                if (t.q == 0) photon(t); else electron(t);
            }
        }
        double rel = std::fabs(led_dep + led_esc - led_src) / led_src;
        if (rel > st.max_ledger_rel) st.max_ledger_rel = rel;
    }

    void history(uint32_t h) {
        hist = h; led_src = led_dep = led_esc = 0; first_vox = -1; first_chan = -1;
        Particle p;
        st.n_hist += 1;
        if (source(p)) {
            stack.clear();
            stack.push_back(p);
            while (!stack.empty()) {
                Particle q = stack.back(); stack.pop_back();
                if (q.q == 0) photon(q); else electron(q);
            }
        }
        double rel = std::fabs(led_dep + led_esc - led_src) / led_src;
        if (rel > st.max_ledger_rel) st.max_ledger_rel = rel;
    }
};

// ------------------------------------------------------------------------------------------------
// fp32 arithmetic-contract path for the attenuation-only mode (R20).  IEEE single
// +,-,*,/,sqrt and explicit fmaf only; compiled with -ffp-contract=off.
static inline float c_ln(float x) {
    uint32_t b; std::memcpy(&b, &x, 4);
    int e = (int)(b >> 23) - 127;
    b = (b & 0x007fffffu) | 0x3f800000u;
    float m; std::memcpy(&m, &b, 4);
    if (m > 1.41421354f) { m = m * 0.5f; e += 1; }
    float f = m - 1.0f;
    float s = f / (2.0f + f);
    float z = s * s;
    float p = fmaf(z, 0.0909090936f, 0.111111112f);
    p = fmaf(z, p, 0.142857149f);
    p = fmaf(z, p, 0.2f);
    p = fmaf(z, p, 0.333333343f);
    p = p * z;
    float t = s + s;
    float r = fmaf(t, p, t);
    return fmaf((float)e, 0.693147182f, r);
}
static inline float c_u(uint32_t w) { return ((float)(w >> 9) + 0.5f) * 1.1920928955078125e-07f; }

struct TabF {  // fp32 photon tables handed in by the caller (see orc_run_atten)
    int N, n_mat; float lnE0, inv_dln;
    const float *mu_maj, *mu_tot, *mu_C, *mu_pp;  // per material arrays are [n_mat][N]
};
static inline void c_lookup(const TabF& t, float lnE, int& i, float& f) {
    float x = (lnE - t.lnE0) * t.inv_dln;
    i = (int)x; if (i > t.N - 2) i = t.N - 2; if (i < 0) i = 0;
    f = x - (float)i;
}
static inline float c_lerp(const float* a, int i, float f) { return fmaf(f, a[i + 1] - a[i], a[i]); }

// ------------------------------------------------------------------------------------------------
extern "C" {

struct orc_material { int32_t n_elem; const int32_t* Z; const float* A; const float* w; float I_eV; float rho_nominal; };
struct orc_params { float e_cut_MeV, g_cut_MeV, e_max_MeV; int32_t n_grid; float d_maxs_cm, f_maxe; uint32_t flags; };
struct orc_beam { int32_t particle, shape; float entry_cm[3], axis[3], ssd_cm, field_cm[2]; int32_t n_nodes; const float* E_nodes_MeV; const float* pdf_nodes; };

static Material to_material(const orc_material& m) {
    Material M;
    for (int i = 0; i < m.n_elem; ++i) { M.Z.push_back(m.Z[i]); M.A.push_back(m.A[i]); M.w.push_back(m.w[i]); }
    M.I_eV = m.I_eV; M.rho_nominal = m.rho_nominal; M.derive();
    return M;
}
static void to_beam(const orc_beam* b, Beam& B) {
    B.particle = b->particle; B.shape = b->shape; B.ssd = b->ssd_cm;
    for (int a = 0; a < 3; ++a) { B.entry[a] = b->entry_cm[a]; B.axis[a] = b->axis[a]; }
    B.field[0] = b->field_cm[0]; B.field[1] = b->field_cm[1];
    for (int i = 0; i < b->n_nodes; ++i) { B.E.push_back(b->E_nodes_MeV[i]); B.pdf.push_back(b->pdf_nodes[i]); }
    B.cdf.assign(B.E.size(), 0.0);
    double tot = 0;
    for (size_t j = 0; j + 1 < B.E.size(); ++j) { tot += 0.5 * (B.pdf[j] + B.pdf[j + 1]) * (B.E[j + 1] - B.E[j]); B.cdf[j + 1] = tot; }
    for (auto& v : B.cdf) v = tot > 0 ? v / tot : 0.0;
}

void orc_philox(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { philox4x32_10(ctr, key, out); }
float orc_contract_ln(float x) { return c_ln(x); }

int orc_create(const uint8_t* mat, const float* rho, const int32_t* dims, const float* vox, const float* org, Ctx** out) {
    if (!mat || !rho || !out || dims[0] <= 0 || dims[1] <= 0 || dims[2] <= 0) return 1;
    for (int a = 0; a < 3; ++a) if (!(vox[a] > 0)) return 1;
    Ctx* c = new Ctx();
    c->nx = dims[0]; c->ny = dims[1]; c->nz = dims[2];
    size_t n = (size_t)c->nx * c->ny * c->nz;
    for (int a = 0; a < 3; ++a) { c->h[a] = vox[a]; c->org[a] = org[a]; }
    c->mat.assign(mat, mat + n);
    c->rho.assign(rho, rho + n);
    c->rho_f.assign(rho, rho + n);
    for (size_t i = 0; i < n; ++i) if (!(rho[i] > 0)) { delete c; return 1; }
    *out = c;
    return 0;
}
void orc_destroy(Ctx* c) { delete c; }

int orc_build_tables(Ctx* c, const orc_material* mats, int n_mats, const orc_params* p) {
    if (!c || !mats || n_mats <= 0 || !p || p->n_grid < 8) return 1;
    for (uint8_t m : c->mat) if (m >= n_mats) return 1;
    c->p = Params{p->e_cut_MeV, p->g_cut_MeV, p->e_max_MeV, p->n_grid, p->d_maxs_cm, p->f_maxe, p->flags};
    c->mats.clear();
    for (int i = 0; i < n_mats; ++i) c->mats.push_back(to_material(mats[i]));
    if (!make_grid(*c)) return 1;
    build_tables(*c);
    return 0;
}
void orc_set_flags(Ctx* c, uint32_t flags) { c->p.flags = flags; if (flags & F_MS_GS) g_gs.build(); }

// grid description: out[0]=lnE0, out[1]=dln, out[2]=N, out[3]=k_cut
void orc_grid(const Ctx* c, double* out) { out[0] = c->lnE0; out[1] = c->dln; out[2] = c->N; out[3] = c->k_cut; }
// table export (fp64), which: 0 mu_tot 1 mu_C 2 mu_pp 3 R 4 L 5 S_hard 6 S_M 7 S_max 8 K1 ; m=-1,which=9: mu_maj
int orc_table(const Ctx* c, int m, int which, double* out) {
    if (!c->have_tables) return 2;
    const std::vector<double>* v = nullptr;
    if (which == 9) v = &c->mu_maj;
    else {
        if (m < 0 || m >= (int)c->tab.size()) return 1;
        const MatTables& t = c->tab[m];
        const std::vector<double>* all[11] = {&t.mu_tot, &t.mu_C, &t.mu_pp, &t.R, &t.L, &t.S_hard, &t.S_M, &t.S_max, &t.K1, nullptr, &t.lnA};
        if (which < 0 || which > 10 || which == 9) return 1;
        v = all[which];
    }
    std::memcpy(out, v->data(), sizeof(double) * v->size());
    return 0;
}
double orc_material_scalar(const Ctx* c, int m, int which) {
    const Material& M = c->mats[m];
    return which == 0 ? M.ne : which == 1 ? M.ZA : which == 2 ? M.Cbr : M.Lscr;
}
// closed-form evaluation at one energy (for the pins): which: 0 sigma_KN(k=E/mc2) [cm2/electron], 1 mu_C/rho,
// 2 mu_pe/rho, 3 mu_pp/rho, 4 L_col(E, arg), 5 L_rad(E, kmax=arg), 6 ne*sigma_Moller(E, e_cut=arg),
// 7 Sigma_br(E, g_cut=arg), 8 K1, 9 density effect, 10 k dSigma/dk (E, k=arg), 11 moller dsigma/deps (E, eps=arg) per electron
double orc_eval(const Ctx* c, int m, int which, double E, double arg) {
    const Material& M = c->mats[m];
    switch (which) {
        case 0: return sigma_kn(E / MEC2);
        case 1: return mu_compton(M, E);
        case 2: return mu_pe(M, E);
        case 3: return mu_pp(M, E);
        case 4: return L_col(M, E, arg);
        case 5: return L_rad(M, E, arg);
        case 6: return M.ne * moller_sigma(E, arg);
        case 7: return brems_sigma(M, E, arg);
        case 8: return K1(M, E);
        case 12: return S_el(M, E);
        case 9: return density_effect(M, E);
        case 10: return brems_kdsdk(M, E, arg);
        case 11: return moller_dsde(E, arg);
    }
    return -1;
}
double orc_sigma_pp_atom(int Z, double k) { return sigma_pp(Z, k) / (ALPHA * RE * RE * Z * Z); }
double orc_lerp(const Ctx* c, int m, int which, double E) {
    const MatTables& t = c->tab[m < 0 ? 0 : m];
    const std::vector<double>* all[10] = {&t.mu_tot, &t.mu_C, &t.mu_pp, &t.R, &t.L, &t.S_hard, &t.S_M, &t.S_max, &t.K1, &c->mu_maj};
    return lerp_tab(*c, *all[which], E);
}
double orc_inv_range(const Ctx* c, int m, double Rt) { return inv_range(*c, c->tab[m].R, Rt); }

// Run histories [h0, h1) of a job of n_total histories split into n_batches contiguous batches
// (batch of history h = floor(h*B/N), R18).  edep: [n_batches][nvox] fp64, accumulated (+=), MeV.
int orc_run(Ctx* c, const orc_beam* b, uint64_t h0, uint64_t h1, uint64_t n_total, uint64_t seed, int n_batches,
            double* edep, double* stats_out, int32_t* first_vox_out, int32_t* first_chan_out) {
    if (!c || !c->have_tables) return 2;
    if (!b || n_batches < 1 || n_total >= (1ull << 32) || h1 > n_total || h0 > h1 || b->n_nodes < 1) return 1;
    Beam B; to_beam(b, B);
    for (double E : B.E) if (E > c->p.e_max) return 3;
    Stats st; std::memset(&st, 0, sizeof st);
    Run run(*c, B, seed, st);
    size_t nvox = c->mat.size();
    for (uint64_t h = h0; h < h1; ++h) {
        uint64_t bi = (h * (uint64_t)n_batches) / n_total;
        run.edep = edep + bi * nvox;
        run.history((uint32_t)h);
        if (first_vox_out) first_vox_out[h - h0] = run.first_vox;
        if (first_chan_out) first_chan_out[h - h0] = run.first_chan;
    }
    if (stats_out) std::memcpy(stats_out, &st, sizeof st);
    return 0;
}
int orc_n_stats() { return N_STATS; }

// Particle-list source: histories [h0, h1) are particles[h0 .. h1) (records of 7 floats + int32, as mc_particle).
struct orc_particle { float x, y, z, u, v, w, E; int32_t particle; };
int orc_run_particles(Ctx* c, const orc_particle* particles, uint64_t h0, uint64_t h1, uint64_t n_total, uint64_t seed,
                      int n_batches, double* edep, double* stats_out) {
    if (!c || !c->have_tables) return 2;
    if (!particles || n_batches < 1 || n_total >= (1ull << 32) || h1 > n_total || h0 > h1) return 1;
    Beam B; B.particle = 0; B.shape = 0;
    Stats st; std::memset(&st, 0, sizeof st);
    Run run(*c, B, seed, st);
    size_t nvox = c->mat.size();
    for (uint64_t h = h0; h < h1; ++h) {
        const orc_particle& q = particles[h];
        if (q.E > c->p.e_max) return 3;
        uint64_t bi = (h * (uint64_t)n_batches) / n_total;
        run.edep = edep + bi * nvox;
        double x[3] = {q.x, q.y, q.z}, d[3] = {q.u, q.v, q.w};
        run.history_listed((uint32_t)h, q.particle == 0 ? 0 : (q.particle > 0 ? 1 : -1), x, d, q.E);
    }
    if (stats_out) std::memcpy(stats_out, &st, sizeof st);
    return 0;
}

// Dose and batch uncertainty (R17, R18): D_b = E_b/(rho V N_b); mean over batches; standard error.
int orc_finalize(const Ctx* c, const double* edep, uint64_t n_total, int n_batches, double* dose, double* sigma) {
    size_t nvox = c->mat.size();
    double V = c->h[0] * c->h[1] * c->h[2];
    std::vector<double> nb(n_batches);
    for (int b = 0; b < n_batches; ++b) {
        // histories with floor(h*B/N) == b : h in [ceil(b*N/B), ceil((b+1)*N/B))
        uint64_t lo = ((uint64_t)b * n_total + n_batches - 1) / n_batches, hi = ((uint64_t)(b + 1) * n_total + n_batches - 1) / n_batches;
        nb[b] = (double)(hi - lo);
    }
    for (size_t v = 0; v < nvox; ++v) {
        double mass = c->rho[v] * V, mean = 0;
        for (int b = 0; b < n_batches; ++b) mean += edep[(size_t)b * nvox + v] / (mass * nb[b]);
        mean /= n_batches;
        double ss = 0;
        for (int b = 0; b < n_batches; ++b) { double d = edep[(size_t)b * nvox + v] / (mass * nb[b]) - mean; ss += d * d; }
        dose[v] = mean;
        sigma[v] = n_batches > 1 ? std::sqrt(ss / ((double)n_batches * (n_batches - 1))) : 0.0;
    }
    return 0;
}

// ---- samplers exposed one interaction at a time, for the chi-square / moment / conservation pins ----
// Each entry draws from history stream h = i (track 0) and calls the SAME sampler function the transport code calls.
static Stream pin_stream(uint64_t i, uint64_t seed) {
    Stream s; s.h = (uint32_t)i; s.seed_lo = (uint32_t)seed; s.seed_hi = (uint32_t)(seed >> 32); s.trk_lo = s.trk_hi = 0; s.block = 0;
    return s;
}
// KN: out[4*i+0]=eps, [1]=cos(theta_photon), [2]=dot(electron dir, incoming), [3]=|p_in - p_g - p_e|/p_in residual
void orc_sample_kn(double E, uint64_t n, uint64_t seed, double* out) {
    for (uint64_t i = 0; i < n; ++i) {
        Stream s = pin_stream(i, seed);
        KNSample kn = sample_kn(s, E);
        s.next();
        const double d0[3] = {0.6, 0.0, 0.8};
        double d1[3] = {0.6, 0.0, 0.8}, ed[3];
        compton_kinematics(E, kn, 2.0 * PI * s.u(2), d1, ed);
        double E1 = kn.eps * E, Te = E - E1, pe = std::sqrt(Te * (Te + 2.0 * MEC2));
        double res = 0, dot = 0;
        for (int a = 0; a < 3; ++a) { double r = E * d0[a] - E1 * d1[a] - pe * ed[a]; res += r * r; dot += ed[a] * d0[a]; }
        out[4 * i] = kn.eps; out[4 * i + 1] = d0[0] * d1[0] + d0[1] * d1[1] + d0[2] * d1[2]; out[4 * i + 2] = dot; out[4 * i + 3] = std::sqrt(res) / E;
    }
}
// Moller: out[3*i+0]=eps, [1]=cos theta primary, [2]=cos theta delta
void orc_sample_moller(double T0, double e_cut, uint64_t n, uint64_t seed, double* out) {
    for (uint64_t i = 0; i < n; ++i) {
        Stream s = pin_stream(i, seed);
        double eps = sample_moller(s, T0, e_cut);
        out[3 * i] = eps;
        moller_angles(T0, eps * T0, out[3 * i + 1], out[3 * i + 2]);
    }
}
// brems photon energy k for material m of ctx
void orc_sample_brems(const Ctx* c, int m, double T0, uint64_t n, uint64_t seed, double* out) {
    for (uint64_t i = 0; i < n; ++i) {
        Stream s = pin_stream(i, seed);
        out[i] = sample_brems(s, c->mats[m], T0, c->p.g_cut);
    }
}
// MS polar cosine for a given a = 1 - exp(-K1 rho d) (word 2 of the step block, as in transport)
// ---- Goudsmit-Saunderson entries for the pins (the functions transport calls) ----------------------------------------
void orc_gs_dims(int* out) { out[0] = GS_NT; out[1] = GS_NA; out[2] = GS_NQ; }
void orc_gs_nodes(double* t, double* A, double* r) {
    for (int i = 0; i < GS_NT; ++i) t[i] = gs_t_node(i);
    for (int j = 0; j < GS_NA; ++j) A[j] = gs_A_node(j);
    for (int k = 0; k < GS_NQ; ++k) r[k] = gs_r_node(k);
}
void orc_gs_table(double* out) { g_gs.build(); std::memcpy(out, g_gs.y.data(), sizeof(double) * g_gs.y.size()); }
void orc_gs_moments(double A, int lmax, double* out) { std::vector<double> g = gs_moments(A, lmax); std::memcpy(out, g.data(), sizeof(double) * (lmax + 1)); }
double orc_gs_G1(double A) { return gs_G1(A); }
void orc_gs_cdf(double lambda, double A, const double* x, int n, double* out) {
    std::vector<double> S = gs_cdf(lambda, A, std::vector<double>(x, x + n));
    std::memcpy(out, S.data(), sizeof(double) * n);
}
// n samples of mu = cos(theta) for scattering power t and screening A, words 2 and 3 of block 0 of stream (seed, history i)
void orc_gs_sample(double t, double A, uint64_t n, uint64_t seed, double* out) {
    g_gs.build();
    for (uint64_t i = 0; i < n; ++i) {
        Stream s = pin_stream(i, seed);
        s.next();
        out[i] = 1.0 - gs_sample_omu(g_gs, t, A, s.w[2], s.w[3]);
    }
}

void orc_sample_ms(double am, uint64_t n, uint64_t seed, double* out) {
    for (uint64_t i = 0; i < n; ++i) {
        Stream s = pin_stream(i, seed);
        s.next();
        out[i] = 1.0 - sample_ms_omu(am, s.u(2));
    }
}
// annihilation photon direction (words 2, 3 of the block, as in transport): out[3*i..] = unit vector
void orc_sample_iso(uint64_t n, uint64_t seed, double* out) {
    for (uint64_t i = 0; i < n; ++i) {
        Stream s = pin_stream(i, seed);
        s.next();
        iso_direction(s.u(2), s.u(3), out + 3 * i);
    }
}
// the direction rotation of the transport code (R25), one call
void orc_rotate(const double* d, double mu, double phi, double* out) {
    out[0] = d[0]; out[1] = d[1]; out[2] = d[2];
    rotate_dir(out, mu, phi);
}
// run-time switches of the readings R8 / R8b (defaults: hinge_overrun 0.25, ms_carry 1)
int orc_set_option(Ctx* c, const char* name, double value) {
    if (!c || !name) return 1;
    std::string n(name);
    if (n == "hinge_overrun") { if (!(value >= 0.0 && value <= 1.0)) return 1; c->hinge_overrun = value; }
    else if (n == "ms_carry") c->ms_carry = value != 0.0;
    else return 1;
    return 0;
}
int orc_n_probe() { return N_PROBE; }
// Per-history probe of the PRIMARY electron / positron track, for the transport-level pins (hard-event rate, MS in
// transport, hinge rule).  Runs histories [h0, h1) like orc_run (dose goes to a scratch grid) and writes N_PROBE doubles
// per history: [0] first real hard event (0 none, 1 Moller, 2 bremsstrahlung), [1] kinetic energy at that event,
// [2..4] final position, [5..7] final direction, [8] path length, [9] steps, [10] final kinetic energy,
// [11] end (0 absorbed at the cut-off, 1 left the phantom), [12] path length at the first hard event,
// [13] fictitious candidates before it, [14] sum of the scattering powers the MS angles were sampled for,
// [15] sum of K1 rho x path actually travelled, [16..18] sum of the two annihilation-photon directions (positron),
// [19] z direction cosine of the first annihilation photon, [20] cosine between the primary's direction and its first
// bremsstrahlung photon's, [21] the primary's kinetic energy at that emission (0 = no bremsstrahlung event).
int orc_run_probe(Ctx* c, const orc_beam* b, uint64_t h0, uint64_t h1, uint64_t n_total, uint64_t seed, double* out, double* stats_out) {
    if (!c || !c->have_tables) return 2;
    if (!b || !out || n_total >= (1ull << 32) || h1 > n_total || h0 > h1 || b->n_nodes < 1) return 1;
    Beam B; to_beam(b, B);
    for (double E : B.E) if (E > c->p.e_max) return 3;
    Stats st; std::memset(&st, 0, sizeof st);
    Run run(*c, B, seed, st);
    std::vector<double> scratch(c->mat.size(), 0.0);
    run.edep = scratch.data();
    for (uint64_t h = h0; h < h1; ++h) {
        run.probe = out + (h - h0) * N_PROBE;
        for (int k = 0; k < N_PROBE; ++k) run.probe[k] = 0.0;
        run.history((uint32_t)h);
    }
    if (stats_out) std::memcpy(stats_out, &st, sizeof st);
    return 0;
}
// primaries only: energy, position, direction (7 doubles per history) — source pins
void orc_sample_source(Ctx* c, const orc_beam* b, uint64_t n, uint64_t seed, double* out) {
    Beam B; to_beam(b, B);
    Stats st; std::memset(&st, 0, sizeof st);
    Run run(*c, B, seed, st);
    std::vector<double> dummy(c->mat.size(), 0.0);
    run.edep = dummy.data();
    for (uint64_t i = 0; i < n; ++i) {
        run.hist = (uint32_t)i;
        Particle p; run.source(p);
        out[7 * i] = p.E;
        for (int a = 0; a < 3; ++a) { out[7 * i + 1 + a] = p.x[a]; out[7 * i + 4 + a] = p.d[a]; }
    }
}

// ---- attenuation-only mode, fp32 arithmetic contract (R20) ------------------------------------
// Photon primaries only; for each history the voxel index (-1 = escaped) and channel (0 Compton,
// 1 pair, 2 photoelectric, 255 none) of the first real interaction.  The fp32 photon tables are
// INPUTS (any builder's): mu_maj[N] (1/cm), mu_tot/mu_C/mu_pp [n_mat][N] (cm^2/g).
int orc_run_atten(const Ctx* c, const orc_beam* b, uint64_t n, uint64_t seed, int N, int n_mat, float lnE0, float inv_dln,
                  const float* mu_maj, const float* mu_tot, const float* mu_C, const float* mu_pp,
                  int32_t* voxel_out, uint8_t* channel_out, uint32_t* flights_out) {
    if (!c || !b || b->particle != 0) return 1;
    TabF t{N, n_mat, lnE0, inv_dln, mu_maj, mu_tot, mu_C, mu_pp};
    int nn = b->n_nodes;
    // spectrum cdf: fp64 running trapezoid sum in node order, normalised, rounded to fp32
    std::vector<float> cdf(nn, 0.0f);
    {
        std::vector<double> cd(nn, 0.0); double tot = 0;
        for (int j = 0; j + 1 < nn; ++j) { tot += 0.5 * ((double)b->pdf_nodes[j] + (double)b->pdf_nodes[j + 1]) * ((double)b->E_nodes_MeV[j + 1] - (double)b->E_nodes_MeV[j]); cd[j + 1] = tot; }
        for (int j = 0; j < nn; ++j) cdf[j] = tot > 0 ? (float)(cd[j] / tot) : 0.0f;
    }
    const float org[3] = {(float)c->org[0], (float)c->org[1], (float)c->org[2]};
    const float ih[3] = {1.0f / (float)c->h[0], 1.0f / (float)c->h[1], 1.0f / (float)c->h[2]};
    const int nd[3] = {c->nx, c->ny, c->nz};
    for (uint64_t h = 0; h < n; ++h) {
        Stream s; s.h = (uint32_t)h; s.seed_lo = (uint32_t)seed; s.seed_hi = (uint32_t)(seed >> 32); s.trk_lo = s.trk_hi = 0; s.block = 0;
        s.next();
        float E;
        if (nn == 1) E = b->E_nodes_MeV[0];
        else {
            float u0 = c_u(s.w[0]), u1 = c_u(s.w[1]);
            int j = 0;
            while (j + 2 < nn && u0 >= cdf[j + 1]) ++j;
            float p0 = b->pdf_nodes[j], p1 = b->pdf_nodes[j + 1];
            float q = fmaf(u1, p1 * p1 - p0 * p0, p0 * p0);
            float tt = (u1 * (p0 + p1)) / (p0 + std::sqrt(q));
            E = fmaf(tt, b->E_nodes_MeV[j + 1] - b->E_nodes_MeV[j], b->E_nodes_MeV[j]);
        }
        float x[3], d[3];
        if (b->shape == 0) { for (int a = 0; a < 3; ++a) { x[a] = b->entry_cm[a]; d[a] = b->axis[a]; } }
        else {
            float fx = (c_u(s.w[2]) - 0.5f) * b->field_cm[0], fy = (c_u(s.w[3]) - 0.5f) * b->field_cm[1];
            x[0] = b->entry_cm[0] + fx; x[1] = b->entry_cm[1] + fy; x[2] = b->entry_cm[2];
            float n2 = fmaf(fx, fx, fmaf(fy, fy, b->ssd_cm * b->ssd_cm));
            float nr = std::sqrt(n2);
            d[0] = fx / nr; d[1] = fy / nr; d[2] = b->ssd_cm / nr;
        }
        int vox = -1; uint8_t chan = 255; uint32_t nfl = 0;
        int v[3]; bool in = true;
        for (int a = 0; a < 3; ++a) { float f = (x[a] - org[a]) * ih[a]; if (f < 0.0f || f >= (float)nd[a]) in = false; }
        if (in && E >= (float)c->p.g_cut) {
            int i; float f;
            c_lookup(t, c_ln(E), i, f);
            float maj = c_lerp(t.mu_maj, i, f);
            bool done = false;
            while (!done) {
                s.next();
                for (int k = 0; k < 2 && !done; ++k) {
                    float sl = (-c_ln(c_u(s.w[2 * k]))) / maj;
                    ++nfl;
                    bool inside = true;
                    for (int a = 0; a < 3; ++a) {
                        x[a] = fmaf(sl, d[a], x[a]);
                        float fa = (x[a] - org[a]) * ih[a];
                        if (fa < 0.0f || fa >= (float)nd[a]) inside = false; else v[a] = (int)fa;
                    }
                    if (!inside) { done = true; break; }
                    int vi = v[0] + nd[0] * (v[1] + nd[1] * v[2]);
                    int m = c->mat[vi]; float rho = c->rho_f[vi];
                    float r = c_u(s.w[2 * k + 1]) * maj;
                    float mu = rho * c_lerp(t.mu_tot + (size_t)m * N, i, f);
                    if (r <= mu) {
                        float vc = c_lerp(t.mu_C + (size_t)m * N, i, f), vp = c_lerp(t.mu_pp + (size_t)m * N, i, f);
                        chan = r < rho * vc ? 0 : (r < rho * (vc + vp) ? 1 : 2);
                        vox = vi; done = true;
                    }
                }
            }
        }
        voxel_out[h] = vox; channel_out[h] = chan; if (flights_out) flights_out[h] = nfl;
    }
    return 0;
}

}  // extern "C"
