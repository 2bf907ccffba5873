// ORACLE -- TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, single-threaded, double-precision CPU implementation of the
// ARCHER-EPID hot path as scoped by SURVEY.md section 8(c): coupled photon /
// electron Monte Carlo transport source -> air -> voxel phantom -> air -> EPID
// slab stack, plus the k(t,s) response post-pass (PAPER.md:88-94, 104, 108-110,
// 114-123, 147-153; BASELINE.json:north_star).  It follows the algorithm of
// SURVEY.md 8(c) step by step in that order and notation; there is no blocking,
// fusion or reordering.  It shares no code with the CUDA library
// (paper_2510_24154_b200/csrc) -- only the generated input arrays (gen/).
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
// reference legs may load it.  The product path never does.
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): P1 Philox known answers, P2 source
// chi-square, P3 Beer-Lambert transmission, P4 Woodcock == surface tracking and
// analytic first-collision depth, P5 Klein-Nishina moments and chi-square, P6
// PE-only pencil-beam deposit, P7 CSDA path length, P8 Highland width, P9 energy
// ledger, P10 symmetry, P11 Table 1 / Eq. 1 / slab thickness.
// parity unpinned: physical realism of the parametric tables and agreement with
// measurement (no data in the container; SURVEY.md 8(c) last pin row).
//
// Units: cm, MeV, g/cm^3.  World frame = phantom frame.  Beam frame: source at
// the origin, axes (u, v, w) = rows of beam_axes, beam along +w.

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <limits>
#include <string>
#include <utility>
#include <vector>

namespace {

constexpr double MEC2 = 0.51099895;       // SURVEY 8(c) constants
constexpr double RHO_AIR = 1.205e-3;      // world filler, material 0 (SURVEY 8(c) "Geometry")
constexpr int MAT_AIR = 0;
constexpr double WORLD_HALF = 100.0;      // |u|,|v| <= 100 cm
constexpr double WORLD_WMIN = -1.0;       // -1 <= w <= EPID bottom
constexpr double PI = 3.14159265358979323846;
constexpr double INF = std::numeric_limits<double>::infinity();

enum Region { AIR = 0, PHANTOM = 1, EPID = 2 };
enum PType { PHOTON = 0, ELECTRON = 1, POSITRON = 2 };

// ---------------------------------------------------------------- Philox4x32-10
// Counter-based RNG (Salmon et al. 2011): 10 rounds, multipliers 0xD2511F53 /
// 0xCD9E8D57, Weyl key increments 0x9E3779B9 / 0xBB67AE85.  Pin P1.
inline void philox_round(uint32_t c[4], const uint32_t k[2]) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * c[0];
    const uint64_t p1 = (uint64_t)0xCD9E8D57u * c[2];
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c[1] ^ k[0];
    const uint32_t n1 = (uint32_t)p1;
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c[3] ^ k[1];
    const uint32_t n3 = (uint32_t)p0;
    c[0] = n0; c[1] = n1; c[2] = n2; c[3] = n3;
}
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c[4] = {ctr[0], ctr[1], ctr[2], ctr[3]};
    uint32_t k[2] = {key[0], key[1]};
    for (int r = 0; r < 10; ++r) {
        if (r > 0) { k[0] += 0x9E3779B9u; k[1] += 0xBB67AE85u; }
        philox_round(c, k);
    }
    for (int i = 0; i < 4; ++i) out[i] = c[i];
}

// Per-particle stream, reading A1: key = seed, counter = (h_lo, h_hi, particle_id, block).
struct Rng {
    uint32_t key[2], ctr[4], buf[4];
    int pos;
    void init(uint64_t seed, uint64_t h, uint32_t pid) {
        key[0] = (uint32_t)seed; key[1] = (uint32_t)(seed >> 32);
        ctr[0] = (uint32_t)h; ctr[1] = (uint32_t)(h >> 32); ctr[2] = pid; ctr[3] = 0;
        pos = 4;
    }
    double u() {                                   // uniform in (0,1): (r + 0.5) 2^-32
        if (pos == 4) { philox4x32_10(ctr, key, buf); ctr[3]++; pos = 0; }
        return ((double)buf[pos++] + 0.5) * (1.0 / 4294967296.0);
    }
    uint32_t child_id(int sibling) const {         // A1: schedule-independent secondary id
        return ctr[2] * 0x9E3779B1u + ctr[3] * 2u + (uint32_t)sibling + 1u;
    }
    void skip_block() { pos = 4; }                 // after a creation event: next draw opens a new block
};

struct Vec3 { double x, y, z; };
inline Vec3 operator+(Vec3 a, Vec3 b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
inline Vec3 operator-(Vec3 a, Vec3 b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
inline Vec3 operator*(double s, Vec3 a) { return {s * a.x, s * a.y, s * a.z}; }
inline double dot(Vec3 a, Vec3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
inline Vec3 normalize(Vec3 a) { double n = std::sqrt(dot(a, a)); return {a.x / n, a.y / n, a.z / n}; }
inline double comp(const Vec3& a, int i) { return i == 0 ? a.x : (i == 1 ? a.y : a.z); }
inline void setcomp(Vec3& a, int i, double v) { if (i == 0) a.x = v; else if (i == 1) a.y = v; else a.z = v; }

// Rotate unit vector d by polar angle (cos_t, sin_t) and azimuth phi about itself.
Vec3 rotate(Vec3 d, double cos_t, double sin_t, double phi) {
    const double cp = std::cos(phi), sp = std::sin(phi);
    Vec3 n;
    const double a2 = 1.0 - d.z * d.z;
    if (a2 > 1e-12) {
        const double a = std::sqrt(a2);
        n.x = d.x * cos_t + sin_t * (d.x * d.z * cp - d.y * sp) / a;
        n.y = d.y * cos_t + sin_t * (d.y * d.z * cp + d.x * sp) / a;
        n.z = d.z * cos_t - a * sin_t * cp;
    } else {
        const double sg = d.z >= 0 ? 1.0 : -1.0;
        n.x = sin_t * cp; n.y = sin_t * sp; n.z = sg * cos_t;
    }
    return normalize(n);
}

struct Particle {
    int type;            // PType
    double E;            // photon energy or kinetic energy [MeV]
    Vec3 pos, dir;       // world frame in AIR / PHANTOM; beam frame (u, v, w) in EPID
    int region;
    int iv[3];           // voxel index (PHANTOM)
    int layer;           // EPID layer index
    Rng rng;
    bool uncollided;     // primary photon that has not interacted yet
};

struct Ctx {
    std::string err;
    // materials (as handed over by gen/)
    int n_mat = 0, n_E = 0, n_T = 0;
    std::vector<double> Eg, lnEg, muC, muPE, muPP, Tg, lnTg, S, X0;
    // phantom
    int n[3] = {0, 0, 0};
    double h[3] = {0, 0, 0}, org[3] = {0, 0, 0};
    std::vector<float> rho;
    std::vector<uint8_t> mat;
    std::vector<double> mu_maj;            // node values of the majorant [n_E]
    // EPID
    int n_layers = 0, nu = 0, nv = 0;
    double sid = 0, pitch = 0;
    std::vector<double> lt, lrho, ztop;    // thickness, density, top w of each layer (+ bottom)
    std::vector<int> lmat, lscored;
    // source
    Vec3 src{0, 0, 0}, au{1, 0, 0}, av{0, 1, 0}, aw{0, 0, 1};
    int n_bins = 0, fu = 0, fv = 0;
    double fpitch = 0, fdist = 0;
    std::vector<double> Eedges, cdfE, cdfF;
    std::vector<float> fluence;
    // physics
    int mode = 1;
    double photon_cut = 0.010, electron_cut = 0.200, f_E = 0.10, s_max = 1.0;
    std::vector<double> ne;                // electrons per gram [n_mat] (mode 2: Class II, reading A31)
    int tracking = 0;                      // 0 Woodcock, 1 exact voxel-by-voxel surface tracking
    int eq1_printed = 0;                   // 1: use Eq. 1 exactly as printed
    // fixed-primary override (pencil beams for pins)
    bool fixed = false; int fx_type = 0; double fx_E = 0; Vec3 fx_pos{0, 0, 0}, fx_dir{0, 0, 1};
    // tallies
    int rebin = 1;
    bool want_phantom_sq = true;
    std::vector<double> ep_sum, ep_sq, rb_sum, rb_sq, ph_sum, ph_sq, unc;
    double ledger[8] = {0};
    uint64_t counters[16] = {0};
    double aux[4] = {0};                   // 0: electron path length [cm], 1: sum rho*s [g/cm^2], 2 / 3: Moller events in the phantom / elsewhere
    int fc_bins = 0; double fc_w0 = 0, fc_dw = 0; std::vector<double> fc_hist;
    // per-history scratch
    std::vector<std::pair<int64_t, double>> hpix, hvox;
    std::vector<Particle> stack;
    // Phase Space 3 (reading A30): every particle arriving at the EPID top plane from the air,
    // 8 doubles per record = {type, E, u, v, du, dv, dw (beam frame), history index}
    bool ps3_on = false; uint64_t cur_h = 0; std::vector<double> ps3;
    // coarse phantom tally (history-by-history, like the re-binned image): blocks of prb[0] x prb[1] x prb[2] voxels
    int prb[3] = {1, 1, 1}; bool prb_on = false; std::vector<double> pc_sum, pc_sq;
    // second moments of the ledger channels over histories (sum over histories of (per-history amount)^2)
    double ledger_sq[8] = {0}, ledger_prev[8] = {0};
    // event log for the pins (tests/test_oracle_pins_events.py): 16 doubles per record, see log_event
    size_t log_cap = 0; std::vector<double> evlog;
    // collimation stage (readings A35-A37): Phase Space 1 records on the plane
    // w = w_ps1 (beam frame) and tungsten slabs with per-row openings between it and the Phase Space 2 plane w = w_ps2
    struct Slab { double w0, w1; int axis; double row0, pitch; std::vector<double> lo, hi; };
    std::vector<Slab> slabs; int col_mat = 0; double col_rho = 0, w_ps2 = 0; bool have_col = false;
    std::vector<float> ps1; size_t n_ps1 = 0; double w_ps1 = 0;
    double head[4] = {0};                  // PS2 particles, their energy, energy absorbed in the stage, interactions in the stage
    bool ps2_on = false; std::vector<double> ps2;   // Phase Space 2 dump: {E, u, v, du, dv, dw, history, uncollided}
};

// ---------------------------------------------------------------- tables
// Interpolation rule: linear in (ln E, ln mu) for Compton /
// photoelectric / stopping power; linear in ln E on mu for pair (zero below threshold).
struct Cell { int i; double t; };
Cell locate(const std::vector<double>& g, const std::vector<double>& lng, double x) {
    const int n = (int)g.size();
    if (x <= g[0]) return {0, 0.0};
    if (x >= g[n - 1]) return {n - 2, 1.0};
    int i = (int)(std::upper_bound(g.begin(), g.end(), x) - g.begin()) - 1;
    if (i > n - 2) i = n - 2;
    const double t = (std::log(x) - lng[i]) / (lng[i + 1] - lng[i]);
    return {i, t};
}
inline double lerp_loglog(double a, double b, double t) {
    if (a > 0 && b > 0) return std::exp(std::log(a) + t * (std::log(b) - std::log(a)));
    return a + t * (b - a);
}
void mu_partial(const Ctx& c, int m, double E, double out[3]) {   // [pe, compton, pair] cm^2/g
    const Cell k = locate(c.Eg, c.lnEg, E);
    const size_t o = (size_t)m * c.n_E + k.i;
    out[0] = lerp_loglog(c.muPE[o], c.muPE[o + 1], k.t);
    out[1] = lerp_loglog(c.muC[o], c.muC[o + 1], k.t);
    // pair: linear in ln E on mu; impossible at or below the threshold 2 m_e c^2 (reading A34: the linear
    // interpolant across the grid cell that straddles the threshold would otherwise be > 0 just below it)
    out[2] = E > 2.0 * MEC2 ? c.muPP[o] + k.t * (c.muPP[o + 1] - c.muPP[o]) : 0.0;
}
double mu_tot(const Ctx& c, int m, double E) {
    double p[3]; mu_partial(c, m, E, p); return p[0] + p[1] + p[2];
}
double stop_pow(const Ctx& c, int m, double T) {
    const Cell k = locate(c.Tg, c.lnTg, T);
    const size_t o = (size_t)m * c.n_T + k.i;
    return lerp_loglog(c.S[o], c.S[o + 1], k.t);
}
// Majorant (reading A7, corrected in DESIGN.md): node values max_m rho_max,m * mu_tot,m(E_j),
// interpolated LINEARLY in ln E (an upper bound of every material's interpolant) times (1 + 1e-6).
double majorant(const Ctx& c, double E) {
    const Cell k = locate(c.Eg, c.lnEg, E);
    return (c.mu_maj[k.i] + k.t * (c.mu_maj[k.i + 1] - c.mu_maj[k.i])) * (1.0 + 1e-6);
}
void build_majorant(Ctx& c) {
    std::vector<double> rmax(c.n_mat, 0.0);
    const size_t nv = (size_t)c.n[0] * c.n[1] * c.n[2];
    for (size_t i = 0; i < nv; ++i) rmax[c.mat[i]] = std::max(rmax[c.mat[i]], (double)c.rho[i]);
    c.mu_maj.assign(c.n_E, 0.0);
    for (int j = 0; j < c.n_E; ++j)
        for (int m = 0; m < c.n_mat; ++m) {
            if (rmax[m] <= 0) continue;
            const size_t o = (size_t)m * c.n_E + j;
            c.mu_maj[j] = std::max(c.mu_maj[j], rmax[m] * (c.muPE[o] + c.muC[o] + c.muPP[o]));
        }
}

// ---------------------------------------------------------------- frames
inline Vec3 to_beam(const Ctx& c, Vec3 p) { Vec3 r = p - c.src; return {dot(c.au, r), dot(c.av, r), dot(c.aw, r)}; }
inline Vec3 dir_to_beam(const Ctx& c, Vec3 d) { return {dot(c.au, d), dot(c.av, d), dot(c.aw, d)}; }
inline Vec3 dir_to_world(const Ctx& c, Vec3 b) { return b.x * c.au + b.y * c.av + b.z * c.aw; }
inline Vec3 to_world(const Ctx& c, Vec3 b) { return c.src + dir_to_world(c, b); }

// ---------------------------------------------------------------- tallies
inline size_t vox_index(const Ctx& c, const int iv[3]) { return ((size_t)iv[2] * c.n[1] + iv[1]) * c.n[0] + iv[0]; }
void dep_phantom(Ctx& c, const int iv[3], double e) {
    c.ledger[1] += e; c.hvox.emplace_back((int64_t)vox_index(c, iv), e);
}
void dep_epid(Ctx& c, int layer, double u, double v, double e) {
    // Pixel (iu, iv) = floor((u + nu p/2)/p), floor((v + nv p/2)/p)   (SURVEY 8(c) "Geometry")
    if (c.lscored[layer]) {
        const double fu = std::floor((u + 0.5 * c.nu * c.pitch) / c.pitch);
        const double fv = std::floor((v + 0.5 * c.nv * c.pitch) / c.pitch);
        if (fu >= 0 && fu < c.nu && fv >= 0 && fv < c.nv) {
            c.ledger[2] += e; c.hpix.emplace_back((int64_t)fv * c.nu + (int64_t)fu, e);
            return;
        }
    }
    c.ledger[3] += e;
}
inline void dep_air(Ctx& c, double e) { c.ledger[4] += e; }
inline void escape(Ctx& c, double e) { c.ledger[5] += e; }

void deposit_here(Ctx& c, const Particle& p, double e) {          // deposit at the particle's position
    if (p.region == AIR) dep_air(c, e);
    else if (p.region == PHANTOM) dep_phantom(c, p.iv, e);
    else dep_epid(c, p.layer, p.pos.x, p.pos.y, e);
}

void merge_history(std::vector<std::pair<int64_t, double>>& h) {
    std::sort(h.begin(), h.end(), [](const auto& a, const auto& b) { return a.first < b.first; });
    size_t o = 0;
    for (size_t i = 0; i < h.size(); ++i) {
        if (o > 0 && h[o - 1].first == h[i].first) h[o - 1].second += h[i].second;
        else h[o++] = h[i];
    }
    h.resize(o);
}
// History-by-history estimator: add x and x^2 per touched bin at history end.
void flush_history(Ctx& c) {
    if (!c.hpix.empty()) {
        merge_history(c.hpix);
        for (auto& kv : c.hpix) { c.ep_sum[kv.first] += kv.second; c.ep_sq[kv.first] += kv.second * kv.second; }
        if (c.rebin > 1) {
            const int r = c.rebin, cu = c.nu / r;
            for (auto& kv : c.hpix) {
                const int64_t iu = kv.first % c.nu, iv = kv.first / c.nu;
                kv.first = (iv / r) * cu + (iu / r);
            }
            merge_history(c.hpix);
        }
        for (auto& kv : c.hpix) { c.rb_sum[kv.first] += kv.second; c.rb_sq[kv.first] += kv.second * kv.second; }
        c.hpix.clear();
    }
    if (!c.hvox.empty()) {
        merge_history(c.hvox);
        for (auto& kv : c.hvox) {
            c.ph_sum[kv.first] += kv.second;
            if (c.want_phantom_sq) c.ph_sq[kv.first] += kv.second * kv.second;
        }
        if (c.prb_on) {
            const int64_t nx = c.n[0], ny = c.n[1], cx = c.n[0] / c.prb[0], cy = c.n[1] / c.prb[1];
            for (auto& kv : c.hvox) {
                const int64_t ix = kv.first % nx, iy = (kv.first / nx) % ny, iz = kv.first / (nx * ny);
                kv.first = ((iz / c.prb[2]) * cy + iy / c.prb[1]) * cx + ix / c.prb[0];
            }
            merge_history(c.hvox);
            for (auto& kv : c.hvox) { c.pc_sum[kv.first] += kv.second; c.pc_sq[kv.first] += kv.second * kv.second; }
        }
        c.hvox.clear();
    }
    for (int k = 0; k < 8; ++k) {
        const double d = c.ledger[k] - c.ledger_prev[k];
        c.ledger_sq[k] += d * d; c.ledger_prev[k] = c.ledger[k];
    }
}

// ---------------------------------------------------------------- geometry helpers
// Ray / phantom-AABB entry distance for a particle in AIR (slab method).  Returns INF when the
// box is not hit ahead; 0 when the particle sits on the surface heading inward.  *axis gets the entry axis.
double aabb_entry(const Ctx& c, Vec3 p, Vec3 d, int* axis) {
    double tn = -INF, tf = INF; int ax = -1;
    for (int a = 0; a < 3; ++a) {
        const double lo = c.org[a], hi = c.org[a] + c.n[a] * c.h[a];
        const double pa = comp(p, a), da = comp(d, a);
        if (da == 0.0) { if (pa < lo || pa >= hi) return INF; continue; }
        double t1 = (lo - pa) / da, t2 = (hi - pa) / da;
        if (t1 > t2) std::swap(t1, t2);
        if (t1 > tn) { tn = t1; ax = a; }
        if (t2 < tf) tf = t2;
    }
    if (!(tf > 0.0) || tn > tf || tn >= tf) return INF;
    *axis = ax;
    return tn > 0.0 ? tn : 0.0;
}
// Exit distance from inside the AABB along d; *axis = crossed axis.
double aabb_exit(const Ctx& c, Vec3 p, Vec3 d, int* axis) {
    double tf = INF; int ax = 0;
    for (int a = 0; a < 3; ++a) {
        const double lo = c.org[a], hi = c.org[a] + c.n[a] * c.h[a];
        const double pa = comp(p, a), da = comp(d, a);
        double t = INF;
        if (da > 0) t = (hi - pa) / da; else if (da < 0) t = (lo - pa) / da;
        if (t < tf) { tf = t; ax = a; }
    }
    *axis = ax;
    return tf > 0 ? tf : 0.0;
}
inline bool inside_grid(const Ctx& c, Vec3 p) {
    for (int a = 0; a < 3; ++a) {
        const double g = comp(p, a);
        if (g < c.org[a] || g >= c.org[a] + c.n[a] * c.h[a]) return false;
    }
    return true;
}
inline void locate_voxel(const Ctx& c, Vec3 p, int iv[3]) {
    for (int a = 0; a < 3; ++a) {
        int i = (int)std::floor((comp(p, a) - c.org[a]) / c.h[a]);
        iv[a] = std::min(std::max(i, 0), c.n[a] - 1);
    }
}
// Distance along beam-frame ray (pb, db) to the world box sides |u| = |v| = 100 and w = -1.
double world_exit_air(Vec3 pb, Vec3 db) {
    double t = INF;
    if (db.x > 0) t = std::min(t, (WORLD_HALF - pb.x) / db.x); else if (db.x < 0) t = std::min(t, (-WORLD_HALF - pb.x) / db.x);
    if (db.y > 0) t = std::min(t, (WORLD_HALF - pb.y) / db.y); else if (db.y < 0) t = std::min(t, (-WORLD_HALF - pb.y) / db.y);
    if (db.z < 0) t = std::min(t, (WORLD_WMIN - pb.z) / db.z);
    return t > 0 ? t : 0.0;
}
double world_exit_lateral(Vec3 pb, Vec3 db) {
    double t = INF;
    if (db.x > 0) t = std::min(t, (WORLD_HALF - pb.x) / db.x); else if (db.x < 0) t = std::min(t, (-WORLD_HALF - pb.x) / db.x);
    if (db.y > 0) t = std::min(t, (WORLD_HALF - pb.y) / db.y); else if (db.y < 0) t = std::min(t, (-WORLD_HALF - pb.y) / db.y);
    return t > 0 ? t : 0.0;
}

// Boundaries seen from AIR (AIR case).
struct AirHit { double t; int kind; int axis; };   // kind 0 phantom, 1 EPID top, 2 world exit
AirHit air_boundary(const Ctx& c, const Particle& p) {
    int ax = -1;
    const double tp = aabb_entry(c, p.pos, p.dir, &ax);
    const Vec3 pb = to_beam(c, p.pos), db = dir_to_beam(c, p.dir);
    double te = INF;
    if (db.z > 0) { te = (c.sid - pb.z) / db.z; if (te < 0) te = 0; }
    const double tw = world_exit_air(pb, db);
    AirHit h{tp, 0, ax};
    if (te < h.t) h = {te, 1, -1};
    if (tw < h.t) h = {tw, 2, -1};
    return h;
}
void enter_phantom(const Ctx& c, Particle& p, double t, int axis) {
    p.pos = p.pos + t * p.dir;
    const double lo = c.org[axis], hi = c.org[axis] + c.n[axis] * c.h[axis];
    const bool from_lo = comp(p.dir, axis) > 0;
    setcomp(p.pos, axis, from_lo ? lo : hi);          // snap exactly onto the entry face
    locate_voxel(c, p.pos, p.iv);
    p.iv[axis] = from_lo ? 0 : c.n[axis] - 1;
    p.region = PHANTOM;
}
void enter_epid(Ctx& c, Particle& p, double t) {
    p.pos = p.pos + t * p.dir;
    Vec3 pb = to_beam(c, p.pos); pb.z = c.sid;
    p.dir = dir_to_beam(c, p.dir); p.pos = pb; p.region = EPID; p.layer = 0;
    if (c.ps3_on) { const double rec[8] = {(double)p.type, p.E, pb.x, pb.y, p.dir.x, p.dir.y, p.dir.z, (double)c.cur_h}; c.ps3.insert(c.ps3.end(), rec, rec + 8); }
    if (p.type == PHOTON && p.uncollided) {                        // pin P3 / P10 tally
        c.counters[10]++;
        const double fu = std::floor((pb.x + 0.5 * c.nu * c.pitch) / c.pitch);
        const double fv = std::floor((pb.y + 0.5 * c.nv * c.pitch) / c.pitch);
        if (fu >= 0 && fu < c.nu && fv >= 0 && fv < c.nv) c.unc[(size_t)fv * c.nu + (size_t)fu] += 1.0;
    }
}
void epid_to_air(const Ctx& c, Particle& p) {                       // leaving through the top face
    Vec3 pb = p.pos; pb.z = c.sid;
    p.pos = to_world(c, pb); p.dir = dir_to_world(c, p.dir); p.region = AIR;
}

// ---------------------------------------------------------------- event log (pins only; off unless orc_set_event_log)
// record = {kind (1 interaction, 2 birth), history, particle id, particle type, its energy when the event starts,
//           its direction xyz, [8] channel 0 PE / 1 Compton / 2 pair (kind 1) or child type (kind 2),
//           [9] material (kind 1) or child energy (kind 2), child direction xyz, sibling, region, child id}
void log_event(Ctx& c, int kind, const Particle& p, double a8, double a9, Vec3 cd, int sibling, uint32_t child_pid) {
    if (c.evlog.size() / 16 >= c.log_cap) return;
    const double rec[16] = {(double)kind, (double)c.cur_h, (double)p.rng.ctr[2], (double)p.type, p.E, p.dir.x, p.dir.y, p.dir.z,
                            a8, a9, cd.x, cd.y, cd.z, (double)sibling, (double)p.region, (double)child_pid};
    c.evlog.insert(c.evlog.end(), rec, rec + 16);
}

// ---------------------------------------------------------------- secondaries
Particle make_child(Ctx& c, const Particle& parent, int sibling, int type, double E, Vec3 dir, uint64_t seed) {
    Particle s = parent;
    s.type = type; s.E = E; s.dir = dir; s.uncollided = false;
    const uint64_t h = ((uint64_t)parent.rng.ctr[1] << 32) | parent.rng.ctr[0];
    s.rng.init(seed, h, parent.rng.child_id(sibling));
    if (c.log_cap) log_event(c, 2, parent, (double)type, E, dir, sibling, s.rng.ctr[2]);
    return s;
}
struct Run { uint64_t seed; };

// Two 0.511 MeV photons, isotropic, back to back (reading A11).  Directions are drawn from `p`'s stream.
void annihilate(Ctx& c, Particle& p, const Run& r) {
    const double ct = 2.0 * p.rng.u() - 1.0, phi = 2.0 * PI * p.rng.u();
    const double st = std::sqrt(std::max(0.0, 1.0 - ct * ct));
    Vec3 d{st * std::cos(phi), st * std::sin(phi), ct};
    c.stack.push_back(make_child(c, p, 0, PHOTON, MEC2, d, r.seed));
    c.stack.push_back(make_child(c, p, 1, PHOTON, MEC2, -1.0 * d, r.seed));
    c.counters[9] += 2;
    p.rng.skip_block();
}

// Klein-Nishina sampling: epsilon-mixture rejection on
// f(eps) ~ (1/eps + eps)(1 - eps sin^2 / (1 + eps^2)), eps in [1/(1+2k), 1].  Pin P5.
void sample_kn(Rng& rng, double E, double* eps_out, double* cos_out, uint64_t* iters) {
    const double k = E / MEC2, e0 = 1.0 / (1.0 + 2.0 * k);
    const double a1 = std::log(1.0 / e0), a2 = 0.5 * (1.0 - e0 * e0);
    for (;;) {
        if (iters) (*iters)++;
        const double x1 = rng.u(), x2 = rng.u(), x3 = rng.u();
        double eps;
        if (x1 * (a1 + a2) < a1) eps = std::exp(-x2 * a1);
        else eps = std::sqrt(e0 * e0 + (1.0 - e0 * e0) * x2);
        const double t = (1.0 - eps) / (k * eps);            // 1 - cos(theta)
        const double sin2 = t * (2.0 - t);
        const double g = 1.0 - eps * sin2 / (1.0 + eps * eps);
        if (g >= x3) { *eps_out = eps; *cos_out = 1.0 - t; return; }
    }
}

// Compton event: photon (E, d) -> photon (E1, d1) + electron (T = E - E1, de), phi uniform,
// electron direction from momentum conservation, de ~ E d - E1 d1.
void compton_scatter(Rng& rng, double E, Vec3 d, double* E1, Vec3* d1, double* T, Vec3* de, uint64_t* iters) {
    double eps, ct;
    sample_kn(rng, E, &eps, &ct, iters);
    const double phi = 2.0 * PI * rng.u();
    *E1 = eps * E; *T = E - *E1;
    *d1 = rotate(d, ct, std::sqrt(std::max(0.0, 1.0 - ct * ct)), phi);
    *de = normalize(E * d - (*E1) * (*d1));
}

// Interaction of a photon in material m.  Returns false when the photon is gone.
bool interact(Ctx& c, Particle& p, int m, const Run& r) {
    p.uncollided = false;
    double mu[3]; mu_partial(c, m, p.E, mu);
    const double x = p.rng.u() * (mu[0] + mu[1] + mu[2]);
    if (x < mu[0]) {                                               // photoelectric
        c.counters[3]++;
        if (c.log_cap) log_event(c, 1, p, 0.0, (double)m, Vec3{0, 0, 0}, 0, 0);
        if (c.mode == 0) deposit_here(c, p, p.E);
        else { c.stack.push_back(make_child(c, p, 0, ELECTRON, p.E, p.dir, r.seed)); c.counters[9]++; p.rng.skip_block(); }
        return false;
    }
    if (x < mu[0] + mu[1]) {                                       // Compton
        c.counters[4]++;
        if (c.log_cap) log_event(c, 1, p, 1.0, (double)m, Vec3{0, 0, 0}, 0, 0);
        double E1, T; Vec3 d1, de;
        compton_scatter(p.rng, p.E, p.dir, &E1, &d1, &T, &de, &c.counters[12]);
        if (c.mode == 0) deposit_here(c, p, T);
        else {
            c.stack.push_back(make_child(c, p, 0, ELECTRON, T, de, r.seed)); c.counters[9]++;
            p.rng.skip_block();
        }
        p.E = E1; p.dir = d1;
        return true;
    }
    c.counters[5]++;                                               // pair
    if (c.log_cap) log_event(c, 1, p, 2.0, (double)m, Vec3{0, 0, 0}, 0, 0);
    const double Ttot = p.E - 2.0 * MEC2;
    const double Tm = p.rng.u() * Ttot, Tp = Ttot - Tm;          // uniform split (reading A10)
    if (c.mode == 0) {
        deposit_here(c, p, Ttot);
        annihilate(c, p, r);                                       // 2 m_e c^2 re-emitted at the interaction point (A11)
    } else {
        c.stack.push_back(make_child(c, p, 0, ELECTRON, Tm, p.dir, r.seed));
        c.stack.push_back(make_child(c, p, 1, POSITRON, Tp, p.dir, r.seed));
        c.counters[9] += 2;
        p.rng.skip_block();
    }
    return false;
}

void score_first_collision(Ctx& c, const Particle& p) {            // pin P4 histogram along w
    if (!p.uncollided || c.fc_bins <= 0) return;
    const double w = (p.region == EPID) ? p.pos.z : to_beam(c, p.pos).z;
    const int b = (int)std::floor((w - c.fc_w0) / c.fc_dw);
    if (b >= 0 && b < c.fc_bins) c.fc_hist[b] += 1.0;
}

// ---------------------------------------------------------------- photon transport
void photon_exit_phantom(const Ctx& c, Particle& p, Vec3 from) {
    int ax; const double t = aabb_exit(c, from, p.dir, &ax);
    p.pos = from + t * p.dir;
    setcomp(p.pos, ax, comp(p.dir, ax) > 0 ? c.org[ax] + c.n[ax] * c.h[ax] : c.org[ax]);
    p.region = AIR;
}

// Exact voxel-by-voxel surface tracking inside the phantom (used by pin P4 to validate Woodcock).
// Returns true when a collision site was reached (p.pos, p.iv set), false when the photon left the grid.
bool surface_track(Ctx& c, Particle& p) {
    double tau = -std::log(p.rng.u());
    int iv[3]; locate_voxel(c, p.pos, iv);
    for (int a = 0; a < 3; ++a) {                                   // on an upper face heading inward
        const double hi = c.org[a] + c.n[a] * c.h[a];
        if (comp(p.pos, a) >= hi) iv[a] = c.n[a] - 1;
    }
    for (;;) {
        c.counters[0]++;
        double tmin = INF; int ax = 0;
        for (int a = 0; a < 3; ++a) {
            const double da = comp(p.dir, a);
            double t = INF;
            if (da > 0) t = (c.org[a] + (iv[a] + 1) * c.h[a] - comp(p.pos, a)) / da;
            else if (da < 0) t = (c.org[a] + iv[a] * c.h[a] - comp(p.pos, a)) / da;
            if (t < tmin) { tmin = t; ax = a; }
        }
        if (tmin < 0) tmin = 0;
        const size_t vi = vox_index(c, iv);
        const double mu = c.rho[vi] * mu_tot(c, c.mat[vi], p.E);
        if (mu * tmin > tau) {
            p.pos = p.pos + (tau / mu) * p.dir;
            p.iv[0] = iv[0]; p.iv[1] = iv[1]; p.iv[2] = iv[2];
            return true;
        }
        tau -= mu * tmin;
        p.pos = p.pos + tmin * p.dir;
        const bool up = comp(p.dir, ax) > 0;
        setcomp(p.pos, ax, c.org[ax] + (iv[ax] + (up ? 1 : 0)) * c.h[ax]);
        iv[ax] += up ? 1 : -1;
        if (iv[ax] < 0 || iv[ax] >= c.n[ax]) { p.region = AIR; return false; }
    }
}

void transport_photon(Ctx& c, Particle p, const Run& r) {
    for (;;) {
        if (p.E < c.photon_cut) { c.counters[13]++; deposit_here(c, p, p.E); return; }   // PAPER.md:104 (10 keV)
        if (p.region == AIR) {
            const AirHit hb = air_boundary(c, p);
            const double mu = RHO_AIR * mu_tot(c, MAT_AIR, p.E);
            const double s = -std::log(p.rng.u()) / mu;
            c.counters[1]++;
            if (s < hb.t) {
                p.pos = p.pos + s * p.dir;
                score_first_collision(c, p);
                if (!interact(c, p, MAT_AIR, r)) return;
            } else if (hb.kind == 0) enter_phantom(c, p, hb.t, hb.axis);
            else if (hb.kind == 1) enter_epid(c, p, hb.t);
            else { escape(c, p.E); return; }
        } else if (p.region == PHANTOM) {
            if (c.tracking == 1) {
                if (!surface_track(c, p)) continue;
                score_first_collision(c, p);
                const size_t vi = vox_index(c, p.iv);
                if (!interact(c, p, c.mat[vi], r)) return;
                continue;
            }
            // Woodcock (delta) tracking against the majorant
            const double mm = majorant(c, p.E);
            const double s = -std::log(p.rng.u()) / mm;
            c.counters[0]++;
            const Vec3 xn = p.pos + s * p.dir;
            if (!inside_grid(c, xn)) { photon_exit_phantom(c, p, p.pos); continue; }
            p.pos = xn;
            locate_voxel(c, p.pos, p.iv);
            const size_t vi = vox_index(c, p.iv);
            const int m = c.mat[vi];
            if (p.rng.u() * mm < c.rho[vi] * mu_tot(c, m, p.E)) {
                score_first_collision(c, p);
                if (!interact(c, p, m, r)) return;
            }
        } else {                                                    // EPID: surface tracking layer by layer
            const int l = p.layer;
            const double mu = c.lrho[l] * mu_tot(c, c.lmat[l], p.E);
            const double s = -std::log(p.rng.u()) / mu;
            c.counters[2]++;
            double tf = INF;
            if (p.dir.z > 0) tf = (c.ztop[l + 1] - p.pos.z) / p.dir.z;
            else if (p.dir.z < 0) tf = (c.ztop[l] - p.pos.z) / p.dir.z;
            if (tf < 0) tf = 0;
            const double tl = world_exit_lateral(p.pos, p.dir);
            if (s < tf && s < tl) {
                p.pos = p.pos + s * p.dir;
                score_first_collision(c, p);
                if (!interact(c, p, c.lmat[l], r)) return;
            } else if (tl < tf) { escape(c, p.E); return; }
            else {
                p.pos = p.pos + tf * p.dir;
                if (p.dir.z > 0) { p.pos.z = c.ztop[l + 1]; p.layer = l + 1; if (p.layer >= c.n_layers) { escape(c, p.E); return; } }
                else { p.pos.z = c.ztop[l]; p.layer = l - 1; if (p.layer < 0) epid_to_air(c, p); }
            }
        }
    }
}

// ---------------------------------------------------------------- electron / positron
// Highland width for a step of mass thickness rho*s in material m at mid-step kinetic energy Tm.
// ---------------------------------------------------------------- Class II collisions (mode 2; "Class II
// condensed history"; reading A31): discrete Moller events with energy transfer W above Tc = the electron
// cut-off, continuous loss with the restricted stopping power below it.  With eps = W / T, tau = T / m_e c^2,
//   d sigma / d eps = (2 pi r_e^2 m_e c^2 / (beta^2 T)) [1/eps^2 + 1/(1-eps)^2 + (tau/(tau+1))^2 - (2 tau+1)/(tau+1)^2 / (eps (1-eps))]
// per electron, eps in [Tc/T, 1/2] (the faster outgoing electron is the primary); zero for T <= 2 Tc.
constexpr double R_E = 2.8179403262e-13;   // cm
struct MollerXs { double sigma, hard; };    // cross section per electron [cm^2]; int W d sigma [MeV cm^2]
MollerXs moller_xs(double T, double Tc) {
    MollerXs r{0.0, 0.0};
    if (!(T > 2.0 * Tc)) return r;
    const double tau = T / MEC2, b2 = tau * (tau + 2.0) / ((tau + 1.0) * (tau + 1.0));
    const double c1 = (tau / (tau + 1.0)) * (tau / (tau + 1.0)), c2 = (2.0 * tau + 1.0) / ((tau + 1.0) * (tau + 1.0));
    const double a = Tc / T, K = 2.0 * PI * R_E * R_E * MEC2 / (b2 * T);
    // antiderivatives between a and 1/2
    r.sigma = K * (1.0 / a - 1.0 / (1.0 - a) + c1 * (0.5 - a) - c2 * std::log((1.0 - a) / a));
    const double i1 = std::log(0.5 / a);                                              // int eps / eps^2
    const double i2 = (2.0 + std::log(0.5)) - (1.0 / (1.0 - a) + std::log(1.0 - a));   // int eps / (1-eps)^2
    const double i3 = c1 * (0.125 - 0.5 * a * a);                                     // int c1 eps
    const double i4 = c2 * std::log(2.0 * (1.0 - a));                                 // int c2 / (1-eps)
    r.hard = K * T * (i1 + i2 + i3 - i4);
    return r;
}
// eps from the Moller density on [a, 1/2] by rejection from 1/eps^2 (envelope: the bracket times eps^2 without its
// negative term is at most 2 + c1/4)
double sample_moller_eps(Rng& rng, double T, double Tc, uint64_t* trials) {
    const double tau = T / MEC2, a = Tc / T;
    const double c1 = (tau / (tau + 1.0)) * (tau / (tau + 1.0)), c2 = (2.0 * tau + 1.0) / ((tau + 1.0) * (tau + 1.0));
    const double gmax = 2.0 + 0.25 * c1;
    for (;;) {
        const double x1 = rng.u(), x2 = rng.u();
        if (trials) ++*trials;
        const double eps = a / (1.0 - x1 * (1.0 - 2.0 * a));
        const double x = eps / (1.0 - eps);
        const double g = 1.0 + x * x + c1 * eps * eps - c2 * x;
        if (x2 * gmax <= g) return eps;
    }
}
// scattering angles of the two outgoing electrons (energy-momentum conservation, target at rest)
inline double moller_cos(double Tout, double Tin) { return std::sqrt(Tout * (Tin + 2.0 * MEC2) / (Tin * (Tout + 2.0 * MEC2))); }

// Bremsstrahlung (mode 3; reading A32): parametric, complete-screening shape normalised by the radiation length,
//   d Sigma / d k = (1 / (X0 k)) (4/3 - 4/3 y + y^2),  y = k / T,  0 < k <= T      [cm^2/g per MeV]
// so that the total radiative stopping power is T / X0.  Photons above kc (the photon cut-off) are discrete events,
// the loss to photons below kc is continuous.
struct BremsXs { double sigma, soft; };     // Sigma(k > kc) [cm^2/g]; restricted radiative stopping power [MeV cm^2/g]
BremsXs brems_xs(double T, double kc, double X0) {
    BremsXs r{0.0, T / X0};
    if (!(T > kc)) return r;                                         // everything is soft
    const double a = kc / T;
    r.sigma = (4.0 / 3.0 * std::log(1.0 / a) - 4.0 / 3.0 * (1.0 - a) + 0.5 * (1.0 - a * a)) / X0;
    r.soft = T * (4.0 / 3.0 * a - 2.0 / 3.0 * a * a + a * a * a / 3.0) / X0;
    return r;
}
// photon energy from the density above on [kc, T]: rejection from 1/k with (4/3 - 4/3 y + y^2) / (4/3) <= 1
double sample_brems_k(Rng& rng, double T, double kc) {
    for (;;) {
        const double x1 = rng.u(), x2 = rng.u();
        const double k = kc * std::pow(T / kc, x1), y = k / T;
        if (x2 <= 1.0 - y + 0.75 * y * y) return k;
    }
}

double highland_theta0(const Ctx& c, int m, double rho_s, double Tm) {
    const double t = rho_s / c.X0[m];
    if (!(t > 0)) return 0.0;
    const double bpc = Tm * (Tm + 2.0 * MEC2) / (Tm + MEC2);
    return (13.6 / bpc) * std::sqrt(t) * std::max(0.25, 1.0 + 0.038 * std::log(t));
}

void transport_electron(Ctx& c, Particle p, const Run& r) {
    c.counters[14]++;
    for (;;) {
        if (p.E <= c.electron_cut) {                                // PAPER.md:104 (200 keV): local deposit
            deposit_here(c, p, p.E);
            if (p.type == POSITRON) annihilate(c, p, r);
            return;
        }
        double rho; int m; double tb = INF; int kind = -1, axis = -1; AirHit hb{INF, 0, -1};
        if (p.region == AIR) {
            rho = RHO_AIR; m = MAT_AIR; hb = air_boundary(c, p); tb = hb.t;
        } else if (p.region == PHANTOM) {
            const size_t vi = vox_index(c, p.iv); rho = c.rho[vi]; m = c.mat[vi];
            for (int a = 0; a < 3; ++a) {
                const double da = comp(p.dir, a);
                double t = INF;
                if (da > 0) t = (c.org[a] + (p.iv[a] + 1) * c.h[a] - comp(p.pos, a)) / da;
                else if (da < 0) t = (c.org[a] + p.iv[a] * c.h[a] - comp(p.pos, a)) / da;
                if (t < tb) { tb = t; axis = a; }
            }
            if (tb < 0) tb = 0;
        } else {
            const int l = p.layer; rho = c.lrho[l]; m = c.lmat[l];
            double tf = INF;
            if (p.dir.z > 0) tf = (c.ztop[l + 1] - p.pos.z) / p.dir.z;
            else if (p.dir.z < 0) tf = (c.ztop[l] - p.pos.z) / p.dir.z;
            if (tf < 0) tf = 0;
            const double tl = world_exit_lateral(p.pos, p.dir);
            if (tl < tf) { tb = tl; kind = 2; } else { tb = tf; kind = 0; }
        }
        // mode 2: restricted stopping power L = S - n_e int W d sigma and a distance to the next hard (Moller) collision,
        // both from the cross section at the energy the step starts with (reading A31)
        // mode 3 adds bremsstrahlung (reading A32): photons above the photon cut-off are discrete, the rest is continuous loss
        const bool class2 = c.mode >= 2, brems = c.mode == 3;
        auto loss = [&](double T) {
            return stop_pow(c, m, T) - (class2 ? c.ne[m] * moller_xs(T, c.electron_cut).hard : 0.0)
                   + (brems ? brems_xs(T, c.photon_cut, c.X0[m]).soft : 0.0);
        };
        const double S = loss(p.E);
        double s_hard = INF, sig_b = 0.0, sig_all = 0.0;
        if (class2) {
            sig_b = brems ? brems_xs(p.E, c.photon_cut, c.X0[m]).sigma : 0.0;
            sig_all = c.ne[m] * moller_xs(p.E, c.electron_cut).sigma + sig_b;
            const double xh = p.rng.u();                                    // drawn every step, also when no hard collision is possible
            if (sig_all > 0) s_hard = -std::log(xh) / (rho * sig_all);
        }
        double s = std::min(std::min(tb, s_hard), std::min(c.f_E * p.E / (rho * S), c.s_max));
        const bool on_face = (s == tb);
        const bool hard = class2 && !on_face && s == s_hard;
        const double dE = std::min(p.E, rho * s * loss(p.E - 0.5 * rho * s * S));   // midpoint rule
        const double Tmid = p.E - 0.5 * dE;
        const Vec3 mid = p.pos + (0.5 * s) * p.dir;
        p.pos = p.pos + s * p.dir;
        if (p.region == AIR) { dep_air(c, dE); c.counters[7]++; }
        else if (p.region == PHANTOM) { dep_phantom(c, p.iv, dE); c.counters[6]++; }
        else { dep_epid(c, p.layer, mid.x, mid.y, dE); c.counters[8]++; }   // pixel of the step midpoint (reading A24)
        p.E -= dE;
        c.aux[0] += s; c.aux[1] += rho * s;
        // Highland deflection, applied at the end of the step (reading A13).  The face crossing below is
        // decided by the direction the step was taken in; the new direction applies from the next step on.
        double th = 0.0, phi = 0.0;
        const bool deflect = s > 0;
        if (deflect) {
            const double th0 = highland_theta0(c, m, rho * s, Tmid);
            const double xa = p.rng.u(), xb = p.rng.u();
            th = std::min(PI, th0 * std::sqrt(-2.0 * std::log(xa)));
            phi = 2.0 * PI * xb;
        } else c.counters[15]++;
        if (on_face) {
            // the step ended on a face: the particle is now in the neighbouring voxel / layer / region
            const double e_out = p.E + (p.type == POSITRON ? 2.0 * MEC2 : 0.0);   // A11: rest energy leaves with the positron
            if (p.region == AIR) {
                if (hb.kind == 0) enter_phantom(c, p, 0.0, hb.axis);
                else if (hb.kind == 1) enter_epid(c, p, 0.0);
                else { escape(c, e_out); return; }
            } else if (p.region == PHANTOM) {
                const bool up = comp(p.dir, axis) > 0;
                setcomp(p.pos, axis, c.org[axis] + (p.iv[axis] + (up ? 1 : 0)) * c.h[axis]);
                p.iv[axis] += up ? 1 : -1;
                if (p.iv[axis] < 0 || p.iv[axis] >= c.n[axis]) {
                    p.iv[axis] = std::min(std::max(p.iv[axis], 0), c.n[axis] - 1);
                    p.region = AIR;
                }
            } else {
                if (kind == 2) { escape(c, e_out); return; }
                const int l = p.layer;
                if (p.dir.z > 0) { p.pos.z = c.ztop[l + 1]; p.layer = l + 1; if (p.layer >= c.n_layers) { escape(c, e_out); return; } }
                else { p.pos.z = c.ztop[l]; p.layer = l - 1; if (p.layer < 0) epid_to_air(c, p); }
            }
        }
        if (deflect) p.dir = rotate(p.dir, std::cos(th), std::sin(th), phi);
        // which kind of hard event: by the cross sections the distance was drawn with
        const bool is_brems = hard && brems && p.rng.u() * sig_all < sig_b;
        if (is_brems) {
            if (p.E > c.photon_cut) {                                       // photon along the electron's direction (reading A32)
                const double k = sample_brems_k(p.rng, p.E, c.photon_cut);
                Particle ph = make_child(c, p, 0, PHOTON, k, p.dir, r.seed);
                p.E -= k;
                p.rng.skip_block();
                c.counters[9]++;
                c.stack.push_back(ph);
            }
        } else if (hard && p.E > 2.0 * c.electron_cut) {                   // Moller event where the step ended, at the energy left
            const double eps = sample_moller_eps(p.rng, p.E, c.electron_cut, nullptr);
            const double W = eps * p.E, T1 = p.E - W, phi2 = 2.0 * PI * p.rng.u();
            const double cd = moller_cos(W, p.E), cp = moller_cos(T1, p.E);
            const Vec3 d0 = p.dir;
            Particle dl = make_child(c, p, 0, ELECTRON, W, rotate(d0, cd, std::sqrt(std::max(0.0, 1.0 - cd * cd)), phi2 + PI), r.seed);
            p.dir = rotate(d0, cp, std::sqrt(std::max(0.0, 1.0 - cp * cp)), phi2);
            p.E = T1;
            c.counters[9]++;
            c.aux[p.region == PHANTOM ? 2 : 3] += 1.0;                     // hard collisions in the phantom / elsewhere (pins)
            p.rng.skip_block();
            c.stack.push_back(dl);                                         // followed after the primary (LIFO; the order is immaterial, A27)
        }
    }
}

// ---------------------------------------------------------------- mode 4: multi-voxel condensed-history steps with a random hinge
// the patient transport "was developed based on DPM", a Class II condensed-history code whose electron steps cross
// voxel boundaries and are split at a random hinge.  The paper says no more; reading A38 in the notation of SURVEY 8(c)
// step 4, with the physics of mode 1 (CSDA loss, Highland deflection, no discrete events):
//   * a STEP is an energy loss dE_k = f_E T_k (T_k = energy at its start); faces do not end it;
//   * at its start one Philox block gives xi (hinge position) and (xi_a, xi_b) (deflection): the step is travelled in two LEGS,
//     losing xi dE_k before and (1 - xi) dE_k after the HINGE, where the direction is rotated by the polar angle
//     min(pi, theta0 sqrt(-2 ln xi_a)) and the azimuth 2 pi xi_b;
//   * theta0 is Highland's width for the whole step in the medium m where the hinge lies (the medium of the segment that ends
//     the first leg): mass thickness dE_k / S_m(T_k - dE_k / 2) (density cancels), mid-step energy T_k - dE_k / 2;
//   * a leg is a chain of straight SEGMENTS, each ending on a voxel / layer / region face or where the leg's energy budget R is
//     used up: ds = R / (rho S_m(T - R/2)) if that is nearer than the face (the segment then loses exactly R), else the distance
//     to the face with the midpoint-rule loss of mode 1; every segment deposits its loss in the voxel / pixel (mid-point, A24) /
//     scalar it lies in; crossing a face changes the voxel index / layer / region exactly as in mode 1;
//   * T <= T_cut ends the track as in mode 1; s_max is not used.
void transport_electron_hinge(Ctx& c, Particle p, const Run& r) {
    c.counters[14]++;
    double R = 0.0, R_after = 0.0, dEk = 0.0, Tm = 0.0, xa = 0.5, xb = 0.0;   // budget of the current leg and of the leg after the hinge; the step's loss, mid energy and deflection draws
    bool before_hinge = false;
    for (;;) {
        if (p.E <= c.electron_cut) {                                // PAPER.md:104 (200 keV): local deposit
            deposit_here(c, p, p.E);
            if (p.type == POSITRON) annihilate(c, p, r);
            return;
        }
        double rho; int m; double tb = INF; int kind = -1, axis = -1; AirHit hb{INF, 0, -1};
        if (p.region == AIR) {
            rho = RHO_AIR; m = MAT_AIR; hb = air_boundary(c, p); tb = hb.t;
        } else if (p.region == PHANTOM) {
            const size_t vi = vox_index(c, p.iv); rho = c.rho[vi]; m = c.mat[vi];
            for (int a = 0; a < 3; ++a) {
                const double da = comp(p.dir, a);
                double t = INF;
                if (da > 0) t = (c.org[a] + (p.iv[a] + 1) * c.h[a] - comp(p.pos, a)) / da;
                else if (da < 0) t = (c.org[a] + p.iv[a] * c.h[a] - comp(p.pos, a)) / da;
                if (t < tb) { tb = t; axis = a; }
            }
            if (tb < 0) tb = 0;
        } else {
            const int l = p.layer; rho = c.lrho[l]; m = c.lmat[l];
            double tf = INF;
            if (p.dir.z > 0) tf = (c.ztop[l + 1] - p.pos.z) / p.dir.z;
            else if (p.dir.z < 0) tf = (c.ztop[l] - p.pos.z) / p.dir.z;
            if (tf < 0) tf = 0;
            const double tl = world_exit_lateral(p.pos, p.dir);
            if (tl < tf) { tb = tl; kind = 2; } else { tb = tf; kind = 0; }
        }
        if (!(R > 0.0) && !before_hinge) {                          // a new step starts here, in this medium
            dEk = c.f_E * p.E; Tm = p.E - 0.5 * dEk;
            const double xi = p.rng.u(); xa = p.rng.u(); xb = p.rng.u();
            p.rng.skip_block();                                     // one block per step
            R = xi * dEk; R_after = dEk - R; before_hinge = true;
            c.counters[15]++;                                       // (mode 4: counter 15 counts steps, counters 6-8 segments)
        }
        // one segment: to the face, or to where the leg's budget is used up
        const double s_R = R / (rho * stop_pow(c, m, p.E - 0.5 * R));
        const bool on_face = !(s_R < tb);
        const double s = on_face ? tb : s_R;
        const double dE = on_face ? std::min(p.E, rho * s * stop_pow(c, m, p.E - 0.5 * rho * s * stop_pow(c, m, p.E))) : R;
        const Vec3 mid = p.pos + (0.5 * s) * p.dir;
        p.pos = p.pos + s * p.dir;
        if (p.region == AIR) { dep_air(c, dE); c.counters[7]++; }
        else if (p.region == PHANTOM) { dep_phantom(c, p.iv, dE); c.counters[6]++; }
        else { dep_epid(c, p.layer, mid.x, mid.y, dE); c.counters[8]++; }
        p.E -= dE; R -= dE;
        c.aux[0] += s; c.aux[1] += rho * s;
        if (on_face) {
            const double e_out = p.E + (p.type == POSITRON ? 2.0 * MEC2 : 0.0);
            if (p.region == AIR) {
                if (hb.kind == 0) enter_phantom(c, p, 0.0, hb.axis);
                else if (hb.kind == 1) enter_epid(c, p, 0.0);
                else { escape(c, e_out); return; }
            } else if (p.region == PHANTOM) {
                const bool up = comp(p.dir, axis) > 0;
                setcomp(p.pos, axis, c.org[axis] + (p.iv[axis] + (up ? 1 : 0)) * c.h[axis]);
                p.iv[axis] += up ? 1 : -1;
                if (p.iv[axis] < 0 || p.iv[axis] >= c.n[axis]) {
                    p.iv[axis] = std::min(std::max(p.iv[axis], 0), c.n[axis] - 1);
                    p.region = AIR;
                }
            } else {
                if (kind == 2) { escape(c, e_out); return; }
                const int l = p.layer;
                if (p.dir.z > 0) { p.pos.z = c.ztop[l + 1]; p.layer = l + 1; if (p.layer >= c.n_layers) { escape(c, e_out); return; } }
                else { p.pos.z = c.ztop[l]; p.layer = l - 1; if (p.layer < 0) epid_to_air(c, p); }
            }
        }
        if (!(R > 0.0) && before_hinge) {                           // the hinge: deflect (medium m of the segment just travelled), then the second leg
            const double th0 = highland_theta0(c, m, dEk / stop_pow(c, m, Tm), Tm);
            const double th = std::min(PI, th0 * std::sqrt(-2.0 * std::log(xa))), phi = 2.0 * PI * xb;
            p.dir = rotate(p.dir, std::cos(th), std::sin(th), phi);
            R = R_after; before_hinge = false;
        }
    }
}

// ---------------------------------------------------------------- collimation stage (section 2.1.1)
// "Particles are sampled from Phase Space 1 and transported through the jaws and MLC ... The resulting phase space (Phase Space
// 2) is ... streamed directly into the next simulation stage."  Readings (A35-A37): the stage lies between the planes
// w = w_ps1 and w = w_ps2 of the beam frame; inside the w-range of a slab every point outside the opening of its row is tungsten,
// every other point of the stage is air.  Photons are tracked by Woodcock flights against the tungsten coefficient (exact for
// any arrangement of openings); charged particles are not followed (their energy stays where the photon interacted, pair
// production included: annihilation quanta born in the head are dropped); a photon that turns upstream (dw <= 0) or leaves
// the world sideways has left the stage (escaped).  Energy absorbed in the stage is booked in the ledger's air channel.
int head_material(const Ctx& c, Vec3 q) {
    for (const Ctx::Slab& sl : c.slabs) {
        if (q.z < sl.w0 || q.z >= sl.w1) continue;
        const double across = sl.axis == 0 ? q.y : q.x, along = sl.axis == 0 ? q.x : q.y;
        const double fr = std::floor((across - sl.row0) / sl.pitch);
        if (fr < 0 || fr >= (double)sl.lo.size()) return c.col_mat;
        const size_t r = (size_t)fr;
        return (along >= sl.lo[r] && along < sl.hi[r]) ? MAT_AIR : c.col_mat;
    }
    return MAT_AIR;
}
// p.pos / p.dir in the BEAM frame, on or below the Phase Space 1 plane.  Returns true with p on the Phase Space 2 plane.
bool head_stage(Ctx& c, Particle& p) {
    auto absorb = [&](double e) { dep_air(c, e); c.head[2] += e; };
    for (;;) {
        if (p.E < c.photon_cut) { absorb(p.E); return false; }
        const double mm = std::max(c.col_rho * mu_tot(c, c.col_mat, p.E), RHO_AIR * mu_tot(c, MAT_AIR, p.E)) * (1.0 + 1e-6);
        const double s = -std::log(p.rng.u()) / mm;
        const Vec3 q = p.pos + s * p.dir;
        if (q.z >= c.w_ps2) {                                              // reaches the Phase Space 2 plane first
            const double t = (c.w_ps2 - p.pos.z) / p.dir.z;
            p.pos = p.pos + t * p.dir; p.pos.z = c.w_ps2;
            if (std::fabs(p.pos.x) >= WORLD_HALF || std::fabs(p.pos.y) >= WORLD_HALF) { escape(c, p.E); return false; }
            return true;
        }
        if (std::fabs(q.x) >= WORLD_HALF || std::fabs(q.y) >= WORLD_HALF) { escape(c, p.E); return false; }
        p.pos = q;
        const int m = head_material(c, q);
        const double rho = m == MAT_AIR ? RHO_AIR : c.col_rho;
        double mu[3]; mu_partial(c, m, p.E, mu);
        if (!(p.rng.u() * mm < rho * (mu[0] + mu[1] + mu[2]))) continue;   // virtual collision
        p.uncollided = false; c.head[3] += 1.0;
        const double x = p.rng.u() * (mu[0] + mu[1] + mu[2]);
        if (x < mu[0] || !(x < mu[0] + mu[1])) { absorb(p.E); return false; }   // photoelectric, or pair (all of E stays, reading A36)
        double E1, T; Vec3 d1, de;
        compton_scatter(p.rng, p.E, p.dir, &E1, &d1, &T, &de, nullptr);
        absorb(T);
        p.E = E1; p.dir = d1;
        if (!(p.dir.z > 0.0)) { escape(c, p.E); return false; }           // turned upstream: out of the stage
    }
}

// ---------------------------------------------------------------- source
struct SourceSample { double E; Vec3 dir_world; Vec3 dir_beam; int pixel; double u, v; };
SourceSample sample_source(const Ctx& c, Rng& rng) {
    const double x0 = rng.u(), x1 = rng.u(), x2 = rng.u(), x3 = rng.u();
    SourceSample s;
    {   // inverse of the piecewise-linear CDF of the histogram pdf
        const double target = x0 * c.cdfE[c.n_bins];
        int i = 0;
        while (i < c.n_bins - 1 && !(c.cdfE[i + 1] > target)) ++i;
        const double w = c.cdfE[i + 1] - c.cdfE[i];
        const double t = w > 0 ? (target - c.cdfE[i]) / w : 0.0;
        s.E = c.Eedges[i] + t * (c.Eedges[i + 1] - c.Eedges[i]);
    }
    {   // smallest j with CDF_F[j+1] > xi1 * CDF_F[last], row-major (v-major, u fastest)
        const double target = x1 * c.cdfF.back();
        const size_t j = (size_t)(std::upper_bound(c.cdfF.begin() + 1, c.cdfF.end(), target) - (c.cdfF.begin() + 1));
        s.pixel = (int)std::min(j, (size_t)c.fu * c.fv - 1);
    }
    const int ju = s.pixel % c.fu, jv = s.pixel / c.fu;
    s.u = (ju - 0.5 * c.fu + x2) * c.fpitch;
    s.v = (jv - 0.5 * c.fv + x3) * c.fpitch;
    s.dir_beam = normalize(Vec3{s.u, s.v, c.fdist});
    s.dir_world = dir_to_world(c, s.dir_beam);
    return s;
}

int check_ready(Ctx& c) {
    if (c.n_mat <= 0) { c.err = "init_materials not called"; return -2; }
    if (c.n[0] <= 0) { c.err = "load_phantom not called"; return -2; }
    if (c.n_layers <= 0) { c.err = "load_epid_layers not called"; return -2; }
    if (c.fu <= 0) { c.err = "load_source not called"; return -2; }
    if (c.have_col && c.n_ps1 == 0) { c.err = "a collimator needs a phase-space source"; return -2; }
    if ((c.mode == 2 || c.mode == 3) && (int)c.ne.size() != c.n_mat) { c.err = "modes 2 and 3 need orc_set_class2 (electrons per gram)"; return -2; }
    // phantom AABB must lie inside the air part of the world box
    for (int k = 0; k < 8; ++k) {
        Vec3 p{c.org[0] + ((k & 1) ? c.n[0] * c.h[0] : 0), c.org[1] + ((k & 2) ? c.n[1] * c.h[1] : 0), c.org[2] + ((k & 4) ? c.n[2] * c.h[2] : 0)};
        const Vec3 b = to_beam(c, p);
        if (std::fabs(b.x) >= WORLD_HALF || std::fabs(b.y) >= WORLD_HALF || b.z <= WORLD_WMIN || b.z >= c.sid) { c.err = "phantom outside the air region of the world"; return -3; }
    }
    if (inside_grid(c, c.src)) { c.err = "source inside the phantom"; return -3; }
    return 0;
}

void alloc_tallies(Ctx& c) {
    const size_t np = (size_t)c.nu * c.nv, nvx = (size_t)c.n[0] * c.n[1] * c.n[2];
    const size_t nr = (size_t)(c.nu / c.rebin) * (c.nv / c.rebin);
    c.ep_sum.assign(np, 0); c.ep_sq.assign(np, 0); c.unc.assign(np, 0);
    c.rb_sum.assign(nr, 0); c.rb_sq.assign(nr, 0);
    c.ph_sum.assign(nvx, 0); c.ph_sq.assign(c.want_phantom_sq ? nvx : 0, 0);
    std::fill(c.ledger, c.ledger + 8, 0.0); std::fill(c.counters, c.counters + 16, (uint64_t)0);
    std::fill(c.aux, c.aux + 4, 0.0); std::fill(c.head, c.head + 4, 0.0); c.ps2.clear();
    std::fill(c.ledger_sq, c.ledger_sq + 8, 0.0); std::fill(c.ledger_prev, c.ledger_prev + 8, 0.0);
    if (c.prb_on) { const size_t nc = (size_t)(c.n[0] / c.prb[0]) * (c.n[1] / c.prb[1]) * (c.n[2] / c.prb[2]); c.pc_sum.assign(nc, 0); c.pc_sq.assign(nc, 0); }
    else { c.pc_sum.clear(); c.pc_sq.clear(); }
    c.evlog.clear();
    c.fc_hist.assign(std::max(c.fc_bins, 0), 0.0);
}

}  // namespace

// ================================================================ C ABI (ctypes)
extern "C" {

struct orc_ctx;   // opaque = Ctx
#define C(x) (*reinterpret_cast<Ctx*>(x))

void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) { philox4x32_10(ctr, key, out); }

orc_ctx* orc_create() { return reinterpret_cast<orc_ctx*>(new Ctx()); }
void orc_destroy(orc_ctx* x) { delete reinterpret_cast<Ctx*>(x); }
const char* orc_last_error(orc_ctx* x) { return C(x).err.c_str(); }

int orc_init_materials(orc_ctx* x, int n_mat, int n_E, const float* E, const float* muC, const float* muPE, const float* muPP,
                       int n_T, const float* T, const float* S, const float* X0) {
    Ctx& c = C(x);
    if (n_mat <= 0 || n_E < 2 || n_T < 2) { c.err = "bad table sizes"; return -1; }
    c.n_mat = n_mat; c.n_E = n_E; c.n_T = n_T;
    c.Eg.assign(E, E + n_E); c.Tg.assign(T, T + n_T);
    c.lnEg.resize(n_E); c.lnTg.resize(n_T);
    for (int i = 0; i < n_E; ++i) c.lnEg[i] = std::log(c.Eg[i]);
    for (int i = 0; i < n_T; ++i) c.lnTg[i] = std::log(c.Tg[i]);
    c.muC.assign(muC, muC + (size_t)n_mat * n_E); c.muPE.assign(muPE, muPE + (size_t)n_mat * n_E);
    c.muPP.assign(muPP, muPP + (size_t)n_mat * n_E); c.S.assign(S, S + (size_t)n_mat * n_T);
    c.X0.assign(X0, X0 + n_mat);
    return 0;
}
int orc_load_phantom(orc_ctx* x, int nx, int ny, int nz, const float sp[3], const float org[3], const float* rho, const uint8_t* mat) {
    Ctx& c = C(x);
    if (c.n_mat <= 0) { c.err = "init_materials first"; return -2; }
    if (nx <= 0 || ny <= 0 || nz <= 0) { c.err = "bad grid"; return -1; }
    c.n[0] = nx; c.n[1] = ny; c.n[2] = nz;
    for (int a = 0; a < 3; ++a) { c.h[a] = sp[a]; c.org[a] = org[a]; }
    const size_t nv = (size_t)nx * ny * nz;
    c.rho.assign(rho, rho + nv); c.mat.assign(mat, mat + nv);
    for (size_t i = 0; i < nv; ++i) if (c.mat[i] >= c.n_mat) { c.err = "material index out of range"; return -1; }
    build_majorant(c);
    return 0;
}
int orc_load_epid_layers(orc_ctx* x, int nl, const float* th, const uint8_t* mat, const float* rho, const uint8_t* scored,
                         float sid, int nu, int nv, float pitch) {
    Ctx& c = C(x);
    if (nl <= 0 || nu <= 0 || nv <= 0 || !(pitch > 0)) { c.err = "bad EPID"; return -1; }
    c.n_layers = nl; c.nu = nu; c.nv = nv; c.sid = sid; c.pitch = pitch;
    c.lt.assign(th, th + nl); c.lrho.assign(rho, rho + nl);
    c.lmat.assign(mat, mat + nl); c.lscored.assign(scored, scored + nl);
    c.ztop.assign(nl + 1, 0.0); c.ztop[0] = sid;
    for (int l = 0; l < nl; ++l) c.ztop[l + 1] = c.ztop[l] + c.lt[l];
    return 0;
}
int orc_load_source(orc_ctx* x, const float src[3], const float axes[9], int nb, const float* edges, const float* pdf,
                    int fu, int fv, float fpitch, float fdist, const float* fl) {
    Ctx& c = C(x);
    if (nb <= 0 || fu <= 0 || fv <= 0) { c.err = "bad source"; return -1; }
    c.src = {src[0], src[1], src[2]};
    c.au = {axes[0], axes[1], axes[2]}; c.av = {axes[3], axes[4], axes[5]}; c.aw = {axes[6], axes[7], axes[8]};
    c.n_bins = nb; c.Eedges.assign(edges, edges + nb + 1);
    c.cdfE.assign(nb + 1, 0.0);
    for (int i = 0; i < nb; ++i) c.cdfE[i + 1] = c.cdfE[i] + (double)pdf[i];
    c.fu = fu; c.fv = fv; c.fpitch = fpitch; c.fdist = fdist;
    c.fluence.assign(fl, fl + (size_t)fu * fv);
    c.cdfF.assign((size_t)fu * fv + 1, 0.0);
    for (size_t j = 0; j < (size_t)fu * fv; ++j) c.cdfF[j + 1] = c.cdfF[j] + (double)fl[j];
    if (!(c.cdfE[nb] > 0) || !(c.cdfF.back() > 0)) { c.err = "empty spectrum or fluence"; return -1; }
    return 0;
}
int orc_set_physics(orc_ctx* x, int mode, double pcut, double ecut, double fE, double smax) {
    Ctx& c = C(x); c.mode = mode; c.photon_cut = pcut; c.electron_cut = ecut; c.f_E = fE; c.s_max = smax; return 0;
}
// options: tracking (0 Woodcock / 1 surface), rebin factor, keep phantom sum of squares, first-collision histogram
// mode 2 input: electrons per gram of every material
int orc_set_class2(orc_ctx* x, int n_mat, const float* ne) { Ctx& c = C(x); c.ne.assign(ne, ne + n_mat); return 0; }
// unit-level: Moller cross section per electron and hard-loss integral; n samples of eps
int orc_moller_xs(double T, double Tc, double out[2]) { const MollerXs r = moller_xs(T, Tc); out[0] = r.sigma; out[1] = r.hard; return 0; }
int orc_sample_moller(double T, double Tc, uint64_t seed, uint64_t n, double* eps) {
    Rng rng; rng.init(seed, 0, 0);
    for (uint64_t i = 0; i < n; ++i) eps[i] = sample_moller_eps(rng, T, Tc, nullptr);
    return 0;
}
double orc_moller_cos(double Tout, double Tin) { return moller_cos(Tout, Tin); }
int orc_brems_xs(double T, double kc, double X0, double out[2]) { const BremsXs r = brems_xs(T, kc, X0); out[0] = r.sigma; out[1] = r.soft; return 0; }
int orc_sample_brems(double T, double kc, uint64_t seed, uint64_t n, double* k) {
    Rng rng; rng.init(seed, 0, 0);
    for (uint64_t i = 0; i < n; ++i) k[i] = sample_brems_k(rng, T, kc);
    return 0;
}
int orc_set_options(orc_ctx* x, int tracking, int rebin, int want_phantom_sq, int fc_bins, double fc_w0, double fc_dw) {
    Ctx& c = C(x);
    if (rebin < 1) { c.err = "rebin < 1"; return -1; }
    c.tracking = tracking; c.rebin = rebin; c.want_phantom_sq = want_phantom_sq != 0;
    c.fc_bins = fc_bins; c.fc_w0 = fc_w0; c.fc_dw = fc_dw;
    return 0;
}
// type < 0 clears the override.  pos / dir in the world frame.
int orc_set_fixed_primary(orc_ctx* x, int type, double E, const double pos[3], const double dir[3]) {
    Ctx& c = C(x);
    if (type < 0) { c.fixed = false; return 0; }
    c.fixed = true; c.fx_type = type; c.fx_E = E; c.fx_pos = {pos[0], pos[1], pos[2]};
    c.fx_dir = normalize(Vec3{dir[0], dir[1], dir[2]});
    return 0;
}
int orc_reset(orc_ctx* x) {
    Ctx& c = C(x);
    int rc = check_ready(c); if (rc) return rc;
    if (c.nu % c.rebin || c.nv % c.rebin) { c.err = "rebin must divide nu and nv"; return -1; }
    alloc_tallies(c); return 0;
}
// Histories [first, first + n); accumulates into the tallies (call orc_reset first).
int orc_run(orc_ctx* x, uint64_t first, uint64_t n, uint64_t seed) {
    Ctx& c = C(x);
    if (c.ep_sum.empty()) { int rc = orc_reset(x); if (rc) return rc; }
    Run r{seed};
    for (uint64_t h = first; h < first + n; ++h) {
        Particle p{};
        c.cur_h = h;
        p.rng.init(seed, h, 0);
        bool through = true;
        if (c.n_ps1 > 0) {
            // Phase Space 1 source (reading A35): record floor(xi0 n) of the table, xi0 = first draw of block 0; the other
            // three draws of the block are not used
            const double x0 = p.rng.u(); p.rng.skip_block();
            const size_t j = std::min((size_t)(x0 * (double)c.n_ps1), c.n_ps1 - 1);
            const float* q = c.ps1.data() + 8 * j;
            p.type = PHOTON; p.E = q[5]; p.region = AIR; p.uncollided = true;
            p.pos = {q[0], q[1], c.w_ps1}; p.dir = normalize(Vec3{q[2], q[3], q[4]});
            c.ledger[0] += p.E; c.ledger[6] += 1.0;
            if (c.have_col) through = head_stage(c, p);
            if (through) {
                c.head[0] += 1.0; c.head[1] += p.E;
                if (c.ps2_on) { const double rec[8] = {p.E, p.pos.x, p.pos.y, p.dir.x, p.dir.y, p.dir.z, (double)h, p.uncollided ? 1.0 : 0.0}; c.ps2.insert(c.ps2.end(), rec, rec + 8); }
                p.pos = to_world(c, p.pos); p.dir = dir_to_world(c, p.dir);
            }
            c.stack.clear();
            if (through) c.stack.push_back(p);
            while (!c.stack.empty()) {
                Particle q2 = c.stack.back(); c.stack.pop_back();
                if (q2.type == PHOTON) transport_photon(c, q2, r); else if (c.mode == 4) transport_electron_hinge(c, q2, r); else transport_electron(c, q2, r);
            }
            flush_history(c);
            continue;
        }
        const SourceSample s = sample_source(c, p.rng);             // block 0 of particle 0 (reading A1)
        p.type = PHOTON; p.E = s.E; p.pos = c.src; p.dir = s.dir_world; p.region = AIR; p.uncollided = true;
        if (c.fixed) {
            p.type = c.fx_type; p.E = c.fx_E; p.pos = c.fx_pos; p.dir = c.fx_dir;
            p.uncollided = (p.type == PHOTON);
            if (inside_grid(c, p.pos)) { p.region = PHANTOM; locate_voxel(c, p.pos, p.iv); }
            else {
                const Vec3 b = to_beam(c, p.pos);
                if (b.z >= c.sid && b.z < c.ztop[c.n_layers]) {
                    p.region = EPID; p.dir = dir_to_beam(c, p.dir); p.pos = b; p.layer = 0;
                    while (p.layer < c.n_layers - 1 && b.z >= c.ztop[p.layer + 1]) p.layer++;
                }
            }
        }
        c.ledger[0] += p.E + (p.type == POSITRON ? 2.0 * MEC2 : 0.0);
        c.ledger[6] += 1.0;
        c.stack.clear(); c.stack.push_back(p);
        while (!c.stack.empty()) {                                  // LIFO
            c.counters[11] = std::max<uint64_t>(c.counters[11], c.stack.size());
            Particle q = c.stack.back(); c.stack.pop_back();
            if (q.type == PHOTON) transport_photon(c, q, r); else if (c.mode == 4) transport_electron_hinge(c, q, r); else transport_electron(c, q, r);
        }
        flush_history(c);
    }
    return 0;
}
// Raw accumulators (any pointer may be NULL).  Sizes: epid nu*nv, rebinned (nu/r)*(nv/r), phantom nx*ny*nz.
int orc_read(orc_ctx* x, double* ep_sum, double* ep_sq, double* rb_sum, double* rb_sq, double* ph_sum, double* ph_sq,
             double* unc, double ledger[8], uint64_t counters[16], double aux[4], double* fc_hist) {
    Ctx& c = C(x);
    auto cp = [](double* d, const std::vector<double>& s) { if (d && !s.empty()) std::memcpy(d, s.data(), s.size() * sizeof(double)); };
    cp(ep_sum, c.ep_sum); cp(ep_sq, c.ep_sq); cp(rb_sum, c.rb_sum); cp(rb_sq, c.rb_sq);
    cp(ph_sum, c.ph_sum); cp(ph_sq, c.ph_sq); cp(unc, c.unc); cp(fc_hist, c.fc_hist);
    if (ledger) std::memcpy(ledger, c.ledger, sizeof(c.ledger));
    if (counters) std::memcpy(counters, c.counters, sizeof(c.counters));
    if (aux) std::memcpy(aux, c.aux, sizeof(c.aux));
    return 0;
}

// Coarse phantom tally: blocks of rx x ry x rz voxels (must divide the grid; 1,1,1 switches it off).  Takes effect at orc_reset.
int orc_set_phantom_rebin(orc_ctx* x, int rx, int ry, int rz) {
    Ctx& c = C(x);
    if (rx < 1 || ry < 1 || rz < 1) { c.err = "phantom rebin < 1"; return -1; }
    if (c.n[0] > 0 && (c.n[0] % rx || c.n[1] % ry || c.n[2] % rz)) { c.err = "phantom rebin must divide the grid"; return -1; }
    c.prb[0] = rx; c.prb[1] = ry; c.prb[2] = rz; c.prb_on = rx * ry * rz > 1;
    return 0;
}
// Coarse phantom sums / sums of squares [(nz/rz)][(ny/ry)][(nx/rx)] and the second moments of the ledger channels (any may be NULL).
int orc_read_extra(orc_ctx* x, double* pc_sum, double* pc_sq, double ledger_sq[8]) {
    Ctx& c = C(x);
    if (pc_sum && !c.pc_sum.empty()) std::memcpy(pc_sum, c.pc_sum.data(), c.pc_sum.size() * sizeof(double));
    if (pc_sq && !c.pc_sq.empty()) std::memcpy(pc_sq, c.pc_sq.data(), c.pc_sq.size() * sizeof(double));
    if (ledger_sq) std::memcpy(ledger_sq, c.ledger_sq, sizeof(c.ledger_sq));
    return 0;
}
// Event log for the pins: keep up to `capacity` records of 16 doubles (0 switches it off); cleared by orc_reset.
int orc_set_event_log(orc_ctx* x, uint64_t capacity) { Ctx& c = C(x); c.log_cap = (size_t)capacity; c.evlog.clear(); return 0; }
uint64_t orc_event_log_count(orc_ctx* x) { return C(x).evlog.size() / 16; }
int orc_read_event_log(orc_ctx* x, double* out) { Ctx& c = C(x); if (!c.evlog.empty()) std::memcpy(out, c.evlog.data(), c.evlog.size() * sizeof(double)); return 0; }

// Collimation stage.  Slab k spans w in [w0[k], w1[k]) of the beam frame, its rows are stacked along v (axis 0: openings in u) or
// along u (axis 1: openings in v) from row0[k] with pitch[k]; row r opens [lo, hi) (concatenated arrays, n_rows[k] entries per
// slab); outside the rows and outside the openings the slab is material `mat` at `rho`.  n_slabs = 0 removes the collimator.
int orc_load_collimator(orc_ctx* x, int n_slabs, const float* w0, const float* w1, const int* axis, const int* n_rows, const float* row0,
                        const float* pitch, const float* lo, const float* hi, int mat, double rho, double w_ps2) {
    Ctx& c = C(x);
    c.slabs.clear(); c.have_col = false;
    if (n_slabs == 0) return 0;
    if (mat < 0 || mat >= c.n_mat || !(rho > 0)) { c.err = "bad collimator material"; return -1; }
    size_t o = 0; double prev = -INF;
    for (int k = 0; k < n_slabs; ++k) {
        if (!(w1[k] > w0[k]) || !(w0[k] >= prev) || n_rows[k] < 1 || !(pitch[k] > 0)) { c.err = "bad collimator slab"; return -1; }
        Ctx::Slab sl{w0[k], w1[k], axis[k], row0[k], pitch[k], {}, {}};
        for (int r = 0; r < n_rows[k]; ++r, ++o) { sl.lo.push_back(lo[o]); sl.hi.push_back(hi[o]); }
        c.slabs.push_back(sl); prev = w1[k];
    }
    if (!(w_ps2 >= prev)) { c.err = "Phase Space 2 plane above the last slab"; return -1; }
    c.col_mat = mat; c.col_rho = rho; c.w_ps2 = w_ps2; c.have_col = true;
    return 0;
}
// Phase Space 1 records [n][8] = {u, v, du, dv, dw, E, -, -} on the plane w = w_plane of the beam frame; n = 0 goes back to the
// fluence-map source.  The beam frame is the one of orc_load_source (source position and axes).
int orc_load_phase_space_source(orc_ctx* x, uint64_t n, const float* rec, double w_plane) {
    Ctx& c = C(x);
    c.ps1.assign(rec, rec + 8 * n); c.n_ps1 = (size_t)n; c.w_ps1 = w_plane;
    return 0;
}
int orc_read_head(orc_ctx* x, double out[4]) { std::memcpy(out, C(x).head, 4 * sizeof(double)); return 0; }
int orc_set_ps2(orc_ctx* x, int on) { Ctx& c = C(x); c.ps2_on = on != 0; c.ps2.clear(); return 0; }
uint64_t orc_ps2_count(orc_ctx* x) { return C(x).ps2.size() / 8; }
int orc_read_ps2(orc_ctx* x, double* out) { Ctx& c = C(x); if (!c.ps2.empty()) std::memcpy(out, c.ps2.data(), c.ps2.size() * sizeof(double)); return 0; }

// Phase Space 3: switch the recording on / off (clears the store), number of records, copy out [n][8].
int orc_set_ps3(orc_ctx* x, int on) { Ctx& c = C(x); c.ps3_on = on != 0; c.ps3.clear(); return 0; }
uint64_t orc_ps3_count(orc_ctx* x) { return C(x).ps3.size() / 8; }
int orc_read_ps3(orc_ctx* x, double* out) { Ctx& c = C(x); if (!c.ps3.empty()) std::memcpy(out, c.ps3.data(), c.ps3.size() * sizeof(double)); return 0; }

// ---- unit-level entry points for the pins
int orc_mu_partial(orc_ctx* x, int m, double E, double out[3]) { mu_partial(C(x), m, E, out); return 0; }
double orc_stop_pow(orc_ctx* x, int m, double T) { return stop_pow(C(x), m, T); }
double orc_majorant(orc_ctx* x, double E) { return majorant(C(x), E); }
double orc_highland_theta0(orc_ctx* x, int m, double rho_s, double Tm) { return highland_theta0(C(x), m, rho_s, Tm); }
// K1 for histories [first, first+n): out[h] = {E, dir_world xyz, pixel, u, v} (7 doubles each)
int orc_sample_source(orc_ctx* x, uint64_t first, uint64_t n, uint64_t seed, double* out) {
    Ctx& c = C(x);
    if (c.fu <= 0) { c.err = "load_source first"; return -2; }
    for (uint64_t k = 0; k < n; ++k) {
        Rng rng; rng.init(seed, first + k, 0);
        const SourceSample s = sample_source(c, rng);
        double* o = out + 7 * k;
        o[0] = s.E; o[1] = s.dir_world.x; o[2] = s.dir_world.y; o[3] = s.dir_world.z; o[4] = s.pixel; o[5] = s.u; o[6] = s.v;
    }
    return 0;
}
// n Klein-Nishina samples at energy E from stream (seed, history k, particle 0)
int orc_sample_compton(double E, uint64_t seed, uint64_t n, double* eps, double* cost) {
    for (uint64_t k = 0; k < n; ++k) { Rng rng; rng.init(seed, k, 0); sample_kn(rng, E, eps + k, cost + k, nullptr); }
    return 0;
}
// n full Compton events of a photon (E, d0): out[k] = {E1, d1 xyz, T, de xyz} (8 doubles each)
int orc_compton_events(double E, const double d0[3], uint64_t seed, uint64_t n, double* out) {
    const Vec3 d = normalize(Vec3{d0[0], d0[1], d0[2]});
    for (uint64_t k = 0; k < n; ++k) {
        Rng rng; rng.init(seed, k, 0);
        double E1, T; Vec3 d1, de;
        compton_scatter(rng, E, d, &E1, &d1, &T, &de, nullptr);
        double* o = out + 8 * k;
        o[0] = E1; o[1] = d1.x; o[2] = d1.y; o[3] = d1.z; o[4] = T; o[5] = de.x; o[6] = de.y; o[7] = de.z;
    }
    return 0;
}
// n Highland deflections of direction d0 with width theta0 (the step-4 sampling rule): out[k] = new direction
int orc_sample_deflection(const double d0[3], double theta0, uint64_t seed, uint64_t n, double* out) {
    const Vec3 d = normalize(Vec3{d0[0], d0[1], d0[2]});
    for (uint64_t k = 0; k < n; ++k) {
        Rng rng; rng.init(seed, k, 0);
        const double xa = rng.u(), xb = rng.u();
        const double th = std::min(PI, theta0 * std::sqrt(-2.0 * std::log(xa)));
        const Vec3 r = rotate(d, std::cos(th), std::sin(th), 2.0 * PI * xb);
        out[3 * k] = r.x; out[3 * k + 1] = r.y; out[3 * k + 2] = r.z;
    }
    return 0;
}

// ---- K8 response post-pass
// Effective field size (Eq. 1; reading A16): a, b = extent at the isocentre plane (w = 100 cm) of the
// bounding box of fluence pixels with weight > 0.  Equivalent square s = 2ab/(a+b); printed form ab/(2(a+b)) behind a flag.
double orc_field_size(orc_ctx* x, int printed_form) {
    Ctx& c = C(x);
    int u0 = c.fu, u1 = -1, v0 = c.fv, v1 = -1;
    for (int j = 0; j < c.fv; ++j) for (int i = 0; i < c.fu; ++i)
        if (c.fluence[(size_t)j * c.fu + i] > 0) { u0 = std::min(u0, i); u1 = std::max(u1, i); v0 = std::min(v0, j); v1 = std::max(v1, j); }
    if (u1 < 0) return 0.0;
    const double sc = 100.0 / c.fdist;
    const double a = (u1 - u0 + 1) * c.fpitch * sc, b = (v1 - v0 + 1) * c.fpitch * sc;
    return printed_form ? a * b / (2.0 * (a + b)) : 2.0 * a * b / (a + b);
}
// Radiological thickness map (reading A17): exact Siddon line integral of rho/(1 g cm^-3) from the source
// to each pixel centre on the EPID top plane, through the phantom grid only.  out[nv*nu].
int orc_tmap(orc_ctx* x, double* out) {
    Ctx& c = C(x);
    int rc = check_ready(c); if (rc) return rc;
    for (int jv = 0; jv < c.nv; ++jv) for (int ju = 0; ju < c.nu; ++ju) {
        const Vec3 pb{(ju + 0.5 - 0.5 * c.nu) * c.pitch, (jv + 0.5 - 0.5 * c.nv) * c.pitch, c.sid};
        const Vec3 end = to_world(c, pb);
        const Vec3 d = end - c.src;                                  // parameter a in [0,1]
        double a0 = 0.0, a1 = 1.0; bool hit = true;
        for (int a = 0; a < 3; ++a) {
            const double lo = c.org[a], hi = c.org[a] + c.n[a] * c.h[a], pa = comp(c.src, a), da = comp(d, a);
            if (da == 0) { if (pa < lo || pa >= hi) hit = false; continue; }
            double t1 = (lo - pa) / da, t2 = (hi - pa) / da; if (t1 > t2) std::swap(t1, t2);
            a0 = std::max(a0, t1); a1 = std::min(a1, t2);
        }
        double acc = 0.0;
        if (hit && a0 < a1) {
            const double len = std::sqrt(dot(d, d));
            // merge the sorted plane crossings of the three axes
            std::vector<double> al; al.push_back(a0); al.push_back(a1);
            for (int a = 0; a < 3; ++a) {
                const double da = comp(d, a); if (da == 0) continue;
                for (int k = 0; k <= c.n[a]; ++k) {
                    const double t = (c.org[a] + k * c.h[a] - comp(c.src, a)) / da;
                    if (t > a0 && t < a1) al.push_back(t);
                }
            }
            std::sort(al.begin(), al.end());
            for (size_t k = 0; k + 1 < al.size(); ++k) {
                const double am = 0.5 * (al[k] + al[k + 1]);
                const Vec3 pm = c.src + am * d;
                if (!inside_grid(c, pm)) continue;
                int iv[3]; locate_voxel(c, pm, iv);
                acc += (al[k + 1] - al[k]) * len * c.rho[vox_index(c, iv)];
            }
        }
        out[(size_t)jv * c.nu + ju] = acc;
    }
    return 0;
}
// k(t, s) by bilinear interpolation in lut[it*ns + is] on uniform axes, (t, s) clamped into the table (reading A18).
double orc_lut_bilinear(const double* lut, int nt, int ns, double t_min, double t_max, double s_min, double s_max, double t, double s) {
    double ft = nt > 1 ? (std::min(std::max(t, t_min), t_max) - t_min) / (t_max - t_min) * (nt - 1) : 0.0;
    double fs = ns > 1 ? (std::min(std::max(s, s_min), s_max) - s_min) / (s_max - s_min) * (ns - 1) : 0.0;
    int it = std::min((int)std::floor(ft), std::max(nt - 2, 0)), is = std::min((int)std::floor(fs), std::max(ns - 2, 0));
    const double wt = ft - it, ws = fs - is;
    const int it1 = std::min(it + 1, nt - 1), is1 = std::min(is + 1, ns - 1);
    return (1 - wt) * ((1 - ws) * lut[it * ns + is] + ws * lut[it * ns + is1]) + wt * ((1 - ws) * lut[it1 * ns + is] + ws * lut[it1 * ns + is1]);
}
// signal = dose * k(t_uv, s).  n = nu*nv.
int orc_apply_lut(const double* lut, int nt, int ns, double t_min, double t_max, double s_min, double s_max,
                  double s_eff, const double* dose, const double* tmap, size_t n, double* out) {
    for (size_t i = 0; i < n; ++i) out[i] = dose[i] * orc_lut_bilinear(lut, nt, ns, t_min, t_max, s_min, s_max, tmap[i], s_eff);
    return 0;
}

}  // extern "C"
