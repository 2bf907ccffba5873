// Host side of the C-ABI declared in include/aepid.h: argument checking, workspace layout, table
// preparation (ln-domain tables, majorant, integer CDF thresholds) and kernel launches.  No device
// allocation happens here: every device byte lives in the caller's workspace.
#include <cuda_runtime.h>
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "../../include/aepid.h"
#include "params.h"

using namespace aepid;

namespace {

constexpr size_t kAlign = 256;
constexpr size_t kMaxLut = 65536;
inline size_t up(size_t x) { return (x + kAlign - 1) & ~(kAlign - 1); }

struct Layout {
    size_t vox, ph_batch, ep_batch, out_ph, out_ep, tmap, signal, dose_in, lut, blob, thrE, edges, thrF, guideF, queues, small, ps1, head_rows, total;
    size_t nvox, npix, blob_bytes;
};

bool dims_ok(const aepid_dims* d) {
    if (!d) return false;
    if (d->n_mat < 1 || d->n_mat > kMaxMat || d->n_E < 2 || d->n_E > 4096 || d->n_T < 2 || d->n_T > 4096) return false;
    if (d->nx < 1 || d->ny < 1 || d->nz < 1 || d->nx > 1024 || d->ny > 1024 || d->nz > 1024) return false;
    if (d->n_layers < 1 || d->n_layers > kMaxLayers || d->nu < 1 || d->nv < 1 || d->nu > 16384 || d->nv > 16384) return false;
    if (d->n_bins < 1 || d->n_bins > 65536 || d->fu < 1 || d->fv < 1 || d->fu > 4096 || d->fv > 4096) return false;
    if (d->n_batches < 2 || d->n_batches > 255) return false;
    if (d->max_live_per_cta != 0 && (d->max_live_per_cta < 64 || d->max_live_per_cta > kMaxPoolSlots / 2)) return false;
    if (d->n_ps1 < 0) return false;
    return true;
}

// records per class queue of a CTA: twice the most particles a CTA keeps alive (queue protocol in transport.cu), a power of two
int pool_log_for(const aepid_dims& d) {
    const int live = d.max_live_per_cta ? d.max_live_per_cta : kDefaultLive;
    int lg = 7;
    while ((1 << lg) < 2 * live) ++lg;
    return lg;
}

Layout make_layout(const aepid_dims& d) {
    Layout L{};
    L.nvox = (size_t)d.nx * d.ny * d.nz;
    L.npix = (size_t)d.nu * d.nv;
    L.blob_bytes = ((size_t)d.n_mat * d.n_E * 4 + d.n_E + (size_t)d.n_mat * d.n_T * 4 + d.n_mat + d.n_E + kEGuide + 1) * 4;
    size_t o = 0;
    auto take = [&](size_t bytes) { const size_t at = o; o += up(bytes); return at; };
    L.vox = take(L.nvox * 4);
    L.ph_batch = take(L.nvox * 4 * d.n_batches);
    L.ep_batch = take(L.npix * 4 * d.n_batches);
    L.out_ph = take(L.nvox * 8);
    L.out_ep = take(L.npix * 8);
    L.tmap = take(L.npix * 4);
    L.signal = take(L.npix * 4);
    L.dose_in = take(L.npix * 4);
    L.lut = take(kMaxLut * 4);
    L.blob = take(L.blob_bytes);
    L.thrE = take(((size_t)d.n_bins + 1) * 4);
    L.edges = take(((size_t)d.n_bins + 1) * 4);
    L.thrF = take(((size_t)d.fu * d.fv + 1) * 4);
    L.guideF = take(((size_t)kGuideSize + 1) * 4);
    L.queues = take((size_t)kMaxCtas * kRingCount * ((size_t)1 << pool_log_for(d)) * kRecordBytes);   // class queues of the transport kernel (scratch)
    L.small = take(1024);            // ledger [8] f64 @0 | chunk counter @64 | bad-material flag @68 | rho_max [32] f32 @128 | counters [32] u64 @256 | gamma stats [4] f64 @512, max bits @544 | PS3 count u64 @576 | head stats [4] f64 @640 | body box [6] i32 @704, f_out bits @728 | kfac [32] f32 @768
    L.ps1 = take((size_t)d.n_ps1 * 32);                 // Phase Space 1 records (collimation stage), 0 if not used
    L.head_rows = take((size_t)kMaxHeadRows * 8);        // openings lo[] | hi[] of the collimator rows
    L.total = o;
    return L;
}

}  // namespace

struct aepid_ctx {
    int device = 0, sm_count = 148;
    cudaStream_t stream = nullptr;
    aepid_dims dims{};
    Layout lay{};
    char* ws = nullptr;
    std::string err;
    // host copies of what the tables are built from
    int n_mat = 0, n_E = 0, n_T = 0;
    std::vector<float> Eg, Tg, muC, muPE, muPP, S, X0;
    std::vector<float> rho_max;
    bool have_mat = false, have_phantom = false, have_epid = false, have_source = false, tables_dirty = true;
    Geom g{};
    Physics ph{1, 0.010f, 0.200f, 0.10f, 1.0f};
    Tables tb{};
    Source so{};
    int bb_u0 = 0, bb_u1 = -1, bb_v0 = 0, bb_v1 = -1;    // bounding box of positive fluence pixels
    unsigned long long n_done = 0;                         // histories since the last reset
    unsigned long long first_history = 0;                  // global index of history 0 of this context (multi-GPU sharding)
    double hist[256] = {0};
    std::vector<float> ne; bool have_ne = false;               // electrons per gram (aepid_set_class2)
    bool counting = false;
    int pool_log = kMaxPoolLog;                                // log2 of the records per class queue of a CTA (from dims.max_live_per_cta)
    int live_max = kMaxPoolSlots / 2;
    float4* ps3 = nullptr; unsigned long long ps3_cap = 0;       // caller-owned Phase Space 3 buffer (aepid_set_phase_space)
    Head hd{};                                                   // collimation stage (aepid_load_phase_space_source, aepid_load_collimator)

    uint32_t* d_vox() { return reinterpret_cast<uint32_t*>(ws + lay.vox); }
    float* d_ph_batch() { return reinterpret_cast<float*>(ws + lay.ph_batch); }
    float* d_ep_batch() { return reinterpret_cast<float*>(ws + lay.ep_batch); }
    float* d_out_ph() { return reinterpret_cast<float*>(ws + lay.out_ph); }
    float* d_out_ep() { return reinterpret_cast<float*>(ws + lay.out_ep); }
    float* d_tmap() { return reinterpret_cast<float*>(ws + lay.tmap); }
    float* d_signal() { return reinterpret_cast<float*>(ws + lay.signal); }
    float* d_dose_in() { return reinterpret_cast<float*>(ws + lay.dose_in); }
    float* d_lut() { return reinterpret_cast<float*>(ws + lay.lut); }
    uint32_t* d_blob() { return reinterpret_cast<uint32_t*>(ws + lay.blob); }
    uint32_t* d_thrE() { return reinterpret_cast<uint32_t*>(ws + lay.thrE); }
    float* d_edges() { return reinterpret_cast<float*>(ws + lay.edges); }
    uint32_t* d_thrF() { return reinterpret_cast<uint32_t*>(ws + lay.thrF); }
    uint32_t* d_guideF() { return reinterpret_cast<uint32_t*>(ws + lay.guideF); }
    double* d_ledger() { return reinterpret_cast<double*>(ws + lay.small); }
    unsigned long long* d_counters() { return reinterpret_cast<unsigned long long*>(ws + lay.small + 256); }
    unsigned int* d_chunk() { return reinterpret_cast<unsigned int*>(ws + lay.small + 64); }
    unsigned int* d_bad_mat() { return reinterpret_cast<unsigned int*>(ws + lay.small + 68); }
    float* d_rho_max() { return reinterpret_cast<float*>(ws + lay.small + 128); }
    double* d_gamma_stats() { return reinterpret_cast<double*>(ws + lay.small + 512); }
    unsigned int* d_gamma_max() { return reinterpret_cast<unsigned int*>(ws + lay.small + 544); }
    unsigned long long* d_ps3_count() { return reinterpret_cast<unsigned long long*>(ws + lay.small + 576); }
    double* d_head_stats() { return reinterpret_cast<double*>(ws + lay.small + 640); }      // [4]
    int* d_body_box() { return reinterpret_cast<int*>(ws + lay.small + 704); }                // [6] + the f_out bits
    float* d_kfac() { return reinterpret_cast<float*>(ws + lay.small + 768); }                // [kMaxMat]
    float4* d_ps1() { return reinterpret_cast<float4*>(ws + lay.ps1); }
    float* d_head_rows() { return reinterpret_cast<float*>(ws + lay.head_rows); }
};

namespace {

int fail(aepid_ctx* c, int code, const std::string& msg) { if (c) c->err = msg; return code; }
#define CU(call)                                                                                         \
    do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return fail(ctx, AEPID_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e_)); } while (0)

enum MemKind { MEM_HOST_PAGEABLE, MEM_HOST_PINNED, MEM_DEVICE };
MemKind classify(const void* p) {
    cudaPointerAttributes a{};
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return MEM_HOST_PAGEABLE; }
    if (a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged) return MEM_DEVICE;
    if (a.type == cudaMemoryTypeHost) return MEM_HOST_PINNED;
    return MEM_HOST_PAGEABLE;
}
// Copy a host-or-device input array to a host vector (small arrays the host needs to see).
template <class T>
int fetch(aepid_ctx* ctx, const T* src, size_t n, std::vector<T>& out) {
    out.resize(n);
    if (classify(src) == MEM_DEVICE) {
        CU(cudaMemcpyAsync(out.data(), src, n * sizeof(T), cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
    } else std::memcpy(out.data(), src, n * sizeof(T));
    return 0;
}
// Deliver a device result to a host-or-device output pointer.
int deliver(aepid_ctx* ctx, void* dst, const void* dev_src, size_t bytes, bool* need_sync) {
    const MemKind k = classify(dst);
    CU(cudaMemcpyAsync(dst, dev_src, bytes, k == MEM_DEVICE ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, ctx->stream));
    if (k != MEM_DEVICE) *need_sync = true;
    return 0;
}

// The transport kernel reports what must never happen (a secondary without head room, a scheduler that found no runnable
// phase) in ledger[7]; tallies of such a run are incomplete.  Called right after a stream synchronisation.
int check_internal(aepid_ctx* ctx, const double* host_ledger) {
    if (host_ledger[7] != 0.0) {
        char buf[320];
        std::snprintf(buf, sizeof buf, "transport kernel raised internal error flags %.0f (2: secondary dropped for want of head room, 8: scheduler stalled, 16: index or queue-protocol check of the checked build failed); tallies are incomplete", host_ledger[7]);
        return fail(ctx, AEPID_ERR_INTERNAL, buf);
    }
    return 0;
}

int reset_tallies(aepid_ctx* ctx) {
    const size_t B = ctx->dims.n_batches;
    CU(cudaMemsetAsync(ctx->d_ph_batch(), 0, ctx->lay.nvox * 4 * B, ctx->stream));
    CU(cudaMemsetAsync(ctx->d_ep_batch(), 0, ctx->lay.npix * 4 * B, ctx->stream));
    CU(cudaMemsetAsync(ctx->ws + ctx->lay.small, 0, 128, ctx->stream));
    CU(cudaMemsetAsync(ctx->ws + ctx->lay.small + 256, 0, 256, ctx->stream));
    CU(cudaMemsetAsync(ctx->d_ps3_count(), 0, 8, ctx->stream));
    CU(cudaMemsetAsync(ctx->d_head_stats(), 0, 32, ctx->stream));
    ctx->n_done = 0; ctx->first_history = 0;
    std::fill(ctx->hist, ctx->hist + 256, 0.0);
    return 0;
}

// Moller cross section per electron for energy transfers above Tc, and the energy-weighted integral (reading A31):
// d sigma / d eps = (2 pi r_e^2 m c^2 / (beta^2 T)) [1/eps^2 + 1/(1-eps)^2 + (tau/(tau+1))^2 - (2 tau+1)/(tau+1)^2 / (eps (1-eps))],
// integrated over eps = W / T from Tc / T to 1/2.  Host side, double.
void moller_integrals(double T, double Tc, double& sigma, double& hard) {
    sigma = 0.0; hard = 0.0;
    if (!(T > 2.0 * Tc)) return;
    const double mec2 = 0.51099895, re = 2.8179403262e-13, pi = 3.14159265358979323846;
    const double tau = T / mec2, t1 = tau + 1.0, beta2 = tau * (tau + 2.0) / (t1 * t1);
    const double q1 = tau * tau / (t1 * t1), q2 = (2.0 * tau + 1.0) / (t1 * t1);
    const double lo = Tc / T, pref = 2.0 * pi * re * re * mec2 / (beta2 * T);
    sigma = pref * ((1.0 / lo - 2.0) + (2.0 - 1.0 / (1.0 - lo)) + q1 * (0.5 - lo) - q2 * std::log((1.0 - lo) / lo));
    const double w1 = -std::log(2.0 * lo);
    const double w2 = (2.0 - std::log(2.0)) - (1.0 / (1.0 - lo) + std::log(1.0 - lo));
    const double w3 = 0.5 * q1 * (0.25 - lo * lo);
    const double w4 = q2 * (std::log(1.0 - lo) + std::log(2.0));
    hard = pref * T * (w1 + w2 + w3 - w4);
}

bool log_uniform(const std::vector<float>& g) {
    const int n = (int)g.size();
    if (!(g[0] > 0)) return false;
    const double l0 = std::log((double)g[0]), d = (std::log((double)g[n - 1]) - l0) / (n - 1);
    if (!(d > 0)) return false;
    for (int i = 0; i < n; ++i) if (std::fabs(std::log((double)g[i]) - (l0 + i * d)) > 1e-3 * d) return false;
    return true;
}

// ln-domain photon tables, majorant (reading A7 as corrected in DESIGN.md), ln stopping power, 1/X0.
int build_tables(aepid_ctx* ctx) {
    const int nm = ctx->n_mat, nE = ctx->n_E, nT = ctx->n_T;
    const bool nonuni = !log_uniform(ctx->Eg);
    const size_t base_words = (size_t)nm * nE * 4 + nE + (size_t)nm * nT * 4 + nm;
    std::vector<float> blob(base_words + (nonuni ? (size_t)nE + kEGuide + 1 : 0), 0.0f);
    float* phot = blob.data();
    float* maj = phot + (size_t)nm * nE * 4;
    float* lnS = maj + nE;
    float* invX0 = lnS + (size_t)nm * nT;
    float* lnL = invX0 + nm;                       // mode 2: ln restricted stopping power, Moller cross section (cm^2/g)
    float* sig = lnL + (size_t)nm * nT;
    float* sigb = sig + (size_t)nm * nT;           // mode 3: the bremsstrahlung part of sig
    for (int m = 0; m < nm; ++m)
        for (int j = 0; j < nE; ++j) {
            const size_t o = (size_t)m * nE + j;
            phot[o * 4 + 0] = (float)std::log(std::max((double)ctx->muPE[o], 1e-37));
            phot[o * 4 + 1] = (float)std::log(std::max((double)ctx->muC[o], 1e-37));
            phot[o * 4 + 2] = ctx->muPP[o];
            phot[o * 4 + 3] = 0.0f;
        }
    for (int j = 0; j < nE; ++j) {
        double mx = 1e-30;
        for (int m = 0; m < nm; ++m) {
            const double r = m < (int)ctx->rho_max.size() ? ctx->rho_max[m] : 0.0;
            if (r <= 0) continue;
            const size_t o = (size_t)m * nE + j;
            mx = std::max(mx, r * ((double)ctx->muPE[o] + ctx->muC[o] + ctx->muPP[o]));
        }
        maj[j] = (float)(mx * (1.0 + 1e-4));      // margin covers float32 rounding of the fast exp / log path
    }
    for (int m = 0; m < nm; ++m) {
        for (int j = 0; j < nT; ++j) lnS[(size_t)m * nT + j] = (float)std::log(std::max((double)ctx->S[(size_t)m * nT + j], 1e-37));
        invX0[m] = 1.0f / ctx->X0[m];
    }
    // Body box (params.h Geom::glo).  kfac[m] = max_j mu_tot,m(E_j) / maj_j: a voxel (rho, m) attenuates at most
    // rho kfac[m] maj(E) at EVERY energy, by the argument of reading A7 (each material's interpolant lies below the chord of its
    // node values, the chord of rho kfac[m] maj_j is rho kfac[m] times the majorant's interpolant).  B = bounding box of the
    // voxels with rho kfac > kBodyThr; f_out = the largest rho kfac outside B.
    {
        constexpr float kBodyThr = 0.05f;
        float kfac[kMaxMat] = {0};
        for (int m = 0; m < nm && m < kMaxMat; ++m)
            for (int j = 0; j < nE; ++j) {
                const size_t o = (size_t)m * nE + j;
                kfac[m] = std::max(kfac[m], (float)(((double)ctx->muPE[o] + ctx->muC[o] + ctx->muPP[o]) / (double)maj[j] * (1.0 + 1e-6)));
            }
        Geom& g = ctx->g;
        CU(cudaMemcpyAsync(ctx->d_kfac(), kfac, sizeof(kfac), cudaMemcpyHostToDevice, ctx->stream));
        launch_body_box(ctx->d_vox(), g.nx, g.ny, g.nz, ctx->d_kfac(), kBodyThr, ctx->d_body_box(), reinterpret_cast<unsigned int*>(ctx->d_body_box() + 6), ctx->stream);
        CU(cudaGetLastError());
        int box[7];
        CU(cudaMemcpyAsync(box, ctx->d_body_box(), sizeof(box), cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
        const int nn[3] = {g.nx, g.ny, g.nz};
        const float lo[3] = {g.lox, g.loy, g.loz}, hi[3] = {g.hix, g.hiy, g.hiz}, h[3] = {g.hx, g.hy, g.hz};
        for (int a = 0; a < 3; ++a) {
            if (box[3 + a] < box[a]) { g.glo[a] = g.ghi[a] = lo[a]; continue; }            // no voxel above the threshold: G is empty
            const int i0 = std::max(box[a] - 1, 0), i1 = std::min(box[3 + a] + 2, nn[a]);   // one voxel of cushion: a point that rounding puts
            g.glo[a] = i0 == 0 ? lo[a] : lo[a] + (float)i0 * h[a];                           // on the wrong side of a face of G is still outside B
            g.ghi[a] = i1 == nn[a] ? hi[a] : lo[a] + (float)i1 * h[a];
        }
        float fo; std::memcpy(&fo, &box[6], 4);
        g.f_out = std::min(std::max(fo, 1e-6f), 1.0f);
    }
    if (ctx->have_ne)
        for (int m = 0; m < nm; ++m)
            for (int j = 0; j < nT; ++j) {
                double sg, hd;
                moller_integrals((double)ctx->Tg[j], (double)ctx->ph.ecut, sg, hd);
                const size_t o = (size_t)m * nT + j;
                double bs = 0.0, bsoft = 0.0;                  // mode 3 (reading A32): photons above the photon cut-off, soft radiative loss
                if (ctx->ph.mode == 3) {
                    const double T = ctx->Tg[j], kc = ctx->ph.pcut, X0 = ctx->X0[m], lo = kc / T;
                    if (T > kc) {
                        bs = (4.0 / 3.0 * std::log(1.0 / lo) - 4.0 / 3.0 * (1.0 - lo) + 0.5 * (1.0 - lo * lo)) / X0;
                        bsoft = T * (4.0 / 3.0 * lo - 2.0 / 3.0 * lo * lo + lo * lo * lo / 3.0) / X0;
                    } else bsoft = T / X0;
                }
                lnL[o] = (float)std::log(std::max((double)ctx->S[o] - (double)ctx->ne[m] * hd + bsoft, 1e-37));
                sig[o] = (float)((double)ctx->ne[m] * sg + bs);
                sigb[o] = (float)bs;
            }
    // A photon grid that is not log-uniform (a real tabulation: irregular spacing, refined around absorption edges): the kernel
    // finds the cell from a guide table that is uniform in ln E, then interpolates exactly as on a uniform grid.
    ctx->tb.nonuni_E = nonuni ? 1 : 0; ctx->tb.inv_dg = 0.0f; ctx->tb.lnEg_off = (int)base_words;
    if (nonuni) {
        float* lnEg = blob.data() + base_words;
        uint32_t* guide = reinterpret_cast<uint32_t*>(lnEg + nE);
        for (int j = 0; j < nE; ++j) lnEg[j] = (float)std::log((double)ctx->Eg[j]);
        const double l0 = lnEg[0], span = (double)lnEg[nE - 1] - l0;
        ctx->tb.inv_dg = (float)(kEGuide / span);
        int i = 0;
        for (int k = 0; k <= kEGuide; ++k) {       // the cell of the bucket's left edge, taken a hair to the left so that float rounding
            const float x = (float)(l0 + (k - 1e-3) * span / kEGuide);   // of the bucket index never starts the search past the cell
            while (i < nE - 2 && lnEg[i + 1] <= x) ++i;
            guide[k] = (uint32_t)i;
        }
    }
    CU(cudaMemcpyAsync(ctx->d_blob(), blob.data(), blob.size() * 4, cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));       // blob is a local vector
    ctx->tb.n_mat = nm; ctx->tb.n_E = nE; ctx->tb.n_T = nT;
    ctx->tb.lnE0 = (float)std::log((double)ctx->Eg[0]);
    ctx->tb.inv_dlnE = (float)((nE - 1) / (std::log((double)ctx->Eg[nE - 1]) - std::log((double)ctx->Eg[0])));
    ctx->tb.lnT0 = (float)std::log((double)ctx->Tg[0]);
    ctx->tb.inv_dlnT = (float)((nT - 1) / (std::log((double)ctx->Tg[nT - 1]) - std::log((double)ctx->Tg[0])));
    ctx->tb.blob = ctx->d_blob();
    ctx->tb.blob_words = (int)blob.size();
    ctx->tables_dirty = false;
    return 0;
}

int check_geometry(aepid_ctx* ctx) {
    const Geom& g = ctx->g;
    for (int k = 0; k < 8; ++k) {
        const double p[3] = {(k & 1) ? g.hix : g.lox, (k & 2) ? g.hiy : g.loy, (k & 4) ? g.hiz : g.loz};
        const double r[3] = {p[0] - g.src[0], p[1] - g.src[1], p[2] - g.src[2]};
        const double u = g.au[0] * r[0] + g.au[1] * r[1] + g.au[2] * r[2];
        const double v = g.av[0] * r[0] + g.av[1] * r[1] + g.av[2] * r[2];
        const double w = g.aw[0] * r[0] + g.aw[1] * r[1] + g.aw[2] * r[2];
        if (std::fabs(u) >= kWorldHalf || std::fabs(v) >= kWorldHalf || w <= kWorldWMin || w >= g.sid)
            return fail(ctx, AEPID_ERR_GEOMETRY, "phantom reaches outside the air region of the world box (|u|,|v| < 100 cm, -1 < w < sid)");
    }
    if (g.src[0] >= g.lox && g.src[0] < g.hix && g.src[1] >= g.loy && g.src[1] < g.hiy && g.src[2] >= g.loz && g.src[2] < g.hiz)
        return fail(ctx, AEPID_ERR_GEOMETRY, "source lies inside the phantom");
    return 0;
}

int fill_params(aepid_ctx* ctx, TransportParams& p) {
    if (!ctx->have_mat) return fail(ctx, AEPID_ERR_BAD_STATE, "aepid_init_materials has not been called");
    if (!ctx->have_phantom) return fail(ctx, AEPID_ERR_BAD_STATE, "aepid_load_phantom has not been called");
    if (!ctx->have_epid) return fail(ctx, AEPID_ERR_BAD_STATE, "aepid_load_epid_layers has not been called");
    if (!ctx->have_source) return fail(ctx, AEPID_ERR_BAD_STATE, "aepid_load_source has not been called");
    if (ctx->ph.mode >= 2 && !ctx->have_ne) return fail(ctx, AEPID_ERR_BAD_STATE, "physics modes 2 and 3 need aepid_set_class2 (after aepid_init_materials)");
    if (int rc = check_geometry(ctx)) return rc;
    for (int l = 0; l < ctx->g.n_layers; ++l)
        if (ctx->g.lmat[l] >= ctx->n_mat) return fail(ctx, AEPID_ERR_BAD_ARG, "EPID layer material index out of range");
    if (ctx->tables_dirty) if (int rc = build_tables(ctx)) return rc;
    if (transport_smem_bytes(ctx->tb) > 227 * 1024) return fail(ctx, AEPID_ERR_NOMEM, "material tables do not fit in shared memory");
    p.g = ctx->g; p.ph = ctx->ph; p.tb = ctx->tb; p.so = ctx->so;
    p.vox = ctx->d_vox(); p.ep_batch = ctx->d_ep_batch(); p.ph_batch = ctx->d_ph_batch();
    p.ledger = ctx->d_ledger(); p.counters = ctx->d_counters(); p.hist_counter = ctx->d_chunk();
    p.queues = reinterpret_cast<uint4*>(ctx->ws + ctx->lay.queues);
    p.n_batches = ctx->dims.n_batches; p.nvox = ctx->lay.nvox; p.npix = ctx->lay.npix; p.live_max = ctx->live_max;
    // physics mode 4 carries 64-byte records (the leg's energy budget): half as many fit the class queues
    p.pool_log = ctx->ph.mode == 4 ? ctx->pool_log - 1 : ctx->pool_log;
    if (ctx->ph.mode == 4) p.live_max = std::min(p.live_max, (1 << p.pool_log) / 2);
    p.hd = ctx->hd; p.hd.stats = ctx->d_head_stats(); p.hd.ps1 = ctx->d_ps1();
    p.hd.lo = ctx->d_head_rows(); p.hd.hi = ctx->d_head_rows() + kMaxHeadRows;
    if (p.hd.n_slabs > 0 && p.hd.n_ps1 == 0) return fail(ctx, AEPID_ERR_BAD_STATE, "a collimator needs a phase-space source (aepid_load_phase_space_source)");
    if (p.hd.n_slabs > 0 && p.hd.mat >= ctx->n_mat) return fail(ctx, AEPID_ERR_BAD_ARG, "collimator material index out of range");
    if (p.hd.n_slabs == 0) p.hd.w_ps2 = p.hd.w_ps1;
    if (p.hd.n_ps1 != 0 && !(p.hd.w_ps2 < ctx->g.sid)) return fail(ctx, AEPID_ERR_GEOMETRY, "Phase Space 2 plane below the EPID");
    p.ps3 = ctx->ps3; p.ps3_count = ctx->d_ps3_count(); p.ps3_cap = ctx->ps3 ? ctx->ps3_cap : 0;
    p.base = 0; set_seed(p, 0); p.n = 0; p.hist_per_batch = 1;
    return 0;
}

}  // namespace

extern "C" {

size_t aepid_workspace_bytes(const aepid_dims* dims) {
    if (!dims_ok(dims)) return 0;
    return make_layout(*dims).total;
}

int aepid_create(aepid_ctx** out, int device, void* cuda_stream, const aepid_dims* dims, void* workspace, size_t workspace_bytes) {
    if (!out) return AEPID_ERR_BAD_ARG;
    *out = nullptr;
    aepid_ctx* ctx = new aepid_ctx();
    *out = ctx;                                   // returned even on failure so that aepid_last_error works
    if (!dims_ok(dims)) return fail(ctx, AEPID_ERR_BAD_ARG, "dims out of range");
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev <= 0) { cudaGetLastError(); return fail(ctx, AEPID_ERR_CUDA, "no CUDA device: this library has no CPU fallback"); }
    if (device < 0 || device >= n_dev) return fail(ctx, AEPID_ERR_BAD_ARG, "device index out of range");
    CU(cudaSetDevice(device));
    cudaDeviceProp prop{};
    CU(cudaGetDeviceProperties(&prop, device));
    ctx->device = device; ctx->sm_count = prop.multiProcessorCount;
    ctx->stream = (cudaStream_t)cuda_stream;
    ctx->dims = *dims; ctx->lay = make_layout(*dims);
    ctx->pool_log = pool_log_for(*dims); ctx->live_max = (1 << ctx->pool_log) / 2;
    if (!workspace || ((uintptr_t)workspace & (kAlign - 1))) return fail(ctx, AEPID_ERR_BAD_ARG, "workspace must be a 256-byte aligned device pointer");
    if (classify(workspace) != MEM_DEVICE) return fail(ctx, AEPID_ERR_BAD_ARG, "workspace is not device memory");
    if (workspace_bytes < ctx->lay.total) return fail(ctx, AEPID_ERR_NOMEM, "workspace smaller than aepid_workspace_bytes(dims)");
    ctx->ws = static_cast<char*>(workspace);
    return reset_tallies(ctx);
}

void aepid_destroy(aepid_ctx* ctx) { delete ctx; }

const char* aepid_last_error(const aepid_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }

int aepid_synchronize(aepid_ctx* ctx) {
    if (!ctx) return AEPID_ERR_BAD_ARG;
    double led[8] = {0};
    if (ctx->ws) CU(cudaMemcpyAsync(led, ctx->d_ledger(), sizeof(led), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return check_internal(ctx, led);
}

int aepid_init_materials(aepid_ctx* ctx, int n_mat, int n_E, const float* E, const float* muC, const float* muPE, const float* muPP,
                         int n_T, const float* T, const float* S, const float* X0) {
    if (!ctx || !ctx->ws) return AEPID_ERR_BAD_STATE;
    if (!E || !muC || !muPE || !muPP || !T || !S || !X0) return fail(ctx, AEPID_ERR_BAD_ARG, "null table pointer");
    if (n_mat < 1 || n_E < 2 || n_T < 2) return fail(ctx, AEPID_ERR_BAD_ARG, "table sizes out of range");
    if (n_mat > ctx->dims.n_mat || n_E > ctx->dims.n_E || n_T > ctx->dims.n_T) return fail(ctx, AEPID_ERR_NOMEM, "tables exceed dims");
    if (int rc = fetch(ctx, E, (size_t)n_E, ctx->Eg)) return rc;
    if (int rc = fetch(ctx, T, (size_t)n_T, ctx->Tg)) return rc;
    if (int rc = fetch(ctx, muC, (size_t)n_mat * n_E, ctx->muC)) return rc;
    if (int rc = fetch(ctx, muPE, (size_t)n_mat * n_E, ctx->muPE)) return rc;
    if (int rc = fetch(ctx, muPP, (size_t)n_mat * n_E, ctx->muPP)) return rc;
    if (int rc = fetch(ctx, S, (size_t)n_mat * n_T, ctx->S)) return rc;
    if (int rc = fetch(ctx, X0, (size_t)n_mat, ctx->X0)) return rc;
    for (int j = 0; j < n_E; ++j) if (!(ctx->Eg[j] > 0) || (j && !(ctx->Eg[j] > ctx->Eg[j - 1]))) return fail(ctx, AEPID_ERR_BAD_ARG, "photon energy grid must be positive and strictly increasing");
    if (!log_uniform(ctx->Tg)) return fail(ctx, AEPID_ERR_BAD_ARG, "the electron energy grid must be increasing and log-uniform (the photon grid may be any increasing grid)");
    for (float v : ctx->muC) if (!(v >= 0)) return fail(ctx, AEPID_ERR_BAD_ARG, "negative or NaN cross section");
    for (float v : ctx->muPE) if (!(v >= 0)) return fail(ctx, AEPID_ERR_BAD_ARG, "negative or NaN cross section");
    for (float v : ctx->muPP) if (!(v >= 0)) return fail(ctx, AEPID_ERR_BAD_ARG, "negative or NaN cross section");
    for (float v : ctx->S) if (!(v > 0)) return fail(ctx, AEPID_ERR_BAD_ARG, "stopping power must be positive");
    for (float v : ctx->X0) if (!(v > 0)) return fail(ctx, AEPID_ERR_BAD_ARG, "radiation length must be positive");
    ctx->n_mat = n_mat; ctx->n_E = n_E; ctx->n_T = n_T;
    ctx->have_mat = true; ctx->tables_dirty = true; ctx->have_ne = false;
    return 0;
}

int aepid_load_phantom(aepid_ctx* ctx, int nx, int ny, int nz, const float sp[3], const float org[3],
                       const float* rho, const unsigned char* mat) {
    if (!ctx || !ctx->ws) return AEPID_ERR_BAD_STATE;
    if (!ctx->have_mat) return fail(ctx, AEPID_ERR_BAD_STATE, "aepid_init_materials must come first");
    if (!sp || !org || !rho || !mat) return fail(ctx, AEPID_ERR_BAD_ARG, "null phantom pointer");
    if (nx < 1 || ny < 1 || nz < 1 || !(sp[0] > 0) || !(sp[1] > 0) || !(sp[2] > 0)) return fail(ctx, AEPID_ERR_BAD_ARG, "bad grid");
    if (nx != ctx->dims.nx || ny != ctx->dims.ny || nz != ctx->dims.nz) return fail(ctx, AEPID_ERR_NOMEM, "phantom grid differs from dims");
    const size_t n = (size_t)nx * ny * nz;
    const MemKind kr = classify(rho), km = classify(mat);
    const float* d_rho = rho; const unsigned char* d_mat = mat;
    // host inputs are staged in the (about to be zeroed) phantom batch buffers: B >= 2 gives 8 bytes per voxel
    char* stage = reinterpret_cast<char*>(ctx->d_ph_batch());
    if (kr != MEM_DEVICE) { CU(cudaMemcpyAsync(stage, rho, n * 4, cudaMemcpyHostToDevice, ctx->stream)); d_rho = reinterpret_cast<const float*>(stage); }
    if (km != MEM_DEVICE) { CU(cudaMemcpyAsync(stage + n * 4, mat, n, cudaMemcpyHostToDevice, ctx->stream)); d_mat = reinterpret_cast<const unsigned char*>(stage + n * 4); }
    launch_pack_voxels(d_rho, d_mat, ctx->d_vox(), n, ctx->d_rho_max(), ctx->n_mat, ctx->d_bad_mat(), ctx->stream);
    CU(cudaGetLastError());
    ctx->rho_max.assign(kMaxMat, 0.0f);
    unsigned int bad = 0;
    CU(cudaMemcpyAsync(ctx->rho_max.data(), ctx->d_rho_max(), kMaxMat * 4, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaMemcpyAsync(&bad, ctx->d_bad_mat(), sizeof(bad), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    if (bad) { ctx->have_phantom = false; return fail(ctx, AEPID_ERR_BAD_ARG, "material index out of range in the phantom (a material byte >= n_mat)"); }
    Geom& g = ctx->g;
    g.nx = nx; g.ny = ny; g.nz = nz;
    g.hx = sp[0]; g.hy = sp[1]; g.hz = sp[2];
    g.ihx = 1.0f / sp[0]; g.ihy = 1.0f / sp[1]; g.ihz = 1.0f / sp[2];
    g.lox = org[0]; g.loy = org[1]; g.loz = org[2];
    g.hix = org[0] + nx * sp[0]; g.hiy = org[1] + ny * sp[1]; g.hiz = org[2] + nz * sp[2];
    ctx->have_phantom = true; ctx->tables_dirty = true;
    return reset_tallies(ctx);
}

int aepid_load_epid_layers(aepid_ctx* ctx, int nl, const float* th, const unsigned char* mat, const float* rho,
                           const unsigned char* scored, float sid, int nu, int nv, float pitch) {
    if (!ctx || !ctx->ws) return AEPID_ERR_BAD_STATE;
    if (!th || !mat || !rho || !scored) return fail(ctx, AEPID_ERR_BAD_ARG, "null layer pointer");
    if (nl < 1 || nl > ctx->dims.n_layers) return fail(ctx, AEPID_ERR_NOMEM, "layer count exceeds dims");
    if (nu != ctx->dims.nu || nv != ctx->dims.nv) return fail(ctx, AEPID_ERR_NOMEM, "EPID image differs from dims");
    if (!(pitch > 0) || !(sid > 0)) return fail(ctx, AEPID_ERR_BAD_ARG, "pitch and sid must be positive");
    Geom& g = ctx->g;
    g.n_layers = nl; g.nu = nu; g.nv = nv; g.sid = sid; g.pitch = pitch; g.inv_pitch = 1.0f / pitch;
    g.half_u = 0.5f * nu * pitch; g.half_v = 0.5f * nv * pitch;
    double z = 0.0; g.zt[0] = 0.0f;
    for (int l = 0; l < nl; ++l) {
        if (!(th[l] > 0) || !(rho[l] > 0)) return fail(ctx, AEPID_ERR_BAD_ARG, "layer thickness and density must be positive");
        z += th[l]; g.zt[l + 1] = (float)z;
        g.lrho[l] = rho[l]; g.lmat[l] = mat[l]; g.lscored[l] = scored[l] ? 1 : 0;
    }
    for (int l = nl; l < kMaxLayers; ++l) { g.zt[l + 1] = g.zt[nl]; g.lrho[l] = 1.0f; g.lmat[l] = 0; g.lscored[l] = 0; }
    ctx->have_epid = true;
    return 0;
}

int aepid_load_source(aepid_ctx* ctx, const float src[3], const float axes[9], int nb, const float* edges, const float* pdf,
                      int fu, int fv, float fpitch, float fdist, const float* fluence) {
    if (!ctx || !ctx->ws) return AEPID_ERR_BAD_STATE;
    if (!src || !axes || !edges || !pdf || !fluence) return fail(ctx, AEPID_ERR_BAD_ARG, "null source pointer");
    if (nb < 1 || fu < 1 || fv < 1 || !(fpitch > 0) || !(fdist > 0)) return fail(ctx, AEPID_ERR_BAD_ARG, "bad source sizes");
    if (nb > ctx->dims.n_bins || (size_t)fu * fv > (size_t)ctx->dims.fu * ctx->dims.fv) return fail(ctx, AEPID_ERR_NOMEM, "source exceeds dims");
    for (int r = 0; r < 3; ++r) {                          // rows must be orthonormal
        for (int q = r; q < 3; ++q) {
            const double d = (double)axes[3 * r] * axes[3 * q] + (double)axes[3 * r + 1] * axes[3 * q + 1] + (double)axes[3 * r + 2] * axes[3 * q + 2];
            if (std::fabs(d - (r == q ? 1.0 : 0.0)) > 1e-4) return fail(ctx, AEPID_ERR_BAD_ARG, "beam_axes rows are not orthonormal");
        }
    }
    std::vector<float> he, hp, hf;
    if (int rc = fetch(ctx, edges, (size_t)nb + 1, he)) return rc;
    if (int rc = fetch(ctx, pdf, (size_t)nb, hp)) return rc;
    if (int rc = fetch(ctx, fluence, (size_t)fu * fv, hf)) return rc;
    // integer thresholds on the raw draw r: bin = #{k >= 1 : (r + 0.5) 2^-32 * total >= cdf[k]}
    auto thresholds = [](const std::vector<float>& w, std::vector<uint32_t>& thr, double& total) {
        const size_t n = w.size();
        std::vector<double> cdf(n + 1, 0.0);
        for (size_t i = 0; i < n; ++i) { if (!(w[i] >= 0)) return false; cdf[i + 1] = cdf[i] + (double)w[i]; }
        total = cdf[n];
        if (!(total > 0)) return false;
        thr.resize(n + 1);
        for (size_t k = 0; k <= n; ++k) {
            const double t = std::ceil(cdf[k] / total * 4294967296.0 - 0.5);
            thr[k] = t <= 0 ? 0u : (t >= 4294967295.0 ? 0xFFFFFFFFu : (uint32_t)t);
        }
        return true;
    };
    std::vector<uint32_t> tE, tF; double totE = 0, totF = 0;
    if (!thresholds(hp, tE, totE)) return fail(ctx, AEPID_ERR_BAD_ARG, "spectrum pdf must be non-negative with a positive sum");
    if (!thresholds(hf, tF, totF)) return fail(ctx, AEPID_ERR_BAD_ARG, "fluence must be non-negative with a positive sum");
    tE[nb] = 0u;                                           // 2^32 mod 2^32: widths come out right by wrap-around
    // guide table of the fluence search: guide[k] = #{j < n : thrF[1 + j] <= k 2^(32 - kGuideLog)}, so that the upper
    // bound of a draw r lies in [guide[r >> s], guide[(r >> s) + 1]] and the search touches 2-3 words instead of 16
    std::vector<uint32_t> gF((size_t)kGuideSize + 1);
    {
        const size_t n = (size_t)fu * fv - 1;
        size_t j = 0;
        for (int k = 0; k < kGuideSize; ++k) {
            const uint32_t key = (uint32_t)k << (32 - kGuideLog);
            while (j < n && tF[1 + j] <= key) ++j;
            gF[k] = (uint32_t)j;
        }
        gF[kGuideSize] = (uint32_t)n;
    }
    int j_last = 0;
    ctx->bb_u0 = fu; ctx->bb_u1 = -1; ctx->bb_v0 = fv; ctx->bb_v1 = -1;
    for (int j = 0; j < fv; ++j) for (int i = 0; i < fu; ++i)
        if (hf[(size_t)j * fu + i] > 0) {
            j_last = j * fu + i;
            ctx->bb_u0 = std::min(ctx->bb_u0, i); ctx->bb_u1 = std::max(ctx->bb_u1, i);
            ctx->bb_v0 = std::min(ctx->bb_v0, j); ctx->bb_v1 = std::max(ctx->bb_v1, j);
        }
    CU(cudaMemcpyAsync(ctx->d_thrE(), tE.data(), tE.size() * 4, cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemcpyAsync(ctx->d_edges(), he.data(), he.size() * 4, cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemcpyAsync(ctx->d_thrF(), tF.data(), tF.size() * 4, cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemcpyAsync(ctx->d_guideF(), gF.data(), gF.size() * 4, cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));                // sources are local vectors
    Geom& g = ctx->g;
    for (int k = 0; k < 3; ++k) { g.src[k] = src[k]; g.au[k] = axes[k]; g.av[k] = axes[3 + k]; g.aw[k] = axes[6 + k]; }
    Source& so = ctx->so;
    so.n_bins = nb; so.fu = fu; so.fv = fv; so.j_last = j_last; so.fpitch = fpitch; so.fdist = fdist;
    so.thrE = ctx->d_thrE(); so.edges = ctx->d_edges(); so.thrF = ctx->d_thrF(); so.guideF = ctx->d_guideF();
    ctx->have_source = true;
    return 0;
}

int aepid_set_physics(aepid_ctx* ctx, int mode, float pcut, float ecut, float fE, float smax) {
    if (!ctx) return AEPID_ERR_BAD_ARG;
    if (mode < 0 || mode > 4 || !(pcut > 0) || !(ecut > 0) || !(fE > 0) || !(fE <= 0.5f) || !(smax > 0)) return fail(ctx, AEPID_ERR_BAD_ARG, "physics parameters out of range");
    if (ecut != ctx->ph.ecut || pcut != ctx->ph.pcut || mode != ctx->ph.mode) ctx->tables_dirty = true;   // the restricted stopping powers depend on the cut-offs and the mode
    ctx->ph.mode = mode; ctx->ph.pcut = pcut; ctx->ph.ecut = ecut; ctx->ph.fE = fE; ctx->ph.smax = smax;
    return 0;
}

int aepid_reset_tallies(aepid_ctx* ctx) {
    if (!ctx || !ctx->ws) return AEPID_ERR_BAD_STATE;
    return reset_tallies(ctx);
}

int aepid_set_counting(aepid_ctx* ctx, int on) { if (!ctx) return AEPID_ERR_BAD_ARG; ctx->counting = on != 0; return 0; }

int aepid_simulate(aepid_ctx* ctx, unsigned long long n_histories, unsigned long long seed) {
    if (!ctx || !ctx->ws) return AEPID_ERR_BAD_STATE;
    TransportParams p{};
    if (int rc = fill_params(ctx, p)) return rc;
    const int B = ctx->dims.n_batches;
    unsigned long long left = n_histories;
    while (left > 0) {
        const unsigned long long n = std::min<unsigned long long>(left, 1ull << 31);
        p.base = ctx->first_history + ctx->n_done; set_seed(p, seed); p.n = (uint32_t)n;
        const uint64_t hpb = (n + B - 1) / B;                  // history k of the launch -> batch k / hpb, exactly as in the kernel
        p.hist_per_batch = (uint32_t)hpb;
        CU(cudaMemsetAsync(ctx->d_chunk(), 0, sizeof(unsigned int), ctx->stream));
        const int rc = launch_transport(p, ctx->counting, ctx->sm_count, ctx->stream);
        if (rc != 0) return fail(ctx, AEPID_ERR_CUDA, std::string("transport launch: ") + cudaGetErrorString((cudaError_t)rc));
        for (int b = 0; b < B; ++b) {
            const uint64_t h0 = std::min<uint64_t>((uint64_t)b * hpb, n), h1 = std::min<uint64_t>((uint64_t)(b + 1) * hpb, n);
            ctx->hist[b] += (double)(h1 - h0);
        }
        ctx->n_done += n; left -= n;
    }
    return 0;
}

int aepid_read_tallies(aepid_ctx* ctx, float* ep_mean, float* ep_sigma, float* ph_mean, float* ph_sigma, double ledger[8]) {
    if (!ctx || !ctx->ws) return AEPID_ERR_BAD_STATE;
    bool need_sync = false;
    auto fold = [&](const float* batches, size_t n, float* mean, float* sigma, float* scratch) -> int {
        if (!mean && !sigma) return 0;
        FoldParams f{};
        f.batches = batches; f.n = n; f.n_batches = ctx->dims.n_batches; f.total = (double)ctx->n_done;
        std::copy(ctx->hist, ctx->hist + 256, f.hist);
        const bool dm = mean && classify(mean) == MEM_DEVICE, ds = sigma && classify(sigma) == MEM_DEVICE;
        f.mean = mean ? (dm ? mean : scratch) : nullptr;
        f.sigma = sigma ? (ds ? sigma : scratch + n) : nullptr;
        launch_fold(f, ctx->stream);
        CU(cudaGetLastError());
        if (mean && !dm) if (int rc = deliver(ctx, mean, scratch, n * 4, &need_sync)) return rc;
        if (sigma && !ds) if (int rc = deliver(ctx, sigma, scratch + n, n * 4, &need_sync)) return rc;
        return 0;
    };
    if (int rc = fold(ctx->d_ep_batch(), ctx->lay.npix, ep_mean, ep_sigma, ctx->d_out_ep())) return rc;
    if (int rc = fold(ctx->d_ph_batch(), ctx->lay.nvox, ph_mean, ph_sigma, ctx->d_out_ph())) return rc;
    double led[8] = {0};
    if (ledger) need_sync = true;
    if (need_sync) {                                       // the call synchronises anyway: look at the kernel's error flags too
        CU(cudaMemcpyAsync(led, ctx->d_ledger(), sizeof(led), cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
    }
    if (ledger) { std::copy(led, led + 8, ledger); ledger[6] = (double)ctx->n_done; }
    return need_sync ? check_internal(ctx, led) : 0;
}

int aepid_set_history_offset(aepid_ctx* ctx, unsigned long long first_history) {
    if (!ctx) return AEPID_ERR_BAD_ARG;
    if (ctx->n_done != 0) return fail(ctx, AEPID_ERR_BAD_STATE, "set the history offset right after aepid_reset_tallies");
    ctx->first_history = first_history;
    return 0;
}

int aepid_read_moments(aepid_ctx* ctx, double* ep_s1, double* ep_s2, double* ph_s1, double* ph_s2, double totals[2]) {
    if (!ctx || !ctx->ws) return AEPID_ERR_BAD_STATE;
    for (const double* q : {ep_s1, ep_s2, ph_s1, ph_s2})
        if (q && classify(q) != MEM_DEVICE) return fail(ctx, AEPID_ERR_BAD_ARG, "moment outputs must be device pointers");
    FoldParams f{};
    f.n_batches = ctx->dims.n_batches; f.total = (double)ctx->n_done;
    std::copy(ctx->hist, ctx->hist + 256, f.hist);
    if (ep_s1 || ep_s2) { f.batches = ctx->d_ep_batch(); f.n = ctx->lay.npix; launch_moments(f, ep_s1, ep_s2, ctx->stream); CU(cudaGetLastError()); }
    if (ph_s1 || ph_s2) { f.batches = ctx->d_ph_batch(); f.n = ctx->lay.nvox; launch_moments(f, ph_s1, ph_s2, ctx->stream); CU(cudaGetLastError()); }
    if (totals) {                                          // host output: synchronise and look at the kernel's error flags
        totals[0] = (double)ctx->n_done; totals[1] = 0.0;
        for (int b = 0; b < ctx->dims.n_batches; ++b) if (ctx->hist[b] > 0) totals[1] += 1.0;
        double led[8] = {0};
        CU(cudaMemcpyAsync(led, ctx->d_ledger(), sizeof(led), cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
        return check_internal(ctx, led);
    }
    return 0;
}

int aepid_finalize_moments(aepid_ctx* ctx, const double* s1, const double* s2, size_t n, double n_histories, double n_batches,
                           float* mean, float* sigma) {
    if (!ctx || !ctx->ws) return AEPID_ERR_BAD_STATE;
    if (!s1 || (sigma && !s2)) return fail(ctx, AEPID_ERR_BAD_ARG, "null moment pointer");
    for (const void* q : {(const void*)s1, (const void*)s2, (const void*)mean, (const void*)sigma})
        if (q && classify(q) != MEM_DEVICE) return fail(ctx, AEPID_ERR_BAD_ARG, "moment buffers must be device pointers");
    launch_finalize_moments(s1, s2, n, n_histories, n_batches, mean, sigma, ctx->stream);
    CU(cudaGetLastError());
    return 0;
}

int aepid_read_batches(aepid_ctx* ctx, float* epid_batches, double* histories_per_batch) {
    if (!ctx || !ctx->ws) return AEPID_ERR_BAD_STATE;
    bool need_sync = false;
    if (epid_batches) if (int rc = deliver(ctx, epid_batches, ctx->d_ep_batch(), ctx->lay.npix * 4 * ctx->dims.n_batches, &need_sync)) return rc;
    if (need_sync) CU(cudaStreamSynchronize(ctx->stream));
    if (histories_per_batch) std::copy(ctx->hist, ctx->hist + ctx->dims.n_batches, histories_per_batch);
    return 0;
}

int aepid_read_counters(aepid_ctx* ctx, unsigned long long counters[32]) {
    if (!ctx || !ctx->ws || !counters) return AEPID_ERR_BAD_ARG;
    CU(cudaMemcpyAsync(counters, ctx->d_counters(), 32 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return 0;
}

int aepid_sample_source(aepid_ctx* ctx, unsigned long long first, unsigned long long n, unsigned long long seed, float* out) {
    if (!ctx || !ctx->ws) return AEPID_ERR_BAD_STATE;
    if (!out) return fail(ctx, AEPID_ERR_BAD_ARG, "null output");
    if (!ctx->have_source) return fail(ctx, AEPID_ERR_BAD_STATE, "aepid_load_source has not been called");
    TransportParams p{};
    p.g = ctx->g; p.so = ctx->so; set_seed(p, seed);
    if (classify(out) == MEM_DEVICE) {
        launch_sample_source(p, first, n, out, ctx->stream);
        CU(cudaGetLastError());
        return 0;
    }
    const size_t cap = ctx->lay.nvox * 8 / 32;             // samples that fit in the phantom output scratch
    if (cap == 0) return fail(ctx, AEPID_ERR_NOMEM, "scratch too small");
    for (unsigned long long k = 0; k < n; k += cap) {
        const unsigned long long m = std::min<unsigned long long>(cap, n - k);
        launch_sample_source(p, first + k, m, ctx->d_out_ph(), ctx->stream);
        CU(cudaGetLastError());
        CU(cudaMemcpyAsync(out + 8 * k, ctx->d_out_ph(), m * 32, cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
    }
    return 0;
}

int aepid_field_size(aepid_ctx* ctx, int printed_form, float* s_cm) {
    if (!ctx || !s_cm) return AEPID_ERR_BAD_ARG;
    if (!ctx->have_source) return fail(ctx, AEPID_ERR_BAD_STATE, "aepid_load_source has not been called");
    if (ctx->bb_u1 < 0) { *s_cm = 0.0f; return 0; }
    const double sc = 100.0 / ctx->so.fdist;
    const double a = (ctx->bb_u1 - ctx->bb_u0 + 1) * (double)ctx->so.fpitch * sc, b = (ctx->bb_v1 - ctx->bb_v0 + 1) * (double)ctx->so.fpitch * sc;
    *s_cm = (float)(printed_form ? a * b / (2.0 * (a + b)) : 2.0 * a * b / (a + b));
    return 0;
}

int aepid_apply_response_lut(aepid_ctx* ctx, const float* lut, int nt, int ns, float t_min, float t_max, float s_min, float s_max,
                             float s_eff, const float* epid_in, float* signal_out, float* tmap_out) {
    if (!ctx || !ctx->ws) return AEPID_ERR_BAD_STATE;
    if (!lut || !signal_out) return fail(ctx, AEPID_ERR_BAD_ARG, "null lut or output");
    if (nt < 1 || ns < 1 || (size_t)nt * ns > kMaxLut) return fail(ctx, AEPID_ERR_BAD_ARG, "LUT size out of range");
    if ((nt > 1 && !(t_max > t_min)) || (ns > 1 && !(s_max > s_min))) return fail(ctx, AEPID_ERR_BAD_ARG, "LUT axes must be increasing");
    if (!ctx->have_phantom || !ctx->have_epid || !ctx->have_source) return fail(ctx, AEPID_ERR_BAD_STATE, "phantom, EPID and source must be loaded");
    const size_t n = ctx->lay.npix;
    bool need_sync = false;
    const float* d_lut = lut;
    if (classify(lut) != MEM_DEVICE) {
        CU(cudaMemcpyAsync(ctx->d_lut(), lut, (size_t)nt * ns * 4, cudaMemcpyHostToDevice, ctx->stream));
        if (classify(lut) == MEM_HOST_PINNED) need_sync = true;
        d_lut = ctx->d_lut();
    }
    if (s_eff < 0) if (int rc = aepid_field_size(ctx, 0, &s_eff)) return rc;
    launch_tmap(ctx->g, ctx->d_vox(), ctx->d_tmap(), ctx->stream);
    CU(cudaGetLastError());
    const float* d_dose;
    if (!epid_in) {
        FoldParams f{};
        f.batches = ctx->d_ep_batch(); f.n = n; f.n_batches = ctx->dims.n_batches; f.total = (double)ctx->n_done;
        std::copy(ctx->hist, ctx->hist + 256, f.hist);
        f.mean = ctx->d_dose_in(); f.sigma = nullptr;
        launch_fold(f, ctx->stream);
        CU(cudaGetLastError());
        d_dose = ctx->d_dose_in();
    } else if (classify(epid_in) == MEM_DEVICE) d_dose = epid_in;
    else {
        CU(cudaMemcpyAsync(ctx->d_dose_in(), epid_in, n * 4, cudaMemcpyHostToDevice, ctx->stream));
        if (classify(epid_in) == MEM_HOST_PINNED) need_sync = true;
        d_dose = ctx->d_dose_in();
    }
    const bool dev_out = classify(signal_out) == MEM_DEVICE;
    float* d_out = dev_out ? signal_out : ctx->d_signal();
    launch_apply_lut(d_lut, nt, ns, t_min, t_max, s_min, s_max, s_eff, d_dose, ctx->d_tmap(), d_out, n, ctx->stream);
    CU(cudaGetLastError());
    if (!dev_out) if (int rc = deliver(ctx, signal_out, d_out, n * 4, &need_sync)) return rc;
    if (tmap_out) if (int rc = deliver(ctx, tmap_out, ctx->d_tmap(), n * 4, &need_sync)) return rc;
    if (need_sync) CU(cudaStreamSynchronize(ctx->stream));
    return 0;
}

int aepid_set_class2(aepid_ctx* ctx, const float* electrons_per_gram) {
    if (!ctx || !ctx->ws) return AEPID_ERR_BAD_STATE;
    if (!ctx->have_mat) return fail(ctx, AEPID_ERR_BAD_STATE, "aepid_init_materials has not been called");
    if (!electrons_per_gram) return fail(ctx, AEPID_ERR_BAD_ARG, "null pointer");
    if (int rc = fetch(ctx, electrons_per_gram, (size_t)ctx->n_mat, ctx->ne)) return rc;
    for (float v : ctx->ne) if (!(v > 0)) return fail(ctx, AEPID_ERR_BAD_ARG, "electrons per gram must be positive");
    ctx->have_ne = true; ctx->tables_dirty = true;
    return 0;
}

int aepid_load_phase_space_source(aepid_ctx* ctx, unsigned long long n_records, const float* records, float w_plane_cm) {
    if (!ctx || !ctx->ws) return AEPID_ERR_BAD_STATE;
    if (n_records == 0) { ctx->hd.n_ps1 = 0; return 0; }                  // back to the fluence-map source
    if (!records) return fail(ctx, AEPID_ERR_BAD_ARG, "null records");
    if (n_records > (unsigned long long)ctx->dims.n_ps1) return fail(ctx, AEPID_ERR_NOMEM, "phase-space records exceed dims.n_ps1");
    if (!(w_plane_cm > kWorldWMin)) return fail(ctx, AEPID_ERR_GEOMETRY, "Phase Space 1 plane outside the world");
    CU(cudaMemcpyAsync(ctx->d_ps1(), records, (size_t)n_records * 32, classify(records) == MEM_DEVICE ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    ctx->hd.n_ps1 = (uint32_t)n_records; ctx->hd.w_ps1 = w_plane_cm;
    return 0;
}

int aepid_load_collimator(aepid_ctx* ctx, int n_slabs, const float* w0, const float* w1, const int* axis, const int* n_rows,
                          const float* row0, const float* pitch, const float* lo, const float* hi, int material, float density, float w_ps2) {
    if (!ctx || !ctx->ws) return AEPID_ERR_BAD_STATE;
    Head& H = ctx->hd;
    if (n_slabs == 0) { H.n_slabs = 0; return 0; }
    if (n_slabs < 0 || n_slabs > kMaxSlabs) return fail(ctx, AEPID_ERR_BAD_ARG, "at most 4 collimator slabs");
    if (!w0 || !w1 || !axis || !n_rows || !row0 || !pitch || !lo || !hi) return fail(ctx, AEPID_ERR_BAD_ARG, "null collimator pointer");
    if (material < 0 || material >= kMaxMat || !(density > 0)) return fail(ctx, AEPID_ERR_BAD_ARG, "bad collimator material or density");
    int total = 0; float prev = -1e30f;
    for (int k = 0; k < n_slabs; ++k) {
        if (!(w1[k] > w0[k]) || !(w0[k] >= prev) || n_rows[k] < 1 || !(pitch[k] > 0) || (axis[k] != 0 && axis[k] != 1))
            return fail(ctx, AEPID_ERR_BAD_ARG, "collimator slabs must be sorted along w, non-overlapping, with positive thickness and pitch");
        total += n_rows[k]; prev = w1[k];
    }
    if (total > kMaxHeadRows) return fail(ctx, AEPID_ERR_NOMEM, "more than 1024 collimator rows");
    if (!(w_ps2 >= prev)) return fail(ctx, AEPID_ERR_GEOMETRY, "Phase Space 2 plane above the last slab");
    CU(cudaMemcpyAsync(ctx->d_head_rows(), lo, (size_t)total * 4, cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemcpyAsync(ctx->d_head_rows() + kMaxHeadRows, hi, (size_t)total * 4, cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    int off = 0;
    for (int k = 0; k < n_slabs; ++k) {
        H.w0[k] = w0[k]; H.w1[k] = w1[k]; H.axis[k] = axis[k]; H.n_rows[k] = n_rows[k]; H.row0[k] = row0[k]; H.inv_pitch[k] = 1.0f / pitch[k];
        H.off[k] = off; off += n_rows[k];
    }
    H.n_slabs = n_slabs; H.mat = material; H.rho = density; H.w_ps2 = w_ps2;
    return 0;
}

int aepid_read_head(aepid_ctx* ctx, double out[4]) {
    if (!ctx || !ctx->ws) return AEPID_ERR_BAD_STATE;
    if (!out) return fail(ctx, AEPID_ERR_BAD_ARG, "null output");
    CU(cudaMemcpyAsync(out, ctx->d_head_stats(), 4 * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return 0;
}

int aepid_set_live_limit(aepid_ctx* ctx, int max_live_per_cta) {
    if (!ctx) return AEPID_ERR_BAD_ARG;
    const int cap = (1 << ctx->pool_log) / 2;
    if (max_live_per_cta == 0) max_live_per_cta = cap;
    if (max_live_per_cta < 64 || max_live_per_cta > cap) return fail(ctx, AEPID_ERR_BAD_ARG, "live limit out of range (64 .. half a class queue = dims.max_live_per_cta)");
    ctx->live_max = max_live_per_cta;
    return 0;
}

int aepid_set_phase_space(aepid_ctx* ctx, void* records, unsigned long long capacity) {
    if (!ctx || !ctx->ws) return AEPID_ERR_BAD_STATE;
    if (records && (classify(records) != MEM_DEVICE || ((uintptr_t)records & 15))) return fail(ctx, AEPID_ERR_BAD_ARG, "phase-space buffer must be 16-byte aligned device memory");
    if (records && capacity == 0) return fail(ctx, AEPID_ERR_BAD_ARG, "phase-space capacity is zero");
    ctx->ps3 = reinterpret_cast<float4*>(records); ctx->ps3_cap = records ? capacity : 0;
    CU(cudaMemsetAsync(ctx->d_ps3_count(), 0, 8, ctx->stream));
    return 0;
}

int aepid_read_phase_space_count(aepid_ctx* ctx, unsigned long long* n_arrived) {
    if (!ctx || !ctx->ws) return AEPID_ERR_BAD_STATE;
    if (!n_arrived) return fail(ctx, AEPID_ERR_BAD_ARG, "null output");
    CU(cudaMemcpyAsync(n_arrived, ctx->d_ps3_count(), 8, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return 0;
}

int aepid_roi_mean(aepid_ctx* ctx, const float* image, int nu, int nv, float pitch_cm, float roi_cm, double* mean_out) {
    if (!ctx || !ctx->ws) return AEPID_ERR_BAD_STATE;
    if (!mean_out) return fail(ctx, AEPID_ERR_BAD_ARG, "null output");
    if (!(roi_cm > 0)) return fail(ctx, AEPID_ERR_BAD_ARG, "ROI size must be positive");
    const float* d_img = image;
    if (!image) {                                                       // the current mean EPID image
        if (!ctx->have_epid) return fail(ctx, AEPID_ERR_BAD_STATE, "aepid_load_epid_layers has not been called");
        FoldParams f{};
        f.batches = ctx->d_ep_batch(); f.n = ctx->lay.npix; f.n_batches = ctx->dims.n_batches; f.total = (double)ctx->n_done;
        std::copy(ctx->hist, ctx->hist + 256, f.hist);
        f.mean = ctx->d_dose_in(); f.sigma = nullptr;
        launch_fold(f, ctx->stream);
        d_img = ctx->d_dose_in(); nu = ctx->g.nu; nv = ctx->g.nv; pitch_cm = ctx->g.pitch;
    } else {
        if (nu < 1 || nv < 1 || nu > 32768 || nv > 32768 || !(pitch_cm > 0)) return fail(ctx, AEPID_ERR_BAD_ARG, "image size or pitch out of range");
        if (classify(image) != MEM_DEVICE) return fail(ctx, AEPID_ERR_BAD_ARG, "aepid_roi_mean takes a device pointer (or NULL for the current image)");
    }
    launch_roi_sum(d_img, nu, nv, pitch_cm, roi_cm, ctx->d_gamma_stats(), ctx->stream);
    CU(cudaGetLastError());
    double h[2];
    CU(cudaMemcpyAsync(h, ctx->d_gamma_stats(), sizeof(h), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    *mean_out = h[1] > 0 ? h[0] / h[1] : std::nan("");
    return 0;
}

int aepid_upsample(aepid_ctx* ctx, const float* in, int nu, int nv, float* out, int mu, int mv) {
    if (!ctx || !ctx->ws) return AEPID_ERR_BAD_STATE;
    if (!in || !out) return fail(ctx, AEPID_ERR_BAD_ARG, "null image pointer");
    if (nu < 1 || nv < 1 || mu < 1 || mv < 1 || nu > 32768 || nv > 32768 || mu > 32768 || mv > 32768) return fail(ctx, AEPID_ERR_BAD_ARG, "image size out of range");
    if (classify(in) != MEM_DEVICE || classify(out) != MEM_DEVICE) return fail(ctx, AEPID_ERR_BAD_ARG, "aepid_upsample takes device pointers");
    launch_upsample(in, nu, nv, out, mu, mv, ctx->stream);
    CU(cudaGetLastError());
    return 0;
}

int aepid_gamma_index(aepid_ctx* ctx, const float* ref, const float* eval, int nu, int nv, float pitch_cm, float dose_frac, float dta_cm,
                      float threshold_frac, float gamma_cap, float* gamma_out, double stats[4]) {
    if (!ctx || !ctx->ws) return AEPID_ERR_BAD_STATE;
    if (!ref || !eval || !gamma_out) return fail(ctx, AEPID_ERR_BAD_ARG, "null image pointer");
    if (nu < 1 || nv < 1 || nu > 32768 || nv > 32768) return fail(ctx, AEPID_ERR_BAD_ARG, "image size out of range");
    if (!(pitch_cm > 0) || !(dose_frac > 0) || !(dta_cm > 0) || !(threshold_frac >= 0) || !(gamma_cap >= 1))
        return fail(ctx, AEPID_ERR_BAD_ARG, "gamma criteria out of range (pitch, dose fraction, DTA > 0; threshold >= 0; cap >= 1)");
    if (classify(ref) != MEM_DEVICE || classify(eval) != MEM_DEVICE || classify(gamma_out) != MEM_DEVICE)
        return fail(ctx, AEPID_ERR_BAD_ARG, "aepid_gamma_index takes device pointers for the images");
    if (launch_gamma(ref, eval, gamma_out, nu, nv, pitch_cm, dose_frac, dta_cm, threshold_frac, gamma_cap, ctx->d_gamma_max(),
                     ctx->d_gamma_stats(), ctx->stream) != 0)
        return fail(ctx, AEPID_ERR_NOMEM, "search window (cap x DTA / pitch pixels) does not fit in shared memory");
    CU(cudaGetLastError());
    if (stats) {
        double h[4];
        CU(cudaMemcpyAsync(h, ctx->d_gamma_stats(), sizeof(h), cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
        stats[0] = h[0]; stats[1] = h[1]; stats[2] = h[0] > 0 ? h[2] / h[0] : 0.0;
        stats[3] = h[3];                                               // kept on the device as the bit pattern of a non-negative double
    }
    return 0;
}

}  // extern "C"
