// Kernel parameter blocks shared by the host API (api.cu) and the kernels (transport.cu, postpass.cu).
// Plain structs, passed by value as __grid_constant__ kernel arguments.
#pragma once
#include <cstdint>
#include <cstddef>
#include <type_traits>
#include <vector_types.h>

namespace aepid {

constexpr int kMaxLayers = 8;
constexpr int kMaxMat = 32;
constexpr float kRhoAir = 1.205e-3f;  // world filler, material 0 (SURVEY 8(c) "Geometry")
constexpr float kWorldHalf = 100.0f;  // |u|, |v| <= 100 cm
constexpr float kWorldWMin = -1.0f;   // -1 <= w
constexpr float kMec2 = 0.51099895f;
#ifndef AEPID_POOL_LOG
#define AEPID_POOL_LOG 19
#endif
constexpr int kMaxPoolLog = AEPID_POOL_LOG;       // largest class queue: 2^19 records per class per CTA (262144 particles alive per CTA)
constexpr int kDefaultLive = 65536;               // aepid_dims.max_live_per_cta = 0
constexpr int kMaxPoolSlots = 1 << kMaxPoolLog;   // the size in force comes from aepid_dims.max_live_per_cta (TransportParams::pool_log)
constexpr int kRingCount = 5;         // class queues per CTA: the five event classes
constexpr int kRecordBytes = 48;      // three 16-byte vectors per particle
constexpr int kMaxCtas = 160;         // CTAs of the transport kernel the workspace provides class queues for (one per SM)
constexpr int kGuideLog = 12;         // the fluence search starts from a guide table indexed by the top kGuideLog bits of the draw
constexpr int kGuideSize = 1 << kGuideLog;

enum Region : uint32_t { R_AIR = 0, R_PHANTOM = 1, R_EPID = 2 };
enum PType : uint32_t { T_PHOTON = 0, T_ELECTRON = 1, T_POSITRON = 2 };

struct Geom {
    // phantom grid in the world frame
    int nx, ny, nz;
    float hx, hy, hz, ihx, ihy, ihz;
    float lox, loy, loz, hix, hiy, hiz;
    // Body box: an axis-aligned box G of whole voxels, one voxel wider on every side than the bounding box B of
    // the voxels whose attenuation can exceed a small fraction of the majorant; outside B no voxel exceeds f_out x majorant(E)
    // at any energy, so Woodcock flights outside G run against f_out x majorant (the margin of air around a patient costs no
    // virtual collisions).  An empty B gives glo == ghi.
    float glo[3], ghi[3], f_out;
    // beam frame
    float src[3], au[3], av[3], aw[3];
    // EPID slab stack; zt[] = depth of the layer tops below the EPID top plane (zt[0] = 0)
    int n_layers, nu, nv;
    float sid, pitch, inv_pitch, half_u, half_v;
    float zt[kMaxLayers + 1];
    float lrho[kMaxLayers];
    int lmat[kMaxLayers];
    int lscored[kMaxLayers];
};

struct Physics {
    int mode;                          // 0 kerma, 1 coupled
    float pcut, ecut, fE, smax;
};

// Table blob layout in global memory (copied verbatim into shared memory by every block):
//   float4 phot[n_mat][n_E]  = {ln mu_pe, ln mu_compton, mu_pair, 0}
//   float  maj[n_E]          majorant node values, safety margin included
//   float  lnS[n_mat][n_T]   ln stopping power
//   float  invX0[n_mat]
//   -- only if the photon grid is not log-uniform (nonuni_E) --
//   float  lnEg[n_E]         ln of the photon grid points
//   uint32 guide[kEGuide+1]  guide[k] = cell of the photon grid that holds ln E = lnE0 + k / inv_dg (start of the search)
constexpr int kEGuide = 1024;
struct Tables {
    int n_mat, n_E, n_T;
    float lnE0, inv_dlnE, lnT0, inv_dlnT;
    int nonuni_E;                      // the photon grid is an arbitrary increasing one: cell found through the guide table
    float inv_dg;                      // guide buckets per unit of ln E
    int lnEg_off;                      // word offset of lnEg in the blob (guide follows it)
    const uint32_t* blob;
    int blob_words;
};

struct Source {
    int n_bins, fu, fv, j_last;
    float fpitch, fdist;
    const uint32_t* thrE;              // [n_bins+1] integer CDF thresholds on the raw 32-bit draw
    const float* edges;                // [n_bins+1]
    const uint32_t* thrF;              // [fu*fv+1]
    const uint32_t* guideF;            // [kGuideSize+1] bracket of the search in thrF per top-bits bucket of the draw
};

// Collimation stage: Phase Space 1 records and tungsten slabs with per-row openings
// between the planes w = w_ps1 and w = w_ps2 of the beam frame (include/aepid.h: aepid_load_phase_space_source, aepid_load_collimator).
constexpr int kMaxSlabs = 4;
constexpr int kMaxHeadRows = 1024;     // rows (leaf pairs, jaw openings) over all slabs
struct Head {
    uint32_t n_ps1;                    // 0: fluence-map source
    float w_ps1;
    const float4* ps1;                 // [n_ps1][2] = {u, v, du, dv} {dw, E, -, -}
    int n_slabs, mat;                  // slabs sorted by w; material index and density of the jaws / leaves
    float rho, w_ps2;
    float w0[kMaxSlabs], w1[kMaxSlabs], row0[kMaxSlabs], inv_pitch[kMaxSlabs];
    int axis[kMaxSlabs], n_rows[kMaxSlabs], off[kMaxSlabs];
    const float* lo; const float* hi;  // openings of all rows, slab after slab
    double* stats;                     // [4]: Phase Space 2 particles, their energy, energy absorbed in the stage, unused
};

struct TransportParams {
    Geom g;
    Head hd;
    Physics ph;
    Tables tb;
    Source so;
    const uint32_t* vox;               // packed voxels: density (19 mantissa bits) | material (5 bits)
    float* ep_batch;                   // [B][nv*nu]
    float* ph_batch;                   // [B][nz*ny*nx]
    double* ledger;                    // [8]
    unsigned long long* counters;      // [32]
    unsigned int* hist_counter;        // next history of this launch that has not been started
    uint4* queues;                     // class queues of particle records [kMaxCtas][kRingCount][1 << pool_log][3], scratch of one launch
    int pool_log;                      // log2 of the records per class queue of a CTA
    float4* ps3;                       // Phase Space 3 records [ps3_cap][2] (null: not recorded), see aepid_set_phase_space
    unsigned long long* ps3_count;     // arrivals at the EPID top plane so far (also beyond the capacity)
    unsigned long long ps3_cap;
    uint64_t base;                     // global index of relative history 0 of this launch
    uint64_t seed;
    uint32_t rk[20];                   // Philox round keys of `seed` (set_seed): rk[2r], rk[2r+1] = key of round r
    uint32_t n;                        // histories in this launch (< 2^32)
    uint32_t hist_per_batch;           // history k of the launch scores into batch min(k / hist_per_batch, B - 1)
    int n_batches;
    int live_max;                      // most particles alive per CTA (<= half a class queue), aepid_set_live_limit
    size_t nvox, npix;
};

struct FoldParams {
    const float* batches;              // [B][n]
    size_t n;
    int n_batches;
    float* mean;                       // may be null
    float* sigma;                      // may be null
    double hist[256];                  // histories per batch
    double total;
};

inline void set_seed(TransportParams& p, uint64_t seed) {
    p.seed = seed;
    for (int r = 0; r < 10; ++r) { p.rk[2 * r] = (uint32_t)seed + 0x9E3779B9u * (uint32_t)r; p.rk[2 * r + 1] = (uint32_t)(seed >> 32) + 0xBB67AE85u * (uint32_t)r; }
}

// launchers (defined in transport.cu / postpass.cu)
int launch_transport(const TransportParams& p, bool counting, int sm_count, void* stream);
size_t transport_smem_bytes(const Tables& t);
void launch_pack_voxels(const float* rho, const unsigned char* mat, uint32_t* out, size_t n, float* rho_max, int n_mat, unsigned int* bad, void* stream);
void launch_body_box(const uint32_t* vox, int nx, int ny, int nz, const float* kfac, float thr, int* box, unsigned int* fout_bits, void* stream);
void launch_fold(const FoldParams& p, void* stream);
void launch_moments(const FoldParams& p, double* s1, double* s2, void* stream);
void launch_finalize_moments(const double* s1, const double* s2, size_t n, double total, double batches, float* mean, float* sigma, void* stream);
void launch_sample_source(const TransportParams& p, uint64_t first, uint64_t n, float* out, void* stream);
void launch_tmap(const Geom& g, const uint32_t* vox, float* tmap, void* stream);
void launch_apply_lut(const float* lut, int nt, int ns, float t_min, float t_max, float s_min, float s_max,
                      float s_eff, const float* dose, const float* tmap, float* out, size_t n, void* stream);
// analysis.cu
void launch_upsample(const float* in, int nu, int nv, float* out, int mu, int mv, void* stream);
void launch_roi_sum(const float* img, int nu, int nv, float pitch, float roi, double* acc, void* stream);
int launch_gamma(const float* ref, const float* ev, float* gamma, int nu, int nv, float pitch, float dose_frac, float dta,
                 float thr_frac, float cap, unsigned int* dmax_bits, double* stats, void* stream);

}  // namespace aepid
