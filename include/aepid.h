/* aepid.h -- C-ABI of the B200-native ARCHER-EPID hot path.
 *
 * What the library computes (Fig. 1, 104, 108-110, 114-123, 147-153;
 * BASELINE.json:north_star): analog coupled photon/electron
 * Monte Carlo transport of source photons through air, a CT-derived voxel phantom, air
 * and a multi-layer EPID slab stack, scoring absorbed energy into the EPID image and the
 * phantom grid, followed by the paper's dose-to-signal correction k(t, s).
 *
 * Conventions
 *   - Units: cm, MeV, g/cm^3.  Tallies are energy per history [MeV]; dose is a constant
 *     scaling by (density x voxel or pixel-layer volume) left to the caller.
 *   - World frame = the phantom's own axis-aligned (CT) frame.  Beam frame: source at the
 *     origin, axes u, v, w = rows of `beam_axes` written in world coordinates, beam along
 *     +w.  Everything that is not phantom or EPID inside the world box |u|,|v| <= 100 cm,
 *     -1 <= w <= EPID bottom is air (material 0, 1.205e-3 g/cm^3); leaving the box is
 *     escape (SURVEY.md 8(c) "Geometry").
 *   - Every function returns 0 on success or a negative aepid_status; nothing throws,
 *     prints or exits.  aepid_last_error() gives the reason.
 *   - Pointer arguments marked "host or device" are classified with
 *     cudaPointerGetAttributes.  Inputs are copied / repacked into the workspace during
 *     the call and may be freed on return.  Outputs are caller-owned buffers of exactly
 *     the stated size.
 *   - The library never allocates device memory: the caller hands it one workspace of
 *     aepid_workspace_bytes(dims) bytes (e.g. a torch uint8 tensor) and a CUDA stream.
 *     All work is stream-ordered; calls that fill HOST outputs synchronise the stream
 *     before returning, calls with DEVICE outputs do not.
 *   - One context per GPU; a context is not thread-safe.
 *   - There is no CPU fallback: without a CUDA device aepid_create fails with AEPID_ERR_CUDA.
 */
#ifndef AEPID_H
#define AEPID_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct aepid_ctx aepid_ctx;

enum aepid_status {
    AEPID_OK = 0,
    AEPID_ERR_BAD_ARG = -1,   /* null pointer, size out of range, malformed table */
    AEPID_ERR_BAD_STATE = -2, /* call order: something required has not been loaded */
    AEPID_ERR_GEOMETRY = -3,  /* phantom / EPID / source overlap or lie outside the world box */
    AEPID_ERR_CUDA = -4,      /* a CUDA runtime call failed (message holds cudaGetErrorString) */
    AEPID_ERR_NOMEM = -5,     /* workspace smaller than aepid_workspace_bytes(dims), or an input exceeds dims */
    AEPID_ERR_INTERNAL = -6   /* the transport kernel raised an error flag (ledger[7] != 0): a secondary was dropped for want of
                                 head room or the scheduler stalled; the tallies of that run are incomplete.  Reported by the calls
                                 that synchronise: aepid_read_tallies (with a ledger or a host output), aepid_read_moments (with
                                 totals), aepid_synchronize. */
};

/* Capacities the workspace is laid out for.  Loads may use less (fewer energy bins, a smaller
 * fluence map, fewer layers) but never more. */
typedef struct aepid_dims {
    int n_mat, n_E, n_T;      /* materials (<= 32), photon grid points, electron grid points */
    int nx, ny, nz;           /* phantom grid (each <= 1024) */
    int n_layers;             /* EPID layers (<= 8) */
    int nu, nv;               /* EPID image */
    int n_bins;               /* spectrum bins */
    int fu, fv;               /* fluence map */
    int n_batches;            /* B independent tally buffers for the batch variance estimate (2..255) */
    int n_ps1;                /* capacity for Phase Space 1 records (aepid_load_phase_space_source), 0 if not used */
    int max_live_per_cta;     /* most particles one CTA of the transport kernel keeps alive, 64..262144 (0 = 65536); the workspace
                                 holds 160 x 5 class queues of twice that many 48-byte records (rounded up to a power of two):
                                 20 GB at 262144, 5.0 GB at 65536, 80 MB at 1024.  Results do not depend on it; small runs want it
                                 small, runs of 1e9 histories are 8 % faster at 262144 than at 65536 (profiles/r02_README.md). */
} aepid_dims;

/* Bytes of device memory the context needs for `dims` (0 if dims are invalid). */
size_t aepid_workspace_bytes(const aepid_dims* dims);

/* Create a context on CUDA device `device`, ordered on `cuda_stream` (a cudaStream_t, e.g.
 * torch.cuda.current_stream().cuda_stream; NULL = legacy default stream), owning nothing but
 * host-side bookkeeping.  `workspace` is DEVICE memory, 256-byte aligned, that must outlive
 * the context.  Tallies start zeroed. */
int aepid_create(aepid_ctx** out, int device, void* cuda_stream, const aepid_dims* dims,
                 void* workspace, size_t workspace_bytes);
void aepid_destroy(aepid_ctx* ctx);
const char* aepid_last_error(const aepid_ctx* ctx);   /* NUL-terminated, owned by the context */

/* Material tables (SURVEY.md 8(c) "Cross-section / stopping-power tables"; physics list PAPER.md:104).
 * All arrays host or device, float32.  E_grid_MeV [n_E]: positive and strictly increasing, otherwise free (a tabulation
 * refined around absorption edges; an edge is two grid points a hair apart): a log-uniform grid is indexed directly, any other
 * through a guide table of 1024 buckets in ln E (AEPID_ERR_BAD_ARG if not increasing).  T_grid_MeV [n_T] must be log-uniform
 * and increasing (stopping powers are smooth; the charged-particle step looks it up twice per step).  mu_* [n_mat][n_E] are mass coefficients in cm^2/g: Compton and photoelectric are
 * interpolated linearly in (ln E, ln mu), pair linearly in (ln E, mu).  stop_pow [n_mat][n_T] in
 * MeV cm^2/g (log-log interpolation), rad_len_g_cm2 [n_mat].  Material 0 is the air that fills the world. */
int aepid_init_materials(aepid_ctx* ctx, int n_mat,
                         int n_E, const float* E_grid_MeV,
                         const float* mu_compton, const float* mu_pe, const float* mu_pair,
                         int n_T, const float* T_grid_MeV,
                         const float* stop_pow, const float* rad_len_g_cm2);

/* Voxel phantom ("three-dimensional density matrix").  density_g_cm3 and material are
 * [nz][ny][nx] with x fastest, host or device; origin_cm is the world position of the corner of voxel
 * (0,0,0).  The grid is repacked to one 32-bit word per voxel (density rounded to 19 mantissa bits,
 * material in the low 5 bits).  Resets the tallies. */
int aepid_load_phantom(aepid_ctx* ctx, int nx, int ny, int nz, const float spacing_cm[3],
                       const float origin_cm[3], const float* density_g_cm3, const unsigned char* material);

/* EPID slab stack: n_layers slabs normal to w, listed along +w, the upstream face of
 * layer 0 at w = sid_cm (reading A6).  Per-layer arrays are HOST pointers [n_layers].  Energy deposited in
 * layers with scored != 0 is binned to pixel (iu, iv) = floor((u + nu p/2)/p), floor((v + nv p/2)/p) of an
 * nu x nv image centred on the beam axis; everything else in the stack goes to ledger[3]. */
int aepid_load_epid_layers(aepid_ctx* ctx, int n_layers, const float* thickness_cm,
                           const unsigned char* material, const float* density_g_cm3,
                           const unsigned char* scored, float sid_cm, int nu, int nv, float pitch_cm);

/* Source (BASELINE.json:north_star (2)): point source at src_pos_cm (world), energy
 * from the histogram spectrum E_edges_MeV [n_bins+1] / E_pdf [n_bins] (one zero-width bin = monoenergetic),
 * position from the planar fluence map fluence [fv][fu] (u fastest, pitch f_pitch_cm, centred on the axis) on
 * the plane w = f_plane_dist_cm.  src_pos_cm and beam_axes are HOST pointers; the arrays host or device.
 * May be called again between fields; it does not touch the tallies. */
int aepid_load_source(aepid_ctx* ctx, const float src_pos_cm[3], const float beam_axes[9],
                      int n_bins, const float* E_edges_MeV, const float* E_pdf,
                      int fu, int fv, float f_pitch_cm, float f_plane_dist_cm, const float* fluence);

/* mode 0: kerma (charged-particle energy deposited at the interaction point, configs[0]);
 * mode 1: coupled (CSDA electron steps with Highland deflection);
 * mode 2: coupled with Class II collisions ("Class II condensed history"; reading A31): discrete Moller events
 * with energy transfer above the electron cut-off, each starting a delta ray, and the restricted collision stopping
 * power below it;
 * mode 3: mode 2 plus bremsstrahlung (reading A32): photons above the photon cut-off are emitted as discrete events along the
 * particle's direction, the loss to softer photons is continuous; the spectrum (4/3 - 4/3 y + y^2) / (X0 k), y = k / T, makes the
 * total radiative stopping power T / X0.  Modes 2 and 3 need aepid_set_class2;
 * mode 4: the physics of mode 1 with DPM-style steps ("developed based on DPM"; reading A38): a step loses f_E T in two
 * legs split at a uniformly drawn hinge where the Highland deflection of the whole step is applied; voxel, layer and region faces
 * end straight segments (each deposits rho S ds of its own medium), not steps; s_max is not used.  The class queues hold half as
 * many (64-byte) records in this mode.  Cutoffs PAPER.md:104 (defaults 0.010 / 0.200 MeV); step rule f_E = 0.10,
 * s_max = 1 cm (reading A13). */
int aepid_set_physics(aepid_ctx* ctx, int mode, float photon_cut_MeV, float electron_cut_MeV,
                      float f_E, float s_max_cm);

/* Zero the B batch buffers, the energy ledger, the counters, the history count and the history offset: the start of a new
 * field (every IMRT field is simulated on its own; aepid_load_source "implies nothing about
 * tallies").  Asynchronous on the stream. */
int aepid_reset_tallies(aepid_ctx* ctx);

/* The hot path, K1-K7 of SURVEY.md 8(a).  One history = one particle of Phase Space 2, i.e. one source photon entering the
 * patient stage (section 2.1.1); it and all its descendants are followed through the phantom (photoelectric,
 * Compton and pair interactions, electrons down to 200 keV, photons down to 10 keV: section 2.1.2), the air gap
 * and the EPID layers, scoring energy into the phantom grid and the image.
 * Transports histories [first, first + n) where first = history offset + histories run since the last reset; history h
 * draws from Philox4x32-10 keyed by `seed` with counter (h_lo, h_hi, particle, block) (reading A1).
 * Accumulates into the B batch buffers (history k of a launch scores into batch min(k / ceil(n / B), B - 1)); asynchronous
 * on the stream; n_histories above 2^31 is split into several launches. */
int aepid_simulate(aepid_ctx* ctx, unsigned long long n_histories, unsigned long long seed);

/* The results of the path: the three-dimensional energy deposition in the patient grid ("3-D dose") and the
 * EPID image, each as the mean energy per history and its standard error, which is what the paper's
 * "statistical uncertainty below 1 %" is a statement about (reading A19; estimator: DESIGN.md section 3, B
 * independent batches).  Images [nv][nu], volumes [nz][ny][nx]; any of the four may be NULL; host or device.  ledger (HOST,
 * may be NULL): {emitted, dep_phantom, dep_epid_scored, dep_epid_other, dep_air, escaped, n_histories, error flags of the
 * transport kernel}.  With a ledger or any host output the call synchronises and returns AEPID_ERR_INTERNAL if the error
 * flags are set (the outputs are still written). */
int aepid_read_tallies(aepid_ctx* ctx, float* epid_mean, float* epid_sigma,
                       float* phantom_mean, float* phantom_sigma, double ledger[8]);

/* Multi-GPU sharding: histories are independent, so rank r of G runs a disjoint block of the
 * global history range.  aepid_set_history_offset makes the next aepid_simulate start at global history index
 * `first_history` (Philox is keyed by the global index); call it after aepid_reset_tallies. */
int aepid_set_history_offset(aepid_ctx* ctx, unsigned long long first_history);

/* Per-bin sufficient statistics of this context's B batches, for the one exchange step of 8(e):
 * s1 = sum_b x_b and s2 = sum_b x_b^2 / n_b (float64; images [nv][nu], volumes [nz][ny][nx]; DEVICE pointers, any may be
 * NULL).  totals (HOST [2]) = {histories, non-empty batches}.  After an all-reduce(sum) of s1, s2 and totals over ranks,
 * aepid_finalize_moments turns them into the mean per history and its standard error:
 * mean = s1 / N, sigma^2 = (s2 - N mean^2) / ((B - 1) N).  n = number of bins; all pointers DEVICE. */
int aepid_read_moments(aepid_ctx* ctx, double* epid_s1, double* epid_s2, double* phantom_s1, double* phantom_s2, double totals[2]);
int aepid_finalize_moments(aepid_ctx* ctx, const double* s1, const double* s2, size_t n, double n_histories, double n_batches,
                           float* mean, float* sigma);

/* Raw per-batch EPID sums [B][nv][nu] (host or device, may be NULL) and histories per batch (HOST [B]). */
int aepid_read_batches(aepid_ctx* ctx, float* epid_batches, double* histories_per_batch);

/* Event and scheduler counters since the last reset (HOST [32]), only counted while aepid_set_counting(ctx, 1) (an
 * instrumented instantiation of the transport kernel runs then).  Counter map, index name (the binding's COUNTER_NAMES):
 *    0 woodcock_flights    1 air_flights        2 epid_flights       3 n_pe
 *    4 n_compton           5 n_pair             6 esteps_phantom     7 esteps_air
 *    8 esteps_epid         9 n_secondaries     10 unused10          11 unused11
 *   12 kn_iterations      13 photon_cutoffs    14 e_tracks          15 zero_steps
 *   16 iter_A             17 iter_W            18 iter_E            19 iter_P
 *   20 iter_X             21 lanes_A           22 lanes_W           23 lanes_E
 *   24 lanes_P            25 lanes_X           26 phases            27 particles_stored
 *   28 particles_loaded   29 particles_parked  30 source_tasks      31 majorant_violations
 * 0-9, 12-15: events of the physics (flights per region, interactions per channel, charged-particle steps per region,
 * secondaries created, Klein-Nishina trials, photons ended by the 10 keV cut-off, charged tracks, zero-length steps);
 * 16-20: warp-level event iterations of the scheduler phases A, W, E, P, X (transport.cu), 21-25: live lanes summed over
 * those iterations, 26 phases run (all CTAs), 27 / 28 particle records written to / read from the class queues, 29 lanes
 * that parked their particle for want of head room, 30 source tasks, 31 tentative Woodcock collisions in a voxel whose
 * attenuation coefficient exceeds the majorant of its segment (body box): must stay 0. */
int aepid_set_counting(aepid_ctx* ctx, int on);
int aepid_read_counters(aepid_ctx* ctx, unsigned long long counters[32]);

/* K1 alone: source samples of histories [first, first+n): out[n][8] = {E, dx, dy, dz (world), fluence pixel,
 * u, v on the fluence plane, 0}; host or device. */
int aepid_sample_source(aepid_ctx* ctx, unsigned long long first, unsigned long long n,
                        unsigned long long seed, float* out);

/* Effective field size (Eq. 1; reading A16): equivalent square s = 2ab/(a+b) of the bounding
 * box a x b (at the isocentre plane w = 100 cm) of fluence pixels with weight > 0; printed_form != 0 gives
 * ab/(2(a+b)) exactly as printed. */
int aepid_field_size(aepid_ctx* ctx, int printed_form, float* s_cm);

/* Response post-pass: t_uv = line integral of density/(1 g cm^-3) from the source
 * to the centre of pixel (u, v) on the EPID top plane through the phantom grid (reading A17);
 * signal = dose * k(t_uv, s) with k bilinear in lut[it*ns + is] on uniform axes, (t, s) clamped into the table
 * (reading A18).  s_eff_cm < 0 derives s from the loaded fluence.  epid_in NULL = current mean image.
 * lut (nt*ns <= 65536), epid_in, signal_out [nv][nu], tmap_out [nv][nu] (may be NULL): host or device. */
int aepid_apply_response_lut(aepid_ctx* ctx, const float* lut, int nt, int ns,
                             float t_min, float t_max, float s_min, float s_max, float s_eff_cm,
                             const float* epid_in, float* signal_out, float* tmap_out);

/* Input of physics mode 2: electrons per gram of every material, N_A sum_i w_i Z_i / A_i ([n_mat], host or device, copied).
 * Call after aepid_init_materials (which forgets it). */
int aepid_set_class2(aepid_ctx* ctx, const float* electrons_per_gram);

/* Collimation stage (section 2.1.1: "particles are sampled from Phase Space 1 and transported through the
 * jaws and MLC ... the resulting phase space (Phase Space 2) is ... streamed directly into the next simulation stage";
 * SURVEY.md 8(f) NEXT-3; readings A35-A37 in DESIGN.md).
 * aepid_load_phase_space_source: n_records x 8 floats = {u, v, du, dv, dw, E, -, -} (host or device, copied): position on the
 * plane w = w_plane_cm of the beam frame (the frame of aepid_load_source: source position and axes), direction, energy.  While
 * a table is loaded, history h starts from record floor(xi n_records), xi = the first draw of its Philox block 0, instead of
 * the fluence-map sampler (one history = one Phase Space 1 particle; aepid_read_head counts the Phase Space 2 particles).
 * n_records = 0 goes back to the fluence-map source.  n_records <= dims.n_ps1.
 * aepid_load_collimator: n_slabs (<= 4) tungsten slabs sorted along w between the Phase Space 1 plane and w_ps2_cm.  Slab k spans
 * [w0[k], w1[k]); its rows are stacked along v (axis[k] = 0: the MLC and the x-jaws, openings in u) or along u (axis[k] = 1: the
 * y-jaws, openings in v), row r covering [row0[k] + r pitch[k], row0[k] + (r+1) pitch[k]); row r is open on [lo, hi) (lo, hi:
 * concatenated over the slabs, n_rows[k] entries each, at most 1024 in all; a closed leaf pair has lo = hi), all in cm at the slab
 * itself (straight, unfocused edges).  Everything else inside a slab's w-range is `material` at `density`.  All pointers HOST.
 * Photons are followed through the stage with the photon physics of the path; charged particles are not (their energy stays in
 * the head and is booked in ledger[4]), annihilation quanta born in the head are dropped, photons that turn upstream escape.
 * n_slabs = 0 removes the collimator.
 * aepid_read_head (synchronises): {Phase Space 2 particles, their energy [MeV], energy absorbed in the stage [MeV], 0} since the
 * last aepid_reset_tallies. */
int aepid_load_phase_space_source(aepid_ctx* ctx, unsigned long long n_records, const float* records, float w_plane_cm);
int aepid_load_collimator(aepid_ctx* ctx, int n_slabs, const float* w0_cm, const float* w1_cm, const int* axis, const int* n_rows,
                          const float* row0_cm, const float* pitch_cm, const float* lo_cm, const float* hi_cm,
                          int material, float density_g_cm3, float w_ps2_cm);
int aepid_read_head(aepid_ctx* ctx, double out[4]);

/* Scheduler knob of the transport kernel: the most particles a CTA keeps alive at a time, 64 .. what the
 * context was created for (0 = that: dims.max_live_per_cta, half a class queue).  Results do not depend on it (every particle has its own Philox stream);
 * small values make lanes wait for head room and exist to test exactly that path. */
int aepid_set_live_limit(aepid_ctx* ctx, int max_live_per_cta);

/* Phase Space 3 ("an additional scoring plane, Phase Space 3, is generated to store all particles exiting
 * the patient"; reading A30): while a buffer is set, every particle that arrives at the EPID top plane (w = sid) from the
 * air is copied into it as two float4 = {u, v, du, dv} {dw, E, type bits, history bits}: position and direction in the beam
 * frame (cm; dw > 0), photon energy or kinetic energy (MeV), type 0 photon / 1 electron / 2 positron and the global history
 * index modulo 2^32 as raw 32-bit patterns.  The particle itself flies on (the hand-off stays in flight); the order of the
 * records is not defined.  records: DEVICE, 16-byte aligned, 32 * capacity bytes, caller-owned and kept alive while set;
 * NULL switches the recording off.  Setting a buffer and aepid_reset_tallies zero the arrival count.
 * aepid_read_phase_space_count (synchronises): arrivals since then; only the first `capacity` claimed records are stored. */
int aepid_set_phase_space(aepid_ctx* ctx, void* records, unsigned long long capacity);
int aepid_read_phase_space_count(aepid_ctx* ctx, unsigned long long* n_arrived);

/* Eq. 2 of the paper, k(t, s) = M(t, s) / S(t, s): S is "the average simulated dose" in the central
 * roi_cm x roi_cm region (the paper: 1 cm x 1 cm) of the EPID image.  mean_out (HOST) = mean over the pixels whose centre
 * lies in the closed central square (reading A33); nan if there is none.  image: DEVICE [nv][nu] with its pitch, or NULL
 * for the current mean EPID image of the context (nu, nv, pitch_cm are then ignored).  Synchronises. */
int aepid_roi_mean(aepid_ctx* ctx, const float* image, int nu, int nv, float pitch_cm, float roi_cm, double* mean_out);

/* Analysis chain (section 2.3.3).
 * aepid_upsample: out [mv][mu] = bilinear interpolant of in [nv][nu] over the same physical area: output pixel (j, i)
 * is taken at x = (i + 0.5) nu/mu - 0.5, y = (j + 0.5) nv/mv - 0.5 in input pixels (centres at the integers), clamped to
 * [0, n - 1] (reading A28).  DEVICE pointers, caller-owned; asynchronous on the context's stream.
 * aepid_gamma_index: global 2-D gamma of `eval` against `ref` (same grid [nv][nu], non-negative, pixel pitch pitch_cm):
 * gamma = min over evaluated pixels within gamma_cap * dta_cm of sqrt(dist^2/dta^2 + (D_e - D_r)^2/(dose_frac max(ref))^2),
 * reported as min(gamma_cap, gamma); reference pixels below threshold_frac * max(ref) get -1 and are not counted
 * (reading A29).  ref, eval, gamma_out: DEVICE [nv][nu].  stats (HOST [4], may be NULL; when given the call
 * synchronises) = tested pixels, pixels with gamma <= 1, mean gamma, max gamma over the tested pixels.
 * AEPID_ERR_NOMEM if the window of gamma_cap * dta_cm / pitch_cm pixels does not fit in shared memory (about 90 pixels). */
int aepid_upsample(aepid_ctx* ctx, const float* in, int nu, int nv, float* out, int mu, int mv);
int aepid_gamma_index(aepid_ctx* ctx, const float* ref, const float* eval, int nu, int nv, float pitch_cm,
                      float dose_frac, float dta_cm, float threshold_frac, float gamma_cap,
                      float* gamma_out, double stats[4]);

/* Block until everything queued on the context's stream has finished. */
int aepid_synchronize(aepid_ctx* ctx);

/* The analysis chain of PAPER.md:141 (up-sample the predicted image to the grid of the measured one, reading A28, then the
 * global gamma index of it against the measured image, reading A29) for callers that cannot allocate device memory: code
 * under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  No context, no workspace: the call
 * allocates NOTHING (no cudaMalloc / cudaFree, no allocating library routine).  Its scratch (the up-sampled image, the image
 * maximum, the gamma statistics) is a file-scope `static __device__` array of the library, AEPID_STATIC_MAX_PIXELS floats +
 * 256 bytes = 6.25 MiB, which every GPU that loads the library holds until the process exits.
 *   predicted [nv][nu], measured [mv][mu] (the reference; non-negative; pixel pitch pitch_cm), gamma_out [mv][mu]: DEVICE,
 *   caller-owned.  stats_out: DEVICE [4] doubles or NULL = {tested pixels, pixels with gamma <= 1, mean gamma, max gamma}.
 *   The criteria are those of aepid_gamma_index; gamma_out = gamma of the up-sampled predicted image (evaluated) against
 *   `measured` (reference), identical to aepid_upsample followed by aepid_gamma_index(measured, up-sampled, ...).
 * Asynchronous on cuda_stream of CUDA device `device` (made current for the call, the previous one restored).  The first
 * call per device resolves the array's device address (cudaGetSymbolAddress): make one call before a graph capture.
 * Every call shares the one array: it keeps the last call's contents (what must start at zero is cleared on the stream by
 * every call), and two calls that OVERLAP on the GPU (different streams, no ordering) race: order them.
 * Errors: AEPID_ERR_NOMEM if mu * mv > AEPID_STATIC_MAX_PIXELS (use aepid_upsample + aepid_gamma_index with caller memory)
 * or if the search window does not fit in shared memory; AEPID_ERR_BAD_ARG; AEPID_ERR_CUDA.  error_text (HOST, may be NULL)
 * receives a NUL-terminated message of at most error_text_bytes bytes. */
#define AEPID_STATIC_MAX_PIXELS (1280 * 1280)
int aepid_gamma_of_upsampled_static(int device, void* cuda_stream, const float* predicted, int nu, int nv,
                                    const float* measured, int mu, int mv, float pitch_cm, float dose_frac, float dta_cm,
                                    float threshold_frac, float gamma_cap, float* gamma_out, double* stats_out,
                                    char* error_text, size_t error_text_bytes);

#ifdef __cplusplus
}
#endif
#endif /* AEPID_H */
