// Transport kernel: K1 source sampling, K2 air navigation, K3 Woodcock tracking, K4 interaction
// sampling, K5 CSDA electron steps with Highland deflection, K6 EPID slab transport and K7 tally
// scoring (physics of SURVEY.md 8(c)).
//
// Design (sm_100a): ONE persistent CTA per SM that runs a LOCAL WAVEFRONT.  Measured on B200 (profiles/r01_history.md,
// DESIGN.md 6.2): warps of one SM that execute different parts of a code body larger than the
// 32 KB instruction cache starve on instruction fetch (IPC 0.3-1.1 of 4), warps that execute the same part do not.
// So all warps of a CTA work on the same event class at any time:
//   * Event classes: A photon in air (new histories start here), W photon in the phantom, E charged particle in the
//     phantom, P photon inside the EPID or with a collision pending outside the phantom, X charged particle outside
//     the phantom.  The CTA runs PHASES, one class per phase, separated by block barriers; thread 0 picks the next
//     phase: new histories while there is head room for them, else the class with the most waiting particles.
//   * Particle records (48 B, three 16 B vectors) live in per-CTA CLASS QUEUES in global memory: one ring of kPool
//     records per event class (L2 / HBM, written and read once with streaming .cs accesses so that they do not push the
//     voxels and tallies out of the L2; consecutive tickets = consecutive records,
//     so a refill is one coalesced, prefetchable read with no index to chase).  Shared memory holds the material tables
//     (ln domain, one LDS.128 per node) and the scheduler state.  Up to kLiveMax = 65536 particles for 1024 lanes
//     (262144 for launches of 4e8 histories and more, aepid_dims.max_live_per_cta) make a phase many waves long, so that the
//     phase switch (two barriers, every lane refilled at once, a cold instruction cache: about 35 us) and the tail of a phase
//     cost little (measured on 1e9 histories of C3: 32768 alive +2.5 %, 65536 the reference, 262144 -7 %).
//   * Within a phase every lane follows its particle event by event while it stays in the class; a lane whose
//     particle has died or changed class writes it back (record appended to the queue of the new class) and is
//     refilled IN PLACE from the queue of the phase, so warps run one code path with nearly all lanes active.
//     Secondaries are appended straight to the queue of their class.
//   * Queue protocol: head/tail are monotonic ticket counters; a push takes a ticket from tail and writes the record;
//     pops take tickets from head but only below the SNAPSHOT of tail taken at the last barrier, so a record is never
//     read before the barrier that publishes it and no generation tags or spin waits are needed.  What is pushed
//     during a phase (also into the phase's own queue: parked or evicted particles) becomes visible in the next phase.
//     A push may not wrap onto a record that can still be read in this phase: tail at the end of the phase minus head
//     at its start must stay <= kPool.  That difference is (particles popped) + (particles in the queue at the end),
//     each at most the number of particles alive in the CTA, which s_live keeps <= kLiveMax = kPool / 2.
//   * A phase ends softly: a warp that can no longer keep its lanes full (ring exhausted, kRefillMin lanes empty)
//     writes its particles back and leaves, so all warps reach the barrier within about one event of each other and
//     the survivors join the next phase of their class (a write-back and reload costs a fraction of one event).
//     In a phase that starts with fewer than two waves of particles a warp stays for at least kMinIter events.
//   * Head room: s_live counts the particles alive in the CTA plus the credits held by lanes.  A lane runs an event
//     that can create a secondary only while it holds a credit (its own count when its particle died, else a fresh
//     one), otherwise it parks its particle; new histories start only while kReserve of head room stays free.  Hence
//     s_live <= kLiveMax always, and writing a particle back never needs anything.
//   * A particle's trajectory does not depend on the schedule: its Philox stream is keyed by (history, particle
//     id, block) and every event consumes whole blocks (reading A1).
//   * The phantom is one packed 32-bit word per voxel gathered through the read-only path; phantom deposits of
//     consecutive steps in one voxel are merged in registers and flushed with one RED; the energy ledger is summed
//     per lane in float, reduced over the warp and accumulated per warp in double.
// No tensor cores / TMA: random gathers and scalar arithmetic, nothing here is a dense contraction.
#include <cuda_runtime.h>
#include <cstdint>
#include "params.h"

namespace aepid {

#ifndef AEPID_WARPS
#define AEPID_WARPS 32
#endif
constexpr int kWarps = AEPID_WARPS;
constexpr int kThreads = kWarps * 32;
// Records per class queue of a CTA: kPool = 1 << TransportParams::pool_log (from aepid_dims.max_live_per_cta, at most 2^19);
// the most particles alive in a CTA at any time is half a queue (see "queue protocol" above), the limit in force is
// TransportParams::live_max <= kPool / 2 (s_live_max).
#ifndef AEPID_RESERVE_8THS
#define AEPID_RESERVE_8THS 3
#endif
#ifndef AEPID_REFILL_MIN
#define AEPID_REFILL_MIN 3
#endif
constexpr int kReserve8ths = AEPID_RESERVE_8THS;             // eighths of the limit that must remain free for secondaries when new histories start
constexpr int kRefillMin = AEPID_REFILL_MIN;                 // a warp refills its empty lanes once this many are empty
#ifndef AEPID_MIN_ITER
#define AEPID_MIN_ITER 12
#endif
constexpr uint32_t kMinIter = AEPID_MIN_ITER;   // events per lane before a warp may leave a short phase early
#ifndef AEPID_SHARE_NUM
#define AEPID_SHARE_NUM 1u
#define AEPID_SHARE_DEN 1u
#endif
#ifndef AEPID_PREFETCH
#define AEPID_PREFETCH 2048
#endif
#ifndef AEPID_STEPS_E
#define AEPID_STEPS_E 4
#endif
#ifndef AEPID_STEPS_X
#define AEPID_STEPS_X 4
#endif
constexpr int kStepsE = AEPID_STEPS_E, kStepsX = AEPID_STEPS_X;   // steps per event of a charged particle in / outside the phantom
#ifdef AEPID_PHASE_CLOCK
constexpr bool kPhaseClock = true;        // analysis build: counters 10, 11, 16-25, 27-31 hold phase clocks instead
#else
constexpr bool kPhaseClock = false;
#endif
constexpr int kLongPhase = 2 * kThreads;      // phases that start with at least this many particles end softly
#ifndef AEPID_HIT_MIN
#define AEPID_HIT_MIN 16
#endif
constexpr int kHitMin = AEPID_HIT_MIN;          // photon flights go on until this many lanes of the warp have a collision to sample
constexpr int kMaxRounds = 8;                 // ... but no more than this many flights per event
constexpr int kStarved = 256;                 // less head room than this: prefer phases that need none
constexpr uint32_t kIterLimit = 1u << 20;     // iterations of one warp in one phase before it hands its particles back
constexpr uint32_t kPhaseLimit = 1u << 24;
constexpr float kPi = 3.14159265358979f;
constexpr float kInf = 3.0e38f;
constexpr uint32_t kNone = 0xffffffffu;

// event classes = rings = phases
enum : int { C_A = 0, C_W = 1, C_E = 2, C_P = 3, C_X = 4, kClasses = 5, kRings = kRingCount };

#define FULL_MASK 0xffffffffu
// flags: bits 0-1 type, 2-3 region, 4-6 layer, 7 collision pending (photon outside the phantom), 16-23 batch
#define F_TYPE(f) ((f) & 3u)
#define F_REGION(f) (((f) >> 2) & 3u)
#define F_LAYER(f) (((f) >> 4) & 7u)
#define F_HIT (1u << 7)
#define F_LEGA (1u << 8)      // physics mode 4: a charged particle on the first leg of its step (before the hinge)
#define F_BATCH(f) (((f) >> 16) & 255u)
#define SET_TYPE(f, t) ((f) = ((f) & ~3u) | (t))
#define SET_REGION(f, r) ((f) = ((f) & ~(3u << 2)) | ((r) << 2))
#define SET_LAYER(f, l) ((f) = ((f) & ~(7u << 4)) | ((uint32_t)(l) << 4))

// event class of a particle: which ring it waits in, which phase works on it
__device__ __forceinline__ int class_of(uint32_t flags) {
    const uint32_t reg = F_REGION(flags);
    if (F_TYPE(flags) == T_PHOTON) return reg == R_PHANTOM ? C_W : ((reg == R_EPID || (flags & F_HIT)) ? C_P : C_A);
    return reg == R_PHANTOM ? C_E : C_X;
}

// is the particle with these flags in class C?  (class_of(flags) == C, as two or three bit tests)
template <int C>
__device__ __forceinline__ bool in_class(uint32_t flags) {
    constexpr uint32_t kTR = 3u | (3u << 2);                                    // type and region bits
    if (C == C_W) return (flags & kTR) == (T_PHOTON | (R_PHANTOM << 2));
    if (C == C_A) return (flags & (kTR | F_HIT)) == (T_PHOTON | (R_AIR << 2));
    if (C == C_P) return (flags & 3u) == T_PHOTON && (flags & (3u << 2)) != (R_PHANTOM << 2) && (flags & ((3u << 2) | F_HIT)) != (R_AIR << 2);
    if (C == C_E) return (flags & 3u) != T_PHOTON && (flags & (3u << 2)) == (R_PHANTOM << 2);
    return (flags & 3u) != T_PHOTON && (flags & (3u << 2)) != (R_PHANTOM << 2);
}

// Scheduler state and the geometry copy: static shared memory, so that the out-of-line helpers reach them
// without arguments.
__shared__ unsigned int s_tail[kRings];             // tickets handed to pushers
__shared__ unsigned int s_head[kRings];             // tickets handed to poppers
__shared__ unsigned int s_snap[kRings];             // tail at the last barrier: pops stay below it
__shared__ int s_flag[2];                           // [0] no histories left, [1] error bits
__shared__ int s_phase, s_keep, s_budget, s_left;   // class of the phase (-1: done), soft-end threshold, new histories allowed, warps gone
__shared__ int s_stuck;                             // bit c: class c was stuck in its last phase (choose_phase: progress check)
__shared__ int s_did, s_parked;                     // set by any warp whose lanes ran an event / parked a particle for want of a credit in the
                                                    // current phase (choose_phase: progress check)
__shared__ unsigned int s_nphase;
__shared__ Geom s_g;
__shared__ float* s_ep_batch;
__shared__ unsigned long long s_npix;
__shared__ uint4* s_queue;                          // this CTA's class queues of particle records [kClasses][kPool][3]
__shared__ int s_live_max;                          // limit of s_live for this launch
__shared__ int s_live;                              // particles alive in this CTA (in the queues, in lanes) + head-room credits held by lanes
extern __shared__ __align__(16) unsigned char smem_raw[];   // per-warp ledger | table blob

// error bits (summed over CTAs into ledger[7]): 2 no head room for a secondary, 8 scheduler found no
// runnable phase or ran out of phases
__device__ __forceinline__ void raise_error(int bit) { atomicOr(s_flag + 1, bit); }
// Checked build (-DAEPID_CHECKED, tests/test_gpu_checked_build.py): every index that reaches global memory (voxel words, tally
// bins, queue records) and the invariants of the queue protocol are tested in the kernel; a violation raises error bit 16,
// which aepid_read_tallies / aepid_synchronize return as AEPID_ERR_INTERNAL.  (compute-sanitizer is closed on the GPU pool
// this was developed on; the checks cost about 4 % and are compiled out of the product build.)
#ifdef AEPID_CHECKED
#define AEPID_CHECK(cond) do { if (!(cond)) raise_error(16); } while (0)
__shared__ unsigned int s_head0[kRings];            // head of every queue when the phase began (queue protocol: tail - head0 <= kPool)
#else
#define AEPID_CHECK(cond) do { } while (0)
#endif


__shared__ uint32_t s_pool_mask;                    // records per class queue - 1
__shared__ int s_pool_log;
__shared__ uint32_t s_rec_vec;                      // 16-byte vectors per particle record: 3, or 4 in physics mode 4 (the leg's energy budget)
#ifndef AEPID_RING_BASE
#define AEPID_RING_BASE 1
#endif
__shared__ uint4* s_ring_base[kRings];              // first record of every class queue of this CTA
#if AEPID_RING_BASE
__device__ __forceinline__ uint4* queue_rec(int r, uint32_t ticket) { return s_ring_base[r] + (ticket & s_pool_mask) * s_rec_vec; }
#else
__device__ __forceinline__ uint4* queue_rec(int r, uint32_t ticket) { return s_queue + ((((size_t)r) << s_pool_log) + (ticket & s_pool_mask)) * s_rec_vec; }
#endif
struct Shared {
    const float4* phot;
    const float* maj;
    const float* lnS;
    const float* invX0;
    const float* sig;               // mode 2: Moller cross section [n_mat][n_T] (cm^2/g), linear in ln T; lnS then holds the restricted stopping power
    const float* lnEg;              // photon grid that is not log-uniform: ln E_j, and the guide table of the cell search (params.h)
    const uint32_t* guide;
};

struct Lane {
    float x, y, z, dx, dy, dz, E;   // position: world (AIR, photon in PHANTOM), voxel fraction (charged in PHANTOM), beam (u, v, depth) in EPID
    uint32_t vox;                   // packed voxel index ix | iy << 10 | iz << 20
    uint32_t flags;
    uint32_t h, pid, blk;           // history (relative to the launch base), particle id, Philox block counter
    uint32_t cw, vlin;              // packed word and linear index of the current voxel (charged particle in PHANTOM)
    int ci; float ct, mumaj;        // photon: table cell, fraction, majorant at E
    uint32_t pidx; float pval;      // pending phantom deposit (merged while the voxel does not change)
    float R;                        // physics mode 4: energy the particle still loses on the current leg of its step
    uint32_t counted;               // 1: the lane holds a particle that is counted in s_live (alive, or dead and not yet released); kNone: none
    uint32_t spare;                 // 1: the lane holds a head-room credit for its next secondary (kNone: none)
    float a_emit, a_ph, a_eps, a_epo, a_air, a_esc;   // ledger sums since the last flush
    bool alive;
};

// ---------------------------------------------------------------- Philox4x32-10 (own implementation; pinned on the GPU by tests)
__device__ __noinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return make_uint4(c0, c1, c2, c3);
}
// uniform in (0,1) from the top 23 bits: ((r >> 9) + 0.5) 2^-23 is exact in float32 and never 0 or 1
// (built in the mantissa of a float in [1, 2), no integer conversion; the subtraction is exact)
__device__ __forceinline__ float u01(uint32_t r) { return __uint_as_float(0x3f800000u | (r >> 9)) - 0.99999994f; }

// approximate reciprocal (MUFU.RCP): geometry distances and sampling formulas do not need the IEEE one
__device__ __forceinline__ float rcp(float x) { return __fdividef(1.0f, x); }

__device__ __forceinline__ uint4 rng_block(Lane& L, const TransportParams& P) {
    const uint64_t h = P.base + L.h;
    const uint4 o = philox4x32_10((uint32_t)h, (uint32_t)(h >> 32), L.pid, L.blk, (uint32_t)P.seed, (uint32_t)(P.seed >> 32));
    L.blk++;
    return o;
}
// The same block, expanded in place with the round keys taken from the kernel parameters (constant-bank operands: no
// key arithmetic, no call): for the three hottest draw sites (electron steps, Woodcock flights, Klein-Nishina trials).
__device__ __forceinline__ uint4 rng_block_hot(Lane& L, const TransportParams& P) {
    const uint64_t h = P.base + L.h;
    uint32_t c0 = (uint32_t)h, c1 = (uint32_t)(h >> 32), c2 = L.pid, c3 = L.blk;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ P.rk[2 * r], n2 = hi0 ^ c3 ^ P.rk[2 * r + 1];
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    }
    L.blk++;
    return make_uint4(c0, c1, c2, c3);
}
__device__ __forceinline__ uint32_t child_id(const Lane& L, uint32_t sibling) {    // reading A1
    return L.pid * 0x9E3779B1u + L.blk * 2u + sibling + 1u;
}

// ---------------------------------------------------------------- tables
// (pe, co, pp) of material m for a photon of energy E in table cell (ci, ct).  Pair production is impossible at or below
// 2 m_e c^2 although the linear interpolant across the cell that straddles the threshold is positive there (reading A34).
__device__ __forceinline__ void mu3(const TransportParams& P, const Shared& sh, int m, int ci, float ct, float E, float& pe, float& co, float& pp) {
    const float4 a = sh.phot[m * P.tb.n_E + ci], b = sh.phot[m * P.tb.n_E + ci + 1];
    pe = __expf(fmaf(ct, b.x - a.x, a.x));
    co = __expf(fmaf(ct, b.y - a.y, a.y));
    pp = E > 2.0f * kMec2 ? fmaf(ct, b.z - a.z, a.z) : 0.0f;
}
__device__ __forceinline__ void set_energy(Lane& L, const TransportParams& P, const Shared& sh) {
    const float lnE = __logf(L.E);
    int i; float t;
    if (P.tb.nonuni_E) {            // any increasing grid (a tabulation with absorption edges): guide bucket, then a short walk
        const float gk = fminf(fmaxf((lnE - P.tb.lnE0) * P.tb.inv_dg, 0.0f), (float)kEGuide);
        i = (int)sh.guide[(int)gk];
        while (i < P.tb.n_E - 2 && sh.lnEg[i + 1] <= lnE) ++i;
        t = fminf(fmaxf(__fdividef(lnE - sh.lnEg[i], sh.lnEg[i + 1] - sh.lnEg[i]), 0.0f), 1.0f);
    } else {
        float f = (lnE - P.tb.lnE0) * P.tb.inv_dlnE;
        f = fminf(fmaxf(f, 0.0f), (float)(P.tb.n_E - 1));
        i = min((int)f, P.tb.n_E - 2);
        t = f - (float)i;
    }
    L.ci = i; L.ct = t;
    L.mumaj = fmaf(t, sh.maj[i + 1] - sh.maj[i], sh.maj[i]);
}
__device__ __forceinline__ float stop_pow(const TransportParams& P, const Shared& sh, int m, float T) {
    float f = (__logf(T) - P.tb.lnT0) * P.tb.inv_dlnT;
    f = fminf(fmaxf(f, 0.0f), (float)(P.tb.n_T - 1));
    const int i = min((int)f, P.tb.n_T - 2);
    const float* r = sh.lnS + m * P.tb.n_T + i;
    return __expf(fmaf(f - (float)i, r[1] - r[0], r[0]));
}

// ---------------------------------------------------------------- frames
__device__ __forceinline__ void to_beam(const Geom& g, float x, float y, float z, float& u, float& v, float& w) {
    const float rx = x - g.src[0], ry = y - g.src[1], rz = z - g.src[2];
    u = g.au[0] * rx + g.au[1] * ry + g.au[2] * rz;
    v = g.av[0] * rx + g.av[1] * ry + g.av[2] * rz;
    w = g.aw[0] * rx + g.aw[1] * ry + g.aw[2] * rz;
}
__device__ __forceinline__ void dir_to_beam(const Geom& g, float x, float y, float z, float& u, float& v, float& w) {
    u = g.au[0] * x + g.au[1] * y + g.au[2] * z;
    v = g.av[0] * x + g.av[1] * y + g.av[2] * z;
    w = g.aw[0] * x + g.aw[1] * y + g.aw[2] * z;
}
__device__ __forceinline__ void dir_to_world(const Geom& g, float u, float v, float w, float& x, float& y, float& z) {
    x = u * g.au[0] + v * g.av[0] + w * g.aw[0];
    y = u * g.au[1] + v * g.av[1] + w * g.aw[1];
    z = u * g.au[2] + v * g.av[2] + w * g.aw[2];
}

// Rotate the unit vector d by polar (ct, st) and azimuth (cp, sp) using a branch-free orthonormal basis.
__device__ __forceinline__ void rotate(float& dx, float& dy, float& dz, float ct, float st, float cp, float sp) {
    const float sg = copysignf(1.0f, dz);
    const float a = -rcp(sg + dz), b = dx * dy * a;
    const float b1x = 1.0f + sg * dx * dx * a, b1y = sg * b, b1z = -sg * dx;
    const float b2x = b, b2y = sg + dy * dy * a, b2z = -dy;
    const float sc = st * cp, ss = st * sp;
    float nx = ct * dx + sc * b1x + ss * b2x;
    float ny = ct * dy + sc * b1y + ss * b2y;
    float nz = ct * dz + sc * b1z + ss * b2z;
    const float inv = rsqrtf(nx * nx + ny * ny + nz * nz);
    dx = nx * inv; dy = ny * inv; dz = nz * inv;
}

// voxel word through the read-only path; -DAEPID_VOX_EVICT_LAST=1 asks the L2 to keep voxel lines in preference to the streaming
// queue records and tallies (measured: profiles/r02_README.md)
#ifndef AEPID_VOX_EVICT_LAST
#define AEPID_VOX_EVICT_LAST 0
#endif
__device__ __forceinline__ uint32_t ld_vox(const uint32_t* p) {
#if AEPID_VOX_EVICT_LAST
    uint64_t pol; uint32_t v;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    asm volatile("ld.global.nc.L2::cache_hint.u32 %0, [%1], %2;" : "=r"(v) : "l"(p), "l"(pol));
    return v;
#else
    return __ldg(p);
#endif
}
// ---------------------------------------------------------------- tallies
// One RED per deposit.  -DAEPID_MATCH_TALLY=1 is the measured alternative north_star names (warp-aggregated atomics): the lanes
// of the warp that score into the same bin are found with match.any, their values are summed by shuffles and the lowest lane
// issues one RED (profiles/r02_README.md has both timings).
#ifndef AEPID_MATCH_TALLY
#define AEPID_MATCH_TALLY 0
#endif
__device__ __forceinline__ void tally_add(float* addr, float v) {
#if AEPID_MATCH_TALLY
    const unsigned act = __activemask();
    const unsigned peers = __match_any_sync(act, (unsigned long long)addr);
    float sum = 0.0f;
    for (unsigned m = peers; m; m &= m - 1u) sum += __shfl_sync(peers, v, __ffs(m) - 1);
    if ((threadIdx.x & 31u) == (unsigned)(__ffs(peers) - 1)) atomicAdd(addr, sum);
#else
    atomicAdd(addr, v);
#endif
}
__device__ __forceinline__ void flush_pending(Lane& L, const TransportParams& P) {
    if (L.pval != 0.0f) {
        AEPID_CHECK(L.pidx < P.nvox && F_BATCH(L.flags) < (uint32_t)P.n_batches);
        tally_add(P.ph_batch + (size_t)F_BATCH(L.flags) * P.nvox + L.pidx, L.pval);
        L.pval = 0.0f;
    }
}
__device__ __forceinline__ uint32_t vox_linear(const Geom& g, uint32_t v) {
    return (((v >> 20) & 1023u) * (uint32_t)g.ny + ((v >> 10) & 1023u)) * (uint32_t)g.nx + (v & 1023u);
}
__device__ __forceinline__ void dep_vox(Lane& L, const TransportParams& P, uint32_t idx, float e) {
    if (idx != L.pidx) { flush_pending(L, P); L.pidx = idx; }
    L.pval += e;
    L.a_ph += e;
}
// Energy e deposited at (u, v) of an EPID layer: scores the pixel and returns true if the layer is scored and
// (u, v) lies inside the image (SURVEY 8(c) "Geometry").
__device__ __noinline__ bool score_epid(uint32_t flags, float u, float v, float e) {
    if (!s_g.lscored[F_LAYER(flags)]) return false;
    const float fu = floorf((u + s_g.half_u) * s_g.inv_pitch), fv = floorf((v + s_g.half_v) * s_g.inv_pitch);
    if (!(fu >= 0.0f && fu < (float)s_g.nu && fv >= 0.0f && fv < (float)s_g.nv)) return false;
    AEPID_CHECK((size_t)fv * s_g.nu + (size_t)fu < s_npix);
    tally_add(s_ep_batch + (size_t)F_BATCH(flags) * s_npix + (size_t)fv * s_g.nu + (size_t)fu, e);
    return true;
}
__device__ __forceinline__ void dep_epid(Lane& L, float u, float v, float e) {
    if (score_epid(L.flags, u, v, e)) L.a_eps += e; else L.a_epo += e;
}
// deposit at the particle's position
__device__ __forceinline__ void dep_here(Lane& L, const TransportParams& P, float e) {
    const uint32_t reg = F_REGION(L.flags);
    if (reg == R_PHANTOM) dep_vox(L, P, vox_linear(P.g, L.vox), e);
    else if (reg == R_AIR) L.a_air += e;
    else dep_epid(L, L.x, L.y, e);
}

// ---------------------------------------------------------------- geometry
// Nearest boundary seen from AIR: kind 0 phantom AABB entry, 1 EPID top plane, 2 world exit.
struct AirHit { float t; int code; };      // code = kind | axis << 2
__device__ __noinline__ AirHit air_boundary(float x, float y, float z, float dx, float dy, float dz) {
    const Geom& g = s_g;
    float tn = -kInf, tf = kInf; int ax = 0; bool miss = false;
#define SLAB(P_, D_, LO_, HI_, A_)                                            \
    if (fabsf(D_) > 1e-20f) {                                                  \
        const float inv = rcp(D_);                                       \
        float t1 = ((LO_) - (P_)) * inv, t2 = ((HI_) - (P_)) * inv;           \
        if (t1 > t2) { const float t = t1; t1 = t2; t2 = t; }                  \
        if (t1 > tn) { tn = t1; ax = A_; }                                     \
        tf = fminf(tf, t2);                                                    \
    } else if ((P_) < (LO_) || (P_) >= (HI_)) miss = true;
    SLAB(x, dx, g.lox, g.hix, 0)
    SLAB(y, dy, g.loy, g.hiy, 1)
    SLAB(z, dz, g.loz, g.hiz, 2)
#undef SLAB
    float tb = (miss || !(tf > 0.0f) || tn >= tf) ? kInf : fmaxf(tn, 0.0f);
    int kind = 0;
    float pu, pv, pw, du, dv, dw;
    to_beam(g, x, y, z, pu, pv, pw);
    dir_to_beam(g, dx, dy, dz, du, dv, dw);
    if (dw > 0.0f) { const float te = fmaxf((g.sid - pw) / dw, 0.0f); if (te < tb) { tb = te; kind = 1; } }
    float tw = kInf;
    if (du > 0.0f) tw = fminf(tw, (kWorldHalf - pu) / du); else if (du < 0.0f) tw = fminf(tw, (-kWorldHalf - pu) / du);
    if (dv > 0.0f) tw = fminf(tw, (kWorldHalf - pv) / dv); else if (dv < 0.0f) tw = fminf(tw, (-kWorldHalf - pv) / dv);
    if (dw < 0.0f) tw = fminf(tw, (kWorldWMin - pw) / dw);
    tw = fmaxf(tw, 0.0f);
    if (tw < tb) { tb = tw; kind = 2; }
    AirHit r; r.t = tb; r.code = kind | (ax << 2);
    return r;
}
__device__ __forceinline__ float lateral_exit(float u, float v, float du, float dv) {
    float t = kInf;
    if (du > 0.0f) t = fminf(t, (kWorldHalf - u) / du); else if (du < 0.0f) t = fminf(t, (-kWorldHalf - u) / du);
    if (dv > 0.0f) t = fminf(t, (kWorldHalf - v) / dv); else if (dv < 0.0f) t = fminf(t, (-kWorldHalf - v) / dv);
    return fmaxf(t, 0.0f);
}
__device__ __forceinline__ float comp3(float a, float b, float c, int i) { return i == 0 ? a : (i == 1 ? b : c); }

// Particle at world position (already moved) enters the phantom through the face of `axis`.
__device__ __forceinline__ void enter_phantom(Lane& L, const TransportParams& P, int axis) {
    const Geom& g = P.g;
    const bool pos_dir = comp3(L.dx, L.dy, L.dz, axis) > 0.0f;
    if (axis == 0) L.x = pos_dir ? g.lox : g.hix; else if (axis == 1) L.y = pos_dir ? g.loy : g.hiy; else L.z = pos_dir ? g.loz : g.hiz;
    SET_REGION(L.flags, R_PHANTOM);
    if (F_TYPE(L.flags) != T_PHOTON) {                        // charged: voxel index + in-voxel fraction
        const float gx = (L.x - g.lox) * g.ihx, gy = (L.y - g.loy) * g.ihy, gz = (L.z - g.loz) * g.ihz;
        int ix = min(max((int)floorf(gx), 0), g.nx - 1), iy = min(max((int)floorf(gy), 0), g.ny - 1), iz = min(max((int)floorf(gz), 0), g.nz - 1);
        float fx = fminf(fmaxf(gx - (float)ix, 0.0f), 1.0f), fy = fminf(fmaxf(gy - (float)iy, 0.0f), 1.0f), fz = fminf(fmaxf(gz - (float)iz, 0.0f), 1.0f);
        if (axis == 0) { ix = pos_dir ? 0 : g.nx - 1; fx = pos_dir ? 0.0f : 1.0f; }
        else if (axis == 1) { iy = pos_dir ? 0 : g.ny - 1; fy = pos_dir ? 0.0f : 1.0f; }
        else { iz = pos_dir ? 0 : g.nz - 1; fz = pos_dir ? 0.0f : 1.0f; }
        L.x = fx; L.y = fy; L.z = fz;
        L.vox = (uint32_t)ix | ((uint32_t)iy << 10) | ((uint32_t)iz << 20);
        L.vlin = vox_linear(g, L.vox);
        AEPID_CHECK(L.vlin < P.nvox);
        L.cw = ld_vox(P.vox + L.vlin);
    }
}
__device__ __forceinline__ void enter_epid(Lane& L, const Geom& g) {       // position already on the top plane
    float pu, pv, pw, du, dv, dw;
    to_beam(g, L.x, L.y, L.z, pu, pv, pw);
    dir_to_beam(g, L.dx, L.dy, L.dz, du, dv, dw);
    L.x = pu; L.y = pv; L.z = 0.0f; L.dx = du; L.dy = dv; L.dz = dw;
    SET_REGION(L.flags, R_EPID); SET_LAYER(L.flags, 0);
}
// Phase Space 3 (reading A30): the particle has just arrived at the EPID top plane from the air (position
// (u, v, 0) and direction already in the beam frame).  One counter request per group of lanes that arrive together; the
// hand-off stays in flight, the record is a copy.
__device__ __noinline__ void record_ps3(float4* rec, unsigned long long* count, unsigned long long cap,
                                        float u, float v, float du, float dv, float dw, float E, uint32_t type, uint32_t hist) {
    const unsigned act = __activemask(), lane = threadIdx.x & 31u;
    const int leader = __ffs(act) - 1;
    unsigned long long base = 0;
    if ((int)lane == leader) base = atomicAdd(count, (unsigned long long)__popc(act));
    base = __shfl_sync(act, base, leader);
    const unsigned long long k = base + (unsigned long long)__popc(act & ((1u << lane) - 1u));
    if (k < cap) {
        __stcs(rec + 2 * k, make_float4(u, v, du, dv));
        __stcs(rec + 2 * k + 1, make_float4(dw, E, __uint_as_float(type), __uint_as_float(hist)));
    }
}
__device__ __forceinline__ void enter_epid_ps3(Lane& L, const TransportParams& P) {
    enter_epid(L, P.g);
    if (P.ps3) record_ps3(P.ps3, P.ps3_count, P.ps3_cap, L.x, L.y, L.dx, L.dy, L.dz, L.E, F_TYPE(L.flags), (uint32_t)(P.base + L.h));
}
__device__ __forceinline__ void epid_to_air(Lane& L, const Geom& g) {      // leaving through the top face
    const float u = L.x, v = L.y, w = g.sid;
    float x, y, z;
    dir_to_world(g, u, v, w, x, y, z);
    L.x = x + g.src[0]; L.y = y + g.src[1]; L.z = z + g.src[2];
    dir_to_world(g, L.dx, L.dy, L.dz, x, y, z);
    L.dx = x; L.dy = y; L.dz = z;
    SET_REGION(L.flags, R_AIR);
}
// charged particle in PHANTOM: (vox, fraction) -> world
__device__ __forceinline__ void frac_to_world(Lane& L, const Geom& g) {
    L.x = fmaf(((float)(L.vox & 1023u) + L.x), g.hx, g.lox);
    L.y = fmaf(((float)((L.vox >> 10) & 1023u) + L.y), g.hy, g.loy);
    L.z = fmaf(((float)((L.vox >> 20) & 1023u) + L.z), g.hz, g.loz);
}
// photon (world position in PHANTOM) -> charged particle representation
__device__ __forceinline__ void world_to_frac(const Geom& g, uint32_t vox, float& x, float& y, float& z) {
    const float gx = (x - g.lox) * g.ihx - (float)(vox & 1023u);
    const float gy = (y - g.loy) * g.ihy - (float)((vox >> 10) & 1023u);
    const float gz = (z - g.loz) * g.ihz - (float)((vox >> 20) & 1023u);
    x = fminf(fmaxf(gx, 0.0f), 1.0f); y = fminf(fmaxf(gy, 0.0f), 1.0f); z = fminf(fmaxf(gz, 0.0f), 1.0f);
}

// ---------------------------------------------------------------- class queues (protocol in the header comment)

// lane 0 claims up to `want` entries of ring r; returns count | first ticket << 32 (warp-uniform, all lanes call)
__device__ __noinline__ unsigned long long ring_claim(int r, int want) {
    int n = 0; uint32_t t = 0;
    if ((threadIdx.x & 31u) == 0 && want > 0 && (int)(s_snap[r] - *((volatile unsigned int*)(s_head + r))) > 0) {
        t = atomicAdd(s_head + r, (unsigned)want);
        n = min(max((int)(s_snap[r] - t), 0), want);
        if (n < want) atomicSub(s_head + r, (unsigned)(want - n));
    }
    n = __shfl_sync(FULL_MASK, n, 0);
    t = __shfl_sync(FULL_MASK, t, 0);
    return (unsigned long long)(uint32_t)n | ((unsigned long long)t << 32);
}
// lane 0 claims up to `want` of the new histories this phase may start (warp-uniform, all lanes call)
__device__ __noinline__ int budget_claim(int want) {
    int n = 0;
    if ((threadIdx.x & 31u) == 0 && want > 0 && *((volatile int*)&s_budget) > 0) {
        const int b = atomicSub(&s_budget, want);
        n = min(max(b, 0), want);
        if (n < want) atomicAdd(&s_budget, want - n);
    }
    return __shfl_sync(FULL_MASK, n, 0);
}

// Append a particle record to the queue of its class (one lane, divergent code); visible to poppers after the next barrier.
// Inlined, like take_credit: out of line the two cost 3.9 % of the kernel time on C3 in call overhead (profiles/r02_README.md).
__device__ __forceinline__ void queue_particle(float x, float y, float z, float dx, float dy, float dz, float E,
                                            uint32_t vox, uint32_t flags, uint32_t h, uint32_t pid, uint32_t blk, float R = 0.0f) {
    const int r = class_of(flags);
    const uint32_t tk = atomicAdd(s_tail + r, 1u);
    // the record written must not be one a pop of this phase may still read: tickets in flight fit one queue (header comment)
#ifdef AEPID_CHECKED
    AEPID_CHECK(r >= 0 && r < kClasses && tk - s_head0[r] <= s_pool_mask);
#endif
    uint4* rec = queue_rec(r, tk);
    __stcs(rec + 0, make_uint4(__float_as_uint(x), __float_as_uint(y), __float_as_uint(z), __float_as_uint(dx)));
    __stcs(rec + 1, make_uint4(__float_as_uint(dy), __float_as_uint(dz), __float_as_uint(E), vox));
    __stcs(rec + 2, make_uint4(flags, h, pid, blk));
    if (s_rec_vec == 4u) __stcs(rec + 3, make_uint4(__float_as_uint(R), 0u, 0u, 0u));
}
// Head room: s_live counts the particles alive in the CTA plus the credits lanes hold for secondaries they may create; it
// never exceeds kLiveMax, which is what keeps every queue from wrapping onto unread records (header comment).  A lane
// keeps at most one credit (its own, when its particle died, else a fresh one) and only runs an event that can create a
// secondary while it holds one.
__device__ __forceinline__ uint32_t take_credit() {
    if (*((volatile int*)&s_live) >= s_live_max) return kNone;
    if (atomicAdd(&s_live, 1) >= s_live_max) { atomicSub(&s_live, 1); return kNone; }
    return 1u;
}
__device__ __forceinline__ bool ensure_spare(Lane& L) {
    if (L.spare == kNone) L.spare = take_credit();
    return L.spare != kNone;
}
// A secondary goes straight into the queue of its class, on the lane's credit.  Without one (cannot happen: see
// ensure_spare; flagged) its energy is booked as escaped so that the ledger still closes.
__device__ __forceinline__ void spawn_from(Lane& L, float x, float y, float z, float dx, float dy, float dz, float E,
                                           uint32_t flags, uint32_t pid) {
    if (L.spare == kNone) { raise_error(2); L.a_esc += E + (F_TYPE(flags) == T_POSITRON ? 2.0f * kMec2 : 0.0f); return; }
    L.spare = kNone;
    queue_particle(x, y, z, dx, dy, dz, E, L.vox, flags, L.h, pid, 0u);
}
// Two 0.511 MeV photons, isotropic and back to back (reading A11): the lane becomes the first, the second is spawned.
// Position must already be in the frame photons use in this region.
__device__ __forceinline__ void annihilate(Lane& L, const TransportParams& P) {
    const uint4 r = rng_block(L, P);
    const float ct = 2.0f * u01(r.x) - 1.0f, st = sqrtf(fmaxf(0.0f, 1.0f - ct * ct));
    float sp, cp; __sincosf(2.0f * kPi * u01(r.y) - kPi, &sp, &cp);
    const float dx = st * cp, dy = st * sp, dz = ct;
    uint32_t f = L.flags & ~F_LEGA; SET_TYPE(f, T_PHOTON);
    spawn_from(L, L.x, L.y, L.z, -dx, -dy, -dz, kMec2, f, child_id(L, 1));
    L.pid = child_id(L, 0); L.blk = 0;
    L.flags = f;
    L.dx = dx; L.dy = dy; L.dz = dz; L.E = kMec2;
}

// ---------------------------------------------------------------- K4 interaction
// Klein-Nishina by epsilon-mixture rejection for a photon of energy L.E: eps = E'/E, t = 1 - cos(theta), x4 = a spare uniform for
// the azimuth; one Philox block per trial.
template <bool COUNT>
__device__ __forceinline__ void sample_kn(Lane& L, const TransportParams& P, float& eps, float& t, float& x4, uint32_t* cnt) {
    const float k = L.E * (1.0f / kMec2), e0 = rcp(1.0f + 2.0f * k), e02 = e0 * e0;
    const float a1 = -__logf(e0), a2 = 0.5f * (1.0f - e02);
#pragma unroll 1
    for (;;) {
        const uint4 r = rng_block_hot(L, P);                               // one block per trial
        const float x1 = u01(r.x), x2 = u01(r.y), x3 = u01(r.z); x4 = u01(r.w);
        if (COUNT) cnt[12]++;
        eps = (x1 * (a1 + a2) < a1) ? __expf(-x2 * a1) : sqrtf(fmaf(1.0f - e02, x2, e02));
        t = __fdividef(1.0f - eps, k * eps);
        const float g = 1.0f - __fdividef(eps * t * (2.0f - t), 1.0f + eps * eps);
        if (g >= x3) break;
    }
}
template <bool COUNT>
__device__ __forceinline__ void interact(Lane& L, const TransportParams& P, const Shared& sh, float xsel, float pe, float co, uint32_t* cnt) {
    const bool coupled = P.ph.mode != 0;
    const uint32_t reg = F_REGION(L.flags);
    if (xsel < pe) {                                                       // photoelectric: electron T = E along d
        if (COUNT) cnt[3]++;
        if (!coupled || L.E <= P.ph.ecut) { if (COUNT && coupled) { cnt[9]++; cnt[14]++; } dep_here(L, P, L.E); L.alive = false; return; }
        SET_TYPE(L.flags, T_ELECTRON);
        L.pid = child_id(L, 0); L.blk = 0; L.R = 0.0f;
        if (COUNT) { cnt[9]++; cnt[14]++; }
        if (reg == R_PHANTOM) { world_to_frac(P.g, L.vox, L.x, L.y, L.z); }
        return;
    }
    if (xsel < pe + co) {                                                  // Compton: Klein-Nishina by epsilon-mixture rejection
        if (COUNT) cnt[4]++;
        float eps, t, x4;
        sample_kn<COUNT>(L, P, eps, t, x4, cnt);
        const float ct = 1.0f - t, st = sqrtf(fmaxf(0.0f, t * (2.0f - t)));
        float sp, cp; __sincosf(2.0f * kPi * x4 - kPi, &sp, &cp);
        const float E0 = L.E, E1 = eps * E0, T = E0 - E1;
        float d1x = L.dx, d1y = L.dy, d1z = L.dz;
        rotate(d1x, d1y, d1z, ct, st, cp, sp);
        if (coupled && T > P.ph.ecut) {
            // electron from momentum conservation: queued with its own stream (reading A1)
            float ex = E0 * L.dx - E1 * d1x, ey = E0 * L.dy - E1 * d1y, ez = E0 * L.dz - E1 * d1z;
            const float inv = rsqrtf(ex * ex + ey * ey + ez * ez);
            float px = L.x, py = L.y, pz = L.z;
            if (reg == R_PHANTOM) world_to_frac(P.g, L.vox, px, py, pz);
            uint32_t f = L.flags; SET_TYPE(f, T_ELECTRON);
            if (COUNT) { cnt[9]++; cnt[14]++; }
            spawn_from(L, px, py, pz, ex * inv, ey * inv, ez * inv, T, f, child_id(L, 0));
        } else {                                                           // kerma, or electron born below its cutoff: local deposit
            dep_here(L, P, T);
            if (COUNT && coupled) { cnt[9]++; cnt[14]++; }
        }
        // the scattered photon keeps its own stream
        L.E = E1; L.dx = d1x; L.dy = d1y; L.dz = d1z;
        if (E1 < P.ph.pcut) { if (COUNT) cnt[13]++; dep_here(L, P, E1); L.alive = false; return; }
        set_energy(L, P, sh);
        return;
    }
    // pair production: uniform kinetic split, both along d (reading A10)
    if (COUNT) cnt[5]++;
    const float a = u01(rng_block(L, P).x);
    const float Ttot = L.E - 2.0f * kMec2;
    const float Tm = a * Ttot, Tp = Ttot - Tm;
    if (!coupled) {
        dep_here(L, P, Ttot);
        if (COUNT) cnt[9] += 2;
        annihilate(L, P);                                                  // 2 m_e c^2 re-emitted at the interaction point (A11)
        set_energy(L, P, sh);
        return;
    }
    if (COUNT) { cnt[9] += 2; cnt[14] += 2; }
    uint32_t fpos = L.flags; SET_TYPE(fpos, T_POSITRON);
    const uint32_t id0 = child_id(L, 0), id1 = child_id(L, 1);
    if (reg == R_PHANTOM) world_to_frac(P.g, L.vox, L.x, L.y, L.z);
    spawn_from(L, L.x, L.y, L.z, L.dx, L.dy, L.dz, Tp, fpos, id1);
    SET_TYPE(L.flags, T_ELECTRON);
    L.pid = id0; L.blk = 0; L.R = 0.0f;
    L.E = Tm;
}

// ---------------------------------------------------------------- photon flights.  Each returns true with (xsel, pe, co)
// set if the photon collides at its new position (K4 follows).
// K3: one Woodcock flight in the phantom.  One exponential optical depth nl is spent along the ray against a majorant that is
// piecewise constant in two regions (params.h Geom::glo): the global majorant mumaj(E) inside the body box G,
// f_out x mumaj(E) in the margin between G and the faces of the grid (air around a patient: f_out ~ 1e-3), so that the margin
// costs no virtual collisions and no extra Philox blocks: a ray meets the convex G in at most one chord, hence at most three
// segments margin | chord | margin.  The tentative collision is accepted with mu(voxel) / (majorant of its segment).  Same
// distribution as tracking against one global majorant (pin P4 of the oracle covers any exact tracker).
#ifndef AEPID_BODY_BOX
#define AEPID_BODY_BOX 1
#endif
__device__ __forceinline__ bool in_box(const float* lo, const float* hi, float x, float y, float z) {
    return x >= lo[0] && x < hi[0] && y >= lo[1] && y < hi[1] && z >= lo[2] && z < hi[2];
}
template <bool COUNT>
__device__ __forceinline__ bool woodcock_flight(Lane& L, const TransportParams& P, const Shared& sh, float& xsel, float& pe, float& co, uint32_t* cnt) {
    const Geom& g = P.g;
    const uint4 rr = rng_block_hot(L, P);
    const float u1 = u01(rr.x), u2 = u01(rr.y);
    if (COUNT) cnt[0]++;
    float nl = -__logf(u1), sig = L.mumaj;
    bool collide = false;
#if AEPID_BODY_BOX
    const float glo[3] = {g.glo[0], g.glo[1], g.glo[2]}, ghi[3] = {g.ghi[0], g.ghi[1], g.ghi[2]};
#else
    const float glo[3] = {g.lox, g.loy, g.loz}, ghi[3] = {g.hix, g.hiy, g.hiz};
#endif
    if (!AEPID_BODY_BOX || in_box(glo, ghi, L.x, L.y, L.z)) {          // (without a body box the start is not tested: a photon that
        const float s = __fdividef(nl, sig);                               //  came in through a high face sits ON it)
        const float nx = fmaf(s, L.dx, L.x), ny = fmaf(s, L.dy, L.y), nz = fmaf(s, L.dz, L.z);
        if (in_box(glo, ghi, nx, ny, nz)) { L.x = nx; L.y = ny; L.z = nz; collide = true; }   // the common case: ends inside G
#if AEPID_BODY_BOX
        else {                                                             // leaves G first: on to the margin with what is left of nl
            float tx = kInf, ty = kInf, tz = kInf;
            if (L.dx != 0.0f) tx = ((L.dx > 0.0f ? ghi[0] : glo[0]) - L.x) * rcp(L.dx);
            if (L.dy != 0.0f) ty = ((L.dy > 0.0f ? ghi[1] : glo[1]) - L.y) * rcp(L.dy);
            if (L.dz != 0.0f) tz = ((L.dz > 0.0f ? ghi[2] : glo[2]) - L.z) * rcp(L.dz);
            const float t = fmaxf(fminf(tx, fminf(ty, tz)), 0.0f);
            nl = fmaxf(nl - sig * t, 0.0f);
            L.x = fmaf(t, L.dx, L.x); L.y = fmaf(t, L.dy, L.y); L.z = fmaf(t, L.dz, L.z);
            sig = g.f_out * L.mumaj;
        }
#endif
    }
#if AEPID_BODY_BOX
    else {                                                                 // starts in the margin: does the ray meet G?
        sig = g.f_out * L.mumaj;
        float tn = -kInf, tf = kInf; bool miss = false;
#define SLAB(P_, D_, LO_, HI_)                                                 \
        if (fabsf(D_) > 1e-20f) {                                              \
            const float inv = rcp(D_);                                         \
            const float t1 = ((LO_) - (P_)) * inv, t2 = ((HI_) - (P_)) * inv;  \
            tn = fmaxf(tn, fminf(t1, t2)); tf = fminf(tf, fmaxf(t1, t2));      \
        } else if ((P_) < (LO_) || (P_) >= (HI_)) miss = true;
        SLAB(L.x, L.dx, glo[0], ghi[0])
        SLAB(L.y, L.dy, glo[1], ghi[1])
        SLAB(L.z, L.dz, glo[2], ghi[2])
#undef SLAB
        if (!miss && tf > 0.0f && tn < tf) {
            tn = fmaxf(tn, 0.0f);
            if (nl < sig * tn) {                                           // collides in the margin before G
                const float s = __fdividef(nl, sig);
                L.x = fmaf(s, L.dx, L.x); L.y = fmaf(s, L.dy, L.y); L.z = fmaf(s, L.dz, L.z); collide = true;
            } else {
                nl -= sig * tn;
                const float chord = tf - tn;
                if (nl < L.mumaj * chord) {                                // collides on the chord through G
                    const float s = tn + __fdividef(nl, L.mumaj);
                    L.x = fmaf(s, L.dx, L.x); L.y = fmaf(s, L.dy, L.y); L.z = fmaf(s, L.dz, L.z); collide = true; sig = L.mumaj;
                } else {                                                   // through G: the margin behind it
                    nl -= L.mumaj * chord;
                    L.x = fmaf(tf, L.dx, L.x); L.y = fmaf(tf, L.dy, L.y); L.z = fmaf(tf, L.dz, L.z);
                }
            }
        }
    }
#endif
    if (!collide) {
        // margin up to the faces of the grid (without a body box: the photon is on its way out, sig x t = 0 < nl never holds)
        float tx = kInf, ty = kInf, tz = kInf;
        if (L.dx != 0.0f) tx = ((L.dx > 0.0f ? g.hix : g.lox) - L.x) * rcp(L.dx);
        if (L.dy != 0.0f) ty = ((L.dy > 0.0f ? g.hiy : g.loy) - L.y) * rcp(L.dy);
        if (L.dz != 0.0f) tz = ((L.dz > 0.0f ? g.hiz : g.loz) - L.z) * rcp(L.dz);
        const float t = fmaxf(fminf(tx, fminf(ty, tz)), 0.0f);
        if (AEPID_BODY_BOX && nl < sig * t) {
            const float s = __fdividef(nl, sig);
            L.x = fmaf(s, L.dx, L.x); L.y = fmaf(s, L.dy, L.y); L.z = fmaf(s, L.dz, L.z); collide = true;
        } else {
            // left the grid: place on the AABB exit point, snapped onto the crossed face
            L.x = fmaf(t, L.dx, L.x); L.y = fmaf(t, L.dy, L.y); L.z = fmaf(t, L.dz, L.z);
            if (tx <= ty && tx <= tz) L.x = L.dx > 0.0f ? g.hix : g.lox;
            else if (ty <= tz) L.y = L.dy > 0.0f ? g.hiy : g.loy;
            else L.z = L.dz > 0.0f ? g.hiz : g.loz;
            SET_REGION(L.flags, R_AIR);
            return false;
        }
    }
    const int ix = min(max((int)((L.x - g.lox) * g.ihx), 0), g.nx - 1), iy = min(max((int)((L.y - g.loy) * g.ihy), 0), g.ny - 1),
              iz = min(max((int)((L.z - g.loz) * g.ihz), 0), g.nz - 1);
    AEPID_CHECK(ix >= 0 && iy >= 0 && iz >= 0 && ((size_t)iz * g.ny + iy) * g.nx + ix < P.nvox);
    const uint32_t w = ld_vox(P.vox + ((size_t)iz * g.ny + iy) * g.nx + ix);
    const float rho = __uint_as_float(w & ~31u);
    float pp;
    mu3(P, sh, (int)(w & 31u), L.ci, L.ct, L.E, pe, co, pp);
    xsel = u2 * sig;
    if (COUNT && rho * (pe + co + pp) > sig) cnt[31]++;                    // the majorant of the segment does not bound this voxel: must never happen
    if (xsel < rho * (pe + co + pp)) {
        xsel = __fdividef(xsel, rho);                                      // reuse the accept draw for the channel (reading A8)
        L.cw = w; L.vox = (uint32_t)ix | ((uint32_t)iy << 10) | ((uint32_t)iz << 20);
        return true;
    }
    return false;
}
// K2 + K6: a photon in AIR flies to wherever it goes.  One exponential optical depth is spent along the straight
// path through the air and - if the path crosses the whole EPID stack inside the world box - through the layers (a
// sequence of exponential flights that stop at boundaries is one exponential flight in optical depth).  Outcomes:
// collision in air or in a layer (true), phantom entry, EPID entry (the rare path that leaves the stack sideways:
// left to the layer-by-layer code), escape.
template <bool COUNT>
__device__ __forceinline__ bool air_transit(Lane& L, const TransportParams& P, const Shared& sh, float& xsel, float& pe, float& co, uint32_t* cnt) {
    const Geom& g = P.g;
    if (COUNT) cnt[1]++;
    const AirHit ah = air_boundary(L.x, L.y, L.z, L.dx, L.dy, L.dz);
    const uint4 rr = rng_block(L, P);
    const float u1 = u01(rr.x), u2 = u01(rr.y);
    float nl = -__logf(u1);
    float pp;
    mu3(P, sh, 0, L.ci, L.ct, L.E, pe, co, pp);
    float mt = pe + co + pp;
    const float mua = kRhoAir * mt;
    if (nl < mua * ah.t) {                                                 // collision in air
        const float s = __fdividef(nl, mua);
        L.x = fmaf(s, L.dx, L.x); L.y = fmaf(s, L.dy, L.y); L.z = fmaf(s, L.dz, L.z);
        xsel = u2 * mt;
        return true;
    }
    L.x = fmaf(ah.t, L.dx, L.x); L.y = fmaf(ah.t, L.dy, L.y); L.z = fmaf(ah.t, L.dz, L.z);
    const int kind = ah.code & 3;
    if (kind == 0) { enter_phantom(L, P, ah.code >> 2); return false; }
    if (kind == 2) { L.a_esc += L.E; L.alive = false; return false; }
    enter_epid_ps3(L, P);                                                  // (u, v, depth 0), beam-frame direction, dw > 0
    const float idw = rcp(L.dz);
    if (lateral_exit(L.x, L.y, L.dx, L.dy) < g.zt[g.n_layers] * idw) return false;   // leaves the stack sideways: layer-by-layer code
    nl -= mua * ah.t;
    if (COUNT) cnt[2]++;
#pragma unroll 1
    for (int l = 0; l < g.n_layers; ++l) {
        mu3(P, sh, g.lmat[l], L.ci, L.ct, L.E, pe, co, pp);
        mt = pe + co + pp;
        const float mul = g.lrho[l] * mt, path = (g.zt[l + 1] - g.zt[l]) * idw;
        if (nl < mul * path) {                                             // collision in layer l
            const float s = __fdividef(nl, mul) + g.zt[l] * idw;           // path length from the top plane
            L.x = fmaf(s, L.dx, L.x); L.y = fmaf(s, L.dy, L.y); L.z = fminf(fmaxf(s * L.dz, g.zt[l]), g.zt[l + 1]);
            SET_LAYER(L.flags, l);
            xsel = u2 * mt;
            return true;
        }
        nl -= mul * path;
    }
    L.a_esc += L.E; L.alive = false;                                       // through the bottom of the stack
    return false;
}
// K6: one flight of a photon inside the EPID, surface tracking layer by layer.
template <bool COUNT>
__device__ __forceinline__ bool epid_flight(Lane& L, const TransportParams& P, const Shared& sh, float& xsel, float& pe, float& co, uint32_t* cnt) {
    const Geom& g = P.g;
    const uint4 rr = rng_block(L, P);
    const float u1 = u01(rr.x), u2 = u01(rr.y);
    if (COUNT) cnt[2]++;
    const int l = F_LAYER(L.flags);
    float pp;
    mu3(P, sh, g.lmat[l], L.ci, L.ct, L.E, pe, co, pp);
    const float mt = pe + co + pp;
    const float s = __fdividef(-__logf(u1), g.lrho[l] * mt);
    float tf = kInf;
    if (L.dz > 0.0f) tf = (g.zt[l + 1] - L.z) / L.dz; else if (L.dz < 0.0f) tf = (g.zt[l] - L.z) / L.dz;
    tf = fmaxf(tf, 0.0f);
    const float tl = lateral_exit(L.x, L.y, L.dx, L.dy);
    if (s < tf && s < tl) { L.x = fmaf(s, L.dx, L.x); L.y = fmaf(s, L.dy, L.y); L.z = fmaf(s, L.dz, L.z); xsel = u2 * mt; return true; }
    if (tl < tf) { L.a_esc += L.E; L.alive = false; return false; }
    L.x = fmaf(tf, L.dx, L.x); L.y = fmaf(tf, L.dy, L.y);
    if (L.dz > 0.0f) {
        L.z = g.zt[l + 1];
        if (l + 1 >= g.n_layers) { L.a_esc += L.E; L.alive = false; }
        else SET_LAYER(L.flags, l + 1);
    } else {
        L.z = g.zt[l];
        if (l == 0) epid_to_air(L, g); else SET_LAYER(L.flags, l - 1);
    }
    return false;
}

// ---------------------------------------------------------------- K5 electron / positron step
// Energy loss of the step (midpoint rule), deposit-independent part shared by the two step functions.
// Class II (C2, physics mode 2, reading A31): sh.lnS holds the restricted stopping power, and the step also stops at the
// next hard (Moller) collision, whose distance is drawn with the cross section at the energy the step starts with (draw rh).
struct StepLoss { float s, dep, Tmid, sig, sigb; bool hard; };
template <int PH>
__device__ __forceinline__ StepLoss step_loss(Lane& L, const TransportParams& P, const Shared& sh, int m, float rho, float tb, uint32_t rh) {
    const float T = L.E;
    const float S = stop_pow(P, sh, m, T);
    StepLoss r;
    r.s = fminf(tb, fminf(__fdividef(P.ph.fE * T, rho * S), P.ph.smax));
    r.hard = false; r.sig = 0.0f; r.sigb = 0.0f;
    if (PH == 2 || PH == 3) {
        float f = (__logf(T) - P.tb.lnT0) * P.tb.inv_dlnT;
        f = fminf(fmaxf(f, 0.0f), (float)(P.tb.n_T - 1));
        const int i = min((int)f, P.tb.n_T - 2);
        const float* q = sh.sig + m * P.tb.n_T + i;
        const float sg = fmaf(f - (float)i, q[1] - q[0], q[0]);
        r.sig = sg;
        if (PH == 3) { const float* qb = q + P.tb.n_mat * P.tb.n_T; r.sigb = fmaf(f - (float)i, qb[1] - qb[0], qb[0]); }   // bremsstrahlung part
        const float sh_ = sg > 0.0f ? __fdividef(-__logf(u01(rh)), rho * sg) : kInf;
        r.hard = sh_ < r.s;                                                // strictly inside the step: a step that ends on a face does not collide
        r.s = fminf(r.s, sh_);
    }
    const float S2 = stop_pow(P, sh, m, T - 0.5f * rho * r.s * S);        // midpoint rule
    const float dE = fminf(T, rho * r.s * S2);
    const float Tn = T - dE;
    r.dep = T - Tn;                                                        // exactly what the particle loses (ledger closes)
    r.Tmid = T - 0.5f * dE;
    L.E = Tn;
    return r;
}
// Highland deflection angles for a step of mass thickness rho*s at mid-step energy Tmid from the draws (ra, rb)
// (reading A13).  A zero-length step gives theta = 0, i.e. no deflection.
__device__ __forceinline__ void highland(const Shared& sh, int m, float rho_s, float Tmid, uint32_t ra, uint32_t rb,
                                         float& ct, float& st, float& cp, float& sp) {
    const float t = fmaxf(rho_s * sh.invX0[m], 1e-30f);
    const float ibpc = __fdividef(Tmid + kMec2, Tmid * (Tmid + 2.0f * kMec2));
    const float th0 = 13.6f * ibpc * sqrtf(t) * fmaxf(0.25f, fmaf(0.038f, __logf(t), 1.0f));
    const float th = rho_s > 0.0f ? fminf(kPi, th0 * sqrtf(-2.0f * __logf(u01(ra)))) : 0.0f;
    __sincosf(th, &st, &ct);
    __sincosf(2.0f * kPi * u01(rb) - kPi, &sp, &cp);
}
// Hard (Moller) collision of a charged particle of kinetic energy L.E > 2 Tc where its step ended (reading A31): the energy
// transfer W = eps E, eps in [Tc / E, 1/2], is sampled from the Moller density by rejection from 1 / eps^2 (one Philox block
// per trial: two draws for the trial, the third for the azimuth); both outgoing directions follow from energy-momentum
// conservation.  The delta ray is an electron queued on the lane's credit, the lane goes on with the rest.
template <bool COUNT>
__device__ __forceinline__ void moller_event(Lane& L, const TransportParams& P, uint32_t* cnt) {
    const float T = L.E, tau = T * (1.0f / kMec2), a = __fdividef(P.ph.ecut, T);
    const float t1 = rcp(tau + 1.0f), c1 = tau * tau * t1 * t1, c2 = (2.0f * tau + 1.0f) * t1 * t1;
    const float gmax = 2.0f + 0.25f * c1;
    float eps, phi;
#pragma unroll 1
    for (;;) {
        const uint4 r = rng_block(L, P);
        eps = __fdividef(a, 1.0f - u01(r.x) * (1.0f - 2.0f * a));
        const float x = __fdividef(eps, 1.0f - eps);
        const float g = 1.0f + x * x + c1 * eps * eps - c2 * x;
        phi = 2.0f * kPi * u01(r.z) - kPi;
        if (u01(r.y) * gmax <= g) break;
    }
    const float W = eps * T, T1 = T - W;
    const float cd = sqrtf(__fdividef(W * (T + 2.0f * kMec2), T * (W + 2.0f * kMec2)));
    const float cpm = sqrtf(__fdividef(T1 * (T + 2.0f * kMec2), T * (T1 + 2.0f * kMec2)));
    float sphi, cphi; __sincosf(phi, &sphi, &cphi);
    float ex = L.dx, ey = L.dy, ez = L.dz;
    rotate(ex, ey, ez, cd, sqrtf(fmaxf(0.0f, 1.0f - cd * cd)), -cphi, -sphi);     // the delta ray: opposite azimuth
    uint32_t f = L.flags; SET_TYPE(f, T_ELECTRON);
    if (COUNT) { cnt[9]++; cnt[14]++; }
    spawn_from(L, L.x, L.y, L.z, ex, ey, ez, W, f, child_id(L, 0));
    rotate(L.dx, L.dy, L.dz, cpm, sqrtf(fmaxf(0.0f, 1.0f - cpm * cpm)), cphi, sphi);
    L.E = T1;
}
// Bremsstrahlung event of a charged particle of kinetic energy L.E > kc = the photon cut-off (physics mode 3, reading A32):
// photon energy k in [kc, E] from (4/3 - 4/3 y + y^2) / k, y = k / E, by rejection from 1/k (one Philox block per trial);
// the photon leaves along the particle's direction with its own stream, the particle keeps E - k.  IN_PHANTOM: the lane
// holds voxel fractions, the photon record wants the world position.
template <bool COUNT, bool IN_PHANTOM>
__device__ __forceinline__ void brems_event(Lane& L, const TransportParams& P, uint32_t* cnt) {
    const float T = L.E, lr = __logf(__fdividef(T, P.ph.pcut));
    float k;
#pragma unroll 1
    for (;;) {
        const uint4 r = rng_block(L, P);
        k = P.ph.pcut * __expf(u01(r.x) * lr);
        const float y = __fdividef(k, T);
        if (u01(r.y) <= 1.0f - y + 0.75f * y * y) break;
    }
    k = fminf(k, T);
    float px = L.x, py = L.y, pz = L.z;
    if (IN_PHANTOM) {
        px = fmaf(((float)(L.vox & 1023u) + L.x), P.g.hx, P.g.lox);
        py = fmaf(((float)((L.vox >> 10) & 1023u) + L.y), P.g.hy, P.g.loy);
        pz = fmaf(((float)((L.vox >> 20) & 1023u) + L.z), P.g.hz, P.g.loz);
    }
    uint32_t f = L.flags; SET_TYPE(f, T_PHOTON);
    if (COUNT) cnt[9]++;
    spawn_from(L, px, py, pz, L.dx, L.dy, L.dz, k, f, child_id(L, 0));
    L.E = T - k;
}
// charged particle at or below its cutoff (PAPER.md:104, 200 keV): local deposit; a positron annihilates
template <bool COUNT>
__device__ __forceinline__ void stop_charged(Lane& L, const TransportParams& P, uint32_t* cnt) {
    dep_here(L, P, L.E);
    if (F_TYPE(L.flags) == T_POSITRON) {
        if (F_REGION(L.flags) == R_PHANTOM) frac_to_world(L, P.g);
        if (COUNT) cnt[9] += 2;
        annihilate(L, P);
    } else L.alive = false;
}
// One step inside the phantom with the draws (ra, rb): the hot loop of the whole path, written without branches up
// to the rare exit from the grid (selects instead of per-axis branches: a face is crossed by a few lanes of nearly
// every warp, so divergent code there is paid by all).  The particle is above its cutoff.  Invariant of class E: the
// pending deposit of the lane belongs to the current voxel (L.pidx == L.vlin, set when the particle is loaded).
template <bool COUNT, int PH>
__device__ __forceinline__ void electron_step_phantom(Lane& L, const TransportParams& P, const Shared& sh, uint32_t ra, uint32_t rb, uint32_t rh, uint32_t rw, uint32_t* cnt) {
    constexpr bool C2 = PH == 2 || PH == 3, PHANTOM_FRAME = true;
    const Geom& g = P.g;
    const float rho = __uint_as_float(L.cw & ~31u); const int m = (int)(L.cw & 31u);
    // distance to the voxel face in the direction of travel, per axis (a vanishing component gives a huge distance)
    const float tx = (L.dx > 0.0f ? 1.0f - L.x : L.x) * g.hx * rcp(fabsf(L.dx) + 1e-30f);
    const float ty = (L.dy > 0.0f ? 1.0f - L.y : L.y) * g.hy * rcp(fabsf(L.dy) + 1e-30f);
    const float tz = (L.dz > 0.0f ? 1.0f - L.z : L.z) * g.hz * rcp(fabsf(L.dz) + 1e-30f);
    const float tb = fmaxf(fminf(tx, fminf(ty, tz)), 0.0f);
    const bool ax0 = tx <= ty && tx <= tz, ax1 = !ax0 && ty <= tz, ax2 = !ax0 && !ax1;
    const StepLoss sl = step_loss<PH>(L, P, sh, m, rho, tb, rh);
    if (COUNT) { cnt[6]++; if (!(sl.s > 0.0f)) cnt[15]++; }
    L.pval += sl.dep; L.a_ph += sl.dep;
    L.x = fmaf(sl.s * g.ihx, L.dx, L.x); L.y = fmaf(sl.s * g.ihy, L.dy, L.y); L.z = fmaf(sl.s * g.ihz, L.dz, L.z);
    float ct, st, cp, sp;
    highland(sh, m, rho * sl.s, sl.Tmid, ra, rb, ct, st, cp, sp);
    // the step ended on a face: neighbouring voxel (index +-1 on the crossed axis, never re-derived from the position) or out of the grid
    const bool cross = sl.s == tb;
    const bool up = (ax0 ? L.dx : (ax1 ? L.dy : L.dz)) > 0.0f;
    const float nf = up ? 0.0f : 1.0f;
    const int sh10 = ax0 ? 0 : (ax1 ? 10 : 20);
    const int nmax = ax0 ? g.nx : (ax1 ? g.ny : g.nz);
    const int stride = ax0 ? 1 : (ax1 ? g.nx : g.nx * g.ny);
    const int ni = (int)((L.vox >> sh10) & 1023u) + (up ? 1 : -1);
    const bool inside = ni >= 0 && ni < nmax;
    L.x = (cross && ax0) ? nf : L.x; L.y = (cross && ax1) ? nf : L.y; L.z = (cross && ax2) ? nf : L.z;
    if (cross && inside) {
        if (L.pval != 0.0f) tally_add(P.ph_batch + (size_t)F_BATCH(L.flags) * P.nvox + L.vlin, L.pval);
        L.pval = 0.0f;
        L.vox = (L.vox & ~(1023u << sh10)) | ((uint32_t)ni << sh10);
        L.vlin += (uint32_t)(up ? stride : -stride);
        L.pidx = L.vlin;
        AEPID_CHECK(L.vlin < P.nvox && L.vlin == vox_linear(g, L.vox));
        L.cw = ld_vox(P.vox + L.vlin);
    }
    if (cross && !inside) {                                                // rare: leaves the grid
        frac_to_world(L, g);                                               // uses the old index; then snap the crossed axis
        if (ax0) L.x = up ? g.hix : g.lox; else if (ax1) L.y = up ? g.hiy : g.loy; else L.z = up ? g.hiz : g.loz;
        SET_REGION(L.flags, R_AIR);
    }
    rotate(L.dx, L.dy, L.dz, ct, st, cp, sp);
    if (C2 && sl.hard) {                                                   // hard event at the end of the step, with the energy left;
        if (PH == 3 && u01(rw) * sl.sig < sl.sigb) {                       // its kind by the cross sections the distance was drawn with
            if (L.E > P.ph.pcut) brems_event<COUNT, PHANTOM_FRAME>(L, P, cnt);
        } else if (L.E > 2.0f * P.ph.ecut) moller_event<COUNT>(L, P, cnt);
    }
}
// one step in the air or inside the EPID (the particle is above its cutoff)
template <bool COUNT, int PH>
__device__ __forceinline__ void electron_step_outside(Lane& L, const TransportParams& P, const Shared& sh, uint32_t ra, uint32_t rb, uint32_t rh, uint32_t rw, uint32_t* cnt) {
    constexpr bool C2 = PH == 2 || PH == 3, PHANTOM_FRAME = false;
    const Geom& g = P.g;
    const bool in_air = F_REGION(L.flags) == R_AIR;
    float rho, tb; int m, axis = 0, kind = 0;
    if (in_air) {
        rho = kRhoAir; m = 0;
        // Open air: farther than s_max from the phantom box, the EPID top plane and the world walls, so the step (at most
        // s_max long) cannot reach a boundary and the exact distances are not needed.  An electron crosses the air gap in
        // hundreds of such steps.
        const float far = P.ph.smax * 1.0001f;
        const float gap = fmaxf(fmaxf(fmaxf(g.lox - L.x, L.x - g.hix), fmaxf(g.loy - L.y, L.y - g.hiy)), fmaxf(g.loz - L.z, L.z - g.hiz));
        float pu, pv, pw;
        to_beam(g, L.x, L.y, L.z, pu, pv, pw);
        const float wall = fminf(fminf(kWorldHalf - fabsf(pu), kWorldHalf - fabsf(pv)), fminf(pw - kWorldWMin, g.sid - pw));
        if (gap > far && wall > far) { tb = kInf; }
        else {
            const AirHit ah = air_boundary(L.x, L.y, L.z, L.dx, L.dy, L.dz);
            tb = ah.t; kind = ah.code & 3; axis = ah.code >> 2;
        }
    } else {
        const int l = F_LAYER(L.flags);
        rho = g.lrho[l]; m = g.lmat[l];
        float tf = kInf;
        if (L.dz > 0.0f) tf = (g.zt[l + 1] - L.z) / L.dz; else if (L.dz < 0.0f) tf = (g.zt[l] - L.z) / L.dz;
        tf = fmaxf(tf, 0.0f);
        const float tl = lateral_exit(L.x, L.y, L.dx, L.dy);
        if (tl < tf) { tb = tl; kind = 2; } else { tb = tf; kind = 0; }
    }
    const StepLoss sl = step_loss<PH>(L, P, sh, m, rho, tb, rh);
    if (COUNT && !(sl.s > 0.0f)) cnt[15]++;
    if (in_air) { if (COUNT) cnt[7]++; L.a_air += sl.dep; }
    else { if (COUNT) cnt[8]++; dep_epid(L, fmaf(0.5f * sl.s, L.dx, L.x), fmaf(0.5f * sl.s, L.dy, L.y), sl.dep); }   // pixel of the step midpoint (A24)
    L.x = fmaf(sl.s, L.dx, L.x); L.y = fmaf(sl.s, L.dy, L.y); L.z = fmaf(sl.s, L.dz, L.z);
    float ct, st, cp, sp;
    highland(sh, m, rho * sl.s, sl.Tmid, ra, rb, ct, st, cp, sp);
    if (sl.s == tb) {                                                      // the step ended on a boundary
        const float e_out = L.E + (F_TYPE(L.flags) == T_POSITRON ? 2.0f * kMec2 : 0.0f);
        if (in_air) {
            if (kind == 0) enter_phantom(L, P, axis);
            else if (kind == 1) enter_epid_ps3(L, P);
            else { L.a_esc += e_out; L.alive = false; return; }
        } else {
            const int l = F_LAYER(L.flags);
            if (kind == 2) { L.a_esc += e_out; L.alive = false; return; }
            if (L.dz > 0.0f) {
                L.z = g.zt[l + 1];
                if (l + 1 >= g.n_layers) { L.a_esc += e_out; L.alive = false; return; }
                SET_LAYER(L.flags, l + 1);
            } else {
                L.z = g.zt[l];
                if (l == 0) epid_to_air(L, g); else SET_LAYER(L.flags, l - 1);
            }
        }
    }
    rotate(L.dx, L.dy, L.dz, ct, st, cp, sp);
    if (C2 && sl.hard) {                                                   // hard event at the end of the step, with the energy left;
        if (PH == 3 && u01(rw) * sl.sig < sl.sigb) {                       // its kind by the cross sections the distance was drawn with
            if (L.E > P.ph.pcut) brems_event<COUNT, PHANTOM_FRAME>(L, P, cnt);
        } else if (L.E > 2.0f * P.ph.ecut) moller_event<COUNT>(L, P, cnt);
    }
}
// ---------------------------------------------------------------- physics mode 4 (reading A38): multi-voxel steps with a random hinge
// A step loses dE_k = f_E T_k in two legs, xi dE_k before the hinge and the rest after it; faces end SEGMENTS, not steps.  The
// lane carries the budget of its leg (L.R) and the leg bit (F_LEGA); everything else about the step is recomputed at the hinge
// from the step's own Philox block (the last one the particle drew): xi gives T_k = T / (1 - xi f_E), (xi_a, xi_b) the deflection.
__device__ __forceinline__ void hinge_begin_step(Lane& L, const TransportParams& P) {
    const uint4 r = rng_block_hot(L, P);
    L.R = u01(r.x) * P.ph.fE * L.E;
    L.flags |= F_LEGA;
}
__device__ __forceinline__ void hinge_deflect(Lane& L, const TransportParams& P, const Shared& sh, int m) {
    L.blk--;                                                               // the step's block again: (xi, xi_a, xi_b)
    const uint4 r = rng_block_hot(L, P);
    const float xi = u01(r.x);
    const float Tk = __fdividef(L.E, 1.0f - xi * P.ph.fE), dEk = P.ph.fE * Tk, Tm = Tk - 0.5f * dEk;
    float ct, st, cp, sp;
    highland(sh, m, __fdividef(dEk, stop_pow(P, sh, m, Tm)), Tm, r.y, r.z, ct, st, cp, sp);
    rotate(L.dx, L.dy, L.dz, ct, st, cp, sp);
    L.R = (1.0f - xi) * dEk;
    L.flags &= ~F_LEGA;
}
// length and loss of one segment in medium (rho, m): to the face at tb, or to where the leg's budget is used up
struct Segment { float s, dE; bool on_face; };
__device__ __forceinline__ Segment hinge_segment(Lane& L, const TransportParams& P, const Shared& sh, int m, float rho, float tb) {
    Segment g;
    const float T = L.E;
    const float sR = __fdividef(L.R, rho * stop_pow(P, sh, m, T - 0.5f * L.R));
    g.on_face = !(sR < tb);
    if (g.on_face) {
        const float S = stop_pow(P, sh, m, T);
        g.s = tb;
        g.dE = fminf(T, rho * tb * stop_pow(P, sh, m, T - 0.5f * rho * tb * S));   // midpoint rule, as in mode 1
        L.R -= g.dE;
    } else { g.s = sR; g.dE = fminf(L.R, T); L.R = 0.0f; }
    const float Tn = T - g.dE;
    g.dE = T - Tn;                                                         // exactly what the particle loses (ledger closes)
    L.E = Tn;
    return g;
}
template <bool COUNT>
__device__ __forceinline__ void hinge_segment_phantom(Lane& L, const TransportParams& P, const Shared& sh, uint32_t* cnt) {
    const Geom& g = P.g;
    const float rho = __uint_as_float(L.cw & ~31u); const int m = (int)(L.cw & 31u);
    if (!(L.R > 0.0f) && !(L.flags & F_LEGA)) { hinge_begin_step(L, P); if (COUNT) cnt[15]++; }
    const float tx = (L.dx > 0.0f ? 1.0f - L.x : L.x) * g.hx * rcp(fabsf(L.dx) + 1e-30f);
    const float ty = (L.dy > 0.0f ? 1.0f - L.y : L.y) * g.hy * rcp(fabsf(L.dy) + 1e-30f);
    const float tz = (L.dz > 0.0f ? 1.0f - L.z : L.z) * g.hz * rcp(fabsf(L.dz) + 1e-30f);
    const float tb = fmaxf(fminf(tx, fminf(ty, tz)), 0.0f);
    const bool ax0 = tx <= ty && tx <= tz, ax1 = !ax0 && ty <= tz, ax2 = !ax0 && !ax1;
    const Segment sg = hinge_segment(L, P, sh, m, rho, tb);
    if (COUNT) cnt[6]++;
    L.pval += sg.dE; L.a_ph += sg.dE;
    L.x = fmaf(sg.s * g.ihx, L.dx, L.x); L.y = fmaf(sg.s * g.ihy, L.dy, L.y); L.z = fmaf(sg.s * g.ihz, L.dz, L.z);
    if (sg.on_face) {
        const bool up = (ax0 ? L.dx : (ax1 ? L.dy : L.dz)) > 0.0f;
        const float nf = up ? 0.0f : 1.0f;
        const int sh10 = ax0 ? 0 : (ax1 ? 10 : 20);
        const int nmax = ax0 ? g.nx : (ax1 ? g.ny : g.nz);
        const int stride = ax0 ? 1 : (ax1 ? g.nx : g.nx * g.ny);
        const int ni = (int)((L.vox >> sh10) & 1023u) + (up ? 1 : -1);
        L.x = ax0 ? nf : L.x; L.y = ax1 ? nf : L.y; L.z = ax2 ? nf : L.z;
        if (ni >= 0 && ni < nmax) {
            if (L.pval != 0.0f) tally_add(P.ph_batch + (size_t)F_BATCH(L.flags) * P.nvox + L.vlin, L.pval);
            L.pval = 0.0f;
            L.vox = (L.vox & ~(1023u << sh10)) | ((uint32_t)ni << sh10);
            L.vlin += (uint32_t)(up ? stride : -stride);
            L.pidx = L.vlin;
            AEPID_CHECK(L.vlin < P.nvox && L.vlin == vox_linear(g, L.vox));
            L.cw = ld_vox(P.vox + L.vlin);
        } else {                                                           // leaves the grid
            frac_to_world(L, g);
            if (ax0) L.x = up ? g.hix : g.lox; else if (ax1) L.y = up ? g.hiy : g.loy; else L.z = up ? g.hiz : g.loz;
            SET_REGION(L.flags, R_AIR);
        }
    }
    if (!(L.R > 0.0f) && (L.flags & F_LEGA)) hinge_deflect(L, P, sh, m);  // the hinge, in the medium of the segment that ended the leg
}
template <bool COUNT>
__device__ __forceinline__ void hinge_segment_outside(Lane& L, const TransportParams& P, const Shared& sh, uint32_t* cnt) {
    const Geom& g = P.g;
    const bool in_air = F_REGION(L.flags) == R_AIR;
    float rho, tb; int m, axis = 0, kind = 0;
    if (in_air) {
        rho = kRhoAir; m = 0;
        const AirHit ah = air_boundary(L.x, L.y, L.z, L.dx, L.dy, L.dz);
        tb = ah.t; kind = ah.code & 3; axis = ah.code >> 2;
    } else {
        const int l = F_LAYER(L.flags);
        rho = g.lrho[l]; m = g.lmat[l];
        float tf = kInf;
        if (L.dz > 0.0f) tf = (g.zt[l + 1] - L.z) / L.dz; else if (L.dz < 0.0f) tf = (g.zt[l] - L.z) / L.dz;
        tf = fmaxf(tf, 0.0f);
        const float tl = lateral_exit(L.x, L.y, L.dx, L.dy);
        if (tl < tf) { tb = tl; kind = 2; } else { tb = tf; kind = 0; }
    }
    if (!(L.R > 0.0f) && !(L.flags & F_LEGA)) { hinge_begin_step(L, P); if (COUNT) cnt[15]++; }
    const Segment sg = hinge_segment(L, P, sh, m, rho, tb);
    if (in_air) { if (COUNT) cnt[7]++; L.a_air += sg.dE; }
    else { if (COUNT) cnt[8]++; dep_epid(L, fmaf(0.5f * sg.s, L.dx, L.x), fmaf(0.5f * sg.s, L.dy, L.y), sg.dE); }   // pixel of the segment's mid-point (A24)
    L.x = fmaf(sg.s, L.dx, L.x); L.y = fmaf(sg.s, L.dy, L.y); L.z = fmaf(sg.s, L.dz, L.z);
    if (sg.on_face) {
        const float e_out = L.E + (F_TYPE(L.flags) == T_POSITRON ? 2.0f * kMec2 : 0.0f);
        if (in_air) {
            if (kind == 0) enter_phantom(L, P, axis);
            else if (kind == 1) enter_epid_ps3(L, P);
            else { L.a_esc += e_out; L.alive = false; return; }
        } else {
            const int l = F_LAYER(L.flags);
            if (kind == 2) { L.a_esc += e_out; L.alive = false; return; }
            if (L.dz > 0.0f) {
                L.z = g.zt[l + 1];
                if (l + 1 >= g.n_layers) { L.a_esc += e_out; L.alive = false; return; }
                SET_LAYER(L.flags, l + 1);
            } else {
                L.z = g.zt[l];
                if (l == 0) epid_to_air(L, g); else SET_LAYER(L.flags, l - 1);
            }
        }
    }
    if (!(L.R > 0.0f) && (L.flags & F_LEGA)) hinge_deflect(L, P, sh, m);
}

// K5 for one lane: up to kStepsE / kStepsX consecutive steps per event, one Philox block per two steps
template <bool COUNT, bool PHANTOM, int PH>
__device__ __forceinline__ void charged_event(Lane& L, const TransportParams& P, const Shared& sh, uint32_t* cnt) {
    constexpr bool C2 = PH == 2 || PH == 3;
    if (L.E <= P.ph.ecut) { stop_charged<COUNT>(L, P, cnt); return; }
    if (PH == 4) {
#pragma unroll 1
        for (int k = 0; k < (PHANTOM ? kStepsE : kStepsX); ++k) {
            if (PHANTOM) hinge_segment_phantom<COUNT>(L, P, sh, cnt); else hinge_segment_outside<COUNT>(L, P, sh, cnt);
            if (!L.alive) break;
            if (L.E <= P.ph.ecut) {
                if (F_TYPE(L.flags) == T_ELECTRON) { dep_here(L, P, L.E); L.alive = false; }
                break;
            }
            if ((F_REGION(L.flags) == R_PHANTOM) != PHANTOM) break;
        }
        return;
    }
    uint4 r = PHANTOM ? rng_block_hot(L, P) : rng_block(L, P);
#pragma unroll 1
    for (int k = 0; k < (PHANTOM ? kStepsE : kStepsX); ++k) {
        if (C2) {                                                          // a block per step: deflection (x, y), hard-collision distance (z), kind (w)
            if (k) r = PHANTOM ? rng_block_hot(L, P) : rng_block(L, P);
            if (PHANTOM) electron_step_phantom<COUNT, PH>(L, P, sh, r.x, r.y, r.z, r.w, cnt);
            else electron_step_outside<COUNT, PH>(L, P, sh, r.x, r.y, r.z, r.w, cnt);
        } else {
            if (k && !(k & 1)) r = PHANTOM ? rng_block_hot(L, P) : rng_block(L, P);
            if (PHANTOM) electron_step_phantom<COUNT, 1>(L, P, sh, (k & 1) ? r.z : r.x, (k & 1) ? r.w : r.y, 0u, 0u, cnt);
            else electron_step_outside<COUNT, 1>(L, P, sh, (k & 1) ? r.z : r.x, (k & 1) ? r.w : r.y, 0u, 0u, cnt);
        }
        if (!L.alive) break;
        if (L.E <= P.ph.ecut) {                                            // cutoff reached: an electron stops here and now;
            if (F_TYPE(L.flags) == T_ELECTRON) { dep_here(L, P, L.E); L.alive = false; }   // a positron first needs a credit for its second photon
            break;
        }
        if ((F_REGION(L.flags) == R_PHANTOM) != PHANTOM) break;
        if (C2 && L.spare == kNone) break;                                 // the credit went into a delta ray: the next step needs a new one
    }
}

// ---------------------------------------------------------------- collimation stage
// A photon sampled from Phase Space 1 is followed through the jaws and the MLC down to the Phase Space 2 plane (readings
// A35-A37): inside the w-range of a slab every point outside the opening of its row is tungsten, everything else is air;
// charged particles are not followed (their energy stays in the head: the ledger's air channel), annihilation quanta born in
// the head are dropped, a photon that turns upstream or leaves the world sideways has escaped.  The oracle tracks the whole
// stage by Woodcock flights against the tungsten coefficient; the same distribution costs less here: air gaps and slab
// crossings that provably stay inside the openings are one exponential flight in air, and only a slab whose tungsten the ray
// may touch is tracked by Woodcock flights (exact for any arrangement of openings), ended at the slab's faces.
__device__ __forceinline__ bool head_blocked(const Head& H, int k, float x, float y) {
    const float across = H.axis[k] == 0 ? y : x, along = H.axis[k] == 0 ? x : y;
    const float fr = floorf((across - H.row0[k]) * H.inv_pitch[k]);
    if (!(fr >= 0.0f && fr < (float)H.n_rows[k])) return true;
    const int r = H.off[k] + (int)fr;
    return !(along >= __ldg(H.lo + r) && along < __ldg(H.hi + r));
}
// does the straight path from (x, y, w) to the bottom face of slab k stay inside the openings of every row it passes?
__device__ __forceinline__ bool head_clear(const Head& H, int k, float x, float y, float w, float dx, float dy, float dz) {
    const float t = (H.w1[k] - w) / dz;
    const float x1 = fmaf(t, dx, x), y1 = fmaf(t, dy, y);
    const bool ax0 = H.axis[k] == 0;
    const float a0 = ax0 ? y : x, a1 = ax0 ? y1 : x1, l0 = ax0 ? x : y, l1 = ax0 ? x1 : y1;
    const float f0 = floorf((fminf(a0, a1) - H.row0[k]) * H.inv_pitch[k]), f1 = floorf((fmaxf(a0, a1) - H.row0[k]) * H.inv_pitch[k]);
    if (!(f0 >= 0.0f && f1 < (float)H.n_rows[k])) return false;
    const float lmin = fminf(l0, l1), lmax = fmaxf(l0, l1);
    for (int r = (int)f0; r <= (int)f1; ++r)
        if (!(lmin >= __ldg(H.lo + H.off[k] + r) && lmax < __ldg(H.hi + H.off[k] + r))) return false;
    return true;
}
// The lane's photon: (L.x, L.y, L.z) = (u, v, w) and direction in the BEAM frame, dw > 0.  Returns true with the photon on the
// Phase Space 2 plane; false if it ended in the stage (energy booked).  dep sums what the stage absorbed.
template <bool COUNT>
__device__ __forceinline__ bool head_stage(Lane& L, const TransportParams& P, const Shared& sh, float& dep, uint32_t* cnt) {
    const Head& H = P.hd;
    int k = 0;
#pragma unroll 1
    for (;;) {
        if (L.E < P.ph.pcut) { dep += L.E; L.a_air += L.E; return false; }
        set_energy(L, P, sh);
        while (k < H.n_slabs && L.z >= H.w1[k]) ++k;
        const bool in_slab = k < H.n_slabs && L.z >= H.w0[k];
        const float w_end = in_slab ? H.w1[k] : (k < H.n_slabs ? H.w0[k] : H.w_ps2);
        if (!in_slab && k >= H.n_slabs && L.z >= H.w_ps2) return true;
        const float t_end = fmaxf((w_end - L.z) / L.dz, 0.0f);
        const uint4 rr = rng_block(L, P);
        const float nl = -__logf(u01(rr.x)), u2 = u01(rr.y);
        float pe, co, pp;
        mu3(P, sh, 0, L.ci, L.ct, L.E, pe, co, pp);
        const float mta = pe + co + pp, mua = kRhoAir * mta;
        float xsel;
        bool tungsten = false;
        if (!(in_slab && !head_clear(H, k, L.x, L.y, L.z, L.dx, L.dy, L.dz))) {
            // air gap, or a slab crossed inside its openings: one exponential flight in air up to the next plane
            if (!(nl < mua * t_end)) {
                L.x = fmaf(t_end, L.dx, L.x); L.y = fmaf(t_end, L.dy, L.y); L.z = w_end;
                if (!(fabsf(L.x) < kWorldHalf && fabsf(L.y) < kWorldHalf)) { L.a_esc += L.E; return false; }
                if (in_slab) ++k;
                continue;
            }
            const float s = __fdividef(nl, mua);
            L.x = fmaf(s, L.dx, L.x); L.y = fmaf(s, L.dy, L.y); L.z = fminf(fmaf(s, L.dz, L.z), w_end);
            xsel = u2 * mta;
        } else {
            // Woodcock flight inside slab k against the tungsten coefficient
            float pw, cw, ppw;
            mu3(P, sh, H.mat, L.ci, L.ct, L.E, pw, cw, ppw);
            const float mtw = pw + cw + ppw, muw = H.rho * mtw, mm = fmaxf(muw, mua) * 1.0001f;
            if (!(nl < mm * t_end)) {
                L.x = fmaf(t_end, L.dx, L.x); L.y = fmaf(t_end, L.dy, L.y); L.z = w_end; ++k;
                if (!(fabsf(L.x) < kWorldHalf && fabsf(L.y) < kWorldHalf)) { L.a_esc += L.E; return false; }
                continue;
            }
            const float s = __fdividef(nl, mm);
            L.x = fmaf(s, L.dx, L.x); L.y = fmaf(s, L.dy, L.y); L.z = fminf(fmaf(s, L.dz, L.z), w_end);
            tungsten = head_blocked(H, k, L.x, L.y);
            const float acc = u2 * mm;
            if (!(acc < (tungsten ? muw : mua))) continue;                 // virtual collision
            xsel = tungsten ? __fdividef(acc, H.rho) : __fdividef(acc, kRhoAir);   // reuse the accept draw for the channel (reading A8)
            if (tungsten) { pe = pw; co = cw; }
        }
        if (!(fabsf(L.x) < kWorldHalf && fabsf(L.y) < kWorldHalf)) { L.a_esc += L.E; return false; }
        if (COUNT) cnt[11]++;
        if (xsel < pe || !(xsel < pe + co)) { dep += L.E; L.a_air += L.E; return false; }   // photoelectric, or pair: all of E stays (A36)
        float eps, t, x4;
        sample_kn<COUNT>(L, P, eps, t, x4, cnt);
        const float ct = 1.0f - t, st = sqrtf(fmaxf(0.0f, t * (2.0f - t)));
        float sp, cp; __sincosf(2.0f * kPi * x4 - kPi, &sp, &cp);
        const float E1 = eps * L.E, T = L.E - E1;
        dep += T; L.a_air += T;
        L.E = E1;
        rotate(L.dx, L.dy, L.dz, ct, st, cp, sp);
        if (!(L.dz > 0.0f)) { L.a_esc += L.E; return false; }              // turned upstream: out of the stage
    }
}

// ---------------------------------------------------------------- K1 source
__device__ __forceinline__ uint32_t upper_bound_u32(const uint32_t* a, uint32_t n, uint32_t key) {   // #{k in [0,n): a[k] <= key}
    uint32_t lo = 0, hi = n;
    while (lo < hi) { const uint32_t mid = (lo + hi) >> 1; if (__ldg(a + mid) <= key) lo = mid + 1; else hi = mid; }
    return lo;
}
struct SourceSample { float E, dx, dy, dz, u, v; uint32_t pixel; };
__device__ __forceinline__ SourceSample sample_source(const TransportParams& P, uint32_t r0, uint32_t r1, uint32_t r2, uint32_t r3) {
    const Source& so = P.so; const Geom& g = P.g;
    SourceSample s;
    {   // energy: bin by the integer thresholds on r0, linear inside the bin
        uint32_t i = 0; float t;
        if (so.n_bins > 1) {
            i = upper_bound_u32(so.thrE + 1, so.n_bins - 1, r0);
            const uint32_t lo = __ldg(so.thrE + i), hi = __ldg(so.thrE + i + 1);
            const uint32_t wdt = hi - lo;                                  // thrE[n_bins] = 2^32 wraps to 0: the difference is still right
            t = wdt ? ((float)(r0 - lo) + 0.5f) / (float)wdt : 0.0f;
        } else t = ((float)r0 + 0.5f) * 2.3283064365386963e-10f;
        const float e0 = __ldg(so.edges + i), e1 = __ldg(so.edges + i + 1);
        s.E = fmaf(t, e1 - e0, e0);
    }
    uint32_t j;
    {   // fluence pixel: #{k : thrF[1 + k] <= r1}, searched inside the bracket the guide table gives for the top bits of r1
        uint32_t lo = __ldg(so.guideF + (r1 >> (32 - kGuideLog))), hi = __ldg(so.guideF + (r1 >> (32 - kGuideLog)) + 1);
        while (lo < hi) { const uint32_t mid = (lo + hi) >> 1; if (__ldg(so.thrF + 1 + mid) <= r1) lo = mid + 1; else hi = mid; }
        j = lo;
    }
    j = min(j, (uint32_t)so.j_last);
    s.pixel = j;
    const int ju = (int)(j % (uint32_t)so.fu), jv = (int)(j / (uint32_t)so.fu);
    s.u = ((float)ju - 0.5f * (float)so.fu + u01(r2)) * so.fpitch;
    s.v = ((float)jv - 0.5f * (float)so.fv + u01(r3)) * so.fpitch;
    const float inv = rsqrtf(s.u * s.u + s.v * s.v + so.fdist * so.fdist);
    dir_to_world(g, s.u * inv, s.v * inv, so.fdist * inv, s.dx, s.dy, s.dz);
    return s;
}

// ---------------------------------------------------------------- the kernel
// Add the warp's sum of v to *dst (lane 0); all lanes must call.
__device__ __noinline__ void ledger_add(float v, double* dst, bool atomic = false) {
    if (__ballot_sync(FULL_MASK, v != 0.0f) == 0u) return;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL_MASK, v, o);
    if ((threadIdx.x & 31u) == 0) { if (atomic) atomicAdd(dst, (double)v); else *dst += (double)v; }
}
__device__ __forceinline__ void ledger_flush(Lane& L, double* led) {
    ledger_add(L.a_emit, led + 0); ledger_add(L.a_ph, led + 1); ledger_add(L.a_eps, led + 2);
    ledger_add(L.a_epo, led + 3); ledger_add(L.a_air, led + 4); ledger_add(L.a_esc, led + 5);
    L.a_emit = L.a_ph = L.a_eps = L.a_epo = L.a_air = L.a_esc = 0.0f;
}

// Thread 0, between two barriers: publish what the last phase pushed (snapshot of every tail) and pick the next
// phase: new histories (class A) while there is head room for a full wave of them, else the class with the most
// waiting particles.  W and P need credits for their secondaries, so they wait while the head room is nearly used up
// and another class can run (particles that die in E and X give it back).
__device__ __noinline__ void choose_phase(const TransportParams& P, unsigned long long* phase_count) {
    int n[kRings];
#pragma unroll
    for (int r = 0; r < kRings; ++r) { s_snap[r] = s_tail[r]; n[r] = (int)(s_snap[r] - s_head[r]); }
#ifdef AEPID_CHECKED
    for (int r = 0; r < kRings; ++r) { s_head0[r] = s_head[r]; AEPID_CHECK(n[r] >= 0 && n[r] <= s_live_max); }
#endif
    int n_live = 0;
#pragma unroll
    for (int c = 0; c < kClasses; ++c) n_live += n[c];
    AEPID_CHECK(s_nphase == 0u || s_live == n_live);           // every credit was given back, every death was counted
    s_live = n_live;                                           // between phases every particle sits in a queue and no lane holds a credit
    // Progress check.  A phase in which every lane that could have run an event parked its particle for want of a head-room
    // credit is STUCK (possible with a small aepid_set_live_limit, or in physics modes 2 and 3 where every charged step needs a
    // credit, when pair / annihilation / bremsstrahlung photons multiply).  A stuck class is passed over until some phase makes
    // progress again (a particle that dies gives its count back); if every class that has particles is stuck, the limit set by
    // the caller, which is a soft one, is raised, up to the hard bound the queue protocol needs (half a class queue); beyond
    // that the run cannot go on and the error is flagged.
    if (s_did != 0) s_stuck = 0;
    else if (s_nphase > 0u && s_parked != 0 && s_phase >= 0) s_stuck |= 1 << s_phase;
    s_did = 0; s_parked = 0;
    if (s_stuck != 0) {
        bool any_free = false;
#pragma unroll
        for (int c = 0; c < kClasses; ++c) any_free |= n[c] > 0 && !((s_stuck >> c) & 1);
        if (!any_free) {
            const int hard = (1 << P.pool_log) / 2;
            if (s_live_max < hard) { s_live_max = min(2 * s_live_max, hard); s_stuck = 0; }
            else { raise_error(8); for (int r = 0; r < kRings; ++r) n[r] = 0; s_flag[0] = 1; }
        }
    }
    const int nf = s_live_max - n_live;
    bool more = s_flag[0] == 0;
    int budget = 0;
    if (more) {
        const uint32_t done = *((volatile unsigned int*)P.hist_counter);
        const uint32_t left = done < P.n ? P.n - done : 0u;
        if (left == 0u) { more = false; s_flag[0] = 1; }
        // take no more than this CTA's share of what is left, so that the CTAs finish together
        const uint32_t share = max((uint32_t)((unsigned long long)left * AEPID_SHARE_NUM / (AEPID_SHARE_DEN * gridDim.x)), (uint32_t)kThreads);
        budget = (int)min((uint32_t)max(nf - kReserve8ths * s_live_max / 8, 0), share);
    }
    int ph = -1;
    if (more && budget >= kThreads) ph = C_A;
    else {
        const bool starved = nf < kStarved && (n[C_E] + n[C_X] + n[C_A]) > 0;
        int nb = 0;
#pragma unroll
        for (int c = 0; c < kClasses; ++c) {
            if (starved && (c == C_W || c == C_P)) continue;
            if ((s_stuck >> c) & 1) continue;                  // its lanes could only park last time: let another class free head room first
            if (n[c] > nb) { nb = n[c]; ph = c; }
        }
        if (ph < 0 && n_live > 0) {                            // whatever waits must run: first a class that is not stuck, else any
#pragma unroll
            for (int c = 0; c < kClasses; ++c) if (!((s_stuck >> c) & 1) && n[c] > nb) { nb = n[c]; ph = c; }
#pragma unroll
            for (int c = 0; c < kClasses; ++c) if (ph < 0 && n[c] > nb) { nb = n[c]; ph = c; }
        }
        if (ph >= 0) budget = 0;
        else if (more && budget > 0) ph = C_A;                 // fewer histories left than lanes
        else if (more) raise_error(8);                         // cannot happen: nothing queued, yet no room for a history
    }
    if (ph >= 0 && ++s_nphase > kPhaseLimit) { raise_error(8); ph = -1; }
    s_phase = ph; s_left = 0; s_budget = ph == C_A ? budget : 0;
    const int n_start = ph < 0 ? 0 : n[ph] + (ph == C_A ? budget : 0);
    // soft end (header comment): at once for a long phase; for a short one not before kMinIter events per lane, so
    // that every phase makes progress (a short phase that restarts runs with its particles packed into fewer warps)
    s_keep = n_start >= kLongPhase ? 1 : 2;
    if (phase_count && ph >= 0) atomicAdd(phase_count, 1ull);
}

// One phase of class C for one warp (header comment).  On return every lane is empty and holds no credit.
template <bool COUNT, int C, int PH, bool HEAD>
__device__ __forceinline__ void run_phase(Lane& L, const TransportParams& P, const Shared& sh, double* led, uint32_t* cnt) {
    const unsigned lane = threadIdx.x & 31u;
    const unsigned lt_mask = (1u << lane) - 1u;
    constexpr bool C2 = PH == 2 || PH == 3;
    constexpr bool kSpawns = C == C_W || C == C_P || (C2 && (C == C_E || C == C_X));   // classes whose events create secondaries all the time
    const int keep = *((volatile int*)&s_keep);
    bool leaving = false, park = false, did = false, parked = false;
    float h_n = 0.0f, h_E = 0.0f, h_dep = 0.0f;                 // collimation stage (class A only): Phase Space 2 particles, their energy, absorbed
    // every lane enters a phase empty: saying so lets the compiler drop what this class never touches from the registers
    L.a_emit = L.a_ph = L.a_eps = L.a_epo = L.a_air = L.a_esc = 0.0f;
    L.alive = false; L.counted = kNone; L.spare = kNone; L.pval = 0.0f; L.pidx = kNone;
#pragma unroll 1
    for (uint32_t it = 1;; ++it) {
        // ---- A: particles that left the class (or all of them, when the warp leaves) go to the queue of their class;
        //         the count of a dead particle becomes the lane's credit or is given back
        if (!(L.alive && !leaving && !park && in_class<C>(L.flags))) {
            flush_pending(L, P);
            if (L.alive) {
                queue_particle(L.x, L.y, L.z, L.dx, L.dy, L.dz, L.E, L.vox, L.flags, L.h, L.pid, L.blk, PH == 4 ? L.R : 0.0f);
                if (COUNT && !kPhaseClock) cnt[27]++;
                L.alive = false; L.counted = kNone;
            } else if (L.counted != kNone) {
                if (kSpawns && !leaving && L.spare == kNone) L.spare = 1u; else atomicSub(&s_live, 1);
                L.counted = kNone;
            }
            park = false;
        }
        if (leaving) break;
        // ---- B: refill the empty lanes from the ring of the class; class A then starts new histories
        unsigned empty = __ballot_sync(FULL_MASK, !L.alive);
        if (__popc(empty) >= kRefillMin || it >= kIterLimit) {
            const unsigned long long cl = ring_claim(C, __popc(empty));
            const int got = (int)(uint32_t)cl;
            const int rk = __popc(empty & lt_mask);
            if (!L.alive && rk < got) {
                const uint32_t tk = (uint32_t)(cl >> 32) + (uint32_t)rk;
                AEPID_CHECK((int)(s_snap[C] - tk) > 0 && (int)(*((volatile unsigned int*)(s_tail + C)) - tk) <= (int)(s_pool_mask + 1u));   // published, not yet overwritten
                const uint4* rec = queue_rec(C, tk);
                const uint4 a = __ldcs(rec), b = __ldcs(rec + 1), c = __ldcs(rec + 2);
                if (PH == 4) L.R = __uint_as_float(__ldcs(rec + 3).x);
#if AEPID_PREFETCH > 0
                // the records a later refill will want (same queue, AEPID_PREFETCH tickets ahead, if published): into the L2
                if ((int)(s_snap[C] - (tk + AEPID_PREFETCH)) > 0) {
                    const uint4* nx = queue_rec(C, tk + AEPID_PREFETCH);
                    asm volatile("prefetch.global.L2 [%0];" :: "l"(nx));
                    asm volatile("prefetch.global.L2 [%0];" :: "l"(nx + 2));
                }
#endif
                L.x = __uint_as_float(a.x); L.y = __uint_as_float(a.y); L.z = __uint_as_float(a.z); L.dx = __uint_as_float(a.w);
                L.dy = __uint_as_float(b.x); L.dz = __uint_as_float(b.y); L.E = __uint_as_float(b.z); L.vox = b.w;
                L.flags = c.x; L.h = c.y; L.pid = c.z; L.blk = c.w;
                L.counted = 1u; L.alive = true;
                L.pval = 0.0f; L.pidx = kNone;
                if (COUNT && !kPhaseClock) cnt[28]++;
                if (C == C_A || C == C_W || C == C_P) set_energy(L, P, sh);
                if (C == C_E) { L.vlin = vox_linear(P.g, L.vox); AEPID_CHECK(L.vlin < P.nvox); L.cw = ld_vox(P.vox + L.vlin); L.pidx = L.vlin; }
            }
            if (C == C_A) {
                // K1: new histories in the lanes that are still empty (the budget of the phase is head room set aside for them)
                empty = __ballot_sync(FULL_MASK, !L.alive);
                const int nnew = budget_claim(__popc(empty));
                if (nnew > 0) {
                    const int rk2 = __popc(empty & lt_mask);
                    uint32_t h0 = 0;
                    if (lane == 0) { h0 = atomicAdd(P.hist_counter, (unsigned)nnew); atomicAdd(&s_live, nnew); }
                    h0 = __shfl_sync(FULL_MASK, h0, 0);
                    if (!L.alive && rk2 < nnew) {
                        const uint32_t h = h0 + (uint32_t)rk2;
                        if (h >= P.n) { atomicSub(&s_live, 1); atomicExch(s_flag, 1); }
                        else {
                            L.h = h; L.pid = 0; L.blk = 0;
                            const uint4 r = rng_block(L, P);               // block 0 of particle 0: E, pixel, u, v (reading A1)
                            L.vox = 0;
                            L.flags = T_PHOTON | (R_AIR << 2) | (min(h / P.hist_per_batch, (uint32_t)P.n_batches - 1u) << 16);
                            L.alive = true; L.counted = 1u;
                            L.pval = 0.0f; L.pidx = kNone; L.R = 0.0f;
                            if (!HEAD) {                                   // HEAD: the instantiation with the collimation stage (launch_transport)
                                const SourceSample s = sample_source(P, r.x, r.y, r.z, r.w);
                                L.x = P.g.src[0]; L.y = P.g.src[1]; L.z = P.g.src[2];
                                L.dx = s.dx; L.dy = s.dy; L.dz = s.dz; L.E = s.E;
                                L.a_emit += s.E;
                                set_energy(L, P, sh);
                            } else {
                                // Phase Space 1 source (reading A35): record floor(xi0 n), xi0 = (r + 0.5) 2^-32 = the first draw of block 0
                                const uint32_t j = (uint32_t)((((unsigned long long)r.x * 2ull + 1ull) * (unsigned long long)P.hd.n_ps1) >> 33);
                                const float4 qa = __ldg(P.hd.ps1 + 2 * (size_t)j), qb = __ldg(P.hd.ps1 + 2 * (size_t)j + 1);
                                const float inv = rsqrtf(qa.z * qa.z + qa.w * qa.w + qb.x * qb.x);
                                L.x = qa.x; L.y = qa.y; L.z = P.hd.w_ps1;
                                L.dx = qa.z * inv; L.dy = qa.w * inv; L.dz = qb.x * inv; L.E = qb.y;
                                L.a_emit += L.E;
                                const bool through = P.hd.n_slabs > 0 ? head_stage<COUNT>(L, P, sh, h_dep, cnt) : true;
                                if (through) {
                                    h_n += 1.0f; h_E += L.E;
                                    if (COUNT) cnt[10]++;
                                    float x, y, z;                         // beam frame -> world frame
                                    dir_to_world(P.g, L.x, L.y, L.z, x, y, z);
                                    L.x = x + P.g.src[0]; L.y = y + P.g.src[1]; L.z = z + P.g.src[2];
                                    dir_to_world(P.g, L.dx, L.dy, L.dz, x, y, z);
                                    L.dx = x; L.dy = y; L.dz = z;
                                    set_energy(L, P, sh);
                                } else L.alive = false;                    // ended in the head: the lane's count goes back in section A
                            }
                        }
                    }
                    if (COUNT && !kPhaseClock && lane == 0) cnt[30]++;
                }
            }
            // ---- C: leave the phase?
            const int n_live = __popc(__ballot_sync(FULL_MASK, L.alive));
            int go = 0;                                                        // 0 carry on, 1 nothing to do right now, 2 write back and leave, 3 leave
            {   // every lane reads the same shared words (one broadcast load each): the decision is uniform without a shuffle
                bool dry = (int)(s_snap[C] - *((volatile unsigned int*)(s_head + C))) <= 0;
                if (C == C_A && *((volatile int*)&s_budget) > 0 && *((volatile int*)s_flag) == 0) dry = false;
                if (n_live == 0) go = dry ? 3 : 1;
                else if (it >= kIterLimit) go = 2;
                else if (dry && 32 - n_live >= kRefillMin && (keep == 1 || (keep == 2 && it >= kMinIter))) go = 2;    // cannot keep its lanes full any more
            }
            if (go == 3) break;
            if (go == 2) { leaving = true; continue; }
            if (go == 1) continue;
        }
        // ---- D: one event per live lane
        #ifndef AEPID_PHASE_CLOCK
        if (COUNT) { if (lane == 0) cnt[16 + C]++; if (L.alive) cnt[21 + C]++; }
#endif
        bool on = L.alive;
        if (C == C_W || C == C_P) {
            if (on && !ensure_spare(L)) { park = true; on = false; if (COUNT && !kPhaseClock) cnt[29]++; }   // an interaction may create a secondary
        } else if (C2 && (C == C_E || C == C_X)) {
            if (on && !ensure_spare(L)) { park = true; on = false; if (COUNT && !kPhaseClock) cnt[29]++; }   // a step may end in a Moller event
        } else if (C == C_E || C == C_X) {
            if (on && F_TYPE(L.flags) == T_POSITRON && L.E <= P.ph.ecut && !ensure_spare(L)) { park = true; on = false; if (COUNT && !kPhaseClock) cnt[29]++; }   // annihilation needs a credit
        }
        did |= on; parked |= park;
        if (C == C_W) {
            // K3 + K4: flights against the majorant until at least kHitMin lanes have a collision to sample (or nobody flies
            // any more), then the interactions together: keeps both halves of the event well filled when few flights collide
            bool fly = on;
            if (on && L.E < P.ph.pcut) { if (COUNT) cnt[13]++; dep_here(L, P, L.E); L.alive = false; fly = false; }   // PAPER.md:104, 10 keV
            bool hit = false; float xsel = 0.0f, pe = 0.0f, co = 0.0f;
#pragma unroll 1
            for (int round = 0; round < kMaxRounds; ++round) {
                if (fly) { hit = woodcock_flight<COUNT>(L, P, sh, xsel, pe, co, cnt); fly = !hit && F_REGION(L.flags) == R_PHANTOM; }
                if (__popc(__ballot_sync(FULL_MASK, hit)) >= kHitMin || __ballot_sync(FULL_MASK, fly) == 0u) break;
            }
            if (hit) interact<COUNT>(L, P, sh, xsel, pe, co, cnt);
        } else if (on) {
            if (C == C_E) charged_event<COUNT, true, PH>(L, P, sh, cnt);
            else if (C == C_X) charged_event<COUNT, false, PH>(L, P, sh, cnt);
            else if (L.E < P.ph.pcut) { if (COUNT) cnt[13]++; dep_here(L, P, L.E); L.alive = false; }   // PAPER.md:104, 10 keV
            else {
                bool hit = false; float xsel = 0.0f, pe = 0.0f, co = 0.0f;
                if (C == C_A) {
                    if (air_transit<COUNT>(L, P, sh, xsel, pe, co, cnt)) L.flags |= F_HIT;   // collision in air or in a layer: class P
                } else {
                    if (L.flags & F_HIT) {                                 // collision found by the transit: channel from a fresh draw (reading A8)
                        L.flags &= ~F_HIT;
                        const bool in_air = F_REGION(L.flags) == R_AIR;
                        float pp;
                        mu3(P, sh, in_air ? 0 : P.g.lmat[F_LAYER(L.flags)], L.ci, L.ct, L.E, pe, co, pp);
                        xsel = u01(rng_block(L, P).x) * (pe + co + pp);
                        hit = true;
                    } else hit = epid_flight<COUNT>(L, P, sh, xsel, pe, co, cnt);
                }
                if (hit) interact<COUNT>(L, P, sh, xsel, pe, co, cnt);
            }
        }
        // ---- E: ledger of the last iterations: float per lane -> warp sum -> the warp's double accumulators
        if ((it & 63u) == 0u) ledger_flush(L, led);
    }
    if (L.spare != kNone) { atomicSub(&s_live, 1); L.spare = kNone; }
    if (L.counted != kNone) { atomicSub(&s_live, 1); L.counted = kNone; }   // a history that ended in the collimation stage right before the warp left
    ledger_flush(L, led);
    if (C == C_A && HEAD) {
        ledger_add(h_n, P.hd.stats + 0, true); ledger_add(h_E, P.hd.stats + 1, true); ledger_add(h_dep, P.hd.stats + 2, true);
    }
    if (__any_sync(FULL_MASK, did) && lane == 0) s_did = 1;
    if (__any_sync(FULL_MASK, parked) && lane == 0) s_parked = 1;
    if (lane == 0) atomicAdd(&s_left, 1);
}

template <bool COUNT, int PH, bool HEAD>
__global__ void __launch_bounds__(kThreads, 1) transport_kernel(const __grid_constant__ TransportParams P) {
    // dynamic shared memory: per-warp ledger | table blob
    double* const led_all = reinterpret_cast<double*>(smem_raw);
    uint32_t* const blob = reinterpret_cast<uint32_t*>(smem_raw + kWarps * 8 * sizeof(double));
    for (int i = threadIdx.x; i < P.tb.blob_words; i += kThreads) blob[i] = __ldg(P.tb.blob + i);
    Shared sh;
    sh.phot = reinterpret_cast<const float4*>(blob);
    sh.maj = reinterpret_cast<const float*>(sh.phot + P.tb.n_mat * P.tb.n_E);
    sh.lnS = sh.maj + P.tb.n_E;
    sh.invX0 = sh.lnS + P.tb.n_mat * P.tb.n_T;
    sh.sig = sh.invX0 + P.tb.n_mat + P.tb.n_mat * P.tb.n_T;
    sh.lnEg = reinterpret_cast<const float*>(blob) + P.tb.lnEg_off;
    sh.guide = reinterpret_cast<const uint32_t*>(sh.lnEg + P.tb.n_E);
    if (PH == 2 || PH == 3) sh.lnS = sh.invX0 + P.tb.n_mat;                    // the restricted stopping power takes the place of the total one
    for (int i = threadIdx.x; i < kWarps * 8; i += kThreads) led_all[i] = 0.0;
    if (threadIdx.x < kRings) { s_tail[threadIdx.x] = 0u; s_head[threadIdx.x] = 0u; s_snap[threadIdx.x] = 0u; }
    if (threadIdx.x < 2) s_flag[threadIdx.x] = 0;
    if (threadIdx.x == 0) {
        s_g = P.g; s_ep_batch = P.ep_batch; s_npix = P.npix; s_nphase = 0u;
        s_pool_log = P.pool_log; s_pool_mask = (1u << P.pool_log) - 1u; s_rec_vec = PH == 4 ? 4u : 3u;
        s_queue = P.queues + (((size_t)blockIdx.x * kClasses) << P.pool_log) * (PH == 4 ? 4 : 3);
        for (int r = 0; r < kRings; ++r) s_ring_base[r] = s_queue + (((size_t)r) << P.pool_log) * (PH == 4 ? 4 : 3);
        s_live = 0; s_live_max = min(max(P.live_max, 64), (1 << P.pool_log) / 2); s_did = 0; s_parked = 0; s_stuck = 0; s_phase = -1;
    }
    __syncthreads();

    uint32_t cnt[COUNT ? 32 : 1];
    if (COUNT) {
#pragma unroll
        for (int i = 0; i < 32; ++i) cnt[i] = 0;
    }
    const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    double* const led = led_all + warp * 8;
    Lane L;
    L.x = L.y = L.z = 0.0f; L.dx = L.dy = 0.0f; L.dz = 1.0f; L.E = 0.0f; L.vox = 0; L.flags = 0; L.h = L.pid = L.blk = 0;
    L.cw = 0; L.vlin = 0; L.ci = 0; L.ct = 0.0f; L.mumaj = 1.0f;
    L.pval = 0.0f; L.pidx = kNone; L.counted = kNone; L.spare = kNone; L.alive = false; L.R = 0.0f;
    L.a_emit = L.a_ph = L.a_eps = L.a_epo = L.a_air = L.a_esc = 0.0f;

#pragma unroll 1
    for (;;) {
        if (threadIdx.x == 0) choose_phase(P, COUNT ? P.counters + 26 : nullptr);
        __syncthreads();
        const int ph = s_phase;
        if (ph < 0) break;
#ifdef AEPID_PHASE_CLOCK
        const long long t0 = clock64();
#endif
        switch (ph) {
            case C_A: run_phase<COUNT, C_A, PH, HEAD>(L, P, sh, led, cnt); break;
            case C_W: run_phase<COUNT, C_W, PH, HEAD>(L, P, sh, led, cnt); break;
            case C_E: run_phase<COUNT, C_E, PH, HEAD>(L, P, sh, led, cnt); break;
            case C_P: run_phase<COUNT, C_P, PH, HEAD>(L, P, sh, led, cnt); break;
            default:  run_phase<COUNT, C_X, PH, HEAD>(L, P, sh, led, cnt); break;
        }
#ifdef AEPID_PHASE_CLOCK
        if (COUNT && lane == 0) { atomicAdd(P.counters + 10, (unsigned long long)(clock64() - t0)); atomicAdd(P.counters + 27 + ph, (unsigned long long)(clock64() - t0)); }   // busy warp-cycles
#endif
        __syncthreads();
#ifdef AEPID_PHASE_CLOCK
        if (COUNT && threadIdx.x == 0) {
            atomicAdd(P.counters + 16 + ph, (unsigned long long)(clock64() - t0));                  // cycles per class
            atomicAdd(P.counters + 21 + ph, 1ull);                                                    // phases per class
            atomicAdd(P.counters + 11, (unsigned long long)(clock64() - t0) * kWarps);
        }
#endif
    }

    if (threadIdx.x < 6) {
        double v = 0.0;
        for (int w = 0; w < kWarps; ++w) v += led_all[w * 8 + threadIdx.x];
        if (v != 0.0) atomicAdd(P.ledger + threadIdx.x, v);
    }
    if (threadIdx.x == 0 && s_flag[1]) atomicAdd(P.ledger + 7, (double)s_flag[1]);
    if (COUNT) {
#pragma unroll
        for (int i = 0; i < 32; ++i) {
            uint32_t v = cnt[i];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL_MASK, v, o);
            if (lane == 0 && v) atomicAdd(P.counters + i, (unsigned long long)v);
        }
    }
}

constexpr size_t kDynSmemFixed = kWarps * 8 * sizeof(double);

size_t transport_smem_bytes(const Tables& t) {      // dynamic + static shared memory of the kernel
    return kDynSmemFixed + (size_t)t.blob_words * 4 + sizeof(Geom) + 512;
}

template <bool COUNT, int PH, bool HEAD>
static int launch_inst(const TransportParams& p, unsigned blocks, size_t smem, cudaStream_t stream) {
    const cudaError_t e = cudaFuncSetAttribute(transport_kernel<COUNT, PH, HEAD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return (int)e;
    transport_kernel<COUNT, PH, HEAD><<<blocks, kThreads, smem, stream>>>(p);
    return (int)cudaGetLastError();
}
// The collimation stage (Phase Space 1 source + jaws / MLC) has its own instantiations: the fluence-map source pays nothing for it
template <bool COUNT, int PH>
static int launch_one(const TransportParams& p, unsigned blocks, size_t smem, cudaStream_t stream) {
    return p.hd.n_ps1 != 0u ? launch_inst<COUNT, PH, true>(p, blocks, smem, stream) : launch_inst<COUNT, PH, false>(p, blocks, smem, stream);
}
int launch_transport(const TransportParams& p, bool counting, int sm_count, void* stream) {
    const size_t smem = kDynSmemFixed + (size_t)p.tb.blob_words * 4;
    // persistent grid: one CTA per SM (each with its own class queues), but no more CTAs than there is work for
    long long blocks = sm_count < kMaxCtas ? sm_count : kMaxCtas;
    const long long need = ((long long)p.n + 255) / 256;
    if (blocks > need) blocks = need;
    if (blocks < 1) blocks = 1;
    // Class II physics (mode 2: Moller delta rays, mode 3: + bremsstrahlung) has its own instantiations: modes 0 and 1 pay nothing
    const cudaStream_t st = (cudaStream_t)stream; const unsigned nb = (unsigned)blocks;
    if (p.ph.mode == 4) return counting ? launch_one<true, 4>(p, nb, smem, st) : launch_one<false, 4>(p, nb, smem, st);
    if (p.ph.mode == 3) return counting ? launch_one<true, 3>(p, nb, smem, st) : launch_one<false, 3>(p, nb, smem, st);
    if (p.ph.mode == 2) return counting ? launch_one<true, 2>(p, nb, smem, st) : launch_one<false, 2>(p, nb, smem, st);
    return counting ? launch_one<true, 1>(p, nb, smem, st) : launch_one<false, 1>(p, nb, smem, st);
}
// K1 alone (aepid_sample_source): out[k] = {E, dx, dy, dz, pixel, u, v, 0} for history first + k
__global__ void sample_source_kernel(const __grid_constant__ TransportParams P, uint64_t first, uint64_t n, float* __restrict__ out) {
    const uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const uint64_t h = first + k;
    const uint4 r = philox4x32_10((uint32_t)h, (uint32_t)(h >> 32), 0u, 0u, (uint32_t)P.seed, (uint32_t)(P.seed >> 32));
    const SourceSample s = sample_source(P, r.x, r.y, r.z, r.w);
    float4* o = reinterpret_cast<float4*>(out + 8 * k);
    o[0] = make_float4(s.E, s.dx, s.dy, s.dz);
    o[1] = make_float4((float)s.pixel, s.u, s.v, 0.0f);
}
void launch_sample_source(const TransportParams& p, uint64_t first, uint64_t n, float* out, void* stream) {
    if (n == 0) return;
    sample_source_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(p, first, n, out);
}

}  // namespace aepid
