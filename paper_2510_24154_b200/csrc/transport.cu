// Transport kernel: K1 source sampling, K2 air navigation, K3 Woodcock tracking, K4 interaction
// sampling, K5 CSDA electron steps with Highland deflection, K6 EPID slab transport and K7 tally
// scoring (physics of SURVEY.md 8(c)).
//
// Design (sm_100a): one persistent grid, one particle per lane.  Every loop iteration a lane executes ONE
// event of its particle (one photon flight or one electron step) so that lanes holding different particle
// kinds share as much of the instruction stream as possible; a lane whose particle ends pops its private
// secondary stack or takes the next history of the warp's chunk (chunks of 64 histories are handed out by
// one global atomic, so the tail is balanced over the whole GPU).  Material tables live in shared memory in
// the ln domain (one LDS.128 per node), the phantom is one packed 32-bit word per voxel gathered through
// the read-only path (L2-resident up to ~30 M voxels), phantom deposits of consecutive steps in one voxel are
// merged in registers and flushed with one RED, the energy ledger is kept in double.
// No tensor cores / TMA: random gathers and scalar arithmetic, nothing here is a dense contraction.
#include <cuda_runtime.h>
#include <cstdint>
#include "params.h"

namespace aepid {

constexpr int kBlock = 256;
constexpr int kMinBlocks = 3;
constexpr int kStackDepth = 4;
constexpr float kPi = 3.14159265358979f;
constexpr float kInf = 3.0e38f;

#define FULL_MASK 0xffffffffu
// flags: bits 0-1 type, 2-3 region, 4-6 layer, 8 two spare randoms buffered, 16-23 batch
#define F_TYPE(f) ((f) & 3u)
#define F_REGION(f) (((f) >> 2) & 3u)
#define F_LAYER(f) (((f) >> 4) & 7u)
#define F_BATCH(f) (((f) >> 16) & 255u)
#define F_HAS2 (1u << 8)
#define SET_TYPE(f, t) ((f) = ((f) & ~3u) | (t))
#define SET_REGION(f, r) ((f) = ((f) & ~(3u << 2)) | ((r) << 2))
#define SET_LAYER(f, l) ((f) = ((f) & ~(7u << 4)) | ((uint32_t)(l) << 4))

struct Shared {
    const float4* phot;
    const float* maj;
    const float* lnS;
    const float* invX0;
    double* led;        // [8] block-level ledger
};

struct StackEntry { float x, y, z, dx, dy, dz, E; uint32_t flags, vox, pid, blk; };

struct Lane {
    float x, y, z, dx, dy, dz, E;   // position: world (AIR, photon in PHANTOM), voxel fraction (charged in PHANTOM), beam (u, v, depth) in EPID
    uint32_t vox;                   // packed voxel index ix | iy << 10 | iz << 20
    uint32_t flags;
    uint32_t h, pid, blk;           // history (relative to the launch base), particle id, Philox block counter
    uint32_t r2, r3;                // buffered raw draws
    uint32_t cw;                    // packed word of the current voxel (charged particle in PHANTOM)
    int ci; float ct, mumaj;        // photon: table cell, fraction, majorant at E
    uint32_t pidx; float pval;      // pending phantom deposit (merged while the voxel does not change)
    double lph;                     // thread-local ledger: energy deposited in the phantom
    int sp;
    bool alive;
};

// ---------------------------------------------------------------- Philox4x32-10 (own implementation; pinned on the GPU by tests)
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1,
                                              uint32_t& o0, uint32_t& o1, uint32_t& o2, uint32_t& o3) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    o0 = c0; o1 = c1; o2 = c2; o3 = c3;
}
// uniform in (0,1) from the top 23 bits: ((r >> 9) + 0.5) 2^-23 is exact in float32 and never 0 or 1
__device__ __forceinline__ float u01(uint32_t r) { return ((float)(r >> 9) + 0.5f) * 1.1920928955078125e-7f; }

__device__ __forceinline__ void rng_block(Lane& L, const TransportParams& P, uint32_t& o0, uint32_t& o1, uint32_t& o2, uint32_t& o3) {
    const uint64_t h = P.base + L.h;
    philox4x32_10((uint32_t)h, (uint32_t)(h >> 32), L.pid, L.blk, (uint32_t)P.seed, (uint32_t)(P.seed >> 32), o0, o1, o2, o3);
    L.blk++;
}
__device__ __forceinline__ void rng_pair(Lane& L, const TransportParams& P, float& a, float& b) {
    if (L.flags & F_HAS2) { a = u01(L.r2); b = u01(L.r3); L.flags &= ~F_HAS2; }
    else {
        uint32_t o0, o1;
        rng_block(L, P, o0, o1, L.r2, L.r3);
        a = u01(o0); b = u01(o1); L.flags |= F_HAS2;
    }
}
__device__ __forceinline__ uint32_t child_id(const Lane& L, uint32_t sibling) {    // reading A1
    return L.pid * 0x9E3779B1u + L.blk * 2u + sibling + 1u;
}

// ---------------------------------------------------------------- tables
__device__ __forceinline__ void mu3(const TransportParams& P, const Shared& sh, int m, int ci, float ct, float& pe, float& co, float& pp) {
    const float4 a = sh.phot[m * P.tb.n_E + ci], b = sh.phot[m * P.tb.n_E + ci + 1];
    pe = __expf(fmaf(ct, b.x - a.x, a.x));
    co = __expf(fmaf(ct, b.y - a.y, a.y));
    pp = fmaf(ct, b.z - a.z, a.z);
}
__device__ __forceinline__ void set_energy(Lane& L, const TransportParams& P, const Shared& sh) {
    float f = (__logf(L.E) - P.tb.lnE0) * P.tb.inv_dlnE;
    f = fminf(fmaxf(f, 0.0f), (float)(P.tb.n_E - 1));
    const int i = min((int)f, P.tb.n_E - 2);
    L.ci = i; L.ct = f - (float)i;
    L.mumaj = fmaf(L.ct, sh.maj[i + 1] - sh.maj[i], sh.maj[i]);
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
    const float a = -1.0f / (sg + dz), b = dx * dy * a;
    const float b1x = 1.0f + sg * dx * dx * a, b1y = sg * b, b1z = -sg * dx;
    const float b2x = b, b2y = sg + dy * dy * a, b2z = -dy;
    const float sc = st * cp, ss = st * sp;
    float nx = ct * dx + sc * b1x + ss * b2x;
    float ny = ct * dy + sc * b1y + ss * b2y;
    float nz = ct * dz + sc * b1z + ss * b2z;
    const float inv = rsqrtf(nx * nx + ny * ny + nz * nz);
    dx = nx * inv; dy = ny * inv; dz = nz * inv;
}

// ---------------------------------------------------------------- tallies
__device__ __forceinline__ void flush_pending(Lane& L, const TransportParams& P) {
    if (L.pval != 0.0f) {
        atomicAdd(P.ph_batch + (size_t)F_BATCH(L.flags) * P.nvox + L.pidx, L.pval);
        L.pval = 0.0f;
    }
}
__device__ __forceinline__ uint32_t vox_linear(const Geom& g, uint32_t v) {
    return (((v >> 20) & 1023u) * (uint32_t)g.ny + ((v >> 10) & 1023u)) * (uint32_t)g.nx + (v & 1023u);
}
__device__ __forceinline__ void dep_vox(Lane& L, const TransportParams& P, uint32_t idx, float e) {
    if (idx != L.pidx) { flush_pending(L, P); L.pidx = idx; }
    L.pval += e;
    L.lph += (double)e;
}
__device__ __forceinline__ void dep_epid(Lane& L, const TransportParams& P, const Shared& sh, int layer, float u, float v, float e) {
    if (P.g.lscored[layer]) {
        const float fu = floorf((u + P.g.half_u) * P.g.inv_pitch), fv = floorf((v + P.g.half_v) * P.g.inv_pitch);
        if (fu >= 0.0f && fu < (float)P.g.nu && fv >= 0.0f && fv < (float)P.g.nv) {
            atomicAdd(P.ep_batch + (size_t)F_BATCH(L.flags) * P.npix + (size_t)fv * P.g.nu + (size_t)fu, e);
            atomicAdd(&sh.led[2], (double)e);
            return;
        }
    }
    atomicAdd(&sh.led[3], (double)e);
}
// deposit at the particle's position
__device__ __forceinline__ void dep_here(Lane& L, const TransportParams& P, const Shared& sh, float e) {
    const uint32_t reg = F_REGION(L.flags);
    if (reg == R_PHANTOM) dep_vox(L, P, vox_linear(P.g, L.vox), e);
    else if (reg == R_AIR) atomicAdd(&sh.led[4], (double)e);
    else dep_epid(L, P, sh, F_LAYER(L.flags), L.x, L.y, e);
}

// ---------------------------------------------------------------- geometry
// Nearest boundary seen from AIR: kind 0 phantom AABB entry, 1 EPID top plane, 2 world exit.
__device__ __forceinline__ float air_boundary(const Geom& g, const Lane& L, int& kind, int& axis) {
    float tn = -kInf, tf = kInf; int ax = 0; bool miss = false;
#define SLAB(P_, D_, LO_, HI_, A_)                                            \
    if (fabsf(D_) > 1e-20f) {                                                  \
        const float inv = 1.0f / (D_);                                         \
        float t1 = ((LO_) - (P_)) * inv, t2 = ((HI_) - (P_)) * inv;           \
        if (t1 > t2) { const float t = t1; t1 = t2; t2 = t; }                  \
        if (t1 > tn) { tn = t1; ax = A_; }                                     \
        tf = fminf(tf, t2);                                                    \
    } else if ((P_) < (LO_) || (P_) >= (HI_)) miss = true;
    SLAB(L.x, L.dx, g.lox, g.hix, 0)
    SLAB(L.y, L.dy, g.loy, g.hiy, 1)
    SLAB(L.z, L.dz, g.loz, g.hiz, 2)
#undef SLAB
    float tb = (miss || !(tf > 0.0f) || tn >= tf) ? kInf : fmaxf(tn, 0.0f);
    kind = 0; axis = ax;
    float pu, pv, pw, du, dv, dw;
    to_beam(g, L.x, L.y, L.z, pu, pv, pw);
    dir_to_beam(g, L.dx, L.dy, L.dz, du, dv, dw);
    if (dw > 0.0f) { const float te = fmaxf((g.sid - pw) / dw, 0.0f); if (te < tb) { tb = te; kind = 1; } }
    float tw = kInf;
    if (du > 0.0f) tw = fminf(tw, (kWorldHalf - pu) / du); else if (du < 0.0f) tw = fminf(tw, (-kWorldHalf - pu) / du);
    if (dv > 0.0f) tw = fminf(tw, (kWorldHalf - pv) / dv); else if (dv < 0.0f) tw = fminf(tw, (-kWorldHalf - pv) / dv);
    if (dw < 0.0f) tw = fminf(tw, (kWorldWMin - pw) / dw);
    tw = fmaxf(tw, 0.0f);
    if (tw < tb) { tb = tw; kind = 2; }
    return tb;
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
        L.cw = __ldg(P.vox + vox_linear(g, L.vox));
    }
}
__device__ __forceinline__ void enter_epid(Lane& L, const Geom& g) {       // position already on the top plane
    float pu, pv, pw, du, dv, dw;
    to_beam(g, L.x, L.y, L.z, pu, pv, pw);
    dir_to_beam(g, L.dx, L.dy, L.dz, du, dv, dw);
    L.x = pu; L.y = pv; L.z = 0.0f; L.dx = du; L.dy = dv; L.dz = dw;
    SET_REGION(L.flags, R_EPID); SET_LAYER(L.flags, 0);
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

// ---------------------------------------------------------------- stack
__device__ __forceinline__ void push(Lane& L, StackEntry* stk, float x, float y, float z, float dx, float dy, float dz, float E,
                                     uint32_t flags, uint32_t vox, uint32_t pid, uint32_t blk, const Shared& sh) {
    if (L.sp >= kStackDepth) { atomicAdd(&sh.led[7], 1.0); atomicAdd(&sh.led[5], (double)E); return; }   // cannot happen (depth <= 2); flagged
    StackEntry& s = stk[L.sp++];
    s.x = x; s.y = y; s.z = z; s.dx = dx; s.dy = dy; s.dz = dz; s.E = E; s.flags = flags & ~F_HAS2; s.vox = vox; s.pid = pid; s.blk = blk;
}

// Two 0.511 MeV photons, isotropic and back to back (reading A11): the lane becomes the first, the second is pushed.
// Position must already be in the frame photons use in this region.
__device__ __forceinline__ void annihilate(Lane& L, const TransportParams& P, const Shared& sh, StackEntry* stk) {
    float a, b; rng_pair(L, P, a, b);
    const float ct = 2.0f * a - 1.0f, st = sqrtf(fmaxf(0.0f, 1.0f - ct * ct));
    float sp, cp; __sincosf(2.0f * kPi * b - kPi, &sp, &cp);
    const float dx = st * cp, dy = st * sp, dz = ct;
    uint32_t f = L.flags; SET_TYPE(f, T_PHOTON);
    push(L, stk, L.x, L.y, L.z, -dx, -dy, -dz, kMec2, f, L.vox, child_id(L, 1), 0u, sh);
    L.pid = child_id(L, 0); L.blk = 0;
    L.flags = f & ~F_HAS2;
    L.dx = dx; L.dy = dy; L.dz = dz; L.E = kMec2;
    set_energy(L, P, sh);
}

// photon (world position in PHANTOM) -> charged particle representation
__device__ __forceinline__ void world_to_frac(Lane& L, const Geom& g) {
    const float gx = (L.x - g.lox) * g.ihx - (float)(L.vox & 1023u);
    const float gy = (L.y - g.loy) * g.ihy - (float)((L.vox >> 10) & 1023u);
    const float gz = (L.z - g.loz) * g.ihz - (float)((L.vox >> 20) & 1023u);
    L.x = fminf(fmaxf(gx, 0.0f), 1.0f); L.y = fminf(fmaxf(gy, 0.0f), 1.0f); L.z = fminf(fmaxf(gz, 0.0f), 1.0f);
}

// ---------------------------------------------------------------- K4 interaction
template <bool COUNT>
__device__ __forceinline__ void interact(Lane& L, const TransportParams& P, const Shared& sh, StackEntry* stk,
                                         float xsel, float pe, float co, uint32_t* cnt) {
    const bool coupled = P.ph.mode != 0;
    const uint32_t reg = F_REGION(L.flags);
    if (xsel < pe) {                                                       // photoelectric: electron T = E along d
        if (COUNT) cnt[3]++;
        if (!coupled || L.E <= P.ph.ecut) { dep_here(L, P, sh, L.E); L.alive = false; return; }
        SET_TYPE(L.flags, T_ELECTRON);
        L.pid = child_id(L, 0); L.blk = 0; L.flags &= ~F_HAS2;
        if (COUNT) { cnt[9]++; cnt[14]++; }
        if (reg == R_PHANTOM) world_to_frac(L, P.g);
        return;
    }
    if (xsel < pe + co) {                                                  // Compton: Klein-Nishina by epsilon-mixture rejection
        if (COUNT) cnt[4]++;
        const float k = L.E * (1.0f / kMec2), e0 = 1.0f / (1.0f + 2.0f * k), e02 = e0 * e0;
        const float a1 = -__logf(e0), a2 = 0.5f * (1.0f - e02);
        float eps, t, x4;
        for (;;) {
            float x1, x2, x3;
            rng_pair(L, P, x1, x2); rng_pair(L, P, x3, x4);
            if (COUNT) cnt[12]++;
            eps = (x1 * (a1 + a2) < a1) ? __expf(-x2 * a1) : sqrtf(fmaf(1.0f - e02, x2, e02));
            t = (1.0f - eps) / (k * eps);
            const float g = 1.0f - eps * t * (2.0f - t) / (1.0f + eps * eps);
            if (g >= x3) break;
        }
        const float ct = 1.0f - t, st = sqrtf(fmaxf(0.0f, t * (2.0f - t)));
        float sp, cp; __sincosf(2.0f * kPi * x4 - kPi, &sp, &cp);
        const float E1 = eps * L.E, T = L.E - E1;
        float d1x = L.dx, d1y = L.dy, d1z = L.dz;
        rotate(d1x, d1y, d1z, ct, st, cp, sp);
        if (!coupled || T <= P.ph.ecut) {                                  // kerma, or electron born below its cutoff: local deposit
            dep_here(L, P, sh, T);
            if (COUNT && coupled) { cnt[9]++; cnt[14]++; }
            L.E = E1; L.dx = d1x; L.dy = d1y; L.dz = d1z;
            set_energy(L, P, sh);
            return;
        }
        // electron from momentum conservation; the scattered photon waits on the stack
        float ex = L.E * L.dx - E1 * d1x, ey = L.E * L.dy - E1 * d1y, ez = L.E * L.dz - E1 * d1z;
        const float inv = rsqrtf(ex * ex + ey * ey + ez * ez);
        const uint32_t epid = child_id(L, 0);
        if (E1 < P.ph.pcut) dep_here(L, P, sh, E1);
        else {
            // the scattered photon keeps its own stream (same particle id, block counter carried on the stack)
            push(L, stk, L.x, L.y, L.z, d1x, d1y, d1z, E1, L.flags, L.vox, L.pid, L.blk, sh);
        }
        SET_TYPE(L.flags, T_ELECTRON);
        L.pid = epid; L.blk = 0; L.flags &= ~F_HAS2;
        L.E = T; L.dx = ex * inv; L.dy = ey * inv; L.dz = ez * inv;
        if (COUNT) { cnt[9]++; cnt[14]++; }
        if (reg == R_PHANTOM) world_to_frac(L, P.g);
        return;
    }
    // pair production: uniform kinetic split, both along d (reading A10)
    if (COUNT) cnt[5]++;
    float a, b; rng_pair(L, P, a, b);
    const float Ttot = L.E - 2.0f * kMec2;
    const float Tm = a * Ttot, Tp = Ttot - Tm;
    if (!coupled) {
        dep_here(L, P, sh, Ttot);
        if (COUNT) cnt[9] += 2;
        annihilate(L, P, sh, stk);                                         // 2 m_e c^2 re-emitted at the interaction point (A11)
        return;
    }
    if (COUNT) { cnt[9] += 2; cnt[14] += 2; }
    uint32_t fpos = L.flags; SET_TYPE(fpos, T_POSITRON);
    const uint32_t id0 = child_id(L, 0), id1 = child_id(L, 1);
    if (reg == R_PHANTOM) world_to_frac(L, P.g);
    push(L, stk, L.x, L.y, L.z, L.dx, L.dy, L.dz, Tp, fpos, L.vox, id1, 0u, sh);
    SET_TYPE(L.flags, T_ELECTRON);
    L.pid = id0; L.blk = 0; L.flags &= ~F_HAS2;
    L.E = Tm;
}

// ---------------------------------------------------------------- photon event: one flight (K2, K3, K6) + interaction (K4)
template <bool COUNT>
__device__ __forceinline__ void photon_event(Lane& L, const TransportParams& P, const Shared& sh, StackEntry* stk, uint32_t* cnt) {
    const Geom& g = P.g;
    if (L.E < P.ph.pcut) { if (COUNT) cnt[13]++; dep_here(L, P, sh, L.E); L.alive = false; return; }   // PAPER.md:104, 10 keV
    float u1, u2; rng_pair(L, P, u1, u2);
    const float nl = -__logf(u1);
    const uint32_t reg = F_REGION(L.flags);
    float pe, co, pp, xsel = 0.0f; bool hit = false;
    if (reg == R_PHANTOM) {                                                // Woodcock flight against the majorant
        if (COUNT) cnt[0]++;
        const float s = __fdividef(nl, L.mumaj);
        const float nx = fmaf(s, L.dx, L.x), ny = fmaf(s, L.dy, L.y), nz = fmaf(s, L.dz, L.z);
        if (!(nx >= g.lox && nx < g.hix && ny >= g.loy && ny < g.hiy && nz >= g.loz && nz < g.hiz)) {
            // left the grid: place on the AABB exit point, snapped onto the crossed face
            float tx = kInf, ty = kInf, tz = kInf;
            if (L.dx > 0.0f) tx = (g.hix - L.x) / L.dx; else if (L.dx < 0.0f) tx = (g.lox - L.x) / L.dx;
            if (L.dy > 0.0f) ty = (g.hiy - L.y) / L.dy; else if (L.dy < 0.0f) ty = (g.loy - L.y) / L.dy;
            if (L.dz > 0.0f) tz = (g.hiz - L.z) / L.dz; else if (L.dz < 0.0f) tz = (g.loz - L.z) / L.dz;
            const float t = fmaxf(fminf(tx, fminf(ty, tz)), 0.0f);
            L.x = fmaf(t, L.dx, L.x); L.y = fmaf(t, L.dy, L.y); L.z = fmaf(t, L.dz, L.z);
            if (tx <= ty && tx <= tz) L.x = L.dx > 0.0f ? g.hix : g.lox;
            else if (ty <= tz) L.y = L.dy > 0.0f ? g.hiy : g.loy;
            else L.z = L.dz > 0.0f ? g.hiz : g.loz;
            SET_REGION(L.flags, R_AIR);
            return;
        }
        L.x = nx; L.y = ny; L.z = nz;
        const int ix = min((int)((nx - g.lox) * g.ihx), g.nx - 1), iy = min((int)((ny - g.loy) * g.ihy), g.ny - 1), iz = min((int)((nz - g.loz) * g.ihz), g.nz - 1);
        const uint32_t w = __ldg(P.vox + ((size_t)iz * g.ny + iy) * g.nx + ix);
        const float rho = __uint_as_float(w & ~31u);
        mu3(P, sh, (int)(w & 31u), L.ci, L.ct, pe, co, pp);
        xsel = u2 * L.mumaj;
        if (xsel < rho * (pe + co + pp)) {
            hit = true; xsel = __fdividef(xsel, rho);                      // reuse the accept draw for the channel (reading A8)
            L.cw = w; L.vox = (uint32_t)ix | ((uint32_t)iy << 10) | ((uint32_t)iz << 20);
        }
    } else if (reg == R_AIR) {
        if (COUNT) cnt[1]++;
        int kind, axis;
        const float tb = air_boundary(g, L, kind, axis);
        mu3(P, sh, 0, L.ci, L.ct, pe, co, pp);
        const float mt = pe + co + pp;
        const float s = nl / (kRhoAir * mt);
        if (s < tb) { L.x = fmaf(s, L.dx, L.x); L.y = fmaf(s, L.dy, L.y); L.z = fmaf(s, L.dz, L.z); hit = true; xsel = u2 * mt; }
        else {
            L.x = fmaf(tb, L.dx, L.x); L.y = fmaf(tb, L.dy, L.y); L.z = fmaf(tb, L.dz, L.z);
            if (kind == 0) enter_phantom(L, P, axis);
            else if (kind == 1) enter_epid(L, g);
            else { atomicAdd(&sh.led[5], (double)L.E); L.alive = false; }
            return;
        }
    } else {                                                               // EPID: surface tracking layer by layer
        if (COUNT) cnt[2]++;
        const int l = F_LAYER(L.flags);
        mu3(P, sh, g.lmat[l], L.ci, L.ct, pe, co, pp);
        const float mt = pe + co + pp;
        const float s = nl / (g.lrho[l] * mt);
        float tf = kInf;
        if (L.dz > 0.0f) tf = (g.zt[l + 1] - L.z) / L.dz; else if (L.dz < 0.0f) tf = (g.zt[l] - L.z) / L.dz;
        tf = fmaxf(tf, 0.0f);
        const float tl = lateral_exit(L.x, L.y, L.dx, L.dy);
        if (s < tf && s < tl) { L.x = fmaf(s, L.dx, L.x); L.y = fmaf(s, L.dy, L.y); L.z = fmaf(s, L.dz, L.z); hit = true; xsel = u2 * mt; }
        else if (tl < tf) { atomicAdd(&sh.led[5], (double)L.E); L.alive = false; return; }
        else {
            L.x = fmaf(tf, L.dx, L.x); L.y = fmaf(tf, L.dy, L.y);
            if (L.dz > 0.0f) {
                L.z = g.zt[l + 1];
                if (l + 1 >= g.n_layers) { atomicAdd(&sh.led[5], (double)L.E); L.alive = false; }
                else SET_LAYER(L.flags, l + 1);
            } else {
                L.z = g.zt[l];
                if (l == 0) epid_to_air(L, g); else SET_LAYER(L.flags, l - 1);
            }
            return;
        }
    }
    if (hit) interact<COUNT>(L, P, sh, stk, xsel, pe, co, cnt);
}

// ---------------------------------------------------------------- K5 electron / positron step
template <bool COUNT>
__device__ __forceinline__ void electron_event(Lane& L, const TransportParams& P, const Shared& sh, StackEntry* stk, uint32_t* cnt) {
    const Geom& g = P.g;
    const uint32_t reg = F_REGION(L.flags);
    if (L.E <= P.ph.ecut) {                                                // PAPER.md:104, 200 keV: local deposit
        dep_here(L, P, sh, L.E);
        if (F_TYPE(L.flags) == T_POSITRON) {
            if (reg == R_PHANTOM) frac_to_world(L, g);
            if (COUNT) cnt[9] += 2;
            annihilate(L, P, sh, stk);
        } else L.alive = false;
        return;
    }
    float rho, tb; int m, axis = 0, kind = 0;
    if (reg == R_PHANTOM) {
        rho = __uint_as_float(L.cw & ~31u); m = (int)(L.cw & 31u);
        float tx = kInf, ty = kInf, tz = kInf;
        if (L.dx > 0.0f) tx = (1.0f - L.x) * g.hx / L.dx; else if (L.dx < 0.0f) tx = -L.x * g.hx / L.dx;
        if (L.dy > 0.0f) ty = (1.0f - L.y) * g.hy / L.dy; else if (L.dy < 0.0f) ty = -L.y * g.hy / L.dy;
        if (L.dz > 0.0f) tz = (1.0f - L.z) * g.hz / L.dz; else if (L.dz < 0.0f) tz = -L.z * g.hz / L.dz;
        if (tx <= ty && tx <= tz) { tb = tx; axis = 0; } else if (ty <= tz) { tb = ty; axis = 1; } else { tb = tz; axis = 2; }
        tb = fmaxf(tb, 0.0f);
    } else if (reg == R_AIR) {
        rho = kRhoAir; m = 0;
        tb = air_boundary(g, L, kind, axis);
    } else {
        const int l = F_LAYER(L.flags);
        rho = g.lrho[l]; m = g.lmat[l];
        float tf = kInf;
        if (L.dz > 0.0f) tf = (g.zt[l + 1] - L.z) / L.dz; else if (L.dz < 0.0f) tf = (g.zt[l] - L.z) / L.dz;
        tf = fmaxf(tf, 0.0f);
        const float tl = lateral_exit(L.x, L.y, L.dx, L.dy);
        if (tl < tf) { tb = tl; kind = 2; } else { tb = tf; kind = 0; }
    }
    const float T = L.E;
    const float S = stop_pow(P, sh, m, T);
    const float s = fminf(tb, fminf(P.ph.fE * T / (rho * S), P.ph.smax));
    const float S2 = stop_pow(P, sh, m, T - 0.5f * rho * s * S);          // midpoint rule
    const float dE = fminf(T, rho * s * S2);
    const float Tn = T - dE;
    const float dep = T - Tn;                                              // exactly what the particle loses (ledger closes)
    const float Tmid = T - 0.5f * dE;
    if (reg == R_PHANTOM) {
        if (COUNT) cnt[6]++;
        dep_vox(L, P, vox_linear(g, L.vox), dep);
        L.x = fmaf(s * g.ihx, L.dx, L.x); L.y = fmaf(s * g.ihy, L.dy, L.y); L.z = fmaf(s * g.ihz, L.dz, L.z);
    } else if (reg == R_AIR) {
        if (COUNT) cnt[7]++;
        atomicAdd(&sh.led[4], (double)dep);
        L.x = fmaf(s, L.dx, L.x); L.y = fmaf(s, L.dy, L.y); L.z = fmaf(s, L.dz, L.z);
    } else {
        if (COUNT) cnt[8]++;
        dep_epid(L, P, sh, F_LAYER(L.flags), fmaf(0.5f * s, L.dx, L.x), fmaf(0.5f * s, L.dy, L.y), dep);   // pixel of the step midpoint (A24)
        L.x = fmaf(s, L.dx, L.x); L.y = fmaf(s, L.dy, L.y); L.z = fmaf(s, L.dz, L.z);
    }
    L.E = Tn;
    // Highland deflection, applied at the end of the step (reading A13)
    const bool deflect = s > 0.0f;
    float ct = 1.0f, st = 0.0f, cp = 1.0f, sp = 0.0f;
    if (deflect) {
        const float t = rho * s * sh.invX0[m];
        const float bpc = Tmid * (Tmid + 2.0f * kMec2) / (Tmid + kMec2);
        const float th0 = (13.6f / bpc) * sqrtf(t) * fmaxf(0.25f, fmaf(0.038f, __logf(t), 1.0f));
        float ua, ub; rng_pair(L, P, ua, ub);
        const float th = fminf(kPi, th0 * sqrtf(-2.0f * __logf(ua)));
        __sincosf(th, &st, &ct);
        __sincosf(2.0f * kPi * ub - kPi, &sp, &cp);
    } else if (COUNT) cnt[15]++;
    if (s == tb) {                                                         // the step ended on a face: neighbouring voxel / layer / region
        const float e_out = L.E + (F_TYPE(L.flags) == T_POSITRON ? 2.0f * kMec2 : 0.0f);
        if (reg == R_PHANTOM) {
            const bool up = comp3(L.dx, L.dy, L.dz, axis) > 0.0f;
            int ix = (int)(L.vox & 1023u), iy = (int)((L.vox >> 10) & 1023u), iz = (int)((L.vox >> 20) & 1023u);
            bool out;
            if (axis == 0) { ix += up ? 1 : -1; L.x = up ? 0.0f : 1.0f; out = ix < 0 || ix >= g.nx; }
            else if (axis == 1) { iy += up ? 1 : -1; L.y = up ? 0.0f : 1.0f; out = iy < 0 || iy >= g.ny; }
            else { iz += up ? 1 : -1; L.z = up ? 0.0f : 1.0f; out = iz < 0 || iz >= g.nz; }
            if (out) {
                frac_to_world(L, g);                                       // uses the old index; then snap the crossed axis
                if (axis == 0) L.x = up ? g.hix : g.lox; else if (axis == 1) L.y = up ? g.hiy : g.loy; else L.z = up ? g.hiz : g.loz;
                SET_REGION(L.flags, R_AIR);
            } else {
                L.vox = (uint32_t)ix | ((uint32_t)iy << 10) | ((uint32_t)iz << 20);
                L.cw = __ldg(P.vox + vox_linear(g, L.vox));
            }
        } else if (reg == R_AIR) {
            if (kind == 0) enter_phantom(L, P, axis);
            else if (kind == 1) enter_epid(L, g);
            else { atomicAdd(&sh.led[5], (double)e_out); L.alive = false; return; }
        } else {
            const int l = F_LAYER(L.flags);
            if (kind == 2) { atomicAdd(&sh.led[5], (double)e_out); L.alive = false; return; }
            if (L.dz > 0.0f) {
                L.z = g.zt[l + 1];
                if (l + 1 >= g.n_layers) { atomicAdd(&sh.led[5], (double)e_out); L.alive = false; return; }
                SET_LAYER(L.flags, l + 1);
            } else {
                L.z = g.zt[l];
                if (l == 0) epid_to_air(L, g); else SET_LAYER(L.flags, l - 1);
            }
        }
    }
    if (deflect) rotate(L.dx, L.dy, L.dz, ct, st, cp, sp);
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
    uint32_t j = upper_bound_u32(so.thrF + 1, (uint32_t)(so.fu * so.fv - 1), r1);
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
template <bool COUNT>
__global__ void __launch_bounds__(kBlock, kMinBlocks) transport_kernel(const __grid_constant__ TransportParams P) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    {
        uint32_t* dst = reinterpret_cast<uint32_t*>(smem_raw);
        for (int i = threadIdx.x; i < P.tb.blob_words; i += kBlock) dst[i] = __ldg(P.tb.blob + i);
    }
    Shared sh;
    sh.phot = reinterpret_cast<const float4*>(smem_raw);
    sh.maj = reinterpret_cast<const float*>(sh.phot + P.tb.n_mat * P.tb.n_E);
    sh.lnS = sh.maj + P.tb.n_E;
    sh.invX0 = sh.lnS + P.tb.n_mat * P.tb.n_T;
    sh.led = reinterpret_cast<double*>(smem_raw + (((size_t)P.tb.blob_words * 4 + 15) & ~(size_t)15));
    if (threadIdx.x < 8) sh.led[threadIdx.x] = 0.0;
    __syncthreads();

    StackEntry stk[kStackDepth];
    uint32_t cnt[16];
    if (COUNT) {
#pragma unroll
        for (int i = 0; i < 16; ++i) cnt[i] = 0;
    }
    Lane L;
    L.alive = false; L.sp = 0; L.pval = 0.0f; L.pidx = 0xffffffffu; L.lph = 0.0; L.flags = 0; L.blk = 0; L.pid = 0; L.h = 0;
    L.x = L.y = L.z = 0.0f; L.dx = L.dy = 0.0f; L.dz = 1.0f; L.E = 0.0f; L.vox = 0; L.cw = 0; L.ci = 0; L.ct = 0.0f; L.mumaj = 1.0f; L.r2 = L.r3 = 0;
    const unsigned lane = threadIdx.x & 31u;
    const unsigned lt_mask = (1u << lane) - 1u;
    uint32_t wnext = 0, wend = 0, wbatch = 0;      // warp-uniform: current chunk of relative history indices
    bool wdone = false;
    double emitted = 0.0;
    uint32_t max_sp = 0;

    for (;;) {
        if (!L.alive && L.sp > 0) {                // next secondary of this lane's history
            const StackEntry& s = stk[--L.sp];
            L.x = s.x; L.y = s.y; L.z = s.z; L.dx = s.dx; L.dy = s.dy; L.dz = s.dz; L.E = s.E;
            L.flags = s.flags; L.vox = s.vox; L.pid = s.pid; L.blk = s.blk;
            L.alive = true;
            if (F_TYPE(L.flags) == T_PHOTON) set_energy(L, P, sh);
            else if (F_REGION(L.flags) == R_PHANTOM) L.cw = __ldg(P.vox + vox_linear(P.g, L.vox));
        }
        if (!wdone) {
            const unsigned need = __ballot_sync(FULL_MASK, !L.alive);
            if (need) {
                if (wnext == wend) {               // grab the next chunk
                    uint32_t c = 0;
                    if (lane == 0) c = atomicAdd(P.chunk_counter, 1u);
                    c = __shfl_sync(FULL_MASK, c, 0);
                    if (c >= P.n_chunks) wdone = true;
                    else {
                        wnext = c * (uint32_t)kChunk;
                        wend = min(P.n, wnext + (uint32_t)kChunk);
                        wbatch = (uint32_t)(((uint64_t)c * (uint64_t)P.n_batches) / P.n_chunks);
                    }
                }
                if (!wdone) {
                    const uint32_t rank = __popc(need & lt_mask);
                    const uint32_t avail = wend - wnext;
                    if (!L.alive && rank < avail) {                        // start history wnext + rank
                        flush_pending(L, P);
                        L.h = wnext + rank; L.pid = 0; L.blk = 0;
                        uint32_t r0, r1, r2, r3;
                        rng_block(L, P, r0, r1, r2, r3);                   // block 0 of particle 0: E, pixel, u, v (reading A1)
                        const SourceSample s = sample_source(P, r0, r1, r2, r3);
                        L.x = P.g.src[0]; L.y = P.g.src[1]; L.z = P.g.src[2];
                        L.dx = s.dx; L.dy = s.dy; L.dz = s.dz; L.E = s.E;
                        L.flags = T_PHOTON | (R_AIR << 2) | (wbatch << 16);
                        L.alive = true; L.sp = 0;
                        emitted += (double)s.E;
                        set_energy(L, P, sh);
                    }
                    wnext += min((uint32_t)__popc(need), avail);
                }
            }
        }
        if (!__any_sync(FULL_MASK, L.alive)) { if (wdone) break; else continue; }
        if (L.alive) {
            if (F_TYPE(L.flags) == T_PHOTON) photon_event<COUNT>(L, P, sh, stk, cnt);
            else electron_event<COUNT>(L, P, sh, stk, cnt);
            if (COUNT) max_sp = max(max_sp, (uint32_t)L.sp);
        }
    }
    flush_pending(L, P);
    atomicAdd(&sh.led[0], emitted);
    atomicAdd(&sh.led[1], L.lph);
    __syncthreads();
    if (threadIdx.x < 8 && threadIdx.x != 6) { const double v = sh.led[threadIdx.x]; if (v != 0.0) atomicAdd(P.ledger + threadIdx.x, v); }
    if (COUNT) {
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            if (i == 11) continue;
            uint32_t v = cnt[i];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL_MASK, v, o);
            if (lane == 0 && v) atomicAdd(P.counters + i, (unsigned long long)v);
        }
        atomicMax(P.counters + 11, (unsigned long long)max_sp);
    }
}

size_t transport_smem_bytes(const Tables& t) { return (((size_t)t.blob_words * 4 + 15) & ~(size_t)15) + 8 * sizeof(double); }

int launch_transport(const TransportParams& p, bool counting, int sm_count, void* stream) {
    const size_t smem = transport_smem_bytes(p.tb);
    cudaError_t e;
    if (counting) e = cudaFuncSetAttribute(transport_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    else e = cudaFuncSetAttribute(transport_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return (int)e;
    int per_sm = 0;
    if (counting) cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, transport_kernel<true>, kBlock, smem);
    else cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, transport_kernel<false>, kBlock, smem);
    if (per_sm < 1) per_sm = 1;
    // persistent grid: every resident CTA slot of every SM, but no more warps than chunks
    long long blocks = (long long)sm_count * per_sm;
    const long long need = ((long long)p.n_chunks + (kBlock / 32) - 1) / (kBlock / 32);
    if (blocks > need) blocks = need;
    if (blocks < 1) blocks = 1;
    if (counting) transport_kernel<true><<<(unsigned)blocks, kBlock, smem, (cudaStream_t)stream>>>(p);
    else transport_kernel<false><<<(unsigned)blocks, kBlock, smem, (cudaStream_t)stream>>>(p);
    return (int)cudaGetLastError();
}

// K1 alone (aepid_sample_source): out[k] = {E, dx, dy, dz, pixel, u, v, 0} for history first + k
__global__ void sample_source_kernel(const __grid_constant__ TransportParams P, uint64_t first, uint64_t n, float* __restrict__ out) {
    const uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const uint64_t h = first + k;
    uint32_t r0, r1, r2, r3;
    philox4x32_10((uint32_t)h, (uint32_t)(h >> 32), 0u, 0u, (uint32_t)P.seed, (uint32_t)(P.seed >> 32), r0, r1, r2, r3);
    const SourceSample s = sample_source(P, r0, r1, r2, r3);
    float4* o = reinterpret_cast<float4*>(out + 8 * k);
    o[0] = make_float4(s.E, s.dx, s.dy, s.dz);
    o[1] = make_float4((float)s.pixel, s.u, s.v, 0.0f);
}
void launch_sample_source(const TransportParams& p, uint64_t first, uint64_t n, float* out, void* stream) {
    if (n == 0) return;
    sample_source_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(p, first, n, out);
}

}  // namespace aepid
