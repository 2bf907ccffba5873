// Elementwise / reduction kernels around the transport kernel (SURVEY.md 8(a) K7 fold, K8 response post-pass;
// PAPER.md:114-123, 151-153) and the voxel repacking done by aepid_load_phantom.  All HBM-bound streaming
// kernels: coalesced 128-bit accesses, grid-stride loops sized to the SM count.
#include <cuda_runtime.h>
#include <cstdint>
#include "params.h"

namespace aepid {

static inline unsigned grid_for(size_t n, int per_block) {
    size_t b = (n + per_block - 1) / per_block;
    const size_t cap = 148 * 16;                  // a few waves of the 148 SMs
    if (b > cap) b = cap;
    if (b < 1) b = 1;
    return (unsigned)b;
}

// ---- voxel repacking: density (rounded to 19 mantissa bits) | material (5 bits); per-material max density
// A material byte >= n_mat raises *bad (aepid_load_phantom then fails) instead of aliasing to a valid material.
__global__ void pack_voxels_kernel(const float* __restrict__ rho, const unsigned char* __restrict__ mat, uint32_t* __restrict__ out,
                                   size_t n, float* __restrict__ rho_max, int n_mat, unsigned int* __restrict__ bad) {
    __shared__ unsigned int s_max[kMaxMat];
    if (threadIdx.x < kMaxMat) s_max[threadIdx.x] = 0u;
    __syncthreads();
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const float r = fmaxf(rho[i], 0.0f);
        if ((int)mat[i] >= n_mat) atomicOr(bad, 1u);
        const uint32_t m = mat[i] & 31u;
        const uint32_t bits = (__float_as_uint(r) + 16u) & ~31u;     // round to nearest on the kept mantissa
        out[i] = bits | m;
        atomicMax(&s_max[m], bits);                                   // positive floats order like their bit patterns
    }
    __syncthreads();
    if (threadIdx.x < kMaxMat && s_max[threadIdx.x]) atomicMax(reinterpret_cast<unsigned int*>(rho_max) + threadIdx.x, s_max[threadIdx.x]);
}
void launch_pack_voxels(const float* rho, const unsigned char* mat, uint32_t* out, size_t n, float* rho_max, int n_mat, unsigned int* bad, void* stream) {
    cudaMemsetAsync(rho_max, 0, kMaxMat * sizeof(float), (cudaStream_t)stream);
    cudaMemsetAsync(bad, 0, sizeof(unsigned int), (cudaStream_t)stream);
    pack_voxels_kernel<<<grid_for(n, 256), 256, 0, (cudaStream_t)stream>>>(rho, mat, out, n, rho_max, n_mat, bad);
}

// ---- body box of the phantom (params.h: Geom::glo).  f_v = rho_v kfac[m_v] bounds the voxel's attenuation coefficient
// relative to the majorant at every energy (kfac[m] = max over the energy nodes of mu_m(E_j) / majorant(E_j), api.cu).
// Pass 1: index bounding box B of the voxels with f_v > thr (box[0..2] = min, box[3..5] = max, inclusive; empty: max < min).
// Pass 2: the largest f_v among the voxels outside B (as float bits; positive floats order like their bit patterns).
__global__ void body_box_kernel(const uint32_t* __restrict__ vox, int nx, int ny, int nz, const float* __restrict__ kfac, float thr, int* __restrict__ box) {
    __shared__ int s_box[6];
    if (threadIdx.x < 3) s_box[threadIdx.x] = 0x7fffffff; else if (threadIdx.x < 6) s_box[threadIdx.x] = -1;
    __syncthreads();
    const size_t n = (size_t)nx * ny * nz;
    int lo[3] = {0x7fffffff, 0x7fffffff, 0x7fffffff}, hi[3] = {-1, -1, -1};
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const uint32_t w = __ldg(vox + i);
        if (__uint_as_float(w & ~31u) * __ldg(kfac + (w & 31u)) > thr) {
            const int ix = (int)(i % (size_t)nx), iy = (int)((i / (size_t)nx) % (size_t)ny), iz = (int)(i / ((size_t)nx * ny));
            lo[0] = min(lo[0], ix); lo[1] = min(lo[1], iy); lo[2] = min(lo[2], iz);
            hi[0] = max(hi[0], ix); hi[1] = max(hi[1], iy); hi[2] = max(hi[2], iz);
        }
    }
    for (int a = 0; a < 3; ++a) { if (hi[a] >= 0) { atomicMin(&s_box[a], lo[a]); atomicMax(&s_box[3 + a], hi[a]); } }
    __syncthreads();
    if (threadIdx.x < 3) { if (s_box[threadIdx.x] != 0x7fffffff) atomicMin(box + threadIdx.x, s_box[threadIdx.x]); }
    else if (threadIdx.x < 6) { if (s_box[threadIdx.x] >= 0) atomicMax(box + threadIdx.x, s_box[threadIdx.x]); }
}
__global__ void body_out_kernel(const uint32_t* __restrict__ vox, int nx, int ny, int nz, const float* __restrict__ kfac, const int* __restrict__ box,
                                unsigned int* __restrict__ fout_bits) {
    __shared__ unsigned int s_max;
    if (threadIdx.x == 0) s_max = 0u;
    __syncthreads();
    const int b0 = box[0], b1 = box[1], b2 = box[2], b3 = box[3], b4 = box[4], b5 = box[5];
    const size_t n = (size_t)nx * ny * nz;
    unsigned int mx = 0u;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const int ix = (int)(i % (size_t)nx), iy = (int)((i / (size_t)nx) % (size_t)ny), iz = (int)(i / ((size_t)nx * ny));
        if (ix >= b0 && ix <= b3 && iy >= b1 && iy <= b4 && iz >= b2 && iz <= b5) continue;
        const uint32_t w = __ldg(vox + i);
        mx = max(mx, __float_as_uint(__uint_as_float(w & ~31u) * __ldg(kfac + (w & 31u))));
    }
    if (mx) atomicMax(&s_max, mx);
    __syncthreads();
    if (threadIdx.x == 0 && s_max) atomicMax(fout_bits, s_max);
}
// box: 6 ints, fout_bits: 1 uint (device); kfac: [kMaxMat] floats (device)
void launch_body_box(const uint32_t* vox, int nx, int ny, int nz, const float* kfac, float thr, int* box, unsigned int* fout_bits, void* stream) {
    const int init[6] = {0x7fffffff, 0x7fffffff, 0x7fffffff, -1, -1, -1};
    cudaMemcpyAsync(box, init, sizeof(init), cudaMemcpyHostToDevice, (cudaStream_t)stream);
    cudaMemsetAsync(fout_bits, 0, sizeof(unsigned int), (cudaStream_t)stream);
    const size_t n = (size_t)nx * ny * nz;
    body_box_kernel<<<grid_for(n, 256), 256, 0, (cudaStream_t)stream>>>(vox, nx, ny, nz, kfac, thr, box);
    body_out_kernel<<<grid_for(n, 256), 256, 0, (cudaStream_t)stream>>>(vox, nx, ny, nz, kfac, box, fout_bits);
}

// ---- K7 fold: mean per history and standard error of the mean from B independent batch sums
// mean = sum_b x_b / N;  sigma^2 = sum_b n_b (x_b/n_b - mean)^2 / ((B_eff - 1) N)
// One pass over the batches (HBM-bound: 4 B n_batches per bin read once, 8 B written): with s1 = sum_b x_b and
// s2 = sum_b x_b^2 / n_b the sum of squares above is s2 - N mean^2 (doubles; the batch sums are floats).
template <int V>
__device__ __forceinline__ void fold_bins(const FoldParams& p, size_t i) {
    double s1[V], s2[V];
#pragma unroll
    for (int v = 0; v < V; ++v) { s1[v] = 0.0; s2[v] = 0.0; }
    int nb = 0;
    for (int b = 0; b < p.n_batches; ++b) {
        const double nh = p.hist[b];
        float x[V];
        if (V == 4) {
            const float4 q = __ldcs(reinterpret_cast<const float4*>(p.batches + (size_t)b * p.n + i));
            x[0] = q.x; x[1 % V] = q.y; x[2 % V] = q.z; x[3 % V] = q.w;
        } else x[0] = __ldcs(p.batches + (size_t)b * p.n + i);
        const double inh = nh > 0.0 ? 1.0 / nh : 0.0;
        nb += nh > 0.0 ? 1 : 0;
#pragma unroll
        for (int v = 0; v < V; ++v) { const double d = (double)x[v]; s1[v] += d; s2[v] += d * d * inh; }
    }
#pragma unroll
    for (int v = 0; v < V; ++v) {
        const double mean = p.total > 0.0 ? s1[v] / p.total : 0.0;
        if (p.mean) p.mean[i + v] = (float)mean;
        if (p.sigma) p.sigma[i + v] = nb > 1 ? (float)sqrt(fmax(s2[v] - p.total * mean * mean, 0.0) / ((double)(nb - 1) * p.total)) : 0.0f;
    }
}
__global__ void fold_kernel(const __grid_constant__ FoldParams p, int vec) {
    const size_t stride = (size_t)gridDim.x * blockDim.x, t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (vec) { for (size_t i = 4 * t; i < p.n; i += 4 * stride) fold_bins<4>(p, i); }
    else { for (size_t i = t; i < p.n; i += stride) fold_bins<1>(p, i); }
}
void launch_fold(const FoldParams& p, void* stream) {
    if (p.n == 0) return;
    const int vec = p.n % 4 == 0 && ((uintptr_t)p.batches % 16) == 0;     // 128-bit loads: every batch row stays 16-byte aligned
    fold_kernel<<<grid_for(vec ? p.n / 4 : p.n, 256), 256, 0, (cudaStream_t)stream>>>(p, vec);
}

// ---- multi-GPU exchange: per-bin moments of the batches, and their finalisation after the all-reduce
__global__ void moments_kernel(const __grid_constant__ FoldParams p, double* __restrict__ s1, double* __restrict__ s2) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < p.n; i += (size_t)gridDim.x * blockDim.x) {
        double a = 0.0, q = 0.0;
        for (int b = 0; b < p.n_batches; ++b) {
            const double nh = p.hist[b];
            if (nh <= 0.0) continue;
            const double x = (double)p.batches[(size_t)b * p.n + i];
            a += x; q += x * x / nh;
        }
        if (s1) s1[i] = a;
        if (s2) s2[i] = q;
    }
}
void launch_moments(const FoldParams& p, double* s1, double* s2, void* stream) {
    if (p.n == 0) return;
    moments_kernel<<<grid_for(p.n, 256), 256, 0, (cudaStream_t)stream>>>(p, s1, s2);
}
__global__ void finalize_moments_kernel(const double* __restrict__ s1, const double* __restrict__ s2, size_t n, double total, double batches,
                                        float* __restrict__ mean, float* __restrict__ sigma) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const double m = total > 0.0 ? s1[i] / total : 0.0;
        if (mean) mean[i] = (float)m;
        if (sigma) sigma[i] = batches > 1.0 ? (float)sqrt(fmax(s2[i] - total * m * m, 0.0) / ((batches - 1.0) * total)) : 0.0f;
    }
}
void launch_finalize_moments(const double* s1, const double* s2, size_t n, double total, double batches, float* mean, float* sigma, void* stream) {
    if (n == 0) return;
    finalize_moments_kernel<<<grid_for(n, 256), 256, 0, (cudaStream_t)stream>>>(s1, s2, n, total, batches, mean, sigma);
}

// ---- K8 radiological thickness: one ray per EPID pixel, 3-D DDA through the packed grid (reading A17)
__global__ void tmap_kernel(const __grid_constant__ Geom g, const uint32_t* __restrict__ vox, float* __restrict__ tmap) {
    const int ju = blockIdx.x * blockDim.x + threadIdx.x, jv = blockIdx.y * blockDim.y + threadIdx.y;
    if (ju >= g.nu || jv >= g.nv) return;
    const float pu = ((float)ju + 0.5f) * g.pitch - g.half_u, pv = ((float)jv + 0.5f) * g.pitch - g.half_v, pw = g.sid;
    // ray source -> pixel centre, world frame, parameter a in [0, 1]
    const float ex = pu * g.au[0] + pv * g.av[0] + pw * g.aw[0], ey = pu * g.au[1] + pv * g.av[1] + pw * g.aw[1], ez = pu * g.au[2] + pv * g.av[2] + pw * g.aw[2];
    const float len = sqrtf(ex * ex + ey * ey + ez * ez);
    const float d[3] = {ex, ey, ez}, s[3] = {g.src[0], g.src[1], g.src[2]};
    const float lo[3] = {g.lox, g.loy, g.loz}, hi[3] = {g.hix, g.hiy, g.hiz}, h[3] = {g.hx, g.hy, g.hz};
    const int n[3] = {g.nx, g.ny, g.nz};
    float a0 = 0.0f, a1 = 1.0f; bool hit = true;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        if (fabsf(d[a]) < 1e-20f) { if (s[a] < lo[a] || s[a] >= hi[a]) hit = false; continue; }
        float t1 = (lo[a] - s[a]) / d[a], t2 = (hi[a] - s[a]) / d[a];
        if (t1 > t2) { const float t = t1; t1 = t2; t2 = t; }
        a0 = fmaxf(a0, t1); a1 = fminf(a1, t2);
    }
    float acc = 0.0f;
    if (hit && a0 < a1) {
        int iv[3], step[3]; float tnext[3], dt[3];
        const float am = a0 + 1e-6f * (a1 - a0);
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const float p = s[a] + am * d[a];
            iv[a] = min(max((int)floorf((p - lo[a]) / h[a]), 0), n[a] - 1);
            if (d[a] > 1e-20f) { step[a] = 1; dt[a] = h[a] / d[a]; tnext[a] = (lo[a] + (float)(iv[a] + 1) * h[a] - s[a]) / d[a]; }
            else if (d[a] < -1e-20f) { step[a] = -1; dt[a] = -h[a] / d[a]; tnext[a] = (lo[a] + (float)iv[a] * h[a] - s[a]) / d[a]; }
            else { step[a] = 0; dt[a] = 3e38f; tnext[a] = 3e38f; }
        }
        float a = a0;
        for (;;) {
            const int ax = (tnext[0] <= tnext[1] && tnext[0] <= tnext[2]) ? 0 : (tnext[1] <= tnext[2] ? 1 : 2);
            const float an = fminf(tnext[ax], a1);
            const uint32_t w = __ldg(vox + ((size_t)iv[2] * g.ny + iv[1]) * g.nx + iv[0]);
            acc += fmaxf(an - a, 0.0f) * __uint_as_float(w & ~31u);
            a = an;
            if (tnext[ax] >= a1) break;
            iv[ax] += step[ax]; tnext[ax] += dt[ax];
            if (iv[ax] < 0 || iv[ax] >= n[ax]) break;
        }
    }
    tmap[(size_t)jv * g.nu + ju] = acc * len;
}
void launch_tmap(const Geom& g, const uint32_t* vox, float* tmap, void* stream) {
    dim3 b(32, 8), gr((g.nu + 31) / 32, (g.nv + 7) / 8);
    tmap_kernel<<<gr, b, 0, (cudaStream_t)stream>>>(g, vox, tmap);
}

// ---- K8 apply: signal = dose * bilinear k(t, s), (t, s) clamped into the table (reading A18)
__global__ void apply_lut_kernel(const float* __restrict__ lut, int nt, int ns, float t_min, float t_max, float s_min, float s_max,
                                 float s_eff, const float* __restrict__ dose, const float* __restrict__ tmap, float* __restrict__ out, size_t n) {
    const float fs = ns > 1 ? (fminf(fmaxf(s_eff, s_min), s_max) - s_min) / (s_max - s_min) * (float)(ns - 1) : 0.0f;
    const int is = min((int)floorf(fs), max(ns - 2, 0)), is1 = min(is + 1, ns - 1);
    const float ws = fs - (float)is;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const float ft = nt > 1 ? (fminf(fmaxf(tmap[i], t_min), t_max) - t_min) / (t_max - t_min) * (float)(nt - 1) : 0.0f;
        const int it = min((int)floorf(ft), max(nt - 2, 0)), it1 = min(it + 1, nt - 1);
        const float wt = ft - (float)it;
        const float k0 = (1.0f - ws) * __ldg(lut + it * ns + is) + ws * __ldg(lut + it * ns + is1);
        const float k1 = (1.0f - ws) * __ldg(lut + it1 * ns + is) + ws * __ldg(lut + it1 * ns + is1);
        out[i] = dose[i] * ((1.0f - wt) * k0 + wt * k1);
    }
}
void launch_apply_lut(const float* lut, int nt, int ns, float t_min, float t_max, float s_min, float s_max,
                      float s_eff, const float* dose, const float* tmap, float* out, size_t n, void* stream) {
    if (n == 0) return;
    apply_lut_kernel<<<grid_for(n, 256), 256, 0, (cudaStream_t)stream>>>(lut, nt, ns, t_min, t_max, s_min, s_max, s_eff, dose, tmap, out, n);
}

}  // namespace aepid
