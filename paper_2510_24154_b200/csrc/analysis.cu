// Analysis chain of PAPER.md:141 (section 2.3.3): K9 bilinear up-sampling of the predicted image to the grid of the
// measured one (reading A28) and K10 global 2-D gamma index between two images on the same grid (reading A29).
// K9 is a streaming kernel (HBM-bound: 4 B written per output pixel, the input stays in L2).  K10 is a stencil: every
// reference pixel scans the evaluated pixels inside the disc of radius cap x DTA (about 1000 for 3 mm on a 0.34 mm
// grid), staged once per tile in shared memory, so it is bound by shared-memory reads and FMAs, not by HBM.
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>
#include <mutex>
#include "../../include/aepid.h"
#include "params.h"

namespace aepid {

// ---- K9: out[j][i] = bilinear interpolant of in[nv][nu] at x = (i + 0.5) nu/mu - 0.5, y = (j + 0.5) nv/mv - 0.5
// (input pixel centres at the integers), coordinates clamped to [0, n - 1]
// Position of output pixel i of n_out on the input axis of n_in pixels: x = (i + 0.5) n_in/n_out - 0.5 clamped to
// [0, n_in - 1], returned as cell index i0 and fraction f in integer arithmetic (2 n_out x = (2 i + 1) n_in - n_out),
// so that the cell is exact and f carries one float rounding (sizes <= 32768: everything fits 32 bits).
__device__ __forceinline__ void upsample_coord(int i, int n_in, int n_out, int& i0, float& f) {
    const unsigned num = (2u * (unsigned)i + 1u) * (unsigned)n_in, den = 2u * (unsigned)n_out;
    i0 = 0; f = 0.0f;
    if (n_in == 1 || num <= (unsigned)n_out) return;                        // x <= 0
    const unsigned t = num - (unsigned)n_out, q = t / den, r = t - q * den;
    if (q >= (unsigned)(n_in - 1)) { i0 = n_in - 2; f = 1.0f; }             // x >= n_in - 1
    else { i0 = (int)q; f = (float)r / (float)den; }
}
__global__ void upsample_kernel(const float* __restrict__ in, int nu, int nv, float* __restrict__ out, int mu, int mv) {
    const size_t n = (size_t)mu * mv;
    for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (size_t)gridDim.x * blockDim.x) {
        const int j = (int)(k / mu), i = (int)(k - (size_t)j * mu);
        int i0, j0; float fx, fy;
        upsample_coord(i, nu, mu, i0, fx);
        upsample_coord(j, nv, mv, j0, fy);
        const int i1 = min(i0 + 1, nu - 1), j1 = min(j0 + 1, nv - 1);
        const float a = __ldg(in + (size_t)j0 * nu + i0), b = __ldg(in + (size_t)j0 * nu + i1);
        const float c = __ldg(in + (size_t)j1 * nu + i0), d = __ldg(in + (size_t)j1 * nu + i1);
        const float top = fmaf(fx, b - a, a), bot = fmaf(fx, d - c, c);
        __stcs(out + k, fmaf(fy, bot - top, top));
    }
}
void launch_upsample(const float* in, int nu, int nv, float* out, int mu, int mv, void* stream) {
    const size_t n = (size_t)mu * mv;
    if (n == 0) return;
    size_t b = (n + 255) / 256;
    if (b > 148 * 16) b = 148 * 16;
    upsample_kernel<<<(unsigned)b, 256, 0, (cudaStream_t)stream>>>(in, nu, nv, out, mu, mv);
}

// ---- global maximum of a non-negative image (the bit pattern of a non-negative float orders like the value)
__global__ void image_max_kernel(const float* __restrict__ a, size_t n, unsigned int* __restrict__ out) {
    float m = 0.0f;
    for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (size_t)gridDim.x * blockDim.x) m = fmaxf(m, __ldg(a + k));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0 && m > 0.0f) atomicMax(out, __float_as_uint(m));
}

// ---- K10: gamma[j][i] = min(cap, min over evaluated pixels e within cap x DTA of
//      sqrt(|x_e - x_r|^2 / DTA^2 + (D_e - D_r)^2 / (dose_frac D_max)^2)); -1 below the low-dose threshold.
// stats[0..3] += tested pixels, passing pixels (gamma <= 1), sum of gamma; stats[3] = max gamma (as bits).
constexpr int kGTx = 32, kGTy = 16;
struct GammaParams {
    const float* ref; const float* ev; float* gamma;
    int nu, nv, w;                       // half-width of the search window in pixels
    float c_dist;                        // pitch^2 / DTA^2
    float dose_frac, thr_frac, cap;
    const unsigned int* dmax_bits;
    double* stats;
};
__global__ void __launch_bounds__(kGTx * kGTy) gamma_kernel(const __grid_constant__ GammaParams p) {
    extern __shared__ float tile[];      // evaluated image, (kGTy + 2w) x (kGTx + 2w), +inf-like outside the image
    const int w = p.w, tw = kGTx + 2 * w, th = kGTy + 2 * w;
    const int u0 = blockIdx.x * kGTx - w, v0 = blockIdx.y * kGTy - w;
    for (int k = threadIdx.y * kGTx + threadIdx.x; k < tw * th; k += kGTx * kGTy) {
        const int tj = k / tw, ti = k - tj * tw;
        const int j = v0 + tj, i = u0 + ti;
        tile[k] = (i >= 0 && i < p.nu && j >= 0 && j < p.nv) ? __ldg(p.ev + (size_t)j * p.nu + i) : 3.0e38f;
    }
    __syncthreads();
    const int i = blockIdx.x * kGTx + threadIdx.x, j = blockIdx.y * kGTy + threadIdx.y;
    const float dmax = __uint_as_float(*p.dmax_bits);
    float g = -1.0f; bool tested = false;
    if (i < p.nu && j < p.nv) {
        const float dr = __ldg(p.ref + (size_t)j * p.nu + i);
        tested = dmax > 0.0f && dr >= p.thr_frac * dmax;
        if (tested) {
            const float inv_dd = 1.0f / (p.dose_frac * dmax);
            const float cap2 = p.cap * p.cap;
            float best = cap2;
            const float* row0 = tile + (size_t)threadIdx.y * tw + threadIdx.x;      // window origin (dj = di = -w)
            for (int dj = -w; dj <= w; ++dj) {
                const float dj2 = (float)(dj * dj) * p.c_dist;
                if (dj2 > cap2) continue;
                const float* row = row0 + (size_t)(dj + w) * tw + w;
                // |di| <= floor(sqrt((cap2 - dj2) / c_dist)): the chord of the disc on this row
                const int m = min(w, (int)sqrtf(fmaxf(cap2 - dj2, 0.0f) / p.c_dist + 1e-4f));
                for (int di = -m; di <= m; ++di) {
                    const float d = (row[di] - dr) * inv_dd;
                    const float c = fmaf(d, d, fmaf((float)(di * di), p.c_dist, dj2));
                    best = fminf(best, c);
                }
            }
            g = sqrtf(fminf(best, cap2));
        }
        p.gamma[(size_t)j * p.nu + i] = g;
    }
    // block statistics
    float cnt = tested ? 1.0f : 0.0f, pass = (tested && g <= 1.0f) ? 1.0f : 0.0f, sum = tested ? g : 0.0f, mx = tested ? g : 0.0f;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        cnt += __shfl_xor_sync(0xffffffffu, cnt, o); pass += __shfl_xor_sync(0xffffffffu, pass, o);
        sum += __shfl_xor_sync(0xffffffffu, sum, o); mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    }
    if (threadIdx.x == 0 && cnt > 0.0f) {
        atomicAdd(p.stats + 0, (double)cnt); atomicAdd(p.stats + 1, (double)pass); atomicAdd(p.stats + 2, (double)sum);
        atomicMax(reinterpret_cast<unsigned long long*>(p.stats + 3), (unsigned long long)__double_as_longlong((double)mx));
    }
}
// Returns 0, or -1 if the search window does not fit in shared memory.
int launch_gamma(const float* ref, const float* ev, float* gamma, int nu, int nv, float pitch, float dose_frac, float dta,
                 float thr_frac, float cap, unsigned int* dmax_bits, double* stats, void* stream) {
    cudaStream_t st = (cudaStream_t)stream;
    const size_t n = (size_t)nu * nv;
    cudaMemsetAsync(dmax_bits, 0, 4, st);
    cudaMemsetAsync(stats, 0, 4 * sizeof(double), st);
    size_t b = (n + 255) / 256;
    if (b > 148 * 8) b = 148 * 8;
    image_max_kernel<<<(unsigned)b, 256, 0, st>>>(ref, n, dmax_bits);
    GammaParams p;
    p.ref = ref; p.ev = ev; p.gamma = gamma; p.nu = nu; p.nv = nv;
    p.w = (int)floor((double)cap * (double)dta / (double)pitch + 1e-9);
    p.c_dist = (pitch / dta) * (pitch / dta);
    p.dose_frac = dose_frac; p.thr_frac = thr_frac; p.cap = cap; p.dmax_bits = dmax_bits; p.stats = stats;
    const size_t smem = (size_t)(kGTx + 2 * p.w) * (kGTy + 2 * p.w) * sizeof(float);
    if (smem > 200 * 1024) return -1;
    if (cudaFuncSetAttribute(gamma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -1;
    dim3 grid((nu + kGTx - 1) / kGTx, (nv + kGTy - 1) / kGTy), block(kGTx, kGTy);
    gamma_kernel<<<grid, block, smem, st>>>(p);
    return 0;
}

// ---- Eq. 2 (reading A33): mean of the image over the pixels whose centre lies in the central roi x roi
// square; acc[0] += sum, acc[1] += number of pixels (doubles).  A reduction over a few hundred pixels: latency-bound.
__global__ void roi_sum_kernel(const float* __restrict__ img, int nu, int nv, float pitch, float half_roi, double* __restrict__ acc) {
    const size_t n = (size_t)nu * nv;
    double s = 0.0, c = 0.0;
    for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (size_t)gridDim.x * blockDim.x) {
        const int j = (int)(k / nu), i = (int)(k - (size_t)j * nu);
        const float u = ((float)i + 0.5f - 0.5f * (float)nu) * pitch, v = ((float)j + 0.5f - 0.5f * (float)nv) * pitch;
        if (fabsf(u) <= half_roi && fabsf(v) <= half_roi) { s += (double)__ldg(img + k); c += 1.0; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { s += __shfl_xor_sync(0xffffffffu, s, o); c += __shfl_xor_sync(0xffffffffu, c, o); }
    if ((threadIdx.x & 31) == 0 && c > 0.0) { atomicAdd(acc, s); atomicAdd(acc + 1, c); }
}
void launch_roi_sum(const float* img, int nu, int nv, float pitch, float roi, double* acc, void* stream) {
    cudaStream_t st = (cudaStream_t)stream;
    cudaMemsetAsync(acc, 0, 2 * sizeof(double), st);
    size_t b = ((size_t)nu * nv + 255) / 256;
    if (b > 148 * 4) b = 148 * 4;
    roi_sum_kernel<<<(unsigned)b, 256, 0, st>>>(img, nu, nv, pitch, 0.5f * roi, acc);
}

// ---------------------------------------------------------------- the entry point that allocates nothing (include/aepid.h:
// aepid_gamma_of_upsampled_static).  K9 + K10 in one call with NO context and NO workspace: the up-sampled image (the
// intermediate of the chain), the image maximum and the gamma statistics live in this file-scope device array, which every GPU
// that loads the library holds until the process exits (6.25 MiB + 256 B).  All calls share it: it keeps the last call's
// contents, what must start at zero is cleared on the stream at the start of every call, and calls that overlap on the GPU race.
constexpr size_t kStaticMaxPixels = (size_t)AEPID_STATIC_MAX_PIXELS;                 // 1280 x 1280: the paper's 1190 x 1190 fits
constexpr size_t kStaticStatsOff = kStaticMaxPixels * sizeof(float);                 // double stats[4] | uint32 dmax bits
static __device__ __align__(256) unsigned char g_static_scratch[kStaticStatsOff + 256];

// device code names the array directly: {tested, passing, mean gamma, max gamma} from the raw accumulators
__global__ void static_stats_kernel(double* __restrict__ out) {
    const double* st = reinterpret_cast<const double*>(g_static_scratch + kStaticStatsOff);
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        out[0] = st[0]; out[1] = st[1]; out[2] = st[0] > 0.0 ? st[2] / st[0] : 0.0; out[3] = st[3];
    }
}

// In host code `g_static_scratch` is a host-side stand-in, not a device address: the address a kernel can use comes from
// cudaGetSymbolAddress, once per device, with that device current.
constexpr int kStaticMaxDevices = 64;
static std::mutex g_static_mutex;
static void* g_static_addr[kStaticMaxDevices] = {nullptr};
static cudaError_t static_scratch_address(int device, unsigned char** out) {
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_addr[device]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);              // the current device is `device` (caller)
        if (e != cudaSuccess) return e;
        g_static_addr[device] = p;
    }
    *out = static_cast<unsigned char*>(g_static_addr[device]);
    return cudaSuccess;
}
static bool is_device_pointer(const void* p) {
    cudaPointerAttributes a{};
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

}  // namespace aepid

extern "C" int aepid_gamma_of_upsampled_static(int device, void* cuda_stream, const float* predicted, int nu, int nv,
                                               const float* measured, int mu, int mv, float pitch_cm, float dose_frac, float dta_cm,
                                               float threshold_frac, float gamma_cap, float* gamma_out, double* stats_out,
                                               char* error_text, size_t error_text_bytes) {
    using namespace aepid;
    auto fail = [&](int code, const char* what) {
        if (error_text && error_text_bytes) std::snprintf(error_text, error_text_bytes, "%s", what);
        return code;
    };
    if (error_text && error_text_bytes) error_text[0] = 0;
    if (device < 0 || device >= kStaticMaxDevices) return fail(AEPID_ERR_BAD_ARG, "device index out of range (0..63)");
    if (!predicted || !measured || !gamma_out) return fail(AEPID_ERR_BAD_ARG, "null image pointer");
    if (nu < 1 || nv < 1 || mu < 1 || mv < 1 || nu > 32768 || nv > 32768) return fail(AEPID_ERR_BAD_ARG, "image size out of range");
    if ((size_t)mu * (size_t)mv > kStaticMaxPixels) {
        char buf[320];
        std::snprintf(buf, sizeof buf, "measured grid of %d x %d pixels exceeds the static scratch of aepid_gamma_of_upsampled_static "
                      "(AEPID_STATIC_MAX_PIXELS = %zu, e.g. 1280 x 1280): use aepid_upsample + aepid_gamma_index", mu, mv, kStaticMaxPixels);
        return fail(AEPID_ERR_NOMEM, buf);
    }
    if (!(pitch_cm > 0) || !(dose_frac > 0) || !(dta_cm > 0) || !(threshold_frac >= 0) || !(gamma_cap >= 1))
        return fail(AEPID_ERR_BAD_ARG, "gamma criteria out of range (pitch, dose fraction, DTA > 0; threshold >= 0; cap >= 1)");
    int prev = -1;
    if (cudaGetDevice(&prev) != cudaSuccess) return fail(AEPID_ERR_CUDA, "cudaGetDevice failed");
    if (prev != device && cudaSetDevice(device) != cudaSuccess) return fail(AEPID_ERR_CUDA, "cudaSetDevice failed");
    int rc = 0;
    do {
        if (!is_device_pointer(predicted) || !is_device_pointer(measured) || !is_device_pointer(gamma_out) || (stats_out && !is_device_pointer(stats_out))) {
            rc = fail(AEPID_ERR_BAD_ARG, "aepid_gamma_of_upsampled_static takes device pointers (images, gamma_out, stats_out)"); break;
        }
        unsigned char* scratch = nullptr;
        const cudaError_t e = static_scratch_address(device, &scratch);
        if (e != cudaSuccess) { rc = fail(AEPID_ERR_CUDA, cudaGetErrorString(e)); break; }
        float* up = reinterpret_cast<float*>(scratch);
        double* stats = reinterpret_cast<double*>(scratch + kStaticStatsOff);
        unsigned int* dmax = reinterpret_cast<unsigned int*>(scratch + kStaticStatsOff + 4 * sizeof(double));
        launch_upsample(predicted, nu, nv, up, mu, mv, cuda_stream);                   // K9 into the static scratch (fully overwritten)
        // K10: launch_gamma clears dmax and stats on the stream before it uses them
        if (launch_gamma(measured, up, gamma_out, mu, mv, pitch_cm, dose_frac, dta_cm, threshold_frac, gamma_cap, dmax, stats, cuda_stream) != 0) {
            rc = fail(AEPID_ERR_NOMEM, "search window (cap x DTA / pitch pixels) does not fit in shared memory"); break;
        }
        if (stats_out) static_stats_kernel<<<1, 32, 0, (cudaStream_t)cuda_stream>>>(stats_out);
        const cudaError_t le = cudaGetLastError();
        if (le != cudaSuccess) { rc = fail(AEPID_ERR_CUDA, cudaGetErrorString(le)); break; }
    } while (false);
    if (prev != device) cudaSetDevice(prev);
    return rc;
}
