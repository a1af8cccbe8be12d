// sl1m_noalloc.cu -- sl1m_forward_noalloc: the forward apply v = M x of eq (9) (delta pixels, unit
// gains) for callers that must not allocate device memory.
//
// Who that is.  Every other entry point of this library works on a plan, and sl1m_plan_create reserves the plan's
// workspaces with cudaMalloc.  Some programs cannot afford that call at the point where they need an apply:
//   * a real-time correlator back-end or imaging loop that keeps the GPU busy on other streams -- cudaMalloc and cudaFree
//     wait for (and hold up) all work on the device, so one allocation stalls every stream of the process;
//   * a process whose device memory has been handed, all of it, to a pool owned by someone else (a framework's caching
//     allocator, a job scheduler's fixed carve-up): a raw cudaMalloc there fails or eats into another tenant's share;
//   * code that runs under a "no driver allocations after start-up" rule (long-running services that want a flat,
//     auditable memory footprint).
// For them this file gives one plan-less call.  The caller passes inputs and outputs that already live on the device;
// the only other global memory the kernels touch -- the per-split partial sums of the pixel-split forward, the same
// role sl1m_plan's ws_v workspace plays for sl1m_forward -- is the file-scope array g_scratch below.  It is part of
// the library image: every GPU on which the library's module gets loaded carries these 4 MiB until the process exits,
// whether or not this entry point is ever called.  No cudaMalloc, cudaFree, cudaMallocAsync, cudaMallocHost or
// allocating library routine is called here.
//
// The kernel is the pixel-split fp64-phase forward (the shape of fwd_kernel_p64 in sl1m_kernels.cuh) without a plan:
// no Morton sort, no tile centres, no zero-skipping; l, m are read as given (fp64) and n_k - 1 = -r^2/(1+n_k), 1/n_k
// are formed in fp64 per pixel while the tile is staged.  The whole phase u l + v m + w (n - 1) is accumulated in fp64
// turns, its fraction is taken exactly, and sin/cos come from MUFU -- so accuracy does not depend on the pixel order or
// the baseline length.  Partials are summed in a fixed order by a second kernel: results are bit-stable run to run.
#include "../../include/sl1m.h"
#include "sl1m_internal.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cstdio>
#include <mutex>

namespace {

constexpr int NA_NT = 256;                         // threads per CTA
constexpr int NA_RV = 2;                           // visibilities per thread
constexpr int NA_TP = 256;                         // pixels per staged tile
constexpr long long NA_SLOTS = SL1M_NOALLOC_MAX_VIS;   // float2 partial slots: n_vis * splits <= NA_SLOTS
constexpr int NA_MAX_SPLIT = 64;
constexpr int NA_MAX_DEVICES = 64;

// The scratch.  In HOST code this name is only a handle for cudaGetSymbolAddress (below); passing it to a kernel as
// if it were a pointer would hand the kernel a host address.  Device code may name it directly.
static __device__ __align__(256) float2 g_scratch[NA_SLOTS];

std::mutex g_setup_mutex;
float2 *g_scratch_ptr[NA_MAX_DEVICES] = {};       // device address of g_scratch on each device, 0 = not looked up yet

// frac(turns) * 2 pi as an fp32 angle in [-pi, pi): magic-number add (1.5 * 2^20, ulp 2^-32) leaves
// round(turns * 2^32) mod 2^32 in the low word; 23 bits of it go to sin.approx / cos.approx.
__device__ __forceinline__ float turns_to_radians(double turns) {
    const int frac32 = __double2loint(turns + 1572864.0);
    const int s23 = frac32 >> 9;
    const float f = __int_as_float(0x4B400000 + s23) - 12582912.0f;
    return f * 7.490140565847157e-07f;             // 2 pi / 2^23
}

// part[split][n_vis] = sum over the split's pixels of x_k / n_k * exp(-2 pi i (u l_k + v m_k + w (n_k - 1)))
__global__ void __launch_bounds__(NA_NT) noalloc_fwd_kernel(int n_vis, const double *__restrict__ uvw, long long n_pix,
                                                            const double *__restrict__ l, const double *__restrict__ m,
                                                            const float *__restrict__ x, long long tiles_per_split,
                                                            float2 *__restrict__ part) {
    __shared__ double s_l[NA_TP], s_m[NA_TP], s_n[NA_TP];
    __shared__ float s_ax[NA_TP];
    const int tid = threadIdx.x;
    const int jbase = blockIdx.x * (NA_NT * NA_RV);
    double u[NA_RV], v[NA_RV], w[NA_RV];
    float re[NA_RV], im[NA_RV];
#pragma unroll
    for (int r = 0; r < NA_RV; ++r) {
        const int j = min(jbase + r * NA_NT + tid, n_vis - 1);
        u[r] = uvw[3 * (size_t)j + 0];
        v[r] = uvw[3 * (size_t)j + 1];
        w[r] = uvw[3 * (size_t)j + 2];
        re[r] = 0.f;
        im[r] = 0.f;
    }
    const long long k0 = (long long)blockIdx.y * tiles_per_split * NA_TP;
    const long long k1 = min(k0 + tiles_per_split * NA_TP, n_pix);
    for (long long kb = k0; kb < k1; kb += NA_TP) {
        const long long k = kb + tid;                  // NA_TP == NA_NT: one pixel per thread
        double lk = 0.0, mk = 0.0, nk = 0.0;
        float ax = 0.f;
        if (k < k1) {
            lk = l[k];
            mk = m[k];
            const double r2 = lk * lk + mk * mk;
            const double n = sqrt(1.0 - r2);           // NaN for l^2 + m^2 > 1: not validated here (sl1m.h)
            nk = -r2 / (1.0 + n);                      // n - 1 without cancellation
            ax = (float)((double)x[k] / n);
        }
        __syncthreads();                               // the previous tile has been consumed
        s_l[tid] = lk;
        s_m[tid] = mk;
        s_n[tid] = nk;
        s_ax[tid] = ax;
        __syncthreads();
        const int np = (int)min((long long)NA_TP, k1 - kb);
#pragma unroll 2
        for (int p = 0; p < np; ++p) {
            const double pl = s_l[p], pm = s_m[p], pn = s_n[p];
            const float wt = s_ax[p];
#pragma unroll
            for (int r = 0; r < NA_RV; ++r) {
                const float X = turns_to_radians(fma(u[r], pl, fma(v[r], pm, w[r] * pn)));
                float s, c;
                __sincosf(X, &s, &c);
                re[r] = fmaf(wt, c, re[r]);
                im[r] = fmaf(-wt, s, im[r]);
            }
        }
    }
    float2 *out = part + (size_t)blockIdx.y * (size_t)n_vis;
#pragma unroll
    for (int r = 0; r < NA_RV; ++r) {
        const int j = jbase + r * NA_NT + tid;
        if (j < n_vis) out[j] = make_float2(re[r], im[r]);
    }
}

// vis[j] = part[0][j] + part[1][j] + ... in that order
__global__ void __launch_bounds__(256) noalloc_reduce_kernel(int n_vis, int n_split, const float2 *__restrict__ part,
                                                             float2 *__restrict__ vis) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n_vis) return;
    float2 a = part[j];
    for (int s = 1; s < n_split; ++s) {
        const float2 b = part[(size_t)s * (size_t)n_vis + j];
        a.x += b.x;
        a.y += b.y;
    }
    vis[j] = a;
}

// Device address of g_scratch on the current device, looked up once per device.
int scratch_for_current_device(float2 **out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return sl1m_fail(SL1M_ERR_CUDA, cudaGetErrorString(e));
    if (dev < 0 || dev >= NA_MAX_DEVICES) return sl1m_fail(SL1M_ERR_CUDA, "sl1m_forward_noalloc: device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_scratch_ptr[dev]) {
        float2 *ptr = nullptr;
        e = cudaGetSymbolAddress((void **)&ptr, g_scratch);      // `dev` is current: the address is this device's copy
        if (e != cudaSuccess || !ptr) {
            char msg[160];
            snprintf(msg, sizeof msg, "sl1m_forward_noalloc: cudaGetSymbolAddress(scratch) on device %d: %s", dev,
                     e != cudaSuccess ? cudaGetErrorString(e) : "null address");
            return sl1m_fail(SL1M_ERR_CUDA, msg);
        }
        g_scratch_ptr[dev] = ptr;
    }
    *out = g_scratch_ptr[dev];
    return SL1M_OK;
}

}  // namespace

extern "C" int sl1m_forward_noalloc(int64_t n_vis, const double *uvw_dev, int64_t n_pix, const double *l_dev,
                                    const double *m_dev, const float *x_dev, float *vis_dev, void *stream) {
    if (!uvw_dev || !l_dev || !m_dev || !x_dev || !vis_dev)
        return sl1m_fail(SL1M_ERR_NULL, "sl1m_forward_noalloc: uvw_dev, l_dev, m_dev, x_dev and vis_dev are all required");
    if (n_vis < 1 || n_pix < 1) return sl1m_fail(SL1M_ERR_SIZE, "sl1m_forward_noalloc: n_vis and n_pix must be >= 1");
    if (n_vis > SL1M_NOALLOC_MAX_VIS || n_pix > SL1M_NOALLOC_MAX_PIX) {
        char msg[384];
        snprintf(msg, sizeof msg,
                 "sl1m_forward_noalloc: n_vis = %lld, n_pix = %lld is beyond what the static scratch array serves "
                 "(at most %lld visibilities and %lld pixels per call); use a plan (sl1m_plan_create + sl1m_forward) or "
                 "split the visibilities over several calls",
                 (long long)n_vis, (long long)n_pix, (long long)SL1M_NOALLOC_MAX_VIS, (long long)SL1M_NOALLOC_MAX_PIX);
        return sl1m_fail(SL1M_ERR_SIZE, msg);
    }
    float2 *scratch = nullptr;
    if (int st = scratch_for_current_device(&scratch)) return st;

    // launch shape: visibility tiles x pixel splits, about 4 CTAs per SM, splits bounded by the scratch slots
    int n_sm = 148, dev = 0;
    cudaGetDevice(&dev);
    if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n_sm < 1) n_sm = 148;
    const long long vis_tiles = (n_vis + NA_NT * NA_RV - 1) / (NA_NT * NA_RV);
    const long long n_tiles = (n_pix + NA_TP - 1) / NA_TP;
    long long split = std::max<long long>(1, (4LL * n_sm + vis_tiles - 1) / vis_tiles);
    split = std::min<long long>({split, n_tiles, NA_SLOTS / n_vis, (long long)NA_MAX_SPLIT});
    const long long tiles_per_split = (n_tiles + split - 1) / split;
    split = (n_tiles + tiles_per_split - 1) / tiles_per_split;   // no empty split: every slot read below is written first

    cudaStream_t s = (cudaStream_t)stream;
    noalloc_fwd_kernel<<<dim3((unsigned)vis_tiles, (unsigned)split), NA_NT, 0, s>>>(
        (int)n_vis, uvw_dev, (long long)n_pix, l_dev, m_dev, x_dev, tiles_per_split, scratch);
    noalloc_reduce_kernel<<<(unsigned)((n_vis + 255) / 256), 256, 0, s>>>((int)n_vis, (int)split, scratch,
                                                                         (float2 *)vis_dev);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return sl1m_fail(SL1M_ERR_CUDA, cudaGetErrorString(e));
    return SL1M_OK;
}
