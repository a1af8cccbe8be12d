// sl1m.cu -- host side of the C ABI declared in include/sl1m.h: argument validation, the fp64
// plan-time precompute (step a0 of SURVEY.md 8(a)), launch configuration and the solver loop.
// All arithmetic of the method on the hot path runs in the kernels of sl1m_kernels.cuh /
// sl1m_epilogue.cuh; there is no CPU fallback.
#include "../../include/sl1m.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>
#ifdef SL1M_BOUNDS
#include <map>
#include <mutex>
#endif

#include "sl1m_epilogue.cuh"
#include "sl1m_internal.h"
#include "sl1m_kernels.cuh"
#include "sl1m_persist.cuh"

using namespace sl1m;

namespace {

thread_local std::string g_last_error;

int fail(int st, const std::string &msg) {
    g_last_error = msg;
    return st;
}

}  // namespace

int sl1m_fail(int st, const char *msg) { return fail(st, msg ? msg : ""); }

namespace {

#define CUDA_TRY(expr)                                                                      \
    do {                                                                                    \
        cudaError_t e_ = (expr);                                                            \
        if (e_ != cudaSuccess)                                                              \
            return fail(e_ == cudaErrorMemoryAllocation ? SL1M_ERR_ALLOC : SL1M_ERR_CUDA,   \
                        std::string(#expr) + ": " + cudaGetErrorString(e_));                \
    } while (0)

#ifdef SL1M_BOUNDS
// Debug build (-DSL1M_BOUNDS; SURVEY.md:184 asks for memcheck, which the GPU pool refuses to run): every device buffer
// this file allocates gets a 4 KiB canary band of 0xA5 on both sides; sl1m_debug_check() verifies all bands.  The
// kernels over-read by design in two documented places (register prefetch of gain rows) and those are asserted in
// range on the device (ldg_gain); a stray WRITE by any kernel lands in a band and is caught here.
constexpr size_t CANARY = 4096;
struct BoundsAlloc { size_t bytes; };
std::map<void *, BoundsAlloc> g_allocs;      // user pointer -> size
std::mutex g_allocs_mu;
cudaError_t bounds_malloc(void **q, size_t bytes) {
    unsigned char *base = nullptr;
    const size_t padded = (bytes + 255) / 256 * 256;          // keep the trailing band aligned
    cudaError_t e = (cudaMalloc)((void **)&base, padded + 2 * CANARY);
    if (e != cudaSuccess) return e;
    (cudaMemset)(base, 0xA5, CANARY);
    (cudaMemset)(base + CANARY + bytes, 0xA5, padded - bytes + CANARY);
    *q = base + CANARY;
    std::lock_guard<std::mutex> lk(g_allocs_mu);
    g_allocs[*q] = BoundsAlloc{bytes};
    return cudaSuccess;
}
cudaError_t bounds_free(void *q) {
    if (!q) return cudaSuccess;
    {
        std::lock_guard<std::mutex> lk(g_allocs_mu);
        auto it = g_allocs.find(q);
        if (it == g_allocs.end()) return (cudaFree)(q);       // not ours (e.g. a caller's buffer)
        g_allocs.erase(it);
    }
    return (cudaFree)((unsigned char *)q - CANARY);
}
#define cudaMalloc(q, n) bounds_malloc((void **)(q), (n))
#define cudaFree(q) bounds_free((void *)(q))
#endif

constexpr int SM_COUNT_B200 = 148;
constexpr int GAIN_ROW_PAD = 4;   // rows of padding behind the forward-layout gain tables (prefetch distance of the kernels)

}  // namespace

struct sl1m_plan {
    int64_t n_vis = 0, n_pix = 0;
    int n_vis_int = 0;           // internal (possibly baseline-grouped, padded) visibility count
    int gk = 0;                  // 0 unit gains, 1 per-term gains, 2 baseline-grouped gains
    int *vperm = nullptr;        // internal position -> caller index (-1 = padding); NULL = identity
    int n_pix_pad = 0, n_tiles = 0, n_ant = 0;
    bool gauss = false, gains = false;
    int pk = 0;                  // pixel kind of the kernels: 0 delta, 1 Gaussian (per-pixel sigma), 2 Gaussian with one sigma per tile
    // device arrays
    double *u64 = nullptr, *v64 = nullptr, *w64 = nullptr;
    int *ant_p = nullptr, *ant_q = nullptr;
    float4 *pix4 = nullptr;
    float4 *pixc = nullptr;       // [n_chan][n_pix_pad] compact tiles of the zero-skipping forward (NULL = dense forward)
    int *tile_cnt = nullptr;      // [n_chan][n_tiles] pixels per compact tile
    float2 *gFc = nullptr;        // [n_chan][n_pix_pad][n_ant] gain rows of the compact entries (gain plans only)
    float2 *gAc = nullptr;        // [n_chan][n_ant][n_pix_pad] the same in the antenna-major layout, for plans whose forward is the
                                  // packed gain kernel (gk == 2, delta pixels): that kernel reads gA / gAc, and gF / gFc do not exist
    bool dense_forward = false;   // SL1M_DENSE_FORWARD: never skip
    float2 *pixg = nullptr;
    double4 *cen = nullptr;
    float *amp = nullptr;
    int *perm = nullptr;
    float2 *gF = nullptr, *gA = nullptr;
    // launch configuration
    int fwd_rv = 8, fwd_vtiles = 0, fwd_split = 1, fwd_per_split = 0;
    int adj_rp = 8, adj_pgroups = 0, adj_split = 1, adj_per_split = 0;
    // workspaces
    float2 *ws_v = nullptr;      // [fwd_split][n_vis]
    float *ws_p = nullptr;       // [adj_split][n_pix_pad]
    float2 *resid = nullptr;     // [n_vis]   residual / forward result
    float2 *rpol = nullptr;      // [n_vis]   residual in polar form (|r|, arg r) for the one-cosine adjoint kernels
    float *I_sorted = nullptr, *y_sorted = nullptr, *g_sorted = nullptr;   // [n_pix_pad]
    double *part_a = nullptr, *part_b = nullptr, *part_c = nullptr;        // block partials
    int n_part = 0;
    double *scalars = nullptr;   // [4] device scalars (norm2, l2, l1, nnz)
    // host-buffer variants
    float *h_x = nullptr, *h_vis = nullptr, *h_img = nullptr;   // device staging for *_host calls
    bool phase64 = false;         // fp64-phase kernels (delta pixels, unit gains) -- flag or automatic
    bool phase64_flag = false;    // SL1M_PHASE_FP64 was given
    bool phase64_capable = false; // delta pixels with unit gains: pixd exists, the fp64-phase kernels can be switched to
    double4 *pixdc = nullptr;     // [n_chan][n_pix_pad] compact copy of pixd for the zero-skipping fp64-phase forward
    float2 *pixgc = nullptr;      // [n_chan][n_pix_pad] compact copy of pixg for the zero-skipping per-pixel-sigma forward
    double4 *pixd = nullptr;      // DEV [n_pix_pad] (dl, dm, dn', 0) as doubles, only with phase64
    double phase_span = 0.0;      // plan-time bound on the fp32 phase remainder, radians
    int n_chan = 1;               // batched channels (NEXT-4): every per-image / per-visibility buffer is [n_chan][.]
    double *chan_scale = nullptr; // DEV [n_chan] nu_c / nu_0, NULL while n_chan == 1
    float2 *step_c = nullptr;     // DEV [n_chan] (1/L_c, lambda_c/L_c) for the batched solver
    double *trace_buf = nullptr;  // plan-owned trace for sl1m_solve_stop when the caller passes none
    size_t trace_cap = 0;         // doubles
    // FISTA state of the stepping API (sl1m_fista_begin / _step / _image); the solve calls are built on it
    bool f_active = false;
    const float2 *f_vis = nullptr;   // BORROWED measured visibilities
    std::vector<float> f_lam, f_L;   // per channel
    float f_inv_L = 0.f, f_thr = 0.f;
    double f_t = 1.0;                // t_{k+1} of the listing (fp64 on the host; beta is a kernel argument)
    int f_k = 0;                     // iterations enqueued since begin
    // device-side termination (sl1m_solve_stop): ctl_i = {done[C], n_done[C], all_done}
    int *ctl_i = nullptr;
    double *lam2 = nullptr;          // DEV [n_chan] 2 lambda_c (the weight of sum I in E, reading R21)
    const int *done_ptr = nullptr;   // == ctl_i while a stopping solve is enqueueing, else NULL
    int *h_flag = nullptr;           // pinned HOST [2]: all_done as seen by the last two polls
    cudaEvent_t poll_ev[2] = {nullptr, nullptr};
    // persistent single-kernel FISTA of small problems (sl1m_persist.cuh)
    bool persist = false, no_persist = false;
    int persist_grid = 0;
    float4 *pvis4 = nullptr;         // [n_vis] 2 pi (u, v, w)
    float *px0 = nullptr;            // [n_tiles][n_vis] centre phases
    double *ppart = nullptr;         // [2][3][persist_grid]
    unsigned *pbar = nullptr;        // grid-barrier counter
    bool persist_small = false;      // <= 1,024 padded pixels and visibilities: fista_persistent_small_kernel (all operands in registers)
    float *pybuf = nullptr;          // DEV [2][n_pix_pad] its double-buffered a*y
    float *pbeta = nullptr;          // DEV [pbeta_cap] momentum coefficients of one launch
    int pbeta_cap = 0;
    std::vector<float> pbeta_host;   // staging of the same (must outlive the asynchronous copy: plan-owned)
    int64_t launches = 0;
    int device = 0;
};

namespace {

int single_channel_only(const sl1m_plan *p, const char *what) {
    if (p && p->n_chan != 1)
        return fail(SL1M_ERR_PARAM, std::string(what) + ": the plan has several channels; use the *_batch call");
    return SL1M_OK;
}

void free_plan(sl1m_plan *p) {
    if (!p) return;
    void *ptrs[] = {p->u64, p->v64, p->w64, p->ant_p, p->ant_q, p->pix4, p->pixg, p->cen, p->amp,
                    p->perm, p->vperm, p->gF, p->gA, p->ws_v, p->ws_p, p->resid, p->I_sorted, p->y_sorted,
                    p->g_sorted, p->part_a, p->part_b, p->part_c, p->scalars, p->h_x, p->h_vis, p->h_img,
                    p->trace_buf, p->chan_scale, p->step_c, p->pixd, p->pixc, p->tile_cnt, p->gFc, p->rpol, p->ctl_i,
                    p->lam2, p->pixdc, p->pixgc, p->pvis4, p->px0, p->ppart, p->pbar, p->pbeta, p->gAc, p->pybuf};
    for (void *q : ptrs)
        if (q) cudaFree(q);
    if (p->h_flag) cudaFreeHost(p->h_flag);
    for (cudaEvent_t e : p->poll_ev)
        if (e) cudaEventDestroy(e);
    delete p;
}

inline uint32_t spread16(uint32_t x) {  // interleave 16 bits with zeros
    x &= 0xffffu;
    x = (x | (x << 8)) & 0x00ff00ffu;
    x = (x | (x << 4)) & 0x0f0f0f0fu;
    x = (x | (x << 2)) & 0x33333333u;
    x = (x | (x << 1)) & 0x55555555u;
    return x;
}

template <typename T>
int upload(T **dst, const T *src, size_t n) {
    CUDA_TRY(cudaMalloc((void **)dst, std::max<size_t>(n, 1) * sizeof(T)));
    if (n) CUDA_TRY(cudaMemcpy(*dst, src, n * sizeof(T), cudaMemcpyHostToDevice));
    return SL1M_OK;
}

ApplyParams make_params(const sl1m_plan *p) {
    ApplyParams P;
    memset(&P, 0, sizeof(P));
    P.n_vis = p->n_vis_int;
    P.u64 = p->u64;
    P.v64 = p->v64;
    P.w64 = p->w64;
    P.ant_p = p->ant_p;
    P.ant_q = p->ant_q;
    P.n_pix_pad = p->n_pix_pad;
    P.n_tiles = p->n_tiles;
    P.pix4 = p->pix4;
    P.pixg = p->pixg;
    P.cen = p->cen;
    P.n_ant = p->n_ant;
    P.gF = p->gF;
    P.gA = p->gA;
    P.ws_v = p->ws_v;
    P.ws_p = p->ws_p;
    P.chan_scale = p->chan_scale;
    P.ws_v_stride = (size_t)p->fwd_split * (size_t)p->n_vis_int;
    P.ws_p_stride = (size_t)p->adj_split * (size_t)p->n_pix_pad;
    P.done = p->done_ptr;
    P.gAc = p->gAc;
#ifdef SL1M_BOUNDS
    P.gA_end = p->gA ? p->gA + (size_t)p->n_ant * (size_t)p->n_pix_pad + GAIN_ROW_PAD : nullptr;
    P.gAc_end = p->gAc ? p->gAc + (size_t)p->n_chan * (size_t)p->n_ant * (size_t)p->n_pix_pad + GAIN_ROW_PAD : nullptr;
    P.gF_end = p->gF ? p->gF + ((size_t)p->n_pix_pad + GAIN_ROW_PAD) * (size_t)p->n_ant : nullptr;
    P.gFc_end = p->gFc ? p->gFc + ((size_t)p->n_chan * p->n_pix_pad + GAIN_ROW_PAD) * (size_t)p->n_ant : nullptr;
#endif
    return P;
}

// Split count of an apply: `units` CTAs per split (visibility tiles / pixel groups) x n_chan channels, `n_items` work
// items (pixel tiles / visibility chunks) to divide among the splits, `slots` CTAs resident on the GPU at one time.
// Every CTA of an apply costs the same, so the launch takes ceil(CTAs / slots) CTA-durations: around the wanted
// number of waves, take the split count that wastes the least of the last wave (config 5: 24 forward splits = 16.09
// waves run as 17; 25 = 16.77).  A CTA with few items pays its fixed start-up cost more often: mild penalty.
int pick_split(int units, int n_items, int slots, int waves, int n_chan) {
    const double want = (double)slots * waves / std::max(1, n_chan);          // CTAs per channel
    const int s_lo = std::max(1, (int)(0.75 * want / units)), s_hi = std::max(s_lo, (int)(1.6 * want / units) + 1);
    int best = std::min(n_items, std::max(1, (int)((want + units - 1) / units)));
    double best_score = -1.0;
    for (int s0 = s_lo; s0 <= std::min(s_hi, n_items); ++s0) {
        const int per = (n_items + s0 - 1) / s0, s_eff = (n_items + per - 1) / per;
        const double w = (double)units * s_eff * n_chan / slots;
        const double eff = w / std::ceil(w - 1e-9);
        const double score = eff * per / (per + 0.25);
        if (score > best_score + 1e-12) { best_score = score; best = s_eff; }
    }
    return best;
}

// Launch configuration (enough CTAs for 148 SMs x 4 resident CTAs x several waves, shared between the
// channels of a batch) and the workspaces, all [n_chan][.].  Called at plan creation and again by
// sl1m_plan_set_channels.
int configure_and_allocate(sl1m_plan *p) {
    // ---- launch configuration: enough CTAs for 148 SMs x 4 resident CTAs x several waves ----
    // Waves of CTAs per apply: 8, or 16 when every CTA still gets several (visibility tile, pixel tile)
    // pairs -- more, shorter CTAs shrink the tail of the last wave (config 5: 317.8 -> 314.2 ms per iteration).
    const int64_t tile_pairs = (int64_t)((p->n_vis_int + NT * 8 - 1) / (NT * 8)) * p->n_tiles;
    const int waves = tile_pairs >= (int64_t)4 * 16 * SM_COUNT_B200 * 4 ? 16 : 8;
    const int target = std::max(SM_COUNT_B200 * 2, SM_COUNT_B200 * 4 * waves / p->n_chan);   // CTAs per channel
    {
        const int64_t nvi = p->n_vis_int;
        int rv = 8;
        while (rv > 1 && p->gk != 2 && (int64_t)((nvi + NT * rv - 1) / (NT * rv)) * p->n_tiles * p->n_chan < 2 * SM_COUNT_B200)
            rv >>= 1;
        if (p->phase64) rv = std::min(rv, 4);   // fp64 uvw live in registers
        p->fwd_rv = rv;
        p->fwd_vtiles = (int)((nvi + NT * rv - 1) / (NT * rv));
        // resident CTAs per SM of the forward kernel this plan launches (its __launch_bounds__)
        const int fwd_ctas = (rv == 8 || p->gk == 2) ? 4 : (p->pk == 0 && p->gk == 0 ? SL1M_FWD_MIN_CTAS : 4);
        int split = (nvi * (int64_t)p->n_tiles >= (int64_t)64 * SM_COUNT_B200)
                        ? pick_split(p->fwd_vtiles, p->n_tiles, SM_COUNT_B200 * fwd_ctas, waves, p->n_chan)
                        : std::min(p->n_tiles, std::max(1, (target + p->fwd_vtiles - 1) / p->fwd_vtiles));
        p->fwd_per_split = (p->n_tiles + split - 1) / split;
        p->fwd_split = (p->n_tiles + p->fwd_per_split - 1) / p->fwd_per_split;
    }
    {
        const int n_chunks = (p->n_vis_int + VC - 1) / VC;
        int rp = 8;
        while (rp > 1 && (int64_t)(p->n_pix_pad / (NT * rp)) * n_chunks * p->n_chan < 2 * SM_COUNT_B200) rp >>= 1;
        if (p->phase64) rp = std::min(rp, 4);
        p->adj_rp = rp;
        p->adj_pgroups = p->n_pix_pad / (NT * rp);
        const bool one_cos = rp == 8 && p->pk == 0 && p->gk == 0 && !p->phase64;
        const int adj_ctas = one_cos ? SL1M_ADJ_C1_MIN_CTAS : (rp == 8 ? 5 : (p->pk == 0 && p->gk == 0 ? SL1M_ADJ_MIN_CTAS : 4));
        int split = ((int64_t)p->adj_pgroups * n_chunks >= (int64_t)64 * SM_COUNT_B200)
                        ? pick_split(p->adj_pgroups, n_chunks, SM_COUNT_B200 * adj_ctas, waves, p->n_chan)
                        : std::min(n_chunks, std::max(1, (target + p->adj_pgroups - 1) / p->adj_pgroups));
        p->adj_per_split = (n_chunks + split - 1) / split;
        p->adj_split = (n_chunks + p->adj_per_split - 1) / p->adj_per_split;
    }

    // ---- workspaces ----
    const size_t npad = (size_t)p->n_pix_pad, C = (size_t)p->n_chan;
    for (void **q : {(void **)&p->ws_v, (void **)&p->ws_p, (void **)&p->resid, (void **)&p->I_sorted, (void **)&p->y_sorted,
                     (void **)&p->g_sorted, (void **)&p->part_a, (void **)&p->part_b, (void **)&p->part_c, (void **)&p->scalars,
                     (void **)&p->pixc, (void **)&p->tile_cnt, (void **)&p->gFc, (void **)&p->rpol, (void **)&p->pixdc,
                     (void **)&p->pixgc, (void **)&p->gAc}) {
        if (*q) cudaFree(*q);
        *q = nullptr;
    }
    CUDA_TRY(cudaMalloc((void **)&p->ws_v, C * (size_t)p->fwd_split * (size_t)p->n_vis_int * sizeof(float2)));
    CUDA_TRY(cudaMalloc((void **)&p->ws_p, C * (size_t)p->adj_split * npad * sizeof(float)));
    CUDA_TRY(cudaMalloc((void **)&p->resid, C * (size_t)p->n_vis_int * sizeof(float2)));
    CUDA_TRY(cudaMalloc((void **)&p->rpol, C * (size_t)p->n_vis_int * sizeof(float2)));
    CUDA_TRY(cudaMalloc((void **)&p->I_sorted, C * npad * sizeof(float)));
    CUDA_TRY(cudaMalloc((void **)&p->y_sorted, C * npad * sizeof(float)));
    CUDA_TRY(cudaMalloc((void **)&p->g_sorted, C * npad * sizeof(float)));
    p->n_part = (int)std::max<size_t>((npad + ET - 1) / ET, ((size_t)p->n_vis_int + ET - 1) / ET);
    CUDA_TRY(cudaMalloc((void **)&p->part_a, C * (size_t)p->n_part * sizeof(double)));
    CUDA_TRY(cudaMalloc((void **)&p->part_b, C * (size_t)p->n_part * sizeof(double)));
    CUDA_TRY(cudaMalloc((void **)&p->part_c, C * (size_t)p->n_part * sizeof(double)));
    CUDA_TRY(cudaMalloc((void **)&p->scalars, C * 4 * sizeof(double)));
    CUDA_TRY(cudaMemset(p->scalars, 0, C * 4 * sizeof(double)));
    // zero-skipping forward: every forward kernel; the kernels with a per-pixel side array in shared memory
    // (per-pixel sigma, fp64 offsets) get a compact copy of that array too.  Gain plans keep a compact copy of the
    // gain rows next to the compact tiles (n_chan x the table; not beyond 8 GiB -- such a plan keeps the dense forward).
    const size_t gfc_bytes = p->gk != 0 ? (C * npad + GAIN_ROW_PAD) * (size_t)p->n_ant * sizeof(float2) : 0;
    if (!p->dense_forward && gfc_bytes <= ((size_t)8 << 30)) {
        if (p->phase64) {   // side arrays are compacted too
            CUDA_TRY(cudaMalloc((void **)&p->pixdc, C * npad * sizeof(double4)));
            CUDA_TRY(cudaMemset(p->pixdc, 0, C * npad * sizeof(double4)));
        }
        if (p->pk == 1) {
            CUDA_TRY(cudaMalloc((void **)&p->pixgc, C * npad * sizeof(float2)));
            CUDA_TRY(cudaMemset(p->pixgc, 0, C * npad * sizeof(float2)));
        }
        CUDA_TRY(cudaMalloc((void **)&p->pixc, C * npad * sizeof(float4)));
        CUDA_TRY(cudaMalloc((void **)&p->tile_cnt, C * (size_t)p->n_tiles * sizeof(int)));
        CUDA_TRY(cudaMemset(p->pixc, 0, C * npad * sizeof(float4)));
        CUDA_TRY(cudaMemset(p->tile_cnt, 0, C * (size_t)p->n_tiles * sizeof(int)));
        if (gfc_bytes) {
            float2 **dst = (p->gk == 2 && p->pk == 0) ? &p->gAc : &p->gFc;   // packed gain forward: antenna-major
            CUDA_TRY(cudaMalloc((void **)dst, gfc_bytes));
            CUDA_TRY(cudaMemset(*dst, 0, gfc_bytes));
        }
    }
    CUDA_TRY(cudaDeviceSynchronize());

    return SL1M_OK;
}

// Small problems (delta pixels, unit gains, one channel, fp32 phase) run the FISTA loop as ONE persistent
// cooperative kernel (sl1m_persist.cuh).  "Small": below ~6.7e7 generated terms per apply the ~19 us of launch
// latency per multi-launch iteration outweighs what the tuned (packed, pipe-balanced) apply kernels gain per term.
constexpr double PERSIST_MAX_TERMS = 67108864.0;
int persist_setup(sl1m_plan *p) {
    p->persist = false;
    if (p->no_persist || p->dense_forward || p->pk != 0 || p->gk != 0 || p->phase64 || p->n_tiles > PERSIST_MAX_TILES ||
        (double)p->n_pix_pad * (double)p->n_vis_int > PERSIST_MAX_TERMS)
        return SL1M_OK;
    int coop = 0, per_sm = 0, sms = 0;
    CUDA_TRY(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, p->device));
    CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, p->device));
    CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fista_persistent_kernel, PT, 0));
    if (!coop || per_sm < 1) return SL1M_OK;
    p->persist_grid = sms;                                   // one CTA per SM
    const size_t nv = (size_t)p->n_vis_int, nt = (size_t)p->n_tiles;
    CUDA_TRY(cudaMalloc((void **)&p->pvis4, nv * sizeof(float4)));
    CUDA_TRY(cudaMalloc((void **)&p->px0, nt * nv * sizeof(float)));
    CUDA_TRY(cudaMalloc((void **)&p->ppart, 2 * 3 * (size_t)p->persist_grid * sizeof(double)));
    CUDA_TRY(cudaMalloc((void **)&p->pbar, sizeof(unsigned)));
    persist_tables_kernel<<<dim3((unsigned)((nv + 255) / 256), (unsigned)std::min<size_t>(nt, 64)), 256>>>(
        p->u64, p->v64, p->w64, p->cen, p->n_vis_int, p->n_tiles, p->pvis4, p->px0);
    p->launches++;
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaDeviceSynchronize());
    p->persist = true;
    // the smallest problems: every operand in registers, one work item per CTA and phase, the last CTA idle
    if (p->n_pix_pad <= PW * PBLK && p->n_vis_int <= 4 * PT && p->persist_grid >= 130) {
        CUDA_TRY(cudaMalloc((void **)&p->pybuf, 2 * (size_t)p->n_pix_pad * sizeof(float)));
        CUDA_TRY(cudaMemset(p->pybuf, 0, 2 * (size_t)p->n_pix_pad * sizeof(float)));
        p->persist_small = true;
    }
    return SL1M_OK;
}

}  // namespace

// ------------------------------------------------------------------------------------------
// plan creation
// ------------------------------------------------------------------------------------------
extern "C" int sl1m_plan_create(sl1m_plan **out, int64_t n_vis, const double *uvw, const int32_t *ant_p,
                                const int32_t *ant_q, int64_t n_pix, const double *l, const double *m,
                                const double *sigma, int32_t n_ant, const float *gains, int gauss_model,
                                uint32_t flags) {
    if (!out) return fail(SL1M_ERR_NULL, "out is NULL");
    *out = nullptr;
    if (!uvw || !l || !m) return fail(SL1M_ERR_NULL, "uvw, l or m is NULL");
    if (gains && (!ant_p || !ant_q)) return fail(SL1M_ERR_NULL, "gains given without ant_p/ant_q");
    if (n_vis < 1 || n_pix < 1) return fail(SL1M_ERR_SIZE, "n_vis and n_pix must be >= 1");
    if (n_vis > (int64_t)1 << 30 || n_pix > (int64_t)1 << 30) return fail(SL1M_ERR_SIZE, "size beyond 2^30");
    if (gains && n_ant < 1) return fail(SL1M_ERR_SIZE, "n_ant must be >= 1 with gains");
    if (gauss_model != SL1M_GAUSS_PARAXIAL && gauss_model != SL1M_GAUSS_WIDEFIELD)
        return fail(SL1M_ERR_PARAM, "unknown gauss_model");
    if (flags & ~(SL1M_GAINS_ON_DEVICE | SL1M_PHASE_FP64 | SL1M_DENSE_FORWARD | SL1M_NO_PERSISTENT))
        return fail(SL1M_ERR_PARAM, "unknown flag");
    for (int64_t j = 0; j < 3 * n_vis; ++j)
        if (!std::isfinite(uvw[j])) return fail(SL1M_ERR_DOMAIN, "non-finite uvw");
    bool any_gauss = false;
    for (int64_t k = 0; k < n_pix; ++k) {
        if (!std::isfinite(l[k]) || !std::isfinite(m[k])) return fail(SL1M_ERR_DOMAIN, "non-finite l/m");
        if (l[k] * l[k] + m[k] * m[k] >= 1.0) return fail(SL1M_ERR_DOMAIN, "l^2 + m^2 >= 1");
        if (sigma) {
            if (!std::isfinite(sigma[k]) || sigma[k] < 0.0) return fail(SL1M_ERR_DOMAIN, "sigma < 0 or non-finite");
            any_gauss |= sigma[k] > 0.0;
        }
    }
    if (gains)
        for (int64_t j = 0; j < n_vis; ++j)
            if (ant_p[j] < 0 || ant_p[j] >= n_ant || ant_q[j] < 0 || ant_q[j] >= n_ant)
                return fail(SL1M_ERR_INDEX, "antenna index outside [0, n_ant)");

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(SL1M_ERR_CUDA, "no CUDA device: the SL1M library has no CPU fallback");
    }

    sl1m_plan *p = new (std::nothrow) sl1m_plan();
    if (!p) return fail(SL1M_ERR_ALLOC, "host allocation failed");
    struct Guard {
        sl1m_plan *p;
        ~Guard() { if (p) free_plan(p); }
    } guard{p};
    CUDA_TRY(cudaGetDevice(&p->device));
    p->dense_forward = (flags & SL1M_DENSE_FORWARD) != 0;
    p->no_persist = (flags & SL1M_NO_PERSISTENT) != 0;
    p->n_vis = n_vis;
    p->n_pix = n_pix;
    p->n_ant = gains ? n_ant : 0;
    p->gauss = any_gauss;
    p->gains = gains != nullptr;

    try {
        // ---- Morton sort of the pixel list: consecutive runs are spatially compact ----
        double lmin = l[0], lmax = l[0], mmin = m[0], mmax = m[0];
        for (int64_t k = 1; k < n_pix; ++k) {
            lmin = std::min(lmin, l[k]); lmax = std::max(lmax, l[k]);
            mmin = std::min(mmin, m[k]); mmax = std::max(mmax, m[k]);
        }
        const double ext = std::max(std::max(lmax - lmin, mmax - mmin), 1e-300);
        std::vector<std::pair<uint32_t, int>> keys((size_t)n_pix);
        for (int64_t k = 0; k < n_pix; ++k) {
            const uint32_t ix = (uint32_t)std::min(65535.0, (l[k] - lmin) / ext * 65535.0);
            const uint32_t iy = (uint32_t)std::min(65535.0, (m[k] - mmin) / ext * 65535.0);
            keys[(size_t)k] = {spread16(ix) | (spread16(iy) << 1), (int)k};
        }
        // Gaussian plans with few distinct sigma values (multi-scale layers) are sorted by
        // sigma class first, each class padded to whole tiles: every tile then has ONE sigma, which
        // makes q = w sigma^2, 1/(1+q^2) and the exponent scale per-(visibility, tile) constants
        // instead of per-term work (kernels with PK == 2).  Otherwise plain Morton order (PK == 1).
        std::vector<double> classes;
        if (any_gauss) {
            for (int64_t k = 0; k < n_pix && classes.size() <= 16; ++k)
                if (std::find(classes.begin(), classes.end(), sigma[k]) == classes.end()) classes.push_back(sigma[k]);
            if (classes.size() > 16) classes.clear();
            std::sort(classes.begin(), classes.end());
        }
        const bool by_class = !classes.empty() && !gains;
        auto class_of = [&](int k) -> int {
            return by_class ? (int)(std::find(classes.begin(), classes.end(), sigma[k]) - classes.begin()) : 0;
        };
        std::stable_sort(keys.begin(), keys.end(),
                         [&](const std::pair<uint32_t, int> &a, const std::pair<uint32_t, int> &b) {
                             const int ca = class_of(a.second), cb = class_of(b.second);
                             return ca != cb ? ca < cb : a.first < b.first;
                         });
        // slots: sorted position -> caller pixel, -1 on padding (class boundaries and the tail)
        std::vector<int> slots;
        slots.reserve((size_t)n_pix + (classes.size() + 1) * TP + PIX_PAD);
        for (size_t i = 0; i < keys.size(); ++i) {
            if (by_class && i > 0 && class_of(keys[i].second) != class_of(keys[i - 1].second))
                while (slots.size() % TP) slots.push_back(-1);
            slots.push_back(keys[i].second);
        }
        while (slots.size() % PIX_PAD) slots.push_back(-1);
        if (slots.size() > ((size_t)1 << 30)) return fail(SL1M_ERR_SIZE, "padded pixel count beyond 2^30");
        p->n_pix_pad = (int)slots.size();
        p->n_tiles = p->n_pix_pad / TP;
        p->pk = any_gauss ? (by_class ? 2 : 1) : 0;

        // ---- per-tile fp64 centres, per-pixel fp32 offsets (step a0) ----
        const size_t npad = (size_t)p->n_pix_pad;
        std::vector<float4> pix4(npad, make_float4(0.f, 0.f, 0.f, 0.f));
        std::vector<float2> pixg(any_gauss ? npad : 0, make_float2(0.f, 0.f));
        std::vector<double4> cen((size_t)p->n_tiles, make_double4(0.0, 0.0, 0.0, 0.0));
        std::vector<float> amp(npad, 0.f);
        std::vector<int> perm(npad, -1);
        std::vector<double4> pixd(npad, make_double4(0.0, 0.0, 0.0, 0.0));
        double umax = 0.0, vmax = 0.0, wmax = 0.0, span = 0.0;
        for (int64_t j = 0; j < n_vis; ++j) {
            umax = std::max(umax, std::fabs(uvw[3 * j]));
            vmax = std::max(vmax, std::fabs(uvw[3 * j + 1]));
            wmax = std::max(wmax, std::fabs(uvw[3 * j + 2]));
        }
        const double PI = 3.14159265358979323846, LOG2E = 1.4426950408889634074;
        for (int t = 0; t < p->n_tiles; ++t) {
            const size_t k0 = (size_t)t * TP, k1 = k0 + TP;
            double a0 = 1e300, a1 = -1e300, b0 = 1e300, b1 = -1e300, sig_tile = 0.0;
            for (size_t s = k0; s < k1; ++s) {
                const int k = slots[s];
                if (k < 0) continue;
                a0 = std::min(a0, l[k]); a1 = std::max(a1, l[k]);
                b0 = std::min(b0, m[k]); b1 = std::max(b1, m[k]);
                if (sigma) sig_tile = sigma[k];
            }
            if (a0 > a1) continue;   // a tile of padding only
            const double lc = 0.5 * (a0 + a1), mc = 0.5 * (b0 + b1);
            const double rc2 = lc * lc + mc * mc;
            const double nc = -rc2 / (1.0 + std::sqrt(1.0 - rc2));   // n - 1 at the centre
            cen[(size_t)t] = make_double4(lc, mc, nc, sig_tile * sig_tile);   // .w = sigma^2 of the tile (PK == 2)
            for (size_t s = k0; s < k1; ++s) {
                const int k = slots[s];
                if (k < 0) continue;
                const double r2 = l[k] * l[k] + m[k] * m[k];
                const double n = std::sqrt(1.0 - r2);
                const double sg = sigma ? sigma[k] : 0.0;
                // eq (9)/(17): n' = n - 1 (cancellation-free); eq (16): n' = -r^2/2; sigma == 0 => eq (9)
                const double npr = (sg > 0.0 && gauss_model == SL1M_GAUSS_PARAXIAL) ? -0.5 * r2
                                                                                     : -r2 / (1.0 + n);
                pix4[s] = make_float4((float)(l[k] - lc), (float)(m[k] - mc), (float)(npr - nc), 0.f);
                pixd[s] = make_double4(l[k] - lc, m[k] - mc, npr - nc, 0.0);
                span = std::max(span, 2.0 * PI * (umax * std::fabs(l[k] - lc) + vmax * std::fabs(m[k] - mc) +
                                                  wmax * std::fabs(npr - nc)));
                amp[s] = (float)(1.0 / n);
                perm[s] = k;
                if (any_gauss) pixg[s] = make_float2((float)(sg * sg), (float)(-PI * LOG2E * sg * sg));
            }
        }

        // ---- visibilities: SoA fp64 in the INTERNAL order ----
        // With gains, visibilities are grouped by baseline (p, q) into groups of 8 samples (padded):
        // the gain product g_p conj(g_q) of a group is then loaded once per pixel instead of once
        // per term.  Sample r of group g sits at (g / 128) * 1024 + r * 128 + g % 128, which is the
        // forward kernel's thread layout.  Used when the groups are at least 34 % full on average: measured at
        // config 4, a grouped apply costs the same whatever its fill (8.2 + 5.0 ms per forward + adjoint for 8 slots)
        // and the per-term kernels run at 0.52 / 1.4e12 terms/s, so 3 samples per baseline are still 1.3x faster
        // grouped (13.2 against 17.2 ms) and 5 samples 2.1x; below that, per-term gains.
        std::vector<int> vperm;
        std::vector<int> ip, iq;
        p->n_vis_int = (int)n_vis;
        p->gk = gains ? 1 : 0;
        if (gains) {
            std::vector<int> order((size_t)n_vis);
            for (int64_t j = 0; j < n_vis; ++j) order[(size_t)j] = (int)j;
            std::stable_sort(order.begin(), order.end(), [&](int a, int b) {
                return ant_p[a] != ant_p[b] ? ant_p[a] < ant_p[b] : ant_q[a] < ant_q[b];
            });
            int64_t n_groups = 0;
            for (int64_t s0 = 0; s0 < n_vis;) {
                int64_t s1 = s0;
                while (s1 < n_vis && ant_p[order[(size_t)s1]] == ant_p[order[(size_t)s0]] &&
                       ant_q[order[(size_t)s1]] == ant_q[order[(size_t)s0]]) ++s1;
                n_groups += (s1 - s0 + 7) / 8;
                s0 = s1;
            }
            const int64_t n_groups_pad = ((n_groups + NT - 1) / NT) * NT;
            if ((double)n_vis >= 0.34 * (double)(n_groups * 8) && n_groups_pad * 8 < ((int64_t)1 << 30)) {
                p->gk = 2;
                p->n_vis_int = (int)(n_groups_pad * 8);
                vperm.assign((size_t)p->n_vis_int, -1);
                ip.assign((size_t)p->n_vis_int, 0);
                iq.assign((size_t)p->n_vis_int, 0);
                int64_t g = 0;
                for (int64_t s0 = 0; s0 < n_vis;) {
                    int64_t s1 = s0;
                    while (s1 < n_vis && ant_p[order[(size_t)s1]] == ant_p[order[(size_t)s0]] &&
                           ant_q[order[(size_t)s1]] == ant_q[order[(size_t)s0]]) ++s1;
                    for (int64_t b = s0; b < s1; b += 8, ++g) {
                        for (int r = 0; r < 8; ++r) {
                            const size_t pos = (size_t)((g / NT) * (NT * 8) + r * NT + g % NT);
                            ip[pos] = ant_p[order[(size_t)s0]];
                            iq[pos] = ant_q[order[(size_t)s0]];
                            if (b + r < s1) vperm[pos] = order[(size_t)(b + r)];
                        }
                    }
                    s0 = s1;
                }
            } else {
                // Per-term gains (baselines with too few samples to group): still ORDER the visibilities by antenna
                // pair.  A warp's 32 consecutive visibilities then share p and have consecutive q, so its two gain
                // loads per term hit one 8-byte word (broadcast) and one contiguous 256-byte run of the pixel's gain
                // row instead of 32 scattered words; in the adjoint consecutive staged visibilities reuse the
                // antenna-p row from L1.
                vperm.assign(order.begin(), order.end());
                ip.resize((size_t)n_vis);
                iq.resize((size_t)n_vis);
                for (int64_t js = 0; js < n_vis; ++js) {
                    ip[(size_t)js] = ant_p[order[(size_t)js]];
                    iq[(size_t)js] = ant_q[order[(size_t)js]];
                }
            }
        }
        const size_t nvi = (size_t)p->n_vis_int;
        std::vector<double> su(nvi, 0.0), sv(nvi, 0.0), sw(nvi, 0.0);
        for (size_t js = 0; js < nvi; ++js) {
            const int64_t j = vperm.empty() ? (int64_t)js : vperm[js];
            if (j < 0) continue;
            su[js] = uvw[3 * j];
            sv[js] = uvw[3 * j + 1];
            sw[js] = uvw[3 * j + 2];
        }

        int st;
        if ((st = upload(&p->u64, su.data(), su.size()))) return st;
        if ((st = upload(&p->v64, sv.data(), sv.size()))) return st;
        if ((st = upload(&p->w64, sw.data(), sw.size()))) return st;
        if ((st = upload(&p->pix4, pix4.data(), npad))) return st;
        if (any_gauss && (st = upload(&p->pixg, pixg.data(), npad))) return st;
        if ((st = upload(&p->cen, cen.data(), cen.size()))) return st;
        if ((st = upload(&p->amp, amp.data(), npad))) return st;
        if ((st = upload(&p->perm, perm.data(), npad))) return st;
        // fp64-phase kernels: on request, or when the fp32 remainder could exceed ~256 rad (sin.approx
        // loses 4e-5 there, profiles/r1_microbench.md); delta pixels with unit gains only.
        p->phase_span = span;
        p->phase64_capable = !any_gauss && !gains;
        p->phase64_flag = (flags & SL1M_PHASE_FP64) != 0;
        p->phase64 = p->phase64_capable && (p->phase64_flag || span > 256.0);
        // kept for every plan that could need it: sl1m_plan_set_channels may switch to the fp64-phase kernels
        if (p->phase64_capable && (st = upload(&p->pixd, pixd.data(), npad))) return st;
        if (gains) {
            if ((st = upload(&p->ant_p, vperm.empty() ? ant_p : ip.data(), nvi))) return st;
            if ((st = upload(&p->ant_q, vperm.empty() ? ant_q : iq.data(), nvi))) return st;
            if (!vperm.empty() && (st = upload(&p->vperm, vperm.data(), nvi))) return st;
        }
    } catch (const std::bad_alloc &) {
        return fail(SL1M_ERR_ALLOC, "host allocation failed");
    }

    // ---- gains: re-layout on the device ----
    if (gains) {
        const size_t raw_n = (size_t)n_ant * (size_t)n_pix;
        float2 *raw = nullptr;
        if (flags & SL1M_GAINS_ON_DEVICE) {
            raw = (float2 *)gains;
        } else {
            CUDA_TRY(cudaMalloc((void **)&raw, raw_n * sizeof(float2)));
            cudaError_t e = cudaMemcpy(raw, gains, raw_n * sizeof(float2), cudaMemcpyHostToDevice);
            if (e != cudaSuccess) { cudaFree(raw); return fail(SL1M_ERR_CUDA, cudaGetErrorString(e)); }
        }
        const size_t lay_n = (size_t)p->n_pix_pad * (size_t)n_ant;
        // gF (pixel-major) serves the scalar forward kernels and carries GAIN_ROW_PAD rows of zero padding (they
        // prefetch rows ahead); the packed gain forward (gk == 2, delta pixels) reads the antenna-major gA instead,
        // which then carries GAIN_ROW_PAD entries of padding, and gF is not built at all.
        const bool fwd_reads_gA = p->gk == 2 && !any_gauss;
        cudaError_t e1 = cudaSuccess;
        if (!fwd_reads_gA) {
            e1 = cudaMalloc((void **)&p->gF, (lay_n + (size_t)GAIN_ROW_PAD * n_ant) * sizeof(float2));
            if (e1 == cudaSuccess) e1 = cudaMemset(p->gF + lay_n, 0, (size_t)GAIN_ROW_PAD * n_ant * sizeof(float2));
        }
        cudaError_t e2 = (e1 == cudaSuccess) ? cudaMalloc((void **)&p->gA, (lay_n + GAIN_ROW_PAD) * sizeof(float2)) : e1;
        if (e2 == cudaSuccess) e2 = cudaMemset(p->gA + lay_n, 0, GAIN_ROW_PAD * sizeof(float2));
        if (e2 == cudaSuccess) {
            // antennas are looped inside the kernel (grid.y would cap n_ant at 65,535; "each (antenna, time)
            // its own row" can exceed that)
            gains_layout_kernel<<<(p->n_pix_pad + ET - 1) / ET, ET>>>(raw, n_ant, (int)n_pix, p->n_pix_pad, p->perm, p->gF, p->gA);
            e2 = cudaGetLastError();
            if (e2 == cudaSuccess) e2 = cudaDeviceSynchronize();
            p->launches++;
        }
        if (!(flags & SL1M_GAINS_ON_DEVICE)) cudaFree(raw);
        if (e2 != cudaSuccess)
            return fail(e2 == cudaErrorMemoryAllocation ? SL1M_ERR_ALLOC : SL1M_ERR_CUDA, cudaGetErrorString(e2));
    }

    {
        int st2 = configure_and_allocate(p);
        if (st2) return st2;
        if ((st2 = persist_setup(p))) return st2;
    }

    guard.p = nullptr;
    *out = p;
    return SL1M_OK;
}

// ------------------------------------------------------------------------------------------
// launches
// ------------------------------------------------------------------------------------------
namespace {

inline int egrid(size_t n) { return (int)((n + ET - 1) / ET); }
inline dim3 cgrid(const sl1m_plan *p, size_t n) { return dim3((unsigned)egrid(n), (unsigned)p->n_chan); }  // x: elements, y: channel
inline ZeroSkip zs_of(const sl1m_plan *p) {
    return ZeroSkip{p->pixc, p->tile_cnt, p->gF, p->gFc, p->n_ant, p->pixd, p->pixdc, p->pixg, p->pixgc, p->gA, p->gAc};
}

template <int PK, int GK, bool B>
void launch_fwd_rv(const sl1m_plan *p, const ApplyParams &P, dim3 grid, cudaStream_t s) {
    if constexpr (GK == 2) {
        if constexpr (PK == 0) fwd_kernel_x2<SL1M_FWD_G2_NPQ, B, true><<<grid, NT, 0, s>>>(P);
        else fwd_kernel<8, PK, 2, B><<<grid, NT, 0, s>>>(P);
    } else {
        switch (p->fwd_rv) {
            case 8:
                if constexpr (PK == 0 && GK == 0) fwd_kernel_x2<SL1M_FWD_NPQ, B><<<grid, NT, 0, s>>>(P);
                else if constexpr (PK == 2 && GK == 0) fwd_kernel_gtx2<B><<<grid, NT, 0, s>>>(P);
                else fwd_kernel<8, PK, GK, B><<<grid, NT, 0, s>>>(P);
                break;
            case 4: fwd_kernel<4, PK, GK, B><<<grid, NT, 0, s>>>(P); break;
            case 2: fwd_kernel<2, PK, GK, B><<<grid, NT, 0, s>>>(P); break;
            default: fwd_kernel<1, PK, GK, B><<<grid, NT, 0, s>>>(P); break;
        }
    }
}

template <int PK, int GK, bool B>
void launch_adj_rp(const sl1m_plan *p, const ApplyParams &P, dim3 grid, cudaStream_t s) {
    switch (p->adj_rp) {
        case 8:
            if constexpr (PK == 0 && GK == 0) {
                ApplyParams Q = P;      // one cosine per term: the kernel reads the residual in polar form
                vis_polar_kernel<<<dim3((unsigned)egrid((size_t)p->n_vis_int), (unsigned)p->n_chan), ET, 0, s>>>(P.r, p->rpol, p->n_vis_int, p->done_ptr);
                Q.r = p->rpol;
                adj_kernel_c1<SL1M_ADJ_C1_NPQ, B><<<grid, NT, 0, s>>>(Q);
            }
            else if constexpr (PK == 0 && GK == 2) adj_kernel_g2x2<SL1M_ADJ_G2_NPQ, B><<<grid, NT, 0, s>>>(P);
            else if constexpr (PK == 2 && GK == 0) adj_kernel_gtx2<B><<<grid, NT, 0, s>>>(P);
            else adj_kernel<8, PK, GK, B><<<grid, NT, 0, s>>>(P);
            break;
        case 4: adj_kernel<4, PK, GK, B><<<grid, NT, 0, s>>>(P); break;
        case 2: adj_kernel<2, PK, GK, B><<<grid, NT, 0, s>>>(P); break;
        default: adj_kernel<1, PK, GK, B><<<grid, NT, 0, s>>>(P); break;
    }
}

// BATCH instantiations (blockIdx.z = channel, per-channel uvw scale) only when the plan has channels.
template <int PK, int GK>
void launch_fwd_rv(const sl1m_plan *p, const ApplyParams &P, dim3 grid, cudaStream_t s) {
    if (p->chan_scale) launch_fwd_rv<PK, GK, true>(p, P, grid, s);
    else launch_fwd_rv<PK, GK, false>(p, P, grid, s);
}
template <int PK, int GK>
void launch_adj_rp(const sl1m_plan *p, const ApplyParams &P, dim3 grid, cudaStream_t s) {
    if (p->chan_scale) launch_adj_rp<PK, GK, true>(p, P, grid, s);
    else launch_adj_rp<PK, GK, false>(p, P, grid, s);
}

// forward main kernel: pix4.w must already hold a*x in sorted order; fills ws_v.
void launch_fwd(sl1m_plan *p, cudaStream_t s) {
    ApplyParams P = make_params(p);
    P.per_split = p->fwd_per_split;
    dim3 grid(p->fwd_vtiles, p->fwd_split, p->n_chan);
    if (p->pixc) {   // zero-skipping: stream the compact tiles the packing kernel left behind
        P.pix4 = p->pixc;
        P.tile_cnt = p->tile_cnt;
        P.gFc = p->gFc;
        if (p->pixgc) P.pixg = p->pixgc;
    }
    if (p->phase64) {
        const double4 *pd = p->pixc ? p->pixdc : p->pixd;
        switch (p->fwd_rv) {
            case 4: fwd_kernel_p64<4><<<grid, NT, 0, s>>>(P, pd); break;
            case 2: fwd_kernel_p64<2><<<grid, NT, 0, s>>>(P, pd); break;
            default: fwd_kernel_p64<1><<<grid, NT, 0, s>>>(P, pd); break;
        }
        p->launches++;
        return;
    }
    const int key = p->pk * 3 + p->gk;   // pk == 2 (one sigma per tile) only exists with unit gains
    switch (key) {
        case 6: launch_fwd_rv<2, 0>(p, P, grid, s); break;
        case 0: launch_fwd_rv<0, 0>(p, P, grid, s); break;
        case 1: launch_fwd_rv<0, 1>(p, P, grid, s); break;
        case 2: launch_fwd_rv<0, 2>(p, P, grid, s); break;
        case 3: launch_fwd_rv<1, 0>(p, P, grid, s); break;
        case 4: launch_fwd_rv<1, 1>(p, P, grid, s); break;
        default: launch_fwd_rv<1, 2>(p, P, grid, s); break;
    }
    p->launches++;
}

// adjoint main kernel on residual r (device, INTERNAL order [n_vis_int]); fills ws_p.
void launch_adj(sl1m_plan *p, const float2 *r, cudaStream_t s) {
    ApplyParams P = make_params(p);
    P.per_split = p->adj_per_split;
    P.r = r;
    dim3 grid(p->adj_pgroups, p->adj_split, p->n_chan);
    if (p->phase64) {
        // one cosine per term here too: the kernel reads the residual in polar form
        vis_polar_kernel<<<dim3((unsigned)egrid((size_t)p->n_vis_int), (unsigned)p->n_chan), ET, 0, s>>>(P.r, p->rpol, p->n_vis_int, p->done_ptr);
        P.r = p->rpol;
        p->launches++;
        switch (p->adj_rp) {
            case 4: adj_kernel_p64<4><<<grid, NT, 0, s>>>(P, p->pixd); break;
            case 2: adj_kernel_p64<2><<<grid, NT, 0, s>>>(P, p->pixd); break;
            default: adj_kernel_p64<1><<<grid, NT, 0, s>>>(P, p->pixd); break;
        }
        p->launches++;
        return;
    }
    const int key = p->pk * 3 + p->gk;
    switch (key) {
        case 6: launch_adj_rp<2, 0>(p, P, grid, s); break;
        case 0: launch_adj_rp<0, 0>(p, P, grid, s); break;
        case 1: launch_adj_rp<0, 1>(p, P, grid, s); break;
        case 2: launch_adj_rp<0, 2>(p, P, grid, s); break;
        case 3: launch_adj_rp<1, 0>(p, P, grid, s); break;
        case 4: launch_adj_rp<1, 1>(p, P, grid, s); break;
        default: launch_adj_rp<1, 2>(p, P, grid, s); break;
    }
    p->launches++;
    if (key == 0 && p->adj_rp == 8) p->launches++;   // vis_polar_kernel in front of the one-cosine kernel
}

int check_launch(const char *what) {
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(SL1M_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
    return SL1M_OK;
}

}  // namespace

extern "C" int sl1m_forward(sl1m_plan *p, const float *x_dev, float *vis_dev, void *stream) {
    if (!p || !x_dev || !vis_dev) return fail(SL1M_ERR_NULL, "sl1m_forward: NULL argument");
    cudaStream_t s = (cudaStream_t)stream;
    pack_caller_kernel<<<cgrid(p, p->n_pix_pad), ET, 0, s>>>(p->pix4, p->amp, p->perm, x_dev, p->n_pix_pad, (int)p->n_pix, zs_of(p));
    launch_fwd(p, s);
    fwd_reduce_kernel<<<cgrid(p, p->n_vis_int), ET, 0, s>>>(p->ws_v, p->fwd_split, p->n_vis_int, p->vperm, nullptr,
                                                            (float2 *)vis_dev, 0, nullptr, (int)p->n_vis, p->n_part);
    p->launches += 2;
    if (p->f_active) {
        // A stepped FISTA run is open and its next iteration reads a*y_{k+1} from the pixel tiles, which now hold the
        // caller's a*x: put them back from y_sorted (every solver path keeps it current), so that
        // begin / step / forward(I_k) / step continues the same run.
        pack_sorted_kernel<<<cgrid(p, p->n_pix_pad), ET, 0, s>>>(p->pix4, p->amp, p->y_sorted, p->n_pix_pad, zs_of(p));
        p->launches++;
    }
    return check_launch("sl1m_forward");
}

extern "C" int sl1m_adjoint(sl1m_plan *p, const float *r_dev, float *img_dev, void *stream) {
    if (!p || !r_dev || !img_dev) return fail(SL1M_ERR_NULL, "sl1m_adjoint: NULL argument");
    cudaStream_t s = (cudaStream_t)stream;
    const float2 *r_int = (const float2 *)r_dev;
    if (p->vperm) {
        vis_gather_kernel<<<cgrid(p, p->n_vis_int), ET, 0, s>>>((const float2 *)r_dev, p->vperm, p->resid, p->n_vis_int,
                                                                (int)p->n_vis);
        p->launches++;
        r_int = p->resid;
    }
    launch_adj(p, r_int, s);
    adj_reduce_kernel<<<cgrid(p, p->n_pix_pad), ET, 0, s>>>(p->ws_p, p->adj_split, p->n_pix_pad, p->amp, p->perm,
                                                            img_dev, nullptr, nullptr, (int)p->n_pix, p->n_part);
    p->launches += 1;
    return check_launch("sl1m_adjoint");
}

namespace {
int ensure_host_staging(sl1m_plan *p) {
    if (!p->h_x) CUDA_TRY(cudaMalloc((void **)&p->h_x, (size_t)p->n_pix * sizeof(float)));
    if (!p->h_img) CUDA_TRY(cudaMalloc((void **)&p->h_img, (size_t)p->n_pix * sizeof(float)));
    if (!p->h_vis) CUDA_TRY(cudaMalloc((void **)&p->h_vis, (size_t)p->n_vis * sizeof(float2)));
    return SL1M_OK;
}
}  // namespace

extern "C" int sl1m_forward_host(sl1m_plan *p, const float *x_host, float *vis_host, void *stream) {
    if (!p || !x_host || !vis_host) return fail(SL1M_ERR_NULL, "sl1m_forward_host: NULL argument");
    if (int stc = single_channel_only(p, "sl1m_forward_host")) return stc;
    cudaStream_t s = (cudaStream_t)stream;
    int st = ensure_host_staging(p);
    if (st) return st;
    CUDA_TRY(cudaMemcpyAsync(p->h_x, x_host, (size_t)p->n_pix * sizeof(float), cudaMemcpyHostToDevice, s));
    if ((st = sl1m_forward(p, p->h_x, p->h_vis, stream))) return st;
    CUDA_TRY(cudaMemcpyAsync(vis_host, p->h_vis, (size_t)p->n_vis * sizeof(float2), cudaMemcpyDeviceToHost, s));
    CUDA_TRY(cudaStreamSynchronize(s));
    return SL1M_OK;
}

extern "C" int sl1m_adjoint_host(sl1m_plan *p, const float *r_host, float *img_host, void *stream) {
    if (!p || !r_host || !img_host) return fail(SL1M_ERR_NULL, "sl1m_adjoint_host: NULL argument");
    if (int stc = single_channel_only(p, "sl1m_adjoint_host")) return stc;
    cudaStream_t s = (cudaStream_t)stream;
    int st = ensure_host_staging(p);
    if (st) return st;
    CUDA_TRY(cudaMemcpyAsync(p->h_vis, r_host, (size_t)p->n_vis * sizeof(float2), cudaMemcpyHostToDevice, s));
    if ((st = sl1m_adjoint(p, p->h_vis, p->h_img, stream))) return st;
    CUDA_TRY(cudaMemcpyAsync(img_host, p->h_img, (size_t)p->n_pix * sizeof(float), cudaMemcpyDeviceToHost, s));
    CUDA_TRY(cudaStreamSynchronize(s));
    return SL1M_OK;
}

// ------------------------------------------------------------------------------------------
// a7: power iteration, entirely on the device; one synchronise at the end
// ------------------------------------------------------------------------------------------
namespace {
// L_out_host: HOST [n_chan]
int max_eig_impl(sl1m_plan *p, int n_pow, float *L_out_host, void *stream) {
    if (!p || !L_out_host) return fail(SL1M_ERR_NULL, "sl1m_max_eig: NULL argument");
    if (n_pow < 1) return fail(SL1M_ERR_PARAM, "n_pow must be >= 1");
    cudaStream_t s = (cudaStream_t)stream;
    const int npad = p->n_pix_pad;
    p->f_active = false;                 // the pixel tiles are about to hold the power iteration's vectors
    // x0 = 1/sqrt(n_pix) on real pixels
    fill_kernel<<<cgrid(p, npad), ET, 0, s>>>(p->g_sorted, (float)(1.0 / std::sqrt((double)p->n_pix)), p->perm, npad);
    pack_sorted_kernel<<<cgrid(p, npad), ET, 0, s>>>(p->pix4, p->amp, p->g_sorted, npad, zs_of(p));
    p->launches += 2;
    if (p->persist && !p->chan_scale) {   // small problem: all rounds in one cooperative launch (sl1m_persist.cuh)
        PersistParams P;
        memset(&P, 0, sizeof(P));
        const int G = p->persist_grid;
        P.n_vis = p->n_vis_int;
        P.n_pix_pad = npad;
        P.n_tiles = p->n_tiles;
        P.nvg = std::max(1, std::min(PG, (p->n_vis_int + G - 1) / G));
        int npg = 1;
        while (npg < PG && npad / npg > G) npg <<= 1;
        P.npg = npg;
        P.vis4 = p->pvis4;
        P.x0 = p->px0;
        P.pix4 = p->pix4;
        P.amp = p->amp;
        P.rpol = p->rpol;
        P.part = p->ppart;
        P.bar = p->pbar;
        P.n_iter = n_pow;
        double *out = p->scalars;
        CUDA_TRY(cudaMemsetAsync(p->pbar, 0, sizeof(unsigned), s));
        void *args[] = {(void *)&P, (void *)&out};
        const cudaError_t le = cudaLaunchCooperativeKernel((const void *)power_persistent_kernel, dim3((unsigned)G), dim3(PT), args, 0, s);
        if (le == cudaSuccess) {
            p->launches++;
            int st = check_launch("sl1m_max_eig(persistent)");
            if (st) return st;
            double h = 0.0;
            CUDA_TRY(cudaMemcpyAsync(&h, p->scalars, sizeof(double), cudaMemcpyDeviceToHost, s));
            CUDA_TRY(cudaStreamSynchronize(s));
            L_out_host[0] = (float)std::sqrt(h);
            return SL1M_OK;
        }
        if (le != cudaErrorCooperativeLaunchTooLarge && le != cudaErrorLaunchOutOfResources) CUDA_TRY(le);
        cudaGetLastError();               // not co-resident right now: the multi-launch rounds below
    }
    for (int it = 0; it < n_pow; ++it) {
        launch_fwd(p, s);
        fwd_reduce_kernel<<<cgrid(p, p->n_vis_int), ET, 0, s>>>(p->ws_v, p->fwd_split, p->n_vis_int, p->vperm, nullptr,
                                                                p->resid, 1, nullptr, (int)p->n_vis, p->n_part);
        launch_adj(p, p->resid, s);
        adj_reduce_kernel<<<cgrid(p, npad), ET, 0, s>>>(p->ws_p, p->adj_split, npad, p->amp, p->perm, nullptr,
                                                        p->g_sorted, p->part_a, (int)p->n_pix, p->n_part);
        sum_partials_kernel<<<p->n_chan, ET, 0, s>>>(p->part_a, nullptr, nullptr, egrid(npad), 0, 0, p->scalars, nullptr,
                                                     nullptr, p->n_part, 4);
        normalize_pack_kernel<<<cgrid(p, npad), ET, 0, s>>>(p->g_sorted, p->scalars, p->amp, p->pix4, npad, zs_of(p));
        p->launches += 4;
    }
    int st = check_launch("sl1m_max_eig");
    if (st) return st;
    std::vector<double> h(4 * (size_t)p->n_chan);
    CUDA_TRY(cudaMemcpyAsync(h.data(), p->scalars, h.size() * sizeof(double), cudaMemcpyDeviceToHost, s));
    CUDA_TRY(cudaStreamSynchronize(s));
    for (int c = 0; c < p->n_chan; ++c) L_out_host[c] = (float)std::sqrt(h[4 * (size_t)c]);
    return SL1M_OK;
}
}  // namespace

extern "C" int sl1m_max_eig(sl1m_plan *p, int n_pow, float *L_out_host, void *stream) {
    if (int st = single_channel_only(p, "sl1m_max_eig")) return st;
    return max_eig_impl(p, n_pow, L_out_host, stream);
}

extern "C" int sl1m_max_eig_batch(sl1m_plan *p, int n_pow, float *L_out_host, void *stream) {
    return max_eig_impl(p, n_pow, L_out_host, stream);
}

// ------------------------------------------------------------------------------------------
// a3-a6: FISTA, listing PAPER.md:188-192; no host round-trip per iteration
// ------------------------------------------------------------------------------------------
namespace {
struct StopOpts {
    double tol, nnz_tol;   // < 0: that rule is off
    int check_every;
};

// y_1 = I_0 = x0 (or 0), t_1 = 1.  lambda_c, L_c: HOST [n_chan], L_c > 0.  vis_dev is BORROWED until the next begin.
int fista_begin_impl(sl1m_plan *p, const float *vis_dev, const float *lambda_c, const float *L_c, const float *x0_dev,
                     cudaStream_t s) {
    const int C = p->n_chan, npad = p->n_pix_pad;
    p->f_active = false;
    p->f_lam.assign(lambda_c, lambda_c + C);
    p->f_L.assign(L_c, L_c + C);
    p->f_inv_L = (float)(1.0 / (double)L_c[0]);
    p->f_thr = (float)((double)lambda_c[0] / (double)L_c[0]);
    {   // per-channel (1/L_c, lambda_c/L_c) and 2 lambda_c on the device
        std::vector<float2> h((size_t)C);
        std::vector<double> l2((size_t)C);
        for (int c = 0; c < C; ++c) {
            h[c] = make_float2((float)(1.0 / (double)L_c[c]), (float)((double)lambda_c[c] / (double)L_c[c]));
            l2[c] = 2.0 * (double)lambda_c[c];
        }
        if (!p->lam2) CUDA_TRY(cudaMalloc((void **)&p->lam2, (size_t)C * sizeof(double)));
        if (!p->ctl_i) CUDA_TRY(cudaMalloc((void **)&p->ctl_i, (2 * (size_t)C + 1) * sizeof(int)));
        CUDA_TRY(cudaMemcpyAsync(p->lam2, l2.data(), (size_t)C * sizeof(double), cudaMemcpyHostToDevice, s));
        if (C > 1) CUDA_TRY(cudaMemcpyAsync(p->step_c, h.data(), (size_t)C * sizeof(float2), cudaMemcpyHostToDevice, s));
        CUDA_TRY(cudaMemsetAsync(p->ctl_i, 0, (2 * (size_t)C + 1) * sizeof(int), s));
        CUDA_TRY(cudaStreamSynchronize(s));   // h, l2 are stack-lifetime staging buffers
    }
    if (x0_dev) {
        gather_kernel<<<cgrid(p, npad), ET, 0, s>>>(x0_dev, p->perm, p->I_sorted, npad, (int)p->n_pix);
        p->launches++;
    } else {
        CUDA_TRY(cudaMemsetAsync(p->I_sorted, 0, (size_t)C * npad * sizeof(float), s));
    }
    CUDA_TRY(cudaMemcpyAsync(p->y_sorted, p->I_sorted, (size_t)C * npad * sizeof(float), cudaMemcpyDeviceToDevice, s));
    pack_sorted_kernel<<<cgrid(p, npad), ET, 0, s>>>(p->pix4, p->amp, p->y_sorted, npad, zs_of(p));
    p->launches++;
    p->f_vis = (const float2 *)vis_dev;
    p->f_t = 1.0;
    p->f_k = 0;
    p->done_ptr = nullptr;
    p->f_active = true;
    return check_launch("sl1m_fista_begin");
}

// n_iter more iterations of the listing from the plan's state (I_k, y_{k+1}, t_{k+1}).  trace_dev (nullable):
// DEV [n_chan][trace_stride doubles]; iteration i of THIS call writes row trace_row0 + i.  stop (nullable): the
// termination rules, decided on the device (stop_rule_kernel) from trace rows k-1, k-2 counted from the state's
// begin -- the caller's trace must then hold every iteration since begin (trace_row0 == p->f_k).
// The host never waits for an iteration: it reads the all-done flag two polls behind what it has enqueued.
// The same iterations as ONE launch of the persistent kernel (small single-channel problems).
int persist_iterate(sl1m_plan *p, int n_iter, double *trace_rows, const StopOpts *stop, cudaStream_t s) {
    if (n_iter < 1) return SL1M_OK;
    PersistParams P;
    memset(&P, 0, sizeof(P));
    const int G = p->persist_grid;
    P.n_vis = p->n_vis_int;
    P.n_pix_pad = p->n_pix_pad;
    P.n_tiles = p->n_tiles;
    P.nvg = std::max(1, std::min(PG, (p->n_vis_int + G - 1) / G));
    int npg = 1;
    while (npg < PG && p->n_pix_pad / npg > G) npg <<= 1;    // power of two: an item never straddles a tile
    P.npg = npg;
    P.vis4 = p->pvis4;
    P.x0 = p->px0;
    P.pix4 = p->pix4;
    P.amp = p->amp;
    P.I_sorted = p->I_sorted;
    P.y_sorted = p->y_sorted;
    P.V = p->f_vis;
    P.rpol = p->rpol;
    P.part = p->ppart;
    P.bar = p->pbar;
    P.trace = trace_rows;
    P.ctl = stop ? p->ctl_i : nullptr;
    P.inv_L = p->f_inv_L;
    P.thr = p->f_thr;
    P.lam2 = 2.0 * (double)p->f_lam[0];
    P.tol = stop ? stop->tol : -1.0;
    P.nnz_tol = stop ? stop->nnz_tol : -1.0;
    P.check_every = stop ? stop->check_every : 0;
    P.k0 = p->f_k;
    P.n_iter = n_iter;
    const double t_before = p->f_t;
    {   // momentum coefficients of this launch's iterations, fp64 on the host as in the multi-launch loop
        if (p->pbeta_cap < n_iter) {
            if (p->pbeta) cudaFree(p->pbeta);
            p->pbeta = nullptr;
            p->pbeta_cap = 0;
            CUDA_TRY(cudaMalloc((void **)&p->pbeta, (size_t)n_iter * sizeof(float)));
            p->pbeta_cap = n_iter;
        }
        p->pbeta_host.resize((size_t)n_iter);
        double t = p->f_t;
        for (int i = 0; i < n_iter; ++i) {
            const double t_next = 0.5 * (1.0 + std::sqrt(1.0 + 4.0 * t * t));
            p->pbeta_host[(size_t)i] = (float)((t - 1.0) / t_next);
            t = t_next;
        }
        CUDA_TRY(cudaMemcpyAsync(p->pbeta, p->pbeta_host.data(), (size_t)n_iter * sizeof(float), cudaMemcpyHostToDevice, s));
        p->f_t = t;
    }
    P.beta = p->pbeta;
    CUDA_TRY(cudaMemsetAsync(p->pbar, 0, sizeof(unsigned), s));
    void *args[] = {(void *)&P};
    const void *kern = (const void *)fista_persistent_kernel;
    if (p->persist_small) {
        P.nvg = std::max(1, (p->n_vis_int + G - 2) / (G - 1));   // the last CTA stays idle: it sums the objective partials
        P.ybuf = p->pybuf;
        kern = (const void *)fista_persistent_small_kernel;
    }
    const cudaError_t le = cudaLaunchCooperativeKernel(kern, dim3((unsigned)G), dim3(PT), args, 0, s);
    if (le == cudaErrorCooperativeLaunchTooLarge || le == cudaErrorLaunchOutOfResources) {
        // the grid cannot be co-resident right now (e.g. the GPU is shared): this plan goes back to the multi-launch
        // loop for good.  Its compact tiles are rebuilt from y (the persistent kernel does not maintain them).
        cudaGetLastError();
        p->f_t = t_before;
        p->persist = false;
        pack_sorted_kernel<<<cgrid(p, p->n_pix_pad), ET, 0, s>>>(p->pix4, p->amp, p->y_sorted, p->n_pix_pad, zs_of(p));
        p->launches++;
        return -1;                                         // caller: carry on with the multi-launch loop
    }
    CUDA_TRY(le);
    p->launches++;
    p->f_k += n_iter;
    return check_launch("sl1m_fista_step(persistent)");
}

int fista_iterate(sl1m_plan *p, int n_iter, double *trace_dev, size_t trace_stride, int trace_row0,
                  const StopOpts *stop, cudaStream_t s) {
    if (p->persist && !p->chan_scale) {
        const int st = persist_iterate(p, n_iter, trace_dev ? trace_dev + 3 * (size_t)trace_row0 : nullptr, stop, s);
        if (st != -1) return st;
    }
    const int C = p->n_chan, npad = p->n_pix_pad;
    const float2 *step_c = C > 1 ? p->step_c : nullptr;
    const int *done = stop ? p->ctl_i : nullptr;
    p->done_ptr = done;
    struct DoneGuard {      // every exit, the CUDA_TRY early returns included, leaves no stale stop flags behind
        sl1m_plan *q;
        ~DoneGuard() { q->done_ptr = nullptr; }
    } done_guard{p};
    int pending[2] = {0, 0}, slot = 0, looks = 0;
    // How far the host may run ahead of the device's decision.  Small problems (an iteration is tens of
    // microseconds): read the flag every >= 16 iterations, two polls behind -- the iterations enqueued past the stop
    // return at once in the O(N) kernels and in every kernel of a batched plan; the main kernels of a
    // single-channel plan carry no flag test (it cost the packed forward 7 %: 157 -> 168 ms at config 5) and run
    // to no effect.  Large problems (an iteration is milliseconds): wait for every look -- a 10 us round-trip
    // against an iteration that costs a thousand times more.
    const bool big = 2.0 * (double)p->n_pix_pad * (double)p->n_vis_int >= 5e8;
    const int looks_per_poll = !stop ? 0 : (big ? 1 : std::max(1, 16 / std::max(1, stop->check_every)));
    if (stop && !p->h_flag) {
        CUDA_TRY(cudaMallocHost((void **)&p->h_flag, 2 * sizeof(int)));
        CUDA_TRY(cudaEventCreateWithFlags(&p->poll_ev[0], cudaEventDisableTiming));
        CUDA_TRY(cudaEventCreateWithFlags(&p->poll_ev[1], cudaEventDisableTiming));
    }
    for (int i = 0; i < n_iter; ++i) {
        const double t = p->f_t, t_next = 0.5 * (1.0 + std::sqrt(1.0 + 4.0 * t * t));
        const float beta = (float)((t - 1.0) / t_next);
        double *tr = trace_dev ? trace_dev + 3 * (size_t)(trace_row0 + i) : nullptr;
        launch_fwd(p, s);
        fwd_reduce_kernel<<<cgrid(p, p->n_vis_int), ET, 0, s>>>(p->ws_v, p->fwd_split, p->n_vis_int, p->vperm, p->f_vis,
                                                                p->resid, 1, tr ? p->part_a : nullptr, (int)p->n_vis,
                                                                p->n_part, done);
        launch_adj(p, p->resid, s);
        fista_update_kernel<<<cgrid(p, npad), ET, 0, s>>>(p->ws_p, p->adj_split, npad, p->amp, p->pix4, p->I_sorted,
                                                          p->y_sorted, p->f_inv_L, p->f_thr, beta,
                                                          tr ? p->part_b : nullptr, tr ? p->part_c : nullptr, step_c,
                                                          p->n_part, zs_of(p), done);
        p->launches += 2;
        if (tr) {
            sum_partials_kernel<<<C, ET, 0, s>>>(p->part_a, p->part_b, p->part_c, egrid(p->n_vis_int), egrid(npad),
                                                 egrid(npad), tr, tr + 1, tr + 2, p->n_part, trace_stride, done);
            p->launches++;
        }
        p->f_t = t_next;
        p->f_k++;
        if (stop && p->f_k >= 2 && p->f_k % stop->check_every == 0) {
            stop_rule_kernel<<<1, ET, 0, s>>>(trace_dev, trace_stride, p->f_k, C, p->lam2, stop->tol, stop->nnz_tol, p->ctl_i);
            p->launches++;
            if (++looks % looks_per_poll == 0) {
                if (pending[slot]) {                       // the poll issued two polls ago
                    CUDA_TRY(cudaEventSynchronize(p->poll_ev[slot]));
                    if (p->h_flag[slot]) break;
                }
                CUDA_TRY(cudaMemcpyAsync(&p->h_flag[slot], p->ctl_i + 2 * C, sizeof(int), cudaMemcpyDeviceToHost, s));
                CUDA_TRY(cudaEventRecord(p->poll_ev[slot], s));
                pending[slot] = 1;
                if (big) {                                 // wait for this look's decision before enqueueing more
                    CUDA_TRY(cudaEventSynchronize(p->poll_ev[slot]));
                    if (p->h_flag[slot]) break;
                    pending[slot] = 0;
                }
                slot ^= 1;
            }
        }
    }
    return check_launch("sl1m_fista_step");
}

int fista_image_impl(sl1m_plan *p, float *x_out_dev, cudaStream_t s) {
    scatter_kernel<<<cgrid(p, p->n_pix_pad), ET, 0, s>>>(p->I_sorted, p->perm, x_out_dev, p->n_pix_pad, (int)p->n_pix);
    p->launches++;
    return check_launch("sl1m_fista_image");
}

// Shared body of sl1m_solve / sl1m_solve_batch (stop == NULL: fixed iteration count) and sl1m_solve_stop(_batch).
int solve_impl(sl1m_plan *p, const float *vis_dev, const float *lambda_c, const float *L_c_in, int n_pow,
               int n_iter, const StopOpts *stop, const float *x0_dev, float *x_out_dev, double *trace_dev,
               sl1m_solve_info *info_host, void *stream) {
    // lambda_c, L_c_in: HOST [n_chan]; vis/x0/x_out: DEV [n_chan][.]; trace: DEV [n_chan][n_iter][3];
    // info_host: HOST [n_chan].
    if (!p || !vis_dev || !x_out_dev || !lambda_c || !L_c_in) return fail(SL1M_ERR_NULL, "sl1m_solve: NULL argument");
    if (n_iter < 0) return fail(SL1M_ERR_PARAM, "n_iter < 0");
    const int C = p->n_chan;
    std::vector<float> L_c(L_c_in, L_c_in + C);
    bool need_L = false;
    for (int c = 0; c < C; ++c) {
        if (!(lambda_c[c] >= 0.f)) return fail(SL1M_ERR_PARAM, "lambda < 0");
        need_L |= !(L_c[c] > 0.f);
    }
    if (need_L && n_pow < 1) return fail(SL1M_ERR_PARAM, "L <= 0 needs n_pow >= 1");
    cudaStream_t s = (cudaStream_t)stream;
    const int npad = p->n_pix_pad;
    int st;
    const size_t trace_stride = 3 * (size_t)std::max(n_iter, 1);   // doubles per channel in trace_dev
    if (stop && !trace_dev) {   // the stopping rule reads the trace: use the plan's own buffer
        if (p->trace_cap < (size_t)C * trace_stride) {
            if (p->trace_buf) cudaFree(p->trace_buf);
            p->trace_buf = nullptr;
            p->trace_cap = 0;
            CUDA_TRY(cudaMalloc((void **)&p->trace_buf, (size_t)C * trace_stride * sizeof(double)));
            p->trace_cap = (size_t)C * trace_stride;
        }
        trace_dev = p->trace_buf;
    }
    if (need_L) {
        std::vector<float> L_pow((size_t)C);
        if ((st = max_eig_impl(p, n_pow, L_pow.data(), stream))) return st;
        for (int c = 0; c < C; ++c) {
            if (!(L_c[c] > 0.f)) L_c[c] = L_pow[c];
            if (!(L_c[c] > 0.f)) return fail(SL1M_ERR_PARAM, "power iteration returned L <= 0 (zero operator)");
        }
    }
    if ((st = fista_begin_impl(p, vis_dev, lambda_c, L_c.data(), x0_dev, s))) return st;
    struct StateGuard {     // whichever way this call ends
        sl1m_plan *q;
        ~StateGuard() { q->f_active = false; q->f_vis = nullptr; }
    } state_guard{p};
    if ((st = fista_iterate(p, n_iter, trace_dev, trace_stride, 0, stop, s))) return st;
    const int n_enqueued = p->f_k;
    if ((st = fista_image_impl(p, x_out_dev, s))) return st;

    if (info_host) {
        // one extra forward for ||M I_K - V||^2 (Table 1's L2 term)
        pack_sorted_kernel<<<cgrid(p, npad), ET, 0, s>>>(p->pix4, p->amp, p->I_sorted, npad, zs_of(p));
        launch_fwd(p, s);
        fwd_reduce_kernel<<<cgrid(p, p->n_vis_int), ET, 0, s>>>(p->ws_v, p->fwd_split, p->n_vis_int, p->vperm,
                                                                (const float2 *)vis_dev, p->resid, 1, p->part_a,
                                                                (int)p->n_vis, p->n_part);
        l1_nnz_kernel<<<cgrid(p, npad), ET, 0, s>>>(p->I_sorted, npad, p->part_b, p->part_c, p->n_part);
        sum_partials_kernel<<<C, ET, 0, s>>>(p->part_a, p->part_b, p->part_c, egrid(p->n_vis_int), egrid(npad),
                                             egrid(npad), p->scalars + 1, p->scalars + 2, p->scalars + 3, p->n_part, 4);
        p->launches += 4;
        p->f_active = false;               // the pixel tiles now hold a*I_K, not a*y_{K+1}: the state cannot be stepped on
        if ((st = check_launch("sl1m_solve(info)"))) return st;
        std::vector<double> h(4 * (size_t)C);
        std::vector<int> ctl(2 * (size_t)C + 1, 0);
        CUDA_TRY(cudaMemcpyAsync(h.data(), p->scalars, h.size() * sizeof(double), cudaMemcpyDeviceToHost, s));
        if (stop) CUDA_TRY(cudaMemcpyAsync(ctl.data(), p->ctl_i, ctl.size() * sizeof(int), cudaMemcpyDeviceToHost, s));
        CUDA_TRY(cudaStreamSynchronize(s));
        for (int c = 0; c < C; ++c) {
            info_host[c].n_iter_done = (stop && ctl[c]) ? ctl[(size_t)C + c] : n_enqueued;
            info_host[c].L_used = L_c[c];
            info_host[c].l2_term = h[4 * c + 1];
            info_host[c].l1_term = h[4 * c + 2];
            info_host[c].nnz = (int64_t)(h[4 * c + 3] + 0.5);
        }
    }
    // Only sl1m_fista_begin opens a state that can be stepped: a solve's vis_dev is the caller's to free on return,
    // so a later sl1m_fista_step / sl1m_fista_image must fail with "no FISTA state" instead of reading it
    // (state_guard above).
    return SL1M_OK;
}
}  // namespace

extern "C" int sl1m_solve(sl1m_plan *p, const float *vis_dev, float lambda, float L, int n_pow, int n_iter,
                          const float *x0_dev, float *x_out_dev, double *trace_dev, sl1m_solve_info *info_host,
                          void *stream) {
    if (int st = single_channel_only(p, "sl1m_solve")) return st;
    return solve_impl(p, vis_dev, &lambda, &L, n_pow, n_iter, nullptr, x0_dev, x_out_dev, trace_dev, info_host, stream);
}

namespace {
int check_stop_args(double tol, double nnz_tol, int check_every, const void *info_host, const char *what) {
    if (tol != tol || nnz_tol != nnz_tol || (tol < 0.0 && nnz_tol < 0.0) || check_every < 1)
        return fail(SL1M_ERR_PARAM, std::string(what) + ": no stopping rule enabled (tol < 0 and nnz_tol < 0) or check_every < 1");
    if (!info_host) return fail(SL1M_ERR_NULL, std::string(what) + ": info_host is required (it carries n_iter_done)");
    return SL1M_OK;
}
}  // namespace

extern "C" int sl1m_solve_tol(sl1m_plan *p, const float *vis_dev, float lambda, float L, int n_pow, int max_iter,
                              double tol, int check_every, const float *x0_dev, float *x_out_dev,
                              double *trace_dev, sl1m_solve_info *info_host, void *stream) {
    if (int st = single_channel_only(p, "sl1m_solve_tol")) return st;
    if (!(tol >= 0.0) || check_every < 1) return fail(SL1M_ERR_PARAM, "sl1m_solve_tol: tol < 0 or check_every < 1");
    if (!info_host) return fail(SL1M_ERR_NULL, "sl1m_solve_tol: info_host is required (it carries n_iter_done)");
    const StopOpts so{tol, -1.0, check_every};
    return solve_impl(p, vis_dev, &lambda, &L, n_pow, max_iter, &so, x0_dev, x_out_dev, trace_dev, info_host, stream);
}

extern "C" int sl1m_solve_stop(sl1m_plan *p, const float *vis_dev, float lambda, float L, int n_pow, int max_iter,
                               double tol, double nnz_tol, int check_every, const float *x0_dev, float *x_out_dev,
                               double *trace_dev, sl1m_solve_info *info_host, void *stream) {
    if (int st = single_channel_only(p, "sl1m_solve_stop")) return st;
    if (int st = check_stop_args(tol, nnz_tol, check_every, info_host, "sl1m_solve_stop")) return st;
    const StopOpts so{tol, nnz_tol, check_every};
    return solve_impl(p, vis_dev, &lambda, &L, n_pow, max_iter, &so, x0_dev, x_out_dev, trace_dev, info_host, stream);
}

extern "C" int sl1m_solve_stop_batch(sl1m_plan *p, const float *vis_dev, const float *lambda_host, const float *L_host,
                                     int n_pow, int max_iter, double tol, double nnz_tol, int check_every,
                                     const float *x0_dev, float *x_out_dev, double *trace_dev,
                                     sl1m_solve_info *info_host, void *stream) {
    if (int st = check_stop_args(tol, nnz_tol, check_every, info_host, "sl1m_solve_stop_batch")) return st;
    const StopOpts so{tol, nnz_tol, check_every};
    return solve_impl(p, vis_dev, lambda_host, L_host, n_pow, max_iter, &so, x0_dev, x_out_dev, trace_dev, info_host,
                      stream);
}

extern "C" int sl1m_solve_batch(sl1m_plan *p, const float *vis_dev, const float *lambda_host, const float *L_host,
                                int n_pow, int n_iter, const float *x0_dev, float *x_out_dev, double *trace_dev,
                                sl1m_solve_info *info_host, void *stream) {
    return solve_impl(p, vis_dev, lambda_host, L_host, n_pow, n_iter, nullptr, x0_dev, x_out_dev, trace_dev,
                      info_host, stream);
}

// Stepping API: the same iteration, driven by the caller a few iterations at a time (interactive imaging,
// bench.py's per-step timing of ONE continuing FISTA run).
extern "C" int sl1m_fista_begin(sl1m_plan *p, const float *vis_dev, const float *lambda_host, const float *L_host,
                                const float *x0_dev, void *stream) {
    if (!p || !vis_dev || !lambda_host || !L_host) return fail(SL1M_ERR_NULL, "sl1m_fista_begin: NULL argument");
    for (int c = 0; c < p->n_chan; ++c)
        if (!(lambda_host[c] >= 0.f) || !(L_host[c] > 0.f)) return fail(SL1M_ERR_PARAM, "sl1m_fista_begin: lambda < 0 or L <= 0");
    return fista_begin_impl(p, vis_dev, lambda_host, L_host, x0_dev, (cudaStream_t)stream);
}

extern "C" int sl1m_fista_step(sl1m_plan *p, int n_iter, double *trace_dev, void *stream) {
    if (!p) return fail(SL1M_ERR_NULL, "sl1m_fista_step: NULL plan");
    if (!p->f_active) return fail(SL1M_ERR_PARAM, "sl1m_fista_step: no FISTA state (call sl1m_fista_begin; a solve that returned info ends the state)");
    if (n_iter < 0) return fail(SL1M_ERR_PARAM, "n_iter < 0");
    return fista_iterate(p, n_iter, trace_dev, 3 * (size_t)std::max(n_iter, 1), 0, nullptr, (cudaStream_t)stream);
}

extern "C" int sl1m_fista_image(sl1m_plan *p, float *x_out_dev, int32_t *n_iter_done_host, void *stream) {
    if (!p || !x_out_dev) return fail(SL1M_ERR_NULL, "sl1m_fista_image: NULL argument");
    if (!p->f_active) return fail(SL1M_ERR_PARAM, "sl1m_fista_image: no FISTA state");
    if (n_iter_done_host) *n_iter_done_host = p->f_k;
    return fista_image_impl(p, x_out_dev, (cudaStream_t)stream);
}

// NEXT-4: turn the plan into a batch of n_chan channels that share pixels, gains and baseline
// geometry; channel c sees uvw * scale[c].
extern "C" int sl1m_plan_set_channels(sl1m_plan *p, int32_t n_chan, const double *scale_host) {
    if (!p || !scale_host) return fail(SL1M_ERR_NULL, "sl1m_plan_set_channels: NULL argument");
    if (n_chan < 1 || n_chan > 65535) return fail(SL1M_ERR_SIZE, "n_chan must be in [1, 65535]");
    double scale_max = 0.0;
    for (int c = 0; c < n_chan; ++c) {
        if (!std::isfinite(scale_host[c]) || !(scale_host[c] > 0.0))
            return fail(SL1M_ERR_DOMAIN, "channel scale must be finite and > 0");
        scale_max = std::max(scale_max, scale_host[c]);
    }
    const size_t npad = (size_t)p->n_pix_pad;
    // Transactional: every buffer whose size depends on n_chan is allocated afresh next to the old one; the plan
    // switches over only when all of them exist, so a failure (out of memory) leaves it exactly as it was.
    sl1m_plan saved = *p;
    auto fields = [](sl1m_plan *q) {
        return std::vector<void **>{(void **)&q->ws_v, (void **)&q->ws_p, (void **)&q->resid, (void **)&q->rpol,
                                    (void **)&q->I_sorted, (void **)&q->y_sorted, (void **)&q->g_sorted,
                                    (void **)&q->part_a, (void **)&q->part_b, (void **)&q->part_c, (void **)&q->scalars,
                                    (void **)&q->pixc, (void **)&q->tile_cnt, (void **)&q->gFc, (void **)&q->gAc, (void **)&q->pixdc,
                                    (void **)&q->pixgc, (void **)&q->pix4,
                                    (void **)&q->chan_scale, (void **)&q->step_c, (void **)&q->h_x, (void **)&q->h_vis,
                                    (void **)&q->h_img, (void **)&q->ctl_i, (void **)&q->lam2, (void **)&q->trace_buf};
    };
    for (void **q : fields(p)) *q = nullptr;
    p->trace_cap = 0;
    p->f_active = false;
    p->n_chan = n_chan;
    // the fp32 phase remainder grows with the channel's frequency: re-evaluate the fp64-phase decision
    p->phase64 = p->phase64_capable && (p->phase64_flag || p->phase_span * scale_max > 256.0);
    auto attempt = [&]() -> int {
        // replicate the pixel tiles: channel c keeps its own a*x in pix4[c][.].w
        CUDA_TRY(cudaMalloc((void **)&p->pix4, (size_t)n_chan * npad * sizeof(float4)));
        for (int c = 0; c < n_chan; ++c)
            CUDA_TRY(cudaMemcpy(p->pix4 + (size_t)c * npad, saved.pix4, npad * sizeof(float4), cudaMemcpyDeviceToDevice));
        CUDA_TRY(cudaMalloc((void **)&p->chan_scale, (size_t)n_chan * sizeof(double)));
        CUDA_TRY(cudaMemcpy(p->chan_scale, scale_host, (size_t)n_chan * sizeof(double), cudaMemcpyHostToDevice));
        CUDA_TRY(cudaMalloc((void **)&p->step_c, (size_t)n_chan * sizeof(float2)));
        if (int st = configure_and_allocate(p)) return st;
        CUDA_TRY(cudaDeviceSynchronize());
        return SL1M_OK;
    };
    const int st = attempt();
    sl1m_plan *loser = st ? p : &saved;       // free the new buffers on failure, the old ones on success
    for (void **q : fields(loser))
        if (*q) cudaFree(*q);
    if (st) {
        const int64_t launches = p->launches;
        *p = saved;
        p->launches = launches;
    }
    return st;
}

extern "C" int32_t sl1m_plan_n_chan(const sl1m_plan *p) { return p ? p->n_chan : 0; }

extern "C" int sl1m_dirty_image(sl1m_plan *p, const float *vis_dev, float scale, float *img_dev, void *stream) {
    if (!p || !vis_dev || !img_dev) return fail(SL1M_ERR_NULL, "sl1m_dirty_image: NULL argument");
    if (!std::isfinite(scale)) return fail(SL1M_ERR_PARAM, "sl1m_dirty_image: non-finite scale");
    int st = sl1m_adjoint(p, vis_dev, img_dev, stream);
    if (st) return st;
    const size_t n_all = (size_t)p->n_chan * (size_t)p->n_pix;      // [n_chan][n_pix] is contiguous
    scale_clip_kernel<<<egrid(n_all), ET, 0, (cudaStream_t)stream>>>(img_dev, scale, n_all);
    p->launches++;
    return check_launch("sl1m_dirty_image");
}

extern "C" int sl1m_solve_host(sl1m_plan *p, const float *vis_host, float lambda, float L, int n_pow, int n_iter,
                               const float *x0_host, float *x_out_host, sl1m_solve_info *info_host,
                               void *stream) {
    if (!p || !vis_host || !x_out_host) return fail(SL1M_ERR_NULL, "sl1m_solve_host: NULL argument");
    if (int stc = single_channel_only(p, "sl1m_solve_host")) return stc;
    cudaStream_t s = (cudaStream_t)stream;
    int st = ensure_host_staging(p);
    if (st) return st;
    CUDA_TRY(cudaMemcpyAsync(p->h_vis, vis_host, (size_t)p->n_vis * sizeof(float2), cudaMemcpyHostToDevice, s));
    if (x0_host)
        CUDA_TRY(cudaMemcpyAsync(p->h_x, x0_host, (size_t)p->n_pix * sizeof(float), cudaMemcpyHostToDevice, s));
    if ((st = sl1m_solve(p, p->h_vis, lambda, L, n_pow, n_iter, x0_host ? p->h_x : nullptr, p->h_img, nullptr,
                         info_host, stream)))
        return st;
    CUDA_TRY(cudaMemcpyAsync(x_out_host, p->h_img, (size_t)p->n_pix * sizeof(float), cudaMemcpyDeviceToHost, s));
    CUDA_TRY(cudaStreamSynchronize(s));
    return SL1M_OK;
}

extern "C" int sl1m_plan_describe(const sl1m_plan *p, sl1m_plan_info *o) {
    if (!p || !o) return fail(SL1M_ERR_NULL, "sl1m_plan_describe: NULL argument");
    memset(o, 0, sizeof(*o));
    o->n_pix_padded = p->n_pix_pad;
    o->n_tiles = p->n_tiles;
    o->gaussian = p->gauss;
    o->gains = p->gk;
    o->fwd_rv = p->fwd_rv;
    o->fwd_vis_tiles = p->fwd_vtiles;
    o->fwd_pixel_splits = p->fwd_split;
    o->fwd_tiles_per_split = p->fwd_per_split;
    o->adj_rp = p->adj_rp;
    o->adj_pixel_groups = p->adj_pgroups;
    o->adj_vis_splits = p->adj_split;
    o->adj_chunks_per_split = p->adj_per_split;
    const int pk = p->gauss ? 1 : 0;
    const bool plain = !pk && p->gk == 0;          // delta pixels, unit gains
    const bool grouped = !pk && p->gk == 2;        // delta pixels, baseline-grouped gains
    o->fwd_poly_per16 = plain ? (p->fwd_rv == 8 ? SL1M_FWD_NPQ : (p->fwd_rv == 4 ? (SL1M_FWD_NPOLY8 / 2) * 4 : 0))
                              : (grouped ? SL1M_FWD_G2_NPQ : 0);
    constexpr int adj_npq8 = SL1M_ADJ_C1_NPQ;
    o->adj_poly_per16 = plain ? (p->adj_rp == 8 ? adj_npq8 : (p->adj_rp == 4 ? (SL1M_ADJ_NPOLY8 / 2) * 4 : 0))
                              : (grouped && p->adj_rp == 8 ? SL1M_ADJ_G2_NPQ : 0);
    o->mufu_per_term_mufu_path = p->pk == 2 ? 3 : (pk ? 4 : 2);
    o->gaussian = p->pk;
    o->phase_fp64 = p->phase64;
    o->phase_span_rad = (float)p->phase_span;
    o->zero_skip = p->pixc != nullptr;
    o->persistent = p->persist && !p->chan_scale;
    o->adj_mufu_per_term = o->mufu_per_term_mufu_path;
    if (p->phase64) o->adj_mufu_per_term = 1;      // adj_kernel_p64: |r| cos(X + arg r)
    if (!p->phase64) {
        if (p->pk == 0) o->adj_mufu_per_term = 1;    // delta pixels: one cosine per term in every adjoint kernel
        if (p->pk == 2 && p->gk == 0 && p->adj_rp == 8) o->adj_mufu_per_term = 2;    // adj_kernel_gtx2: ex2 + cos
    }
    if (o->phase_fp64) o->fwd_poly_per16 = o->adj_poly_per16 = 0;
    const bool tile_gauss = p->pk == 2 && p->gk == 0;
    o->fwd_packed_pairs = ((plain || tile_gauss) && p->fwd_rv == 8) || grouped;
    o->adj_packed_pairs = (plain || grouped || tile_gauss) && p->adj_rp == 8;
    return SL1M_OK;
}

extern "C" int sl1m_forward_active_pixels(sl1m_plan *p, int64_t *n_active_host, void *stream) {
    if (!p || !n_active_host) return fail(SL1M_ERR_NULL, "sl1m_forward_active_pixels: NULL argument");
    const size_t C = (size_t)p->n_chan, T = (size_t)p->n_tiles;
    if (!p->tile_cnt) {   // dense forward: every (padded) pixel is streamed
        for (size_t c = 0; c < C; ++c) n_active_host[c] = (int64_t)p->n_pix_pad;
        return SL1M_OK;
    }
    cudaStream_t s = (cudaStream_t)stream;
    if (p->persist && !p->chan_scale && p->f_active) {
        // A stepped run on the persistent kernels: they skip zero pixels warp by warp from y itself and never touch
        // tile_cnt (it would still say what the last multi-launch pack saw).  Count y_{k+1} != 0 instead -- exactly the
        // pixels the next iteration's forward evaluates.  Persistent plans are small (< 6.7e7 terms per apply).
        std::vector<float> y((size_t)p->n_pix_pad);
        CUDA_TRY(cudaMemcpyAsync(y.data(), p->y_sorted, y.size() * sizeof(float), cudaMemcpyDeviceToHost, s));
        CUDA_TRY(cudaStreamSynchronize(s));
        int64_t n = 0;
        for (float v : y) n += (v != 0.f);
        n_active_host[0] = n;
        return SL1M_OK;
    }
    std::vector<int> h(C * T);
    CUDA_TRY(cudaMemcpyAsync(h.data(), p->tile_cnt, h.size() * sizeof(int), cudaMemcpyDeviceToHost, s));
    CUDA_TRY(cudaStreamSynchronize(s));
    for (size_t c = 0; c < C; ++c) {
        int64_t n = 0;
        for (size_t t = 0; t < T; ++t) n += h[c * T + t];
        n_active_host[c] = n;
    }
    return SL1M_OK;
}

extern "C" int sl1m_debug_check(void) {
#ifdef SL1M_BOUNDS
    cudaError_t e = cudaDeviceSynchronize();                  // also surfaces a device-side assert of ldg_gain
    if (e != cudaSuccess) return fail(SL1M_ERR_CUDA, std::string("sl1m_debug_check: ") + cudaGetErrorString(e));
    std::vector<unsigned char> h(2 * CANARY + 256);
    std::lock_guard<std::mutex> lk(g_allocs_mu);
    for (const auto &kv : g_allocs) {
        const unsigned char *u = (const unsigned char *)kv.first;
        const size_t bytes = kv.second.bytes, tail = (bytes + 255) / 256 * 256 - bytes + CANARY;
        if ((cudaMemcpy)(h.data(), u - CANARY, CANARY, cudaMemcpyDeviceToHost) != cudaSuccess ||
            (cudaMemcpy)(h.data() + CANARY, u + bytes, tail, cudaMemcpyDeviceToHost) != cudaSuccess)
            return fail(SL1M_ERR_CUDA, "sl1m_debug_check: cannot read a canary band");
        for (size_t i = 0; i < CANARY + tail; ++i)
            if (h[i] != 0xA5) {
                char msg[160];
                snprintf(msg, sizeof(msg), "sl1m_debug_check: buffer of %zu bytes overwritten %s its %s (byte %zu of the band)",
                         bytes, i < CANARY ? "before" : "past", i < CANARY ? "start" : "end", i < CANARY ? CANARY - i : i - CANARY);
                return fail(SL1M_ERR_CUDA, msg);
            }
    }
    return SL1M_OK;
#else
    return SL1M_OK;
#endif
}

extern "C" int sl1m_debug_poke_past_end(sl1m_plan *p) {
#ifdef SL1M_BOUNDS
    if (!p) return fail(SL1M_ERR_NULL, "sl1m_debug_poke_past_end: NULL plan");
    const float v = 1.0f;      // 4 bytes just past the residual buffer: what a one-element overrun of a kernel would do
    CUDA_TRY((cudaMemcpy)((unsigned char *)p->resid + (size_t)p->n_chan * (size_t)p->n_vis_int * sizeof(float2), &v, sizeof(v),
                          cudaMemcpyHostToDevice));
    return SL1M_OK;
#else
    (void)p;
    return fail(SL1M_ERR_PARAM, "sl1m_debug_poke_past_end: not a -DSL1M_BOUNDS build");
#endif
}

extern "C" int sl1m_debug_bounds_build(void) {
#ifdef SL1M_BOUNDS
    return 1;
#else
    return 0;
#endif
}

extern "C" int64_t sl1m_launch_count(const sl1m_plan *p) { return p ? p->launches : 0; }
extern "C" int64_t sl1m_plan_n_vis(const sl1m_plan *p) { return p ? p->n_vis : 0; }
extern "C" int64_t sl1m_plan_n_pix(const sl1m_plan *p) { return p ? p->n_pix : 0; }

extern "C" void sl1m_destroy(sl1m_plan *p) { free_plan(p); }

extern "C" const char *sl1m_status_string(int st) {
    switch (st) {
        case SL1M_OK: return "SL1M_OK";
        case SL1M_ERR_NULL: return "SL1M_ERR_NULL";
        case SL1M_ERR_SIZE: return "SL1M_ERR_SIZE";
        case SL1M_ERR_DOMAIN: return "SL1M_ERR_DOMAIN";
        case SL1M_ERR_INDEX: return "SL1M_ERR_INDEX";
        case SL1M_ERR_ALLOC: return "SL1M_ERR_ALLOC";
        case SL1M_ERR_CUDA: return "SL1M_ERR_CUDA";
        case SL1M_ERR_PARAM: return "SL1M_ERR_PARAM";
        default: return "SL1M_ERR_UNKNOWN";
    }
}

extern "C" const char *sl1m_last_error(void) { return g_last_error.c_str(); }
