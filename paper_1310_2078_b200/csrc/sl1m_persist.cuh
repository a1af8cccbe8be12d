// sl1m_persist.cuh -- the whole FISTA loop of a SMALL problem in ONE persistent cooperative kernel.
//
// Why: config 1 (1,024 pixels x 1,000 visibilities) is 2e6 generated terms per iteration -- under a microsecond
// of arithmetic on 148 SMs -- but the multi-launch loop (forward, residual epilogue, polar residual, adjoint, fused
// update, partial sums) costs 18.7 us per iteration in launch latency alone.  The paper's small real
// data set is of this kind: 127 channels of 256^2 pixels x 11,934 visibilities, ~200 iterations each
// (PAPER.md:279-291).  Here one CTA per SM stays resident for all iterations of the listing:
//
//   phase A (forward + residual, a1 + a3):  a CTA owns <= 8 visibilities; its threads split the pixel list, generate
//       the entries (eq 9, tile-centred phase as in sl1m_kernels.cuh), reduce over the CTA in a fixed order, subtract
//       V and leave the residual in POLAR form (|r|, arg r) in global memory.
//   --- grid barrier ---
//   phase B (adjoint + update, a2 + a4 + a5): a CTA owns <= 8 consecutive pixels; its threads split the
//       visibilities, accumulate |r| cos(X + arg r) (one cosine per term: the image is real), reduce, and the pixel's
//       owner thread applies the gradient step, T^{lambda/L} (eq 18), the momentum and re-packs a*y.
//   --- grid barrier ---
//   objective partials (a6), the trace row and the stopping rules (readings R21, R24) from per-CTA
//       partials, on the device; every CTA takes the same decision from the same numbers and leaves together.
//
// The phase of a term is x0(j, tile) + u' dl + v' dm + w' dn' as in the tuned kernels, but x0 -- the fp64 centre
// phase of every (visibility, tile) pair -- is iteration-invariant, so it is tabulated ONCE at plan time
// (n_tiles x n_vis floats).  Data another CTA wrote in the previous phase is read with ld.global.cg (L1 is not
// coherent); constants go through the read-only path.  Sums are formed in a fixed order: results are bit-stable run
// to run, but the order differs from the multi-launch kernels', so the two paths agree to rounding, not bit for bit.
//
// Zero-skipping: a warp compacts its 128-pixel block to the entries with a*y != 0 (ballot + prefix popcount, order
// kept) before generating terms, so the forward costs what the non-zero pixels cost, as in the tuned path.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "sl1m_kernels.cuh"

namespace sl1m {

constexpr int PT = 256;            // threads per CTA
constexpr int PW = PT / 32;        // warps per CTA
constexpr int PG = 8;              // visibilities (phase A) / pixels (phase B) per work item
constexpr int PBLK = 128;          // pixels a warp compacts at a time in phase A
constexpr int PERSIST_MAX_TILES = 512;   // 131,072 pixels: s_x0 is 16 KB of the CTA's 34 KB of static shared memory

struct PersistParams {
    int n_vis, n_pix_pad, n_tiles;
    int nvg, npg;                  // visibilities / pixels per work item (1, 2, 4 or 8; npg divides TP)
    const float4 *vis4;            // [n_vis] (2 pi u, 2 pi v, 2 pi w, 0)
    const float *x0;               // [n_tiles][n_vis] centre phases, radians in [-pi, pi]
    float4 *pix4;                  // [n_pix_pad] (dl, dm, dn', a*y); .w rewritten every iteration
    const float *amp;              // [n_pix_pad] 1/n_k (0 on padding)
    float *I_sorted, *y_sorted;    // [n_pix_pad] I_k, y_{k+1}
    const float2 *V;               // [n_vis] measured visibilities
    float2 *rpol;                  // [n_vis] residual (|r|, arg r)
    double *part;                  // [2][3][gridDim.x] per-CTA partials (||r||^2, sum I, nnz), double-buffered by iteration parity
    unsigned *bar;                 // grid-barrier counter, zero at launch
    double *trace;                 // [.][3] rows of this launch's iterations, or NULL
    int *ctl;                      // {done, n_done, all_done} (sl1m_solve_stop) or NULL
    float inv_L, thr;
    double lam2, tol, nnz_tol;     // stopping rules (tol, nnz_tol < 0: off)
    int check_every;               // 0: no stopping rule
    int k0;                        // iterations done before this launch
    const float *beta;             // [n_iter] momentum coefficients (t_k - 1)/t_{k+1} of this launch's iterations, formed in
                                   // fp64 on the host (a device fp64 sqrt + divide cost 0.3 us per iteration on the critical path)
    int n_iter;
    float *ybuf;                   // [2][n_pix_pad] a*y_k, double-buffered by iteration parity (fista_persistent_small_kernel)
};

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned *p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
// All CTAs of the (cooperatively launched, co-resident) grid meet here.  Monotonic counter: the n-th barrier is
// passed when it reaches n * gridDim.x.
// Default (SL1M_BAR_MODE 2): thread 0 arrives with one red.release.gpu (orders every earlier write of the CTA, which
// the leading __syncthreads made visible to it, before the increment) and polls with ld.acquire.gpu: the poll that
// reads the final count synchronises-with every producer's release (release/acquire pattern of the PTX memory
// model), and the trailing __syncthreads hands that on to the CTA's other threads.  Nothing here leans on how this
// chip happens to order loads.
// SL1M_BAR_MODE bit 1: red.release arrive (else __threadfence + atomicAdd); bit 0: ld.relaxed poll followed by
// fence.acq_rel.gpu (also covered by the model); bit 2: ... without that fence.  Measured at config 1, 2,000-iteration
// solve (profiles/r3_microbench.md): mode 2 4.72 us per iteration, mode 3 5.44, mode 7 4.63.  Mode 7 (no
// consumer-side acquire at all) was the default in round 2; it has never produced a differing bit, but it is correct
// only by an argument about the hardware (consumers use ld.global.cg, in-order issue, control dependency on the
// poll), not by the memory model -- it buys 0.09 us and stays an opt-in for measurements.
#ifndef SL1M_BAR_MODE
#define SL1M_BAR_MODE 2
#endif
__device__ __forceinline__ void grid_barrier(unsigned *bar, unsigned &target) {
    __syncthreads();
    if (threadIdx.x == 0) {
        target += gridDim.x;
#if SL1M_BAR_MODE & 2
        asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(bar), "r"(1u) : "memory");
#else
        __threadfence();
        atomicAdd(bar, 1u);
#endif
#if SL1M_BAR_MODE & 1
        unsigned v;
        do {
            asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(bar) : "memory");
        } while (v < target);
#if !(SL1M_BAR_MODE & 4)
        asm volatile("fence.acq_rel.gpu;" ::: "memory");
#endif
#else
        while (ld_acquire_u32(bar) < target) {}
#endif
    }
    __syncthreads();
}

// Fixed-order CTA sum of N per-thread values: warp shuffles, then PW per-warp partials added in warp order.
// Result valid in threads 0..N-1 (thread i holds sum i).
template <int N>
__device__ __forceinline__ float cta_sum(float (&v)[N], float (*s_red)[PG * 2 + 1]) {
    static_assert(N == 8 || N == 16, "cta_sum: 8 or 16 values per thread");
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // Warp stage: a halving butterfly -- at every step a lane keeps half of its values and sends the other half to its
    // partner, so N values x 32 lanes take N - 1 + (5 - log2 N) shuffles instead of 5 N.  Afterwards lane l holds the
    // warp's sum of value number (l mod N) (bit-reversed bookkeeping below); the order of additions is fixed.
    float w[N];
#pragma unroll
    for (int i = 0; i < N; ++i) w[i] = v[i];
    int idx = 0;                                             // which value this lane ends up holding
    {
        constexpr int STEPS = (N == 16) ? 4 : 3;
#pragma unroll
        for (int s = 0; s < STEPS; ++s) {
            const int half = N >> (s + 1);
            const bool up = (lane >> s) & 1;                 // upper partner keeps the upper half
#pragma unroll
            for (int i = 0; i < half; ++i) {
                const float keep = up ? w[i + half] : w[i];
                const float give = up ? w[i] : w[i + half];
                w[i] = keep + __shfl_xor_sync(0xffffffffu, give, 1 << s);
            }
            idx |= up ? half : 0;
        }
        // remaining lane bits: plain butterfly on the single value left
#pragma unroll
        for (int o = 1 << STEPS; o < 32; o <<= 1) w[0] += __shfl_xor_sync(0xffffffffu, w[0], o);
    }
    __syncthreads();                      // s_red free again
    if (lane < N) s_red[warp][idx] = w[0];                   // lanes 0..N-1 cover every idx exactly once
    __syncthreads();
    float t = 0.f;
    if (threadIdx.x < N) {
#pragma unroll
        for (int ww = 0; ww < PW; ++ww) t += s_red[ww][threadIdx.x];
    }
    return t;
}

// Sum of n doubles at p (written by other CTAs: ld.cg), by one warp in a fixed order; result in every lane.
__device__ __forceinline__ double warp_sum_cg(const double *p, int n) {
    double v = 0.0;
    for (int i = threadIdx.x & 31; i < n; i += 32) v += __ldcg(p + i);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// The three partial arrays at once, every load in flight before the first add (one L2 round trip: this sum sits on
// the critical path of the CTA that writes the trace row).  n <= 32 * 8 elements per array.
__device__ __forceinline__ void warp_sum3_cg(const double *p, int n, double &a, double &b, double &c) {
    const int lane = threadIdx.x & 31;
    double x[8], y[8], z[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        const int i = lane + 32 * q;
        const bool in = i < n;
        x[q] = in ? __ldcg(p + i) : 0.0;
        y[q] = in ? __ldcg(p + n + i) : 0.0;
        z[q] = in ? __ldcg(p + 2 * n + i) : 0.0;
    }
    a = b = c = 0.0;
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        a += x[q];
        b += y[q];
        c += z[q];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a += __shfl_xor_sync(0xffffffffu, a, o);
        b += __shfl_xor_sync(0xffffffffu, b, o);
        c += __shfl_xor_sync(0xffffffffu, c, o);
    }
}

__global__ void __launch_bounds__(PT, 1) fista_persistent_kernel(const PersistParams P) {
    __shared__ __align__(16) float4 s_list[PW][PBLK];       // compacted non-zero pixels of the warp's block
    __shared__ uint16_t s_tile[PW][PBLK];                    // their tile index
    __shared__ __align__(16) float s_x0[PERSIST_MAX_TILES][PG];   // centre phases of the CTA's phase-A item
    __shared__ float s_red[PW][PG * 2 + 1];
    __shared__ int s_stop;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int G = gridDim.x;
    unsigned bar_target = 0;
    const int items_a = (P.n_vis + P.nvg - 1) / P.nvg;
    const int items_b = P.n_pix_pad / P.npg;
    const bool one_item_a = items_a <= G;                    // the CTA's x0 slice never changes: stage it once
    double E_prev = 0.0, N_prev = 0.0;
    int staged_item = -1;
    // the CTA that sums the partials into the trace row: the last one when it has no work item of its own
    const int tracer = (items_a < G && items_b < G) ? G - 1 : 0;
    // Everything that does not change from one iteration to the next stays in registers when the CTA has a single
    // work item per phase (the small-problem case this kernel exists for): an iteration is latency-bound, and every
    // L2 round trip taken off its critical path is 0.15 us.
    const bool one_item_b = items_b <= G;
    const bool res_v = one_item_b && P.n_vis <= 4 * PT;      // phase B: the thread's <= 4 visibilities live in registers
    float uf[PG], vf[PG], wf[PG];                            // phase A: the item's visibilities
    float2 Vj = make_float2(0.f, 0.f);
    bool a_loaded = false, b_loaded = false;
    float dl[PG], dm[PG], dn[PG];                            // phase B: the item's pixels
    float a_own = 0.f, y_own = 0.f, I_own = 0.f;             // ... and the state of the pixel this thread updates
    float4 v4r[4];
    float x0v[4];

    for (int it = 0; it < P.n_iter; ++it) {
        const int k = P.k0 + it + 1;                         // 1-based iteration number of the listing
        double *part = P.part + (size_t)(k & 1) * 3 * G;

        // ------------------------------------------------------------------ phase A: r = M y - V
        double r2 = 0.0;
        for (int item = blockIdx.x; item < items_a; item += G) {
            const int j0 = item * P.nvg;
            if (staged_item != item) {
                __syncthreads();
                for (int i = tid; i < P.n_tiles * PG; i += PT) {
                    const int tl = i / PG, r = i - tl * PG, j = min(j0 + r, P.n_vis - 1);
                    s_x0[tl][r] = __ldg(P.x0 + (size_t)tl * P.n_vis + j);
                }
                __syncthreads();
                staged_item = one_item_a ? item : -1;
            }
            float acc[2 * PG];
#pragma unroll
            for (int r = 0; r < 2 * PG; ++r) acc[r] = 0.f;
            if (!a_loaded) {
#pragma unroll
                for (int r = 0; r < PG; ++r) {
                    const float4 v4 = __ldg(P.vis4 + min(j0 + r, P.n_vis - 1));
                    uf[r] = v4.x;
                    vf[r] = v4.y;
                    wf[r] = v4.z;
                }
                if (tid < 2 * P.nvg && (tid & 1) == 0 && j0 + (tid >> 1) < P.n_vis) Vj = __ldg(P.V + j0 + (tid >> 1));
                a_loaded = one_item_a;
            }
            // the warp's share of the pixel list, PBLK pixels at a time: compact to a*y != 0, then generate
            for (int base = warp * PBLK; base < P.n_pix_pad; base += PW * PBLK) {
                int cnt = 0;
                float4 pxq[PBLK / 32];
#pragma unroll
                for (int q = 0; q < PBLK / 32; ++q) pxq[q] = __ldcg(P.pix4 + base + q * 32 + lane);   // all in flight before the first ballot
#pragma unroll
                for (int q = 0; q < PBLK / 32; ++q) {
                    const int kpx = base + q * 32 + lane;
                    const float4 px = pxq[q];
                    const bool nz = px.w != 0.f;             // NaN counts as non-zero and propagates
                    const unsigned b = __ballot_sync(0xffffffffu, nz);
                    if (nz) {
                        const int pos = cnt + __popc(b & ((1u << lane) - 1u));
                        s_list[warp][pos] = px;
                        s_tile[warp][pos] = (uint16_t)(kpx / TP);
                    }
                    cnt += __popc(b);
                }
                __syncwarp();
                for (int i = lane; i < cnt; i += 32) {
                    const float4 px = s_list[warp][i];
                    const float4 *x0q = reinterpret_cast<const float4 *>(s_x0[s_tile[warp][i]]);
                    const float4 xa = x0q[0], xb = x0q[1];
                    const float x0r[PG] = {xa.x, xa.y, xa.z, xa.w, xb.x, xb.y, xb.z, xb.w};
#pragma unroll
                    for (int r = 0; r < PG; ++r) {
                        if (r < P.nvg) {
                            const float X = fmaf(uf[r], px.x, fmaf(vf[r], px.y, fmaf(wf[r], px.z, x0r[r])));
                            float s, c;
                            __sincosf(X, &s, &c);
                            acc[2 * r] = fmaf(px.w, c, acc[2 * r]);
                            acc[2 * r + 1] = fmaf(-px.w, s, acc[2 * r + 1]);
                        }
                    }
                }
                __syncwarp();
            }
            const float sum = cta_sum<2 * PG>(acc, s_red);   // thread i: re (i even) / im (i odd) of visibility i / 2
            // pair up (re, im) in the even thread
            const float other = __shfl_down_sync(0xffffffffu, sum, 1);
            if (tid < 2 * P.nvg && (tid & 1) == 0) {
                const int j = j0 + (tid >> 1);
                if (j < P.n_vis) {
                    const float re = sum - Vj.x, im = other - Vj.y;
                    P.rpol[j] = make_float2(sqrtf(fmaf(re, re, im * im)), atan2f(im, re));
                    r2 += (double)re * re + (double)im * im;
                }
            }
        }
        if (tid < 32) {                                      // the CTA's ||r||^2 partial (even lanes of warp 0 hold terms)
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) r2 += __shfl_xor_sync(0xffffffffu, r2, o);
            if (tid == 0) part[blockIdx.x] = r2;
        }
        grid_barrier(P.bar, bar_target);

        // ------------------------------------------------------------------ phase B: g = Re M^H r, update
        const float beta = __ldg(P.beta + it);
        double l1 = 0.0, nz = 0.0;
        for (int item = blockIdx.x; item < items_b; item += G) {
            const int p0 = item * P.npg;
            const float *x0row = P.x0 + (size_t)(p0 / TP) * P.n_vis;      // npg divides TP: one tile per item
            float acc[PG];
#pragma unroll
            for (int i = 0; i < PG; ++i) acc[i] = 0.f;
            if (!b_loaded) {
#pragma unroll
                for (int i = 0; i < PG; ++i) {
                    const float4 px = __ldcg(P.pix4 + min(p0 + i, P.n_pix_pad - 1));   // .xyz are constants, .w is rewritten below
                    dl[i] = px.x;
                    dm[i] = px.y;
                    dn[i] = px.z;
                }
                if (tid < P.npg) {
                    a_own = __ldg(P.amp + p0 + tid);
                    y_own = P.y_sorted[p0 + tid];
                    I_own = P.I_sorted[p0 + tid];
                }
                if (res_v) {
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        const int j = min(tid + q * PT, P.n_vis - 1);
                        v4r[q] = __ldg(P.vis4 + j);
                        x0v[q] = __ldg(x0row + j);
                    }
                }
                b_loaded = one_item_b;
            }
            if (res_v) {
                float2 rp[4];
#pragma unroll
                for (int q = 0; q < 4; ++q)                        // the four residual loads are in flight together
                    rp[q] = (tid + q * PT < P.n_vis) ? __ldcg(P.rpol + tid + q * PT) : make_float2(0.f, 0.f);
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const float ph = x0v[q] + rp[q].y;
#pragma unroll
                    for (int i = 0; i < PG; ++i) {
                        if (i < P.npg) {
                            const float X = fmaf(v4r[q].x, dl[i], fmaf(v4r[q].y, dm[i], fmaf(v4r[q].z, dn[i], ph)));
                            acc[i] = fmaf(rp[q].x, __cosf(X), acc[i]);
                        }
                    }
                }
            } else {
                for (int j = tid; j < P.n_vis; j += PT) {
                    const float4 v4 = __ldg(P.vis4 + j);
                    const float2 rp = __ldcg(P.rpol + j);
                    const float ph = __ldg(x0row + j) + rp.y;
#pragma unroll
                    for (int i = 0; i < PG; ++i) {
                        if (i < P.npg) {
                            const float X = fmaf(v4.x, dl[i], fmaf(v4.y, dm[i], fmaf(v4.z, dn[i], ph)));
                            acc[i] = fmaf(rp.x, __cosf(X), acc[i]);
                        }
                    }
                }
            }
            const float gsum = cta_sum<PG>(acc, s_red);
            if (tid < P.npg) {
                const int kk = p0 + tid;
                const float g = gsum * a_own;
                const float z = fmaf(-P.inv_L, g, y_own);
                const float I_new = (z > P.thr) ? z - P.thr : 0.f;
                const float y_new = fmaf(beta, I_new - I_own, I_new);
                I_own = I_new;                                 // with several items per CTA these are reloaded per item
                y_own = y_new;
                if (!one_item_b) {                             // one item: the state stays in registers until the kernel ends
                    P.I_sorted[kk] = I_new;
                    P.y_sorted[kk] = y_new;
                }
                P.pix4[kk].w = a_own * y_new;
                l1 += (double)I_new;
                nz += (I_new != 0.f) ? 1.0 : 0.0;
            }
        }
        if (tid < 32) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                l1 += __shfl_xor_sync(0xffffffffu, l1, o);
                nz += __shfl_xor_sync(0xffffffffu, nz, o);
            }
            if (tid == 0) {
                part[G + blockIdx.x] = l1;
                part[2 * G + blockIdx.x] = nz;
            }
        }
        grid_barrier(P.bar, bar_target);

        // ------------------------------------------------------------------ a6: objective, trace, stopping rules
        const bool look = P.check_every > 0 && k >= 2 && (k % P.check_every) == 0;
        const bool before_look = P.check_every > 0 && ((k + 1) % P.check_every) == 0;
        const bool want = look || before_look || (P.trace && blockIdx.x == tracer);
        if (want) {
            if (warp == 0) {
                double l2s, l1s, nzs;
                warp_sum3_cg(part, G, l2s, l1s, nzs);
                if (lane == 0) {
                    if (P.trace && blockIdx.x == tracer) {
                        P.trace[3 * (size_t)it] = l2s;
                        P.trace[3 * (size_t)it + 1] = l1s;
                        P.trace[3 * (size_t)it + 2] = nzs;
                    }
                    const double E = l2s + P.lam2 * l1s;
                    int stop = 0;
                    if (look)
                        stop = (P.tol >= 0.0 && fabs(E - E_prev) <= P.tol * fabs(E)) ||
                               (P.nnz_tol >= 0.0 && fabs(nzs - N_prev) <= P.nnz_tol * nzs);
                    E_prev = E;
                    N_prev = nzs;
                    s_stop = stop;
                    if (stop && blockIdx.x == 0) {
                        P.ctl[0] = 1;
                        P.ctl[1] = k;
                        P.ctl[2] = 1;
                    }
                }
            }
            if (P.check_every > 0) {
                __syncthreads();
                if (s_stop) break;                           // same numbers, same decision in every CTA
                __syncthreads();
            }
        }
    }
    // the register-resident state of the CTA's pixels goes back to global memory (next launch, sl1m_fista_image)
    if (one_item_b && blockIdx.x < items_b && tid < P.npg) {
        P.I_sorted[blockIdx.x * P.npg + tid] = I_own;
        P.y_sorted[blockIdx.x * P.npg + tid] = y_own;
    }
}

// ------------------------------------------------------------------------------------------
// The smallest problems (<= 1,024 padded pixels, <= 1,024 visibilities, one work item per CTA and phase: config 1).
// The same two phases and barriers as above, specialised: every iteration-invariant operand is in registers (also the
// (dl, dm, dn') of the pixels a thread reads in phase A), and a*y travels as 4-byte floats through a buffer that is
// double-buffered by iteration parity instead of inside the 16-byte pixel records.  4.70 us per iteration at config 1
// against 5.15 us for the general kernel.
// Tried here and dropped: a ONE-barrier mode for sparse iterates, in which every pixel-owning CTA recomputes the whole
// residual itself (nnz * n_vis sincos per CTA; 13 non-zero pixels at config 1) instead of receiving it from the
// visibility owners -- 5.56 us: at 8 warps per SM the recomputation is a latency chain longer than the barrier it saves.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(PT, 1) fista_persistent_small_kernel(const PersistParams P) {
    __shared__ __align__(16) float4 s_list[PW][PBLK];       // compacted non-zero pixels, per warp
    __shared__ uint16_t s_tile[PW][PBLK];
    __shared__ __align__(16) float s_x0[4][PG];              // centre phases of the CTA's phase-A item (<= 4 tiles)
    __shared__ float s_red[PW][PG * 2 + 1];
    __shared__ int s_stop;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int G = gridDim.x, cta = blockIdx.x;
    unsigned bar_target = 0;
    const int items_a = (P.n_vis + P.nvg - 1) / P.nvg, items_b = P.n_pix_pad / P.npg;
    const bool has_a = cta < items_a, has_b = cta < items_b;
    const int tracer = G - 1;                                // idle in both phases (host-side condition)
    double E_prev = 0.0, N_prev = 0.0;

    // ---- iteration-invariant operands
    const int j0 = cta * P.nvg, p0 = cta * P.npg;
    float uf[PG], vf[PG], wf[PG];
    float2 Vj = make_float2(0.f, 0.f);
    if (has_a) {
        for (int i = tid; i < P.n_tiles * PG; i += PT) {
            const int tl = i / PG, r = i - tl * PG;
            s_x0[tl][r] = __ldg(P.x0 + (size_t)tl * P.n_vis + min(j0 + r, P.n_vis - 1));
        }
#pragma unroll
        for (int r = 0; r < PG; ++r) {
            const float4 v4 = __ldg(P.vis4 + min(j0 + r, P.n_vis - 1));
            uf[r] = v4.x;
            vf[r] = v4.y;
            wf[r] = v4.z;
        }
        if (tid < 2 * P.nvg && (tid & 1) == 0 && j0 + (tid >> 1) < P.n_vis) Vj = __ldg(P.V + j0 + (tid >> 1));
    }
    float3 pxc[PBLK / 32];                                   // (dl, dm, dn') of the pixels this thread reads every iteration
#pragma unroll
    for (int q = 0; q < PBLK / 32; ++q) {
        const int kpx = warp * PBLK + q * 32 + lane;
        const float4 px = (kpx < P.n_pix_pad) ? __ldcg(P.pix4 + kpx) : make_float4(0.f, 0.f, 0.f, 0.f);
        pxc[q] = make_float3(px.x, px.y, px.z);
    }
    float dl[PG], dm[PG], dn[PG], a_own = 0.f, y_own = 0.f, I_own = 0.f, x0v[4];
    float4 v4r[4];
    {
        const float *x0row = P.x0 + (size_t)(min(p0, P.n_pix_pad - 1) / TP) * P.n_vis;
#pragma unroll
        for (int i = 0; i < PG; ++i) {
            const float4 px = __ldcg(P.pix4 + min(p0 + i, P.n_pix_pad - 1));
            dl[i] = px.x;
            dm[i] = px.y;
            dn[i] = px.z;
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int j = min(tid + q * PT, P.n_vis - 1);
            v4r[q] = __ldg(P.vis4 + j);
            x0v[q] = __ldg(x0row + j);
        }
        if (has_b && tid < P.npg) {
            a_own = __ldg(P.amp + p0 + tid);
            y_own = P.y_sorted[p0 + tid];
            I_own = P.I_sorted[p0 + tid];
            P.ybuf[(size_t)((P.k0 + 1) & 1) * P.n_pix_pad + p0 + tid] = a_own * y_own;   // a*y of this launch's first iteration
        }
    }
    grid_barrier(P.bar, bar_target);                         // the first iteration's a*y is in place

    for (int it = 0; it < P.n_iter; ++it) {
        const int k = P.k0 + it + 1;
        double *part = P.part + (size_t)(k & 1) * 3 * G;
        const float *ycur = P.ybuf + (size_t)(k & 1) * P.n_pix_pad;
        float *ynext = P.ybuf + (size_t)((k + 1) & 1) * P.n_pix_pad;
        const float beta = __ldg(P.beta + it);
        // ---- read a*y_k, compact the non-zeros of the warp's block
        int cnt = 0;
        {
            float wq[PBLK / 32];
#pragma unroll
            for (int q = 0; q < PBLK / 32; ++q) {
                const int kpx = warp * PBLK + q * 32 + lane;
                wq[q] = (kpx < P.n_pix_pad) ? __ldcg(ycur + kpx) : 0.f;
            }
#pragma unroll
            for (int q = 0; q < PBLK / 32; ++q) {
                const bool nz = wq[q] != 0.f;                // NaN counts as non-zero and propagates
                const unsigned b = __ballot_sync(0xffffffffu, nz);
                if (nz) {
                    const int pos = cnt + __popc(b & ((1u << lane) - 1u));
                    s_list[warp][pos] = make_float4(pxc[q].x, pxc[q].y, pxc[q].z, wq[q]);
                    s_tile[warp][pos] = (uint16_t)((warp * PBLK + q * 32 + lane) / TP);
                }
                cnt += __popc(b);
            }
        }
        __syncwarp();
        float2 rp[4];                                        // residual of the thread's visibilities, polar
        double r2 = 0.0;
        {
            // ---- phase A: the CTA's <= 8 visibilities against every non-zero pixel (each warp: its own compacted block)
            if (has_a) {
                float acc[2 * PG];
#pragma unroll
                for (int r = 0; r < 2 * PG; ++r) acc[r] = 0.f;
                for (int i = lane; i < cnt; i += 32) {
                    const float4 px = s_list[warp][i];
                    const float4 *x0q = reinterpret_cast<const float4 *>(s_x0[s_tile[warp][i]]);
                    const float4 xa = x0q[0], xb = x0q[1];
                    const float x0r[PG] = {xa.x, xa.y, xa.z, xa.w, xb.x, xb.y, xb.z, xb.w};
#pragma unroll
                    for (int r = 0; r < PG; ++r) {
                        if (r < P.nvg) {
                            const float X = fmaf(uf[r], px.x, fmaf(vf[r], px.y, fmaf(wf[r], px.z, x0r[r])));
                            float sn, cs;
                            __sincosf(X, &sn, &cs);
                            acc[2 * r] = fmaf(px.w, cs, acc[2 * r]);
                            acc[2 * r + 1] = fmaf(-px.w, sn, acc[2 * r + 1]);
                        }
                    }
                }
                const float sum = cta_sum<2 * PG>(acc, s_red);
                const float other = __shfl_down_sync(0xffffffffu, sum, 1);
                if (tid < 2 * P.nvg && (tid & 1) == 0 && j0 + (tid >> 1) < P.n_vis) {
                    const float re = sum - Vj.x, im = other - Vj.y;
                    P.rpol[j0 + (tid >> 1)] = make_float2(sqrtf(fmaf(re, re, im * im)), atan2f(im, re));
                    r2 = (double)re * re + (double)im * im;
                }
            }
            if (tid < 32) {
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) r2 += __shfl_xor_sync(0xffffffffu, r2, o);
                if (tid == 0) part[cta] = r2;
            }
            grid_barrier(P.bar, bar_target);
            if (has_b) {
#pragma unroll
                for (int q = 0; q < 4; ++q)
                    rp[q] = (tid + q * PT < P.n_vis) ? __ldcg(P.rpol + tid + q * PT) : make_float2(0.f, 0.f);
            }
        }
        // ---- phase B: g = Re M^H r on the CTA's pixels, gradient step, T^{lambda/L}, momentum
        double l1 = 0.0, nzs = 0.0;
        if (has_b) {
            float acc[PG];
#pragma unroll
            for (int i = 0; i < PG; ++i) acc[i] = 0.f;
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const float ph = x0v[q] + rp[q].y;
#pragma unroll
                for (int i = 0; i < PG; ++i) {
                    if (i < P.npg) {
                        const float X = fmaf(v4r[q].x, dl[i], fmaf(v4r[q].y, dm[i], fmaf(v4r[q].z, dn[i], ph)));
                        acc[i] = fmaf(rp[q].x, __cosf(X), acc[i]);
                    }
                }
            }
            const float gsum = cta_sum<PG>(acc, s_red);
            if (tid < P.npg) {
                const float g = gsum * a_own;
                const float z = fmaf(-P.inv_L, g, y_own);
                const float I_new = (z > P.thr) ? z - P.thr : 0.f;
                const float y_new = fmaf(beta, I_new - I_own, I_new);
                I_own = I_new;
                y_own = y_new;
                ynext[p0 + tid] = a_own * y_new;
                l1 = (double)I_new;
                nzs = (I_new != 0.f) ? 1.0 : 0.0;
            }
        }
        if (tid < 32) {
#pragma unroll
            for (int o = 4; o > 0; o >>= 1) {                // lanes 0..7 hold terms
                l1 += __shfl_xor_sync(0xffffffffu, l1, o);
                nzs += __shfl_xor_sync(0xffffffffu, nzs, o);
            }
            if (tid == 0) {
                part[G + cta] = l1;
                part[2 * G + cta] = nzs;
            }
        }
        grid_barrier(P.bar, bar_target);
        // ---- a6 on the idle CTA (trace row) and, at looked-at iterations, the stopping rules in every CTA
        const bool look = P.check_every > 0 && k >= 2 && (k % P.check_every) == 0;
        const bool before_look = P.check_every > 0 && ((k + 1) % P.check_every) == 0;
        if (look || before_look || (P.trace && cta == tracer)) {
            if (warp == 0) {
                double l2s, l1s, nz3;
                warp_sum3_cg(part, G, l2s, l1s, nz3);
                if (lane == 0) {
                    if (P.trace && cta == tracer) {
                        P.trace[3 * (size_t)it] = l2s;
                        P.trace[3 * (size_t)it + 1] = l1s;
                        P.trace[3 * (size_t)it + 2] = nz3;
                    }
                    const double E = l2s + P.lam2 * l1s;
                    int stop = 0;
                    if (look)
                        stop = (P.tol >= 0.0 && fabs(E - E_prev) <= P.tol * fabs(E)) ||
                               (P.nnz_tol >= 0.0 && fabs(nz3 - N_prev) <= P.nnz_tol * nz3);
                    E_prev = E;
                    N_prev = nz3;
                    s_stop = stop;
                    if (stop && cta == 0) {
                        P.ctl[0] = 1;
                        P.ctl[1] = k;
                        P.ctl[2] = 1;
                    }
                }
            }
            if (P.check_every > 0) {
                __syncthreads();
                if (s_stop) break;
                __syncthreads();
            }
        }
    }
    // ---- the state goes back to global memory (next launch, sl1m_fista_image, the other kernels)
    if (has_b && tid < P.npg) {
        P.I_sorted[p0 + tid] = I_own;
        P.y_sorted[p0 + tid] = y_own;
        P.pix4[p0 + tid].w = a_own * y_own;
    }
}

// ------------------------------------------------------------------------------------------
// a7 for the same small problems: n_iter rounds of the power iteration x <- g / ||g||, g = Re M^H (M x), in one
// cooperative launch (the multi-launch version is 6 launches per round: for config 1, 30 rounds cost more than a
// 100-iteration solve).  Same two phases and barriers as the FISTA kernel.  The normalisation needs ||g|| of the whole
// image: phase B leaves a*g UNNORMALISED in the pixel tiles plus one fp64 partial of sum g^2 per CTA, and phase A of the
// next round divides by the norm while it reads the tiles -- no third barrier.  out_norm2 = sum g^2 of the last round
// (L = its square root, as sl1m_max_eig defines it).  P.pix4.w must hold a*x_0 on entry.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(PT, 1) power_persistent_kernel(const PersistParams P, double *out_norm2) {
    __shared__ __align__(16) float4 s_list[PW][PBLK];
    __shared__ uint16_t s_tile[PW][PBLK];
    __shared__ __align__(16) float s_x0[PERSIST_MAX_TILES][PG];
    __shared__ float s_red[PW][PG * 2 + 1];
    __shared__ float s_inv;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int G = gridDim.x;
    unsigned bar_target = 0;
    const int items_a = (P.n_vis + P.nvg - 1) / P.nvg;
    const int items_b = P.n_pix_pad / P.npg;
    int staged_item = -1;

    for (int it = 0; it < P.n_iter; ++it) {
        // 1 / ||g|| of the previous round, from the per-CTA partials (every CTA forms the same number)
        if (warp == 0) {
            double v = 0.0;
            if (it > 0) {
                const double *prev = P.part + (size_t)((it - 1) & 1) * G;
                for (int i = lane; i < G; i += 32) v += __ldcg(prev + i);
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            }
            if (lane == 0) s_inv = (it > 0) ? ((v > 0.0) ? (float)(1.0 / sqrt(v)) : 0.f) : 1.f;
        }
        __syncthreads();
        const float inv = s_inv;
        // ---- phase A: v = M x  (left in polar form for phase B)
        for (int item = blockIdx.x; item < items_a; item += G) {
            const int j0 = item * P.nvg;
            if (staged_item != item) {
                __syncthreads();
                for (int i = tid; i < P.n_tiles * PG; i += PT) {
                    const int tl = i / PG, r = i - tl * PG, j = min(j0 + r, P.n_vis - 1);
                    s_x0[tl][r] = __ldg(P.x0 + (size_t)tl * P.n_vis + j);
                }
                __syncthreads();
                staged_item = (items_a <= G) ? item : -1;
            }
            float uf[PG], vf[PG], wf[PG], acc[2 * PG];
#pragma unroll
            for (int r = 0; r < PG; ++r) {
                const float4 v4 = __ldg(P.vis4 + min(j0 + r, P.n_vis - 1));
                uf[r] = v4.x;
                vf[r] = v4.y;
                wf[r] = v4.z;
                acc[2 * r] = 0.f;
                acc[2 * r + 1] = 0.f;
            }
            for (int base = warp * PBLK; base < P.n_pix_pad; base += PW * PBLK) {
                int cnt = 0;
                float4 pxq[PBLK / 32];
#pragma unroll
                for (int q = 0; q < PBLK / 32; ++q) pxq[q] = __ldcg(P.pix4 + base + q * 32 + lane);
#pragma unroll
                for (int q = 0; q < PBLK / 32; ++q) {
                    const int kpx = base + q * 32 + lane;
                    float4 px = pxq[q];
                    px.w *= inv;
                    const bool nz = px.w != 0.f;
                    const unsigned b = __ballot_sync(0xffffffffu, nz);
                    if (nz) {
                        const int pos = cnt + __popc(b & ((1u << lane) - 1u));
                        s_list[warp][pos] = px;
                        s_tile[warp][pos] = (uint16_t)(kpx / TP);
                    }
                    cnt += __popc(b);
                }
                __syncwarp();
                for (int i = lane; i < cnt; i += 32) {
                    const float4 px = s_list[warp][i];
                    const float4 *x0q = reinterpret_cast<const float4 *>(s_x0[s_tile[warp][i]]);
                    const float4 xa = x0q[0], xb = x0q[1];
                    const float x0r[PG] = {xa.x, xa.y, xa.z, xa.w, xb.x, xb.y, xb.z, xb.w};
#pragma unroll
                    for (int r = 0; r < PG; ++r) {
                        if (r < P.nvg) {
                            const float X = fmaf(uf[r], px.x, fmaf(vf[r], px.y, fmaf(wf[r], px.z, x0r[r])));
                            float sn, cs;
                            __sincosf(X, &sn, &cs);
                            acc[2 * r] = fmaf(px.w, cs, acc[2 * r]);
                            acc[2 * r + 1] = fmaf(-px.w, sn, acc[2 * r + 1]);
                        }
                    }
                }
                __syncwarp();
            }
            const float sum = cta_sum<2 * PG>(acc, s_red);
            const float other = __shfl_down_sync(0xffffffffu, sum, 1);
            if (tid < 2 * P.nvg && (tid & 1) == 0 && j0 + (tid >> 1) < P.n_vis)
                P.rpol[j0 + (tid >> 1)] = make_float2(sqrtf(fmaf(sum, sum, other * other)), atan2f(other, sum));
        }
        grid_barrier(P.bar, bar_target);
        // ---- phase B: g = Re M^H v; the tiles receive a*g, the partial sum g^2
        double g2 = 0.0;
        for (int item = blockIdx.x; item < items_b; item += G) {
            const int p0 = item * P.npg;
            const float *x0row = P.x0 + (size_t)(p0 / TP) * P.n_vis;
            float dl[PG], dm[PG], dn[PG], acc[PG];
#pragma unroll
            for (int i = 0; i < PG; ++i) {
                const float4 px = __ldcg(P.pix4 + min(p0 + i, P.n_pix_pad - 1));
                dl[i] = px.x;
                dm[i] = px.y;
                dn[i] = px.z;
                acc[i] = 0.f;
            }
            for (int j = tid; j < P.n_vis; j += PT) {
                const float4 v4 = __ldg(P.vis4 + j);
                const float2 rp = __ldcg(P.rpol + j);
                const float ph = __ldg(x0row + j) + rp.y;
#pragma unroll
                for (int i = 0; i < PG; ++i) {
                    if (i < P.npg) {
                        const float X = fmaf(v4.x, dl[i], fmaf(v4.y, dm[i], fmaf(v4.z, dn[i], ph)));
                        acc[i] = fmaf(rp.x, __cosf(X), acc[i]);
                    }
                }
            }
            const float gsum = cta_sum<PG>(acc, s_red);
            if (tid < P.npg) {
                const float a = __ldg(P.amp + p0 + tid);
                const float g = gsum * a;
                P.pix4[p0 + tid].w = a * g;
                if (P.y_sorted) P.y_sorted[p0 + tid] = g;          // the last round's g, for callers that want the vector
                g2 += (double)g * g;
            }
        }
        if (tid < 32) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) g2 += __shfl_xor_sync(0xffffffffu, g2, o);
            if (tid == 0) P.part[(size_t)(it & 1) * G + blockIdx.x] = g2;
        }
        grid_barrier(P.bar, bar_target);
    }
    if (blockIdx.x == 0 && warp == 0) {
        double v = 0.0;
        const double *last = P.part + (size_t)((P.n_iter - 1) & 1) * G;
        for (int i = lane; i < G; i += 32) v += __ldcg(last + i);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) *out_norm2 = v;
    }
}

// Plan-time tables of the persistent kernel: vis4[j] = 2 pi (u, v, w) as floats, x0[t][j] = centre phase (fp64, reduced).
__global__ void __launch_bounds__(256) persist_tables_kernel(const double *u64, const double *v64, const double *w64,
                                                             const double4 *cen, int n_vis, int n_tiles, float4 *vis4,
                                                             float *x0) {
    const int j = blockIdx.x * 256 + threadIdx.x;
    if (j >= n_vis) return;
    const double u = u64[j], v = v64[j], w = w64[j];
    if (blockIdx.y == 0) vis4[j] = make_float4((float)(TWO_PI * u), (float)(TWO_PI * v), (float)(TWO_PI * w), 0.f);
    for (int t = blockIdx.y; t < n_tiles; t += gridDim.y) x0[(size_t)t * n_vis + j] = centre_phase(u, v, w, cen[t]);
}

}  // namespace sl1m
