// sl1m_epilogue.cuh -- the O(N) kernels around the two applies: packing a*x into the pixel tiles,
// fixed-order reduction of the split partials, the fused FISTA update (steps a3-a6 of
// SURVEY.md 8(a); listing PAPER.md:188-192, eq (18)) and power-iteration helpers.
// Every reduction runs in a fixed order (no float atomics), so results are bit-stable run to run.
#pragma once
#include "sl1m_kernels.cuh"

namespace sl1m {

constexpr int ET = 256;  // threads per CTA in the epilogue kernels

// Block-wide sum in fp64 (warp shuffles, then one warp over the per-warp partials).
__device__ __forceinline__ double block_sum(double v) {
    __shared__ double s_part[ET / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    __syncthreads();  // protect s_part across successive calls
    if (lane == 0) s_part[warp] = v;
    __syncthreads();
    double t = (threadIdx.x < ET / 32) ? s_part[threadIdx.x] : 0.0;
    if (warp == 0) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    }
    return t;  // valid in thread 0
}

// Zero-skipping forward.  A CTA of the packing kernels (ET == TP threads) holds exactly
// tile blockIdx.x.  The entries with a*x != 0 move to the front of the COMPACT copy of the tile in their
// original order, padded with a*x = 0 entries to a multiple of 4; zs.cnt[c][tile] = the padded count.  The
// forward kernels stream only that many pixels of the tile: the skipped terms are exactly zero.
// Plans with a gain table: the forward-layout gain rows gF[k][.] of the compact entries are copied next to them
// (gFc, same tile layout), so the kernels keep walking consecutive rows; a full tile is not copied (the kernels
// read gF for it).  A dense image therefore costs nothing extra, a sparse one n_ant * 8 B per non-zero pixel.
struct ZeroSkip {
    float4 *pixc;        // DEV [n_chan][n_pix_pad] compact tiles, NULL = off (per-pixel sigma, fp64 phase)
    int *cnt;            // DEV [n_chan][n_tiles]
    const float2 *gF;    // DEV [n_pix_pad][n_ant] or NULL (unit gains)
    float2 *gFc;         // DEV [n_chan][n_pix_pad][n_ant]
    int n_ant;
    // per-pixel side arrays of the kernels that stage one next to the pixel tile: compacted with it
    const double4 *pixd; // DEV [n_pix_pad] fp64 offsets (fp64-phase plans) or NULL
    double4 *pixdc;      // DEV [n_chan][n_pix_pad]
    const float2 *pixg;  // DEV [n_pix_pad] (sigma^2, -pi log2(e) sigma^2) (per-pixel-sigma plans) or NULL
    float2 *pixgc;       // DEV [n_chan][n_pix_pad]
    // packed gain forward (fwd_kernel_x2<GAINS>): it reads the ANTENNA-MAJOR table, so the compact gains are kept
    // in that layout too (gAc set => gFc unused)
    const float2 *gA;    // DEV [n_ant][n_pix_pad]
    float2 *gAc;         // DEV [n_chan][n_ant][n_pix_pad] or NULL
};
static_assert(ET == TP, "one packing CTA per pixel tile");
__device__ __forceinline__ void compact_tile(const ZeroSkip zs, size_t chan, int n_pix_pad, float4 v) {
    if (!zs.pixc) return;                                // uniform over the grid
    __shared__ int s_wcnt[ET / 32];
    __shared__ uint8_t s_src[ET];                        // original in-tile index of compact entry p (gain rows)
    const bool nz = (v.w != 0.f);                        // NaN counts as non-zero: it propagates as in the dense path
    const unsigned b = __ballot_sync(0xffffffffu, nz);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) s_wcnt[warp] = __popc(b);
    __syncthreads();
    int base = 0, total = 0;
#pragma unroll
    for (int w = 0; w < ET / 32; ++w) {
        const int c = s_wcnt[w];
        base += (w < warp) ? c : 0;
        total += c;
    }
    float4 *tile = zs.pixc + chan * n_pix_pad + (size_t)blockIdx.x * TP;
    const int cnt4 = (total + 3) & ~3;
    const size_t k_own = (size_t)blockIdx.x * TP + threadIdx.x, side0 = chan * n_pix_pad + (size_t)blockIdx.x * TP;
    if (cnt4 == TP) {                                    // (nearly) full: keep the ORIGINAL order -- the gain kernels read
        tile[threadIdx.x] = v;                           // the rows of a tile with TP entries from the table itself
        if (zs.pixdc) zs.pixdc[side0 + threadIdx.x] = zs.pixd[k_own];
        if (zs.pixgc) zs.pixgc[side0 + threadIdx.x] = zs.pixg[k_own];
        if (threadIdx.x == 0) zs.cnt[chan * (size_t)(n_pix_pad / TP) + blockIdx.x] = TP;
        return;                                          // uniform over the CTA
    }
    if (nz) {
        const int pos = base + __popc(b & ((1u << lane) - 1u));
        tile[pos] = v;
        s_src[pos] = (uint8_t)threadIdx.x;
        if (zs.pixdc) zs.pixdc[side0 + pos] = zs.pixd[k_own];
        if (zs.pixgc) zs.pixgc[side0 + pos] = zs.pixg[k_own];
    }
    if ((int)threadIdx.x < cnt4 - total) {               // padding entries: a*x = 0 and finite side values
        tile[total + threadIdx.x] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (zs.pixdc) zs.pixdc[side0 + total + threadIdx.x] = make_double4(0.0, 0.0, 0.0, 0.0);
        if (zs.pixgc) zs.pixgc[side0 + total + threadIdx.x] = make_float2(0.f, 0.f);
    }
    if (threadIdx.x == 0) zs.cnt[chan * (size_t)(n_pix_pad / TP) + blockIdx.x] = cnt4;
    if (zs.gAc && total > 0) {                           // antenna-major: row a of the tile, compact entries in order
        __syncthreads();
        const size_t t0 = (size_t)blockIdx.x * TP;
        const float2 *src = zs.gA + t0;
        float2 *dst = zs.gAc + chan * (size_t)zs.n_ant * n_pix_pad + t0;
        const int n = cnt4 * zs.n_ant;
        for (int i = threadIdx.x; i < n; i += ET) {
            const int a = i / cnt4, pos = i - a * cnt4;
            dst[(size_t)a * n_pix_pad + pos] = src[(size_t)a * n_pix_pad + s_src[min(pos, total - 1)]];
        }
    } else if (zs.gF && total > 0) {                     // gain rows of the compact entries (padding: a*x = 0, any row)
        __syncthreads();
        const size_t row0 = (size_t)blockIdx.x * TP;
        const float2 *src = zs.gF + row0 * zs.n_ant;
        float2 *dst = zs.gFc + (chan * n_pix_pad + row0) * zs.n_ant;
        const int n = cnt4 * zs.n_ant;
        for (int i = threadIdx.x; i < n; i += ET) {
            const int row = i / zs.n_ant, a = i - row * zs.n_ant;
            dst[i] = src[(size_t)s_src[min(row, total - 1)] * zs.n_ant + a];
        }
    }
}

// pix4[k].w = a_k * x[perm[k]]   (caller order -> sorted, padded pixels get 0)
__global__ void __launch_bounds__(ET) pack_caller_kernel(float4 *pix4, const float *amp, const int *perm,
                                                         const float *x, int n_pix_pad, int n_pix, ZeroSkip zs) {
    const int k = blockIdx.x * ET + threadIdx.x;         // n_pix_pad is a multiple of ET: no ragged CTA
    pix4 += (size_t)blockIdx.y * n_pix_pad;   // blockIdx.y = channel (NEXT-4); caller arrays are [n_chan][n_pix]
    x += (size_t)blockIdx.y * n_pix;
    const int src = perm[k];
    float4 v = pix4[k];
    v.w = (src >= 0) ? amp[k] * x[src] : 0.f;
    pix4[k].w = v.w;
    compact_tile(zs, blockIdx.y, n_pix_pad, v);
}

// sorted[k] = caller[perm[k]] (0 on padding)
__global__ void __launch_bounds__(ET) gather_kernel(const float *caller, const int *perm, float *sorted,
                                                    int n_pix_pad, int n_pix) {
    const int k = blockIdx.x * ET + threadIdx.x;
    if (k >= n_pix_pad) return;
    caller += (size_t)blockIdx.y * n_pix;
    sorted += (size_t)blockIdx.y * n_pix_pad;
    const int src = perm[k];
    sorted[k] = (src >= 0) ? caller[src] : 0.f;
}

// caller[perm[k]] = sorted[k]
__global__ void __launch_bounds__(ET) scatter_kernel(const float *sorted, const int *perm, float *caller,
                                                     int n_pix_pad, int n_pix) {
    const int k = blockIdx.x * ET + threadIdx.x;
    if (k >= n_pix_pad) return;
    caller += (size_t)blockIdx.y * n_pix;
    sorted += (size_t)blockIdx.y * n_pix_pad;
    const int dst = perm[k];
    if (dst >= 0) caller[dst] = sorted[k];
}

// pix4[k].w = a_k * xs[k]  (sorted order in)
__global__ void __launch_bounds__(ET) pack_sorted_kernel(float4 *pix4, const float *amp, const float *xs,
                                                         int n_pix_pad, ZeroSkip zs) {
    const int k = blockIdx.x * ET + threadIdx.x;
    pix4 += (size_t)blockIdx.y * n_pix_pad;
    xs += (size_t)blockIdx.y * n_pix_pad;
    float4 v = pix4[k];
    v.w = amp[k] * xs[k];
    pix4[k].w = v.w;
    compact_tile(zs, blockIdx.y, n_pix_pad, v);
}

__global__ void __launch_bounds__(ET) fill_kernel(float *p, float v, const int *perm, int n_pix_pad) {
    const int k = blockIdx.x * ET + threadIdx.x;
    p += (size_t)blockIdx.y * n_pix_pad;
    if (k < n_pix_pad) p[k] = (perm[k] >= 0) ? v : 0.f;
}

// Forward epilogue (a3): value[js] = sum_s ws[s][js] - V[caller(js)] over INTERNAL positions js;
// written to out[js] (internal order, solver residual) or out[caller(js)] (caller order, API
// output).  vperm maps internal -> caller (-1 = padding, value forced to 0); NULL = identity.
// part[block] = sum |value|^2 (fp64).
__global__ void __launch_bounds__(ET) fwd_reduce_kernel(const float2 *ws, int n_split, int n_int,
                                                        const int *vperm, const float2 *V, float2 *out,
                                                        int out_internal, double *part, int n_vis, int n_part,
                                                        const int *done = nullptr) {
    if (done && done[blockIdx.y]) return;                // channel stopped (sl1m_solve_stop)
    const int js = blockIdx.x * ET + threadIdx.x;
    double sq = 0.0;
    ws += (size_t)blockIdx.y * n_split * n_int;          // blockIdx.y = channel
    if (V) V += (size_t)blockIdx.y * n_vis;
    out += (size_t)blockIdx.y * (out_internal ? n_int : n_vis);
    if (part) part += (size_t)blockIdx.y * n_part;
    if (js < n_int) {
        const int jc = vperm ? vperm[js] : js;
        float re = 0.f, im = 0.f;
        if (jc >= 0) {
            for (int s = 0; s < n_split; ++s) {
                const float2 a = ws[(size_t)s * n_int + js];
                re += a.x;
                im += a.y;
            }
            if (V) {
                const float2 v = V[jc];
                re -= v.x;
                im -= v.y;
            }
        }
        if (out_internal) out[js] = make_float2(re, im);
        else if (jc >= 0) out[jc] = make_float2(re, im);
        sq = (double)re * re + (double)im * im;
    }
    if (part) {
        const double t = block_sum(sq);
        if (threadIdx.x == 0) part[blockIdx.x] = t;
    }
}

// internal[js] = caller[vperm[js]] (0 on padding): brings an API residual into the internal order.
__global__ void __launch_bounds__(ET) vis_gather_kernel(const float2 *caller, const int *vperm, float2 *internal,
                                                        int n_int, int n_vis) {
    const int js = blockIdx.x * ET + threadIdx.x;
    if (js >= n_int) return;
    caller += (size_t)blockIdx.y * n_vis;
    internal += (size_t)blockIdx.y * n_int;
    const int jc = vperm[js];
    internal[js] = (jc >= 0) ? caller[jc] : make_float2(0.f, 0.f);
}

// Residual in polar form for the one-cosine adjoint kernels: rp[j] = (|r_j|, arg r_j), evaluated in fp64.
// Re(e^{iX} r) = |r| cos(X + arg r) (the image is real, reading C3).
__global__ void __launch_bounds__(ET) vis_polar_kernel(const float2 *r, float2 *rp, int n_int,
                                                       const int *done = nullptr) {
    if (done && done[blockIdx.y]) return;
    const int js = blockIdx.x * ET + threadIdx.x;
    if (js >= n_int) return;
    r += (size_t)blockIdx.y * n_int;                     // blockIdx.y = channel
    rp += (size_t)blockIdx.y * n_int;
    const float2 v = r[js];
    const double re = (double)v.x, im = (double)v.y;
    rp[js] = make_float2((float)sqrt(re * re + im * im), (float)atan2(im, re));
}

// Adjoint epilogue: g_k = a_k sum_s ws[s][k]; scattered to the caller's order and/or kept sorted.
__global__ void __launch_bounds__(ET) adj_reduce_kernel(const float *ws, int n_split, int n_pix_pad,
                                                        const float *amp, const int *perm, float *img_caller,
                                                        float *g_sorted, double *part, int n_pix, int n_part) {
    const int k = blockIdx.x * ET + threadIdx.x;
    double sq = 0.0;
    ws += (size_t)blockIdx.y * n_split * n_pix_pad;      // blockIdx.y = channel
    if (img_caller) img_caller += (size_t)blockIdx.y * n_pix;
    if (g_sorted) g_sorted += (size_t)blockIdx.y * n_pix_pad;
    if (part) part += (size_t)blockIdx.y * n_part;
    if (k < n_pix_pad) {
        float g = 0.f;
        for (int s = 0; s < n_split; ++s) g += ws[(size_t)s * n_pix_pad + k];
        g *= amp[k];
        const int dst = perm[k];
        if (img_caller && dst >= 0) img_caller[dst] = g;
        if (g_sorted) g_sorted[k] = g;
        sq = (double)g * g;
    }
    if (part) {
        const double t = block_sum(sq);
        if (threadIdx.x == 0) part[blockIdx.x] = t;
    }
}

// Fused FISTA update (a4 + a5 + a6):  g = a sum_s ws;  z = y - g/L;  I = T^{thr}(z) (eq 18);
// y' = I + beta (I - I_old);  writes I, y', a*y' into the pixel tiles, and block partials of
// sum I and nnz I.
__global__ void __launch_bounds__(ET) fista_update_kernel(const float *ws, int n_split, int n_pix_pad,
                                                          const float *amp, float4 *pix4, float *I_sorted,
                                                          float *y_sorted, float inv_L, float thr, float beta,
                                                          double *part_l1, double *part_nnz,
                                                          const float2 *step_c, int n_part, ZeroSkip zs,
                                                          const int *done = nullptr) {
    if (done && done[blockIdx.y]) return;                // channel stopped: I, y and the packed tiles stay as they are
    const int k = blockIdx.x * ET + threadIdx.x;
    double l1 = 0.0, nz = 0.0;
    float4 pv = make_float4(0.f, 0.f, 0.f, 0.f);
    const int c = blockIdx.y;                            // channel; step_c[c] = (1/L_c, lambda_c/L_c) when batched
    ws += (size_t)c * n_split * n_pix_pad;
    pix4 += (size_t)c * n_pix_pad;
    I_sorted += (size_t)c * n_pix_pad;
    y_sorted += (size_t)c * n_pix_pad;
    if (step_c) {
        inv_L = step_c[c].x;
        thr = step_c[c].y;
    }
    if (part_l1) {
        part_l1 += (size_t)c * n_part;
        part_nnz += (size_t)c * n_part;
    }
    if (k < n_pix_pad) {
        float g = 0.f;
        for (int s = 0; s < n_split; ++s) g += ws[(size_t)s * n_pix_pad + k];
        const float a = amp[k];
        g *= a;
        const float y = y_sorted[k];
        const float z = fmaf(-inv_L, g, y);
        const float I_new = (z > thr) ? z - thr : 0.f;
        const float I_old = I_sorted[k];
        const float y_new = fmaf(beta, I_new - I_old, I_new);
        I_sorted[k] = I_new;
        y_sorted[k] = y_new;
        pv = pix4[k];
        pv.w = a * y_new;
        pix4[k].w = pv.w;
        l1 = I_new;
        nz = (I_new != 0.f) ? 1.0 : 0.0;
    }
    compact_tile(zs, c, n_pix_pad, pv);
    if (part_l1) {
        const double t1 = block_sum(l1);
        const double t2 = block_sum(nz);
        if (threadIdx.x == 0) {
            part_l1[blockIdx.x] = t1;
            part_nnz[blockIdx.x] = t2;
        }
    }
}

// out[i] = sum of n partials of array i, i < n_arrays (single CTA, fixed order).
__global__ void __launch_bounds__(ET) sum_partials_kernel(const double *p0, const double *p1, const double *p2,
                                                          int n0, int n1, int n2, double *out0, double *out1,
                                                          double *out2, int n_part, size_t out_stride,
                                                          const int *done = nullptr) {
    if (done && done[blockIdx.x]) return;
    const double *ps[3] = {p0, p1, p2};
    const int ns[3] = {n0, n1, n2};
    double *outs[3] = {out0, out1, out2};
    const size_t c = blockIdx.x;                         // one CTA per channel
    for (int a = 0; a < 3; ++a) {
        if (!ps[a] || !outs[a]) continue;
        double v = 0.0;
        for (int i = threadIdx.x; i < ns[a]; i += ET) v += ps[a][c * n_part + i];
        const double t = block_sum(v);
        if (threadIdx.x == 0) outs[a][c * out_stride] = t;
    }
}

// Termination rules of PAPER.md:194 evaluated ON THE DEVICE after iteration k (1-based; k >= 2), from the trace rows
// the iteration has just written (readings R21, R24):
//   E rule    |E_k - E_{k-1}| <= tol |E_k|,   E_k = ||M y_k - V||^2 + 2 lambda sum I_k        (tol < 0: off)
//   nnz rule  |N_k - N_{k-1}| <= nnz_tol N_k, N_k = nnz(I_k)                                 (nnz_tol < 0: off)
// A channel that meets either enabled rule gets done[c] = 1, n_done[c] = k; every later kernel of that channel
// returns at once.  ctl = {done[C], n_done[C], all_done}.  One CTA; channels strided over its threads.
__global__ void __launch_bounds__(ET) stop_rule_kernel(const double *trace, size_t trace_stride, int k, int n_chan,
                                                       const double *lam2, double tol, double nnz_tol, int *ctl) {
    int *done = ctl, *n_done = ctl + n_chan, *all_done = ctl + 2 * n_chan;
    int mine = 1;
    for (int c = threadIdx.x; c < n_chan; c += ET) {
        if (!done[c]) {
            const double *now = trace + c * trace_stride + 3 * (size_t)(k - 1), *bef = now - 3;
            const double E_now = now[0] + lam2[c] * now[1], E_bef = bef[0] + lam2[c] * bef[1];
            const bool stop = (tol >= 0.0 && fabs(E_now - E_bef) <= tol * fabs(E_now)) ||
                              (nnz_tol >= 0.0 && fabs(now[2] - bef[2]) <= nnz_tol * now[2]);
            if (stop) {
                done[c] = 1;
                n_done[c] = k;
            } else {
                mine = 0;
            }
        }
    }
    const int all = __syncthreads_and(mine);
    if (threadIdx.x == 0) *all_done = all;
}

// Power iteration (a7): x = g / ||g||, packed straight into the pixel tiles; norm2 on device.
__global__ void __launch_bounds__(ET) normalize_pack_kernel(const float *g_sorted, const double *norm2,
                                                            const float *amp, float4 *pix4, int n_pix_pad,
                                                            ZeroSkip zs) {
    const int k = blockIdx.x * ET + threadIdx.x;
    g_sorted += (size_t)blockIdx.y * n_pix_pad;
    pix4 += (size_t)blockIdx.y * n_pix_pad;
    norm2 += (size_t)blockIdx.y * 4;                     // scalars are [n_chan][4]
    const double nrm = sqrt(*norm2);
    const float x = (nrm > 0.0) ? (float)((double)g_sorted[k] / nrm) : 0.f;
    float4 v = pix4[k];
    v.w = amp[k] * x;
    pix4[k].w = v.w;
    compact_tile(zs, blockIdx.y, n_pix_pad, v);
}

// Gain table re-layout: raw [n_ant][n_pix] (re, im; caller order) -> gF [n_pix_pad][n_ant], gA [n_ant][n_pix_pad],
// both in polar form.
__global__ void __launch_bounds__(ET) gains_layout_kernel(const float2 *raw, int n_ant, int n_pix,
                                                          int n_pix_pad, const int *perm, float2 *gF,
                                                          float2 *gA) {
    const int k = blockIdx.x * ET + threadIdx.x;
    if (k >= n_pix_pad) return;
    const int src = perm[k];
    // polar form (|g|, arg g), evaluated in fp64: the kernels multiply the entry by |g_p||g_q| and shift its
    // phase by arg_p - arg_q (G = g_p conj(g_q)); a zero gain has amplitude 0 and phase 0
    for (int a = 0; a < n_ant; ++a) {
        float2 g = make_float2(0.f, 0.f);
        if (src >= 0) {
            const float2 c = raw[(size_t)a * n_pix + src];
            const double re = (double)c.x, im = (double)c.y;
            g = make_float2((float)sqrt(re * re + im * im), (float)atan2(im, re));
        }
        if (gF) gF[(size_t)k * n_ant + a] = g;
        gA[(size_t)a * n_pix_pad + k] = g;
    }
}

// Block partials of sum I and nnz I over a sorted image (for the final info struct).
__global__ void __launch_bounds__(ET) l1_nnz_kernel(const float *I_sorted, int n_pix_pad, double *part_l1,
                                                    double *part_nnz, int n_part) {
    const int k = blockIdx.x * ET + threadIdx.x;
    I_sorted += (size_t)blockIdx.y * n_pix_pad;
    part_l1 += (size_t)blockIdx.y * n_part;
    part_nnz += (size_t)blockIdx.y * n_part;
    const float v = (k < n_pix_pad) ? I_sorted[k] : 0.f;
    const double t1 = block_sum((double)v);
    const double t2 = block_sum(v != 0.f ? 1.0 : 0.0);
    if (threadIdx.x == 0) {
        part_l1[blockIdx.x] = t1;
        part_nnz[blockIdx.x] = t2;
    }
}

// Dirty image as a starting point (reading R22): img = max(0, scale * img).
__global__ void __launch_bounds__(ET) scale_clip_kernel(float *img, float scale, size_t n) {
    const size_t k = (size_t)blockIdx.x * ET + threadIdx.x;
    if (k < n) img[k] = fmaxf(0.f, scale * img[k]);
}

}  // namespace sl1m
