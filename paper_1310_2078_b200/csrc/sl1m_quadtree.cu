// sl1m_quadtree.cu -- NEXT-3 of SURVEY.md 8(f): the paper's coarse-to-fine / adaptive quadtree
// acceleration (section 4.5, Fig. 10) as a host-side driver over the C ABI:
// solve on the current pixel list, split the pixels where emission was found, warm-start the
// children from their parent, re-plan, repeat.  Every solve runs in the CUDA kernels behind
// sl1m_plan_create / sl1m_max_eig / sl1m_solve_tol; this file holds only the tree bookkeeping
// (reading R23) and has no arithmetic of the operator.
#include <cuda_runtime.h>

#include <chrono>
#include <cmath>
#include <new>
#include <vector>

#include "../../include/sl1m.h"
#include "sl1m_internal.h"

extern "C" int sl1m_quadtree_refine(int64_t n, const double *l, const double *m, const double *side, const float *I,
                                    double frac, double min_side, int64_t capacity, double *l_out, double *m_out,
                                    double *side_out, float *I0_out, int64_t *parent_out, int64_t *n_out,
                                    int64_t *n_refined) {
    if (!l || !m || !side || !I || !l_out || !m_out || !side_out || !I0_out || !n_out || !n_refined)
        return sl1m_fail(SL1M_ERR_NULL, "sl1m_quadtree_refine: NULL argument");
    if (n < 1 || capacity < n) return sl1m_fail(SL1M_ERR_SIZE, "sl1m_quadtree_refine: n < 1 or capacity < n");
    if (!std::isfinite(frac) || !std::isfinite(min_side)) return sl1m_fail(SL1M_ERR_PARAM, "sl1m_quadtree_refine: non-finite frac or min_side");
    double top = 0.0;
    for (int64_t k = 0; k < n; ++k) {
        if (!std::isfinite(I[k]) || !(side[k] > 0.0) || !std::isfinite(side[k]))
            return sl1m_fail(SL1M_ERR_DOMAIN, "sl1m_quadtree_refine: non-finite flux or side <= 0");
        if (k == 0 || (double)I[k] > top) top = (double)I[k];
    }
    const double thr = frac * top;
    // first pass: how many split (so that a too-small capacity fails before anything is written)
    int64_t n_split = 0;
    for (int64_t k = 0; k < n; ++k)
        if (top > 0.0 && (double)I[k] > thr && side[k] / 2.0 >= min_side) ++n_split;
    if (n + 3 * n_split > capacity) return sl1m_fail(SL1M_ERR_SIZE, "sl1m_quadtree_refine: capacity < n + 3 * (pixels that split)");
    int64_t o = 0;
    for (int64_t k = 0; k < n; ++k) {
        const double half = side[k] / 2.0;
        if (top > 0.0 && (double)I[k] > thr && half >= min_side) {
            const double q = side[k] / 4.0;
            const double dm[2] = {-q, +q}, dl[2] = {-q, +q};
            for (int a = 0; a < 2; ++a)
                for (int b = 0; b < 2; ++b) {        // l fastest, as in eqs (5)-(6)
                    l_out[o] = l[k] + dl[b];
                    m_out[o] = m[k] + dm[a];
                    side_out[o] = half;
                    I0_out[o] = I[k] / 4.0f;         // flux-conserving upscaling (exact in fp32)
                    if (parent_out) parent_out[o] = k;
                    ++o;
                }
        } else {
            l_out[o] = l[k];
            m_out[o] = m[k];
            side_out[o] = side[k];
            I0_out[o] = I[k];
            if (parent_out) parent_out[o] = k;
            ++o;
        }
    }
    *n_out = o;
    *n_refined = n_split;
    return SL1M_OK;
}

namespace {
struct DevBuf {
    void *p = nullptr;
    ~DevBuf() { if (p) cudaFree(p); }
    int alloc(size_t bytes) {
        if (p) cudaFree(p);
        p = nullptr;
        return cudaMalloc(&p, bytes ? bytes : 1) == cudaSuccess ? SL1M_OK : sl1m_fail(SL1M_ERR_ALLOC, "sl1m_quadtree_solve: device allocation failed");
    }
};
struct PlanGuard {
    sl1m_plan *p = nullptr;
    ~PlanGuard() { sl1m_destroy(p); }
};
}  // namespace

namespace {
// gains0: HOST [n_ant][n0][2] or NULL.  With a table, a child inherits its parent's gain column (reading R25).
int quadtree_solve_impl(int64_t n_vis, const double *uvw, const float *vis_host, const int32_t *ant_p,
                        const int32_t *ant_q, int32_t n_ant, const float *gains0, int64_t n0,
                                   const double *l0, const double *m0, const double *side0, int n_levels,
                                   double frac, double min_side, double sigma_factor, int gauss_model, float lambda,
                                   float L_safety, int n_pow, int max_iter, double tol, int check_every,
                                   int64_t capacity, double *l_out, double *m_out, double *side_out, float *x_out,
                                   int64_t *n_out, sl1m_qt_level *levels_out, int *n_levels_done, void *stream) {
    if (!uvw || !vis_host || !l0 || !m0 || !side0 || !l_out || !m_out || !side_out || !x_out || !n_out || !n_levels_done)
        return sl1m_fail(SL1M_ERR_NULL, "sl1m_quadtree_solve: NULL argument");
    if (n_vis < 1 || n0 < 1 || capacity < n0) return sl1m_fail(SL1M_ERR_SIZE, "sl1m_quadtree_solve: n_vis < 1, n0 < 1 or capacity < n0");
    if (n_levels < 1 || !(L_safety > 0.f) || n_pow < 1 || max_iter < 0 || !(tol >= 0.0) || check_every < 1 ||
        !(sigma_factor >= 0.0) || !std::isfinite(sigma_factor))
        return sl1m_fail(SL1M_ERR_PARAM, "sl1m_quadtree_solve: n_levels < 1, L_safety <= 0, n_pow < 1, max_iter < 0, tol < 0, check_every < 1 or sigma_factor < 0");
    cudaStream_t s = (cudaStream_t)stream;
    *n_out = 0;
    *n_levels_done = 0;
    try {
        std::vector<double> l(l0, l0 + n0), m(m0, m0 + n0), side(side0, side0 + n0), sigma;
        std::vector<float> x0, x;                       // x0 empty on the first level: start from zero
        std::vector<float> g, g2;                       // gain table of the current level, [n_ant][n][2]
        if (gains0) g.assign(gains0, gains0 + (size_t)n_ant * (size_t)n0 * 2);
        DevBuf vis_dev, x0_dev, x_dev;
        int st;
        if ((st = vis_dev.alloc((size_t)n_vis * 2 * sizeof(float)))) return st;
        if (cudaMemcpyAsync(vis_dev.p, vis_host, (size_t)n_vis * 2 * sizeof(float), cudaMemcpyHostToDevice, s) != cudaSuccess)
            return sl1m_fail(SL1M_ERR_CUDA, "sl1m_quadtree_solve: copy of the visibilities to the device failed");
        for (int level = 0; level < n_levels; ++level) {
            const auto t_start = std::chrono::steady_clock::now();
            const int64_t n = (int64_t)l.size();
            const double *sig = nullptr;
            if (sigma_factor > 0.0) {                   // splittable leaves are Gaussian, resolution-limit leaves delta
                sigma.resize((size_t)n);
                for (int64_t k = 0; k < n; ++k) sigma[(size_t)k] = (side[(size_t)k] / 2.0 >= min_side) ? sigma_factor * side[(size_t)k] : 0.0;
                sig = sigma.data();
            }
            PlanGuard plan;
            if ((st = sl1m_plan_create(&plan.p, n_vis, uvw, gains0 ? ant_p : nullptr, gains0 ? ant_q : nullptr, n, l.data(),
                                       m.data(), sig, gains0 ? n_ant : 0, gains0 ? g.data() : nullptr, gauss_model, 0)))
                return st;
            float L = 0.f;
            if ((st = sl1m_max_eig(plan.p, n_pow, &L, stream))) return st;
            L *= L_safety;
            if (!(L > 0.f)) return sl1m_fail(SL1M_ERR_PARAM, "sl1m_quadtree_solve: power iteration returned L <= 0 (zero operator)");
            if ((st = x_dev.alloc((size_t)n * sizeof(float)))) return st;
            const float *x0p = nullptr;
            if (!x0.empty()) {
                if ((st = x0_dev.alloc((size_t)n * sizeof(float)))) return st;
                if (cudaMemcpyAsync(x0_dev.p, x0.data(), (size_t)n * sizeof(float), cudaMemcpyHostToDevice, s) != cudaSuccess)
                    return sl1m_fail(SL1M_ERR_CUDA, "sl1m_quadtree_solve: copy of the warm start to the device failed");
                x0p = (const float *)x0_dev.p;
            }
            sl1m_solve_info info;
            if ((st = sl1m_solve_tol(plan.p, (const float *)vis_dev.p, lambda, L, 0, max_iter, tol, check_every, x0p,
                                     (float *)x_dev.p, nullptr, &info, stream)))
                return st;
            x.resize((size_t)n);
            if (cudaMemcpyAsync(x.data(), x_dev.p, (size_t)n * sizeof(float), cudaMemcpyDeviceToHost, s) != cudaSuccess ||
                cudaStreamSynchronize(s) != cudaSuccess)
                return sl1m_fail(SL1M_ERR_CUDA, "sl1m_quadtree_solve: read-back of the level's image failed");
            if (levels_out) {
                sl1m_qt_level &lv = levels_out[level];
                lv.n_pix = n;
                lv.L = L;
                lv.n_iter_done = info.n_iter_done;
                lv.l2_term = info.l2_term;
                lv.l1_term = info.l1_term;
                lv.nnz = info.nnz;
                lv.seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_start).count();
            }
            *n_levels_done = level + 1;
            if (level == n_levels - 1) break;
            // split where emission was found; children start from a quarter of their parent
            int64_t n_split = 0;
            {
                double top = 0.0;
                for (int64_t k = 0; k < n; ++k) if (k == 0 || (double)x[(size_t)k] > top) top = (double)x[(size_t)k];
                for (int64_t k = 0; k < n; ++k)
                    if (top > 0.0 && (double)x[(size_t)k] > frac * top && side[(size_t)k] / 2.0 >= min_side) ++n_split;
            }
            if (n_split == 0) break;
            const int64_t n_new = n + 3 * n_split;
            if (n_new > capacity) return sl1m_fail(SL1M_ERR_SIZE, "sl1m_quadtree_solve: capacity too small for the next level");
            std::vector<double> l2((size_t)n_new), m2((size_t)n_new), s2((size_t)n_new);
            std::vector<float> i2((size_t)n_new);
            int64_t got = 0, nref = 0;
            std::vector<int64_t> parent(gains0 ? (size_t)n_new : 0);
            if ((st = sl1m_quadtree_refine(n, l.data(), m.data(), side.data(), x.data(), frac, min_side, n_new, l2.data(),
                                           m2.data(), s2.data(), i2.data(), gains0 ? parent.data() : nullptr, &got, &nref)))
                return st;
            if (gains0) {                               // children inherit their parent's gain column
                g2.resize((size_t)n_ant * (size_t)n_new * 2);
                for (int32_t a = 0; a < n_ant; ++a)
                    for (int64_t k = 0; k < n_new; ++k) {
                        const size_t src = ((size_t)a * (size_t)n + (size_t)parent[(size_t)k]) * 2, dst = ((size_t)a * (size_t)n_new + (size_t)k) * 2;
                        g2[dst] = g[src];
                        g2[dst + 1] = g[src + 1];
                    }
                g.swap(g2);
            }
            l.swap(l2);
            m.swap(m2);
            side.swap(s2);
            x0.swap(i2);
        }
        const int64_t n = (int64_t)l.size();
        for (int64_t k = 0; k < n; ++k) {
            l_out[k] = l[(size_t)k];
            m_out[k] = m[(size_t)k];
            side_out[k] = side[(size_t)k];
            x_out[k] = x[(size_t)k];
        }
        *n_out = n;
    } catch (const std::bad_alloc &) {
        return sl1m_fail(SL1M_ERR_ALLOC, "sl1m_quadtree_solve: host allocation failed");
    }
    return SL1M_OK;
}
}  // namespace

extern "C" int sl1m_quadtree_solve(int64_t n_vis, const double *uvw, const float *vis_host, int64_t n0,
                                   const double *l0, const double *m0, const double *side0, int n_levels,
                                   double frac, double min_side, double sigma_factor, int gauss_model, float lambda,
                                   float L_safety, int n_pow, int max_iter, double tol, int check_every,
                                   int64_t capacity, double *l_out, double *m_out, double *side_out, float *x_out,
                                   int64_t *n_out, sl1m_qt_level *levels_out, int *n_levels_done, void *stream) {
    return quadtree_solve_impl(n_vis, uvw, vis_host, nullptr, nullptr, 0, nullptr, n0, l0, m0, side0, n_levels, frac,
                               min_side, sigma_factor, gauss_model, lambda, L_safety, n_pow, max_iter, tol, check_every,
                               capacity, l_out, m_out, side_out, x_out, n_out, levels_out, n_levels_done, stream);
}

extern "C" int sl1m_quadtree_solve_gains(int64_t n_vis, const double *uvw, const float *vis_host,
                                         const int32_t *ant_p, const int32_t *ant_q, int32_t n_ant,
                                         const float *gains0_host, int64_t n0, const double *l0, const double *m0,
                                         const double *side0, int n_levels, double frac, double min_side,
                                         double sigma_factor, int gauss_model, float lambda, float L_safety, int n_pow,
                                         int max_iter, double tol, int check_every, int64_t capacity, double *l_out,
                                         double *m_out, double *side_out, float *x_out, int64_t *n_out,
                                         sl1m_qt_level *levels_out, int *n_levels_done, void *stream) {
    if (!ant_p || !ant_q || !gains0_host) return sl1m_fail(SL1M_ERR_NULL, "sl1m_quadtree_solve_gains: NULL gain argument");
    if (n_ant < 1) return sl1m_fail(SL1M_ERR_SIZE, "sl1m_quadtree_solve_gains: n_ant < 1");
    return quadtree_solve_impl(n_vis, uvw, vis_host, ant_p, ant_q, n_ant, gains0_host, n0, l0, m0, side0, n_levels, frac,
                               min_side, sigma_factor, gauss_model, lambda, L_safety, n_pow, max_iter, tol, check_every,
                               capacity, l_out, m_out, side_out, x_out, n_out, levels_out, n_levels_done, stream);
}
