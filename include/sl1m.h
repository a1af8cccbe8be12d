/*
 * sl1m.h -- C ABI of the B200-native SL1M hot path (arXiv:1310.2078, S. J. Hardy 2013).
 *
 * The library evaluates, on one sm_100a GPU, the direct (ungridded, matrix-free) measurement
 * operator of the paper and the FISTA solver built on it.  Citations are PAPER.md:<line>.
 *
 *   M_jk   eq (9)  PAPER.md:117-120   delta pixels (sigma_k == 0)
 *          eq (16) PAPER.md:160-163   Gaussian pixels, paraxial   (SL1M_GAUSS_PARAXIAL)
 *          eq (17) PAPER.md:171-174   Gaussian pixels, wide field (SL1M_GAUSS_WIDEFIELD)
 *          times G_jk = g_p(k) conj(g_q(k)) for baseline j = (p_j, q_j)
 *   forward  v = M x          eq (8)  PAPER.md:113-115          sl1m_forward
 *   adjoint  g = Re M^H r     PAPER.md:192, 199                 sl1m_adjoint
 *   L = lambda_max(Re M^H M)  PAPER.md:190, 211                 sl1m_max_eig
 *   FISTA + T^d               PAPER.md:188-197 (eq 18)          sl1m_solve
 *
 * Conventions
 *  - Every call returns an sl1m_status (0 = OK).  Nothing throws or aborts across the ABI.
 *    Arguments are validated before any device work.  sl1m_last_error() returns a thread-local
 *    message for the most recent non-OK status.
 *  - "HOST" pointers are ordinary CPU memory, "DEV" pointers are CUDA device memory of the
 *    current device (e.g. torch.Tensor.data_ptr()).  `stream` is a cudaStream_t passed as
 *    void* (NULL = the legacy default stream).
 *  - The plan COPIES every plan-time input; the caller may free them on return.  Vectors passed
 *    to forward/adjoint/solve stay caller-owned; outputs are overwritten, never accumulated.
 *  - forward/adjoint are asynchronous on `stream`.  solve, fista_begin and max_eig copy their scalars
 *    (lambda, L, the momentum table of a persistent plan) to the device from buffers of their own and
 *    therefore synchronise `stream` ONCE, at the start of the call; the iterations are then enqueued
 *    without any host round-trip per iteration (the device-side stopping rules are polled behind the
 *    enqueue front, sl1m_solve_stop), and the call synchronises again at the end only when a host
 *    result (info / L) was asked for.  fista_step never waits.  The *_host variants copy in and out of
 *    HOST buffers on `stream` and synchronise before returning.
 *  - A plan owns its workspaces: do not use one plan from two streams at once.
 *  - Images are real fp32 [n_pix] in the CALLER's pixel order; visibilities are complex fp32,
 *    interleaved (re, im), [n_vis][2], in the caller's order.
 *  - There is no CPU fallback: without a usable CUDA device every call fails with SL1M_ERR_CUDA.
 */
#ifndef SL1M_H_
#define SL1M_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sl1m_plan sl1m_plan; /* opaque; owns all device copies and workspaces */

typedef enum {
    SL1M_OK = 0,
    SL1M_ERR_NULL = 1,   /* a required pointer is NULL */
    SL1M_ERR_SIZE = 2,   /* n_vis < 1, n_pix < 1, n_ant < 1 with gains, sizes beyond 2^31-1 tiles */
    SL1M_ERR_DOMAIN = 3, /* l^2 + m^2 >= 1, sigma < 0, NaN/Inf in uvw, l, m, sigma */
    SL1M_ERR_INDEX = 4,  /* antenna index outside [0, n_ant) */
    SL1M_ERR_ALLOC = 5,  /* host or device allocation failed */
    SL1M_ERR_CUDA = 6,   /* CUDA runtime error (no device, launch failure, ...) */
    SL1M_ERR_PARAM = 7   /* lambda < 0, L <= 0 with n_pow <= 0, n_iter < 0, unknown model/flag */
} sl1m_status;

typedef enum {
    SL1M_GAUSS_PARAXIAL = 0, /* eq (16) */
    SL1M_GAUSS_WIDEFIELD = 1 /* eq (17) */
} sl1m_gauss_model;

/* flags for sl1m_plan_create */
#define SL1M_GAINS_ON_DEVICE 1u /* `gains` is a DEV pointer (default: HOST) */
#define SL1M_PHASE_FP64 2u      /* accumulate the whole phase in fp64 (delta pixels, unit gains).
                                 * Chosen automatically when the fp32 phase remainder inside a pixel tile could
                                 * exceed 256 rad (a tile spanning > 40 fringes of the longest baseline: a badly
                                 * undersampled image); the default kernels are exact enough otherwise. */
#define SL1M_NO_PERSISTENT 8u   /* small problems (delta pixels, unit gains, one channel, < 6.7e7 terms per apply) run the
                                 * whole FISTA loop as ONE persistent cooperative kernel -- two grid barriers per
                                 * iteration instead of six launches (sl1m_plan_info.persistent == 1).  This flag keeps
                                 * the multi-launch loop, for A/B measurements and tests.  Both are deterministic; they sum
                                 * in different orders, so their images agree to rounding, not bit for bit. */
#define SL1M_DENSE_FORWARD 4u   /* switch the zero-skipping forward off (see sl1m_forward_active_pixels): every
                                 * pixel is streamed even where x_k == 0.  For A/B measurements and tests. */

/*
 * sl1m_plan_create -- build the operator for one set of visibilities and pixels.
 *   uvw      HOST [n_vis][3] fp64, baseline coordinates in wavelengths.
 *   ant_p/q  HOST [n_vis] int32 antenna (gain-row) indices; may be NULL iff gains == NULL.
 *   l, m     HOST [n_pix] fp64 direction cosines of the pixel centres, any order, need not lie
 *            on a grid.
 *   sigma    HOST [n_pix] fp64, the paper's sigma_k of eq (11) (NOT a standard
 *            deviation: std = sigma/sqrt(2 pi)); NULL or 0 => delta pixel, which always uses
 *            eq (9).  sigma_k > 0 uses eq (16) or eq (17) according to `gauss_model`.
 *   gains    [n_ant][n_pix][2] fp32 (re, im), HOST (or DEV with SL1M_GAINS_ON_DEVICE);
 *            NULL => unit gains.  Time-varying beams: give each (antenna, time) its own row.
 * Plan-time work (fp64 on the host): n_k, 1/n_k, n_k - 1 in the cancellation-free form
 * -r^2/(1+n), a Morton sort of the pixels into compact tiles of 256 with fp64 tile centres,
 * and the fp32 offsets from those centres that the kernels consume.
 */
int sl1m_plan_create(sl1m_plan **out, int64_t n_vis, const double *uvw, const int32_t *ant_p,
                     const int32_t *ant_q, int64_t n_pix, const double *l, const double *m,
                     const double *sigma, int32_t n_ant, const float *gains, int gauss_model,
                     uint32_t flags);

/* v = M x.  x DEV [n_pix] fp32 (real), vis DEV [n_vis][2] fp32.  Asynchronous on stream.  Safe inside a stepped
 * FISTA run (see sl1m_fista_begin). */
int sl1m_forward(sl1m_plan *plan, const float *x_dev, float *vis_dev, void *stream);

/* g = Re M^H r.  r DEV [n_vis][2] fp32, img DEV [n_pix] fp32.  Asynchronous on stream.
 * The image is real (PAPER.md:192-197 thresholds x_i > d), so only the real part is formed; the kernels evaluate
 * it as sum_j |M_jk| |r_j| cos(arg r_j - arg M_jk): one cosine per term. */
int sl1m_adjoint(sl1m_plan *plan, const float *r_dev, float *img_dev, void *stream);

/* Same applies with HOST buffers: H2D copy, apply, D2H copy, stream synchronise. */
int sl1m_forward_host(sl1m_plan *plan, const float *x_host, float *vis_host, void *stream);
int sl1m_adjoint_host(sl1m_plan *plan, const float *r_host, float *img_host, void *stream);

/*
 * sl1m_max_eig -- L = lambda_max(Re M^H M) by n_pow rounds of power iteration from the
 * deterministic start x = 1/sqrt(n_pix): g = M^H(M x), L = ||g||_2, x = g/L.  Approaches
 * lambda_max FROM BELOW; callers normally multiply by a safety factor (e.g. 1.05) before
 * passing it to sl1m_solve.  Writes *L_out_host (HOST) after one stream synchronise.  Plans that run the persistent
 * kernel (sl1m_plan_info.persistent) do all n_pow rounds in one cooperative launch.  Overwrites the pixel tiles: ends a
 * stepped FISTA run (sl1m_fista_begin).
 */
int sl1m_max_eig(sl1m_plan *plan, int n_pow, float *L_out_host, void *stream);

typedef struct {
    int32_t n_iter_done;
    float L_used;
    double l2_term; /* ||M I_K - V||^2        (Table 1's "L2 term") */
    double l1_term; /* sum_k I_K[k]           (Table 1's "L1 term")                    */
    int64_t nnz;    /* number of non-zero pixels in I_K                                */
} sl1m_solve_info;

/*
 * sl1m_solve -- n_iter FISTA iterations exactly as listed at PAPER.md:188-192:
 *   y_1 = I_0 = x0 (0 if NULL), t_1 = 1;
 *   I_k = T^{lambda/L}( y_k - (1/L) Re M^H (M y_k - V) ),          T^d of eq (18);
 *   t_{k+1} = (1 + sqrt(1 + 4 t_k^2))/2,  y_{k+1} = I_k + ((t_k - 1)/t_{k+1}) (I_k - I_{k-1}).
 * Its fixed point minimises 1/2 ||V - M I||^2 + lambda sum I, I >= 0 (eq (10) with
 * lambda_paper = 2 lambda).
 *   vis_dev   DEV [n_vis][2] measured visibilities V.
 *   L         step constant; L <= 0 => computed by n_pow rounds of sl1m_max_eig (no safety
 *             factor applied).
 *   x0_dev    DEV [n_pix] or NULL.        x_out_dev  DEV [n_pix], receives I_K.
 *   trace_dev DEV [n_iter][3] fp64 or NULL: per iteration {||M y_k - V||^2, sum I_k, nnz I_k},
 *             written on the device, never read by the host.
 *   info_host HOST or NULL; when non-NULL one extra forward evaluates ||M I_K - V||^2 and the
 *             call synchronises `stream` once before returning.
 */
int sl1m_solve(sl1m_plan *plan, const float *vis_dev, float lambda, float L, int n_pow, int n_iter,
               const float *x0_dev, float *x_out_dev, double *trace_dev,
               sl1m_solve_info *info_host, void *stream);

/*
 * sl1m_solve_tol -- sl1m_solve with the paper's termination rule ("terminated when
 * an iteration leads to a sufficiently small change in the total error E, given by equation
 * (10)"; section 4.1.1: "until the total error changes no more than 1 part in 10^6
 * or until 7000 iterations were reached").  E is formed on the device from what the iteration
 * already has: E_k = ||M y_k - V||^2 + 2 lambda sum I_k (eq (10) with lambda_paper = 2 lambda; the
 * residual is that of y_k, because evaluating M I_k as well is what the paper declines to pay
 * for).  After every `check_every`-th iteration k >= 2 the host reads the two
 * newest trace rows (48 bytes) and stops iff |E_k - E_{k-1}| <= tol |E_k|; no other host
 * round-trip happens inside the loop.  max_iter caps the count (the paper's 7000).
 *   tol >= 0, check_every >= 1, info_host REQUIRED (n_iter_done is how the caller learns k).
 *   trace_dev DEV [max_iter][3] fp64 or NULL (then a plan-owned buffer is used).
 */
int sl1m_solve_tol(sl1m_plan *plan, const float *vis_dev, float lambda, float L, int n_pow,
                   int max_iter, double tol, int check_every, const float *x0_dev,
                   float *x_out_dev, double *trace_dev, sl1m_solve_info *info_host, void *stream);

/*
 * sl1m_solve_stop -- sl1m_solve with BOTH termination criteria of PAPER.md:194 ("terminated when an iteration
 * leads to a sufficiently small change in the total error E, given by equation (10), or when there is a
 * sufficiently small change in the number of non-zero entries in I_k"), decided ON THE DEVICE:
 *   E rule    |E_k - E_{k-1}| <= tol |E_k|        E_k = ||M y_k - V||^2 + 2 lambda sum I_k  (reading R21); tol < 0: off
 *   nnz rule  |N_k - N_{k-1}| <= nnz_tol N_k      N_k = nnz(I_k)                          (reading R24); nnz_tol < 0: off
 * looked at after every check_every-th iteration k >= 2; the solve stops at the first k where an enabled rule
 * holds (at least one must be enabled), else at max_iter.  A one-CTA kernel takes the decision from the trace rows
 * the iteration has just written and raises a device flag; every kernel of a stopped solve returns at once, so
 * the image is that of the stopping iteration.  The host never waits for an iteration: it reads the flag two
 * polls (of >= 16 iterations) behind what it has enqueued and synchronises once at the end for info_host.
 * sl1m_solve_tol(tol) == sl1m_solve_stop(tol, nnz_tol = -1).
 *   trace_dev DEV [max_iter][3] fp64 or NULL (a plan-owned buffer is used); rows past n_iter_done are not written.
 *   info_host REQUIRED (n_iter_done is how the caller learns k).
 * sl1m_solve_stop_batch: the same for every channel of a batched plan, each stopping on its own (a stopped
 * channel's CTAs return at once while the others go on); lambda_host, L_host, info_host HOST [n_chan],
 * trace_dev DEV [n_chan][max_iter][3] or NULL.
 */
int sl1m_solve_stop(sl1m_plan *plan, const float *vis_dev, float lambda, float L, int n_pow,
                    int max_iter, double tol, double nnz_tol, int check_every, const float *x0_dev,
                    float *x_out_dev, double *trace_dev, sl1m_solve_info *info_host, void *stream);
int sl1m_solve_stop_batch(sl1m_plan *plan, const float *vis_dev, const float *lambda_host,
                          const float *L_host, int n_pow, int max_iter, double tol, double nnz_tol,
                          int check_every, const float *x0_dev, float *x_out_dev, double *trace_dev,
                          sl1m_solve_info *info_host, void *stream);

/*
 * Stepping API -- the listing of PAPER.md:188-192 driven a few iterations at a time (interactive imaging; bench.py
 * times the steps of ONE continuing FISTA run through it).  The state (I_k, y_{k+1}, t_{k+1}) lives in the plan.
 *   sl1m_fista_begin  y_1 = I_0 = x0 (0 if NULL), t_1 = 1.  lambda_host, L_host HOST [n_chan] (L > 0).  vis_dev
 *                     DEV [n_chan][n_vis][2] is BORROWED: it must stay valid and unchanged until the next begin.
 *   sl1m_fista_step   n_iter more iterations, asynchronous on stream.  trace_dev DEV [n_chan][max(n_iter,1)][3] or
 *                     NULL receives the rows of THIS call's iterations.
 *   sl1m_fista_image  x_out DEV [n_chan][n_pix] = I_k; *n_iter_done_host (nullable) = k.  Asynchronous.
 * Any solve call on the plan, sl1m_max_eig, or sl1m_plan_set_channels ends the state; a later sl1m_fista_step /
 * sl1m_fista_image then fails with SL1M_ERR_PARAM ("no FISTA state").  Only sl1m_fista_begin opens one: every
 * sl1m_solve* variant ends whatever run was open and leaves none behind (its vis_dev is not borrowed past the call),
 * with or without info_host.
 * sl1m_forward / sl1m_adjoint (and their _host and dirty-image forms) may be called BETWEEN steps without disturbing
 * the run -- e.g. step, sl1m_fista_image, sl1m_forward(I_k) to show the model visibilities, step again: the forward
 * restores the run's a*y_{k+1} pixel tiles after using them for the caller's image (one extra O(n_pix) launch).
 */
int sl1m_fista_begin(sl1m_plan *plan, const float *vis_dev, const float *lambda_host,
                     const float *L_host, const float *x0_dev, void *stream);
int sl1m_fista_step(sl1m_plan *plan, int n_iter, double *trace_dev, void *stream);
int sl1m_fista_image(sl1m_plan *plan, float *x_out_dev, int32_t *n_iter_done_host, void *stream);

/*
 * sl1m_dirty_image -- img = max(0, scale * Re M^H V): "use the dirty image as the initial
 * condition", clipped to the positive orthant the solver lives in.  scale is the
 * caller's normalisation (1/n_vis gives unit point-source response for delta pixels near the
 * phase centre).  vis DEV [n_chan][n_vis][2], img DEV [n_chan][n_pix] (every channel of a batched plan, same
 * scale); asynchronous on stream.  Pass the result as x0_dev to sl1m_solve / sl1m_solve_stop(_batch).
 */
int sl1m_dirty_image(sl1m_plan *plan, const float *vis_dev, float scale, float *img_dev, void *stream);

/*
 * Coarse-to-fine / adaptive quadtree acceleration (section 4.5, Fig. 10: "the
 * system is solved at a low resolution, and pixels where emission is detected are then
 * subdivided ... refinement of all pixels greater than 1 per cent of the maximum"; a 13x speed-up
 * in the paper).  What the paper leaves open is fixed by DESIGN.md reading R23:
 *  - a pixel is a square of side s_k centred on (l_k, m_k); it splits iff I_k > frac * max_j I_j
 *    and s_k/2 >= min_side, and is replaced IN PLACE by four children of side s_k/2 centred on
 *    l_k -/+ s_k/4, m_k -/+ s_k/4 (l fastest); every other pixel stays (mixed sizes in one
 *    solve).  frac < 0 splits every pixel of an image with any emission: the plain coarse-to-fine
 *    strategy.  An image that is zero everywhere splits nothing, whatever frac is (no emission was detected: a
 *    level solved with too large a lambda ends the refinement instead of quadrupling an empty grid).
 *  - "upscale the previously calculated solution": a child starts from I_k/4.
 *
 * sl1m_quadtree_refine -- ONE split step, pure host code (needs no GPU).  All pointers HOST.
 *   in:  n pixels (l, m, side fp64; I fp32, e.g. the image a solve returned)
 *   out: l_out, m_out, side_out, I0_out [capacity >= n + 3 * (number split)], parent_out
 *        (nullable: index of the input pixel each output pixel came from), *n_out, *n_refined.
 *   SL1M_ERR_SIZE if capacity is too small (nothing written).
 */
int sl1m_quadtree_refine(int64_t n, const double *l, const double *m, const double *side,
                         const float *I, double frac, double min_side, int64_t capacity,
                         double *l_out, double *m_out, double *side_out, float *I0_out,
                         int64_t *parent_out, int64_t *n_out, int64_t *n_refined);

typedef struct {
    int64_t n_pix;       /* pixels solved at this level                          */
    float L;             /* step constant used (power iteration x L_safety)      */
    int32_t n_iter_done; /* FISTA iterations until the stopping rule / the cap   */
    double l2_term, l1_term;
    int64_t nnz;
    double seconds;      /* wall time of the level: plan + L + solve + read-back */
} sl1m_qt_level;

/*
 * sl1m_quadtree_solve -- the driver: at most n_levels times { plan the current pixel list,
 * L = L_safety * sl1m_max_eig(n_pow), sl1m_solve_tol(lambda, max_iter, tol, check_every) warm-
 * started from the upscaled previous level, split }.  Stops early when no pixel splits.
 * Pixels that can still split are Gaussian pixels of sigma_k = sigma_factor * s_k (eq 16/17 by
 * gauss_model), pixels at the resolution limit (s_k/2 < min_side) and all pixels when
 * sigma_factor == 0 are delta pixels (eq 9).  Unit gains (sl1m_quadtree_solve_gains takes a gain table).
 *   uvw HOST [n_vis][3] fp64; vis_host HOST [n_vis][2] fp32; l0, m0, side0 HOST [n0] fp64.
 *   outputs HOST [capacity]: final leaves (l, m, side) and their fluxes x; *n_out leaves.
 *   levels_out HOST [n_levels] or NULL; *n_levels_done.  Synchronises `stream` at every level.
 */
int sl1m_quadtree_solve(int64_t n_vis, const double *uvw, const float *vis_host, int64_t n0,
                        const double *l0, const double *m0, const double *side0, int n_levels,
                        double frac, double min_side, double sigma_factor, int gauss_model,
                        float lambda, float L_safety, int n_pow, int max_iter, double tol,
                        int check_every, int64_t capacity, double *l_out, double *m_out,
                        double *side_out, float *x_out, int64_t *n_out, sl1m_qt_level *levels_out,
                        int *n_levels_done, void *stream);

/*
 * sl1m_quadtree_solve_gains -- the same driver with direction-dependent gains: ant_p, ant_q HOST [n_vis] int32 and
 * gains0_host HOST [n_ant][n0][2] fp32, the gain table ON THE STARTING PIXEL LIST.  The paper does not say what the
 * gains of a refined pixel are; reading R25: a child inherits the gain column of its parent (the beam is
 * taken as constant over a pixel that is being split).  Everything else as sl1m_quadtree_solve.
 */
int sl1m_quadtree_solve_gains(int64_t n_vis, const double *uvw, const float *vis_host,
                              const int32_t *ant_p, const int32_t *ant_q, int32_t n_ant,
                              const float *gains0_host, int64_t n0, const double *l0, const double *m0,
                              const double *side0, int n_levels, double frac, double min_side,
                              double sigma_factor, int gauss_model, float lambda, float L_safety, int n_pow,
                              int max_iter, double tol, int check_every, int64_t capacity, double *l_out,
                              double *m_out, double *side_out, float *x_out, int64_t *n_out,
                              sl1m_qt_level *levels_out, int *n_levels_done, void *stream);

/*
 * Batched channels (NEXT-4 of the scope table).  The paper's data sets are 61-127 spectral channels
 * (and two polarisations) of ONE observing geometry, each deconvolved independently
 * (PAPER.md:68, 279, 307); the baselines in wavelengths scale with frequency (PAPER.md:61,
 * "b = lambda (u, v, w)").  sl1m_plan_set_channels turns a plan into a batch of n_chan
 * independent problems that share the pixel list, the gain table and the baseline geometry:
 * channel c uses uvw * scale[c] (scale[c] = nu_c / nu_0, HOST [n_chan], > 0).  Afterwards
 *   sl1m_forward   takes x  DEV [n_chan][n_pix]     and writes vis DEV [n_chan][n_vis][2],
 *   sl1m_adjoint   takes r  DEV [n_chan][n_vis][2]  and writes img DEV [n_chan][n_pix],
 * in ONE launch per step (grid z = channel), which is what fills the GPU when one channel's
 * problem is small; sl1m_max_eig_batch / sl1m_solve_batch are the per-channel versions of
 * sl1m_max_eig / sl1m_solve:
 *   L_out_host, lambda_host, L_host, info_host   HOST [n_chan]   (L_host[c] <= 0 => power iteration)
 *   vis_dev DEV [n_chan][n_vis][2]; x0_dev (nullable), x_out_dev DEV [n_chan][n_pix];
 *   trace_dev DEV [n_chan][max(n_iter,1)][3] or NULL.
 * Channels never interact: every result equals the single-channel call on uvw * scale[c].
 * The single-problem calls (sl1m_max_eig, sl1m_solve, sl1m_solve_tol, sl1m_solve_stop, *_host) return
 * SL1M_ERR_PARAM on a plan with more than one channel (use the *_batch call).  Re-allocates the plan's
 * workspaces; synchronises the device.  Transactional: on failure (e.g. out of memory) the plan is unchanged.
 * The fp64-phase decision (SL1M_PHASE_FP64) is re-evaluated for max(scale): a plan whose fp32 phase remainder
 * would exceed 256 rad at its highest channel switches to the fp64-phase kernels, which honour the scales too.
 */
int sl1m_plan_set_channels(sl1m_plan *plan, int32_t n_chan, const double *scale_host);
int32_t sl1m_plan_n_chan(const sl1m_plan *plan);
int sl1m_max_eig_batch(sl1m_plan *plan, int n_pow, float *L_out_host, void *stream);
int sl1m_solve_batch(sl1m_plan *plan, const float *vis_dev, const float *lambda_host,
                     const float *L_host, int n_pow, int n_iter, const float *x0_dev,
                     float *x_out_dev, double *trace_dev, sl1m_solve_info *info_host, void *stream);

/* sl1m_solve with HOST vis / x0 / x_out (trace not available); always synchronises. */
int sl1m_solve_host(sl1m_plan *plan, const float *vis_host, float lambda, float L, int n_pow,
                    int n_iter, const float *x0_host, float *x_out_host,
                    sl1m_solve_info *info_host, void *stream);

/* Launch configuration and instruction mix of a plan (what bench.py's roofline arithmetic uses). */
typedef struct {
    int32_t n_pix_padded, n_tiles;       /* sorted pixel list padded to 1,024; tiles of 256        */
    int32_t gaussian, gains;             /* gaussian: 1 if any sigma_k > 0.  gains: 0 none, 1 per-term
                                          * loads, 2 baseline-grouped (one gain product per 8 samples) */
    int32_t fwd_rv;                      /* visibilities per thread in the forward kernel          */
    int32_t fwd_vis_tiles, fwd_pixel_splits, fwd_tiles_per_split;
    int32_t fwd_poly_per16;              /* of every 16 terms, how many use FMA-pipe polynomial sincos */
    int32_t adj_rp;                      /* pixels per thread in the adjoint kernel                */
    int32_t adj_pixel_groups, adj_vis_splits, adj_chunks_per_split;
    int32_t adj_poly_per16;
    int32_t mufu_per_term_mufu_path;     /* forward: 2 (delta), 3 (Gaussian, one sigma per tile) or 4 (Gaussian) */
    int32_t fwd_packed_pairs;            /* 1 = the packed fp32x2 (FFMA2) forward kernel is in use  */
    int32_t adj_packed_pairs;
    int32_t phase_fp64;                  /* 1 = the fp64-phase kernels are in use                    */
    float phase_span_rad;                /* plan-time bound on the fp32 phase remainder in a tile    */
    int32_t zero_skip;                   /* 1 = the forward streams only pixels with x_k != 0       */
    int32_t persistent;                  /* 1 = the FISTA loop of this plan runs as one persistent cooperative kernel */
    int32_t adj_mufu_per_term;           /* MUFU per MUFU-path term of the ADJOINT: 1 with the one-cosine kernels
                                          * (Re(e^{iX} r) = |r| cos(X + arg r)), 2 with per-tile-sigma Gaussian
                                          * pixels (ex2 + cos), else as the forward                  */
} sl1m_plan_info;
int sl1m_plan_describe(const sl1m_plan *plan, sl1m_plan_info *info_host);

/*
 * Zero-skipping forward.  The image of an L1 solve is sparse and non-negative (eq (18), PAPER.md:194-197:
 * T^d zeroes every x_i <= d), so most terms M_jk x_k of the forward are exactly zero.  Whenever a*x is packed
 * into the pixel tiles (sl1m_forward, every FISTA iteration, the power iteration) the pixels with x_k != 0 are
 * moved to the front of a compact copy of their tile, in their original order, and the forward kernel streams
 * only those; the result is the same sum with the zero terms left out.  With a gain table the gain rows of the
 * compact entries are copied next to them (one more table-sized buffer per channel; a full tile is not copied).
 * Kernels that stage a per-pixel side array next to the tile (per-pixel sigma; the fp64 offsets of the fp64-phase
 * kernels) get a compact copy of that array as well.  Plans whose compact gain rows would exceed 8 GiB keep the dense
 * forward (sl1m_plan_info.zero_skip == 0), as does SL1M_DENSE_FORWARD.  The adjoint always evaluates every term.
 * n_active_host: HOST [n_chan]; pixels the most recently packed forward input streams per channel (padded to
 * 4 per tile; n_pix_padded when the plan does not skip).  During a stepped run on a persistent plan
 * (sl1m_plan_info.persistent; its kernels skip zeros straight from y and keep no compact tiles): the exact number of
 * pixels with y_{k+1} != 0, which is what the next iteration's forward evaluates.  Synchronises `stream`.
 */
int sl1m_forward_active_pixels(sl1m_plan *plan, int64_t *n_active_host, void *stream);

/*
 * sl1m_measure_peaks -- issue-rate micro-benchmark for the roofline the operator is held against.
 * The operator is a GENERATED matrix-vector product (the matrix is never stored), bound by the XU
 * (MUFU.SIN/COS/EX2) and FMA pipes, not by HBM; the denominators are therefore measured with those instructions in
 * the kernels' own launch shape (128-thread CTAs, 8 per SM on every SM, chains of independent instructions).
 * Runs ~10 short kernels on `stream` (about 50 ms in all), synchronises, needs no plan.  All rates are for the
 * whole GPU, timed with CUDA events; the per-clock figures divide by the device's maximum SM clock.
 */
typedef struct {
    int32_t n_sm;
    double sm_clock_mhz;                 /* the device's maximum SM clock (cudaDevAttrClockRate): basis of the per-clock figures */
    double clock64_mhz;                  /* clock64 ticks per second seen by the MUFU probe (not the SM clock on B200; unused)    */
    double mufu_per_s, mufu_per_clk_sm;  /* MUFU.EX2 alone: results/s, results per clock per SM (nominal 16)        */
    double mufu_cos_per_clk_sm;          /* MUFU.COS alone (same pipe)                                              */
    double ffma_per_s, ffma_per_clk_sm;  /* scalar FFMA alone (nominal 128 per clock per SM)                        */
    double ffma2_lanes_per_s, ffma2_lanes_per_clk_sm;   /* packed FFMA2, counted in fp32 lanes (2 per instruction)  */
    double coissue_mufu_per_clk_sm;      /* 4 MUFU + 12 FFMA2 + 4 FMUL.RZ per body: MUFU results per clock per SM   */
    double coissue_ffma2_lanes_per_clk_sm;   /* ... and the FFMA2 lanes per clock per SM achieved beside them       */
    double coissue_cycles_per_iter;      /* sub-partition cycles per warp per body (profiles/r1_microbench.md: 35.3) */
    double coissue_adj_mufu_per_clk_sm;  /* 4 MUFU.COS + 8 FFMA2 + 4 FMUL.RZ per body (the one-cosine adjoint's mix) */
    double dfma_per_s, dfma_per_clk_sm;  /* DFMA alone on the FP64 pipe (the fp64-phase kernels: 4 FP64 ops per term)  */
} sl1m_peaks;
int sl1m_measure_peaks(sl1m_peaks *out_host, void *stream);

/*
 * Memory-safety net without compute-sanitizer (SURVEY.md:184; the GPU pool does not run the tool).  A library
 * built with -DSL1M_BOUNDS (paper_1310_2078_b200.build.build_library(bounds=True) -> libsl1m_bounds.so) puts a 4 KiB
 * canary band on both sides of every device buffer it allocates and asserts, on the device, that the two documented
 * over-reads of the kernels (register prefetch of gain-table rows, up to 4 rows past the pixels in use) stay inside
 * their tables.  sl1m_debug_check synchronises the device and verifies every band: SL1M_ERR_CUDA (with
 * sl1m_last_error naming the buffer size and side) after a stray write or a failed device assertion.  In the normal
 * build it does nothing and returns SL1M_OK.  sl1m_debug_bounds_build: 1 in the debug build, else 0.
 */
int sl1m_debug_check(void);
int sl1m_debug_bounds_build(void);
/* Debug build only (SL1M_ERR_PARAM otherwise): writes 4 bytes just past the plan's residual buffer, so that a test can
 * see sl1m_debug_check report it. */
int sl1m_debug_poke_past_end(sl1m_plan *plan);

/*
 * sl1m_forward_noalloc -- v = M x of eq (9) (delta pixels, unit gains, one channel) WITHOUT a plan
 * and without any allocation, for callers that cannot ask the CUDA driver for memory when they need an apply:
 * a real-time pipeline whose other streams must keep running (cudaMalloc / cudaFree hold up the whole device), a
 * process whose device memory belongs entirely to someone else's pool (a raw cudaMalloc fails there, or takes what a
 * neighbour was promised), a service bound to a fixed memory footprint after start-up.  Every plan-based call is
 * closed to them because sl1m_plan_create allocates the plan's workspaces.
 *   uvw_dev  DEV [n_vis][3] fp64, wavelengths.          l_dev, m_dev  DEV [n_pix] fp64 direction cosines.
 *   x_dev    DEV [n_pix] fp32 image.                                  vis_dev       DEV [n_vis][2] fp32 (re, im), overwritten.
 * All five buffers stay the caller's; they are read / written in the caller's order and not copied.
 * Scratch: the per-split partial sums go to ONE array compiled into the library (4 MiB of device memory on every GPU
 * that loads the library, held until the process exits).  Consequences:
 *  - limits: n_vis <= SL1M_NOALLOC_MAX_VIS and n_pix <= SL1M_NOALLOC_MAX_PIX, else SL1M_ERR_SIZE (checked before any
 *    device work) with sl1m_last_error() naming the limit; larger problems need a plan, or one call per block of
 *    visibilities (rows of M are independent);
 *  - all calls on a device share the array.  Calls issued to the SAME stream are safe back to back.  Calls that may
 *    run at the same time on the GPU (different streams, different host threads) overwrite each other's partial sums
 *    and give wrong visibilities without any error: serialise them yourself;
 *  - the array keeps the previous call's contents; nothing in it has to start at zero, because every slot the final
 *    sum reads is first written by the same call.
 * The FIRST call on each device looks up the array's device address (once per device, the device current at the
 * call) -- make that first call at start-up, outside any stream capture; later calls only launch two kernels.
 * Asynchronous on `stream`; deterministic (fixed summation order).  l^2 + m^2 >= 1 is NOT checked (the inputs are
 * on the device): such a pixel poisons the output with NaN.  Accuracy as sl1m_forward (phase in fp64, relative L2
 * <= 2e-4 against the fp64 definition); slower than a plan's forward -- no sort, no tile centres, no zero skipping.
 */
#define SL1M_NOALLOC_MAX_VIS 524288   /* = 4 MiB of scratch / 8 B per complex partial */
#define SL1M_NOALLOC_MAX_PIX 16777216
int sl1m_forward_noalloc(int64_t n_vis, const double *uvw_dev, int64_t n_pix, const double *l_dev, const double *m_dev,
                         const float *x_dev, float *vis_dev, void *stream);

/* Number of kernels this plan has launched since creation (for bench.py's gpu_launches). */
int64_t sl1m_launch_count(const sl1m_plan *plan);

/* Sizes the plan was created with (0 for a NULL plan). */
int64_t sl1m_plan_n_vis(const sl1m_plan *plan);
int64_t sl1m_plan_n_pix(const sl1m_plan *plan);

void sl1m_destroy(sl1m_plan *plan);     /* NULL-safe */
const char *sl1m_status_string(int st); /* static strings */
const char *sl1m_last_error(void);      /* thread-local detail of the last non-OK status */

#ifdef __cplusplus
}
#endif
#endif /* SL1M_H_ */
