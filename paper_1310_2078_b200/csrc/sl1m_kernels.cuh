// sl1m_kernels.cuh -- sm_100a device code of the SL1M hot path (arXiv:1310.2078).
//
// The matrix M (eq 9 / 16 / 17) is never stored:
// every (visibility j, pixel k) entry is generated on the fly.  Design:
//
//  * Pixels are Morton-sorted at plan time into compact tiles of TP = 256 with an fp64 centre
//    (l_c, m_c, n'_c).  The phase of a term is split as
//        2 pi (u l + v m + w n')  =  x0(j, tile)  +  u' dl_k + v' dm_k + w' dn'_k
//    where x0 = 2 pi frac(u l_c + v m_c + w n'_c) is evaluated ONCE per (visibility, tile) in fp64
//    and range-reduced there, and the small offsets (dl, dm, dn') and u' = 2 pi u ... are fp32.
//    The per-term cost is 3 FFMA + FMUL.RZ + MUFU.SIN + MUFU.COS + 2 FFMA, and the fp32 phase
//    error scales with the tile extent instead of the field extent.
//  * forward: a thread owns RV visibilities in registers, the CTA streams pixel tiles through
//    shared memory with 1-D TMA bulk copies (cp.async.bulk + mbarrier, double buffered); every
//    lane reads the same pixel (broadcast LDS.128).
//  * adjoint: a thread owns RP pixels in registers (a warp's pixels share one tile centre), the
//    CTA stages chunks of visibilities (u', v', w', r, x0 per centre) in shared memory.
//  * Outputs are split across CTAs (pixel splits / visibility splits) into a workspace and
//    reduced in a fixed order by small epilogue kernels: no float atomics, bit-stable results.
//
// Gaussian pixels use the real-arithmetic form of eqs (16)/(17) derived in DESIGN.md and pinned by
// tests/test_oracle_entry.py::test_real_form_identity_used_by_the_cuda_kernels:
//    q = w s^2, den = 1 + q^2, A = -pi s^2 ((u - w l)^2 + (v - w m)^2)/den  (<= 0, no overflow)
//    M = a/den (1 + i q) exp(A) exp(-i (X - q A)),   X = the delta-pixel phase with n' = n - 1
//    (eq 17) or n' = -r^2/2 (eq 16).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <type_traits>
#ifdef SL1M_BOUNDS
#include <cassert>
#endif

namespace sl1m {

constexpr int TP = 256;        // pixels per tile (one fp64 centre per tile)
constexpr int NT = 128;        // threads per CTA in the apply kernels
constexpr int VC = 128;        // visibilities per staged chunk in the adjoint
constexpr int PIX_PAD = 1024;
constexpr int NPAIR_X2 = 4;    // register pairs per thread in the packed kernels  // pixel arrays are padded to a multiple of this
constexpr double TWO_PI = 6.283185307179586476925286766559;

struct ApplyParams {
    // visibilities (caller order)
    int n_vis;
    const double *u64, *v64, *w64;  // [n_vis]
    const int *ant_p, *ant_q;       // [n_vis] (gains only)
    // pixels (sorted order, padded)
    int n_pix_pad;
    int n_tiles;                    // n_pix_pad / TP
    const float4 *pix4;             // [n_pix_pad] (dl, dm, dn', a*x)   .w rewritten per forward
    const float2 *pixg;             // [n_pix_pad] (sigma^2, -pi log2(e) sigma^2)  (Gaussian only)
    const double4 *cen;             // [n_tiles]   (l_c, m_c, n'_c, 0)
    // zero-skipping forward: when tile_cnt != NULL, pix4 is the COMPACT copy of the
    // tiles -- the pixels of tile t with a*x != 0 moved to its front in their original order -- and
    // tile_cnt[c][t] is how many of them the forward has to stream (rounded up to a multiple of 4, the
    // padding entries carry a*x = 0).  Exact: a skipped term is a*x*M_jk = 0.  Unit-gain kernels only.
    const int *tile_cnt;            // [n_chan][n_tiles] or NULL (dense: every tile has TP pixels)
    const float2 *gFc;              // [n_chan][n_pix_pad][n_ant] gain rows of the compact entries of every tile
                                    // that is not full (a full tile is read from gF); gain plans only
    // gains
    int n_ant;
    const float2 *gF;               // [n_pix_pad][n_ant]  forward layout
    const float2 *gA;               // [n_ant][n_pix_pad]  adjoint layout
    // split bookkeeping
    int per_split;                  // forward: pixel tiles per split; adjoint: vis chunks per split
    // I/O
    const float2 *r;                // adjoint input [n_vis] (re, im)
    float2 *ws_v;                   // forward partials [n_split][n_vis]
    float *ws_p;                    // adjoint partials [n_split][n_pix_pad]
    // batched channels (NEXT-4): blockIdx.z = channel c.  Channel c sees the baselines u, v, w
    // scaled by chan_scale[c] (= nu_c / nu_0, "b = lambda (u, v, w)"), its own a*x in
    // pix4[c][.].w, its own residual r[c][.] and its own partials.  chan_scale == NULL: one channel.
    const double *chan_scale;       // [n_chan] or NULL
    size_t ws_v_stride, ws_p_stride;   // elements per channel of ws_v / ws_p
    // device-side termination (sl1m_solve_stop): done[c] != 0 once channel c has met its stopping rule; every
    // kernel of the iteration then returns at once for that channel, so the iterations the host had already
    // enqueued cost a few microseconds and the image stays the one of the stopping iteration.  NULL = never.
    const int *done;                // [n_chan] or NULL
    // antenna-major compact gains of the packed gain forward (fwd_kernel_x2<GAINS>): gAc[c][a][k] holds, for every
    // tile that was compacted, the gains of its compact entries in the row layout of gA
    const float2 *gAc;              // [n_chan][n_ant][n_pix_pad] (+ padding) or NULL
#ifdef SL1M_BOUNDS
    // debug build (-DSL1M_BOUNDS): one-past-the-end of the two gain tables, padding rows included; every
    // forward-layout gain load (the register prefetches run up to 4 rows past the pixels in use) is asserted in range
    const float2 *gF_end, *gFc_end, *gA_end, *gAc_end;
#endif
};

// Forward-layout gain load.  The kernels prefetch rows ahead of the pixel they are on -- up to 4 rows past the last
// pixel in use, which the tables' padding rows absorb.  The debug build asserts that every such address is inside
// one of the two tables (compute-sanitizer is not available on the pool; tests/test_gpu_bounds.py runs this build).
__device__ __forceinline__ float2 ldg_gain(const ApplyParams &P, const float2 *q) {
#ifdef SL1M_BOUNDS
    assert((q >= P.gF && q < P.gF_end) || (P.gFc && q >= P.gFc && q < P.gFc_end));
#endif
    return __ldg(q);
}

// Two consecutive pixels of one antenna's row of the antenna-major tables (gA / gAc), 16-byte aligned.
__device__ __forceinline__ float4 ldg_gain4(const ApplyParams &P, const float4 *q) {
#ifdef SL1M_BOUNDS
    const float2 *q2 = reinterpret_cast<const float2 *>(q);
    assert((q2 >= P.gA && q2 + 2 <= P.gA_end) || (P.gAc && q2 >= P.gAc && q2 + 2 <= P.gAc_end));
#endif
    return __ldg(q);
}

// BATCH is a compile-time switch: the single-channel instantiations carry no channel arithmetic at
// all (measured: even a live fp64 scale register costs the packed forward kernel 7 %).
template <bool BATCH>
__device__ __forceinline__ double chan_scale_of(const ApplyParams &P) {
    return BATCH ? P.chan_scale[blockIdx.z] : 1.0;
}
template <bool BATCH>
__device__ __forceinline__ size_t chan_index() {
    return BATCH ? (size_t)blockIdx.z : (size_t)0;
}
// pixels of tile t the forward streams (a multiple of 4; TP without the zero-skipping compaction)
template <bool BATCH>
__device__ __forceinline__ int tile_pixels(const ApplyParams &P, int t) {
    return P.tile_cnt ? __ldg(P.tile_cnt + chan_index<BATCH>() * P.n_tiles + t) : TP;
}
// Adjoint CTA -> (pixel group, visibility split).  The grid is (pixel groups, splits) and CTAs are scheduled in
// linear order, x fastest.  With a gain table the CTAs resident at one time should share PIXEL GROUPS (their gain
// columns gA[a][group] then stay in L2 across the splits) instead of sharing a split: config 4 read the 256 MiB
// table from DRAM once per split (11.5 GB per launch, profiles/r1_ncu_full_gain_kernels_config4.md).  SWAP makes
// the split the fast index of the linear CTA number.
template <bool SWAP>
__device__ __forceinline__ void adj_cta(int &group, int &split) {
    if (SWAP) {
        const unsigned lin = blockIdx.y * gridDim.x + blockIdx.x;
        group = (int)(lin / gridDim.y);
        split = (int)(lin - (unsigned)group * gridDim.y);
    } else {
        group = (int)blockIdx.x;
        split = (int)blockIdx.y;
    }
}
// forward-layout gain rows of tile t: the compact copy when the tile was compacted (npx < TP), else the table
template <bool BATCH>
__device__ __forceinline__ const float2 *tile_gain_rows(const ApplyParams &P, int t, int npx) {
    const float2 *g = (P.tile_cnt && npx < TP) ? P.gFc + chan_index<BATCH>() * (size_t)P.n_pix_pad * P.n_ant : P.gF;
    return g + (size_t)t * TP * P.n_ant;
}

// ------------------------------------------------------------------------------------------
// PTX helpers: mbarrier + 1-D TMA bulk copy (cp.async.bulk -> SASS UBLKCP)
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    uint32_t ok = 0;
    const uint32_t a = smem_u32(bar);
    while (!ok) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok)
            : "r"(a), "r"(parity)
            : "memory");
    }
}
__device__ __forceinline__ void tma_bulk_g2s(void *dst_smem, const void *src_gmem, uint32_t bytes,
                                             uint64_t *bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
            "r"(smem_u32(dst_smem)),
        "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}
__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcp_approx(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// x0 = 2 pi * frac(u l_c + v m_c + w n'_c), fp64, reduced to [-pi, pi] before rounding to fp32.
__device__ __forceinline__ float centre_phase(double u, double v, double w, const double4 &c) {
    double t = fma(u, c.x, fma(v, c.y, w * c.z));
    t -= rint(t);
    return static_cast<float>(t * TWO_PI);
}

// sin/cos on the FMA pipe (no MUFU): X = k pi + r, r in [-pi/2, pi/2]; sin r by an odd degree-9 and cos r
// by an even degree-8 near-minimax polynomial (Chebyshev-node fits on z = r^2 over [0, (1.02 pi/2)^2];
// max abs error 1.2e-7 / 2.9e-7 in fp32, i.e. at least as accurate as MUFU.SIN/COS).  Returns
// sin r, cos r and the sign bit (-1)^k as a mask to be XOR-ed into whatever multiplies them.
// Used for a fixed fraction of the terms so that the FMA pipe, which the MUFU-bound loop leaves
// two-thirds idle, carries part of the transcendental load.
__device__ __forceinline__ void sincos_poly(float X, float &s, float &c, uint32_t &sign) {
    const float kf = fmaf(X, 0.318309886183790672f, 12582912.0f);  // 1.5*2^23: k in the low mantissa bits
    const float kr = kf - 12582912.0f;
    const float r = fmaf(kr, -3.14159265358979324f, X);
    const float z = r * r;
    float ps = fmaf(z, 2.629978780532838e-06f, -0.00019821235036943108f);
    ps = fmaf(z, ps, 0.008333230391144753f);
    ps = fmaf(z, ps, -0.1666666567325592f);
    s = fmaf(r * z, ps, r);
    float pc = fmaf(z, 2.3423957827617414e-05f, -0.0013866969384253025f);
    pc = fmaf(z, pc, 0.04166554659605026f);
    pc = fmaf(z, pc, -0.49999991059303284f);
    c = fmaf(z, pc, 1.0f);
    sign = __float_as_uint(kf) << 31;
}
__device__ __forceinline__ float fxor(float a, uint32_t m) { return __uint_as_float(__float_as_uint(a) ^ m); }
// sin x, cos x by the same polynomials, signs applied (centre-phase rotations of the gain kernels: once per
// (visibility, tile), as accurate as the polynomial terms, no MUFU, no slow-path stack frame)
__device__ __forceinline__ void sincos_fma(float X, float &s, float &c) {
    uint32_t sg;
    sincos_poly(X, s, c, sg);
    s = fxor(s, sg);
    c = fxor(c, sg);
}

// ------------------------------------------------------------------------------------------
// Packed fp32 pairs (sm_100a FFMA2/FMUL2/FADD2): one issue slot carries two FMAs.  The MUFU-bound
// loop is limited by issue slots as soon as part of the sincos load moves to the FMA pipe, so the
// delta-pixel kernels keep a thread's 8 register-tile entries as 4 pairs.
// ------------------------------------------------------------------------------------------
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float lo, float hi) {
    f32x2 d;
    asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(lo), "f"(hi));
    return d;
}
__device__ __forceinline__ f32x2 bc2(float x) { return pk2(x, x); }
__device__ __forceinline__ void up2(f32x2 d, float &lo, float &hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(d));
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
    f32x2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) {
    f32x2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) {
    f32x2 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}

// sincos_poly on a pair: same reduction and polynomials, 13 packed instructions for two terms.
// sg_lo / sg_hi: the integer k of each lane in the low mantissa bits (bit 0 = parity = sign flip).
__device__ __forceinline__ void sincos_poly2(f32x2 X, f32x2 &s, f32x2 &c, uint32_t &k_lo, uint32_t &k_hi) {
    const f32x2 kf = fma2(X, bc2(0.318309886183790672f), bc2(12582912.0f));
    const f32x2 kr = add2(kf, bc2(-12582912.0f));
    const f32x2 r = fma2(kr, bc2(-3.14159265358979324f), X);
    const f32x2 z = mul2(r, r);
    f32x2 ps = fma2(z, bc2(2.629978780532838e-06f), bc2(-0.00019821235036943108f));
    ps = fma2(z, ps, bc2(0.008333230391144753f));
    ps = fma2(z, ps, bc2(-0.1666666567325592f));
    s = fma2(mul2(r, z), ps, r);
    f32x2 pc = fma2(z, bc2(2.3423957827617414e-05f), bc2(-0.0013866969384253025f));
    pc = fma2(z, pc, bc2(0.04166554659605026f));
    pc = fma2(z, pc, bc2(-0.49999991059303284f));
    c = fma2(z, pc, bc2(1.0f));
    float a, b;
    up2(kf, a, b);
    k_lo = __float_as_uint(a);
    k_hi = __float_as_uint(b);
}
// x with its sign flipped when k is odd: x_bits + (k << 31) (an LEA on the ALU pipe).
__device__ __forceinline__ float flip_if_odd(float x, uint32_t k) {
    return __uint_as_float(__float_as_uint(x) ^ (k << 31));     // SHL + LOP3 (ALU pipe; an IMAD add was measured no faster)
}

// One generated term.  X is the delta-pixel phase (radians).  Returns the complex entry WITHOUT
// the per-pixel amplitude a_k (forward folds a_k x_k into `wt`; adjoint applies a_k at the end).
//   delta:    e = (cos X, -sin X)
//   Gaussian: e = (1/den) 2^E2 (1 + i q)(cos X' - i sin X'),  X' = X - q A,  A = E2 ln 2
// POLY (delta pixels only): sin/cos from sincos_poly; the caller applies `sign` to its multiplier.
template <int PK, bool POLY>
__device__ __forceinline__ void gen_entry(float X, float du, float dv, float w, float sig2,
                                          float nsp, float &ere, float &eim, uint32_t &sign) {
    sign = 0u;
    if (PK == 0) {
        float s, c;
        if (POLY) sincos_poly(X, s, c, sign); else __sincosf(X, &s, &c);
        ere = c;
        eim = -s;
    } else {
        const float q = w * sig2;
        const float den = fmaf(q, q, 1.0f);
        const float rden = rcp_approx(den);
        const float s2 = fmaf(dv, dv, du * du);
        const float E2 = (s2 * rden) * nsp;                 // log2 of the Gaussian amplitude (<= 0)
        const float amp = ex2_approx(E2) * rden;
        const float Xp = fmaf(-0.69314718056f * q, E2, X);  // X - q A
        float s, c;
        __sincosf(Xp, &s, &c);
        ere = amp * fmaf(q, s, c);                          // Re (1+iq)(c - is) = c + q s
        eim = amp * fmaf(q, c, -s);                         // Im               = q c - s
    }
}

// Gaussian pixels with ONE sigma per tile (PK == 2): everything that depends only on (visibility, tile)
// is hoisted out of the term.  With q = w s^2, den = 1 + q^2:
//   E' = s2 * cE + lr,  cE = -pi log2(e) s^2 / den,  lr = log2(1/den)   =>  2^E' = e^A / den
//   X' = X - q A = (X + q ln2 lr) - q ln2 E'                              (the lr part is folded into x0)
//   entry = 2^E' (1 + i q)(cos X' - i sin X')
// per term: 15 FP32 + 3 MUFU (ex2, sin, cos) instead of 20 + 4.
__device__ __forceinline__ void gauss_tile_constants(double w, double sig2, float &q, float &cE, float &lr,
                                                     float &x0) {
    const double qd = w * sig2;
    const double rden = 1.0 / (1.0 + qd * qd);
    q = static_cast<float>(qd);
    cE = static_cast<float>(-3.14159265358979323846 * 1.4426950408889634074 * sig2 * rden);
    const double lrd = log2(rden);
    lr = static_cast<float>(lrd);
    // fold q ln2 lr into the centre phase, reduced again to [-pi, pi]
    double t = (static_cast<double>(x0) + 0.69314718055994530942 * qd * lrd) * (1.0 / TWO_PI);
    t -= rint(t);
    x0 = static_cast<float>(t * TWO_PI);
}
// entry = amp (cr + i ci); the caller folds amp into its own multiplier (a x, or nothing)
__device__ __forceinline__ void gen_entry_tile(float X, float du, float dv, float q, float cE, float lr,
                                               float &amp, float &cr, float &ci) {
    const float s2 = fmaf(dv, dv, du * du);
    const float Ep = fmaf(s2, cE, lr);
    const float Xp = fmaf(-0.69314718056f * q, Ep, X);   // -ln2 q is loop-invariant: hoisted by the compiler
    amp = ex2_approx(Ep);
    float s, c;
    __sincosf(Xp, &s, &c);
    cr = fmaf(q, s, c);                                   // Re (1 + i q)(c - i s)
    ci = fmaf(q, c, -s);                                  // Im
}

// Tuning constants of the delta-pixel / unit-gain kernels (measured on B200):
//   *_NPOLY8   how many of a thread's 8 register-tile entries take the polynomial sincos path
//   *_MIN_CTAS resident CTAs per SM the kernel is compiled for (register budget 65536/(128*n))
#ifndef SL1M_FWD_NPOLY8
#define SL1M_FWD_NPOLY8 1
#endif
#ifndef SL1M_ADJ_NPOLY8
#define SL1M_ADJ_NPOLY8 2
#endif
//   *_NPQ      packed kernels: how many of every 16 register pairs take the polynomial path
#ifndef SL1M_FWD_NPQ
#define SL1M_FWD_NPQ 4
#endif
//   *_GT_MIN_CTAS  the one-sigma-per-tile Gaussian kernels (PK == 2)
#ifndef SL1M_FWD_GT_MIN_CTAS
#define SL1M_FWD_GT_MIN_CTAS 4
#endif
#ifndef SL1M_ADJ_GT_MIN_CTAS
#define SL1M_ADJ_GT_MIN_CTAS 5
#endif
//   *_G2_NPQ   the same fraction for the packed kernels with baseline-grouped gains
#ifndef SL1M_FWD_G2_NPQ
#define SL1M_FWD_G2_NPQ 3
#endif
#ifndef SL1M_ADJ_G2_NPQ
#define SL1M_ADJ_G2_NPQ 1
#endif
#ifndef SL1M_FWD_X2_MIN_CTAS
#define SL1M_FWD_X2_MIN_CTAS 4
#endif
#ifndef SL1M_FWD_MIN_CTAS
#define SL1M_FWD_MIN_CTAS 5
#endif
#ifndef SL1M_ADJ_MIN_CTAS
#define SL1M_ADJ_MIN_CTAS 6
#endif
template <int R, int PK, int GK, int NPOLY8>
struct PolySplit {
    static constexpr int N = (PK != 0 || GK != 0) ? 0 : (R == 8 ? NPOLY8 : (R == 4 ? NPOLY8 / 2 : 0));
};

// ------------------------------------------------------------------------------------------
// forward:  ws_v[split][j] = sum_{k in split} M_jk x_k        (a1)
// grid = (vis tiles of NT*RV, pixel splits); block = NT
// ------------------------------------------------------------------------------------------
template <int RV, int PK, int GK, bool BATCH = false>
#ifndef SL1M_FWD_G1_MIN_CTAS
#define SL1M_FWD_G1_MIN_CTAS 4   // per-term gains: 255 registers (2 CTAs/SM) left the gain loads latency-bound: 9.27 -> 4.67 ms at config 4 with 2 samples per baseline
#endif
__global__ void __launch_bounds__(NT, (PK == 0 && GK == 0) ? SL1M_FWD_MIN_CTAS : (GK == 2 ? 4 : (PK == 2 ? SL1M_FWD_GT_MIN_CTAS : (PK == 0 && GK == 1 ? SL1M_FWD_G1_MIN_CTAS : 1)))) fwd_kernel(const ApplyParams P) {
    if (BATCH && P.done && P.done[blockIdx.z]) return;   // batched solve: this channel has met its stopping rule
    __shared__ __align__(128) float4 s_pix[2][TP];
    __shared__ __align__(128) float2 s_pixg[PK == 1 ? 2 : 1][PK == 1 ? TP : 1];
    __shared__ __align__(8) uint64_t s_bar[2];

    const int tid = threadIdx.x;
    const int t0 = blockIdx.y * P.per_split;
    const int t1 = min(t0 + P.per_split, P.n_tiles);
    const int jbase = blockIdx.x * (NT * RV);

    // fp64 uvw are re-read from global (L1/L2-resident) once per pixel tile instead of living in
    // 6 registers per visibility: the register budget buys occupancy (6 CTAs per SM).
    float uf[RV], vf[RV], wf[RV], wl[RV], re[RV], im[RV];
    int ap[RV], aq[RV];
    const int jlast = P.n_vis - 1;
    const double sc = chan_scale_of<BATCH>(P);
    const float4 *pix4 = P.pix4 + chan_index<BATCH>() * P.n_pix_pad;
#pragma unroll
    for (int r = 0; r < RV; ++r) {
        const int j = min(jbase + r * NT + tid, jlast);
        const double wd = sc * __ldg(P.w64 + j);
        uf[r] = static_cast<float>(TWO_PI * (sc * __ldg(P.u64 + j)));
        vf[r] = static_cast<float>(TWO_PI * (sc * __ldg(P.v64 + j)));
        wf[r] = static_cast<float>(TWO_PI * wd);
        wl[r] = static_cast<float>(wd);
        re[r] = 0.f;
        im[r] = 0.f;
        if (GK) {
            ap[r] = P.ant_p[j];
            aq[r] = P.ant_q[j];
        }
    }
    // GK == 2 ("baseline-grouped" plan): the plan laid the visibilities out so that a thread's RV
    // entries are samples of ONE baseline (p, q): the gain product G is loaded once per pixel.
    static_assert(GK != 2 || RV == 8, "grouped gains need RV == 8");

    constexpr bool ZSKIP = true;        // zero-skipping in every variant; PK == 1 streams the compact copy of its side array too
    if (tid == 0) {
        mbar_init(&s_bar[0], 1);
        mbar_init(&s_bar[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    // P.pixg: the plan's [n_pix_pad] array, or with zero-skipping its per-channel compact copy [n_chan][n_pix_pad]
    const float2 *pixg = (PK == 1 && P.tile_cnt) ? P.pixg + chan_index<BATCH>() * P.n_pix_pad : P.pixg;
    auto issue = [&](int t, int st) {
        const uint32_t n4 = (uint32_t)(ZSKIP ? max(tile_pixels<BATCH>(P, t), 4) : TP);
        const uint32_t b4 = n4 * (uint32_t)sizeof(float4);
        mbar_expect_tx(&s_bar[st], b4 + (PK == 1 ? n4 * (uint32_t)sizeof(float2) : 0u));
        tma_bulk_g2s(&s_pix[st][0], pix4 + (size_t)t * TP, b4, &s_bar[st]);
        if (PK == 1) tma_bulk_g2s(&s_pixg[st][0], pixg + (size_t)t * TP, n4 * (uint32_t)sizeof(float2), &s_bar[st]);
    };
    if (tid == 0) {
        if (t0 < t1) issue(t0, 0);
        if (t0 + 1 < t1) issue(t0 + 1, 1);
    }

    for (int t = t0; t < t1; ++t) {
        const int st = (t - t0) & 1;
        const uint32_t parity = ((t - t0) >> 1) & 1;
        const double4 c = P.cen[t];
        const int npx = ZSKIP ? tile_pixels<BATCH>(P, t) : TP;
        float x0[RV], uc[RV], vc[RV];
        float tq[PK == 2 ? RV : 1], tcE[PK == 2 ? RV : 1], tlr[PK == 2 ? RV : 1];   // per-(visibility, tile) constants
#pragma unroll
        for (int r = 0; r < RV; ++r) {
            if (ZSKIP && npx == 0) continue;     // empty tile (uniform over the CTA): nothing to prepare
            const int j = min(jbase + r * NT + tid, jlast);
            const double ud = sc * __ldg(P.u64 + j), vd = sc * __ldg(P.v64 + j), wd = sc * __ldg(P.w64 + j);
            x0[r] = centre_phase(ud, vd, wd, c);
            if (PK) {
                uc[r] = static_cast<float>(ud - wd * c.x);
                vc[r] = static_cast<float>(vd - wd * c.y);
            }
            if (PK == 2) gauss_tile_constants(wd, c.w, tq[r], tcE[r], tlr[r], x0[r]);
        }
        mbar_wait(&s_bar[st], parity);
        const float2 *gbase = GK ? tile_gain_rows<BATCH>(P, t, npx) : nullptr;
        // grouped gains: register prefetch two pixels ahead (rows are cold in L1 on first touch)
        float2 gp0, gq0, gp1, gq1;
        if (GK == 2) {
            gp0 = ldg_gain(P, gbase + ap[0]);
            gq0 = ldg_gain(P, gbase + aq[0]);
            gp1 = ldg_gain(P, gbase + P.n_ant + ap[0]);
            gq1 = ldg_gain(P, gbase + P.n_ant + aq[0]);
        }
#pragma unroll 2
        for (int p = 0; p < npx; ++p) {
            const float4 px = s_pix[st][p];
            // gains are stored in polar form (|g|, arg g):  G = g_p conj(g_q) = |g_p||g_q| e^{i(arg_p - arg_q)}
            // multiplies the entry by a real factor and shifts its phase: M x = (a x |G|) e^{-i(X - gamma)}
            float Gw = px.w, gam = 0.f;
            if (GK == 2) {
                const float2 gp = gp0, gq = gq0;
                gp0 = gp1;
                gq0 = gq1;
                const int pn = min(p + 2, TP - 1);
                gp1 = ldg_gain(P, gbase + (size_t)pn * P.n_ant + ap[0]);
                gq1 = ldg_gain(P, gbase + (size_t)pn * P.n_ant + aq[0]);
                Gw = px.w * (gp.x * gq.x);
                gam = gp.y - gq.y;
            }
            float sig2 = 0.f, nsp = 0.f;
            if (PK == 1) {
                const float2 pg = s_pixg[st][p];
                sig2 = pg.x;
                nsp = pg.y;
            }
#pragma unroll
            for (int r = 0; r < RV; ++r) {
                float X = fmaf(uf[r], px.x, fmaf(vf[r], px.y, fmaf(wf[r], px.z, x0[r])));
                float wg = Gw;
                if (GK == 2) X -= gam;
                if (GK == 1) {
                    const float2 gp = ldg_gain(P, gbase + (size_t)p * P.n_ant + ap[r]);
                    const float2 gq = ldg_gain(P, gbase + (size_t)p * P.n_ant + aq[r]);
                    wg = px.w * (gp.x * gq.x);
                    X -= gp.y - gq.y;
                }
                float du = 0.f, dv = 0.f;
                if (PK) {
                    du = fmaf(-wl[r], px.x, uc[r]);
                    dv = fmaf(-wl[r], px.y, vc[r]);
                }
                float ere, eim;
                uint32_t sgn;
                if (PK == 2) {
                    float amp;
                    gen_entry_tile(X, du, dv, tq[r], tcE[r], tlr[r], amp, ere, eim);
                    const float t = wg * amp;
                    re[r] = fmaf(t, ere, re[r]);
                    im[r] = fmaf(t, eim, im[r]);
                    continue;
                }
                if (r < PolySplit<RV, PK, GK, SL1M_FWD_NPOLY8>::N) gen_entry<PK, true>(X, du, dv, wl[r], sig2, nsp, ere, eim, sgn);
                else gen_entry<PK, false>(X, du, dv, wl[r], sig2, nsp, ere, eim, sgn);
                const float wt = (r < PolySplit<RV, PK, GK, SL1M_FWD_NPOLY8>::N) ? fxor(wg, sgn) : wg;
                re[r] = fmaf(wt, ere, re[r]);
                im[r] = fmaf(wt, eim, im[r]);
            }
        }
        __syncthreads();  // every thread is done with stage st
        if (tid == 0 && t + 2 < t1) issue(t + 2, st);
    }

    float2 *out = P.ws_v + chan_index<BATCH>() * P.ws_v_stride + (size_t)blockIdx.y * P.n_vis;
#pragma unroll
    for (int r = 0; r < RV; ++r) {
        const int j = jbase + r * NT + tid;
        if (j < P.n_vis) out[j] = make_float2(re[r], im[r]);
    }
}

// ------------------------------------------------------------------------------------------
// forward, delta pixels / unit gains, packed-pair variant (the configs 1, 2, 5 path at RV = 8).
// A thread's 8 visibilities are 4 register pairs; per pixel and pair: 3 FFMA2 (phase) + either
// {2 FMUL.RZ, 4 MUFU} or the 13-instruction packed polynomial + 2 FFMA2 (accumulate).  NP16 of
// every 16 terms (2 consecutive pixels x 8 visibilities) take the polynomial path; NP16 is even
// (whole pairs).  im is accumulated with the opposite sign and negated in the epilogue.
// ------------------------------------------------------------------------------------------
template <int NPQ, bool BATCH = false, bool GAINS = false>
__global__ void __launch_bounds__(NT, SL1M_FWD_X2_MIN_CTAS) fwd_kernel_x2(const ApplyParams P) {
    if (BATCH && P.done && P.done[blockIdx.z]) return;   // batched solve: this channel has met its stopping rule
    constexpr int RV = 8, NPAIR = 4;
    // NPQ of the 16 pairs of 4 consecutive pixels take the polynomial path: pixel q gets (NPQ + 3 - q) / 4
    __shared__ __align__(128) float4 s_pix[2][TP];
    __shared__ __align__(8) uint64_t s_bar[2];
    // GAINS: RE/IM hold the sums of ONE tile without its centre phase; the running totals live here
    // ([pair][thread], own slots only) and take e^{-i x0} (tile sum) at the end of every tile.
    __shared__ __align__(8) f32x2 s_tot[GAINS ? 2 * NPAIR_X2 : 1][GAINS ? NT : 1];

    const int tid = threadIdx.x;
    const int t0 = blockIdx.y * P.per_split;
    const int t1 = min(t0 + P.per_split, P.n_tiles);
    const int jbase = blockIdx.x * (NT * RV);
    const int jlast = P.n_vis - 1;
    const double sc = chan_scale_of<BATCH>(P);
    const float4 *pix4 = P.pix4 + chan_index<BATCH>() * P.n_pix_pad;

    f32x2 U[NPAIR], V[NPAIR], W[NPAIR], RE[NPAIR], IM[NPAIR];
#pragma unroll
    for (int i = 0; i < NPAIR; ++i) {
        const int ja = min(jbase + (2 * i) * NT + tid, jlast), jb = min(jbase + (2 * i + 1) * NT + tid, jlast);
        U[i] = pk2(static_cast<float>(TWO_PI * (sc * __ldg(P.u64 + ja))), static_cast<float>(TWO_PI * (sc * __ldg(P.u64 + jb))));
        V[i] = pk2(static_cast<float>(TWO_PI * (sc * __ldg(P.v64 + ja))), static_cast<float>(TWO_PI * (sc * __ldg(P.v64 + jb))));
        W[i] = pk2(static_cast<float>(TWO_PI * (sc * __ldg(P.w64 + ja))), static_cast<float>(TWO_PI * (sc * __ldg(P.w64 + jb))));
        RE[i] = pk2(0.f, 0.f);
        IM[i] = pk2(0.f, 0.f);
        if (GAINS) {
            s_tot[i][tid] = pk2(0.f, 0.f);
            s_tot[NPAIR + i][tid] = pk2(0.f, 0.f);
        }
    }
    // GAINS ("baseline-grouped" plan, gk == 2): the thread's 8 visibilities are samples of ONE baseline
    // (p, q).  Gains are stored in polar form (|g|, arg g), so G = g_p conj(g_q) = |G| e^{i gamma} with
    // |G| = |g_p||g_q|, gamma = arg_p - arg_q, formed once per pixel and shared by the 4 pairs:
    //     M_jk x_k = (a x |G|) e^{-i (X_rel - gamma)} e^{-i x0(j, tile)}
    // -gamma is the innermost addend of the phase FMA chain (where the unit-gain kernel has x0) and the
    // weight stays real: the term costs what a unit-gain term costs.  e^{-i x0} multiplies the tile's sum.
    int ap = 0, aq = 0;
    if (GAINS) {
        const int j0 = min(jbase + tid, jlast);
        ap = P.ant_p[j0];
        aq = P.ant_q[j0];
    }

    if (tid == 0) {
        mbar_init(&s_bar[0], 1);
        mbar_init(&s_bar[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    auto issue = [&](int t, int st) {   // only the pixels the tile has to stream (an empty tile still moves 64 B: barrier phases stay in step)
        const uint32_t bytes = (uint32_t)max(tile_pixels<BATCH>(P, t), 4) * (uint32_t)sizeof(float4);
        mbar_expect_tx(&s_bar[st], bytes);
        tma_bulk_g2s(&s_pix[st][0], pix4 + (size_t)t * TP, bytes, &s_bar[st]);
    };
    if (tid == 0) {
        if (t0 < t1) issue(t0, 0);
        if (t0 + 1 < t1) issue(t0 + 1, 1);
    }

    // one pixel against the 4 pairs; the first NPOLY pairs use the FMA-pipe polynomial
    // wgt: the real weight of the pixel (a x, times |G| with gains); ngam: -gamma (gains only)
    auto pixel = [&](const float4 px, const f32x2 (&X0)[NPAIR], auto npoly_tag, float wgt, float ngam) {
        constexpr int NPOLY = decltype(npoly_tag)::value;
        const f32x2 pxx = bc2(px.x), pxy = bc2(px.y), pxz = bc2(px.z);
#pragma unroll
        for (int i = 0; i < NPAIR; ++i) {
            const f32x2 X = fma2(U[i], pxx, fma2(V[i], pxy, fma2(W[i], pxz, GAINS ? bc2(ngam) : X0[i])));
            if (i < NPOLY) {
                f32x2 s, c;
                uint32_t ka, kb;
                sincos_poly2(X, s, c, ka, kb);
                const f32x2 wt = pk2(flip_if_odd(wgt, ka), flip_if_odd(wgt, kb));
                RE[i] = fma2(wt, c, RE[i]);
                IM[i] = fma2(wt, s, IM[i]);
            } else {
                float xa, xb, sa, ca, sb, cb;
                up2(X, xa, xb);
                __sincosf(xa, &sa, &ca);
                __sincosf(xb, &sb, &cb);
                const f32x2 wt = bc2(wgt);
                RE[i] = fma2(wt, pk2(ca, cb), RE[i]);
                IM[i] = fma2(wt, pk2(sa, sb), IM[i]);
            }
        }
    };

    for (int t = t0; t < t1; ++t) {
        const int st = (t - t0) & 1;
        const uint32_t parity = ((t - t0) >> 1) & 1;
        const int npx = tile_pixels<BATCH>(P, t);   // zero-skipping: pixels with a*x != 0 (all TP when dense)
        f32x2 X0[NPAIR];
        if (!GAINS && npx > 0) {
            const double4 c = P.cen[t];
#pragma unroll
            for (int i = 0; i < NPAIR; ++i) {
                const int ja = min(jbase + (2 * i) * NT + tid, jlast), jb = min(jbase + (2 * i + 1) * NT + tid, jlast);
                X0[i] = pk2(centre_phase(sc * __ldg(P.u64 + ja), sc * __ldg(P.v64 + ja), sc * __ldg(P.w64 + ja), c),
                            centre_phase(sc * __ldg(P.u64 + jb), sc * __ldg(P.v64 + jb), sc * __ldg(P.w64 + jb), c));
            }
        }
        mbar_wait(&s_bar[st], parity);
        if (GAINS) {
            // Gains of the tile for the thread's two antennas, read from the ANTENNA-MAJOR table gA[a][k] (the
            // adjoint's layout; gAc[c][a][k] holds the compact entries of a tile that was compacted): the thread
            // walks two contiguous rows, so 4 pixels are 4 LDG.128 at pointer + immediate instead of 8 LDG.64 with
            // a 64-bit index computation each (46 -> 6 integer instructions per 32 terms).  A lane's 128-byte line
            // serves its next 16 pixels; a CTA keeps <= 2 x 128 such lines live, well inside L1.  Register prefetch
            // one group of 4 pixels ahead; the rows carry 4 entries of padding behind the last tile.
            const bool compacted = P.tile_cnt && npx < TP;
            const float2 *grow = compacted ? P.gAc + chan_index<BATCH>() * (size_t)P.n_ant * P.n_pix_pad : P.gA;
            const float4 *pp = reinterpret_cast<const float4 *>(grow + (size_t)ap * P.n_pix_pad + (size_t)t * TP);
            const float4 *pq = reinterpret_cast<const float4 *>(grow + (size_t)aq * P.n_pix_pad + (size_t)t * TP);
            float4 gp01 = ldg_gain4(P, pp), gp23 = ldg_gain4(P, pp + 1), gq01 = ldg_gain4(P, pq), gq23 = ldg_gain4(P, pq + 1);
#pragma unroll 1
            for (int p = 0; p < npx; p += 4) {
                float Gw[4], Ng[4];
                Gw[0] = s_pix[st][p].w * (gp01.x * gq01.x);                    // a x |g_p||g_q|
                Ng[0] = gq01.y - gp01.y;                                       // -gamma
                Gw[1] = s_pix[st][p + 1].w * (gp01.z * gq01.z);
                Ng[1] = gq01.w - gp01.w;
                Gw[2] = s_pix[st][p + 2].w * (gp23.x * gq23.x);
                Ng[2] = gq23.y - gp23.y;
                Gw[3] = s_pix[st][p + 3].w * (gp23.z * gq23.z);
                Ng[3] = gq23.w - gp23.w;
                pp += 2;
                pq += 2;
                gp01 = ldg_gain4(P, pp);                     // entries past npx exist (stale, next tile or padding): harmless prefetch
                gp23 = ldg_gain4(P, pp + 1);
                gq01 = ldg_gain4(P, pq);
                gq23 = ldg_gain4(P, pq + 1);
                pixel(s_pix[st][p], X0, std::integral_constant<int, (NPQ + 3) / 4>{}, Gw[0], Ng[0]);
                pixel(s_pix[st][p + 1], X0, std::integral_constant<int, (NPQ + 2) / 4>{}, Gw[1], Ng[1]);
                pixel(s_pix[st][p + 2], X0, std::integral_constant<int, (NPQ + 1) / 4>{}, Gw[2], Ng[2]);
                pixel(s_pix[st][p + 3], X0, std::integral_constant<int, NPQ / 4>{}, Gw[3], Ng[3]);
            }
            if (npx > 0) {   // totals += e^{-i x0} (RE - i IM):  re += RE c0 - IM s0,  -im += RE s0 + IM c0
                const double4 c = P.cen[t];
#pragma unroll
                for (int i = 0; i < NPAIR; ++i) {
                    const int ja = min(jbase + (2 * i) * NT + tid, jlast), jb = min(jbase + (2 * i + 1) * NT + tid, jlast);
                    float sa, ca, sb, cb;
                    sincos_fma(centre_phase(sc * __ldg(P.u64 + ja), sc * __ldg(P.v64 + ja), sc * __ldg(P.w64 + ja), c), sa, ca);
                    sincos_fma(centre_phase(sc * __ldg(P.u64 + jb), sc * __ldg(P.v64 + jb), sc * __ldg(P.w64 + jb), c), sb, cb);
                    const f32x2 C0 = pk2(ca, cb), S0 = pk2(sa, sb);
                    s_tot[i][tid] = add2(s_tot[i][tid], fma2(RE[i], C0, mul2(IM[i], pk2(-sa, -sb))));
                    s_tot[NPAIR + i][tid] = add2(s_tot[NPAIR + i][tid], fma2(RE[i], S0, mul2(IM[i], C0)));
                    RE[i] = pk2(0.f, 0.f);
                    IM[i] = pk2(0.f, 0.f);
                }
            }
        } else {
#pragma unroll 1
            for (int p = 0; p < npx; p += 4) {
                pixel(s_pix[st][p], X0, std::integral_constant<int, (NPQ + 3) / 4>{}, s_pix[st][p].w, 0.f);
                pixel(s_pix[st][p + 1], X0, std::integral_constant<int, (NPQ + 2) / 4>{}, s_pix[st][p + 1].w, 0.f);
                pixel(s_pix[st][p + 2], X0, std::integral_constant<int, (NPQ + 1) / 4>{}, s_pix[st][p + 2].w, 0.f);
                pixel(s_pix[st][p + 3], X0, std::integral_constant<int, NPQ / 4>{}, s_pix[st][p + 3].w, 0.f);
            }
        }
        __syncthreads();  // every thread is done with stage st
        if (tid == 0 && t + 2 < t1) issue(t + 2, st);
    }

    float2 *out = P.ws_v + chan_index<BATCH>() * P.ws_v_stride + (size_t)blockIdx.y * P.n_vis;
#pragma unroll
    for (int i = 0; i < NPAIR; ++i) {
        float ra, rb, ia, ib;
        up2(GAINS ? s_tot[i][tid] : RE[i], ra, rb);
        up2(GAINS ? s_tot[NPAIR + i][tid] : IM[i], ia, ib);
        const int ja = jbase + (2 * i) * NT + tid, jb = jbase + (2 * i + 1) * NT + tid;
        if (ja < P.n_vis) out[ja] = make_float2(ra, -ia);
        if (jb < P.n_vis) out[jb] = make_float2(rb, -ib);
    }
}

// ------------------------------------------------------------------------------------------
// adjoint:  ws_p[split][k] = Re sum_{j in split} conj(M_jk / a_k) r_j      (a2)
// grid = (pixel groups of NT*RP, visibility splits); block = NT.
// Warp w owns the 32*RP consecutive sorted pixels starting at base + w*32*RP; with RP = 8 that
// is exactly one tile (one centre per warp), with RP <= 2 the whole CTA sits inside one tile.
// ------------------------------------------------------------------------------------------
template <int RP, int PK, int GK, bool BATCH = false>
__global__ void __launch_bounds__(NT, (PK == 0 && GK == 0) ? SL1M_ADJ_MIN_CTAS : (GK == 2 ? 4 : (PK == 2 ? SL1M_ADJ_GT_MIN_CTAS : 1))) adj_kernel(const ApplyParams P) {
    if (BATCH && P.done && P.done[blockIdx.z]) return;   // batched solve: this channel has met its stopping rule
    constexpr int NCEN = (NT * RP > TP) ? (NT * RP / TP) : 1;
    __shared__ __align__(16) float4 s_vis[2][VC];        // (u', v', w', w)
    __shared__ __align__(8) float2 s_r[2][VC];           // residual (re, im)
    __shared__ float s_x0[2][VC][NCEN];
    __shared__ __align__(8) float2 s_uc[PK ? 2 : 1][PK ? VC : 1][PK ? NCEN : 1];
    __shared__ __align__(16) float4 s_tc[PK == 2 ? 2 : 1][PK == 2 ? VC : 1][PK == 2 ? NCEN : 1];   // (q, cE, lr, x0')
    __shared__ __align__(8) int2 s_ant[GK ? 2 : 1][GK ? VC : 1];   // GK == 2 uses the first VC/8 only

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    int cta_group, cta_split;
    adj_cta<(GK != 0)>(cta_group, cta_split);
    const int base = cta_group * (NT * RP);
    const int kfirst = base + warp * (32 * RP);
    const int tile0 = base / TP;
    const int mycen = (kfirst / TP) - tile0;

    float dl[RP], dm[RP], dn[RP], acc[RP], sig2[RP], nsp[RP];
#pragma unroll
    for (int i = 0; i < RP; ++i) {
        const int k = kfirst + i * 32 + lane;
        const float4 px = P.pix4[k];
        dl[i] = px.x;
        dm[i] = px.y;
        dn[i] = px.z;
        acc[i] = 0.f;
        if (PK == 1) {
            const float2 pg = P.pixg[k];
            sig2[i] = pg.x;
            nsp[i] = pg.y;
        }
    }

    const int n_chunks = (P.n_vis + VC - 1) / VC;
    const double sc = chan_scale_of<BATCH>(P);
    const int c0 = cta_split * P.per_split;
    const int c1 = min(c0 + P.per_split, n_chunks);

    // GK == 2: a chunk is 16 baseline groups x 8 samples.  The plan stores sample r of group g at
    // internal position (g / 128) * 1024 + r * 128 + g % 128 (the forward's thread layout); here
    // it is staged group-major (slot = group * 8 + sample) so 8 consecutive slots share (p, q).
    auto stage = [&](int chunk, int buf) {
        int j = chunk * VC + tid;   // NT == VC
        int slot = tid;
        if (GK == 2) {
            const int g = chunk * (VC / 8) + (tid & 15), r = tid >> 4;
            j = (g >> 7) * (NT * 8) + r * NT + (g & 127);
            slot = (tid & 15) * 8 + r;
        }
        double u = 0.0, v = 0.0, w = 0.0;
        float2 rr = make_float2(0.f, 0.f);
        int2 a = make_int2(0, 0);
        if (j < P.n_vis) {
            u = sc * P.u64[j];
            v = sc * P.v64[j];
            w = sc * P.w64[j];
            rr = P.r[chan_index<BATCH>() * P.n_vis + j];
            if (GK) a = make_int2(P.ant_p[j], P.ant_q[j]);
        }
        s_vis[buf][slot] = make_float4(static_cast<float>(TWO_PI * u), static_cast<float>(TWO_PI * v),
                                       static_cast<float>(TWO_PI * w), static_cast<float>(w));
        // delta pixels: one cosine per term, Re(e^{iX} r) = |r| cos(X + arg r); arg r joins the centre phases below
        float rphi = 0.f;
        if (PK == 0) {
            rphi = atan2f(rr.y, rr.x);
            rr = make_float2(sqrtf(fmaf(rr.x, rr.x, rr.y * rr.y)), 0.f);
        }
        s_r[buf][slot] = rr;
        if (GK == 1) s_ant[buf][slot] = a;
        if (GK == 2 && tid < 16) s_ant[buf][tid] = a;   // sample 0 carries the group's (p, q)
#pragma unroll
        for (int c = 0; c < NCEN; ++c) {
            const double4 cen = P.cen[tile0 + c];   // L1-resident; not worth 24 registers
            float x0c = centre_phase(u, v, w, cen);
            if (PK)
                s_uc[buf][slot][c] = make_float2(static_cast<float>(u - w * cen.x),
                                                 static_cast<float>(v - w * cen.y));
            if (PK == 2) {
                float q, cE, lr;
                gauss_tile_constants(w, cen.w, q, cE, lr, x0c);
                s_tc[buf][slot][c] = make_float4(q, cE, lr, x0c);
            }
            s_x0[buf][slot][c] = x0c + rphi;
        }
    };

    if (c0 < c1) stage(c0, 0);
    __syncthreads();
    for (int ch = c0; ch < c1; ++ch) {
        const int buf = (ch - c0) & 1;
        if (ch + 1 < c1) stage(ch + 1, buf ^ 1);
        // Gains are stored in polar form (|g|, arg g): M = a |G| e(X - gamma), |G| = |g_p||g_q|, gamma = arg_p - arg_q.
        // Grouped gains: (|G_i|, gamma_i) per pixel is formed once per group of 8 samples; the 8 samples
        // accumulate Z_i = sum Re(conj(e(X - gamma_i)) r) first, then acc_i += |G_i| Z_i.
        float Ga[GK == 2 ? RP : 1], Ng[GK == 2 ? RP : 1], Zr[GK == 2 ? RP : 1];
        float2 gpn[GK == 2 ? RP : 1], gqn[GK == 2 ? RP : 1];
        if (GK == 2) {
            const int2 a = s_ant[buf][0];
#pragma unroll
            for (int i = 0; i < RP; ++i) {
                gpn[i] = __ldg(P.gA + (size_t)a.x * P.n_pix_pad + kfirst + lane + i * 32);
                gqn[i] = __ldg(P.gA + (size_t)a.y * P.n_pix_pad + kfirst + lane + i * 32);
            }
        }
        constexpr int GSZ = (GK == 2) ? 8 : VC;   // slots that share one gain product
        for (int tb = 0; tb < VC; tb += GSZ) {
            if (GK == 2) {
                const int2 a = s_ant[buf][min((tb >> 3) + 1, VC / 8 - 1)];
#pragma unroll
                for (int i = 0; i < RP; ++i) {
                    Ga[i] = gpn[i].x * gqn[i].x;
                    Ng[i] = gqn[i].y - gpn[i].y;      // -gamma
                    Zr[i] = 0.f;
                    gpn[i] = __ldg(P.gA + (size_t)a.x * P.n_pix_pad + kfirst + lane + i * 32);
                    gqn[i] = __ldg(P.gA + (size_t)a.y * P.n_pix_pad + kfirst + lane + i * 32);
                }
            }
#pragma unroll 2
          for (int t = tb; t < tb + GSZ; ++t) {
            const float4 vv = s_vis[buf][t];
            const float2 rr = s_r[buf][t];
            const float x0 = s_x0[buf][t][mycen];
            float4 tc = make_float4(0.f, 0.f, 0.f, 0.f);
            if (PK == 2) tc = s_tc[buf][t][mycen];
            float ucx = 0.f, ucy = 0.f;
            if (PK) {
                const float2 uc = s_uc[buf][t][mycen];
                ucx = uc.x;
                ucy = uc.y;
            }
            const float2 *gpr = nullptr, *gqr = nullptr;
            if (GK == 1) {
                const int2 a = s_ant[buf][t];
                gpr = P.gA + (size_t)a.x * P.n_pix_pad + kfirst + lane;
                gqr = P.gA + (size_t)a.y * P.n_pix_pad + kfirst + lane;
            }
#pragma unroll
            for (int i = 0; i < RP; ++i) {
                float X = fmaf(vv.x, dl[i], fmaf(vv.y, dm[i], fmaf(vv.z, dn[i], x0)));
                float g1 = 1.f;
                if (GK == 2) X += Ng[i];
                if (GK == 1) {
                    const float2 gp = __ldg(gpr + i * 32);
                    const float2 gq = __ldg(gqr + i * 32);
                    g1 = gp.x * gq.x;
                    X -= gp.y - gq.y;
                }
                float du = 0.f, dv = 0.f;
                if (PK) {
                    du = fmaf(-vv.w, dl[i], ucx);
                    dv = fmaf(-vv.w, dm[i], ucy);
                }
                float ere, eim;
                uint32_t sgn;
                if (PK == 0) {   // delta pixel: |r| cos(X + arg r), rr.x = |r| (arg r is inside x0)
                    float cv;
                    if (i < PolySplit<RP, PK, GK, SL1M_ADJ_NPOLY8>::N) {
                        float sv;
                        sincos_poly(X, sv, cv, sgn);         // the unused sine polynomial is dead code
                        cv = fxor(cv, sgn);
                    } else {
                        cv = __cosf(X);
                    }
                    if (GK == 2) Zr[i] = fmaf(cv, rr.x, Zr[i]);
                    else acc[i] = fmaf(GK == 1 ? g1 * rr.x : rr.x, cv, acc[i]);
                    continue;
                }
                if (PK == 2) {   // one sigma per tile: Re conj(M / a) r = amp (cr r_re + ci r_im)
                    float amp;
                    gen_entry_tile(X, du, dv, tc.x, tc.y, tc.z, amp, ere, eim);
                    acc[i] = fmaf(amp, fmaf(eim, rr.y, ere * rr.x), acc[i]);
                    continue;
                }
                if (i < PolySplit<RP, PK, GK, SL1M_ADJ_NPOLY8>::N) {
                    gen_entry<PK, true>(X, du, dv, vv.w, PK ? sig2[i] : 0.f, PK ? nsp[i] : 0.f, ere, eim, sgn);
                    ere = fxor(ere, sgn);
                    eim = fxor(eim, sgn);
                } else {
                    gen_entry<PK, false>(X, du, dv, vv.w, PK ? sig2[i] : 0.f, PK ? nsp[i] : 0.f, ere, eim, sgn);
                }
                // Re(conj(e) r) = ere r_re + eim r_im, e evaluated at the gain-shifted phase
                if (GK == 2) {
                    Zr[i] = fmaf(ere, rr.x, fmaf(eim, rr.y, Zr[i]));
                } else if (GK == 1) {
                    acc[i] = fmaf(g1, fmaf(eim, rr.y, ere * rr.x), acc[i]);
                } else {
                    acc[i] = fmaf(ere, rr.x, fmaf(eim, rr.y, acc[i]));
                }
            }
          }
            if (GK == 2) {
#pragma unroll
                for (int i = 0; i < RP; ++i) acc[i] = fmaf(Ga[i], Zr[i], acc[i]);
            }
        }
        __syncthreads();
    }

    float *out = P.ws_p + chan_index<BATCH>() * P.ws_p_stride + (size_t)cta_split * P.n_pix_pad;
#pragma unroll
    for (int i = 0; i < RP; ++i) out[kfirst + i * 32 + lane] = acc[i];
}

#ifndef SL1M_ADJ_C1_NPQ
#define SL1M_ADJ_C1_NPQ 1
#endif
#ifndef SL1M_ADJ_C1_MIN_CTAS
#define SL1M_ADJ_C1_MIN_CTAS 8
#endif
__device__ __forceinline__ void cos_poly2(f32x2 X, f32x2 &c, uint32_t &k_lo, uint32_t &k_hi) {
    const f32x2 kf = fma2(X, bc2(0.318309886183790672f), bc2(12582912.0f));
    const f32x2 kr = add2(kf, bc2(-12582912.0f));
    const f32x2 r = fma2(kr, bc2(-3.14159265358979324f), X);
    const f32x2 z = mul2(r, r);
    f32x2 pc = fma2(z, bc2(2.3423957827617414e-05f), bc2(-0.0013866969384253025f));
    pc = fma2(z, pc, bc2(0.04166554659605026f));
    pc = fma2(z, pc, bc2(-0.49999991059303284f));
    c = fma2(z, pc, bc2(1.0f));
    float a, b;
    up2(kf, a, b);
    k_lo = __float_as_uint(a);
    k_hi = __float_as_uint(b);
}
template <int NPQ, bool BATCH = false>
__global__ void __launch_bounds__(NT, SL1M_ADJ_C1_MIN_CTAS) adj_kernel_c1(const ApplyParams P) {
    if (BATCH && P.done && P.done[blockIdx.z]) return;   // batched solve: this channel has met its stopping rule
    constexpr int RP = 8, NPAIR = 4, NCEN = NT * RP / TP;
    __shared__ __align__(16) float4 s_vc[2][NCEN][VC];   // (u', v', w', x0 for that centre + arg r)
    __shared__ float s_R[2][VC];                          // |r|

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int base = blockIdx.x * (NT * RP);
    const int kfirst = base + warp * (32 * RP);
    const int tile0 = base / TP;
    const int mycen = (kfirst / TP) - tile0;

    f32x2 DL[NPAIR], DM[NPAIR], DN[NPAIR], ACC[NPAIR];
#pragma unroll
    for (int i = 0; i < NPAIR; ++i) {
        const float4 pa = P.pix4[kfirst + (2 * i) * 32 + lane], pb = P.pix4[kfirst + (2 * i + 1) * 32 + lane];
        DL[i] = pk2(pa.x, pb.x);
        DM[i] = pk2(pa.y, pb.y);
        DN[i] = pk2(pa.z, pb.z);
        ACC[i] = pk2(0.f, 0.f);
    }

    const int n_chunks = (P.n_vis + VC - 1) / VC;
    const double sc = chan_scale_of<BATCH>(P);
    const int c0 = blockIdx.y * P.per_split;
    const int c1 = min(c0 + P.per_split, n_chunks);

    auto stage = [&](int chunk, int buf) {
        const int j = chunk * VC + tid;   // NT == VC
        double u = 0.0, v = 0.0, w = 0.0;
        float2 rp = make_float2(0.f, 0.f);   // (|r|, arg r)
        if (j < P.n_vis) {
            u = sc * P.u64[j];
            v = sc * P.v64[j];
            w = sc * P.w64[j];
            rp = P.r[chan_index<BATCH>() * P.n_vis + j];
        }
        const float uf = static_cast<float>(TWO_PI * u), vf = static_cast<float>(TWO_PI * v),
                    wf = static_cast<float>(TWO_PI * w);
        s_R[buf][tid] = rp.x;
#pragma unroll
        for (int c = 0; c < NCEN; ++c)   // both addends lie in [-pi, pi]
            s_vc[buf][c][tid] = make_float4(uf, vf, wf, centre_phase(u, v, w, P.cen[tile0 + c]) + rp.y);
    };

    auto visibility = [&](const float4 vv, const float R, auto npoly_tag) {
        constexpr int NPOLY = decltype(npoly_tag)::value;
        const f32x2 uu = bc2(vv.x), vvv = bc2(vv.y), ww = bc2(vv.z), x0 = bc2(vv.w);
#pragma unroll
        for (int i = 0; i < NPAIR; ++i) {
            const f32x2 X = fma2(DL[i], uu, fma2(DM[i], vvv, fma2(DN[i], ww, x0)));
            if (i < NPOLY) {
                f32x2 c;
                uint32_t ka, kb;
                cos_poly2(X, c, ka, kb);
                ACC[i] = fma2(c, pk2(flip_if_odd(R, ka), flip_if_odd(R, kb)), ACC[i]);
            } else {
                float xa, xb;
                up2(X, xa, xb);
                ACC[i] = fma2(pk2(__cosf(xa), __cosf(xb)), bc2(R), ACC[i]);
            }
        }
    };

    if (c0 < c1) stage(c0, 0);
    __syncthreads();
    for (int ch = c0; ch < c1; ++ch) {
        const int buf = (ch - c0) & 1;
        if (ch + 1 < c1) stage(ch + 1, buf ^ 1);
#pragma unroll 1
        for (int t = 0; t < VC; t += 4) {
            visibility(s_vc[buf][mycen][t], s_R[buf][t], std::integral_constant<int, (NPQ + 3) / 4>{});
            visibility(s_vc[buf][mycen][t + 1], s_R[buf][t + 1], std::integral_constant<int, (NPQ + 2) / 4>{});
            visibility(s_vc[buf][mycen][t + 2], s_R[buf][t + 2], std::integral_constant<int, (NPQ + 1) / 4>{});
            visibility(s_vc[buf][mycen][t + 3], s_R[buf][t + 3], std::integral_constant<int, NPQ / 4>{});
        }
        __syncthreads();
    }

    float *out = P.ws_p + chan_index<BATCH>() * P.ws_p_stride + (size_t)blockIdx.y * P.n_pix_pad;
#pragma unroll
    for (int i = 0; i < NPAIR; ++i) {
        float a, b;
        up2(ACC[i], a, b);
        out[kfirst + (2 * i) * 32 + lane] = a;
        out[kfirst + (2 * i + 1) * 32 + lane] = b;
    }
}

// ------------------------------------------------------------------------------------------
// adjoint, delta pixels, baseline-grouped gains (gk == 2), packed-pair variant (RP = 8).
// A chunk is 16 baseline groups x 8 samples, staged group-major.  Per group the thread forms
// G_i = g_p(i) conj(g_q(i)) for its 8 pixels once (next group's gain rows prefetched), accumulates
// Z_i = sum_samples conj(e) r over the 8 samples, then acc_i += Re(conj(G_i) Z_i).
// ------------------------------------------------------------------------------------------
#ifndef SL1M_ADJ_G2X2_MIN_CTAS
#define SL1M_ADJ_G2X2_MIN_CTAS 5
#endif
template <int NPQ, bool BATCH = false>
__global__ void __launch_bounds__(NT, SL1M_ADJ_G2X2_MIN_CTAS) adj_kernel_g2x2(const ApplyParams P) {
    if (BATCH && P.done && P.done[blockIdx.z]) return;   // batched solve: this channel has met its stopping rule
    constexpr int RP = 8, NPAIR = 4, NCEN = NT * RP / TP, NG = VC / 8;
    // Gains are stored in polar form (|g|, arg g).  With G = |G| e^{i gamma} (|G| = |g_p||g_q|, gamma = arg_p - arg_q):
    //     Re conj(M_jk) r_j = a |G| Re( e^{i (X_rel - gamma)} r_j e^{i x0(j, centre)} ) = a |G| |r_j| cos(X_rel - gamma + phi'),
    // phi' = arg r_j + x0(j, centre), formed ONCE per (visibility, centre) while the chunk is staged.  -gamma is the
    // innermost addend of the phase FMA chain, phi' one more add; ONE cosine per term, real accumulation.
    __shared__ __align__(16) float4 s_vc[2][VC];          // (u', v', w', -), slot = group * 8 + sample
    __shared__ __align__(8) float2 s_r[2][NCEN][VC];      // (|r|, arg r + x0 of that centre)
    __shared__ __align__(8) int2 s_ant[2][NG];           // the group's (p, q)

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    int cta_group, cta_split;
    adj_cta<true>(cta_group, cta_split);
    const int base = cta_group * (NT * RP);
    const int kfirst = base + warp * (32 * RP);
    const int tile0 = base / TP;
    const int mycen = (kfirst / TP) - tile0;

    f32x2 DL[NPAIR], DM[NPAIR], DN[NPAIR], ACC[NPAIR];
#pragma unroll
    for (int i = 0; i < NPAIR; ++i) {
        const float4 pa = P.pix4[kfirst + (2 * i) * 32 + lane], pb = P.pix4[kfirst + (2 * i + 1) * 32 + lane];
        DL[i] = pk2(pa.x, pb.x);
        DM[i] = pk2(pa.y, pb.y);
        DN[i] = pk2(pa.z, pb.z);
        ACC[i] = pk2(0.f, 0.f);
    }

    const int n_chunks = (P.n_vis + VC - 1) / VC;
    const double sc = chan_scale_of<BATCH>(P);
    const int c0 = cta_split * P.per_split;
    const int c1 = min(c0 + P.per_split, n_chunks);

    // the plan stores sample r of group g at (g / 128) * 1024 + r * 128 + g % 128 (the forward's thread layout)
    auto stage = [&](int chunk, int buf) {
        const int g = chunk * NG + (tid & 15), r = tid >> 4;
        const int j = (g >> 7) * (NT * 8) + r * NT + (g & 127);
        const int slot = (tid & 15) * 8 + r;
        double u = 0.0, v = 0.0, w = 0.0;
        float2 rr = make_float2(0.f, 0.f);
        int2 a = make_int2(0, 0);
        if (j < P.n_vis) {
            u = sc * P.u64[j];
            v = sc * P.v64[j];
            w = sc * P.w64[j];
            rr = P.r[chan_index<BATCH>() * P.n_vis + j];
            a = make_int2(P.ant_p[j], P.ant_q[j]);
        }
        const float uf = static_cast<float>(TWO_PI * u), vf = static_cast<float>(TWO_PI * v),
                    wf = static_cast<float>(TWO_PI * w);
        s_vc[buf][slot] = make_float4(uf, vf, wf, 0.f);
        if (tid < NG) s_ant[buf][tid] = a;   // sample 0 carries the group's (p, q)
        const float R = sqrtf(fmaf(rr.x, rr.x, rr.y * rr.y)), phi = atan2f(rr.y, rr.x);
#pragma unroll
        for (int c = 0; c < NCEN; ++c)
            s_r[buf][c][slot] = make_float2(R, phi + centre_phase(u, v, w, P.cen[tile0 + c]));   // both in [-pi, pi]
    };

    auto load_gains = [&](int2 a, float2 (&gp)[RP], float2 (&gq)[RP]) {
#pragma unroll
        for (int i = 0; i < RP; ++i) {
            gp[i] = __ldg(P.gA + (size_t)a.x * P.n_pix_pad + kfirst + lane + i * 32);
            gq[i] = __ldg(P.gA + (size_t)a.y * P.n_pix_pad + kfirst + lane + i * 32);
        }
    };

    f32x2 Z[NPAIR], NGM[NPAIR];
    // rr = (|r|, phi')
    auto visibility = [&](const float4 vv, const float2 rr, auto npoly_tag) {
        constexpr int NPOLY = decltype(npoly_tag)::value;
        const f32x2 uu = bc2(vv.x), vvv = bc2(vv.y), ww = bc2(vv.z), ph = bc2(rr.y);
#pragma unroll
        for (int i = 0; i < NPAIR; ++i) {
            const f32x2 X = add2(fma2(DL[i], uu, fma2(DM[i], vvv, fma2(DN[i], ww, NGM[i]))), ph);
            if (i < NPOLY) {
                f32x2 c;
                uint32_t ka, kb;
                cos_poly2(X, c, ka, kb);
                Z[i] = fma2(c, pk2(flip_if_odd(rr.x, ka), flip_if_odd(rr.x, kb)), Z[i]);
            } else {
                float xa, xb;
                up2(X, xa, xb);
                Z[i] = fma2(pk2(__cosf(xa), __cosf(xb)), bc2(rr.x), Z[i]);
            }
        }
    };

    if (c0 < c1) stage(c0, 0);
    __syncthreads();
    for (int ch = c0; ch < c1; ++ch) {
        const int buf = (ch - c0) & 1;
        if (ch + 1 < c1) stage(ch + 1, buf ^ 1);
        float2 gp[RP], gq[RP];
        load_gains(s_ant[buf][0], gp, gq);
#pragma unroll 1
        for (int g = 0; g < NG; ++g) {
            f32x2 GA[NPAIR];
#pragma unroll
            for (int i = 0; i < NPAIR; ++i) {
                const float2 pa = gp[2 * i], qa = gq[2 * i], pb = gp[2 * i + 1], qb = gq[2 * i + 1];
                GA[i] = pk2(pa.x * qa.x, pb.x * qb.x);        // |g_p||g_q|
                NGM[i] = pk2(qa.y - pa.y, qb.y - pb.y);       // -gamma
                Z[i] = pk2(0.f, 0.f);
            }
            load_gains(s_ant[buf][min(g + 1, NG - 1)], gp, gq);   // next group's rows
            const int t = g * 8;
            visibility(s_vc[buf][t], s_r[buf][mycen][t], std::integral_constant<int, (NPQ + 3) / 4>{});
            visibility(s_vc[buf][t + 1], s_r[buf][mycen][t + 1], std::integral_constant<int, (NPQ + 2) / 4>{});
            visibility(s_vc[buf][t + 2], s_r[buf][mycen][t + 2], std::integral_constant<int, (NPQ + 1) / 4>{});
            visibility(s_vc[buf][t + 3], s_r[buf][mycen][t + 3], std::integral_constant<int, NPQ / 4>{});
            visibility(s_vc[buf][t + 4], s_r[buf][mycen][t + 4], std::integral_constant<int, (NPQ + 3) / 4>{});
            visibility(s_vc[buf][t + 5], s_r[buf][mycen][t + 5], std::integral_constant<int, (NPQ + 2) / 4>{});
            visibility(s_vc[buf][t + 6], s_r[buf][mycen][t + 6], std::integral_constant<int, (NPQ + 1) / 4>{});
            visibility(s_vc[buf][t + 7], s_r[buf][mycen][t + 7], std::integral_constant<int, NPQ / 4>{});
#pragma unroll
            for (int i = 0; i < NPAIR; ++i) ACC[i] = fma2(GA[i], Z[i], ACC[i]);
        }
        __syncthreads();
    }

    float *out = P.ws_p + chan_index<BATCH>() * P.ws_p_stride + (size_t)cta_split * P.n_pix_pad;
#pragma unroll
    for (int i = 0; i < NPAIR; ++i) {
        float a, b;
        up2(ACC[i], a, b);
        out[kfirst + (2 * i) * 32 + lane] = a;
        out[kfirst + (2 * i + 1) * 32 + lane] = b;
    }
}

// ------------------------------------------------------------------------------------------
// Gaussian pixels with one sigma per tile (PK == 2), unit gains, packed-pair variants (R = 8).
// Same arithmetic as gen_entry_tile, two terms per FFMA2: 14 (forward) / 12 (adjoint) packed ops +
// 2 FMUL.RZ + 6 MUFU per pair.  Next to a scalar FFMA stream every MUFU costs ~2 extra FMA-side
// cycles, next to FFMA2 well under 1 (profiles/r1_microbench.md): packing is what lets the 3-MUFU
// loop run near the MUFU bound.
// ------------------------------------------------------------------------------------------
#ifndef SL1M_FWD_GTX2_MIN_CTAS
#define SL1M_FWD_GTX2_MIN_CTAS 4
#endif
#ifndef SL1M_ADJ_GTX2_MIN_CTAS
#define SL1M_ADJ_GTX2_MIN_CTAS 5
#endif
//   *_GTX2_NP4  of a thread's 4 register pairs, how many take the FMA-pipe polynomial for sin/cos (forward) or
//               cos (adjoint); ex2 stays on the MUFU pipe
#ifndef SL1M_FWD_GTX2_NP4
#define SL1M_FWD_GTX2_NP4 0
#endif
#ifndef SL1M_ADJ_GTX2_NP4
#define SL1M_ADJ_GTX2_NP4 1
#endif
__device__ __forceinline__ void sincos2(f32x2 X, f32x2 &s, f32x2 &c) {
    float xa, xb, sa, ca, sb, cb;
    up2(X, xa, xb);
    __sincosf(xa, &sa, &ca);
    __sincosf(xb, &sb, &cb);
    s = pk2(sa, sb);
    c = pk2(ca, cb);
}
__device__ __forceinline__ f32x2 ex2_2(f32x2 E) {
    float a, b;
    up2(E, a, b);
    return pk2(ex2_approx(a), ex2_approx(b));
}

template <bool BATCH = false>
__global__ void __launch_bounds__(NT, SL1M_FWD_GTX2_MIN_CTAS) fwd_kernel_gtx2(const ApplyParams P) {
    if (BATCH && P.done && P.done[blockIdx.z]) return;   // batched solve: this channel has met its stopping rule
    constexpr int RV = 8, NPAIR = 4;
    __shared__ __align__(128) float4 s_pix[2][TP];
    __shared__ __align__(8) uint64_t s_bar[2];
    // (1 + i q) is the same for every pixel of a tile (q = w sigma_tile^2), so the pixel loop only sums
    // T = sum a x 2^E' (cos X' - i sin X') in registers; at the end of the tile the running totals, kept in
    // shared memory ([pair][thread], own slots only), take (1 + i q) T.  Saves 2 FFMA2 per pair and 24 registers.
    __shared__ __align__(8) f32x2 s_acc[2 * NPAIR_X2][NT];
    const int tid = threadIdx.x;
    const int t0 = blockIdx.y * P.per_split;
    const int t1 = min(t0 + P.per_split, P.n_tiles);
    const int jbase = blockIdx.x * (NT * RV);
    const int jlast = P.n_vis - 1;
    const double sc = chan_scale_of<BATCH>(P);
    const float4 *pix4 = P.pix4 + chan_index<BATCH>() * P.n_pix_pad;

    f32x2 U[NPAIR], V[NPAIR], W[NPAIR], NWL[NPAIR];
#pragma unroll
    for (int i = 0; i < NPAIR; ++i) {
        const int ja = min(jbase + (2 * i) * NT + tid, jlast), jb = min(jbase + (2 * i + 1) * NT + tid, jlast);
        const double wa = sc * __ldg(P.w64 + ja), wb = sc * __ldg(P.w64 + jb);
        U[i] = pk2(static_cast<float>(TWO_PI * (sc * __ldg(P.u64 + ja))), static_cast<float>(TWO_PI * (sc * __ldg(P.u64 + jb))));
        V[i] = pk2(static_cast<float>(TWO_PI * (sc * __ldg(P.v64 + ja))), static_cast<float>(TWO_PI * (sc * __ldg(P.v64 + jb))));
        W[i] = pk2(static_cast<float>(TWO_PI * wa), static_cast<float>(TWO_PI * wb));
        NWL[i] = pk2(static_cast<float>(-wa), static_cast<float>(-wb));
        s_acc[i][tid] = pk2(0.f, 0.f);
        s_acc[NPAIR + i][tid] = pk2(0.f, 0.f);
    }
    if (tid == 0) {
        mbar_init(&s_bar[0], 1);
        mbar_init(&s_bar[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    auto issue = [&](int t, int st) {   // only the pixels the tile has to stream (zero-skipping; >= 64 B)
        const uint32_t bytes = (uint32_t)max(tile_pixels<BATCH>(P, t), 4) * (uint32_t)sizeof(float4);
        mbar_expect_tx(&s_bar[st], bytes);
        tma_bulk_g2s(&s_pix[st][0], pix4 + (size_t)t * TP, bytes, &s_bar[st]);
    };
    if (tid == 0) {
        if (t0 < t1) issue(t0, 0);
        if (t0 + 1 < t1) issue(t0 + 1, 1);
    }
    for (int t = t0; t < t1; ++t) {
        const int st = (t - t0) & 1;
        const uint32_t parity = ((t - t0) >> 1) & 1;
        const double4 c = P.cen[t];
        const int npx = tile_pixels<BATCH>(P, t);
        if (npx == 0) {                          // empty tile (uniform over the CTA): consume the stage and move on
            mbar_wait(&s_bar[st], parity);
            __syncthreads();
            if (tid == 0 && t + 2 < t1) issue(t + 2, st);
            continue;
        }
        f32x2 X0[NPAIR], UC[NPAIR], VC2[NPAIR], CE[NPAIR], LR[NPAIR], CX[NPAIR], TC[NPAIR], TS[NPAIR];
#pragma unroll
        for (int i = 0; i < NPAIR; ++i) {
            float x0[2], uc[2], vc[2], q[2], cE[2], lr[2];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int j = min(jbase + (2 * i + h) * NT + tid, jlast);
                const double ud = sc * __ldg(P.u64 + j), vd = sc * __ldg(P.v64 + j), wd = sc * __ldg(P.w64 + j);
                x0[h] = centre_phase(ud, vd, wd, c);
                uc[h] = static_cast<float>(ud - wd * c.x);
                vc[h] = static_cast<float>(vd - wd * c.y);
                gauss_tile_constants(wd, c.w, q[h], cE[h], lr[h], x0[h]);
            }
            X0[i] = pk2(x0[0], x0[1]);
            UC[i] = pk2(uc[0], uc[1]);
            VC2[i] = pk2(vc[0], vc[1]);
            TC[i] = pk2(0.f, 0.f);
            TS[i] = pk2(0.f, 0.f);
            CE[i] = pk2(cE[0], cE[1]);
            LR[i] = pk2(lr[0], lr[1]);
            CX[i] = pk2(-0.69314718056f * q[0], -0.69314718056f * q[1]);
        }
        mbar_wait(&s_bar[st], parity);
#pragma unroll 1
        for (int p = 0; p < npx; ++p) {
            const float4 px = s_pix[st][p];
            const f32x2 bx = bc2(px.x), by = bc2(px.y), bz = bc2(px.z), bw = bc2(px.w);
#pragma unroll
            for (int i = 0; i < NPAIR; ++i) {
                const f32x2 X = fma2(U[i], bx, fma2(V[i], by, fma2(W[i], bz, X0[i])));
                const f32x2 du = fma2(NWL[i], bx, UC[i]), dv = fma2(NWL[i], by, VC2[i]);
                const f32x2 s2 = fma2(dv, dv, mul2(du, du));
                const f32x2 Ep = fma2(s2, CE[i], LR[i]);
                const f32x2 Xp = fma2(CX[i], Ep, X);
                f32x2 tw = mul2(bw, ex2_2(Ep));                  // a x 2^E'
                f32x2 s, cc;
                if (i < SL1M_FWD_GTX2_NP4) {                     // pipe balance: this pair's sin/cos on the FMA pipe
                    uint32_t ka, kb;
                    sincos_poly2(Xp, s, cc, ka, kb);
                    float ta, tb;
                    up2(tw, ta, tb);
                    tw = pk2(flip_if_odd(ta, ka), flip_if_odd(tb, kb));
                } else {
                    sincos2(Xp, s, cc);
                }
                TC[i] = fma2(tw, cc, TC[i]);
                TS[i] = fma2(tw, s, TS[i]);
            }
        }
#pragma unroll
        for (int i = 0; i < NPAIR; ++i) {   // totals += (1 + i q)(TC - i TS):  re += TC + q TS,  -im += TS - q TC
            const int ja = min(jbase + (2 * i) * NT + tid, jlast), jb = min(jbase + (2 * i + 1) * NT + tid, jlast);
            const f32x2 Q = pk2(static_cast<float>(sc * __ldg(P.w64 + ja) * c.w), static_cast<float>(sc * __ldg(P.w64 + jb) * c.w));
            float qa, qb;
            up2(Q, qa, qb);
            s_acc[i][tid] = add2(s_acc[i][tid], fma2(Q, TS[i], TC[i]));
            s_acc[NPAIR + i][tid] = add2(s_acc[NPAIR + i][tid], fma2(pk2(-qa, -qb), TC[i], TS[i]));
        }
        __syncthreads();
        if (tid == 0 && t + 2 < t1) issue(t + 2, st);
    }
    float2 *out = P.ws_v + chan_index<BATCH>() * P.ws_v_stride + (size_t)blockIdx.y * P.n_vis;
#pragma unroll
    for (int i = 0; i < NPAIR; ++i) {
        float ra, rb, ia, ib;
        up2(s_acc[i][tid], ra, rb);
        up2(s_acc[NPAIR + i][tid], ia, ib);
        const int ja = jbase + (2 * i) * NT + tid, jb = jbase + (2 * i + 1) * NT + tid;
        if (ja < P.n_vis) out[ja] = make_float2(ra, -ia);
        if (jb < P.n_vis) out[jb] = make_float2(rb, -ib);
    }
}

template <bool BATCH = false>
__global__ void __launch_bounds__(NT, SL1M_ADJ_GTX2_MIN_CTAS) adj_kernel_gtx2(const ApplyParams P) {
    if (BATCH && P.done && P.done[blockIdx.z]) return;   // batched solve: this channel has met its stopping rule
    constexpr int RP = 8, NPAIR = 4, NCEN = NT * RP / TP;
    __shared__ __align__(16) float4 s_vis[2][VC];            // (u', v', w', -w)
    __shared__ __align__(16) float4 s_ca[2][NCEN][VC];       // per centre: (x0', uc, vc, cX = -ln2 q)
    __shared__ __align__(16) float4 s_cb[2][NCEN][VC];       // per centre: (cE, lr, R = |(A, B)|, -) with A = r_re + q r_im, B = q r_re - r_im
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int base = blockIdx.x * (NT * RP);
    const int kfirst = base + warp * (32 * RP);
    const int tile0 = base / TP;
    const int mycen = (kfirst / TP) - tile0;
    f32x2 DL[NPAIR], DM[NPAIR], DN[NPAIR], ACC[NPAIR];
#pragma unroll
    for (int i = 0; i < NPAIR; ++i) {
        const float4 pa = P.pix4[kfirst + (2 * i) * 32 + lane], pb = P.pix4[kfirst + (2 * i + 1) * 32 + lane];
        DL[i] = pk2(pa.x, pb.x);
        DM[i] = pk2(pa.y, pb.y);
        DN[i] = pk2(pa.z, pb.z);
        ACC[i] = pk2(0.f, 0.f);
    }
    const int n_chunks = (P.n_vis + VC - 1) / VC;
    const double sc = chan_scale_of<BATCH>(P);
    const int c0 = blockIdx.y * P.per_split;
    const int c1 = min(c0 + P.per_split, n_chunks);
    auto stage = [&](int chunk, int buf) {
        const int j = chunk * VC + tid;
        double u = 0.0, v = 0.0, w = 0.0;
        float2 rr = make_float2(0.f, 0.f);
        if (j < P.n_vis) {
            u = sc * P.u64[j];
            v = sc * P.v64[j];
            w = sc * P.w64[j];
            rr = P.r[chan_index<BATCH>() * P.n_vis + j];
        }
        s_vis[buf][tid] = make_float4(static_cast<float>(TWO_PI * u), static_cast<float>(TWO_PI * v),
                                      static_cast<float>(TWO_PI * w), static_cast<float>(-w));
#pragma unroll
        for (int c = 0; c < NCEN; ++c) {
            const double4 cen = P.cen[tile0 + c];
            float x0 = centre_phase(u, v, w, cen), q, cE, lr;
            gauss_tile_constants(w, cen.w, q, cE, lr, x0);
            // Re conj(M/a) r = amp ((c + q s) r_re + (q c - s) r_im) = amp (c A + s B) = amp R cos(X' - psi),
            // (R, psi) the polar form of (A, B): ONE cosine per term, psi folded into the centre phase
            const float A = fmaf(q, rr.y, rr.x), B = fmaf(q, rr.x, -rr.y);
            s_ca[buf][c][tid] = make_float4(x0 - atan2f(B, A), static_cast<float>(u - w * cen.x),
                                            static_cast<float>(v - w * cen.y), -0.69314718056f * q);
            s_cb[buf][c][tid] = make_float4(cE, lr, sqrtf(fmaf(A, A, B * B)), 0.f);
        }
    };
    if (c0 < c1) stage(c0, 0);
    __syncthreads();
    for (int ch = c0; ch < c1; ++ch) {
        const int buf = (ch - c0) & 1;
        if (ch + 1 < c1) stage(ch + 1, buf ^ 1);
#pragma unroll 2
        for (int t = 0; t < VC; ++t) {
            const float4 vv = s_vis[buf][t], ca = s_ca[buf][mycen][t], cb = s_cb[buf][mycen][t];
            const f32x2 bu = bc2(vv.x), bv = bc2(vv.y), bw = bc2(vv.z), bnw = bc2(vv.w);
            const f32x2 bx0 = bc2(ca.x), buc = bc2(ca.y), bvc = bc2(ca.z), bcx = bc2(ca.w);
            const f32x2 bce = bc2(cb.x), blr = bc2(cb.y), bR = bc2(cb.z);
#pragma unroll
            for (int i = 0; i < NPAIR; ++i) {
                const f32x2 X = fma2(DL[i], bu, fma2(DM[i], bv, fma2(DN[i], bw, bx0)));
                const f32x2 du = fma2(DL[i], bnw, buc), dv = fma2(DM[i], bnw, bvc);
                const f32x2 s2 = fma2(dv, dv, mul2(du, du));
                const f32x2 Ep = fma2(s2, bce, blr);
                const f32x2 Xp = fma2(bcx, Ep, X);
                if (i < SL1M_ADJ_GTX2_NP4) {                     // pipe balance: this pair's cosine on the FMA pipe
                    f32x2 c;
                    uint32_t ka, kb;
                    cos_poly2(Xp, c, ka, kb);
                    float ea, eb;
                    up2(ex2_2(Ep), ea, eb);
                    ACC[i] = fma2(mul2(pk2(flip_if_odd(ea, ka), flip_if_odd(eb, kb)), c), bR, ACC[i]);
                } else {
                    float xa, xb;
                    up2(Xp, xa, xb);
                    ACC[i] = fma2(mul2(ex2_2(Ep), pk2(__cosf(xa), __cosf(xb))), bR, ACC[i]);
                }
            }
        }
        __syncthreads();
    }
    float *out = P.ws_p + chan_index<BATCH>() * P.ws_p_stride + (size_t)blockIdx.y * P.n_pix_pad;
#pragma unroll
    for (int i = 0; i < NPAIR; ++i) {
        float a, b;
        up2(ACC[i], a, b);
        out[kfirst + (2 * i) * 32 + lane] = a;
        out[kfirst + (2 * i + 1) * 32 + lane] = b;
    }
}

// ------------------------------------------------------------------------------------------
// fp64-phase variants (NEXT-2 of the scope table: "higher-precision phase path selectable per
// plan"), delta pixels, unit gains.  The fp32 remainder u' dl + v' dm + w' dn' of the default
// kernels is accurate while it stays within a few hundred radians, i.e. while a 16 x 16-pixel tile
// spans at most a few tens of fringes of the longest baseline -- always true for a sensibly sampled
// image, not for a badly undersampled one.  Here the whole phase is accumulated in fp64 TURNS
// (3 DFMA on the otherwise idle FP64 pipe), its fraction is taken exactly with the magic-number add
// (1.5 * 2^20: the low word of the sum is frac * 2^32), and 23 bits of it are handed to
// sin.approx / cos.approx: phase error <= 4e-7 rad for any baseline length.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ float phase64_to_radians(double turns) {
    const double m = turns + 1572864.0;                        // 1.5 * 2^20: ulp = 2^-32
    const int frac32 = __double2loint(m);                      // round(turns * 2^32) mod 2^32, signed
    const int s23 = frac32 >> 9;                               // [-2^22, 2^22)
    const float f = __int_as_float(0x4B400000 + s23) - 12582912.0f;   // exactly s23
    return f * 7.490140565847157e-07f;                         // 2 pi / 2^23
}

template <int RV>
__global__ void __launch_bounds__(NT, 3) fwd_kernel_p64(const ApplyParams P, const double4 *pixd) {
    if (P.done && P.done[blockIdx.z]) return;   // this channel's solve has met its stopping rule
    __shared__ __align__(128) float4 s_pix[2][TP];
    __shared__ __align__(128) double4 s_pixd[2][TP];   // (dl, dm, dn', 0) as doubles
    __shared__ __align__(8) uint64_t s_bar[2];
    const int tid = threadIdx.x;
    const int t0 = blockIdx.y * P.per_split;
    const int t1 = min(t0 + P.per_split, P.n_tiles);
    const int jbase = blockIdx.x * (NT * RV);
    const int jlast = P.n_vis - 1;
    double ud[RV], vd[RV], wd[RV];
    float re[RV], im[RV];
    // batched channels (blockIdx.z): uvw * nu_c/nu_0 in fp64, the channel's own a*x tiles and partials
    const double sc = P.chan_scale ? P.chan_scale[blockIdx.z] : 1.0;
    const float4 *pix4 = P.pix4 + (size_t)blockIdx.z * P.n_pix_pad;
#pragma unroll
    for (int r = 0; r < RV; ++r) {
        const int j = min(jbase + r * NT + tid, jlast);
        ud[r] = sc * __ldg(P.u64 + j);
        vd[r] = sc * __ldg(P.v64 + j);
        wd[r] = sc * __ldg(P.w64 + j);
        re[r] = 0.f;
        im[r] = 0.f;
    }
    if (tid == 0) {
        mbar_init(&s_bar[0], 1);
        mbar_init(&s_bar[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    // zero-skipping: pix4 / pixd are then the per-channel COMPACT copies and tile_cnt the entries to stream
    const int *tcnt = P.tile_cnt ? P.tile_cnt + (size_t)blockIdx.z * P.n_tiles : nullptr;
    if (tcnt) pixd += (size_t)blockIdx.z * P.n_pix_pad;
    auto issue = [&](int t, int st) {
        const uint32_t n4 = (uint32_t)(tcnt ? max(__ldg(tcnt + t), 4) : TP);
        mbar_expect_tx(&s_bar[st], n4 * (uint32_t)(sizeof(float4) + sizeof(double4)));
        tma_bulk_g2s(&s_pix[st][0], pix4 + (size_t)t * TP, n4 * (uint32_t)sizeof(float4), &s_bar[st]);
        tma_bulk_g2s(&s_pixd[st][0], pixd + (size_t)t * TP, n4 * (uint32_t)sizeof(double4), &s_bar[st]);
    };
    if (tid == 0) {
        if (t0 < t1) issue(t0, 0);
        if (t0 + 1 < t1) issue(t0 + 1, 1);
    }
    for (int t = t0; t < t1; ++t) {
        const int st = (t - t0) & 1;
        const uint32_t parity = ((t - t0) >> 1) & 1;
        const double4 c = P.cen[t];
        double x0[RV];
#pragma unroll
        for (int r = 0; r < RV; ++r) {
            double tt = fma(ud[r], c.x, fma(vd[r], c.y, wd[r] * c.z));
            x0[r] = tt - rint(tt);
        }
        mbar_wait(&s_bar[st], parity);
        const int npx = tcnt ? __ldg(tcnt + t) : TP;
#pragma unroll 2
        for (int p = 0; p < npx; ++p) {
            const double4 pd = s_pixd[st][p];
            const float wt = s_pix[st][p].w;
#pragma unroll
            for (int r = 0; r < RV; ++r) {
                const float X = phase64_to_radians(fma(ud[r], pd.x, fma(vd[r], pd.y, fma(wd[r], pd.z, x0[r]))));
                float s, c2;
                __sincosf(X, &s, &c2);
                re[r] = fmaf(wt, c2, re[r]);
                im[r] = fmaf(-wt, s, im[r]);
            }
        }
        __syncthreads();
        if (tid == 0 && t + 2 < t1) issue(t + 2, st);
    }
    float2 *out = P.ws_v + (size_t)blockIdx.z * P.ws_v_stride + (size_t)blockIdx.y * P.n_vis;
#pragma unroll
    for (int r = 0; r < RV; ++r) {
        const int j = jbase + r * NT + tid;
        if (j < P.n_vis) out[j] = make_float2(re[r], im[r]);
    }
}

template <int RP>
__global__ void __launch_bounds__(NT, 3) adj_kernel_p64(const ApplyParams P, const double4 *pixd) {
    if (P.done && P.done[blockIdx.z]) return;   // this channel's solve has met its stopping rule
    constexpr int NCEN = (NT * RP > TP) ? (NT * RP / TP) : 1;
    __shared__ __align__(32) double4 s_vis[2][VC];       // (u, v, w, 0) in wavelengths
    __shared__ __align__(8) float2 s_r[2][VC];           // residual in polar form (|r|, arg r): one cosine per term
    __shared__ double s_x0[2][VC][NCEN];                 // frac(u l_c + v m_c + w n'_c) + arg r / 2 pi, turns
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int base = blockIdx.x * (NT * RP);
    const int kfirst = base + warp * (32 * RP);
    const int tile0 = base / TP;
    const int mycen = (kfirst / TP) - tile0;
    double dl[RP], dm[RP], dn[RP];
    float acc[RP];
#pragma unroll
    for (int i = 0; i < RP; ++i) {
        const double4 pd = pixd[kfirst + i * 32 + lane];
        dl[i] = pd.x;
        dm[i] = pd.y;
        dn[i] = pd.z;
        acc[i] = 0.f;
    }
    const int n_chunks = (P.n_vis + VC - 1) / VC;
    const int c0 = blockIdx.y * P.per_split;
    const int c1 = min(c0 + P.per_split, n_chunks);
    const double sc = P.chan_scale ? P.chan_scale[blockIdx.z] : 1.0;   // batched channels: uvw * nu_c/nu_0
    const float2 *rin = P.r + (size_t)blockIdx.z * P.n_vis;
    auto stage = [&](int chunk, int buf) {
        const int j = chunk * VC + tid;
        double u = 0.0, v = 0.0, w = 0.0;
        float2 rr = make_float2(0.f, 0.f);
        if (j < P.n_vis) {
            u = sc * P.u64[j];
            v = sc * P.v64[j];
            w = sc * P.w64[j];
            rr = rin[j];
        }
        s_vis[buf][tid] = make_double4(u, v, w, 0.0);
        s_r[buf][tid] = rr;
#pragma unroll
        for (int c = 0; c < NCEN; ++c) {
            const double4 cen = P.cen[tile0 + c];
            const double tt = fma(u, cen.x, fma(v, cen.y, w * cen.z));
            s_x0[buf][tid][c] = (tt - rint(tt)) + (double)rr.y * (1.0 / TWO_PI);
        }
    };
    if (c0 < c1) stage(c0, 0);
    __syncthreads();
    for (int ch = c0; ch < c1; ++ch) {
        const int buf = (ch - c0) & 1;
        if (ch + 1 < c1) stage(ch + 1, buf ^ 1);
#pragma unroll 2
        for (int t = 0; t < VC; ++t) {
            const double4 vv = s_vis[buf][t];
            const float2 rr = s_r[buf][t];
            const double x0 = s_x0[buf][t][mycen];
#pragma unroll
            for (int i = 0; i < RP; ++i) {
                const float X = phase64_to_radians(fma(vv.x, dl[i], fma(vv.y, dm[i], fma(vv.z, dn[i], x0))));
                acc[i] = fmaf(rr.x, __cosf(X), acc[i]);           // Re e^{iX} r = |r| cos(X + arg r)
            }
        }
        __syncthreads();
    }
    float *out = P.ws_p + (size_t)blockIdx.z * P.ws_p_stride + (size_t)blockIdx.y * P.n_pix_pad;
#pragma unroll
    for (int i = 0; i < RP; ++i) out[kfirst + i * 32 + lane] = acc[i];
}

}  // namespace sl1m
