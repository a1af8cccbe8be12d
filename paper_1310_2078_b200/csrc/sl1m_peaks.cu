// sl1m_peaks.cu -- issue-rate micro-benchmark behind bench.py's roofline denominators (SURVEY.md 8(d):
// "the MUFU and FP32 issue rates re-measured by a micro-benchmark on the box").  The SL1M operator is bound by
// instruction issue (MUFU.SIN/COS/EX2 on the XU pipe, FFMA/FFMA2 on the FMA pipe), not by HBM, so the peaks its
// kernels are held against are measured here with the same instructions, launch shape (128-thread CTAs, several per
// SM on all SMs) and clock as the kernels themselves.  Reached through the C ABI: sl1m_measure_peaks().
#include "../../include/sl1m.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cstring>

namespace {

typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float lo, float hi) {
    f32x2 d;
    asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(lo), "f"(hi));
    return d;
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
    f32x2 d;
    asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ float ffma(float a, float b, float c) {
    float d;
    asm volatile("fma.rn.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c));
    return d;
}
__device__ __forceinline__ float mufu_ex2(float x) {
    float y;
    asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float mufu_cos(float x) {
    float y;
    asm volatile("cos.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float fmul_rz(float a, float b) {
    float d;
    asm volatile("mul.rz.f32 %0, %1, %2;" : "=f"(d) : "f"(a), "f"(b));
    return d;
}

// One loop body = N_MUFU independent MUFU chains + N_FMA independent scalar-FFMA chains + N_FMA2 independent
// packed-FFMA2 chains + N_RZ FMUL.RZ (the range-reduction multiply in front of MUFU.SIN/COS), per thread.
// Every chain is 8 deep per iteration so that the loop overhead (one add, one compare, one branch) is < 2 %.
template <int N_MUFU, int N_FMA, int N_FMA2, int N_RZ, bool COS>
__global__ void __launch_bounds__(128) probe_kernel(int iters, float seed, float *sink, long long *cycles) {
    float m[N_MUFU > 0 ? N_MUFU : 1], f[N_FMA > 0 ? N_FMA : 1], z[N_RZ > 0 ? N_RZ : 1];
    f32x2 p[N_FMA2 > 0 ? N_FMA2 : 1];
    const float t = seed + 1e-6f * (float)threadIdx.x;
#pragma unroll
    for (int i = 0; i < N_MUFU; ++i) m[i] = -0.25f * t - 0.01f * i;
#pragma unroll
    for (int i = 0; i < N_FMA; ++i) f[i] = t + i;
#pragma unroll
    for (int i = 0; i < N_FMA2; ++i) p[i] = pk2(t + i, t - i);
#pragma unroll
    for (int i = 0; i < N_RZ; ++i) z[i] = t + 0.5f * i;
    const f32x2 a2 = pk2(0.999f, 1.001f), b2 = pk2(1e-3f, -1e-3f);
    const long long c0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int d = 0; d < 8; ++d) {
#pragma unroll
            for (int i = 0; i < N_MUFU; ++i) m[i] = COS ? mufu_cos(m[i]) : mufu_ex2(m[i]);
#pragma unroll
            for (int i = 0; i < N_FMA; ++i) f[i] = ffma(f[i], 0.999f, 1e-3f);
#pragma unroll
            for (int i = 0; i < N_FMA2; ++i) p[i] = fma2(p[i], a2, b2);
#pragma unroll
            for (int i = 0; i < N_RZ; ++i) z[i] = fmul_rz(z[i], 0.9999f);
        }
    }
    const long long c1 = clock64();
    float acc = 0.f;
#pragma unroll
    for (int i = 0; i < N_MUFU; ++i) acc += m[i];
#pragma unroll
    for (int i = 0; i < N_FMA; ++i) acc += f[i];
#pragma unroll
    for (int i = 0; i < N_FMA2; ++i) acc += __uint_as_float((unsigned)(p[i] & 0xffffffffu)) + __uint_as_float((unsigned)(p[i] >> 32));
#pragma unroll
    for (int i = 0; i < N_RZ; ++i) acc += z[i];
    if (acc == 123.456f) sink[0] = acc;                       // never true: keeps the chains alive
    if (threadIdx.x == 0) cycles[blockIdx.x] = c1 - c0;
}

// FP64 pipe: 8 independent DFMA chains per thread, 8 deep per iteration (the fp64-phase kernels spend 3 DFMA + 1 DADD
// per term on it).
__global__ void __launch_bounds__(128) dfma_probe_kernel(int iters, double seed, float *sink) {
    double d[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) d[i] = seed + 1e-6 * (double)threadIdx.x + (double)i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
#pragma unroll
            for (int i = 0; i < 8; ++i) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(d[i]) : "d"(0.999), "d"(1e-3));
        }
    }
    double acc = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) acc += d[i];
    if (acc == 123.456) sink[0] = (float)acc;                 // never true: keeps the chains alive
}

struct Timed {
    double ms;        // best of the repetitions, CUDA events on the launching stream
    double cyc;       // median-free: mean SM cycles of a CTA's loop (clock64)
};

template <int N_MUFU, int N_FMA, int N_FMA2, int N_RZ, bool COS>
cudaError_t run_probe(int grid, int iters, float *sink, long long *cycles_dev, cudaStream_t s, Timed &out) {
    cudaEvent_t e0, e1;
    cudaError_t e;
    if ((e = cudaEventCreate(&e0)) != cudaSuccess) return e;
    if ((e = cudaEventCreate(&e1)) != cudaSuccess) { cudaEventDestroy(e0); return e; }
    out.ms = 1e30;
    for (int rep = 0; rep < 4; ++rep) {                        // rep 0 warms up (clocks, instruction cache)
        cudaEventRecord(e0, s);
        probe_kernel<N_MUFU, N_FMA, N_FMA2, N_RZ, COS><<<grid, 128, 0, s>>>(iters, 0.5f, sink, cycles_dev);
        cudaEventRecord(e1, s);
        if ((e = cudaEventSynchronize(e1)) != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0) out.ms = std::min(out.ms, (double)ms);
    }
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e == cudaSuccess) {
        long long *h = new long long[grid];
        e = cudaMemcpy(h, cycles_dev, sizeof(long long) * grid, cudaMemcpyDeviceToHost);
        double sum = 0.0;
        for (int i = 0; i < grid; ++i) sum += (double)h[i];
        out.cyc = sum / grid;
        delete[] h;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return e;
}

}  // namespace

extern "C" int sl1m_measure_peaks(sl1m_peaks *o, void *stream) {
    if (!o) return SL1M_ERR_NULL;
    memset(o, 0, sizeof(*o));
    int dev = 0, sms = 0, khz = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev) != cudaSuccess) {
        cudaGetLastError();
        return SL1M_ERR_CUDA;
    }
    cudaStream_t s = (cudaStream_t)stream;
    const int ctas_per_sm = 8, grid = sms * ctas_per_sm, iters = 4096;
    float *sink = nullptr;
    long long *cyc = nullptr;
    if (cudaMalloc((void **)&sink, sizeof(float)) != cudaSuccess) return SL1M_ERR_ALLOC;
    if (cudaMalloc((void **)&cyc, sizeof(long long) * grid) != cudaSuccess) { cudaFree(sink); return SL1M_ERR_ALLOC; }
    const double thr = (double)grid * 128.0, per_it = 8.0 * iters;   // threads, chain steps per chain per thread
    cudaError_t e = cudaSuccess;
    Timed t;
    // Per-clock figures are quoted at the device's maximum SM clock (cudaDevAttrClockRate; bench.py samples the
    // actual clock with nvidia-smi beside this): results per clock per SM = rate / (SMs x clock).  clock64 is
    // recorded too, but on this part it does not tick at the SM clock (measured 1,104 MHz under a 1,965 MHz SM
    // clock), so it is reported as is and used for nothing.
    const double clk_hz = (double)khz * 1e3;
    auto per_clk_sm = [&](double instr_per_thread_total, const Timed &tt) {
        return instr_per_thread_total * thr / (tt.ms * 1e-3) / ((double)sms * clk_hz);
    };
#define PROBE(NM, NF, NF2, NZ, COS) (e == cudaSuccess && (e = run_probe<NM, NF, NF2, NZ, COS>(grid, iters, sink, cyc, s, t)) == cudaSuccess)
    if (PROBE(4, 0, 0, 0, false)) {
        o->mufu_per_s = 4.0 * per_it * thr / (t.ms * 1e-3);
        o->mufu_per_clk_sm = per_clk_sm(4.0 * per_it, t);
        o->sm_clock_mhz = clk_hz * 1e-6;
        o->clock64_mhz = t.cyc / (t.ms * 1e-3) * 1e-6;        // mean clock64 span of a CTA / the event-timed duration
    }
    if (PROBE(4, 0, 0, 0, true)) o->mufu_cos_per_clk_sm = per_clk_sm(4.0 * per_it, t);
    if (PROBE(0, 16, 0, 0, false)) {
        o->ffma_per_s = 16.0 * per_it * thr / (t.ms * 1e-3);
        o->ffma_per_clk_sm = per_clk_sm(16.0 * per_it, t);
    }
    if (PROBE(0, 0, 16, 0, false)) {
        o->ffma2_lanes_per_s = 32.0 * per_it * thr / (t.ms * 1e-3);
        o->ffma2_lanes_per_clk_sm = per_clk_sm(32.0 * per_it, t);
    }
    // MUFU next to a packed-FMA stream: the 12 FFMA2 + 4 FMUL.RZ + 4 MUFU body of profiles/r1_microbench.md (a pair
    // of forward terms on the MUFU path is 5 FFMA2 + 2 FMUL.RZ + 4 MUFU, a polynomial pair 13 FFMA2 and no MUFU).
    if (PROBE(4, 0, 12, 4, false)) {
        o->coissue_mufu_per_clk_sm = per_clk_sm(4.0 * per_it, t);
        o->coissue_ffma2_lanes_per_clk_sm = per_clk_sm(24.0 * per_it, t);
        o->coissue_cycles_per_iter = (t.ms * 1e-3) * clk_hz / per_it / ctas_per_sm;   // sub-partition cycles per warp per body (8 warps each)
    }
    // the one-cosine adjoint's mix per pair of terms: 3 FFMA2 + 2 FMUL.RZ + 2 MUFU.COS + 1 FFMA2 -> x2: 8 FFMA2 + 4 RZ + 4 MUFU
    if (PROBE(4, 0, 8, 4, true)) o->coissue_adj_mufu_per_clk_sm = per_clk_sm(4.0 * per_it, t);
#undef PROBE
    if (e == cudaSuccess) {   // DFMA alone: best of 3 after a warm-up, CUDA events on the launching stream
        cudaEvent_t e0, e1;
        const int d_iters = 512;
        if (cudaEventCreate(&e0) == cudaSuccess && cudaEventCreate(&e1) == cudaSuccess) {
            double best = 1e30;
            for (int rep = 0; rep < 4 && e == cudaSuccess; ++rep) {
                cudaEventRecord(e0, s);
                dfma_probe_kernel<<<grid, 128, 0, s>>>(d_iters, 0.5, sink);
                cudaEventRecord(e1, s);
                e = cudaEventSynchronize(e1);
                float ms = 0.f;
                cudaEventElapsedTime(&ms, e0, e1);
                if (rep > 0) best = std::min(best, (double)ms);
            }
            if (e == cudaSuccess) {
                o->dfma_per_s = 64.0 * d_iters * thr / (best * 1e-3);
                o->dfma_per_clk_sm = o->dfma_per_s / ((double)sms * clk_hz);
            }
            cudaEventDestroy(e0);
            cudaEventDestroy(e1);
        }
    }
    cudaFree(sink);
    cudaFree(cyc);
    o->n_sm = sms;
    if (e != cudaSuccess) { cudaGetLastError(); return SL1M_ERR_CUDA; }
    return SL1M_OK;
}
