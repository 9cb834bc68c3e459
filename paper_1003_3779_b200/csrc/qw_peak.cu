// qw_peak.cu — measured plain-ALU peak of the device, the denominator of the roofline of the temporally blocked /
// resident schedules (bench.py `roofline.peak_source: measured`).  Those kernels are bound by the FP64 pipe
// (complex128) or by the FP32 pipe fed with packed FP32x2 instructions (complex64), not by HBM,
// and their arithmetic is additions and fused multiply-adds on independent amplitudes (eq. 1 evaluated
// as butterflies, qw_coin.cuh).  This kernel issues exactly such instructions — long chains of independent
// DADD / DFMA / FADD2 / FFMA2 on registers, no memory traffic — from every SM and reports thread-level operations
// (a packed instruction counts two) per second.  It computes nothing of the walk.
#include "qw_coin.cuh"

namespace qw {

constexpr int PEAK_ACC = 16;          // independent accumulators per thread (hides the pipe latency)
constexpr int PEAK_INNER = 64;        // unrolled operations per accumulator per outer iteration

template <typename R, bool FMA>
__global__ void __launch_bounds__(256) alu_peak_kernel(R *sink, int outer, R seed) {
    cplx<R> acc[PEAK_ACC];
#pragma unroll
    for (int i = 0; i < PEAK_ACC; ++i) acc[i] = cplx<R>{seed * (R)(i + 1) + (R)threadIdx.x, seed * (R)(i + 2)};
    const cplx<R> inc{seed, -seed};
    const R mul = (R)1 + seed * (R)1e-3;
    for (int o = 0; o < outer; ++o) {
#pragma unroll
        for (int j = 0; j < PEAK_INNER; ++j) {
#pragma unroll
            for (int i = 0; i < PEAK_ACC; ++i) {
                if constexpr (FMA) acc[i] = cx_fma_r(mul, acc[i], inc);      // DFMA x2 / FFMA2
                else acc[i] = cx_add(acc[i], inc);                           // DADD x2 / FADD2
            }
        }
    }
    cplx<R> s{0, 0};
#pragma unroll
    for (int i = 0; i < PEAK_ACC; ++i) s = cx_add(s, acc[i]);
    if (s.re == (R)123.456 && s.im == (R)654.321) sink[0] = s.re;            // never true: keeps the chains alive
}

template <typename R, bool FMA>
static int measure(int sms, double *out) {
    R *sink = nullptr;
    QW_CUDA(cudaMalloc(&sink, sizeof(R)));
    cudaEvent_t a, b;
    QW_CUDA(cudaEventCreate(&a));
    QW_CUDA(cudaEventCreate(&b));
    const int blocks = sms * 8;                       // a multiple of the SM count; 8 x 256 threads fill every scheduler
    const int outer = sizeof(R) == 8 ? 48 : 96;
    double best = 0.0;
    for (int rep = 0; rep < 5; ++rep) {               // first repetition warms up; best of the rest
        QW_CUDA(cudaEventRecord(a, 0));
        alu_peak_kernel<R, FMA><<<blocks, 256>>>(sink, outer, (R)1e-7);
        QW_CUDA(cudaEventRecord(b, 0));
        QW_CUDA(cudaEventSynchronize(b));
        float ms = 0.f;
        QW_CUDA(cudaEventElapsedTime(&ms, a, b));
        // thread-level operations: every complex operation is 2 real ones (one packed FP32x2 instruction)
        const double ops = 2.0 * PEAK_ACC * PEAK_INNER * (double)outer * 256.0 * blocks;
        if (rep > 0 && ms > 0.f && ops / (ms * 1e-3) > best) best = ops / (ms * 1e-3);
    }
    cudaEventDestroy(a); cudaEventDestroy(b); cudaFree(sink);
    QW_CUDA(cudaGetLastError());
    *out = best;
    return QW_OK;
}

}  // namespace qw

using namespace qw;

extern "C" int qw_measure_alu_peak(int dtype, int op, double *ops_per_second) {
    clear_error();
    if (!ops_per_second) return fail(QW_EINVAL, "ops_per_second is NULL");
    if (dtype != QW_C64 && dtype != QW_C128) return fail(QW_EINVAL, "dtype must be QW_C64 or QW_C128");
    if (op != QW_PEAK_ADD && op != QW_PEAK_FMA) return fail(QW_EINVAL, "op must be QW_PEAK_ADD or QW_PEAK_FMA");
    int dev = 0, sms = 0;
    QW_CUDA(cudaGetDevice(&dev));
    QW_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    if (dtype == QW_C128) return op == QW_PEAK_ADD ? measure<double, false>(sms, ops_per_second) : measure<double, true>(sms, ops_per_second);
    return op == QW_PEAK_ADD ? measure<float, false>(sms, ops_per_second) : measure<float, true>(sms, ops_per_second);
}
