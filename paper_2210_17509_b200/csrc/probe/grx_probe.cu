// grx_probe.cu -- the FP64 micro-benchmarks behind bench.py's roofline object (see grx_probe.h).  Bench-side code: built
// as libgrx_probe.so, loaded by bench.py only; libgrx.so does not contain it.
#include <cuda_runtime.h>

#include "grx_probe.h"

namespace {

// 8 independent FMA chains per thread; every lane of the FP64 pipe busy, nothing else going on.
constexpr int DFMA_CHAINS = 8;
constexpr int DFMA_THREADS = 256;
__global__ void __launch_bounds__(DFMA_THREADS) dfma_peak_kernel(int iters, double* sink) {
    double a[DFMA_CHAINS];
    const double m = 1.0 + 1e-9 * threadIdx.x, c = 1e-12 * blockIdx.x;
#pragma unroll
    for (int q = 0; q < DFMA_CHAINS; ++q) a[q] = 0.1 * (q + 1);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
#pragma unroll
            for (int q = 0; q < DFMA_CHAINS; ++q) a[q] = fma(a[q], m, c);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int q = 0; q < DFMA_CHAINS; ++q) s += a[q];
    if (s == 1.2345678) *sink = s;   // keeps the chains alive without a store in the common case
}

constexpr int PROBE_THREADS = 256, PROBE_VALUES = 16, PROBE_MODES = 10;
template <int MODE>
__global__ void __launch_bounds__(PROBE_THREADS) issue_probe_kernel(int iters, double* sink, double k) {
    __shared__ double sh[PROBE_THREADS * 8];
    double r[PROBE_VALUES];
    int x[8];
    const double m = 1.0 - 1e-9 * (threadIdx.x & 7), c = 1e-12 * blockIdx.x;
#pragma unroll
    for (int i = 0; i < PROBE_VALUES; ++i) r[i] = 1.0 + 1e-9 * (threadIdx.x + i);
#pragma unroll
    for (int i = 0; i < 8; ++i) { x[i] = threadIdx.x + i; sh[threadIdx.x + PROBE_THREADS * i] = 1.0; }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < PROBE_VALUES; ++i) {
            const int j = (i + 1) % PROBE_VALUES, l = (i + 7) % PROBE_VALUES, n = (i + 11) % PROBE_VALUES;
            const int e2 = (i + 2) % PROBE_VALUES, e4 = (i + 4) % PROBE_VALUES, s = ((i & ~1) + 8) % PROBE_VALUES;
            if (MODE == 0) r[i] = fma(r[i], m, c);
            if (MODE == 1) r[i] = fma(r[j], r[l], r[n]);
            if (MODE >= 2 && MODE <= 5) r[i] = r[j] * r[l];
            if (MODE == 3) x[i % 8] = x[i % 8] * 5 + x[(i + 3) % 8];
            if (MODE == 4) sh[threadIdx.x + PROBE_THREADS * (i % 8)] = r[n];
            if (MODE == 5) x[i % 8] = __shfl_xor_sync(0xffffffffu, x[i % 8], 1);
            if (MODE == 6) r[i] = fma(r[j], r[e2], r[e4]);
            if (MODE == 7) r[i] = fma(r[j], r[e2], r[i]);
            if (MODE == 8) r[i] = fma(r[j], r[s], r[e4]);
            if (MODE == 9) r[i] = fma(r[j], r[e2], k);
        }
    }
    double t = 0.0;
#pragma unroll
    for (int i = 0; i < PROBE_VALUES; ++i) t += r[i];
#pragma unroll
    for (int i = 0; i < 8; ++i) t += x[i] + sh[(threadIdx.x * 7 + PROBE_THREADS * i) % (PROBE_THREADS * 8)];
    if (t == 1.2345678) *sink = t;
}

cudaError_t sm_count(int* sms) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    return cudaDeviceGetAttribute(sms, cudaDevAttrMultiProcessorCount, dev);
}

template <int MODE>
void launch_mode(int blocks, int iters, double* sink, cudaStream_t st) {
    issue_probe_kernel<MODE><<<blocks, PROBE_THREADS, 0, st>>>(iters, sink, 1.0 - 1e-9);
}

}  // namespace

extern "C" {

int grx_probe_dfma_peak(int iters, double* sink, double* flops_out, void* cuda_stream) {
    if (iters < 1 || !sink) return (int)cudaErrorInvalidValue;
    int sms = 0;
    cudaError_t e = sm_count(&sms);
    if (e != cudaSuccess) return (int)e;
    const int blocks = sms * 4;   // 4 x 256 threads per SM: 8 warps per scheduler
    dfma_peak_kernel<<<blocks, DFMA_THREADS, 0, static_cast<cudaStream_t>(cuda_stream)>>>(iters, sink);
    if (flops_out) *flops_out = 2.0 * 4.0 * DFMA_CHAINS * (double)iters * DFMA_THREADS * (double)blocks;
    return (int)cudaGetLastError();
}

int grx_probe_fp64_issue_modes(void) { return PROBE_MODES; }

int grx_probe_fp64_issue(int mode, int iters, double* sink, double* fp64_instr_out, void* cuda_stream) {
    if (iters < 1 || !sink) return (int)cudaErrorInvalidValue;
    int sms = 0;
    cudaError_t e = sm_count(&sms);
    if (e != cudaSuccess) return (int)e;
    const int blocks = sms * 2;   // 2 x 256 threads per SM: 4 warps per scheduler
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    switch (mode) {
        case 0: launch_mode<0>(blocks, iters, sink, st); break;
        case 1: launch_mode<1>(blocks, iters, sink, st); break;
        case 2: launch_mode<2>(blocks, iters, sink, st); break;
        case 3: launch_mode<3>(blocks, iters, sink, st); break;
        case 4: launch_mode<4>(blocks, iters, sink, st); break;
        case 5: launch_mode<5>(blocks, iters, sink, st); break;
        case 6: launch_mode<6>(blocks, iters, sink, st); break;
        case 7: launch_mode<7>(blocks, iters, sink, st); break;
        case 8: launch_mode<8>(blocks, iters, sink, st); break;
        case 9: launch_mode<9>(blocks, iters, sink, st); break;
        default: return (int)cudaErrorInvalidValue;
    }
    // FP64 thread-instructions of the launch (one per value and iteration)
    if (fp64_instr_out) *fp64_instr_out = (double)PROBE_VALUES * (double)iters * PROBE_THREADS * (double)blocks;
    return (int)cudaGetLastError();
}

}  // extern "C"
