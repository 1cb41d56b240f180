// grx_microbench.cu -- standalone B200 micro-benchmark behind the design numbers in DESIGN.md / profiles/r1_microbench.md:
// accuracy of the MUFU.RCP64H / MUFU.RSQ64H seeds and of the corrections grx_math.cuh applies to them, DFMA latency,
// DFMA throughput against warps per SM and independent chains per thread, MUFU.RCP64H throughput.
// Built by `python -m paper_2210_17509_b200.build` into paper_2210_17509_b200/grx_microbench; not part of libgrx.so.
#include <cstdio>
#include <cmath>
#include <cuda_runtime.h>
#include <vector>

__global__ void seed_err(const double* x, int n, double* out) {
    // out[0]=max rel err rcp seed, [1]=after 3rd-order, [2]=rsqrt seed, [3]=after 3rd-order, [4] rcp after 2nd order (1 newton)
    double e0 = 0, e1 = 0, e2 = 0, e3 = 0, e4 = 0, e5 = 0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        double v = x[i];
        double y; asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(v));
        double ex = 1.0 / v;
        e0 = fmax(e0, fabs(y - ex) / ex);
        double e = fma(-v, y, 1.0);
        double yn = fma(y, e, y);
        e4 = fmax(e4, fabs(yn - ex) / ex);
        double ee = fma(e, e, e);
        double y3 = fma(y, ee, y);
        e1 = fmax(e1, fabs(y3 - ex) / ex);
        double r; asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(v));
        double er = 1.0 / sqrt(v);
        e2 = fmax(e2, fabs(r - er) / er);
        double t = v * r; double h = fma(-t, r, 1.0); double p = fma(0.375, h, 0.5);
        double r3 = fma(r * h, p, r);
        e3 = fmax(e3, fabs(r3 - er) / er);
        double r2 = fma(0.5 * r, h, r);
        e5 = fmax(e5, fabs(r2 - er) / er);
    }
    // crude reduction via atomics on doubles as ull (positive -> monotone)
    atomicMax((unsigned long long*)&out[0], (unsigned long long)__double_as_longlong(e0));
    atomicMax((unsigned long long*)&out[1], (unsigned long long)__double_as_longlong(e1));
    atomicMax((unsigned long long*)&out[2], (unsigned long long)__double_as_longlong(e2));
    atomicMax((unsigned long long*)&out[3], (unsigned long long)__double_as_longlong(e3));
    atomicMax((unsigned long long*)&out[4], (unsigned long long)__double_as_longlong(e4));
    atomicMax((unsigned long long*)&out[5], (unsigned long long)__double_as_longlong(e5));
}

template <int ILP>
__global__ void dfma_chain(int iters, double* sink) {
    double a[ILP];
#pragma unroll
    for (int i = 0; i < ILP; ++i) a[i] = 1.0 + threadIdx.x * 1e-9 + i;
    const double b = 1.0000001, c = 1e-9;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u)
#pragma unroll
            for (int i = 0; i < ILP; ++i) a[i] = fma(a[i], b, c);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < ILP; ++i) s += a[i];
    if (s == 12345.678) sink[0] = s;
}

template <int ILP>
__global__ void rcp_chain(int iters, double* sink) {
    double a[ILP];
#pragma unroll
    for (int i = 0; i < ILP; ++i) a[i] = 1.5 + threadIdx.x * 1e-9 + i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u)
#pragma unroll
            for (int i = 0; i < ILP; ++i) { double y; asm volatile("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a[i])); a[i] = y; }
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < ILP; ++i) s += a[i];
    if (s == 12345.678) sink[0] = s;
}

template <typename K>
float timeit(K k, int blocks, int threads, int iters, double* sink) {
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    k<<<blocks, threads>>>(iters, sink);
    cudaDeviceSynchronize();
    float best = 1e30f;
    for (int r = 0; r < 3; ++r) {
        cudaEventRecord(e0); k<<<blocks, threads>>>(iters, sink); cudaEventRecord(e1); cudaEventSynchronize(e1);
        float ms; cudaEventElapsedTime(&ms, e0, e1); best = fminf(best, ms);
    }
    return best;
}

int main() {
    int n = 1 << 22;
    std::vector<double> h(n);
    unsigned long long s = 88172645463325252ULL;
    for (int i = 0; i < n; ++i) { s ^= s << 13; s ^= s >> 7; s ^= s << 17; double u = (s >> 11) * (1.0 / 9007199254740992.0);
        double ex = ((s >> 3) % 61) - 30.0; h[i] = (1.0 + u) * pow(2.0, ex); }
    double *dx, *dout; cudaMalloc(&dx, n * 8); cudaMalloc(&dout, 64); cudaMemset(dout, 0, 64);
    cudaMemcpy(dx, h.data(), n * 8, cudaMemcpyHostToDevice);
    seed_err<<<296, 256>>>(dx, n, dout);
    double o[6]; cudaMemcpy(o, dout, 48, cudaMemcpyDeviceToHost);
    printf("rcp seed relerr %.3e (2^%.1f)  newton1 %.3e  third-order %.3e\n", o[0], log2(o[0]), o[4], o[1]);
    printf("rsqrt seed relerr %.3e (2^%.1f)  newton1 %.3e  third-order %.3e\n", o[2], log2(o[2]), o[5], o[3]);
    int dev_clk; cudaDeviceGetAttribute(&dev_clk, cudaDevAttrClockRate, 0);
    printf("clock attr %d kHz\n", dev_clk);
    double* sink; cudaMalloc(&sink, 8);
    const int iters = 20000;
    // latency: 1 warp, 1 block, ILP 1
    {
        float ms = timeit(dfma_chain<1>, 1, 32, iters, sink);
        printf("DFMA dependent chain: %.2f ns/op -> %.2f cycles @1.965GHz\n", ms * 1e6 / (iters * 8.0), ms * 1e6 / (iters * 8.0) * 1.965);
        ms = timeit(rcp_chain<1>, 1, 32, iters, sink);
        printf("MUFU.RCP64H dependent chain: %.2f ns/op -> %.2f cycles\n", ms * 1e6 / (iters * 8.0), ms * 1e6 / (iters * 8.0) * 1.965);
    }
    // throughput vs warps/SM and ILP : blocks=148, threads = 32*w
    int ws[] = {4, 8, 12, 16, 24, 32};
    for (int w : ws) {
        float m1 = timeit(dfma_chain<1>, 148, 32 * w, iters, sink);
        float m2 = timeit(dfma_chain<2>, 148, 32 * w, iters, sink);
        float m4 = timeit(dfma_chain<4>, 148, 32 * w, iters, sink);
        auto tf = [&](float ms, int ilp) { return 148.0 * 32 * w * ilp * 8.0 * iters * 2 / (ms * 1e-3) / 1e12; };
        printf("warps/SM %2d: ILP1 %.2f TF  ILP2 %.2f TF  ILP4 %.2f TF\n", w, tf(m1, 1), tf(m2, 2), tf(m4, 4));
    }
    for (int w : {4, 8, 16}) {
        float m1 = timeit(rcp_chain<4>, 148, 32 * w, iters, sink);
        printf("MUFU rcp64h warps/SM %2d ILP4: %.3f Gop/s/SM-equiv -> %.2f lanes/clk/SM @1.965\n", w, 32.0 * w * 4 * 8 * iters / (m1 * 1e-3) / 1e9, 32.0 * w * 4 * 8 * iters / (m1 * 1e-3) / 1.965e9);
    }
    return 0;
}
