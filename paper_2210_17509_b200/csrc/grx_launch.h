// grx_launch.h -- internal: host-side launchers implemented by the kernel translation units.
#pragma once

#include <atomic>

#include <cuda_runtime.h>

#include "grx_common.cuh"

namespace grx {

// Current device of the calling thread and its SM count.  The count is asked from the runtime once per device and kept
// (lock-free; a launch needs it two or three times, and the query is a visible share of a small block's launch latency).
constexpr int MAX_CACHED_DEVICES = 64;
inline cudaError_t current_device_sms(int* dev_out, int* sms_out) {
    static std::atomic<int> cache[MAX_CACHED_DEVICES];   // zero-initialised: 0 = not asked yet
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const bool cached = dev >= 0 && dev < MAX_CACHED_DEVICES;
    int sms = cached ? cache[dev].load(std::memory_order_relaxed) : 0;
    if (sms <= 0) {
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return e;
        if (sms <= 0) return cudaErrorInvalidDevice;
        if (cached) cache[dev].store(sms, std::memory_order_relaxed);
    }
    *dev_out = dev;
    *sms_out = sms;
    return cudaSuccess;
}

// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) of one kernel instantiation, once per device: `done` is that
// instantiation's bit mask over devices (a function-local static of its launcher).
template <typename Kernel>
inline cudaError_t set_max_dynamic_smem_once(Kernel kernel, int dev, size_t smem, std::atomic<unsigned long long>& done) {
    const bool tracked = dev >= 0 && dev < MAX_CACHED_DEVICES;
    if (tracked && (done.load(std::memory_order_acquire) >> dev & 1ULL)) return cudaSuccess;
    const cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess && tracked) done.fetch_or(1ULL << dev, std::memory_order_release);
    return e;
}

// grx_simple.cu: one thread per cell, every thread evaluates its own six faces (cross-check variant)
cudaError_t launch_rhs_simple(const RhsParams& p, int recon, cudaStream_t st);
// grx_fused.cu: the round-1 kernel (operands through L1), the path for arrays the TMA kernel cannot take
cudaError_t launch_rhs_fused(const RhsParams& p, int recon, cudaStream_t st, int tile_nz = 0);   // tile_nz: see grx_fused.cu
cudaError_t launch_rhs_fused_vertex(const RhsParams& p, int recon, cudaStream_t st);   // NEXT-3: p.met, p.K = vertex arrays
double fused_tile_efficiency(const RhsParams& p, int sms);   // expected fill of the launch geometry, in (0, 1]

// grx_tma.cu: the product kernel (TMA-staged planes, shared-memory z rings); needs even Nx and 16-byte aligned arrays
bool tma_supported(const RhsParams& p);
cudaError_t launch_rhs_tma(const RhsParams& p, int recon, int ty, cudaStream_t st);
double tma_tile_efficiency(const RhsParams& p, int sms);

// grx_ct.cu: NEXT-2, flux-CT of calB.  launch_face_bflux fills p.fb on the lines next to the block (all = every face);
// launch_flux_ct replaces out[5..7] by the curl of the edge EMFs.
cudaError_t launch_face_bflux(const RhsParams& p, int recon, bool all, cudaStream_t st);
cudaError_t launch_flux_ct(const RhsParams& p, cudaStream_t st);

// grx_vertex.cu: NEXT-3, metric and K_ij sampled at the cell vertices (p.met / p.K point at vertex arrays)
cudaError_t launch_rhs_vertex(const RhsParams& p, int recon, cudaStream_t st);
cudaError_t launch_tmunu_vertex(const RhsParams& p, double* T, cudaStream_t st);

// grx_support.cu
cudaError_t launch_prim2con(const double* prim, const double* met, long long nc, int nbox, double gamma, double* cons,
                            cudaStream_t st);
cudaError_t launch_con2prim(const double* cons, const double* met, long long nc, int nbox, double gamma, double* prim,
                            unsigned long long* nfail, cudaStream_t st);
cudaError_t launch_rk_axpy(const RhsParams& geom, double a, const double* x, double b, double dt, const double* rhs,
                           double* y, cudaStream_t st);
cudaError_t launch_rk_stage(const RhsParams& geom, double a, const double* Ua, double b, const double* Ub, double h,
                            const double* L, double* Uout, double* acc, double wdt, double* prim, unsigned long long* nfail,
                            cudaStream_t st);
cudaError_t launch_fill_ghosts(const RhsParams& geom, double* prim, int bc, int dirs, cudaStream_t st);
cudaError_t launch_halo_z(const RhsParams& geom, double* prim, double* buf, int side, bool unpack, cudaStream_t st);
cudaError_t launch_halo_z_pull(const RhsParams& geom, double* prim, const double* below, const double* above, cudaStream_t st);
cudaError_t launch_selftest_math(const double* x, double* y, size_t n, cudaStream_t st);

}  // namespace grx
