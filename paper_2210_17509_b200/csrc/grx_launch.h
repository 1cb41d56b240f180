// grx_launch.h -- internal: host-side launchers implemented by the kernel translation units.
#pragma once

#include <cuda_runtime.h>

#include "grx_common.cuh"

namespace grx {

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
cudaError_t launch_dfma_peak(int iters, double* sink, double* flops_out, cudaStream_t st);
cudaError_t launch_issue_probe(int mode, int iters, double* sink, double* fp64_instr_out, cudaStream_t st);

}  // namespace grx
