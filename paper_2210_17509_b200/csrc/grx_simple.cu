// grx_simple.cu -- cross-check variant of the right-hand side: one thread per interior cell, each thread
// evaluates the two faces of its cell in every direction straight from global memory (every interior face
// is therefore computed twice, every reconstruction up to three times).  It exists to validate the fused
// kernel against an independent traversal of the same arithmetic; it is not the product path.
#include "grx_launch.h"

namespace grx {

template <int D, int RECON>
__device__ __forceinline__ void sweep_cell(const RhsParams& p, const double* __restrict__ prim,
                                           const double* __restrict__ met, long long c0, bool last, double acc[8],
                                           unsigned& nfb) {
    double Flo[8], Fhi[8];
    unsigned dummy = 0;
    const long long s = p.stride[D];
    face_from_global<D, RECON>(prim, met, p.nc, s, c0 - s, p.gamma, Flo, nfb);
    // the high face is the next cell's low face: count its fallbacks only at the block edge
    face_from_global<D, RECON>(prim, met, p.nc, s, c0, p.gamma, Fhi, last ? nfb : dummy);
#pragma unroll
    for (int c = 0; c < 8; ++c) acc[c] = fma(-(Fhi[c] - Flo[c]), p.idx[D], acc[c]);
}

template <int RECON>
__global__ void __launch_bounds__(128) rhs_simple_kernel(const __grid_constant__ RhsParams p) {
    const int nxb = (p.n[0] + 127) / 128;
    const int i = (blockIdx.x % nxb) * 128 + threadIdx.x;
    const int row = blockIdx.x / nxb;          // j + ny * k
    const int j = row % p.n[1];
    const int k = row / p.n[1];
    const int box = blockIdx.y;
    if (i >= p.n[0]) return;
    const double* prim = p.prim + (long long)box * 8 * p.nc;
    const double* met = p.met + (long long)box * 10 * p.nc;
    const double* K = p.K + (long long)box * 6 * p.nc;
    double* out = p.out + (long long)box * 8 * p.nc;
    const long long c0 = (i + p.g) + p.stride[1] * (j + p.g) + p.stride[2] * (k + p.g);
    double acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    unsigned nfb = 0;
    sweep_cell<0, RECON>(p, prim, met, c0, i == p.n[0] - 1, acc, nfb);
    sweep_cell<1, RECON>(p, prim, met, c0, j == p.n[1] - 1, acc, nfb);
    sweep_cell<2, RECON>(p, prim, met, c0, k == p.n[2] - 1, acc, nfb);
    double sx, sy, sz, st;
    sources_from_global(p, prim, met, K, c0, sx, sy, sz, st);
    acc[1] += sx; acc[2] += sy; acc[3] += sz; acc[4] += st;
#pragma unroll
    for (int c = 0; c < 8; ++c) out[c * p.nc + c0] = acc[c];
    if (p.nfallback && nfb) atomicAdd(p.nfallback, (unsigned long long)nfb);
}

cudaError_t launch_rhs_simple(const RhsParams& p, int recon, cudaStream_t st) {
    const dim3 block(128);
    const dim3 grid((unsigned)((p.n[0] + 127) / 128) * (unsigned)p.n[1] * (unsigned)p.n[2], p.nbox);
    if (recon == RECON_WENO5) rhs_simple_kernel<RECON_WENO5><<<grid, block, 0, st>>>(p);
    else if (recon == RECON_MC) rhs_simple_kernel<RECON_MC><<<grid, block, 0, st>>>(p);
    else rhs_simple_kernel<RECON_MINMOD><<<grid, block, 0, st>>>(p);
    return cudaGetLastError();
}

}  // namespace grx
