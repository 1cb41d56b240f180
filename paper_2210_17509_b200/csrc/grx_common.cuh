// grx_common.cuh -- launch parameters and global-memory helpers shared by the kernels of the CUDA path.
#pragma once

#include <cuda_runtime.h>

#include "grx_math.cuh"

namespace grx {

// One call's geometry and pointers (passed by value as a __grid_constant__ kernel parameter).
struct RhsParams {
    const double* prim;    // [nbox][8 ][Nz][Ny][Nx]
    const double* met;     // [nbox][10][Nz][Ny][Nx]
    const double* K;       // [nbox][6 ][Nz][Ny][Nx]
    double* out;           // [nbox][8 ][Nz][Ny][Nx]
    unsigned long long* nfallback;   // debug counter or nullptr
    int n[3];              // interior cells
    int N[3];              // cells incl. ghosts
    int g;                 // ghost width
    int nbox;
    long long nc;          // cells per field incl. ghosts = N[0]*N[1]*N[2]
    long long stride[3];   // element stride per direction: 1, Nx, Nx*Ny
    double idx[3];         // 1/dx
    double gamma;
};

__device__ __forceinline__ double ldg(const double* p) { return __ldg(p); }

// Face between cell iL and cell iL + stride[D], everything read from global memory: reconstruct the left
// cell's plus side and the right cell's minus side, average the metric, HLLE.  Used by the simple kernel
// and by the block-edge paths of the fused kernel.
template <int D, int RECON>
__device__ __forceinline__ void face_from_global(const double* __restrict__ prim, const double* __restrict__ met,
                                                 long long nc, long long s, long long iL, double gamma, double Fh[8],
                                                 unsigned& nfb) {
    const long long iR = iL + s;
    double PL[8], PR[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        const double* f = prim + q * nc;
        const double m1 = ldg(f + iL - s), c0 = ldg(f + iL), c1 = ldg(f + iR), p2 = ldg(f + iR + s);
        double m2 = 0.0, p3 = 0.0;
        if (RECON == RECON_WENO5) { m2 = ldg(f + iL - 2 * s); p3 = ldg(f + iR + 2 * s); }
        double qm, qp;
        recon_cell<RECON>(m2, m1, c0, c1, p2, qm, qp);
        PL[q] = qp;
        recon_cell<RECON>(m1, c0, c1, p2, p3, qm, qp);
        PR[q] = qm;
    }
    FaceGeom m;
    m.alp = 0.5 * (ldg(met + iL) + ldg(met + iR));
#pragma unroll
    for (int a = 0; a < 3; ++a) m.beta[a] = 0.5 * (ldg(met + (1 + a) * nc + iL) + ldg(met + (1 + a) * nc + iR));
#pragma unroll
    for (int c = 0; c < 6; ++c) m.g[c] = 0.5 * (ldg(met + (4 + c) * nc + iL) + ldg(met + (4 + c) * nc + iR));
    face_flux<D>(m, PL, PR, prim + iL, prim + iR, nc, gamma, Fh, nfb);
}

// Geometric sources of cell c0 (a8 + a9), everything read from global memory.
__device__ __forceinline__ void sources_from_global(const RhsParams& p, const double* __restrict__ prim,
                                                    const double* __restrict__ met, const double* __restrict__ K,
                                                    long long c0, double& sx, double& sy, double& sz, double& st) {
    double P[8], m[10], Kc[6], dm[3][10];
#pragma unroll
    for (int q = 0; q < 8; ++q) P[q] = ldg(prim + q * p.nc + c0);
#pragma unroll
    for (int c = 0; c < 6; ++c) Kc[c] = ldg(K + c * p.nc + c0);
#pragma unroll
    for (int f = 0; f < 10; ++f) {
        const double* mp = met + f * p.nc + c0;
        m[f] = ldg(mp);
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const long long s = p.stride[a];
            dm[a][f] = d4(ldg(mp - 2 * s), ldg(mp - s), ldg(mp + s), ldg(mp + 2 * s), p.idx[a] * (1.0 / 12.0));
        }
    }
    sources_point(P, m, Kc, dm, p.gamma, sx, sy, sz, st);
}

}  // namespace grx
