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
    double* fb;            // [nbox][6][Nz][Ny][Nx] face fluxes of calB for constrained transport, or nullptr
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

// ---- 32-bit-offset addressing helpers (fused and split kernels) ---------------------------------------------
// Addressing: every thread keeps ONE 64-bit pointer per array (field 0 at its cell); field q and stencil
// neighbours are reached with 32-bit element offsets (nc = cells per field < 2^31, strides < nc), which
// costs one IMAD.WIDE per load instead of a 64-bit add pair.

// Reconstruct the 8 primitives of the cell at pc along a direction with element stride s.
template <int RECON>
__device__ __forceinline__ void recon8s(const double* __restrict__ pc, int nc, int s, double qm[8], double qp[8]) {
    const int s2 = 2 * s;
    const double* f = pc;
#pragma unroll
    for (int q = 0; q < 8; ++q, f += nc) {
        double a = 0.0, e = 0.0;
        if (RECON == RECON_WENO5) { a = ldg(f - s2); e = ldg(f + s2); }
        recon_cell<RECON>(a, ldg(f - s), ldg(f), ldg(f + s), e, qm[q], qp[q]);
    }
}

// Two-point average of the ten metric fields between the cell at mL and the next one along stride s (a1).
__device__ __forceinline__ void face_geom_load(const double* __restrict__ mL, int nc, int s, FaceGeom& m) {
    double v[10];
    const double* mf = mL;
#pragma unroll
    for (int f = 0; f < 10; ++f, mf += nc) v[f] = 0.5 * (ldg(mf) + ldg(mf + s));
    m.alp = v[0];
#pragma unroll
    for (int a = 0; a < 3; ++a) m.beta[a] = v[1 + a];
#pragma unroll
    for (int c = 0; c < 6; ++c) m.g[c] = v[4 + c];
}

// HLLE flux (times `scale` = 1/dx_d) of the face between the cell at (pL, mL) and the next one along stride s.
template <int D>
__device__ __forceinline__ void face8s(const double* __restrict__ pL, const double* __restrict__ mL, int nc, int s,
                                       double PL[8], double PR[8], double gamma, double scale,
                                       double Fh[8], unsigned& nfb) {
    FaceGeom m;
    face_geom_load(mL, nc, s, m);
    face_flux<D>(m, PL, PR, pL, pL + s, nc, gamma, Fh, nfb, scale);
}

// Ten unscaled 4th-order stencil sums of the metric fields along a direction with element stride s.
__device__ __forceinline__ void dmetric(const double* __restrict__ mc, int nc, int s, double d[10]) {
    const int s2 = 2 * s;
    const double* mp = mc;
#pragma unroll
    for (int f = 0; f < 10; ++f, mp += nc) d[f] = d4raw(ldg(mp - s2), ldg(mp - s), ldg(mp + s), ldg(mp + s2));
}

// Geometric sources of the cell at (pc, mc, kc) (a8 + a9) added to acc[1..4]; one direction's ten
// derivatives at a time.  The x stride is the constant 1, so those loads use immediate offsets.
__device__ __forceinline__ void sources_add(const RhsParams& p, const double* __restrict__ pc,
                                            const double* __restrict__ mc, const double* __restrict__ kc, int nc,
                                            int sy, int sz, double acc[8]) {
    SrcState s;
    {
        double P[8], m[10];
        const double* f = pc;
#pragma unroll
        for (int q = 0; q < 8; ++q, f += nc) P[q] = ldg(f);
        f = mc;
#pragma unroll
        for (int q = 0; q < 10; ++q, f += nc) m[q] = ldg(f);
        sources_prepare(P, m, p.gamma, s);
    }
    double st;
    {
        double K[6];
        const double* f = kc;
#pragma unroll
        for (int q = 0; q < 6; ++q, f += nc) K[q] = ldg(f);
        st = sources_K(s, K);
    }
    double d[10];
    dmetric(mc, nc, 1, d);
    acc[1] += sources_dir(s, 0, d, p.idx[0] * (1.0 / 12.0), st);
    dmetric(mc, nc, sy, d);
    acc[2] += sources_dir(s, 1, d, p.idx[1] * (1.0 / 12.0), st);
    dmetric(mc, nc, sz, d);
    acc[3] += sources_dir(s, 2, d, p.idx[2] * (1.0 / 12.0), st);
    acc[4] += st;
}

}  // namespace grx
