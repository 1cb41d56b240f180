// grx_vertex.cuh -- NEXT-3 (reading R31): loads of a vertex-centred metric, shared by the kernels that take one.
// Vertex arrays are [field][Nz+1][Ny+1][Nx+1]; vertex (I, J, K) is the low corner of cell (I, J, K).
#pragma once

#include "grx_common.cuh"

namespace grx {

struct VStride {
    long long s[3];   // vertex strides: 1, Nx+1, (Nx+1)(Ny+1)
    long long nv;     // vertices per field
};

inline VStride vstride(const RhsParams& p) {
    VStride vs;
    vs.s[0] = 1;
    vs.s[1] = p.N[0] + 1;
    vs.s[2] = (long long)(p.N[0] + 1) * (p.N[1] + 1);
    vs.nv = vs.s[2] * (p.N[2] + 1);
    return vs;
}

// mean of the 4 vertices v, v+a, v+b, v+a+b (a face of a cell: a, b = the two transverse vertex strides)
__device__ __forceinline__ double mean4(const double* __restrict__ f, long long v, long long a, long long b) {
    return 0.25 * ((ldg(f + v) + ldg(f + v + b)) + (ldg(f + v + a) + ldg(f + v + a + b)));
}

// Face metric of the low D-face of the cell whose low-corner vertex is vR: mean of the 4 vertices of the face (l.130).
template <int D>
__device__ __forceinline__ void face_geom_vertex(const double* __restrict__ metv, const VStride& vs, long long vR, FaceGeom& m) {
    const long long a = vs.s[(D + 1) % 3], b = vs.s[(D + 2) % 3];
    m.alp = mean4(metv, vR, a, b);
#pragma unroll
    for (int i = 0; i < 3; ++i) m.beta[i] = mean4(metv + (1 + i) * vs.nv, vR, a, b);
#pragma unroll
    for (int c = 0; c < 6; ++c) m.g[c] = mean4(metv + (4 + c) * vs.nv, vR, a, b);
}

// Geometric sources of the cell c0 whose low-corner vertex is v0: cell-centre metric and K_ij = mean of the 8 vertices,
// d_a of a metric field = [27 (m(+1/2) - m(-1/2)) - (m(+3/2) - m(-3/2))] / (24 dx_a) of the transverse 4-vertex means.
__device__ __forceinline__ void sources_from_vertices(const RhsParams& p, const VStride& vs, const double* __restrict__ prim,
                                                      const double* __restrict__ metv, const double* __restrict__ Kv,
                                                      long long c0, long long v0, double& sx, double& sy, double& sz,
                                                      double& st) {
    double P[8], mc[10], Kc[6], dm[3][10];
#pragma unroll
    for (int q = 0; q < 8; ++q) P[q] = ldg(prim + q * p.nc + c0);
#pragma unroll
    for (int f = 0; f < 10; ++f) {
        const double* mv = metv + f * vs.nv;
        double lo = 0.0, hi = 0.0;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const long long sa = vs.s[a], t1 = vs.s[(a + 1) % 3], t2 = vs.s[(a + 2) % 3];
            const double m_m2 = mean4(mv, v0 - sa, t1, t2), m_m1 = mean4(mv, v0, t1, t2);
            const double m_p1 = mean4(mv, v0 + sa, t1, t2), m_p2 = mean4(mv, v0 + 2 * sa, t1, t2);
            dm[a][f] = fma(27.0, m_p1 - m_m1, -(m_p2 - m_m2)) * (p.idx[a] * (1.0 / 24.0));
            if (a == 0) { lo = m_m1; hi = m_p1; }
        }
        mc[f] = 0.5 * (lo + hi);
    }
#pragma unroll
    for (int c = 0; c < 6; ++c)
        Kc[c] = 0.5 * (mean4(Kv + c * vs.nv, v0, vs.s[1], vs.s[2]) + mean4(Kv + c * vs.nv, v0 + 1, vs.s[1], vs.s[2]));
    sources_point(P, mc, Kc, dm, p.gamma, sx, sy, sz, st);
}

}  // namespace grx
