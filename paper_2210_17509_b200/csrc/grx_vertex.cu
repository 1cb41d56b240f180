// grx_vertex.cu -- NEXT-3: the paper's own centring of the spacetime fields (PAPER.md l.84, l.130,
// l.166, l.323; readings R31 / R32 in DESIGN.md).  Metric and K_ij are sampled at the cell VERTICES,
//     metv[box][10][Nz+1][Ny+1][Nx+1],   vertex (I, J, K) = low corner of cell (I, J, K),
// and
//   rhs_vertex_kernel    evaluates the right-hand side with face metric = mean of the 4 vertices of the face (l.130),
//                        cell-centre metric and K_ij = mean of the 8 vertices, and the staggered 4th-order difference
//                        [27 (m(+1/2) - m(-1/2)) - (m(+3/2) - m(-3/2))] / (24 dx) of the transverse 4-vertex means;
//   tmunu_vertex_kernel  interpolates the 8 primitives to the vertices with the tensor product of (-1, 9, 9, -1)/16
//                        ("4th-order symmetric 3D interpolation", l.84) and evaluates T^{mu nu} (Eq. 5) there.
// rhs_vertex_kernel is the cross-check traversal of this centring (one thread per cell straight from global memory, every face
// evaluated by both of its cells, as in grx_simple.cu); the product path of grx_valencia_rhs_vertex is the face-once tile
// traversal rhs_fused_kernel<..., VERTEX> in grx_fused.cu, which shares the vertex loads of grx_vertex.cuh.
#include "grx_launch.h"
#include "grx_vertex.cuh"

namespace grx {

namespace {

// Face between cell iL and cell iR = iL + s along D; vR = vertex index of the low corner of cell iR.
template <int D, int RECON>
__device__ __forceinline__ void face_vertex(const double* __restrict__ prim, const double* __restrict__ metv, long long nc,
                                            const VStride& vs, long long s, long long iL, long long vR, double gamma,
                                            double Fh[8], unsigned& nfb) {
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
    face_geom_vertex<D>(metv, vs, vR, m);
    face_flux<D>(m, PL, PR, prim + iL, prim + iR, nc, gamma, Fh, nfb);
}

template <int D, int RECON>
__device__ __forceinline__ void sweep_vertex(const RhsParams& p, const VStride& vs, const double* __restrict__ prim,
                                             const double* __restrict__ metv, long long c0, long long v0, bool last,
                                             double acc[8], unsigned& nfb) {
    double Flo[8], Fhi[8];
    unsigned dummy = 0;
    const long long s = p.stride[D];
    face_vertex<D, RECON>(prim, metv, p.nc, vs, s, c0 - s, v0, p.gamma, Flo, nfb);
    face_vertex<D, RECON>(prim, metv, p.nc, vs, s, c0, v0 + vs.s[D], p.gamma, Fhi, last ? nfb : dummy);
#pragma unroll
    for (int c = 0; c < 8; ++c) acc[c] = fma(-(Fhi[c] - Flo[c]), p.idx[D], acc[c]);
}

template <int RECON>
__global__ void __launch_bounds__(128) rhs_vertex_kernel(const __grid_constant__ RhsParams p, const VStride vs) {
    const int nxb = (p.n[0] + 127) / 128;
    const int i = (blockIdx.x % nxb) * 128 + threadIdx.x;
    const int row = blockIdx.x / nxb;
    const int j = row % p.n[1], k = row / p.n[1];
    const int box = blockIdx.y;
    if (i >= p.n[0]) return;
    const double* prim = p.prim + (long long)box * 8 * p.nc;
    const double* metv = p.met + (long long)box * 10 * vs.nv;
    const double* Kv = p.K + (long long)box * 6 * vs.nv;
    double* out = p.out + (long long)box * 8 * p.nc;
    const long long c0 = (i + p.g) + p.stride[1] * (j + p.g) + p.stride[2] * (k + p.g);
    const long long v0 = (i + p.g) + vs.s[1] * (j + p.g) + vs.s[2] * (k + p.g);
    double acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    unsigned nfb = 0;
    sweep_vertex<0, RECON>(p, vs, prim, metv, c0, v0, i == p.n[0] - 1, acc, nfb);
    sweep_vertex<1, RECON>(p, vs, prim, metv, c0, v0, j == p.n[1] - 1, acc, nfb);
    sweep_vertex<2, RECON>(p, vs, prim, metv, c0, v0, k == p.n[2] - 1, acc, nfb);
    double sx, sy, sz, st;
    sources_from_vertices(p, vs, prim, metv, Kv, c0, v0, sx, sy, sz, st);
    acc[1] += sx; acc[2] += sy; acc[3] += sz; acc[4] += st;
#pragma unroll
    for (int c = 0; c < 8; ++c) out[c * p.nc + c0] = acc[c];
    if (p.nfallback && nfb) atomicAdd(p.nfallback, (unsigned long long)nfb);
}

// T^{mu nu} = rho h* u^mu u^nu + P* g^{mu nu} - b^mu b^nu (Eq. 5) at one point; T[10] = 00 0x 0y 0z xx xy xz yy yz zz.
__device__ __forceinline__ void tmunu_point(const double P[8], const double met[10], double gamma, double T[10]) {
    const double rho = P[0], eps = P[4];
    const double v[3] = {P[1], P[2], P[3]}, B[3] = {P[5], P[6], P[7]};
    const double alp = met[0], beta[3] = {met[1], met[2], met[3]};
    const double gxx = met[4], gxy = met[5], gxz = met[6], gyy = met[7], gyz = met[8], gzz = met[9];
    const double cof[6] = {fma(gyy, gzz, -gyz * gyz), fma(gxz, gyz, -gxy * gzz), fma(gxy, gyz, -gxz * gyy),
                           fma(gxx, gzz, -gxz * gxz), fma(gxy, gxz, -gxx * gyz), fma(gxx, gyy, -gxy * gxy)};
    const double idet = rcp(fma(gxx, cof[0], fma(gxy, cof[1], gxz * cof[2])));
    const double vl[3] = {fma(gxx, v[0], fma(gxy, v[1], gxz * v[2])), fma(gxy, v[0], fma(gyy, v[1], gyz * v[2])),
                          fma(gxz, v[0], fma(gyz, v[1], gzz * v[2]))};
    const double Bl[3] = {fma(gxx, B[0], fma(gxy, B[1], gxz * B[2])), fma(gxy, B[0], fma(gyy, B[1], gyz * B[2])),
                          fma(gxz, B[0], fma(gyz, B[1], gzz * B[2]))};
    const double v2 = fma(vl[0], v[0], fma(vl[1], v[1], vl[2] * v[2]));
    const double iW2 = 1.0 - v2, W = rsqrt(iW2), ia = rcp(alp);
    const double Bv = fma(Bl[0], v[0], fma(Bl[1], v[1], Bl[2] * v[2]));
    const double B2 = fma(Bl[0], B[0], fma(Bl[1], B[1], Bl[2] * B[2]));
    const double ab0 = W * Bv;                                    // alpha b^0
    const double b2 = fma(B2, iW2, Bv * Bv);
    const double p = (gamma - 1.0) * rho * eps;
    const double rhohs = fma(gamma, rho * eps, rho) + b2, Ps = fma(0.5, b2, p);
    double u[4], b[4];
    u[0] = W * ia;
    b[0] = ab0 * ia;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        const double vt = fma(-beta[i], ia, v[i]);                // v^i - beta^i / alpha
        u[1 + i] = W * vt;
        b[1 + i] = fma(B[i], W * iW2, ab0 * vt);                  // B^i / W + alpha b^0 vtilde^i
    }
    const double ia2 = ia * ia;
    T[0] = fma(rhohs * u[0], u[0], fma(-Ps, ia2, -b[0] * b[0]));
#pragma unroll
    for (int i = 0; i < 3; ++i) T[1 + i] = fma(rhohs * u[0], u[1 + i], fma(Ps * ia2, beta[i], -b[0] * b[1 + i]));
    int n = 4;
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = i; j < 3; ++j) {
            const int c = (i == 0) ? j : (i == 1 ? 2 + j : 5);
            const double gij = fma(cof[c], idet, -beta[i] * beta[j] * ia2);
            T[n++] = fma(rhohs * u[1 + i], u[1 + j], fma(Ps, gij, -b[1 + i] * b[1 + j]));
        }
}

// One thread per vertex COLUMN (i, j) of a z chunk, marching along z: each step interpolates the 8 primitives of one cell
// plane to the column's (x, y) position (4 x 4 cells, symmetric pairs first), keeps the last four planes' values in
// registers and combines them along z -- 128 loads per vertex instead of 512, all of them rows that neighbouring lanes
// share through L1.  T^{mu nu} is then evaluated with the vertex's own metric sample.
constexpr int TMUNU_ZCHUNK = 64;
__global__ void __launch_bounds__(128) tmunu_vertex_kernel(const __grid_constant__ RhsParams p, const VStride vs, double* Tout) {
    const int nxb = (p.n[0] + 1 + 127) / 128;
    const int i = (blockIdx.x % nxb) * 128 + threadIdx.x;
    const int j = blockIdx.x / nxb;
    const int k0 = blockIdx.y * TMUNU_ZCHUNK, k1 = min(k0 + TMUNU_ZCHUNK, p.n[2] + 1);     // vertices k0 .. k1-1
    const int box = blockIdx.z;
    if (i > p.n[0]) return;
    const double* prim = p.prim + (long long)box * 8 * p.nc;
    const double* metv = p.met + (long long)box * 10 * vs.nv;
    double* T = Tout + (long long)box * 10 * vs.nv;
    // the 4 x 4 cells around the column start at cell (i-2, j-2); vertex k needs the cell planes k-2 .. k+1
    long long c = (i - 2 + p.g) + p.stride[1] * (j - 2 + p.g) + p.stride[2] * (k0 - 2 + p.g);
    long long v = (i + p.g) + vs.s[1] * (j + p.g) + vs.s[2] * (k0 + p.g);
    const double w9 = 9.0 / 16.0, w1 = -1.0 / 16.0;
    double r0[8], r1[8], r2[8], r3[8];   // in-plane interpolants of the last four cell planes, oldest first
#pragma unroll
    for (int q = 0; q < 8; ++q) r0[q] = r1[q] = r2[q] = r3[q] = 0.0;
    for (int kz = k0 - 2; kz <= k1; ++kz, c += p.stride[2]) {
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const double* f = prim + q * p.nc + c;
            double h[4];
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                const double* r = f + b * p.stride[1];
                h[b] = fma(w9, ldg(r + 1) + ldg(r + 2), w1 * (ldg(r) + ldg(r + 3)));
            }
            r0[q] = r1[q]; r1[q] = r2[q]; r2[q] = r3[q];
            r3[q] = fma(w9, h[1] + h[2], w1 * (h[0] + h[3]));
        }
        const int k = kz - 1;            // the vertex whose four planes are complete now
        if (k >= k0) {
            double P[8], m[10], T10[10];
#pragma unroll
            for (int q = 0; q < 8; ++q) P[q] = fma(w9, r1[q] + r2[q], w1 * (r0[q] + r3[q]));
#pragma unroll
            for (int f = 0; f < 10; ++f) m[f] = ldg(metv + f * vs.nv + v);
            tmunu_point(P, m, p.gamma, T10);
#pragma unroll
            for (int cc = 0; cc < 10; ++cc) T[cc * vs.nv + v] = T10[cc];
            v += vs.s[2];
        }
    }
}

}  // namespace

cudaError_t launch_rhs_vertex(const RhsParams& p, int recon, cudaStream_t st) {
    const dim3 grid((unsigned)((p.n[0] + 127) / 128) * (unsigned)p.n[1] * (unsigned)p.n[2], p.nbox);
    const VStride vs = vstride(p);
    if (recon == RECON_WENO5) rhs_vertex_kernel<RECON_WENO5><<<grid, 128, 0, st>>>(p, vs);
    else if (recon == RECON_MC) rhs_vertex_kernel<RECON_MC><<<grid, 128, 0, st>>>(p, vs);
    else rhs_vertex_kernel<RECON_MINMOD><<<grid, 128, 0, st>>>(p, vs);
    return cudaGetLastError();
}

cudaError_t launch_tmunu_vertex(const RhsParams& p, double* T, cudaStream_t st) {
    const dim3 grid((unsigned)((p.n[0] + 1 + 127) / 128) * (unsigned)(p.n[1] + 1),
                    (unsigned)((p.n[2] + 1 + TMUNU_ZCHUNK - 1) / TMUNU_ZCHUNK), p.nbox);
    tmunu_vertex_kernel<<<grid, 128, 0, st>>>(p, vstride(p), T);
    return cudaGetLastError();
}

}  // namespace grx
