// host_math_harness.cpp -- TEST INFRASTRUCTURE (CPU box, -m "not gpu").
//
// Compiles the CUDA path's point-wise arithmetic (paper_2210_17509_b200/csrc/grx_math.cuh) as plain C++
// and drives it with the most naive loop possible (every cell evaluates its own six faces), so that the
// arithmetic the kernels use can be compared with the oracle on a machine without a GPU.  On the host the
// MUFU-seeded reciprocals are replaced by IEEE ones; everything else is the device code.  Never part of
// the product path: the library (libgrx.so) has no CPU fallback.
#include <cstddef>
#include <vector>

#include "../paper_2210_17509_b200/csrc/grx_math.cuh"

using namespace grx;

namespace {
struct Box {
    int n[3], g, N[3];
    size_t nc;
    long stride[3];
    size_t idx(int i, int j, int k) const { return (size_t)(i + g) + (size_t)N[0] * ((size_t)(j + g) + (size_t)N[1] * (size_t)(k + g)); }
};

template <int D, int RECON>
void face_at(const Box& B, const double* prim, const double* met, size_t iL, double gamma, double Fh[8], unsigned& nfb) {
    const long s = B.stride[D];
    const size_t iR = iL + s;
    double PL[8], PR[8];
    for (int q = 0; q < 8; ++q) {
        const double* f = prim + q * B.nc;
        double qm, qp;
        recon_cell<RECON>(f[iL - 2 * s], f[iL - s], f[iL], f[iL + s], f[iL + 2 * s], qm, qp);
        PL[q] = qp;
        recon_cell<RECON>(f[iR - 2 * s], f[iR - s], f[iR], f[iR + s], f[iR + 2 * s], qm, qp);
        PR[q] = qm;
    }
    FaceGeom m;
    m.alp = 0.5 * (met[iL] + met[iR]);
    for (int a = 0; a < 3; ++a) m.beta[a] = 0.5 * (met[(1 + a) * B.nc + iL] + met[(1 + a) * B.nc + iR]);
    for (int c = 0; c < 6; ++c) m.g[c] = 0.5 * (met[(4 + c) * B.nc + iL] + met[(4 + c) * B.nc + iR]);
    face_flux<D>(m, PL, PR, prim + iL, prim + iR, (long long)B.nc, gamma, Fh, nfb);
}

template <int D, int RECON>
void sweep(const Box& B, const double* prim, const double* met, double idx, double gamma, double* out, unsigned& nfb) {
    for (int k = 0; k < B.n[2]; ++k)
        for (int j = 0; j < B.n[1]; ++j)
            for (int i = 0; i < B.n[0]; ++i) {
                const size_t c0 = B.idx(i, j, k);
                double Flo[8], Fhi[8];
                unsigned dummy = 0;
                face_at<D, RECON>(B, prim, met, c0 - B.stride[D], gamma, Flo, nfb);
                // the high face is the low face of the next cell: count its fallbacks only at the block edge
                const bool last = ((D == 0 ? i : D == 1 ? j : k) == B.n[D] - 1);
                face_at<D, RECON>(B, prim, met, c0, gamma, Fhi, last ? nfb : dummy);
                for (int c = 0; c < 8; ++c) out[c * B.nc + c0] -= (Fhi[c] - Flo[c]) * idx;
            }
}

template <int RECON>
void rhs_box(const Box& B, const double* prim, const double* met, const double* K, const double dx[3], double gamma,
             double* out, unsigned& nfb) {
    for (int c = 0; c < 8; ++c)
        for (int k = 0; k < B.n[2]; ++k)
            for (int j = 0; j < B.n[1]; ++j)
                for (int i = 0; i < B.n[0]; ++i) out[c * B.nc + B.idx(i, j, k)] = 0.0;
    sweep<0, RECON>(B, prim, met, 1.0 / dx[0], gamma, out, nfb);
    sweep<1, RECON>(B, prim, met, 1.0 / dx[1], gamma, out, nfb);
    sweep<2, RECON>(B, prim, met, 1.0 / dx[2], gamma, out, nfb);
    for (int k = 0; k < B.n[2]; ++k)
        for (int j = 0; j < B.n[1]; ++j)
            for (int i = 0; i < B.n[0]; ++i) {
                const size_t c0 = B.idx(i, j, k);
                double P[8], m[10], Kc[6], dm[3][10];
                for (int q = 0; q < 8; ++q) P[q] = prim[q * B.nc + c0];
                for (int f = 0; f < 10; ++f) m[f] = met[f * B.nc + c0];
                for (int c = 0; c < 6; ++c) Kc[c] = K[c * B.nc + c0];
                for (int a = 0; a < 3; ++a)
                    for (int f = 0; f < 10; ++f) {
                        const double* p = met + f * B.nc + c0;
                        const long s = B.stride[a];
                        dm[a][f] = d4(p[-2 * s], p[-s], p[s], p[2 * s], 1.0 / (12.0 * dx[a]));
                    }
                double sx, sy, sz, st;
                sources_point(P, m, Kc, dm, gamma, sx, sy, sz, st);
                out[1 * B.nc + c0] += sx;
                out[2 * B.nc + c0] += sy;
                out[3 * B.nc + c0] += sz;
                out[4 * B.nc + c0] += st;
            }
}
}  // namespace

extern "C" {

int hm_valencia_rhs(const int n[3], int nbox, const double* prim, const double* met, const double* K, const double dx[3],
                    int g, int recon, double gamma, double* out, unsigned long long* nfallback) {
    Box B;
    for (int a = 0; a < 3; ++a) { B.n[a] = n[a]; B.N[a] = n[a] + 2 * g; }
    B.g = g;
    B.nc = (size_t)B.N[0] * B.N[1] * B.N[2];
    B.stride[0] = 1; B.stride[1] = B.N[0]; B.stride[2] = (long)B.N[0] * B.N[1];
    unsigned nfb = 0;
    for (int b = 0; b < nbox; ++b) {
        const double* p = prim + (size_t)b * 8 * B.nc;
        const double* m = met + (size_t)b * 10 * B.nc;
        const double* k = K + (size_t)b * 6 * B.nc;
        double* o = out + (size_t)b * 8 * B.nc;
        if (recon == RECON_WENO5) rhs_box<RECON_WENO5>(B, p, m, k, dx, gamma, o, nfb);
        else if (recon == RECON_MC) rhs_box<RECON_MC>(B, p, m, k, dx, gamma, o, nfb);
        else rhs_box<RECON_MINMOD>(B, p, m, k, dx, gamma, o, nfb);
    }
    if (nfallback) *nfallback = nfb;
    return 0;
}

void hm_recon_cell(int recon, const double q[5], double* qm, double* qp) {
    if (recon == RECON_WENO5) recon_cell<RECON_WENO5>(q[0], q[1], q[2], q[3], q[4], *qm, *qp);
    else if (recon == RECON_MC) recon_cell<RECON_MC>(q[0], q[1], q[2], q[3], q[4], *qm, *qp);
    else recon_cell<RECON_MINMOD>(q[0], q[1], q[2], q[3], q[4], *qm, *qp);
}

void hm_prim2con(const double P[8], const double met[10], double gamma, double U[8]) { prim2con_point(P, met, gamma, U); }
int hm_con2prim(const double U[8], const double met[10], double gamma, double P[8]) { return con2prim_point(U, met, gamma, P); }
int hm_con2prim_warm(const double U[8], const double met[10], double gamma, const double Pold[8], double P[8]) {
    return con2prim_point_warm(U, met, gamma, Pold, P);
}
// evaluations the warm solve needs from the old state Pold (-1: it gave up and the caller falls back to the bracket)
int hm_con2prim_warm_steps(const double U[8], const double met[10], double gamma, double z0) {
    C2P s;
    con2prim_setup(U, met, gamma, s);
    double z;
    return con2prim_solve_warm(s, z0, z) == 0 ? 0 : -1;
}

}  // extern "C"
