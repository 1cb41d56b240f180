// grx_ct.cu -- NEXT-2: constrained transport of the cell-centred calB^i by flux-CT (reading R30 in
// DESIGN.md; PAPER.md l.287, l.299, l.315 use constrained transport in every multi-dimensional test, l.194-196 name the face
// and edge locations; the paper prints no algorithm).
//
// F^j(calB^i) = eps_{ijk} E_k (d_t B = -curl E):  the EMF on a cell edge is the mean of the four HLLE face fluxes that touch
// it (with those signs), the flux of calB^i through a face is replaced by the mean of the two edge EMFs on that face, and
// d calB^i/dt is the difference of the replaced fluxes.  The vertex-centred divergence of the update vanishes to rounding.
//
// Face fluxes FB[6][cell] = F^x(B^y), F^x(B^z), F^y(B^x), F^y(B^z), F^z(B^x), F^z(B^y) at the LOW face of the cell (normal
// index 0..n, transverse -1..n).  The faces of the interior grid lines come out of the right-hand-side kernel itself
// (rhs_tma_kernel<.,.,true>); face_bflux_kernel adds the one layer of lines next to the block (and does all faces when the
// arrays do not qualify for the TMA kernel).
#include "grx_launch.h"

namespace grx {

namespace {

// One thread per cell of the block extended by one layer; evaluates the low faces of its cell that flux-CT reads and
// that the right-hand-side kernel has not written (all of them if `all`).
template <int RECON>
__global__ void __launch_bounds__(128) face_bflux_kernel(const RhsParams p, const int all) {
    const int ex = p.n[0] + 2, ey = p.n[1] + 2;
    long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int box = blockIdx.y;
    int i, j, k;
    if (all) {
        const long long per_box = (long long)ex * ey * (p.n[2] + 2);
        if (t >= per_box) return;
        i = (int)(t % ex) - 1;
        t /= ex;
        j = (int)(t % ey) - 1;
        k = (int)(t / ey) - 1;
    } else {
        // the cells with an index outside [0, n) only, enumerated region by region so that warps are full:
        // A: the two planes k = -1, n;  B: the rows j = -1, n of the planes between;  C: the columns i = -1, n of the rest
        const long long nA = 2LL * ex * ey, nB = 2LL * ex * p.n[2], nC = 2LL * p.n[1] * p.n[2];
        if (t < nA) {
            i = (int)(t % ex) - 1;
            t /= ex;
            j = (int)(t % ey) - 1;
            k = (t / ey) ? p.n[2] : -1;
        } else if (t < nA + nB) {
            t -= nA;
            i = (int)(t % ex) - 1;
            t /= ex;
            k = (int)(t % p.n[2]);
            j = (t / p.n[2]) ? p.n[1] : -1;
        } else if (t < nA + nB + nC) {
            t -= nA + nB;
            j = (int)(t % p.n[1]);
            t /= p.n[1];
            k = (int)(t % p.n[2]);
            i = (t / p.n[2]) ? p.n[0] : -1;
        } else {
            return;
        }
    }
    const bool ix = (i >= 0 && i < p.n[0]), iy = (j >= 0 && j < p.n[1]), iz = (k >= 0 && k < p.n[2]);   // interior index
    const double* __restrict__ prim = p.prim + (long long)box * 8 * p.nc;
    const double* __restrict__ met = p.met + (long long)box * 10 * p.nc;
    double* __restrict__ fb = p.fb + (long long)box * 6 * p.nc;
    const long long c = (i + p.g) + p.stride[1] * (j + p.g) + p.stride[2] * (k + p.g);
    unsigned nfb = 0;
    double Fh[8];
    // x face i-1/2: normal index 0..n; written by the right-hand-side kernel when (j, k) is an interior line
    if (i >= 0 && (all || !(iy && iz))) {
        face_from_global<0, RECON>(prim, met, p.nc, 1, c - 1, p.gamma, Fh, nfb);
        fb[c] = Fh[6];
        fb[p.nc + c] = Fh[7];
    }
    if (j >= 0 && (all || !(ix && iz))) {
        face_from_global<1, RECON>(prim, met, p.nc, p.stride[1], c - p.stride[1], p.gamma, Fh, nfb);
        fb[2 * p.nc + c] = Fh[5];
        fb[3 * p.nc + c] = Fh[7];
    }
    if (k >= 0 && (all || !(ix && iy))) {
        face_from_global<2, RECON>(prim, met, p.nc, p.stride[2], c - p.stride[2], p.gamma, Fh, nfb);
        fb[4 * p.nc + c] = Fh[5];
        fb[5 * p.nc + c] = Fh[6];
    }
}

// One thread per interior cell: twelve edge EMFs around the cell, replaced face fluxes, update of out[5..7].
__global__ void __launch_bounds__(256) flux_ct_kernel(const RhsParams p) {
    const int i = blockIdx.y * blockDim.x + threadIdx.x;
    if (i >= p.n[0]) return;
    const int j = blockIdx.x % p.n[1], k = blockIdx.x / p.n[1];     // rows in grid.x: up to 2^31 - 1 of them
    const int box = blockIdx.z;
    const long long nc = p.nc, sy = p.stride[1], sz = p.stride[2];
    const double* __restrict__ fb = p.fb + (long long)box * 6 * nc;
    double* __restrict__ out = p.out + (long long)box * 8 * nc;
    const long long c = (i + p.g) + sy * (j + p.g) + sz * (k + p.g);
    const double* FxBy = fb;
    const double* FxBz = fb + nc;
    const double* FyBx = fb + 2 * nc;
    const double* FyBz = fb + 3 * nc;
    const double* FzBx = fb + 4 * nc;
    const double* FzBy = fb + 5 * nc;
    // edge EMFs by the cell whose low-low edge it is: Ez(a) at (i-1/2, j-1/2, k) of cell a, ...
    auto Ez = [&](long long a) { return 0.25 * ((FyBx[a] + FyBx[a - 1]) - (FxBy[a] + FxBy[a - sy])); };
    auto Ex = [&](long long a) { return 0.25 * ((FzBy[a] + FzBy[a - sy]) - (FyBz[a] + FyBz[a - sz])); };
    auto Ey = [&](long long a) { return 0.25 * ((FxBz[a] + FxBz[a - sz]) - (FzBx[a] + FzBx[a - 1])); };
    const double ez00 = Ez(c), ez10 = Ez(c + 1), ez01 = Ez(c + sy), ez11 = Ez(c + sy + 1);
    const double ex00 = Ex(c), ex10 = Ex(c + sy), ex01 = Ex(c + sz), ex11 = Ex(c + sz + sy);
    const double ey00 = Ey(c), ey10 = Ey(c + 1), ey01 = Ey(c + sz), ey11 = Ey(c + sz + 1);
    // d_t B = -curl <E>, <E> = mean of the two edges of a face
    const double hx = 0.5 * p.idx[0], hy = 0.5 * p.idx[1], hz = 0.5 * p.idx[2];
    // dBx = -[ (Ez(j+1) - Ez(j)) / dy - (Ey(k+1) - Ey(k)) / dz ], each E averaged over its two x positions
    out[5 * nc + c] = -(((ez01 + ez11) - (ez00 + ez10)) * hy - ((ey01 + ey11) - (ey00 + ey10)) * hz);
    // dBy = -[ (Ex(k+1) - Ex(k)) / dz - (Ez(i+1) - Ez(i)) / dx ], averaged over the two y positions
    out[6 * nc + c] = -(((ex01 + ex11) - (ex00 + ex10)) * hz - ((ez10 + ez11) - (ez00 + ez01)) * hx);
    // dBz = -[ (Ey(i+1) - Ey(i)) / dx - (Ex(j+1) - Ex(j)) / dy ], averaged over the two z positions
    out[7 * nc + c] = -(((ey10 + ey11) - (ey00 + ey01)) * hx - ((ex10 + ex11) - (ex00 + ex01)) * hy);
}

}  // namespace

cudaError_t launch_face_bflux(const RhsParams& p, int recon, bool all, cudaStream_t st) {
    const long long ex = p.n[0] + 2, ey = p.n[1] + 2;
    const long long threads = all ? ex * ey * (p.n[2] + 2) : 2 * ex * ey + 2 * ex * p.n[2] + 2LL * p.n[1] * p.n[2];
    const dim3 grid((unsigned)((threads + 127) / 128), p.nbox);
    if (recon == RECON_WENO5) face_bflux_kernel<RECON_WENO5><<<grid, 128, 0, st>>>(p, all ? 1 : 0);
    else if (recon == RECON_MC) face_bflux_kernel<RECON_MC><<<grid, 128, 0, st>>>(p, all ? 1 : 0);
    else face_bflux_kernel<RECON_MINMOD><<<grid, 128, 0, st>>>(p, all ? 1 : 0);
    return cudaGetLastError();
}

cudaError_t launch_flux_ct(const RhsParams& p, cudaStream_t st) {
    const long long rows = (long long)p.n[1] * p.n[2];
    if (rows > 2147483647LL) return cudaErrorInvalidConfiguration;
    const int bx = p.n[0] >= 256 ? 256 : (p.n[0] >= 128 ? 128 : (p.n[0] >= 64 ? 64 : 32));
    const dim3 grid((unsigned)rows, (unsigned)((p.n[0] + bx - 1) / bx), p.nbox);
    flux_ct_kernel<<<grid, bx, 0, st>>>(p);
    return cudaGetLastError();
}

}  // namespace grx
