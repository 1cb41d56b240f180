// grx_support.cu -- small kernels around the hot path: prim2con (Eqs. 6-9), the support
// con2prim and RK update (R21/R22), the accuracy self-test of rcp/rsqrt and the DFMA peak micro-benchmark.
#include "grx_launch.h"

namespace grx {

__global__ void __launch_bounds__(256) prim2con_kernel(const double* __restrict__ prim, const double* __restrict__ met,
                                                       long long nc, double gamma, double* __restrict__ cons) {
    const long long c0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (c0 >= nc) return;
    const long long box = blockIdx.y;
    const double* pb = prim + box * 8 * nc;
    const double* mb = met + box * 10 * nc;
    double* cb = cons + box * 8 * nc;
    double P[8], m[10], U[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) P[q] = pb[q * nc + c0];
#pragma unroll
    for (int f = 0; f < 10; ++f) m[f] = mb[f * nc + c0];
    prim2con_point(P, m, gamma, U);
#pragma unroll
    for (int q = 0; q < 8; ++q) cb[q * nc + c0] = U[q];
}

__global__ void __launch_bounds__(128) con2prim_kernel(const double* __restrict__ cons, const double* __restrict__ met,
                                                       long long nc, double gamma, double* __restrict__ prim,
                                                       unsigned long long* nfail) {
    const long long c0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (c0 >= nc) return;
    const long long box = blockIdx.y;
    const double* cb = cons + box * 8 * nc;
    const double* mb = met + box * 10 * nc;
    double* pb = prim + box * 8 * nc;
    double P[8], m[10], U[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) U[q] = cb[q * nc + c0];
#pragma unroll
    for (int f = 0; f < 10; ++f) m[f] = mb[f * nc + c0];
    const int bad = con2prim_point(U, m, gamma, P);
#pragma unroll
    for (int q = 0; q < 8; ++q) pb[q * nc + c0] = P[q];
    if (bad && nfail) atomicAdd(nfail, 1ULL);
}

__global__ void __launch_bounds__(128) rk_axpy_kernel(const __grid_constant__ RhsParams p, double a,
                                                      const double* __restrict__ x, double b, double dt,
                                                      const double* __restrict__ rhs, double* y) {
    const int nxb = (p.n[0] + 127) / 128;
    const int i = (blockIdx.x % nxb) * 128 + threadIdx.x;
    const int row = blockIdx.x / nxb;
    const int j = row % p.n[1], k = row / p.n[1];
    if (i >= p.n[0]) return;
    const long long base = (long long)blockIdx.y * 8 * p.nc + (i + p.g) + p.stride[1] * (j + p.g) + p.stride[2] * (k + p.g);
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        const long long o = base + c * p.nc;
        y[o] = a * x[o] + b * (y[o] + dt * rhs[o]);
    }
}

// NEXT-1: one Runge-Kutta stage on the interior cells, fused with con2prim:
//   U_out = a U_a + b (U_b + h L);   acc += wdt L (RK4 only);   prim = con2prim(U_out).
__global__ void __launch_bounds__(128) rk_stage_kernel(const __grid_constant__ RhsParams p, double a, const double* Ua, double b,
                                                       const double* Ub, double h, const double* __restrict__ L,
                                                       double* Uout, double* acc, double wdt, double* __restrict__ prim,
                                                       unsigned long long* nfail) {
    const int nxb = (p.n[0] + 127) / 128;
    const int i = (blockIdx.x % nxb) * 128 + threadIdx.x;
    const int row = blockIdx.x / nxb;
    const int j = row % p.n[1], k = row / p.n[1];
    if (i >= p.n[0]) return;
    const long long c0 = (i + p.g) + p.stride[1] * (j + p.g) + p.stride[2] * (k + p.g);
    const long long ub = (long long)blockIdx.y * 8 * p.nc + c0;
    const double* mb = p.met + (long long)blockIdx.y * 10 * p.nc + c0;
    double U[8], P[8], Pold[8], m[10];
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        const long long o = ub + c * p.nc;
        const double l = L[o];
        U[c] = a * Ua[o] + b * (Ub[o] + h * l);
        Uout[o] = U[c];
        if (acc) acc[o] += wdt * l;
        Pold[c] = prim[o];      // the state the stage started from: warm start of the solve
    }
#pragma unroll
    for (int f = 0; f < 10; ++f) m[f] = mb[f * p.nc];
    const int bad = con2prim_point_warm(U, m, p.gamma, Pold, P);
#pragma unroll
    for (int c = 0; c < 8; ++c) prim[ub + c * p.nc] = P[c];
    if (bad && nfail) atomicAdd(nfail, 1ULL);
}

// NEXT-1: ghost fill of the 8 primitives at the outer boundary of every box (l.170, l.255, l.329): a ghost cell takes the
// interior cell whose index is its own, clamped (bc = 0, "copy") or wrapped (bc = 1, periodic) direction by direction.
// `dirs`: bit d set = direction d is filled here; a cell that is a ghost cell only in other directions is left alone
// (NEXT-4: the z ghost planes of a slab decomposition come from the neighbour ranks).
__global__ void __launch_bounds__(256) fill_ghosts_kernel(const __grid_constant__ RhsParams p, double* prim, int bc, int dirs) {
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= p.nc) return;
    const int I = (int)(c % p.N[0]), J = (int)((c / p.N[0]) % p.N[1]), Kz = (int)(c / p.stride[2]);
    int s[3] = {I - p.g, J - p.g, Kz - p.g};
    bool ghost = false;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const int n = p.n[d];
        int v = s[d];
        if ((v < 0 || v >= n) && ((dirs >> d) & 1)) {
            ghost = true;
            v = bc == 1 ? ((v % n) + n) % n : (v < 0 ? 0 : n - 1);
        }
        s[d] = v;
    }
    if (!ghost) return;
    // unfilled directions keep their own (ghost) index: s[d] + g is the cell's own coordinate there
    const long long src = (s[0] + p.g) + p.stride[1] * (s[1] + p.g) + p.stride[2] * (s[2] + p.g);
    double* pb = prim + (long long)blockIdx.y * 8 * p.nc;
#pragma unroll
    for (int q = 0; q < 8; ++q) pb[q * p.nc + c] = pb[q * p.nc + src];
}


// NEXT-4: the z ghost planes of a slab decomposition.  side 0: the g lowest
// interior planes (sent to the rank below, whose high ghost planes they fill), side 1: the g highest interior planes.
// buf[box][field][g][Ny][Nx], planes complete with their x and y ghost cells (fill those first: corners come along).
// unpack: side 0 = the g low ghost planes, side 1 = the g high ghost planes.
__global__ void __launch_bounds__(256) halo_z_kernel(const __grid_constant__ RhsParams p, double* prim, double* buf, int side,
                                                     int unpack) {
    const long long slab = (long long)p.g * p.stride[2];
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= slab) return;
    const int bf = blockIdx.y;   // box * 8 + field
    const int k0 = unpack ? (side == 0 ? 0 : p.n[2] + p.g) : (side == 0 ? p.g : p.n[2]);
    double* a = prim + (long long)bf * p.nc + (long long)k0 * p.stride[2] + t;
    double* b = buf + (long long)bf * slab + t;
    if (unpack) *a = *b; else *b = *a;
}

// NEXT-4, peer-memory transport: the z ghost planes are PULLED straight out of the neighbours' arrays -- `below` and `above`
// are the prim arrays of the slabs below and above (same shape), on this device or on a peer whose memory is mapped
// (NVLink peer access): no pack buffer, no staging copy, one kernel.  low ghost planes <- the g highest interior planes of
// `below`, high ghost planes <- the g lowest interior planes of `above`.
__global__ void __launch_bounds__(256) halo_z_pull_kernel(const __grid_constant__ RhsParams p, double* prim,
                                                          const double* __restrict__ below, const double* __restrict__ above) {
    const long long slab = (long long)p.g * p.stride[2];
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= slab) return;
    const long long f = (long long)blockIdx.y * p.nc;   // box * 8 + field
    const int side = blockIdx.z;
    if (side == 0) prim[f + t] = below[f + (long long)p.n[2] * p.stride[2] + t];
    else prim[f + (long long)(p.n[2] + p.g) * p.stride[2] + t] = above[f + (long long)p.g * p.stride[2] + t];
}

__global__ void selftest_math_kernel(const double* __restrict__ x, double* __restrict__ y, size_t n) {
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n) return;
    const double v = x[t];
    y[t] = rcp(v);
    y[n + t] = rsqrt(v);
    y[2 * n + t] = sqrt_nn(v);
}

cudaError_t launch_prim2con(const double* prim, const double* met, long long nc, int nbox, double gamma, double* cons,
                            cudaStream_t st) {
    const dim3 grid((unsigned)((nc + 255) / 256), nbox);
    prim2con_kernel<<<grid, 256, 0, st>>>(prim, met, nc, gamma, cons);
    return cudaGetLastError();
}

cudaError_t launch_con2prim(const double* cons, const double* met, long long nc, int nbox, double gamma, double* prim,
                            unsigned long long* nfail, cudaStream_t st) {
    const dim3 grid((unsigned)((nc + 127) / 128), nbox);
    con2prim_kernel<<<grid, 128, 0, st>>>(cons, met, nc, gamma, prim, nfail);
    return cudaGetLastError();
}

cudaError_t launch_rk_axpy(const RhsParams& p, double a, const double* x, double b, double dt, const double* rhs,
                           double* y, cudaStream_t st) {
    const dim3 grid((unsigned)((p.n[0] + 127) / 128) * (unsigned)p.n[1] * (unsigned)p.n[2], p.nbox);
    rk_axpy_kernel<<<grid, 128, 0, st>>>(p, a, x, b, dt, rhs, y);
    return cudaGetLastError();
}

cudaError_t launch_rk_stage(const RhsParams& p, double a, const double* Ua, double b, const double* Ub, double h,
                            const double* L, double* Uout, double* acc, double wdt, double* prim, unsigned long long* nfail,
                            cudaStream_t st) {
    const dim3 grid((unsigned)((p.n[0] + 127) / 128) * (unsigned)p.n[1] * (unsigned)p.n[2], p.nbox);
    rk_stage_kernel<<<grid, 128, 0, st>>>(p, a, Ua, b, Ub, h, L, Uout, acc, wdt, prim, nfail);
    return cudaGetLastError();
}

cudaError_t launch_fill_ghosts(const RhsParams& p, double* prim, int bc, int dirs, cudaStream_t st) {
    const dim3 grid((unsigned)((p.nc + 255) / 256), p.nbox);
    fill_ghosts_kernel<<<grid, 256, 0, st>>>(p, prim, bc, dirs);
    return cudaGetLastError();
}

cudaError_t launch_halo_z(const RhsParams& p, double* prim, double* buf, int side, bool unpack, cudaStream_t st) {
    const long long slab = (long long)p.g * p.stride[2];
    if (slab == 0) return cudaSuccess;
    const dim3 grid((unsigned)((slab + 255) / 256), (unsigned)(p.nbox * 8));
    halo_z_kernel<<<grid, 256, 0, st>>>(p, prim, buf, side, unpack ? 1 : 0);
    return cudaGetLastError();
}

cudaError_t launch_halo_z_pull(const RhsParams& p, double* prim, const double* below, const double* above, cudaStream_t st) {
    const long long slab = (long long)p.g * p.stride[2];
    if (slab == 0) return cudaSuccess;
    const dim3 grid((unsigned)((slab + 255) / 256), (unsigned)(p.nbox * 8), 2);
    halo_z_pull_kernel<<<grid, 256, 0, st>>>(p, prim, below, above);
    return cudaGetLastError();
}

cudaError_t launch_selftest_math(const double* x, double* y, size_t n, cudaStream_t st) {
    if (n == 0) return cudaSuccess;
    selftest_math_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(x, y, n);
    return cudaGetLastError();
}

}  // namespace grx
