// grx_split.cu -- the right-hand side as TWO barrier-free kernels (steps 2-4):
//
//   rhs_z_kernel   z-direction reconstruct + HLLE + flux difference, plus the geometric sources; WRITES out.
//                  One thread per (i,j) column, marching along z: q^+ of the previous plane and the running
//                  sum of the cell being finished live in registers, so every z-face is evaluated once.
//   rhs_xy_kernel  x- and y-direction reconstruct + HLLE + flux differences; ADDS to out.
//                  One warp per 30-cell row segment (lanes 1..30 own a cell, lanes 0 and 31 are the x-halo),
//                  marching along y.  y works like z above; in x every lane reconstructs its own cell, takes
//                  q^+ of its left neighbour by warp shuffle, evaluates the face on its low side and takes the
//                  flux of its high face by shuffle from its right neighbour.
//
// No __syncthreads, no inter-warp communication: every warp runs on its own, so the FP64 pipe is kept busy
// by whichever of the SM's 16+ resident warps is ready.  The only shared memory is a
// thread-private parking area for the left side's (U, F) while the right side of a face is evaluated, which
// keeps the kernels at 128 registers without spills.
#include <cstdio>
#include <cstdlib>

#include "grx_launch.h"

namespace grx {

constexpr int ST = 128;       // threads per CTA (4 warps)
constexpr int PARK = 16;      // doubles parked per thread: U_L[8], F_L[8]
constexpr int XOWN = 30;      // cells owned by a warp of the xy kernel

struct SplitGeom {
    int ntx;   // tiles along x (z kernel: 32 cells; xy kernel: 30 cells)
    int nty;   // z kernel: groups of 4 rows
    int nch;   // chunks along the marching direction
    int len;   // chunk length
};

// HLLE flux (times `scale` = 1/dx_d) of the face between the cell at (pL, mL) and the next one along a
// direction with element stride s, from given left/right states.  The left side's U and F wait in the
// thread's parking slots while the right side is evaluated.
template <int D>
__device__ __forceinline__ void face_parked(const double* __restrict__ pL, const double* __restrict__ mL, int nc,
                                            int s, const double PL[8], const double PR[8], double gamma,
                                            double scale, volatile double* park, double Fh[8], unsigned& nfb) {
    FaceGeom m;
    face_geom_load(mL, nc, s, m);
    face_geom_complete<D>(m);
    double lmL, lpL;
    {
        double U[8], F[8];
        side_state<D>(PL, pL, nc, m, gamma, U, F, lmL, lpL, nfb);
#pragma unroll
        for (int q = 0; q < 8; ++q) { park[q * ST] = U[q]; park[(8 + q) * ST] = F[q]; }
    }
    double UR[8], FR[8], lmR, lpR;
    side_state<D>(PR, pL + s, nc, m, gamma, UR, FR, lmR, lpR, nfb);
    const double lm = fmin(0.0, fmin(lmL, lmR));
    const double lp = fmax(0.0, fmax(lpL, lpR));
    const double idl = rcp(lp - lm) * (scale * m.sg);
    const double cL = lp * idl, cR = -lm * idl, cU = lp * lm * idl;
#pragma unroll
    for (int q = 0; q < 8; ++q) Fh[q] = fma(cL, park[(8 + q) * ST], fma(cR, FR[q], cU * (UR[q] - park[q * ST])));
}

// ---- z direction + sources -----------------------------------------------------------------------------------
template <int RECON, int MINB>
__global__ void __launch_bounds__(ST, MINB) rhs_z_kernel(const __grid_constant__ RhsParams p, const SplitGeom sg) {
    extern __shared__ double park_raw[];
    const int tid = threadIdx.x, lane = tid & 31, wrp = tid >> 5;
    int t = blockIdx.x;
    const int tix = t % sg.ntx; t /= sg.ntx;
    const int tiy = t % sg.nty; t /= sg.nty;
    const int i = tix * 32 + lane, j = tiy * 4 + wrp;
    if (i >= p.n[0] || j >= p.n[1]) return;
    const int k0 = t * sg.len;
    const int nk = min(sg.len, p.n[2] - k0);
    int nc = (int)p.nc, sy = (int)p.stride[1], sz = (int)p.stride[2];
    asm volatile("" : "+r"(nc), "+r"(sy), "+r"(sz));           // per-thread copies: IMAD.WIDE addressing
    const long long c0 = (long long)blockIdx.y * p.nc;         // box offset in units of fields
    const long long cell = (i + p.g) + (long long)sy * (j + p.g) + (long long)sz * (k0 - 1 + p.g);
    const double* __restrict__ pc = p.prim + 8 * c0 + cell;
    const double* __restrict__ mc = p.met + 10 * c0 + cell;
    const double* __restrict__ kc = p.K + 6 * c0 + cell;
    double* __restrict__ oc = p.out + 8 * c0 + cell;
    volatile double* park = park_raw + tid;
    unsigned nfb = 0;
    double qpz[8], acc[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) { qpz[q] = 0.0; acc[q] = 0.0; }
    for (int kk = -1; kk <= nk; ++kk, pc += sz, mc += sz, kc += sz, oc += sz) {
        {
            double qm[8], qp[8];
            recon8s<RECON>(pc, nc, sz, qm, qp);
            if (kk >= 0) {
                double Fh[8];
                unsigned dup = 0;   // the first face of an inner chunk is the last face of the chunk below
                face_parked<2>(pc - sz, mc - sz, nc, sz, qpz, qm, p.gamma, p.idx[2], park, Fh,
                               (kk == 0 && k0 > 0) ? dup : nfb);
                if (kk >= 1) {
                    double* ob = oc - sz;
#pragma unroll
                    for (int q = 0; q < 8; ++q) ob[(long long)q * nc] = __dsub_rn(acc[q], Fh[q]);
                }
#pragma unroll
                for (int q = 0; q < 8; ++q) acc[q] = Fh[q];
            }
#pragma unroll
            for (int q = 0; q < 8; ++q) qpz[q] = qp[q];
        }
        if (kk >= 0 && kk < nk) sources_add(p, pc, mc, kc, nc, sy, sz, acc);
    }
    if (p.nfallback && nfb) atomicAdd(p.nfallback, (unsigned long long)nfb);
}

// ---- x and y directions ----------------------------------------------------------------------------------------
template <int RECON, int MINB>
__global__ void __launch_bounds__(ST, MINB) rhs_xy_kernel(const __grid_constant__ RhsParams p, const SplitGeom sg) {
    extern __shared__ double park_raw[];
    const int tid = threadIdx.x, lane = tid & 31, wrp = tid >> 5;
    long long wt = (long long)blockIdx.x * (ST / 32) + wrp;
    const int tix = (int)(wt % sg.ntx); wt /= sg.ntx;
    const int yc = (int)(wt % sg.nch); wt /= sg.nch;
    const int k = (int)wt;
    if (k >= p.n[2]) return;                                  // warp-uniform
    const int i = tix * XOWN - 1 + lane;                      // lane 0: left halo cell, lane 31: right halo cell
    const int j0 = yc * sg.len;
    const int nj = min(sg.len, p.n[1] - j0);
    const bool valid = i <= p.n[0];                            // the cell exists (interior or first ghost)
    const bool owned = lane >= 1 && lane <= XOWN && i < p.n[0];
    const bool xface = valid && lane >= 1;                     // evaluates the face on its low side
    const bool count_x = owned || (lane >= 1 && i == p.n[0]);  // a face owned by two warps is counted once
    int nc = (int)p.nc, sy = (int)p.stride[1];
    asm volatile("" : "+r"(nc), "+r"(sy));                     // per-thread copies: IMAD.WIDE addressing
    const long long c0 = (long long)blockIdx.y * p.nc;
    const long long cell = (i + p.g) + (long long)sy * (j0 - 1 + p.g) + p.stride[2] * (k + p.g);
    const double* __restrict__ pc = p.prim + 8 * c0 + cell;
    const double* __restrict__ mc = p.met + 10 * c0 + cell;
    double* __restrict__ oc = p.out + 8 * c0 + cell;
    volatile double* park = park_raw + tid;
    unsigned nfb = 0;
    double qpy[8], acc[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) { qpy[q] = 0.0; acc[q] = 0.0; }
    for (int jj = -1; jj <= nj; ++jj, pc += sy, mc += sy, oc += sy) {
        if (owned) {
            double qm[8], qp[8];
            recon8s<RECON>(pc, nc, sy, qm, qp);
            if (jj >= 0) {
                double Fh[8];
                unsigned dup = 0;
                face_parked<1>(pc - sy, mc - sy, nc, sy, qpy, qm, p.gamma, p.idx[1], park, Fh,
                               (jj == 0 && j0 > 0) ? dup : nfb);
                if (jj >= 1) {
                    double* ob = oc - sy;
#pragma unroll
                    for (int q = 0; q < 8; ++q) {
                        double* o = ob + (long long)q * nc;
                        *o = __dadd_rn(*o, __dsub_rn(acc[q], Fh[q]));
                    }
                }
#pragma unroll
                for (int q = 0; q < 8; ++q) acc[q] = Fh[q];
            }
#pragma unroll
            for (int q = 0; q < 8; ++q) qpy[q] = qp[q];
        }
        if (jj < 0 || jj >= nj) continue;                      // warp-uniform
        double qm[8], qp[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) { qm[q] = 0.0; qp[q] = 0.0; }
        if (valid) recon8s<RECON>(pc, nc, 1, qm, qp);
        double PL[8], Fh[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) { PL[q] = __shfl_up_sync(0xffffffffu, qp[q], 1); Fh[q] = 0.0; }
        if (xface) {
            unsigned dup = 0;
            face_parked<0>(pc - 1, mc - 1, nc, 1, PL, qm, p.gamma, p.idx[0], park, Fh, count_x ? nfb : dup);
        }
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const double hi = __shfl_down_sync(0xffffffffu, Fh[q], 1);
            acc[q] += __dsub_rn(Fh[q], hi);
        }
    }
    if (p.nfallback && nfb) atomicAdd(p.nfallback, (unsigned long long)nfb);
}

// ---- host side ------------------------------------------------------------------------------------------------
namespace {

// Chunks along the marching direction: enough CTAs to fill whole waves, chunks long enough to amortise the
// two one-sided steps at their ends (`ovh` = their cost in units of a full step).
void pick_chunks(long long units_per_chunk_layer, int n, int slots, double ovh, int& nch, int& len) {
    int best = 1;
    double best_eff = -1.0;
    const int maxc = (n + 7) / 8;
    for (int c = 1; c <= maxc; ++c) {
        const int l = (n + c - 1) / c;
        if ((n + l - 1) / l != c) continue;
        const double waves = (double)(units_per_chunk_layer * c) / slots;
        const double fill = waves / (double)(long long)(waves + 0.999999);
        const double eff = fill * l / (l + ovh);
        if (eff > best_eff * 1.001) { best_eff = eff; best = c; }
    }
    len = (n + best - 1) / best;
    nch = (n + len - 1) / len;
}

int sm_count() {
    static int sms = 0;
    if (sms == 0) {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess) return 148;
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) sms = 148;
    }
    return sms;
}

template <int RECON, int MINB>
cudaError_t launch_split_t(const RhsParams& p, cudaStream_t st) {
    const size_t smem = (size_t)PARK * ST * sizeof(double);
    const int slots = sm_count() * MINB;
    // z + sources
    SplitGeom gz;
    gz.ntx = (p.n[0] + 31) / 32;
    gz.nty = (p.n[1] + 3) / 4;
    pick_chunks((long long)gz.ntx * gz.nty * p.nbox, p.n[2], slots, 0.5, gz.nch, gz.len);
    rhs_z_kernel<RECON, MINB><<<dim3((unsigned)(gz.ntx * gz.nty * gz.nch), p.nbox), ST, smem, st>>>(p, gz);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    // x + y
    SplitGeom gx;
    gx.ntx = (p.n[0] + XOWN - 1) / XOWN;
    gx.nty = 0;
    const long long layer = ((long long)gx.ntx * p.n[2] + 3) / 4 * p.nbox;   // CTAs per y-chunk
    pick_chunks(layer, p.n[1], slots, 0.4, gx.nch, gx.len);
    const long long warps = (long long)gx.ntx * gx.nch * p.n[2];
    rhs_xy_kernel<RECON, MINB><<<dim3((unsigned)((warps + 3) / 4), p.nbox), ST, smem, st>>>(p, gx);
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_rhs_split(const RhsParams& p, int recon, cudaStream_t st) {
    if (recon == RECON_WENO5) return launch_split_t<RECON_WENO5, 4>(p, st);
    if (recon == RECON_MC) return launch_split_t<RECON_MC, 4>(p, st);
    return launch_split_t<RECON_MINMOD, 4>(p, st);
}

}  // namespace grx
