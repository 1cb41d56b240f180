// grx_staged.cu -- the fused right-hand side with the current plane STAGED IN SHARED MEMORY.
//
// Same decomposition as grx_fused.cu (a CTA owns a 32 x TY in-plane tile and marches along z; one warp per
// tile row plus one rim warp; every face flux of the block computed once), but at every step the CTA first
// copies the plane it is about to work on -- the 8 primitives with a 3-cell halo and the 10 metric fields
// with a 2-cell halo -- into shared memory with cp.async.  All in-plane stencil reads (x/y reconstruction,
// x/y face metric, the centre values and the x/y metric derivatives of the sources, the rim work) are then
// shared-memory loads at COMPILE-TIME offsets from one per-thread base: no address arithmetic, no L1 misses.
// Only the thread-private z stencil (z reconstruction, z face metric, z metric derivatives, K_ij) still comes
// from global memory, overlapped with the asynchronous copy.  PAPER.md l.127-132; DESIGN.md "Kernels".
#include <cstdio>
#include <cstdlib>

#include "grx_launch.h"

namespace grx {

namespace {

constexpr int TX = 32;
constexpr int PH = 3, MH = 2;          // halo of the staged primitives / metric
constexpr int PX = TX + 2 * PH;        // 38 columns
constexpr int MX = TX + 2 * MH;        // 36 columns

template <int TY>
struct Stage {
    double P[8][TY + 2 * PH][PX];      // primitives of the current plane
    double M[10][TY + 2 * MH][MX];     // metric of the current plane
    double Q[8][TY + 1][TX + 1];       // exchange: q^+ of the low neighbour
    double F[8][TY + 1][TX + 1];       // exchange: face fluxes
};

struct StagedGeom {
    int ntx, nty, nzc, tz;
};

__device__ __forceinline__ void cp_async8(double* dst_shared, const double* src_global) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(dst_shared);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(src_global) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// Reconstruct the 8 primitives of the cell at ps (field 0) along a direction with compile-time stride S;
// FS = element stride between fields.
template <int RECON, int S, int FS>
__device__ __forceinline__ void recon8_sm(const double* ps, double qm[8], double qp[8]) {
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        const double* f = ps + q * FS;
        double a = 0.0, e = 0.0;
        if (RECON == RECON_WENO5) { a = f[-2 * S]; e = f[2 * S]; }
        recon_cell<RECON>(a, f[-S], f[0], f[S], e, qm[q], qp[q]);
    }
}

// HLLE flux (times scale) of the face between the cell at msL and the next one along S, metric from shared
// memory; cenL points at field 0 of the left cell in GLOBAL memory (first-order fallback, R5).
template <int D, int S, int FS>
__device__ __forceinline__ void face8_sm(const double* msL, const double* __restrict__ cenL, int nc, int sg,
                                         const double PL[8], const double PR[8], double gamma, double scale,
                                         double Fh[8], unsigned& nfb) {
    FaceGeom m;
    {
        double v[10];
#pragma unroll
        for (int f = 0; f < 10; ++f) v[f] = 0.5 * (msL[f * FS] + msL[f * FS + S]);
        m.alp = v[0];
#pragma unroll
        for (int a = 0; a < 3; ++a) m.beta[a] = v[1 + a];
#pragma unroll
        for (int c = 0; c < 6; ++c) m.g[c] = v[4 + c];
    }
    face_flux<D>(m, PL, PR, cenL, cenL + sg, nc, gamma, Fh, nfb, scale);
}

template <int S, int FS>
__device__ __forceinline__ void dmetric_sm(const double* ms, double d[10]) {
#pragma unroll
    for (int f = 0; f < 10; ++f) d[f] = d4raw(ms[f * FS - 2 * S], ms[f * FS - S], ms[f * FS + S], ms[f * FS + 2 * S]);
}

// Asynchronous copy of one plane of the tile (with halos) into shared memory; every warp of the CTA takes
// every (TY+1)-th row.  pg/mg: field 0 at the tile origin of that plane; (ax0, ay0): array indices of the origin.
template <int TY>
__device__ __forceinline__ void stage_plane(Stage<TY>& S, const double* __restrict__ pg, const double* __restrict__ mg,
                                            int nc, int sy, int ax0, int ay0, int Nx, int Ny, int warp, int lane) {
    constexpr int NW = TY + 1;
    constexpr int PR = TY + 2 * PH, MR = TY + 2 * MH;
    for (int t = warp; t < 8 * PR; t += NW) {
        const int f = t / PR, r = t - f * PR;
        const int ay = ay0 + r - PH;
        if (ay < 0 || ay >= Ny) continue;
        const double* src = pg + (long long)f * nc + (r - PH) * sy - PH + lane;
        double* dst = &S.P[f][r][lane];
        const int ax = ax0 - PH + lane;
        if (ax >= 0 && ax < Nx) cp_async8(dst, src);
        if (lane < PX - 32 && ax + 32 < Nx) cp_async8(dst + 32, src + 32);
    }
    for (int t = warp; t < 10 * MR; t += NW) {
        const int f = t / MR, r = t - f * MR;
        const int ay = ay0 + r - MH;
        if (ay < 0 || ay >= Ny) continue;
        const double* src = mg + (long long)f * nc + (r - MH) * sy - MH + lane;
        double* dst = &S.M[f][r][lane];
        const int ax = ax0 - MH + lane;
        if (ax >= 0 && ax < Nx) cp_async8(dst, src);
        if (lane < MX - 32 && ax + 32 < Nx) cp_async8(dst + 32, src + 32);
    }
}

// Geometric sources of the thread's cell: centre values and x/y metric derivatives from the staged plane,
// z derivatives and K_ij from global memory.
template <int TY>
__device__ __forceinline__ void sources_staged(const RhsParams& p, const double* ps, const double* ms,
                                               const double* __restrict__ mc, const double* __restrict__ kc, int nc,
                                               int sz, double acc[8]) {
    constexpr int PFS = (TY + 2 * PH) * PX, MFS = (TY + 2 * MH) * MX;
    SrcState s;
    {
        double P[8], m[10];
#pragma unroll
        for (int q = 0; q < 8; ++q) P[q] = ps[q * PFS];
#pragma unroll
        for (int f = 0; f < 10; ++f) m[f] = ms[f * MFS];
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
    dmetric_sm<1, MFS>(ms, d);
    acc[1] += sources_dir(s, 0, d, p.idx[0] * (1.0 / 12.0), st);
    dmetric_sm<MX, MFS>(ms, d);
    acc[2] += sources_dir(s, 1, d, p.idx[1] * (1.0 / 12.0), st);
    dmetric(mc, nc, sz, d);
    acc[3] += sources_dir(s, 2, d, p.idx[2] * (1.0 / 12.0), st);
    acc[4] += st;
}

}  // namespace

namespace {

template <int RECON, int TY>
__global__ void __launch_bounds__((TY + 1) * 32, 1)
rhs_staged_kernel(const __grid_constant__ RhsParams p, const StagedGeom tg) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Stage<TY>& S = *reinterpret_cast<Stage<TY>*>(smem_raw);
    constexpr int PFS = (TY + 2 * PH) * PX, MFS = (TY + 2 * MH) * MX;

    int t = blockIdx.x;
    const int tix = t % tg.ntx; t /= tg.ntx;
    const int tiy = t % tg.nty; t /= tg.nty;
    const int X0 = tix * TX, Y0 = tiy * TY, k0 = t * tg.tz;
    const int txe = min(TX, p.n[0] - X0), tye = min(TY, p.n[1] - Y0);
    const int nk = min(tg.tz, p.n[2] - k0);       // planes owned by this CTA
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    const int nc = (int)p.nc, sy = (int)p.stride[1], sz = (int)p.stride[2];
    const long long c0 = (long long)blockIdx.y * p.nc;
    const long long cell0 = (X0 + p.g) + (long long)sy * (Y0 + p.g) + (long long)sz * (k0 - 1 + p.g);
    const double gamma = p.gamma;
    const int ax0 = X0 + p.g, ay0 = Y0 + p.g;
    // tile origin of the plane being staged (plane k0 first)
    const double* __restrict__ pg = p.prim + 8 * c0 + cell0 + sz;
    const double* __restrict__ mg = p.met + 10 * c0 + cell0 + sz;
    unsigned nfb = 0;

    if (warp < TY) {
        // ------------------------------------------------ regular warp: one cell column per thread
        const bool active = (lane < txe) && (warp < tye);
        const int off = lane + sy * warp;
        const double* __restrict__ pc = p.prim + 8 * c0 + cell0 + off;     // own column, plane k0-1
        const double* __restrict__ mc = p.met + 10 * c0 + cell0 + off;
        const double* __restrict__ kc = p.K + 6 * c0 + cell0 + off;
        double* __restrict__ oc = p.out + 8 * c0 + cell0 + off;
        const double* ps = &S.P[0][warp + PH][lane + PH];
        const double* ms = &S.M[0][warp + MH][lane + MH];
        double qpz[8], acc[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) { qpz[q] = 0.0; acc[q] = 0.0; }
        for (int kk = -1; kk <= nk; ++kk, pc += sz, mc += sz, kc += sz, oc += sz) {
            const bool inplane = (kk >= 0 && kk < nk);   // uniform over the CTA
            if (inplane) stage_plane<TY>(S, pg, mg, nc, sy, ax0, ay0, p.N[0], p.N[1], warp, lane);
            if (active) {
                // z (global memory, overlaps the asynchronous copy): reconstruct this cell, close the face
                // below it, finish the cell below
                double qm[8], qp[8];
                recon8s<RECON>(pc, nc, sz, qm, qp);
                if (kk >= 0) {
                    double Fh[8];
                    unsigned dup = 0;   // the first face of an inner chunk is the last face of the chunk below
                    face8s<2>(pc - sz, mc - sz, nc, sz, qpz, qm, gamma, p.idx[2], Fh, (kk == 0 && k0 > 0) ? dup : nfb);
                    if (kk >= 1) {
                        double* ob = oc - sz;
#pragma unroll
                        for (int q = 0; q < 8; ++q, ob += nc) *ob = __dsub_rn(acc[q], Fh[q]);
                    }
#pragma unroll
                    for (int q = 0; q < 8; ++q) acc[q] = Fh[q];
                }
#pragma unroll
                for (int q = 0; q < 8; ++q) qpz[q] = qp[q];
            }
            if (!inplane) continue;
            pg += sz; mg += sz;
            cp_async_wait_all();
            __syncthreads();                              // the plane has landed
            // x
            double qm[8];
            if (active) {
                double qp[8];
                recon8_sm<RECON, 1, PFS>(ps, qm, qp);
#pragma unroll
                for (int q = 0; q < 8; ++q) S.Q[q][warp][lane + 1] = qp[q];
            }
            __syncthreads();
            if (active) {
                double PL[8], Fh[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) PL[q] = S.Q[q][warp][lane];
                face8_sm<0, 1, MFS>(ms - 1, pc - 1, nc, 1, PL, qm, gamma, p.idx[0], Fh, nfb);
#pragma unroll
                for (int q = 0; q < 8; ++q) S.F[q][warp][lane] = Fh[q];
            }
            __syncthreads();
            // y
            if (active) {
#pragma unroll
                for (int q = 0; q < 8; ++q) acc[q] += __dsub_rn(S.F[q][warp][lane], S.F[q][warp][lane + 1]);
                double qp[8];
                recon8_sm<RECON, PX, PFS>(ps, qm, qp);
#pragma unroll
                for (int q = 0; q < 8; ++q) S.Q[q][warp + 1][lane] = qp[q];
            }
            __syncthreads();
            if (active) {
                double PL[8], Fh[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) PL[q] = S.Q[q][warp][lane];
                face8_sm<1, MX, MFS>(ms - MX, pc - sy, nc, sy, PL, qm, gamma, p.idx[1], Fh, nfb);
#pragma unroll
                for (int q = 0; q < 8; ++q) S.F[q][warp][lane] = Fh[q];
                sources_staged<TY>(p, ps, ms, mc, kc, nc, sz, acc);
            }
            __syncthreads();                              // fluxes published; the staged plane is free again
            if (active) {
#pragma unroll
                for (int q = 0; q < 8; ++q) acc[q] += __dsub_rn(S.F[q][warp][lane], S.F[q][warp + 1][lane]);
            }
        }
    } else {
        // ------------------------------------------------ rim warp: the tile's edge work, all from the staged plane
        // x-rim: lane l < tye          -> cell (X0-1,   Y0+l): its q^+ feeds the first face of row l
        //        lane TY + l, l < tye  -> cell (X0+txe, Y0+l): its q^- and the last face of row l
        // y-rim: lane l < txe          -> cell (X0+l, Y0-1) [q^+] and cell (X0+l, Y0+tye) [q^-, last face of column l]
        const bool xl = lane < tye;
        const bool xr = (TY <= 16) && lane >= TY && (lane - TY) < tye;
        const int xrow = xl ? lane : lane - TY;
        const bool ycol = lane < txe;
        // a rim face is the first face of the next tile too: only the block's last faces are counted here
        const bool count_x = (X0 + txe == p.n[0]), count_y = (Y0 + tye == p.n[1]);
        unsigned dup = 0;
        const int xcol = xl ? -1 : txe;                                   // this lane's x-rim cell (tile coordinates)
        const double* psx = &S.P[0][xrow + PH][xcol + PH];
        const double* msx = &S.M[0][xrow + MH][xcol + MH];
        const double* psb = &S.P[0][PH - 1][lane + PH];                   // bottom y-rim cell
        const double* pst = &S.P[0][PH + tye][lane + PH];                 // top y-rim cell
        const double* mst = &S.M[0][MH + tye][lane + MH];
        // global pointers to the left cells of the two rim faces (first-order fallback only)
        const double* __restrict__ gx = p.prim + 8 * c0 + cell0 + sz + sy * xrow + xcol - 1;
        const double* __restrict__ gy = p.prim + 8 * c0 + cell0 + sz + lane + sy * (tye - 1);
        for (int kk = 0; kk < nk; ++kk, pg += sz, mg += sz, gx += sz, gy += sz) {
            stage_plane<TY>(S, pg, mg, nc, sy, ax0, ay0, p.N[0], p.N[1], warp, lane);
            cp_async_wait_all();
            __syncthreads();                              // the plane has landed
            double yb_qp[8], yt_qm[8], xr_qm[8];
            if (ycol) {
                double tmp[8];
                recon8_sm<RECON, PX, PFS>(psb, tmp, yb_qp);
                recon8_sm<RECON, PX, PFS>(pst, yt_qm, tmp);
            }
            if (xl || xr) {
                double qm[8], qp[8];
                recon8_sm<RECON, 1, PFS>(psx, qm, qp);
                if (xl) {
#pragma unroll
                    for (int q = 0; q < 8; ++q) S.Q[q][xrow][0] = qp[q];
                }
#pragma unroll
                for (int q = 0; q < 8; ++q) xr_qm[q] = qm[q];
            }
            __syncthreads();
            if (xr) {
                double PL[8], Fh[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) PL[q] = S.Q[q][xrow][txe];
                face8_sm<0, 1, MFS>(msx - 1, gx, nc, 1, PL, xr_qm, gamma, p.idx[0], Fh, count_x ? nfb : dup);
#pragma unroll
                for (int q = 0; q < 8; ++q) S.F[q][xrow][txe] = Fh[q];
            }
            __syncthreads();
            if (ycol) {
#pragma unroll
                for (int q = 0; q < 8; ++q) S.Q[q][0][lane] = yb_qp[q];
            }
            __syncthreads();
            if (ycol) {
                double PL[8], Fh[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) PL[q] = S.Q[q][tye][lane];
                face8_sm<1, MX, MFS>(mst - MX, gy, nc, sy, PL, yt_qm, gamma, p.idx[1], Fh, count_y ? nfb : dup);
#pragma unroll
                for (int q = 0; q < 8; ++q) S.F[q][tye][lane] = Fh[q];
            }
            __syncthreads();
        }
    }
    if (p.nfallback && nfb) atomicAdd(p.nfallback, (unsigned long long)nfb);
}

// z-chunking: enough CTAs to fill the machine in whole waves, chunks long enough to amortise the two
// one-sided plane steps at their ends.
StagedGeom make_tiles(const RhsParams& p, int ty, int slots) {
    StagedGeom tg;
    tg.ntx = (p.n[0] + TX - 1) / TX;
    tg.nty = (p.n[1] + ty - 1) / ty;
    const long long inplane = (long long)tg.ntx * tg.nty * p.nbox;
    int best = 1;
    double best_eff = -1.0;
    const int maxc = (p.n[2] + 7) / 8;
    for (int nzc = 1; nzc <= maxc; ++nzc) {
        const int tz = (p.n[2] + nzc - 1) / nzc;
        if ((p.n[2] + tz - 1) / tz != nzc) continue;
        const double waves = (double)(inplane * nzc) / slots;
        const double fill = waves / (double)(long long)(waves + 0.999999);
        const double eff = fill * tz / (tz + 0.45);
        if (eff > best_eff * 1.001) { best_eff = eff; best = nzc; }
    }
    tg.tz = (p.n[2] + best - 1) / best;
    tg.nzc = (p.n[2] + tg.tz - 1) / tg.tz;
    return tg;
}

template <int RECON, int TY>
cudaError_t launch_staged_t(const RhsParams& p, cudaStream_t st) {
    static int sms = 0;
    if (sms == 0) {
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return e;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return e;
    }
    const size_t smem = sizeof(Stage<TY>);
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(rhs_staged_kernel<RECON, TY>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)smem);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    const StagedGeom tg = make_tiles(p, TY, sms);
    const dim3 grid((unsigned)(tg.ntx * tg.nty * tg.nzc), p.nbox);
    rhs_staged_kernel<RECON, TY><<<grid, (TY + 1) * 32, smem, st>>>(p, tg);
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_rhs_staged(const RhsParams& p, int recon, cudaStream_t st) {
    if (recon == RECON_WENO5) return launch_staged_t<RECON_WENO5, 7>(p, st);
    if (recon == RECON_MC) return launch_staged_t<RECON_MC, 7>(p, st);
    return launch_staged_t<RECON_MINMOD, 7>(p, st);
}

}  // namespace grx
