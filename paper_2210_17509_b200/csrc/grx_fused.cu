// grx_fused.cu -- the round-1 kernel, kept as the path for the shapes the TMA kernel (grx_tma.cu) cannot take (odd
// Nx, arrays that are not 16-byte aligned): reconstruct + HLLE + flux divergence in all three directions and the
// geometric sources in ONE pass over the block (steps 2-4), every face flux computed exactly
// once, all operands read through L1 with __ldg.
//
// Decomposition:
//   * A CTA owns an in-plane tile of TX x TY cells (TX = 32 = one warp along x, TY warps along y) and
//     MARCHES along z through a chunk of the block, one plane per step.
//   * z-direction: each thread reconstructs its own cell along z and keeps q^+ of the previous plane in
//     registers, so the face k-1/2 is evaluated once, by the thread that owns the column; the finished
//     right-hand side of cell k-1 is stored at step k.
//   * x- and y-direction: every thread reconstructs its own cell, publishes q^+ in shared memory, evaluates
//     the face on its low side (from its neighbour's q^+ and its own q^-), publishes the flux, and takes the
//     flux of its high face from its neighbour.  The faces and one-sided reconstructions on the rim of the
//     tile belong to one extra "rim warp" per CTA, whose lanes run along the tile edges.
//   * Sources: metric derivatives and the 3+1 source terms per cell, added to the same accumulators.
// Global loads go through L1/L2 (__ldg); lanes run along x, so every load is a contiguous 256 B row segment.
#include "grx_launch.h"
#include "grx_vertex.cuh"

namespace grx {

constexpr int TX = 32;

struct TileGeom {
    int ntx, nty, nzc, tz;   // tiles along x, y; z-chunks and their length
    int pf;                  // software prefetch mode (tuning knob)
};

__device__ __forceinline__ void prefetch_l1(const double* a) { asm volatile("prefetch.global.L1 [%0];" ::"l"(a)); }
__device__ __forceinline__ void prefetch_l2(const double* a) { asm volatile("prefetch.global.L2 [%0];" ::"l"(a)); }

// shared-memory exchange buffer: [8 fields][TY+1 rows][TX+1 columns]
template <int TY>
struct Exch {
    double v[8][TY + 1][TX + 1];
};

// Reconstruct the 8 primitives of cell c along a direction with element stride s.
template <int RECON>
__device__ __forceinline__ void recon8(const double* __restrict__ prim, long long nc, long long c, long long s,
                                       double qm[8], double qp[8]) {
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        const double* f = prim + q * nc + c;
        double a = 0.0, e = 0.0;
        if (RECON == RECON_WENO5) { a = ldg(f - 2 * s); e = ldg(f + 2 * s); }
        recon_cell<RECON>(a, ldg(f - s), ldg(f), ldg(f + s), e, qm[q], qp[q]);
    }
}

// HLLE flux of the face between cells iL and iR = iL + s from given left/right states.  VERTEX (NEXT-3, reading R31): met
// is a vertex array and the face metric is the mean of the 4 vertices of the low D-face of cell iR, whose low-corner
// vertex is vR.
template <int D, bool VERTEX>
__device__ __forceinline__ void face8(const double* __restrict__ prim, const double* __restrict__ met, long long nc,
                                      const VStride& vs, long long iL, long long iR, long long vR, double PL[8],
                                      double PR[8], double gamma, double Fh[8], unsigned& nfb) {
    FaceGeom m;
    if (VERTEX) {
        face_geom_vertex<D>(met, vs, vR, m);
    } else {
        m.alp = 0.5 * (ldg(met + iL) + ldg(met + iR));
#pragma unroll
        for (int a = 0; a < 3; ++a) m.beta[a] = 0.5 * (ldg(met + (1 + a) * nc + iL) + ldg(met + (1 + a) * nc + iR));
#pragma unroll
        for (int c = 0; c < 6; ++c) m.g[c] = 0.5 * (ldg(met + (4 + c) * nc + iL) + ldg(met + (4 + c) * nc + iR));
    }
    face_flux<D>(m, PL, PR, prim + iL, prim + iR, nc, gamma, Fh, nfb);
}

// The running sum of the cell being finished also waits in thread-private shared memory between the points
// where it is updated (4 per step): with the z carry that keeps 32 registers free during the face evaluations.
#define GRX_ACC_LOAD _Pragma("unroll") for (int q_ = 0; q_ < 8; ++q_) acc[q_] = apark[q_ * ((TY + 1) * 32)];
#define GRX_ACC_STORE _Pragma("unroll") for (int q_ = 0; q_ < 8; ++q_) apark[q_ * ((TY + 1) * 32)] = acc[q_];
constexpr int PARK_SLOTS = 16;   // doubles per thread: z carry q^+[8], running sum[8]

template <int RECON, int TY, int MINB, bool VERTEX>
__global__ void __launch_bounds__((TY + 1) * 32, MINB)
rhs_fused_kernel(const __grid_constant__ RhsParams p, const TileGeom tg, const VStride vs) {
    extern __shared__ double smem_raw[];
    Exch<TY>& Qb = *reinterpret_cast<Exch<TY>*>(smem_raw);
    Exch<TY>& Fb = *reinterpret_cast<Exch<TY>*>(smem_raw + sizeof(Exch<TY>) / sizeof(double));

    int t = blockIdx.x;
    const int tix = t % tg.ntx; t /= tg.ntx;
    const int tiy = t % tg.nty; t /= tg.nty;
    const int zc = t;
    const int box = blockIdx.y;
    const int X0 = tix * TX, Y0 = tiy * TY, k0 = zc * tg.tz;
    const int txe = min(TX, p.n[0] - X0), tye = min(TY, p.n[1] - Y0);
    const int nk = min(tg.tz, p.n[2] - k0);       // planes owned by this CTA
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    const double* __restrict__ prim = p.prim + (long long)box * 8 * p.nc;
    const double* __restrict__ met = p.met + (long long)box * 10 * (VERTEX ? vs.nv : p.nc);
    const double* __restrict__ Kf = p.K + (long long)box * 6 * (VERTEX ? vs.nv : p.nc);
    double* __restrict__ out = p.out + (long long)box * 8 * p.nc;
    const long long nc = p.nc, sy = p.stride[1], sz = p.stride[2];
    const double gamma = p.gamma;
    const long long cbase = (X0 + p.g) + sy * (Y0 + p.g) + sz * (k0 - 1 + p.g);   // tile origin, plane k0-1
    const long long vbase = (X0 + p.g) + vs.s[1] * (Y0 + p.g) + vs.s[2] * (k0 - 1 + p.g);   // ... and its low-corner vertex
    unsigned nfb = 0;
    volatile double* apark = smem_raw + 2 * sizeof(Exch<TY>) / sizeof(double) + 8 * (TY + 1) * 32 + threadIdx.x;

    if (warp < TY) {
        // ------------------------------------------------ regular warp: one cell column per thread
        const bool active = (lane < txe) && (warp < tye);
        long long c = cbase + lane + sy * warp;
        long long v = vbase + lane + vs.s[1] * warp;      // low-corner vertex of the cell (VERTEX only)
        // q^+ of the previous plane waits in a thread-private shared-memory slot between two z faces (it is
        // needed once per step; parking it frees 16 registers during the x, y and source phases)
        volatile double* zpark = smem_raw + 2 * sizeof(Exch<TY>) / sizeof(double) + threadIdx.x;
        constexpr int ZS = (TY + 1) * 32;
        double acc[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) acc[q] = 0.0;
        for (int kk = -1; kk <= nk; ++kk, c += sz, v += vs.s[2]) {
            if (!VERTEX && tg.pf && active && kk < nk) {
                // first touches of this column: metric plane k+2 (z derivative at the end of THIS step), K_ij of
                // this plane, primitives of plane k+3 (z stencil at the top of the next step)
                if (tg.pf & 1) {
#pragma unroll
                    for (int f = 0; f < 10; ++f) prefetch_l1(met + f * nc + c + 2 * sz);
#pragma unroll
                    for (int f = 0; f < 6; ++f) prefetch_l1(Kf + f * nc + c);
                }
                // plane k+3 of the primitives is read by WENO5 at the next step; TVD never reads it, and at the last
                // step of the last chunk it would lie past the field when nghost = 2
                if ((tg.pf & 2) && RECON == RECON_WENO5 && kk + 1 < nk) {
#pragma unroll
                    for (int q = 0; q < 8; ++q) prefetch_l1(prim + q * nc + c + 3 * sz);
                }
            }
            if (active) {
                // z: reconstruct this cell, close the face below it, finish the cell below
                double qm[8], qp[8];
                recon8<RECON>(prim, nc, c, sz, qm, qp);
                if (kk >= 0) {
                    double Fh[8];
                    // the first face of an inner chunk is also the last face of the chunk below: count once
                    unsigned dup = 0;
                    double qpz[8];
#pragma unroll
                    for (int q = 0; q < 8; ++q) qpz[q] = zpark[q * ZS];
                    face8<2, VERTEX>(prim, met, nc, vs, c - sz, c, v, qpz, qm, gamma, Fh, (kk == 0 && k0 > 0) ? dup : nfb);
                    // F/dz is rounded once and used with both signs, so a uniform state cancels exactly
#pragma unroll
                    for (int q = 0; q < 8; ++q) Fh[q] = __dmul_rn(Fh[q], p.idx[2]);
                    if (kk >= 1) {
                        GRX_ACC_LOAD
#pragma unroll
                        for (int q = 0; q < 8; ++q) out[q * nc + c - sz] = __dsub_rn(acc[q], Fh[q]);
                    }
#pragma unroll
                    for (int q = 0; q < 8; ++q) acc[q] = Fh[q];
                    GRX_ACC_STORE
                }
#pragma unroll
                for (int q = 0; q < 8; ++q) zpark[q * ZS] = qp[q];
            }
            if (kk < 0 || kk >= nk) continue;   // uniform over the CTA
            // x
            double qm[8];
            if (active) {
                double qp[8];
                recon8<RECON>(prim, nc, c, 1, qm, qp);
#pragma unroll
                for (int q = 0; q < 8; ++q) Qb.v[q][warp][lane + 1] = qp[q];
            }
            __syncthreads();
            if (active) {
                double PL[8], Fh[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) PL[q] = Qb.v[q][warp][lane];
                face8<0, VERTEX>(prim, met, nc, vs, c - 1, c, v, PL, qm, gamma, Fh, nfb);
#pragma unroll
                for (int q = 0; q < 8; ++q) Fb.v[q][warp][lane] = Fh[q];
            }
            __syncthreads();
            // y
            if (active) {
                GRX_ACC_LOAD
#pragma unroll
                for (int q = 0; q < 8; ++q) acc[q] = fma(Fb.v[q][warp][lane] - Fb.v[q][warp][lane + 1], p.idx[0], acc[q]);
                GRX_ACC_STORE
                double qp[8];
                recon8<RECON>(prim, nc, c, sy, qm, qp);
#pragma unroll
                for (int q = 0; q < 8; ++q) Qb.v[q][warp + 1][lane] = qp[q];
            }
            __syncthreads();
            if (active) {
                double PL[8], Fh[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) PL[q] = Qb.v[q][warp][lane];
                face8<1, VERTEX>(prim, met, nc, vs, c - sy, c, v, PL, qm, gamma, Fh, nfb);
#pragma unroll
                for (int q = 0; q < 8; ++q) Fb.v[q][warp][lane] = Fh[q];
            }
            __syncthreads();
            if (active) {
                GRX_ACC_LOAD
#pragma unroll
                for (int q = 0; q < 8; ++q) acc[q] = fma(Fb.v[q][warp][lane] - Fb.v[q][warp + 1][lane], p.idx[1], acc[q]);
                double s1, s2, s3, s4;
                if (VERTEX) sources_from_vertices(p, vs, prim, met, Kf, c, v, s1, s2, s3, s4);
                else sources_from_global(p, prim, met, Kf, c, s1, s2, s3, s4);
                acc[1] += s1; acc[2] += s2; acc[3] += s3; acc[4] += s4;
                GRX_ACC_STORE
            }
        }
    } else {
        // ------------------------------------------------ rim warp: the tile's edge work
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
        for (int kk = 0; kk < nk; ++kk) {
            const long long cp = cbase + sz * (kk + 1);   // tile origin in plane k0+kk
            const long long vp = vbase + vs.s[2] * (kk + 1);
            double yb_qp[8], yt_qm[8], xr_qm[8];
            long long cxr = 0, cyt = 0;
            if (ycol) {
                double tmp[8];
                recon8<RECON>(prim, nc, cp + lane - sy, sy, tmp, yb_qp);
                cyt = cp + lane + sy * tye;
                recon8<RECON>(prim, nc, cyt, sy, yt_qm, tmp);
            }
            if (xl || xr) {
                double qm[8], qp[8];
                cxr = cp + sy * xrow + (xl ? -1 : txe);
                recon8<RECON>(prim, nc, cxr, 1, qm, qp);
                if (xl) {
#pragma unroll
                    for (int q = 0; q < 8; ++q) Qb.v[q][xrow][0] = qp[q];
                }
#pragma unroll
                for (int q = 0; q < 8; ++q) xr_qm[q] = qm[q];
            }
            __syncthreads();
            if (xr) {
                double PL[8], Fh[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) PL[q] = Qb.v[q][xrow][txe];
                face8<0, VERTEX>(prim, met, nc, vs, cxr - 1, cxr, vp + vs.s[1] * xrow + txe, PL, xr_qm, gamma, Fh,
                                 count_x ? nfb : dup);
#pragma unroll
                for (int q = 0; q < 8; ++q) Fb.v[q][xrow][txe] = Fh[q];
            }
            __syncthreads();
            if (ycol) {
#pragma unroll
                for (int q = 0; q < 8; ++q) Qb.v[q][0][lane] = yb_qp[q];
            }
            __syncthreads();
            if (ycol) {
                double PL[8], Fh[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) PL[q] = Qb.v[q][tye][lane];
                face8<1, VERTEX>(prim, met, nc, vs, cyt - sy, cyt, vp + lane + vs.s[1] * tye, PL, yt_qm, gamma, Fh,
                                 count_y ? nfb : dup);
#pragma unroll
                for (int q = 0; q < 8; ++q) Fb.v[q][tye][lane] = Fh[q];
            }
            __syncthreads();
        }
    }
    if (p.nfallback && nfb) atomicAdd(p.nfallback, (unsigned long long)nfb);
}

// ---- host side ------------------------------------------------------------------------------------------------
namespace {

// z-chunking: enough CTAs to fill the machine a few times over, chunks long enough to amortise the two
// one-sided plane steps at their ends.
TileGeom make_tiles(const RhsParams& p, int ty, int slots, double* eff_out = nullptr) {
    TileGeom tg;
    tg.ntx = (p.n[0] + TX - 1) / TX;
    tg.nty = (p.n[1] + ty - 1) / ty;
    const long long inplane = (long long)tg.ntx * tg.nty * p.nbox;
    int best = 1;
    double best_eff = -1.0;
    const int maxc = (p.n[2] + 7) / 8;
    for (int nzc = 1; nzc <= maxc; ++nzc) {
        const int tz = (p.n[2] + nzc - 1) / nzc;
        const int real = (p.n[2] + tz - 1) / tz;
        if (real != nzc) continue;
        const double waves = (double)(inplane * nzc) / slots;
        const double fill = waves / (double)(long long)(waves + 0.999999);
        const double eff = fill * tz / (tz + 0.45);
        if (eff > best_eff * 1.001) { best_eff = eff; best = nzc; }
    }
    tg.tz = (p.n[2] + best - 1) / best;
    tg.nzc = (p.n[2] + tg.tz - 1) / tg.tz;
    tg.pf = 3;   // software prefetch of the first-touch lines (profiles/r1_variants.md)
    if (eff_out) *eff_out = best_eff * p.n[1] / ((double)tg.nty * ty);
    return tg;
}

// The SM count and the shared-memory opt-in are per device: both are asked / set once per device and remembered
// (grx_launch.h; lock-free, so the library still works with several devices and from several host threads).
template <int RECON, int TY, int MINB, bool VERTEX>
cudaError_t launch_one(const RhsParams& p, cudaStream_t st) {
    int dev = 0, sms = 0;
    cudaError_t e = current_device_sms(&dev, &sms);
    if (e != cudaSuccess) return e;
    const size_t smem = 2 * sizeof(Exch<TY>) + PARK_SLOTS * (TY + 1) * 32 * sizeof(double);
    static std::atomic<unsigned long long> smem_set{0};   // per instantiation: devices on which the attribute is set
    e = set_max_dynamic_smem_once(rhs_fused_kernel<RECON, TY, MINB, VERTEX>, dev, smem, smem_set);
    if (e != cudaSuccess) return e;
    const TileGeom tg = make_tiles(p, TY, sms * MINB);
    const dim3 grid((unsigned)(tg.ntx * tg.nty * tg.nzc), p.nbox);
    rhs_fused_kernel<RECON, TY, MINB, VERTEX><<<grid, (TY + 1) * 32, smem, st>>>(p, tg, vstride(p));
    return cudaGetLastError();
}

// 11 rows (12 warps per SM at 168 registers); blocks that are thin along z have too few plane steps per CTA to
// amortise the taller tile and take the 7-row one (8 warps, 255 registers).
// tile_nz: the plane count the tile is chosen for -- that of the whole block when p is a z range of it, so that every
// plane carries the bits of the whole-block call (the two instantiations round differently).
template <int RECON, bool VERTEX>
cudaError_t dispatch(const RhsParams& p, int tile_nz, cudaStream_t st) {
    if (tile_nz < 8) return launch_one<RECON, 7, 1, VERTEX>(p, st);
    return launch_one<RECON, 11, 1, VERTEX>(p, st);
}

}  // namespace

double fused_tile_efficiency(const RhsParams& p, int sms) {
    double eff = 0.0;
    make_tiles(p, p.n[2] < 8 ? 7 : 11, sms, &eff);
    return eff;
}

cudaError_t launch_rhs_fused(const RhsParams& p, int recon, cudaStream_t st, int tile_nz) {
    if (tile_nz <= 0) tile_nz = p.n[2];
    if (recon == RECON_WENO5) return dispatch<RECON_WENO5, false>(p, tile_nz, st);
    if (recon == RECON_MC) return dispatch<RECON_MC, false>(p, tile_nz, st);
    return dispatch<RECON_MINMOD, false>(p, tile_nz, st);
}

// NEXT-3: the same kernel with p.met / p.K pointing at vertex arrays (reading R31)
cudaError_t launch_rhs_fused_vertex(const RhsParams& p, int recon, cudaStream_t st) {
    if (recon == RECON_WENO5) return dispatch<RECON_WENO5, true>(p, p.n[2], st);
    if (recon == RECON_MC) return dispatch<RECON_MC, true>(p, p.n[2], st);
    return dispatch<RECON_MINMOD, true>(p, p.n[2], st);
}

}  // namespace grx
