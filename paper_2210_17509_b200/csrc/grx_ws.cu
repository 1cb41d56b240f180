// grx_ws.cu -- warp-specialised variant of the fused right-hand side (experimental, GRX_VARIANT_WS).
//
// Same tile/march/rim structure as grx_fused.cu, plus ONE EXTRA WARP GROUP (4 warps) per CTA that evaluates the
// geometric sources (a8 + a9: 144 loads and ~290 FP64 operations per cell, the most load-heavy part of a step)
// and hands S_x, S_y, S_z, S_tau to the flux warps through shared memory.  The flux warps take 176 registers,
// the helper group 152 (setmaxnreg; 2 x 176 + 152 = 504 = 3 x 168, the launch allocation), so an SM holds 3 warps per scheduler instead of 2 and the
// helpers' load phases overlap the flux warps' FP64 phases.  Named barriers: 1 = the 8 flux warps;
// 2,3 = "sources of buffer b published"; 4,5 = "buffer b consumed".
#include <cstdio>
#include <cstdlib>

#include "grx_launch.h"

namespace grx {

namespace {

constexpr int WS_MAIN = 256, WS_ALL = 384;
__device__ __forceinline__ void bar_main() { asm volatile("bar.sync 1, 256;" ::: "memory"); }
__device__ __forceinline__ void bar_named_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void bar_named_arrive(int id, int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }

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

// HLLE flux of the face between cells iL and iR = iL + s from given left/right states.
template <int D>
__device__ __forceinline__ void face8(const double* __restrict__ prim, const double* __restrict__ met, long long nc,
                                      long long iL, long long iR, const double PL[8], const double PR[8], double gamma,
                                      double Fh[8], unsigned& nfb) {
    FaceGeom m;
    m.alp = 0.5 * (ldg(met + iL) + ldg(met + iR));
#pragma unroll
    for (int a = 0; a < 3; ++a) m.beta[a] = 0.5 * (ldg(met + (1 + a) * nc + iL) + ldg(met + (1 + a) * nc + iR));
#pragma unroll
    for (int c = 0; c < 6; ++c) m.g[c] = 0.5 * (ldg(met + (4 + c) * nc + iL) + ldg(met + (4 + c) * nc + iR));
    face_flux<D>(m, PL, PR, prim + iL, prim + iR, nc, gamma, Fh, nfb);
}

template <int RECON, int TY>
__global__ void __launch_bounds__((TY + 1) * 32 + 128, 1)
rhs_ws_kernel(const __grid_constant__ RhsParams p, const TileGeom tg) {
    extern __shared__ double smem_raw[];
    Exch<TY>& Qb = *reinterpret_cast<Exch<TY>*>(smem_raw);
    Exch<TY>& Fb = *reinterpret_cast<Exch<TY>*>(smem_raw + sizeof(Exch<TY>) / sizeof(double));
    // sources hand-off: [buffer][S_x, S_y, S_z, S_tau][row][column]
    double (*Ssrc)[4][TY][TX] = reinterpret_cast<double (*)[4][TY][TX]>(smem_raw + 2 * sizeof(Exch<TY>) / sizeof(double));

    int t = blockIdx.x;
    const int tix = t % tg.ntx; t /= tg.ntx;
    const int tiy = t % tg.nty; t /= tg.nty;
    const int zc = t;
    const int box = blockIdx.y;
    const int X0 = tix * TX, Y0 = tiy * TY, k0 = zc * tg.tz;
    const int txe = min(TX, p.n[0] - X0), tye = min(TY, p.n[1] - Y0);
    const int nk = min(tg.tz, p.n[2] - k0);       // planes owned by this CTA
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (warp > TY) {
        // ------------------------------------------------ helper warp group: the geometric sources of the tile
        asm volatile("setmaxnreg.dec.sync.aligned.u32 152;");
        const int h = warp - (TY + 1);
        const int nc32 = (int)p.nc, sy32 = (int)p.stride[1], sz32 = (int)p.stride[2];
        const long long c00 = (long long)blockIdx.y * p.nc;
        const long long cell = (X0 + p.g + lane) + (long long)sy32 * (Y0 + p.g) + (long long)sz32 * (k0 + p.g);
        const double* __restrict__ pc = p.prim + 8 * c00 + cell;
        const double* __restrict__ mc = p.met + 10 * c00 + cell;
        const double* __restrict__ kc = p.K + 6 * c00 + cell;
        for (int kk = 0; kk < nk; ++kk, pc += sz32, mc += sz32, kc += sz32) {
            const int b = kk & 1;
            if (kk >= 2) bar_named_sync(4 + b, WS_ALL);          // the consumers are done with this buffer
            for (int r = h; r < tye; r += 4) {
                if (lane < txe) {
                    double a[8];
#pragma unroll
                    for (int q = 0; q < 8; ++q) a[q] = 0.0;
                    sources_add(p, pc + r * sy32, mc + r * sy32, kc + r * sy32, nc32, sy32, sz32, a);
#pragma unroll
                    for (int q = 0; q < 4; ++q) Ssrc[b][q][r][lane] = a[1 + q];
                }
            }
            __threadfence_block();
            bar_named_arrive(2 + b, WS_ALL);                     // sources of plane k0+kk are in shared memory
        }
        return;
    }
    asm volatile("setmaxnreg.inc.sync.aligned.u32 176;");

    const double* __restrict__ prim = p.prim + (long long)box * 8 * p.nc;
    const double* __restrict__ met = p.met + (long long)box * 10 * p.nc;
    const double* __restrict__ Kf = p.K + (long long)box * 6 * p.nc;
    double* __restrict__ out = p.out + (long long)box * 8 * p.nc;
    const long long nc = p.nc, sy = p.stride[1], sz = p.stride[2];
    const double gamma = p.gamma;
    const long long cbase = (X0 + p.g) + sy * (Y0 + p.g) + sz * (k0 - 1 + p.g);   // tile origin, plane k0-1
    unsigned nfb = 0;

    if (warp < TY) {
        // ------------------------------------------------ regular warp: one cell column per thread
        const bool active = (lane < txe) && (warp < tye);
        long long c = cbase + lane + sy * warp;
        double qpz[8], acc[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) { qpz[q] = 0.0; acc[q] = 0.0; }
        for (int kk = -1; kk <= nk; ++kk, c += sz) {
            if (tg.pf && active && kk < nk) {
                // first touches of this column: metric plane k+2 (z derivative at the end of THIS step), K_ij of
                // this plane, primitives of plane k+3 (z stencil at the top of the next step)
                if (tg.pf & 1) {
#pragma unroll
                    for (int f = 0; f < 10; ++f) prefetch_l1(met + f * nc + c + 2 * sz);
#pragma unroll
                    for (int f = 0; f < 6; ++f) prefetch_l1(Kf + f * nc + c);
                }
                if (tg.pf & 2) {
#pragma unroll
                    for (int q = 0; q < 8; ++q) prefetch_l1(prim + q * nc + c + 3 * sz);
                }
                if (tg.pf & 4) {
#pragma unroll
                    for (int q = 0; q < 8; ++q) prefetch_l2(prim + q * nc + c + 5 * sz);
#pragma unroll
                    for (int f = 0; f < 10; ++f) prefetch_l2(met + f * nc + c + 4 * sz);
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
                    face8<2>(prim, met, nc, c - sz, c, qpz, qm, gamma, Fh, (kk == 0 && k0 > 0) ? dup : nfb);
                    // F/dz is rounded once and used with both signs, so a uniform state cancels exactly
#pragma unroll
                    for (int q = 0; q < 8; ++q) Fh[q] = __dmul_rn(Fh[q], p.idx[2]);
                    if (kk >= 1) {
#pragma unroll
                        for (int q = 0; q < 8; ++q) out[q * nc + c - sz] = __dsub_rn(acc[q], Fh[q]);
                    }
#pragma unroll
                    for (int q = 0; q < 8; ++q) acc[q] = Fh[q];
                }
#pragma unroll
                for (int q = 0; q < 8; ++q) qpz[q] = qp[q];
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
            bar_main();
            if (active) {
                double PL[8], Fh[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) PL[q] = Qb.v[q][warp][lane];
                face8<0>(prim, met, nc, c - 1, c, PL, qm, gamma, Fh, nfb);
#pragma unroll
                for (int q = 0; q < 8; ++q) Fb.v[q][warp][lane] = Fh[q];
            }
            bar_main();
            // y
            if (active) {
#pragma unroll
                for (int q = 0; q < 8; ++q) acc[q] = fma(Fb.v[q][warp][lane] - Fb.v[q][warp][lane + 1], p.idx[0], acc[q]);
                double qp[8];
                recon8<RECON>(prim, nc, c, sy, qm, qp);
#pragma unroll
                for (int q = 0; q < 8; ++q) Qb.v[q][warp + 1][lane] = qp[q];
            }
            bar_main();
            if (active) {
                double PL[8], Fh[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) PL[q] = Qb.v[q][warp][lane];
                face8<1>(prim, met, nc, c - sy, c, PL, qm, gamma, Fh, nfb);
#pragma unroll
                for (int q = 0; q < 8; ++q) Fb.v[q][warp][lane] = Fh[q];
            }
            bar_main();
            if (active) {
#pragma unroll
                for (int q = 0; q < 8; ++q) acc[q] = fma(Fb.v[q][warp][lane] - Fb.v[q][warp + 1][lane], p.idx[1], acc[q]);
            }
            {
                const int b = kk & 1;
                bar_named_sync(2 + b, WS_ALL);                    // the helper group has published this plane's sources
                if (active) {
#pragma unroll
                    for (int q = 0; q < 4; ++q) acc[1 + q] += Ssrc[b][q][warp][lane];
                }
                bar_named_arrive(4 + b, WS_ALL);
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
            bar_main();
            if (xr) {
                double PL[8], Fh[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) PL[q] = Qb.v[q][xrow][txe];
                face8<0>(prim, met, nc, cxr - 1, cxr, PL, xr_qm, gamma, Fh, count_x ? nfb : dup);
#pragma unroll
                for (int q = 0; q < 8; ++q) Fb.v[q][xrow][txe] = Fh[q];
            }
            bar_main();
            if (ycol) {
#pragma unroll
                for (int q = 0; q < 8; ++q) Qb.v[q][0][lane] = yb_qp[q];
            }
            bar_main();
            if (ycol) {
                double PL[8], Fh[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) PL[q] = Qb.v[q][tye][lane];
                face8<1>(prim, met, nc, cyt - sy, cyt, PL, yt_qm, gamma, Fh, count_y ? nfb : dup);
#pragma unroll
                for (int q = 0; q < 8; ++q) Fb.v[q][tye][lane] = Fh[q];
            }
            bar_main();
            bar_named_sync(2 + (kk & 1), WS_ALL);                 // keep the hand-off barrier counts uniform
            bar_named_arrive(4 + (kk & 1), WS_ALL);
        }
    }
    if (p.nfallback && nfb) atomicAdd(p.nfallback, (unsigned long long)nfb);
}


TileGeom make_tiles_ws(const RhsParams& p, int ty, int slots) {
    TileGeom tg;
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
    tg.pf = 3;
    return tg;
}

template <int RECON>
cudaError_t launch_ws_t(const RhsParams& p, cudaStream_t st) {
    constexpr int TY = 7;
    static int sms = 0;
    if (sms == 0) {
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return e;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return e;
    }
    const size_t smem = 2 * sizeof(Exch<TY>) + 2 * 4 * TY * TX * sizeof(double);
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(rhs_ws_kernel<RECON, TY>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    const TileGeom tg = make_tiles_ws(p, TY, sms);
    const dim3 grid((unsigned)(tg.ntx * tg.nty * tg.nzc), p.nbox);
    rhs_ws_kernel<RECON, TY><<<grid, (TY + 1) * 32 + 128, smem, st>>>(p, tg);
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_rhs_ws(const RhsParams& p, int recon, cudaStream_t st) {
    if (recon == RECON_WENO5) return launch_ws_t<RECON_WENO5>(p, st);
    if (recon == RECON_MC) return launch_ws_t<RECON_MC>(p, st);
    return launch_ws_t<RECON_MINMOD>(p, st);
}

}  // namespace grx
