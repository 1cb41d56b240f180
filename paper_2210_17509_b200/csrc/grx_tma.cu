// grx_tma.cu -- the product kernel: the fused right-hand side (steps 2-4: reconstruct -> HLLE ->
// flux divergence + sources, all three directions, every face flux computed once) with every stencil operand served
// from shared memory.
//
// Decomposition: a CTA owns an in-plane tile of 32 x TY cells (one warp per row, lanes along x) and marches along z
// through a chunk of the block, one plane per step; an extra "rim" warp computes the faces on the tile's edge and
// drives the TMA engine.  The memory side is explicit:
//   * the current plane of the 8 primitives with its halo (3 cells for WENO5, 2 for TVD) and of the 10 metric
//     fields with a 2-cell halo is brought in by TMA (cp.async.bulk.tensor, one elected thread, mbarrier
//     completion), one step ahead of its use; all in-plane stencil reads (x/y reconstruction, face averages,
//     x/y metric derivatives) are LDS at compile-time offsets from one per-thread base address;
//   * the z stencils live in thread-private rings in shared memory: the primitives (planes k-2, k-1, k+1; the centre
//     comes from the staged plane) and the metric (planes k-2 .. k+1), so a step touches each plane once;
//   * what is left on the global path per cell and step -- the look-ahead plane of the primitives (8 loads), metric
//     plane k+2 (10), K_ij (6) -- is loaded one step ahead, before the step's last barrier, from lines the producer has
//     pulled into L2 with cp.async.bulk.prefetch.tensor; plus the 8 stores of the finished cell;
//   * x: q^+ and the flux move between neighbouring lanes by warp shuffle; y: one exchange buffer, two barriers per
//     plane.
// Requires even Nx and 16-byte aligned arrays (TMA global strides); grx_api.cu takes grx_fused.cu otherwise.
#include <cuda.h>

#include <cstdio>
#include <cstdlib>
#include <mutex>

#include "grx_launch.h"

namespace grx {

namespace {

constexpr int TX = 32;

struct TmaGeom {
    int ntx, nty, nzc, tz;
};

constexpr int align16(int x) { return (x + 15) & ~15; }

// Shared-memory layout (in doubles) of one CTA.
template <int RECON, int TY>
struct Lay {
    static constexpr int H = (RECON == RECON_WENO5) ? 3 : 2;                  // halo of the staged primitives
    static constexpr int PW = TX + 2 * H + 2, PR = TY + 2 * H, PF = PW * PR;  // row pitch (+2: even box start), rows, field stride
    static constexpr int MH = 2;                                              // halo of the staged metric
    static constexpr int MW = TX + 2 * MH + 2, MR = TY + 2 * MH, MF = MW * MR;
    static constexpr int NT = TY * 32;                                        // row-warp threads
    static constexpr int NRING = (RECON == RECON_WENO5) ? 3 : 1;              // z-history planes of the primitives
    static constexpr int LOOK = H - 1;                                        // look-ahead plane loaded from global
    static constexpr int EF = (TY + 1) * TX;                                  // field stride of the y exchange buffer
    static constexpr int o_ps = 0;
    static constexpr int o_ms = align16(o_ps + 8 * PF);
    static constexpr int o_zr = align16(o_ms + 10 * MF);
    static constexpr int o_qc = o_zr + NRING * 8 * NT;
    static constexpr int o_qf = o_qc + 8 * NT;
    static constexpr int o_fx = o_qf + 8 * EF;
    static constexpr int o_xp = o_fx + 16 * TY;
    static constexpr int o_mz = o_xp + 16 * TY;                               // z ring of the metric: planes k-2 .. k+1 by (plane & 3)
    static constexpr int o_bar = align16(o_mz + 4 * 10 * NT);
    static constexpr int total = o_bar + 16;
    static_assert(total * sizeof(double) <= 227 * 1024, "tile does not fit the 227 KB of shared memory of a CTA");
    static constexpr unsigned ps_bytes = 8u * PF * sizeof(double);
    static constexpr unsigned ms_bytes = 10u * MF * sizeof(double);
};

// ---- mbarrier / TMA primitives (PTX) ---------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
    asm volatile(
        "{\n\t"
        ".reg .pred P1;\n\t"
        "GRX_WAIT:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n\t"
        "@P1 bra GRX_DONE;\n\t"
        "bra GRX_WAIT;\n\t"
        "GRX_DONE:\n\t"
        "}" ::"r"(bar), "r"(parity)
        : "memory");
}
__device__ __forceinline__ void tma_load_4d(unsigned dst, const CUtensorMap* map, unsigned bar, int c0, int c1, int c2,
                                            int c3) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];" ::"r"(dst),
        "l"(reinterpret_cast<unsigned long long>(map)), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
        : "memory");
}

__device__ __forceinline__ void tma_prefetch_4d(const CUtensorMap* map, int c0, int c1, int c2, int c3) {
    asm volatile("cp.async.bulk.prefetch.tensor.4d.L2.global [%0, {%1, %2, %3, %4}];" ::"l"(
                     reinterpret_cast<unsigned long long>(map)),
                 "r"(c0), "r"(c1), "r"(c2), "r"(c3)
                 : "memory");
}

// ---- stencil readers on the staged planes ---------------------------------------------------------------------
// Reconstruct the 8 primitives of the cell at `pb` (field stride PF) along a direction with element stride S.
template <int RECON, int PF, int S>
__device__ __forceinline__ void recon8_smem(const double* pb, double qm[8], double qp[8]) {
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        const double* f = pb + q * PF;
        double a = 0.0, e = 0.0;
        if (RECON == RECON_WENO5) { a = f[-2 * S]; e = f[2 * S]; }
        recon_cell<RECON>(a, f[-S], f[0], f[S], e, qm[q], qp[q]);
    }
}

// Two-point average of the ten metric fields between the cell at mb - S and the cell at mb (a1).
template <int MF, int S>
__device__ __forceinline__ void face_geom_smem(const double* mb, FaceGeom& m) {
    double v[10];
#pragma unroll
    for (int f = 0; f < 10; ++f) v[f] = 0.5 * (mb[f * MF - S] + mb[f * MF]);
    m.alp = v[0];
#pragma unroll
    for (int a = 0; a < 3; ++a) m.beta[a] = v[1 + a];
#pragma unroll
    for (int c = 0; c < 6; ++c) m.g[c] = v[4 + c];
}

template <int MF, int S>
__device__ __forceinline__ void dmetric_smem(const double* mb, double d[10]) {
#pragma unroll
    for (int f = 0; f < 10; ++f) d[f] = d4raw(mb[f * MF - 2 * S], mb[f * MF - S], mb[f * MF + S], mb[f * MF + 2 * S]);
}

// CT: the kernel also writes the HLLE fluxes of the transverse calB components of every face it evaluates to p.fb
// (constrained transport, grx_valencia_rhs_ct): [6][cell] = F^x(B^y), F^x(B^z), F^y(B^x), F^y(B^z), F^z(B^x), F^z(B^y)
// at the LOW face of the cell, unscaled.
template <int RECON, int TY, bool CT>
__global__ void __launch_bounds__((TY + 1) * 32, 1)
rhs_tma_kernel(const __grid_constant__ RhsParams p, const TmaGeom tg, const __grid_constant__ CUtensorMap tmP,
                const __grid_constant__ CUtensorMap tmM, const __grid_constant__ CUtensorMap tmK) {
    using L = Lay<RECON, TY>;
    constexpr int H = L::H, PW = L::PW, PF = L::PF, MH = L::MH, MW = L::MW, MF = L::MF, NT = L::NT, EF = L::EF;
    constexpr unsigned FULL = 0xffffffffu;
    static_assert(4 * TY <= 32, "the rim warp needs four lanes per row");
    extern __shared__ __align__(1024) double sm[];
    double* const PS = sm + L::o_ps;
    double* const MS = sm + L::o_ms;
    double* const QF = sm + L::o_qf;   // [8][TY+1][32] y exchange: q^+ of the row below, then that face's flux
    double* const FX = sm + L::o_fx;   // [2][8][TY] fluxes of the first and the last x face of every row (rim warp)
    double* const XP = sm + L::o_xp;   // [2][8][TY] what the first / last lane of a row parks until those arrive
    const unsigned barP = smem_u32(sm + L::o_bar), barM = barP + 8;

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
    const double* __restrict__ met = p.met + (long long)box * 10 * p.nc;
    const double* __restrict__ Kf = p.K + (long long)box * 6 * p.nc;
    double* __restrict__ out = p.out + (long long)box * 8 * p.nc;
    double* __restrict__ fb = CT ? p.fb + (long long)box * 6 * p.nc : nullptr;
    const long long nc = p.nc, sy = p.stride[1], sz = p.stride[2];
    const double gamma = p.gamma;
    const long long cbase = (X0 + p.g) + sy * (Y0 + p.g) + sz * (k0 - 1 + p.g);   // tile origin, plane k0-1
    unsigned nfb = 0;

    // TMA coordinates of the tile's staged boxes (x, y; z and the field block follow per plane).  A box must start
    // on a 16-byte boundary of global memory (measured: an odd FP64 start coordinate raises "illegal instruction"),
    // so the box starts at the even column at or below the halo and is two columns wider than the halo needs.
    const int dP = (p.g - H) & 1, dM = (p.g - MH) & 1;
    const int pcx = X0 + p.g - H - dP, pcy = Y0 + p.g - H, mcx = X0 + p.g - MH - dM, mcy = Y0 + p.g - MH;
    const int kcx = X0 + p.g - (p.g & 1);   // K_ij is only prefetched: own columns from the even column down
    const bool producer = (threadIdx.x == TY * 32);
    if (producer) {
        mbar_init(barP, 1);
        mbar_init(barM, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (producer) {
        mbar_expect_tx(barP, L::ps_bytes);
        tma_load_4d(smem_u32(PS), &tmP, barP, pcx, pcy, k0 - 1 + p.g, box * 8);
        mbar_expect_tx(barM, L::ms_bytes);
        tma_load_4d(smem_u32(MS), &tmM, barM, mcx, mcy, k0 + p.g, box * 10);
        // L2 prefetch of the planes the first steps load from global memory (later planes: one per step, below)
        for (int j = 0; j <= 3; ++j) {
            tma_prefetch_4d(&tmP, pcx, pcy, k0 + j + p.g, box * 8);
            tma_prefetch_4d(&tmM, mcx, mcy, k0 + j + p.g, box * 10);
            if (j <= 1) tma_prefetch_4d(&tmK, kcx, mcy + MH, k0 + j + p.g, box * 6);
        }
    }

    if (warp < TY) {
        // ------------------------------------------------ row warp: one cell column per thread
        const bool active = (lane < txe) && (warp < tye);
        const bool first = (lane == 0), last = (lane == txe - 1);
        long long c = cbase + lane + sy * warp;
        const double* const psb = PS + (H + warp) * PW + (H + dP + lane);     // this cell in the staged primitives
        const double* const msb = MS + (MH + warp) * MW + (MH + dM + lane);   // ... and in the staged metric
        double* const zr = sm + L::o_zr + threadIdx.x;                        // z ring: [slot][field][thread]
        double* const qc = sm + L::o_qc + threadIdx.x;                        // q^+ of the previous plane: [field][thread]
        double* const qf = QF + warp * 32 + lane;                             // this cell's low y face in the exchange
        double* const mz = sm + L::o_mz + threadIdx.x;                        // z ring of the metric: [plane & 3][field][thread]
        int h2 = 0, h1 = 1;                                                   // ring slots of planes k-2, k-1 (WENO5); slot 2 = k+1
        double acc[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) acc[q] = 0.0;
        if (active) {
            // ring for the first step (plane k0-1): planes k0-3, k0-2 | k0 (WENO5), k0-2 (TVD)
            if (RECON == RECON_WENO5) {
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    zr[(0 * 8 + q) * NT] = ldg(prim + q * nc + c - 2 * sz);
                    zr[(1 * 8 + q) * NT] = ldg(prim + q * nc + c - sz);
                    zr[(2 * 8 + q) * NT] = ldg(prim + q * nc + c + sz);
                }
            } else {
#pragma unroll
                for (int q = 0; q < 8; ++q) zr[q * NT] = ldg(prim + q * nc + c - sz);
            }
            // metric planes k0-2, k0-1, k0 (ring slot = plane index relative to k0, mod 4)
#pragma unroll
            for (int j = -2; j <= 0; ++j)
#pragma unroll
                for (int f = 0; f < 10; ++f) mz[(((j + 4) & 3) * 10 + f) * NT] = ldg(met + f * nc + c + (j + 1) * sz);
        }
        // The global loads of a step -- the look-ahead plane of the primitives, metric plane k+2 and K_ij -- are issued
        // one step ahead, before the last barrier of the step before, so that they are in flight while the CTA waits
        // there (measured: issuing the metric and K_ij at the top of their own step costs 2-5 %).  The producer's TMA
        // prefetch has pulled their lines into L2 by then.
        double qn[8], mn[10], K6[6], dz[10];
        auto issue_loads = [&](int kn, long long cn) {
            if (kn <= nk) {
#pragma unroll
                for (int q = 0; q < 8; ++q) qn[q] = ldg(prim + q * nc + cn + L::LOOK * sz);
            }
            if (kn < nk) {
#pragma unroll
                for (int f = 0; f < 10; ++f) mn[f] = ldg(met + f * nc + cn + 2 * sz);
                if (kn >= 0) {
#pragma unroll
                    for (int f = 0; f < 6; ++f) K6[f] = ldg(Kf + f * nc + cn);
                }
            }
        };
        if (active) issue_loads(-1, c);
        for (int kk = -1; kk <= nk; ++kk, c += sz) {
            // ---------------- z: reconstruct this cell, close the face below it, finish the cell below
            mbar_wait(barP, (unsigned)(kk + 1) & 1u);
            if (active) {
                double qm[8], qp[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    const double c0 = psb[q * PF];
                    if (RECON == RECON_WENO5) {
                        recon_cell<RECON>(zr[(h2 * 8 + q) * NT], zr[(h1 * 8 + q) * NT], c0, zr[(2 * 8 + q) * NT], qn[q],
                                          qm[q], qp[q]);
                        zr[(h2 * 8 + q) * NT] = c0;       // plane k takes the slot of plane k-2
                        zr[(2 * 8 + q) * NT] = qn[q];     // plane k+2 takes the slot of plane k+1 (next centre: staged)
                    } else {
                        recon_cell<RECON>(0.0, zr[q * NT], c0, qn[q], 0.0, qm[q], qp[q]);
                        zr[q * NT] = c0;
                    }
                }
                if (kk >= 0) {
                    double Fh[8], qpz[8];
                    unsigned dup = 0;   // the first face of an inner chunk is the last face of the chunk below: count once
#pragma unroll
                    for (int q = 0; q < 8; ++q) qpz[q] = qc[q * NT];
                    FaceGeom m;
                    {
                        const double* m1 = mz + ((kk + 3) & 3) * 10 * NT;   // plane k-1
                        const double* m0 = mz + (kk & 3) * 10 * NT;         // plane k
                        m.alp = 0.5 * (m1[0] + m0[0]);
#pragma unroll
                        for (int a = 0; a < 3; ++a) m.beta[a] = 0.5 * (m1[(1 + a) * NT] + m0[(1 + a) * NT]);
#pragma unroll
                        for (int g6 = 0; g6 < 6; ++g6) m.g[g6] = 0.5 * (m1[(4 + g6) * NT] + m0[(4 + g6) * NT]);
                    }
                    face_flux<2>(m, qpz, qm, prim + c - sz, prim + c, nc, gamma, Fh, (kk == 0 && k0 > 0) ? dup : nfb);
                    if (CT) { fb[4 * nc + c] = Fh[5]; fb[5 * nc + c] = Fh[6]; }
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
                for (int q = 0; q < 8; ++q) qc[q * NT] = qp[q];
                if (kk < nk) {
                    // z stencil sums of the metric for this cell's sources, then plane k+2 takes the slot of plane k-2
                    const double* m2 = mz + ((kk + 2) & 3) * 10 * NT;
                    const double* m1 = mz + ((kk + 3) & 3) * 10 * NT;
                    const double* p1 = mz + ((kk + 1) & 3) * 10 * NT;
                    if (kk >= 0) {
#pragma unroll
                        for (int f = 0; f < 10; ++f) dz[f] = d4raw(m2[f * NT], m1[f * NT], p1[f * NT], mn[f]);
                    }
#pragma unroll
                    for (int f = 0; f < 10; ++f) mz[(((kk + 2) & 3) * 10 + f) * NT] = mn[f];
                }
            }
            if (RECON == RECON_WENO5) { const int tmp = h2; h2 = h1; h1 = tmp; }
            if (kk < 0 || kk >= nk) {   // uniform over the CTA: no in-plane work on the planes next to the chunk
                if (active) issue_loads(kk + 1, c + sz);
                __syncthreads();
                continue;
            }
            // ---------------- x: q^+ and the flux move between neighbouring lanes by warp shuffle; the first and the
            // last face of the row are the rim warp's (FX), and the lanes next to them park their half of the
            // difference until the first barrier
            double qm[8], qx[8];
#pragma unroll
            for (int q = 0; q < 8; ++q) qx[q] = 0.0;
            if (active) recon8_smem<RECON, PF, 1>(psb, qm, qx);
#pragma unroll
            for (int q = 0; q < 8; ++q) qx[q] = __shfl_up_sync(FULL, qx[q], 1);   // q^+ of the cell to the left
            mbar_wait(barM, (unsigned)kk & 1u);
            double Fx[8];
#pragma unroll
            for (int q = 0; q < 8; ++q) Fx[q] = 0.0;
            if (active && !first) {
                FaceGeom m;
                face_geom_smem<MF, 1>(msb, m);
                face_flux<0>(m, qx, qm, prim + c - 1, prim + c, nc, gamma, Fx, nfb);
                if (CT) { fb[c] = Fx[6]; fb[nc + c] = Fx[7]; }
            }
#pragma unroll
            for (int q = 0; q < 8; ++q) qx[q] = __shfl_down_sync(FULL, Fx[q], 1);   // flux of the high face
            if (active) {
                if (!first && !last) {
#pragma unroll
                    for (int q = 0; q < 8; ++q) acc[q] = fma(Fx[q] - qx[q], p.idx[0], acc[q]);
                } else {
                    if (first) {
#pragma unroll
                        for (int q = 0; q < 8; ++q) XP[q * TY + warp] = qx[q];
                    }
                    if (last) {
#pragma unroll
                        for (int q = 0; q < 8; ++q) XP[(8 + q) * TY + warp] = Fx[q];
                    }
                }
                // ---------------- y
                recon8_smem<RECON, PF, PW>(psb, qm, qx);
#pragma unroll
                for (int q = 0; q < 8; ++q) qf[q * EF + 32] = qx[q];
            }
            __syncthreads();                                   // (A) the staged primitives are free from here on
            double Fh[8];   // flux of this cell's low y face: published for the row below, kept for the own difference
#pragma unroll
            for (int q = 0; q < 8; ++q) Fh[q] = 0.0;
            if (active) {
                if (first || last) {
                    // x difference of the row's end cells: low face from FX[0] / parked, high face from parked / FX[1]
#pragma unroll
                    for (int q = 0; q < 8; ++q) {
                        const double lo = first ? FX[q * TY + warp] : XP[(8 + q) * TY + warp];
                        const double hi = last ? FX[(8 + q) * TY + warp] : XP[q * TY + warp];
                        acc[q] = fma(lo - hi, p.idx[0], acc[q]);
                    }
                }
                // ---------------- sources (a8 + a9): centre primitives from the ring (plane k sits in slot h1 now), x and
                // y stencils of the metric from the staged plane, z stencil sums and K_ij from the top of the step
                {
                    SrcState s;
                    {
                        double P[8], mm[10];
#pragma unroll
                        for (int q = 0; q < 8; ++q) P[q] = (RECON == RECON_WENO5) ? zr[(h1 * 8 + q) * NT] : zr[q * NT];
#pragma unroll
                        for (int f = 0; f < 10; ++f) mm[f] = msb[f * MF];
                        sources_prepare(P, mm, gamma, s);
                    }
                    double st = 0.0, d[10];
                    dmetric_smem<MF, 1>(msb, d);
                    acc[1] += sources_dir(s, 0, d, p.idx[0] * (1.0 / 12.0), st);
                    dmetric_smem<MF, MW>(msb, d);
                    acc[2] += sources_dir(s, 1, d, p.idx[1] * (1.0 / 12.0), st);
                    acc[3] += sources_dir(s, 2, dz, p.idx[2] * (1.0 / 12.0), st);
                    acc[4] += st + sources_K(s, K6);
                }
                // ---------------- y face
                double PL[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) PL[q] = qf[q * EF];
                FaceGeom m;
                face_geom_smem<MF, MW>(msb, m);
                face_flux<1>(m, PL, qm, prim + c - sy, prim + c, nc, gamma, Fh, nfb);
                if (CT) { fb[2 * nc + c] = Fh[5]; fb[3 * nc + c] = Fh[7]; }
#pragma unroll
                for (int q = 0; q < 8; ++q) qf[q * EF] = Fh[q];
                issue_loads(kk + 1, c + sz);
            }
            __syncthreads();                                   // (B) the staged metric is free from here on
            if (active) {
#pragma unroll
                for (int q = 0; q < 8; ++q) acc[q] = fma(Fh[q] - qf[q * EF + 32], p.idx[1], acc[q]);
            }
        }
    } else {
        // ------------------------------------------------ rim warp: the tile's edge faces, and the TMA producer
        // y-rim: lane l < txe -> cell (X0+l, Y0-1) [q^+ for the row warps] and the last face of column l
        // x-rim lanes, four per row: group 0 = cell X0-1, 1 = X0 (the two sides of the row's first face), 2 = X0+txe-1,
        // 3 = X0+txe (its last face); one reconstruction pass covers all four, q^- moves from the odd groups to the
        // even ones by shuffle, and the even groups evaluate the faces
        const int xgrp = lane / TY, xrow = lane - xgrp * TY;
        const bool xrec = (xgrp < 4) && (xrow < tye);
        const bool xface = xrec && !(xgrp & 1);
        const bool ycol = lane < txe;
        // the last faces are the first faces of the next tile too: they count only at the block's end
        const bool count_x = (xgrp == 0) || (X0 + txe == p.n[0]), count_y = (Y0 + tye == p.n[1]);
        unsigned dup = 0;
        // staged positions: this lane's x-rim cell, the y-rim cells of column `lane`
        const int xcol = (xgrp == 0) ? -1 : (xgrp == 1) ? 0 : (xgrp == 2) ? txe - 1 : txe;
        const double* const px = PS + (H + xrow) * PW + (H + dP + xcol);
        const double* const mx = MS + (MH + xrow) * MW + (MH + dM + xcol + 1);   // right cell of the face (even groups)
        const double* const pyb = PS + (H - 1) * PW + (H + dP + lane);
        const double* const pyt = PS + (H + tye) * PW + (H + dP + lane);
        const double* const myt = MS + (MH + tye) * MW + (MH + dM + lane);
        double* const fxo = FX + (xgrp == 0 ? 0 : 8 * TY) + xrow;
        for (int kk = -1; kk <= nk; ++kk) {
            mbar_wait(barP, (unsigned)(kk + 1) & 1u);
            if (kk < 0 || kk >= nk) {
                __syncthreads();
                if (producer && kk < nk) {
                    mbar_expect_tx(barP, L::ps_bytes);
                    tma_load_4d(smem_u32(PS), &tmP, barP, pcx, pcy, k0 + kk + 1 + p.g, box * 8);
                }
                continue;
            }
            const long long cp = cbase + sz * (kk + 1);   // tile origin in plane k0+kk
            // y first: it needs the staged primitives only; the staged metric (x-rim faces) was requested last
            double yt_qm[8];
            if (ycol) {
                double tmp[8], yb_qp[8];
                recon8_smem<RECON, PF, PW>(pyb, tmp, yb_qp);
#pragma unroll
                for (int q = 0; q < 8; ++q) QF[q * EF + lane] = yb_qp[q];
                recon8_smem<RECON, PF, PW>(pyt, yt_qm, tmp);
            }
            mbar_wait(barM, (unsigned)kk & 1u);
            {
                double PL[8], PR[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) PL[q] = PR[q] = 0.0;
                if (xrec) recon8_smem<RECON, PF, 1>(px, PR, PL);
#pragma unroll
                for (int q = 0; q < 8; ++q) PR[q] = __shfl_down_sync(FULL, PR[q], TY);   // q^- of the cell to the right
                if (xface) {
                    double Fh[8];
                    FaceGeom m;
                    face_geom_smem<MF, 1>(mx, m);
                    const long long cxr = cp + sy * xrow + xcol + 1;
                    face_flux<0>(m, PL, PR, prim + cxr - 1, prim + cxr, nc, gamma, Fh, count_x ? nfb : dup);
                    // one writer per face: the face between two tiles is also the first face of the next tile's rows
                    if (CT && count_x) { fb[cxr] = Fh[6]; fb[nc + cxr] = Fh[7]; }
#pragma unroll
                    for (int q = 0; q < 8; ++q) fxo[q * TY] = Fh[q];
                }
            }
            __syncthreads();                                   // (A)
            if (producer) {   // every read of the staged primitives is done: bring in the next plane
                mbar_expect_tx(barP, L::ps_bytes);
                tma_load_4d(smem_u32(PS), &tmP, barP, pcx, pcy, k0 + kk + 1 + p.g, box * 8);
                // ... and pull the planes the row warps load from global memory a step later from HBM into L2
                if (kk + 4 <= nk + 2) {
                    tma_prefetch_4d(&tmP, pcx, pcy, k0 + kk + 4 + p.g, box * 8);
                    tma_prefetch_4d(&tmM, mcx, mcy, k0 + kk + 4 + p.g, box * 10);
                }
                if (kk + 2 < nk) tma_prefetch_4d(&tmK, kcx, mcy + MH, k0 + kk + 2 + p.g, box * 6);
            }
            if (ycol) {
                double PL[8], Fh[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) PL[q] = QF[q * EF + tye * 32 + lane];
                FaceGeom m;
                face_geom_smem<MF, MW>(myt, m);
                const long long cyt = cp + lane + sy * tye;
                face_flux<1>(m, PL, yt_qm, prim + cyt - sy, prim + cyt, nc, gamma, Fh, count_y ? nfb : dup);
                // one writer per face: the face between two row tiles is written by row 0 of the tile above, whose
                // inlined face_flux rounds differently from this one (two writers made the stored bits a race)
                if (CT && count_y) { fb[2 * nc + cyt] = Fh[5]; fb[3 * nc + cyt] = Fh[7]; }
#pragma unroll
                for (int q = 0; q < 8; ++q) QF[q * EF + tye * 32 + lane] = Fh[q];
            }
            __syncthreads();                                   // (B)
            if (producer && kk + 1 < nk) {
                mbar_expect_tx(barM, L::ms_bytes);
                tma_load_4d(smem_u32(MS), &tmM, barM, mcx, mcy, k0 + kk + 1 + p.g, box * 10);
            }
        }
    }
    if (p.nfallback && nfb) atomicAdd(p.nfallback, (unsigned long long)nfb);
}

// ---- host side ------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = nullptr;
    static std::once_flag once;
    std::call_once(once, [] {
        void* sym = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(sym);
    });
    return fn;
}

// 4-D map [field*box][z][y][x] of an FP64 SoA array with boxes of bx x by x 1 x nf elements.
bool make_map(CUtensorMap* map, const double* base, const RhsParams& p, int nf, int bx, int by) {
    EncodeTiledFn enc = encode_fn();
    if (!enc) return false;
    const cuuint64_t dims[4] = {(cuuint64_t)p.N[0], (cuuint64_t)p.N[1], (cuuint64_t)p.N[2], (cuuint64_t)nf * p.nbox};
    const cuuint64_t strides[3] = {(cuuint64_t)p.N[0] * 8, (cuuint64_t)p.stride[2] * 8, (cuuint64_t)p.nc * 8};
    const cuuint32_t box[4] = {(cuuint32_t)bx, (cuuint32_t)by, 1u, (cuuint32_t)nf};
    const cuuint32_t estr[4] = {1u, 1u, 1u, 1u};
    const CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<double*>(base), dims, strides, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

// z-chunking: enough CTAs to fill the machine in whole waves, chunks long enough to amortise what a chunk costs
// besides its planes: the ring fill, the first TMA round trip and the two one-sided plane steps at its ends
// (together about 1.8 plane steps, measured on the 32^3 and 64^3 batches).  Returns the expected efficiency
// (wave fill x chunk factor x used rows of the row tiles) in *eff.
constexpr double CHUNK_OVERHEAD = 1.8;
TmaGeom make_tiles(const RhsParams& p, int ty, int slots, double* eff_out = nullptr) {
    TmaGeom tg;
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
        const double eff = fill * tz / (tz + CHUNK_OVERHEAD);
        if (eff > best_eff * 1.001) { best_eff = eff; best = nzc; }
    }
    tg.tz = (p.n[2] + best - 1) / best;
    tg.nzc = (p.n[2] + tg.tz - 1) / tg.tz;
    if (eff_out) *eff_out = best_eff * p.n[1] / ((double)tg.nty * ty);
    return tg;
}

template <int RECON, int TY, bool CT>
cudaError_t launch_one(const RhsParams& p, cudaStream_t st) {
    using L = Lay<RECON, TY>;
    int dev = 0, sms = 0;
    cudaError_t e = current_device_sms(&dev, &sms);
    if (e != cudaSuccess) return e;
    CUtensorMap tmP, tmM, tmK;
    if (!make_map(&tmP, p.prim, p, 8, L::PW, L::PR) || !make_map(&tmM, p.met, p, 10, L::MW, L::MR) ||
        !make_map(&tmK, p.K, p, 6, TX + 2, TY))
        return cudaErrorNotSupported;
    const size_t smem = (size_t)L::total * sizeof(double);
    static std::atomic<unsigned long long> smem_set{0};   // per instantiation: devices on which the attribute is set
    e = set_max_dynamic_smem_once(rhs_tma_kernel<RECON, TY, CT>, dev, smem, smem_set);
    if (e != cudaSuccess) return e;
    const TmaGeom tg = make_tiles(p, TY, sms);
    const dim3 grid((unsigned)(tg.ntx * tg.nty * tg.nzc), p.nbox);
    rhs_tma_kernel<RECON, TY, CT><<<grid, (TY + 1) * 32, smem, st>>>(p, tg, tmP, tmM, tmK);
    return cudaGetLastError();
}

template <int RECON>
cudaError_t dispatch(const RhsParams& p, int ty, cudaStream_t st) {
    // 7 rows: 8 warps per SM at 254 registers, 211 KB of shared memory (the largest tile whose rings fit)
    if (ty == 7) return p.fb ? launch_one<RECON, 7, true>(p, st) : launch_one<RECON, 7, false>(p, st);
    return cudaErrorInvalidConfiguration;
}

}  // namespace

bool tma_supported(const RhsParams& p) {
    // TMA: global strides are multiples of 16 bytes (even Nx) and the arrays are 16-byte aligned
    if (p.N[0] % 2 != 0) return false;
    if (((uintptr_t)p.prim | (uintptr_t)p.met | (uintptr_t)p.K) & 15u) return false;
    return encode_fn() != nullptr;
}

double tma_tile_efficiency(const RhsParams& p, int sms) {
    double eff = 0.0;
    make_tiles(p, 7, sms, &eff);
    return eff;
}

cudaError_t launch_rhs_tma(const RhsParams& p, int recon, int ty, cudaStream_t st) {
    if (recon == RECON_WENO5) return dispatch<RECON_WENO5>(p, ty, st);
    if (recon == RECON_MC) return dispatch<RECON_MC>(p, ty, st);
    return dispatch<RECON_MINMOD>(p, ty, st);
}

}  // namespace grx
