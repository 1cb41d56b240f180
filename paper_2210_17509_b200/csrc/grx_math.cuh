// grx_math.cuh -- point-wise arithmetic of the Valencia GRMHD right-hand side (CUDA path).
//
// Everything here is per-point math: reconstruction of one cell (a2), face geometry (a1), one HLLE
// face flux (a3-a6) and the geometric sources of one cell (a8-a9).  The kernels in grx_kernels.cu decide
// who computes which point.  Citations are PAPER.md line numbers; R* are the readings in DESIGN.md.
//
// The formulas are algebraically those of the paper but arranged for the FP64 pipe of sm_100a: no IEEE
// divisions (MUFU seed + one third-order correction, error < 1 ulp-ish, see rcp()/rsqrt()), a common
// denominator for the WENO5 weights, a^2 = (b^2 + Gamma p)/(rho h*) for the fast speed, the sources in
// their Eulerian-observer form.  All of these are rounding-level rearrangements (reading R26).
//
// The file also compiles as plain C++ (g++, tests/host_math_harness.cpp) so that the arithmetic can be
// checked on a machine without a GPU; the host build is test infrastructure, never a product path.
#pragma once

#include <math.h>

#if defined(__CUDACC__)
#define GRX_HD __host__ __device__ __forceinline__
#else
#define GRX_HD inline
#endif

namespace grx {

// ---- conventions (R4, R5) ----------------------------------------------------------------------------
constexpr double WENO_EPS = 1e-26;       // Jiang-Shu epsilon
constexpr double V2MAX    = 1.0 - 1e-4;  // admissibility bound on v^2 (W_max = 100)

enum { RECON_MINMOD = 0, RECON_MC = 1, RECON_WENO5 = 2 };

// ---- reciprocal, reciprocal square root, square root without the IEEE slow paths ----------------------
// MUFU.RCP64H / MUFU.RSQ64H seeds are good to 2^-19.9 / 2^-20.1 (measured on B200 over 2^-30..2^30, see
// profiles/r1_microbench.md); ONE third-order correction brings the relative error to 2.2e-16 / 2.6e-16,
// i.e. the rounding level of the IEEE operation (grx_selftest_math + tests/test_gpu_parity.py measure it).
// Arguments are positive, normal numbers everywhere these are used (determinants, lapse, rho h*, ...).
GRX_HD double rcp(double x) {
#if defined(__CUDA_ARCH__)
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x, y, 1.0);
    const double e2 = fma(e, e, e);
    return fma(y, e2, y);                       // y (1 + e + e^2)
#else
    return 1.0 / x;
#endif
}
GRX_HD double rsqrt(double x) {
#if defined(__CUDA_ARCH__)
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double t = x * y;
    const double h = fma(-t, y, 1.0);           // 1 - x y^2
    const double p = fma(0.375, h, 0.5);
    return fma(y * h, p, y);                    // y (1 + h/2 + 3h^2/8)
#else
    return 1.0 / sqrt(x);
#endif
}
// sqrt of a non-negative number (0 -> 0): g = x y ~ sqrt(x), corrected to third order in h = 1 - g y
GRX_HD double sqrt_nn(double x) {
#if defined(__CUDA_ARCH__)
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double g = x * y;
    const double h = fma(-g, y, 1.0);
    const double p = fma(0.375, h, 0.5);
    const double s = fma(g * h, p, g);
    return (x > 0.0) ? s : 0.0;
#else
    return sqrt(x);
#endif
}

// ---- a2: reconstruction of one cell ---------------------------------------------
// (a,b,c,d,e) = (q_{i-2} .. q_{i+2});  qm = value at face i-1/2 from cell i, qp = value at face i+1/2.
template <int RECON>
GRX_HD void recon_cell(double a, double b, double c, double d, double e, double& qm, double& qp) {
    if (RECON == RECON_WENO5) {
        // Jiang-Shu WENO5 (ref [32]); written in first differences so that constant data is exact.
        const double D1 = b - a, D2 = c - b, D3 = d - c, D4 = e - d;
        const double t0 = D2 - D1, t1 = D3 - D2, t2 = D4 - D3;           // second differences
        const double u0 = fma(3.0, D2, -D1);                              // a - 4b + 3c
        const double u1 = D2 + D3;                                        // d - b
        const double u2 = fma(-3.0, D3, D4);                              // 3c - 4d + e
        // 4*beta_k + 4 eps = 13/3 t_k^2 + u_k^2 + 4 eps  (the common factor 4 cancels in the weights; the epsilon rides
        // on the inner FMA)
        const double k133 = 13.0 / 3.0, eps4 = 4.0 * WENO_EPS;
        // t^2 first, then the constant as an FMA operand: a DFMA with a constant operand occupies the pipe 2 cycles, one with
        // three registers 3 (profiles/r2_issue_model.md)
        double e0 = fma(t0 * t0, k133, fma(u0, u0, eps4));
        double e1 = fma(t1 * t1, k133, fma(u1, u1, eps4));
        double e2 = fma(t2 * t2, k133, fma(u2, u2, eps4));
        e0 *= e0; e1 *= e1; e2 *= e2;
        // a_k = d_k / e_k  ->  multiply all three by e0 e1 e2 (common denominator, R26)
        const double e01 = e0 * e1, e02 = e0 * e2, e12 = e1 * e2;
        const double w1 = 6.0 * e02;
        // plus side: weights (1,6,3)/10 on (e12, e02, e01)
        const double wp2 = 3.0 * e01;
        const double Sp = e12 + w1 + wp2;
        // 6 p_k - 6 c in differences: 5 D2 - 2 D1 = 2 u0 - D2,  2 D3 + D2,  4 D3 - D4 = D3 - u2
        const double pp0 = fma(2.0, u0, -D2), pp1 = fma(2.0, D3, D2), pp2 = D3 - u2;
        const double Np = fma(wp2, pp2, fma(w1, pp1, e12 * pp0));
        // minus side: mirrored stencil, weights (1,6,3)/10 on (e01, e02, e12):  2 D4 - 5 D3 = 2 u2 + D3,
        // -(2 D2 + D3),  D1 - 4 D2 = -(u0 + D2)
        const double wm2 = 3.0 * e12;
        const double Sm = e01 + w1 + wm2;
        const double pm0 = fma(2.0, u2, D3), pm1 = -fma(2.0, D2, D3), pm2 = -(u0 + D2);
        const double Nm = fma(wm2, pm2, fma(w1, pm1, e01 * pm0));
        const double r = rcp(Sp * Sm) * (1.0 / 6.0);
        qp = fma(Np, Sm * r, c);
        qm = fma(Nm, Sp * r, c);
    } else {
        const double dm = c - b, dp = d - c;
        double sigma = 0.0;
        if (dm * dp > 0.0) {
            if (RECON == RECON_MC) {
                // monotonised central: sign * min(2|dm|, 2|dp|, |dm+dp|/2)
                const double m = fmin(fmin(2.0 * fabs(dm), 2.0 * fabs(dp)), 0.5 * fabs(dm + dp));
                sigma = (dm > 0.0) ? m : -m;
            } else {
                sigma = (fabs(dm) < fabs(dp)) ? dm : dp;   // minmod (l.255)
            }
        }
        qm = fma(-0.5, sigma, c);
        qp = fma(0.5, sigma, c);
    }
}

// ---- a1: geometry of one face (l.130; R6, R7) -----------------------------------------------------------
struct FaceGeom {
    double alp;            // lapse
    double beta[3];        // shift beta^i
    double g[6];           // gamma_ij: xx xy xz yy yz zz
    double sg;             // sqrt(det gamma)
    double gdd;            // gamma^{dd} for the sweep direction
};
// alp, beta, g already hold the two-point averages; completes sg and gdd.
template <int D>
GRX_HD void face_geom_complete(FaceGeom& m) {
    const double gxx = m.g[0], gxy = m.g[1], gxz = m.g[2], gyy = m.g[3], gyz = m.g[4], gzz = m.g[5];
    const double cxx = fma(gyy, gzz, -gyz * gyz);
    const double cxy = fma(gxz, gyz, -gxy * gzz);
    const double cxz = fma(gxy, gyz, -gxz * gyy);
    const double det = fma(gxx, cxx, fma(gxy, cxy, gxz * cxz));
    const double rs = rsqrt(det);
    m.sg = det * rs;
    const double cdd = (D == 0) ? cxx : (D == 1) ? fma(gxx, gzz, -gxz * gxz) : fma(gxx, gyy, -gxy * gxy);
    m.gdd = cdd * (rs * rs);
}

// ---- a3-a5: one side of a face: admissibility, conserved state, flux, fast speeds -------------------------
// P: reconstructed primitives of this side (replaced in place by the donor cell's centre values cen[q * nc] if the side
// takes the first-order fallback, R5).
// Returns U (Eqs. 6-9, l.88-94) and F^D (Eq. 12, l.108), both WITHOUT their common factor sqrt(gamma), and the two
// characteristic speeds (R8).
template <int D>
GRX_HD void side_state(double P[8], const double* __restrict__ cen, long long nc, const FaceGeom& m,
                       double gamma, double U[8], double F[8], double& lam_m, double& lam_p, unsigned& nfallback) {
    // P is the caller's array and is overwritten IN PLACE by the fallback (it is dead after the face): copying it into
    // conditionally reassigned locals cost 16 register moves per side on the common path.
    const double gxx = m.g[0], gxy = m.g[1], gxz = m.g[2], gyy = m.g[3], gyz = m.g[4], gzz = m.g[5];
    double vlx = fma(gxx, P[1], fma(gxy, P[2], gxz * P[3]));      // v_i = gamma_ij v^j
    double vly = fma(gxy, P[1], fma(gyy, P[2], gyz * P[3]));
    double vlz = fma(gxz, P[1], fma(gyz, P[2], gzz * P[3]));
    double v2 = fma(vlx, P[1], fma(vly, P[2], vlz * P[3]));
    if (!(P[0] > 0.0 && P[4] > 0.0 && v2 < V2MAX)) {          // R5; NaN fails the test
#pragma unroll
        for (int q = 0; q < 8; ++q) P[q] = cen[q * nc];
        vlx = fma(gxx, P[1], fma(gxy, P[2], gxz * P[3]));
        vly = fma(gxy, P[1], fma(gyy, P[2], gyz * P[3]));
        vlz = fma(gxz, P[1], fma(gyz, P[2], gzz * P[3]));
        v2 = fma(vlx, P[1], fma(vly, P[2], vlz * P[3]));
        ++nfallback;
    }
    const double rho = P[0], vx = P[1], vy = P[2], vz = P[3], eps = P[4];
    const double Bx = P[5], By = P[6], Bz = P[7];
    const double iW2 = 1.0 - v2;                             // 1/W^2
    const double W = rsqrt(iW2);                             // l.98
    const double iW = W * iW2;
    const double W2 = W * W;
    const double Blx = fma(gxx, Bx, fma(gxy, By, gxz * Bz));
    const double Bly = fma(gxy, Bx, fma(gyy, By, gyz * Bz));
    const double Blz = fma(gxz, Bx, fma(gyz, By, gzz * Bz));
    const double B2 = fma(Blx, Bx, fma(Bly, By, Blz * Bz));
    const double Bv = fma(Bx, vlx, fma(By, vly, Bz * vlz));
    const double ab0 = W * Bv;                               // alpha b^0
    const double b2 = fma(B2, iW2, Bv * Bv);                 // b^2
    const double blx = fma(Blx, iW, ab0 * vlx);              // b_i
    const double bly = fma(Bly, iW, ab0 * vly);
    const double blz = fma(Blz, iW, ab0 * vlz);
    const double rhoeps = rho * eps;
    const double p = (gamma - 1.0) * rhoeps;                 // l.138
    const double rhoh = fma(gamma, rhoeps, rho);             // rho (1 + eps) + p
    const double rhohs = rhoh + b2;                          // rho h*
    const double Ps = fma(0.5, b2, p);                       // P*
    const double X = rhohs * W2;
    // sqrt(gamma) is common to both sides of a face and to U and F: it is left out here (U, F are the
    // UNDENSITISED state and flux) and rides on the HLLE coefficients in face_flux.
    const double Dd = rho * W;                               // Eq. (6) / sqrt(gamma)
    const double Sx = fma(X, vlx, -ab0 * blx);               // Eq. (7) / sqrt(gamma)
    const double Sy = fma(X, vly, -ab0 * bly);
    const double Sz = fma(X, vlz, -ab0 * blz);
    const double tau = fma(-ab0, ab0, X - Ps) - Dd;          // Eq. (8) / sqrt(gamma)
    U[0] = Dd; U[1] = Sx; U[2] = Sy; U[3] = Sz; U[4] = tau; U[5] = Bx; U[6] = By; U[7] = Bz;   // Eq. (9)
    // flux, Eq. (12): vtilde^i = v^i - beta^i/alpha (l.114); everything carries one factor alpha
    const double alp = m.alp;
    const double avx = fma(alp, vx, -m.beta[0]);             // alpha vtilde^i
    const double avy = fma(alp, vy, -m.beta[1]);
    const double avz = fma(alp, vz, -m.beta[2]);
    const double vd = (D == 0) ? vx : (D == 1) ? vy : vz;
    const double avd = (D == 0) ? avx : (D == 1) ? avy : avz;
    const double Bd = (D == 0) ? Bx : (D == 1) ? By : Bz;
    const double aBdW = alp * Bd * iW;                       // alpha B^d / W
    const double aPs = alp * Ps;
    F[0] = Dd * avd;
    F[1] = fma(Sx, avd, -blx * aBdW);
    F[2] = fma(Sy, avd, -bly * aBdW);
    F[3] = fma(Sz, avd, -blz * aBdW);
    F[1 + D] += aPs;
    F[4] = fma(tau, avd, fma(aPs, vd, -ab0 * aBdW));
    F[5] = fma(Bx, avd, -Bd * avx);
    F[6] = fma(By, avd, -Bd * avy);
    F[7] = fma(Bz, avd, -Bd * avz);
    F[5 + D] = 0.0;
    // fast-magnetosonic speeds (R8).  With N = b^2 + Gamma p, M = rho h - Gamma p, rho h* = N + M:
    //   a^2 = N/(rho h*), 1 - a^2 = M/(rho h*), 1 - v^2 a^2 = Dn/(rho h*) with Dn = rho h* - v^2 N, so
    //   lambda^+- = alpha [v^d M +- sqrt(N (1 - v^2) (gamma^dd Dn - v^d v^d M))] / Dn - beta^d
    // (the factors 1/(rho h*) cancel: one reciprocal, one square root, no cancellation in 1 - a^2).
    const double gp = gamma * p;
    const double N = b2 + gp;
    const double M = rhoh - gp;
    const double Dn = fma(-v2, N, rhohs);
    const double iDn = rcp(Dn);
    const double disc = (N * iW2) * fma(m.gdd, Dn, -(vd * vd) * M);
    const double root = sqrt_nn(fmax(disc, 0.0));
    const double c0 = vd * M;
    const double ai = alp * iDn;
    const double bd = m.beta[D];
    lam_p = fma(ai, c0 + root, -bd);
    lam_m = fma(ai, c0 - root, -bd);
}

// ---- a6: HLLE flux of one face (l.131; R9) -----------------------------------------------------------------
// m holds the averaged alp, beta, g on entry; cenL/cenR point at field 0 of the two donor cells (field stride nc).
template <int D>
GRX_HD void face_flux(FaceGeom& m, double PL[8], double PR[8], const double* __restrict__ cenL,
                      const double* __restrict__ cenR, long long nc, double gamma, double Fh[8], unsigned& nfallback,
                      double scale = 1.0) {
    face_geom_complete<D>(m);
    double UL[8], FL[8], UR[8], FR[8], lmL, lpL, lmR, lpR;
    side_state<D>(PL, cenL, nc, m, gamma, UL, FL, lmL, lpL, nfallback);
    side_state<D>(PR, cenR, nc, m, gamma, UR, FR, lmR, lpR, nfallback);
    const double lm = fmin(0.0, fmin(lmL, lmR));
    const double lp = fmax(0.0, fmax(lpL, lpR));
    const double idl = rcp(lp - lm) * (scale * m.sg);   // 1/dx_d and sqrt(gamma) ride on the three HLLE coefficients
    const double cL = lp * idl, cR = -lm * idl, cU = lp * lm * idl;
#pragma unroll
    for (int c = 0; c < 8; ++c) Fh[c] = fma(cL, FL[c], fma(cR, FR[c], cU * (UR[c] - UL[c])));
}

// ---- a8: 4th-order centred first derivative, grouped so that a constant differentiates to exactly 0 (R12) ---
GRX_HD double d4(double mm2, double mm1, double mp1, double mp2, double inv12dx) {
    return fma(8.0, mp1 - mm1, -(mp2 - mm2)) * inv12dx;
}

// ---- a9: geometric sources of one cell, Eq. (13) (l.112) in 3+1 form (R12-R14) -------------------------------
// With the Eulerian-observer quantities  E = rho h* W^2 - P* - (alpha b^0)^2,  S_k = rho h* W^2 v_k - alpha b^0 b_k,
// S^{kl} = rho h* W^2 v^k v^l + P* gamma^{kl} - bb^k bb^l  (bb^k = B^k/W + alpha b^0 v^k)  Eq. (13) becomes
//   S_{S_j} = sqrt(gamma) [ alpha/2 S^{kl} d_j gamma_kl + S_k d_j beta^k - E d_j alpha ],
//   S_tau   = sqrt(gamma) [ alpha K_kl S^{kl} - S^k d_k alpha ],
// which is term by term the same as the T^{mu nu} form the oracle evaluates.
// P: cell-centre primitives; met: the 10 metric fields at the centre; K: K_ij; dm[j][f] = d_j of metric field f.
GRX_HD void sources_point(const double P[8], const double met[10], const double K[6], const double dm[3][10],
                          double gamma, double& SSx, double& SSy, double& SSz, double& Stau) {
    const double rho = P[0], vx = P[1], vy = P[2], vz = P[3], eps = P[4], Bx = P[5], By = P[6], Bz = P[7];
    const double alp = met[0];
    const double gxx = met[4], gxy = met[5], gxz = met[6], gyy = met[7], gyz = met[8], gzz = met[9];
    const double cxx = fma(gyy, gzz, -gyz * gyz);
    const double cxy = fma(gxz, gyz, -gxy * gzz);
    const double cxz = fma(gxy, gyz, -gxz * gyy);
    const double cyy = fma(gxx, gzz, -gxz * gxz);
    const double cyz = fma(gxy, gxz, -gxx * gyz);
    const double czz = fma(gxx, gyy, -gxy * gxy);
    const double det = fma(gxx, cxx, fma(gxy, cxy, gxz * cxz));
    const double rs = rsqrt(det);
    const double sg = det * rs, idet = rs * rs;
    const double vlx = fma(gxx, vx, fma(gxy, vy, gxz * vz));
    const double vly = fma(gxy, vx, fma(gyy, vy, gyz * vz));
    const double vlz = fma(gxz, vx, fma(gyz, vy, gzz * vz));
    const double v2 = fma(vlx, vx, fma(vly, vy, vlz * vz));
    const double iW2 = 1.0 - v2;
    const double W = rsqrt(iW2), iW = W * iW2, W2 = W * W;
    const double Blx = fma(gxx, Bx, fma(gxy, By, gxz * Bz));
    const double Bly = fma(gxy, Bx, fma(gyy, By, gyz * Bz));
    const double Blz = fma(gxz, Bx, fma(gyz, By, gzz * Bz));
    const double B2 = fma(Blx, Bx, fma(Bly, By, Blz * Bz));
    const double Bv = fma(Bx, vlx, fma(By, vly, Bz * vlz));
    const double ab0 = W * Bv;
    const double b2 = fma(B2, iW2, Bv * Bv);
    const double rhoeps = rho * eps;
    const double p = (gamma - 1.0) * rhoeps;
    const double rhohs = fma(gamma, rhoeps, rho) + b2;
    const double Ps = fma(0.5, b2, p);
    const double X = rhohs * W2;
    const double E = fma(-ab0, ab0, X - Ps);
    // bb^k (upper) and bb_k (lower), momentum density S_k (lower) and S^k (upper)
    const double bux = fma(Bx, iW, ab0 * vx), buy = fma(By, iW, ab0 * vy), buz = fma(Bz, iW, ab0 * vz);
    const double blx = fma(Blx, iW, ab0 * vlx), bly = fma(Bly, iW, ab0 * vly), blz = fma(Blz, iW, ab0 * vlz);
    const double Slx = fma(X, vlx, -ab0 * blx), Sly = fma(X, vly, -ab0 * bly), Slz = fma(X, vlz, -ab0 * blz);
    const double Sux = fma(X, vx, -ab0 * bux), Suy = fma(X, vy, -ab0 * buy), Suz = fma(X, vz, -ab0 * buz);
    // spatial stress S^{kl}
    const double Pi = Ps * idet;   // P* gamma^{kl} = P*/det * cofactor
    const double Xvx = X * vx, Xvy = X * vy, Xvz = X * vz;
    const double Sxx = fma(Xvx, vx, fma(Pi, cxx, -bux * bux));
    const double Sxy = fma(Xvx, vy, fma(Pi, cxy, -bux * buy));
    const double Sxz = fma(Xvx, vz, fma(Pi, cxz, -bux * buz));
    const double Syy = fma(Xvy, vy, fma(Pi, cyy, -buy * buy));
    const double Syz = fma(Xvy, vz, fma(Pi, cyz, -buy * buz));
    const double Szz = fma(Xvz, vz, fma(Pi, czz, -buz * buz));
    const double ha = 0.5 * alp;
    double SS[3];
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        const double* d = dm[j];
        // alpha/2 S^{kl} d_j gamma_kl  (off-diagonal terms count twice)
        const double sdg = fma(Sxx, d[4], fma(Syy, d[7], Szz * d[9])) * ha +
                           alp * fma(Sxy, d[5], fma(Sxz, d[6], Syz * d[8]));
        const double sdb = fma(Slx, d[1], fma(Sly, d[2], Slz * d[3]));
        SS[j] = sg * (sdg + fma(-E, d[0], sdb));
    }
    SSx = SS[0]; SSy = SS[1]; SSz = SS[2];
    const double KS = fma(K[0], Sxx, fma(K[3], Syy, K[5] * Szz)) + 2.0 * fma(K[1], Sxy, fma(K[2], Sxz, K[4] * Syz));
    const double Sda = fma(Sux, dm[0][0], fma(Suy, dm[1][0], Suz * dm[2][0]));
    Stau = sg * fma(alp, KS, -Sda);
}

// ---- a9 in pieces (same formulas as sources_point, arranged so that only one direction's ten metric
// derivatives are live at a time): the cell's Eulerian-observer stress-energy first, then one call per direction.
struct SrcState {
    double alp, sg;        // lapse, sqrt(det gamma)
    double E;              // rho h* W^2 - P* - (alpha b^0)^2
    double Sl[3], Su[3];   // S_k, S^k
    double S2[6];          // S^{kl}: xx xy xz yy yz zz
};
GRX_HD void sources_prepare(const double P[8], const double met[10], double gamma, SrcState& s) {
    const double rho = P[0], vx = P[1], vy = P[2], vz = P[3], eps = P[4], Bx = P[5], By = P[6], Bz = P[7];
    const double gxx = met[4], gxy = met[5], gxz = met[6], gyy = met[7], gyz = met[8], gzz = met[9];
    const double cxx = fma(gyy, gzz, -gyz * gyz);
    const double cxy = fma(gxz, gyz, -gxy * gzz);
    const double cxz = fma(gxy, gyz, -gxz * gyy);
    const double cyy = fma(gxx, gzz, -gxz * gxz);
    const double cyz = fma(gxy, gxz, -gxx * gyz);
    const double czz = fma(gxx, gyy, -gxy * gxy);
    const double det = fma(gxx, cxx, fma(gxy, cxy, gxz * cxz));
    const double rs = rsqrt(det);
    const double idet = rs * rs;
    const double vlx = fma(gxx, vx, fma(gxy, vy, gxz * vz));
    const double vly = fma(gxy, vx, fma(gyy, vy, gyz * vz));
    const double vlz = fma(gxz, vx, fma(gyz, vy, gzz * vz));
    const double v2 = fma(vlx, vx, fma(vly, vy, vlz * vz));
    const double iW2 = 1.0 - v2;
    const double W = rsqrt(iW2), iW = W * iW2, W2 = W * W;
    const double Blx = fma(gxx, Bx, fma(gxy, By, gxz * Bz));
    const double Bly = fma(gxy, Bx, fma(gyy, By, gyz * Bz));
    const double Blz = fma(gxz, Bx, fma(gyz, By, gzz * Bz));
    const double B2 = fma(Blx, Bx, fma(Bly, By, Blz * Bz));
    const double Bv = fma(Bx, vlx, fma(By, vly, Bz * vlz));
    const double ab0 = W * Bv;
    const double b2 = fma(B2, iW2, Bv * Bv);
    const double rhoeps = rho * eps;
    const double p = (gamma - 1.0) * rhoeps;
    const double rhohs = fma(gamma, rhoeps, rho) + b2;
    const double Ps = fma(0.5, b2, p);
    const double X = rhohs * W2;
    s.alp = met[0];
    s.sg = det * rs;
    s.E = fma(-ab0, ab0, X - Ps);
    const double bux = fma(Bx, iW, ab0 * vx), buy = fma(By, iW, ab0 * vy), buz = fma(Bz, iW, ab0 * vz);
    s.Sl[0] = fma(X, vlx, -ab0 * fma(Blx, iW, ab0 * vlx));
    s.Sl[1] = fma(X, vly, -ab0 * fma(Bly, iW, ab0 * vly));
    s.Sl[2] = fma(X, vlz, -ab0 * fma(Blz, iW, ab0 * vlz));
    s.Su[0] = fma(X, vx, -ab0 * bux);
    s.Su[1] = fma(X, vy, -ab0 * buy);
    s.Su[2] = fma(X, vz, -ab0 * buz);
    const double Pi = Ps * idet;   // P* gamma^{kl} = P*/det * cofactor
    const double Xvx = X * vx, Xvy = X * vy, Xvz = X * vz;
    s.S2[0] = fma(Xvx, vx, fma(Pi, cxx, -bux * bux));
    s.S2[1] = fma(Xvx, vy, fma(Pi, cxy, -bux * buy));
    s.S2[2] = fma(Xvx, vz, fma(Pi, cxz, -bux * buz));
    s.S2[3] = fma(Xvy, vy, fma(Pi, cyy, -buy * buy));
    s.S2[4] = fma(Xvy, vz, fma(Pi, cyz, -buy * buz));
    s.S2[5] = fma(Xvz, vz, fma(Pi, czz, -buz * buz));
}
// Direction j: d[f] = 8 (m_{+1} - m_{-1}) - (m_{+2} - m_{-2}) of metric field f along j (unscaled, R12),
// w = 1/(12 dx_j).  Returns S_{S_j} and adds -sqrt(gamma) S^j d_j alpha to Stau.
GRX_HD double sources_dir(const SrcState& s, int j, const double d[10], double w, double& Stau) {
    const double sdg = fma(s.S2[0], d[4], fma(s.S2[3], d[7], s.S2[5] * d[9])) * (0.5 * s.alp) +
                       s.alp * fma(s.S2[1], d[5], fma(s.S2[2], d[6], s.S2[4] * d[8]));
    const double sdb = fma(s.Sl[0], d[1], fma(s.Sl[1], d[2], s.Sl[2] * d[3]));
    const double sw = s.sg * w;
    Stau = fma(-sw * s.Su[j], d[0], Stau);
    return sw * (sdg + fma(-s.E, d[0], sdb));
}
// The extrinsic-curvature term of S_tau: sqrt(gamma) alpha K_kl S^{kl}.
GRX_HD double sources_K(const SrcState& s, const double K[6]) {
    const double KS = fma(K[0], s.S2[0], fma(K[3], s.S2[3], K[5] * s.S2[5])) +
                      2.0 * fma(K[1], s.S2[1], fma(K[2], s.S2[2], K[4] * s.S2[4]));
    return s.sg * s.alp * KS;
}
GRX_HD double d4raw(double mm2, double mm1, double mp1, double mp2) { return fma(8.0, mp1 - mm1, -(mp2 - mm2)); }

// ---- prim2con at one point with the full metric given (Eqs. 6-9) ----------------------------------------------
GRX_HD void prim2con_point(const double P[8], const double met[10], double gamma, double U[8]) {
    const double rho = P[0], vx = P[1], vy = P[2], vz = P[3], eps = P[4], Bx = P[5], By = P[6], Bz = P[7];
    const double gxx = met[4], gxy = met[5], gxz = met[6], gyy = met[7], gyz = met[8], gzz = met[9];
    const double cxx = fma(gyy, gzz, -gyz * gyz);
    const double cxy = fma(gxz, gyz, -gxy * gzz);
    const double cxz = fma(gxy, gyz, -gxz * gyy);
    const double det = fma(gxx, cxx, fma(gxy, cxy, gxz * cxz));
    const double sg = sqrt(det);
    const double vlx = fma(gxx, vx, fma(gxy, vy, gxz * vz));
    const double vly = fma(gxy, vx, fma(gyy, vy, gyz * vz));
    const double vlz = fma(gxz, vx, fma(gyz, vy, gzz * vz));
    const double v2 = fma(vlx, vx, fma(vly, vy, vlz * vz));
    const double iW2 = 1.0 - v2;
    const double W = 1.0 / sqrt(iW2), iW = W * iW2, W2 = W * W;
    const double Blx = fma(gxx, Bx, fma(gxy, By, gxz * Bz));
    const double Bly = fma(gxy, Bx, fma(gyy, By, gyz * Bz));
    const double Blz = fma(gxz, Bx, fma(gyz, By, gzz * Bz));
    const double B2 = fma(Blx, Bx, fma(Bly, By, Blz * Bz));
    const double Bv = fma(Bx, vlx, fma(By, vly, Bz * vlz));
    const double ab0 = W * Bv;
    const double b2 = fma(B2, iW2, Bv * Bv);
    const double rhoeps = rho * eps;
    const double p = (gamma - 1.0) * rhoeps;
    const double rhohs = fma(gamma, rhoeps, rho) + b2;
    const double Ps = fma(0.5, b2, p);
    const double X = rhohs * W2;
    const double Dd = sg * rho * W;
    U[0] = Dd;
    U[1] = sg * fma(X, vlx, -ab0 * fma(Blx, iW, ab0 * vlx));
    U[2] = sg * fma(X, vly, -ab0 * fma(Bly, iW, ab0 * vly));
    U[3] = sg * fma(X, vlz, -ab0 * fma(Blz, iW, ab0 * vlz));
    U[4] = fma(sg, fma(-ab0, ab0, X - Ps), -Dd);
    U[5] = sg * Bx; U[6] = sg * By; U[7] = sg * Bz;
}

// ---- support (R22): Gamma-law con2prim at one point, Newton on z = rho h W^2 ----------------------------------
// f(z) = z + B^2 - p(z) - B^2/(2 W^2) - (S.B)^2/(2 z^2) - (tau + D) on the undensitised conserved variables, with
// v^2(z) = [S^2 z^2 + (S.B)^2 (B^2 + 2z)] / [(z + B^2)^2 z^2].
struct C2P {
    double Dd, E, S2, B2, SB, SB2, gamma;
    double Su[3], B[3];
    double W, rho, p;    // of the last eval
    GRX_HD double eval(double z) {
        double v2 = (S2 * z * z + SB2 * (B2 + 2.0 * z)) / ((z + B2) * (z + B2) * z * z);
        if (v2 > 1.0 - 1e-15) v2 = 1.0 - 1e-15;
        W = 1.0 / sqrt(1.0 - v2);
        rho = Dd / W;
        p = (gamma - 1.0) / gamma * (z / (W * W) - rho);
        return z + B2 - p - B2 / (2.0 * W * W) - SB2 / (2.0 * z * z) - E;
    }
};
GRX_HD void con2prim_setup(const double U[8], const double met[10], double gamma, C2P& s) {
    const double gxx = met[4], gxy = met[5], gxz = met[6], gyy = met[7], gyz = met[8], gzz = met[9];
    const double cxx = fma(gyy, gzz, -gyz * gyz);
    const double cxy = fma(gxz, gyz, -gxy * gzz);
    const double cxz = fma(gxy, gyz, -gxz * gyy);
    const double cyy = fma(gxx, gzz, -gxz * gxz);
    const double cyz = fma(gxy, gxz, -gxx * gyz);
    const double czz = fma(gxx, gyy, -gxy * gxy);
    const double det = fma(gxx, cxx, fma(gxy, cxy, gxz * cxz));
    const double isg = 1.0 / sqrt(det), idet = 1.0 / det;
    s.Dd = U[0] * isg;
    const double tau = U[4] * isg;
    const double Slx = U[1] * isg, Sly = U[2] * isg, Slz = U[3] * isg;
    s.B[0] = U[5] * isg; s.B[1] = U[6] * isg; s.B[2] = U[7] * isg;
    s.Su[0] = (cxx * Slx + cxy * Sly + cxz * Slz) * idet;
    s.Su[1] = (cxy * Slx + cyy * Sly + cyz * Slz) * idet;
    s.Su[2] = (cxz * Slx + cyz * Sly + czz * Slz) * idet;
    const double Blx = gxx * s.B[0] + gxy * s.B[1] + gxz * s.B[2];
    const double Bly = gxy * s.B[0] + gyy * s.B[1] + gyz * s.B[2];
    const double Blz = gxz * s.B[0] + gyz * s.B[1] + gzz * s.B[2];
    s.S2 = Slx * s.Su[0] + Sly * s.Su[1] + Slz * s.Su[2];
    s.B2 = Blx * s.B[0] + Bly * s.B[1] + Blz * s.B[2];
    s.SB = Slx * s.B[0] + Sly * s.B[1] + Slz * s.B[2];
    s.SB2 = s.SB * s.SB;
    s.E = tau + s.Dd;
    s.gamma = gamma;
    s.W = 1.0; s.rho = s.Dd; s.p = 0.0;
}
GRX_HD void con2prim_finish(C2P& s, double z, double P[8]) {
    s.eval(z);
    P[0] = s.rho;
    const double iz = 1.0 / z, izb = 1.0 / (z + s.B2);
    P[1] = (s.Su[0] + s.SB * s.B[0] * iz) * izb;
    P[2] = (s.Su[1] + s.SB * s.B[1] * iz) * izb;
    P[3] = (s.Su[2] + s.SB * s.B[2] * iz) * izb;
    P[4] = s.p / ((s.gamma - 1.0) * s.rho);
    P[5] = s.B[0]; P[6] = s.B[1]; P[7] = s.B[2];
}
// Bracketed solve: grow / shrink a bracket from 2 (E + 1), then Newton with a central-difference slope, bisecting whenever
// a step leaves the bracket.  Returns 0 on convergence (|dz| < 1e-14 z), 1 otherwise.
GRX_HD int con2prim_solve_bracket(C2P& s, double& zout) {
    double zhi = fmax(2.0 * (s.E + 1.0), 1.0);
    for (int it = 0; it < 200 && s.eval(zhi) < 0.0; ++it) zhi *= 2.0;
    double zlo = zhi;
    for (int it = 0; it < 400 && s.eval(zlo) > 0.0; ++it) zlo *= 0.5;
    double z = 0.5 * (zlo + zhi);
    int status = 1;
    for (int it = 0; it < 200; ++it) {
        const double f = s.eval(z);
        if (f > 0.0) zhi = z; else zlo = z;
        const double h = 1e-6 * z;
        const double fp = (s.eval(z + h) - s.eval(z - h)) / (2.0 * h);
        double zn = z - f / fp;
        if (!(zn > zlo && zn < zhi)) zn = 0.5 * (zlo + zhi);
        const double dz = fabs(zn - z);
        z = zn;
        if (dz < 1e-14 * z) { status = 0; break; }
    }
    zout = z;
    return status;
}
// Warm-started solve for time stepping: the old state's z = rho h W^2 is within a time step of the root, so one Newton
// step with a central-difference slope followed by secant steps (one evaluation each) reaches |dz| < 1e-14 z in a handful of
// evaluations.  Returns 0 on convergence; anything else (no convergence in 12 steps, a step to z <= 0 or NaN) makes the
// caller take the bracketed solve.
GRX_HD int con2prim_solve_warm(C2P& s, double z0, double& zout) {
    if (!(z0 > 0.0)) return 1;
    double z = z0, f0 = s.eval(z);
    const double h = 1e-6 * z;
    double slope = (s.eval(z + h) - s.eval(z - h)) / (2.0 * h);
    for (int it = 0; it < 12; ++it) {
        const double zn = z - f0 / slope;
        if (!(zn > 0.0)) return 1;
        const double dz = fabs(zn - z);
        if (dz < 1e-14 * zn) { zout = zn; return 0; }
        const double f1 = s.eval(zn);
        const double sl = (f1 - f0) / (zn - z);
        if (sl > 0.0) slope = sl;      // f is increasing at the root: a secant slope of the wrong sign is rounding noise
        z = zn;
        f0 = f1;
    }
    return 1;
}
// Returns 0 on convergence, 1 otherwise.
GRX_HD int con2prim_point(const double U[8], const double met[10], double gamma, double P[8]) {
    C2P s;
    con2prim_setup(U, met, gamma, s);
    double z;
    const int status = con2prim_solve_bracket(s, z);
    con2prim_finish(s, z, P);
    return status;
}
// Pold: the primitives of the same cell at the previous stage (the warm start); falls back to the bracketed solve.
GRX_HD int con2prim_point_warm(const double U[8], const double met[10], double gamma, const double Pold[8], double P[8]) {
    C2P s;
    con2prim_setup(U, met, gamma, s);
    // z of the old state: rho h W^2 with v^2 = gamma_ij v^i v^j
    const double gxx = met[4], gxy = met[5], gxz = met[6], gyy = met[7], gyz = met[8], gzz = met[9];
    const double vx = Pold[1], vy = Pold[2], vz = Pold[3];
    const double v2 = vx * (gxx * vx + gxy * vy + gxz * vz) + vy * (gxy * vx + gyy * vy + gyz * vz) +
                      vz * (gxz * vx + gyz * vy + gzz * vz);
    const double z0 = Pold[0] * (1.0 + gamma * Pold[4]) / (1.0 - v2);
    double z;
    int status = con2prim_solve_warm(s, z0, z);
    if (status) status = con2prim_solve_bracket(s, z);
    con2prim_finish(s, z, P);
    return status;
}

}  // namespace grx
