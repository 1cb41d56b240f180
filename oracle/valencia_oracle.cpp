// valencia_oracle.cpp -- CPU ORACLE for the FP64 Valencia GRMHD right-hand side.
//
// THIS FILE IS TEST INFRASTRUCTURE.  It is the plain, slow, obviously-correct statement of what
// the hot path computes, written from the paper (GRaM-X, arxiv 2210.17509; citations are
// PAPER.md line numbers + equation) and from the readings R1..R29 listed in DESIGN.md.  Only
// tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call
// it.  It shares no code, header, table or constant generator with the CUDA path
// (paper_2210_17509_b200/csrc) and neither includes the other.
//
// Parity pins: every exported function below is pinned by tests/test_oracle_pins*.py against
// closed forms, invariants and the paper's printed Balsara-1 values (tests/golden/).  Conventions
// that no external value can pin -- WENO_EPS, V2MAX, the fast-speed approximation a^2 (R8), the MC
// limiter and the choice of flux-CT among the constrained-transport schemes (R30; its defining
// properties are pinned) -- are listed as "parity unpinned (convention)" in DESIGN.md.
//
// No blocking, fusion or re-ordering beyond what the algorithm states: per direction, per grid
// line: reconstruct (O2) -> face metric (O1) -> admissibility (O3) -> state (O4) -> flux (O5)
// -> wave speeds (O6) -> HLLE (O7) -> divergence; then derivatives (O8) and sources (O9).
//
// The whole algorithm is templated on the scalar type `R`:
//   double       -- THE oracle
//   long double  -- adjudicator (quantifies the oracle's own rounding, pin P18)
//   Counted      -- a double that counts its operations (official algorithmic flop count)
//
// Build: g++ -O2 -fopenmp -ffp-contract=off -fno-fast-math -shared -fPIC (see oracle/build.py).

#include <cmath>
#include <cstddef>
#include <cstring>
#include <type_traits>
#include <vector>

namespace {

// ---- conventions (R4, R5): compile-time constants -------------------------------------------
constexpr double WENO_EPS = 1e-26;       // R4: Jiang-Shu epsilon
constexpr double V2MAX    = 1.0 - 1e-4;  // R5: admissibility bound on v^2 (W_max = 100)

enum { RECON_MINMOD = 0, RECON_MC = 1, RECON_WENO5 = 2 };

// symmetric 3x3 storage: xx xy xz yy yz zz
constexpr int SYM[3][3] = {{0, 1, 2}, {1, 3, 4}, {2, 4, 5}};

// ---- operation-counting scalar ----------------------------------------------------------------
struct OpCount { unsigned long long add, mul, div, sqrt; };
thread_local OpCount t_ops = {0, 0, 0, 0};

struct Counted {
    double v;
    Counted() : v(0.0) {}
    Counted(double x) : v(x) {}
};
inline Counted operator+(Counted a, Counted b) { ++t_ops.add; return Counted(a.v + b.v); }
inline Counted operator-(Counted a, Counted b) { ++t_ops.add; return Counted(a.v - b.v); }
inline Counted operator*(Counted a, Counted b) { ++t_ops.mul; return Counted(a.v * b.v); }
inline Counted operator/(Counted a, Counted b) { ++t_ops.div; return Counted(a.v / b.v); }
inline Counted operator-(Counted a) { return Counted(-a.v); }   // sign flip: free
inline Counted& operator+=(Counted& a, Counted b) { a = a + b; return a; }
inline Counted& operator-=(Counted& a, Counted b) { a = a - b; return a; }
inline bool operator>(Counted a, Counted b) { return a.v > b.v; }
inline bool operator<(Counted a, Counted b) { return a.v < b.v; }
inline bool operator<=(Counted a, Counted b) { return a.v <= b.v; }
inline bool operator>=(Counted a, Counted b) { return a.v >= b.v; }

inline double      o_sqrt(double x) { return std::sqrt(x); }
inline long double o_sqrt(long double x) { return sqrtl(x); }
inline Counted     o_sqrt(Counted x) { ++t_ops.sqrt; return Counted(std::sqrt(x.v)); }
inline double      o_abs(double x) { return std::fabs(x); }
inline long double o_abs(long double x) { return fabsl(x); }
inline Counted     o_abs(Counted x) { return Counted(std::fabs(x.v)); }
inline double      to_double(double x) { return x; }
inline double      to_double(long double x) { return (double)x; }
inline double      to_double(Counted x) { return x.v; }

template <class R> inline R o_min(R a, R b) { return (b < a) ? b : a; }
template <class R> inline R o_max(R a, R b) { return (b > a) ? b : a; }

// ---- O2: reconstruction of one cell (refs [31],[32]) ---------------------
// Input: the five cell values (a,b,c,d,e) = (q_{i-2}, q_{i-1}, q_i, q_{i+1}, q_{i+2}).
// Output: qm = value at face i-1/2 taken from cell i;  qp = value at face i+1/2 taken from cell i.

// TVD, minmod slope (l.255 "TVD reconstruction with the minmod limiter"; R3)
template <class R> void recon_minmod(R b, R c, R d, R& qm, R& qp) {
    R dm = c - b, dp = d - c;
    R sigma = R(0.0);
    if (dm * dp > R(0.0)) {
        R m = o_min(o_abs(dm), o_abs(dp));
        sigma = (dm > R(0.0)) ? m : -m;
    }
    qm = c - R(0.5) * sigma;
    qp = c + R(0.5) * sigma;
}

// TVD, monotonised-central slope (north_star only; R3)
template <class R> void recon_mc(R b, R c, R d, R& qm, R& qp) {
    R dm = c - b, dp = d - c;
    R sigma = R(0.0);
    if (dm * dp > R(0.0)) {
        R m = o_min(o_min(R(2.0) * o_abs(dm), R(2.0) * o_abs(dp)), R(0.5) * o_abs(dm + dp));
        sigma = (dm > R(0.0)) ? m : -m;
    }
    qm = c - R(0.5) * sigma;
    qp = c + R(0.5) * sigma;
}

// WENO5, Jiang-Shu (ref [32] = Shu 1998; R4).  The three smoothness indicators belong to the cell
// and are shared by its two faces (the mirrored stencil has beta0 <-> beta2).
template <class R> R weno5_combine(R p0, R p1, R p2, R b0, R b1, R b2) {
    R e0 = R(WENO_EPS) + b0, e1 = R(WENO_EPS) + b1, e2 = R(WENO_EPS) + b2;
    R a0 = R(0.1) / (e0 * e0);
    R a1 = R(0.6) / (e1 * e1);
    R a2 = R(0.3) / (e2 * e2);
    return (a0 * p0 + a1 * p1 + a2 * p2) / (a0 + a1 + a2);
}
template <class R> void recon_weno5(R a, R b, R c, R d, R e, R& qm, R& qp) {
    R t;
    t = a - R(2.0) * b + c;              R b0 = R(13.0 / 12.0) * t * t;
    t = a - R(4.0) * b + R(3.0) * c;     b0 = b0 + R(0.25) * t * t;
    t = b - R(2.0) * c + d;              R b1 = R(13.0 / 12.0) * t * t;
    t = b - d;                           b1 = b1 + R(0.25) * t * t;
    t = c - R(2.0) * d + e;              R b2 = R(13.0 / 12.0) * t * t;
    t = R(3.0) * c - R(4.0) * d + e;     b2 = b2 + R(0.25) * t * t;
    // q^+_i : stencil (a,b,c,d,e)
    R p0 = (R(2.0) * a - R(7.0) * b + R(11.0) * c) / R(6.0);
    R p1 = (-b + R(5.0) * c + R(2.0) * d) / R(6.0);
    R p2 = (R(2.0) * c + R(5.0) * d - e) / R(6.0);
    qp = weno5_combine(p0, p1, p2, b0, b1, b2);
    // q^-_i : same formula on the mirrored stencil (e,d,c,b,a); its indicators are (b2,b1,b0)
    R m0 = (R(2.0) * e - R(7.0) * d + R(11.0) * c) / R(6.0);
    R m1 = (-d + R(5.0) * c + R(2.0) * b) / R(6.0);
    R m2 = (R(2.0) * c + R(5.0) * b - a) / R(6.0);
    qm = weno5_combine(m0, m1, m2, b2, b1, b0);
}
template <class R> void recon_cell(int recon, R a, R b, R c, R d, R e, R& qm, R& qp) {
    if (recon == RECON_WENO5) recon_weno5(a, b, c, d, e, qm, qp);
    else if (recon == RECON_MC) recon_mc(b, c, d, qm, qp);
    else recon_minmod(b, c, d, qm, qp);
}

// ---- metric at a point (face or centre) -----------------------------------------------------------
template <class R> struct Metric {
    R alp, beta[3], g[6];   // lapse, shift beta^i, gamma_ij
    R det, sqrtg;           // det(gamma_ij), sqrt of it
    R gu[6];                // inverse gamma^{ij}
};
// determinant by cofactor expansion, inverse = cofactor/det (O1)
template <class R> void metric_complete(Metric<R>& m) {
    const R gxx = m.g[0], gxy = m.g[1], gxz = m.g[2], gyy = m.g[3], gyz = m.g[4], gzz = m.g[5];
    R cxx = gyy * gzz - gyz * gyz;
    R cxy = gxz * gyz - gxy * gzz;
    R cxz = gxy * gyz - gxz * gyy;
    R cyy = gxx * gzz - gxz * gxz;
    R cyz = gxy * gxz - gxx * gyz;
    R czz = gxx * gyy - gxy * gxy;
    m.det = gxx * cxx + gxy * cxy + gxz * cxz;
    m.sqrtg = o_sqrt(m.det);
    m.gu[0] = cxx / m.det; m.gu[1] = cxy / m.det; m.gu[2] = cxz / m.det;
    m.gu[3] = cyy / m.det; m.gu[4] = cyz / m.det; m.gu[5] = czz / m.det;
}
// face metric along d needs only det, sqrt(gamma) and gamma^{dd} (O1)
template <class R> void metric_complete_face(Metric<R>& m, int d) {
    const R gxx = m.g[0], gxy = m.g[1], gxz = m.g[2], gyy = m.g[3], gyz = m.g[4], gzz = m.g[5];
    R cxx = gyy * gzz - gyz * gyz;
    R cxy = gxz * gyz - gxy * gzz;
    R cxz = gxy * gyz - gxz * gyy;
    m.det = gxx * cxx + gxy * cxy + gxz * cxz;
    m.sqrtg = o_sqrt(m.det);
    R cdd = (d == 0) ? cxx : (d == 1) ? gxx * gzz - gxz * gxz : gxx * gyy - gxy * gxy;
    m.gu[SYM[d][d]] = cdd / m.det;
}
template <class R> inline R lower(const Metric<R>& m, const R v[3], int i) {
    return m.g[SYM[i][0]] * v[0] + m.g[SYM[i][1]] * v[1] + m.g[SYM[i][2]] * v[2];
}

// ---- O3: admissibility of a reconstructed state (R5).  Written so NaN fails it. ---------------------
template <class R> bool admissible(const R P[8], const Metric<R>& m) {
    const R v[3] = {P[1], P[2], P[3]};
    R v2 = lower(m, v, 0) * v[0] + lower(m, v, 1) * v[1] + lower(m, v, 2) * v[2];
    return (P[0] > R(0.0)) && (P[4] > R(0.0)) && (v2 < R(V2MAX));
}

// ---- O4: primitive -> conserved, Eqs. (6)-(10) ------------------------------------
// Also returns the scalars the flux, the wave speeds and the sources reuse.
template <class R> struct State {
    R vl[3], v2, W, Bl[3], B2, Bv, ab0, b2, bl[3], p, rhoh, rhohs, Ps;
    R U[8];   // D, S_x, S_y, S_z, tau, calB^x, calB^y, calB^z
};
template <class R> void prim2con_point(const R P[8], const Metric<R>& m, R gamma, State<R>& s) {
    const R rho = P[0], eps = P[4];
    const R v[3] = {P[1], P[2], P[3]};
    const R B[3] = {P[5], P[6], P[7]};
    for (int i = 0; i < 3; ++i) s.vl[i] = lower(m, v, i);                     // v_i = gamma_ij v^j
    s.v2 = s.vl[0] * v[0] + s.vl[1] * v[1] + s.vl[2] * v[2];
    s.W = R(1.0) / o_sqrt(R(1.0) - s.v2);                                      // l.98
    for (int i = 0; i < 3; ++i) s.Bl[i] = lower(m, B, i);
    s.B2 = s.Bl[0] * B[0] + s.Bl[1] * B[1] + s.Bl[2] * B[2];
    s.Bv = s.Bl[0] * v[0] + s.Bl[1] * v[1] + s.Bl[2] * v[2];
    s.ab0 = s.W * s.Bv;                                                        // alpha b^0
    s.b2 = s.B2 / (s.W * s.W) + s.Bv * s.Bv;                                   // b^2
    for (int i = 0; i < 3; ++i) s.bl[i] = s.Bl[i] / s.W + s.ab0 * s.vl[i];     // b_i
    s.p = (gamma - R(1.0)) * rho * eps;                                        // l.138 Gamma-law
    s.rhoh = rho * (R(1.0) + eps) + s.p;                                       // rho h
    s.rhohs = s.rhoh + s.b2;                                                   // rho h*   (Eq. 5)
    s.Ps = s.p + R(0.5) * s.b2;                                                // P*
    const R W2 = s.W * s.W;
    s.U[0] = m.sqrtg * rho * s.W;                                              // Eq. (6)
    for (int j = 0; j < 3; ++j)
        s.U[1 + j] = m.sqrtg * (s.rhohs * W2 * s.vl[j] - s.ab0 * s.bl[j]);     // Eq. (7)
    s.U[4] = m.sqrtg * (s.rhohs * W2 - s.Ps - s.ab0 * s.ab0) - s.U[0];         // Eq. (8)
    for (int k = 0; k < 3; ++k) s.U[5 + k] = m.sqrtg * B[k];                   // Eq. (9)
}

// ---- O5: physical flux along d, Eq. (12) (l.108), vtilde^i = v^i - beta^i/alpha (l.114) -----------------
template <class R> void flux_point(const R P[8], const Metric<R>& m, const State<R>& s, int d, R F[8]) {
    const R v[3] = {P[1], P[2], P[3]};
    R vt[3];
    for (int i = 0; i < 3; ++i) vt[i] = v[i] - m.beta[i] / m.alp;
    const R sgPs = m.sqrtg * s.Ps;
    const R Bd_W = s.U[5 + d] / s.W;                                           // calB^d / W
    F[0] = m.alp * (s.U[0] * vt[d]);
    for (int j = 0; j < 3; ++j) {
        R t = s.U[1 + j] * vt[d] - s.bl[j] * Bd_W;
        if (j == d) t = t + sgPs;
        F[1 + j] = m.alp * t;
    }
    F[4] = m.alp * (s.U[4] * vt[d] + sgPs * v[d] - s.ab0 * Bd_W);
    for (int k = 0; k < 3; ++k) F[5 + k] = m.alp * (s.U[5 + k] * vt[d] - s.U[5 + d] * vt[k]);
}

// ---- O6: fast-magnetosonic characteristic speeds along d (R8) ------------------------------------------
template <class R>
void wavespeeds_point(const R P[8], const Metric<R>& m, const State<R>& s, int d, R gamma, R& lam_m, R& lam_p) {
    const R vd = P[1 + d];
    R cs2 = gamma * s.p / s.rhoh;
    R va2 = s.b2 / s.rhohs;
    R a2 = cs2 + va2 - cs2 * va2;
    R one_v2a2 = R(1.0) - s.v2 * a2;
    R disc = a2 * (R(1.0) - s.v2) * (m.gu[SYM[d][d]] * one_v2a2 - vd * vd * (R(1.0) - a2));
    if (!(disc > R(0.0))) disc = R(0.0);
    R root = o_sqrt(disc);
    lam_p = m.alp * (vd * (R(1.0) - a2) + root) / one_v2a2 - m.beta[d];
    lam_m = m.alp * (vd * (R(1.0) - a2) - root) / one_v2a2 - m.beta[d];
}

// ---- O7: HLLE flux (refs [33-35]; R9) -----------------------------------------------------------------------
template <class R>
void hlle(const R UL[8], const R FL[8], R lmL, R lpL, const R UR[8], const R FR[8], R lmR, R lpR, R Fh[8]) {
    R lm = o_min(R(0.0), o_min(lmL, lmR));
    R lp = o_max(R(0.0), o_max(lpL, lpR));
    for (int c = 0; c < 8; ++c)
        Fh[c] = (lp * FL[c] - lm * FR[c] + lp * lm * (UR[c] - UL[c])) / (lp - lm);
}

// One interface: metric already averaged to the face (alp, beta, g filled), reconstructed left and
// right primitive states PL/PR and the centre values CL/CR of their donor cells (O3 fallback).
template <class R>
void face_flux(Metric<R>& mf, int d, R gamma, const R PLin[8], const R PRin[8], const R CL[8], const R CR[8],
               R Fh[8], unsigned long long* nfallback) {
    metric_complete_face(mf, d);
    R PL[8], PR[8];
    bool okL = admissible(PLin, mf), okR = admissible(PRin, mf);
    for (int q = 0; q < 8; ++q) { PL[q] = okL ? PLin[q] : CL[q]; PR[q] = okR ? PRin[q] : CR[q]; }
    if (nfallback) *nfallback += (okL ? 0 : 1) + (okR ? 0 : 1);
    State<R> sL, sR;
    R FL[8], FR[8], lmL, lpL, lmR, lpR;
    prim2con_point(PL, mf, gamma, sL); flux_point(PL, mf, sL, d, FL); wavespeeds_point(PL, mf, sL, d, gamma, lmL, lpL);
    prim2con_point(PR, mf, gamma, sR); flux_point(PR, mf, sR, d, FR); wavespeeds_point(PR, mf, sR, d, gamma, lmR, lpR);
    hlle(sL.U, FL, lmL, lpL, sR.U, FR, lmR, lpR, Fh);
}

// ---- O9: geometric sources at a cell centre, Eq. (13) (l.112) in 3+1 form (R12-R14) -------------------
// dm[j][f] = d/dx^j of metric field f (f: alp, betax, betay, betaz, gxx, gxy, gxz, gyy, gyz, gzz).
template <class R>
void sources_point(const R P[8], Metric<R>& m, const R K[6], const R dm[3][10], R gamma, R S[8]) {
    metric_complete(m);
    State<R> s;
    prim2con_point(P, m, gamma, s);
    const R v[3] = {P[1], P[2], P[3]};
    const R B[3] = {P[5], P[6], P[7]};
    const R alp = m.alp;
    const R W2 = s.W * s.W;
    R vt[3], bu[3];
    for (int i = 0; i < 3; ++i) vt[i] = v[i] - m.beta[i] / alp;
    for (int i = 0; i < 3; ++i) bu[i] = B[i] / s.W + s.ab0 * vt[i];            // b^i
    // stress-energy tensor, Eq. (5) with u^0 = W/alpha, u^i = W vtilde^i, g^{mu nu} of the 3+1 split
    R T00 = (s.rhohs * W2 - s.Ps - s.ab0 * s.ab0) / (alp * alp);
    R T0[3], T[3][3], T0l[3], betal[3];
    for (int i = 0; i < 3; ++i)
        T0[i] = s.rhohs * W2 * vt[i] / alp + s.Ps * m.beta[i] / (alp * alp) - s.ab0 * bu[i] / alp;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j)
            T[i][j] = s.rhohs * W2 * vt[i] * vt[j] + s.Ps * (m.gu[SYM[i][j]] - m.beta[i] * m.beta[j] / (alp * alp)) -
                      bu[i] * bu[j];
    for (int k = 0; k < 3; ++k) betal[k] = lower(m, m.beta, k);
    for (int k = 0; k < 3; ++k)
        T0l[k] = betal[k] * T00 + m.g[SYM[k][0]] * T0[0] + m.g[SYM[k][1]] * T0[1] + m.g[SYM[k][2]] * T0[2];
    for (int c = 0; c < 8; ++c) S[c] = R(0.0);
    const R pref = alp * m.sqrtg;
    // momentum sources
    for (int j = 0; j < 3; ++j) {
        const R da = dm[j][0];
        R bbdg = R(0.0), t0bdg = R(0.0), tdg = R(0.0), t0ldb = R(0.0);
        for (int k = 0; k < 3; ++k)
            for (int l = 0; l < 3; ++l) {
                const R dg = dm[j][4 + SYM[k][l]];
                bbdg = bbdg + m.beta[k] * m.beta[l] * dg;
                t0bdg = t0bdg + T0[k] * m.beta[l] * dg;
                tdg = tdg + T[k][l] * dg;
            }
        for (int k = 0; k < 3; ++k) t0ldb = t0ldb + T0l[k] * dm[j][1 + k];
        S[1 + j] = pref * (T00 * (R(0.5) * bbdg - alp * da) + t0bdg + t0ldb + R(0.5) * tdg);
    }
    // energy source
    R bbK = R(0.0), tK = R(0.0), bda = R(0.0), t0term = R(0.0);
    for (int i = 0; i < 3; ++i) {
        R bK = R(0.0);
        for (int j = 0; j < 3; ++j) {
            bbK = bbK + m.beta[i] * m.beta[j] * K[SYM[i][j]];
            tK = tK + T[i][j] * K[SYM[i][j]];
            bK = bK + m.beta[j] * K[SYM[i][j]];
        }
        bda = bda + m.beta[i] * dm[i][0];
        t0term = t0term + T0[i] * (R(2.0) * bK - dm[i][0]);
    }
    S[4] = pref * (T00 * (bbK - bda) + t0term + tK);
}

// ---- whole right-hand side of one box ------------------------------------------------------------------------
struct Grid {
    int n[3], g, N[3];
    size_t ncell;
    size_t idx(int i, int j, int k) const {
        return (size_t)(i + g) + (size_t)N[0] * ((size_t)(j + g) + (size_t)N[1] * (size_t)(k + g));
    }
};

template <class R>
void rhs_box(const Grid& G, const double* prim, const double* met, const double* Kc, const double dx[3], int recon,
             double gamma_d, double* out, unsigned long long* fallback_total) {
    const R gamma = R(gamma_d);
    const size_t NC = G.ncell;
    unsigned long long nfb_all = 0;
    OpCount ops_all = {0, 0, 0, 0};

    // accumulator in the working precision R (for R = double it is `out` itself); interior cells start
    // from zero; ghost cells of `out` are never touched (R23)
    std::vector<R> acc_store;
    R* acc;
    if constexpr (std::is_same<R, double>::value) {
        acc = out;
    } else {
        acc_store.assign(8 * NC, R(0.0));
        acc = acc_store.data();
    }
    for (int c = 0; c < 8; ++c)
        for (int k = 0; k < G.n[2]; ++k)
            for (int j = 0; j < G.n[1]; ++j)
                for (int i = 0; i < G.n[0]; ++i) acc[c * NC + G.idx(i, j, k)] = R(0.0);

    // per direction: lines along d
    for (int d = 0; d < 3; ++d) {
        const int d1 = (d + 1) % 3, d2 = (d + 2) % 3;
        const int nd = G.n[d];
        const long nlines = (long)G.n[d1] * G.n[d2];
#pragma omp parallel
        {
            unsigned long long nfb = 0;
            std::vector<R> qm(8 * (size_t)(nd + 2)), qp(8 * (size_t)(nd + 2)), Fh(8 * (size_t)(nd + 1));
#pragma omp for schedule(static)
            for (long line = 0; line < nlines; ++line) {
                int ijk[3];
                ijk[d1] = (int)(line % G.n[d1]);
                ijk[d2] = (int)(line / G.n[d1]);
                auto at = [&](int s) {   // index of cell s along the line
                    int c3[3] = {ijk[0], ijk[1], ijk[2]};
                    c3[d] = s;
                    return G.idx(c3[0], c3[1], c3[2]);
                };
                // O2: reconstruct cells -1 .. nd
                for (int s = -1; s <= nd; ++s)
                    for (int q = 0; q < 8; ++q) {
                        const double* f = prim + q * NC;
                        R a = (recon == RECON_WENO5) ? R(f[at(s - 2)]) : R(0.0);
                        R e = (recon == RECON_WENO5) ? R(f[at(s + 2)]) : R(0.0);
                        recon_cell<R>(recon, a, R(f[at(s - 1)]), R(f[at(s)]), R(f[at(s + 1)]), e,
                                      qm[q * (nd + 2) + s + 1], qp[q * (nd + 2) + s + 1]);
                    }
                // faces f = 0 .. nd between cells f-1 and f
                for (int f = 0; f <= nd; ++f) {
                    const size_t iL = at(f - 1), iR = at(f);
                    Metric<R> mf;
                    mf.alp = R(0.5) * (R(met[0 * NC + iL]) + R(met[0 * NC + iR]));                       // O1
                    for (int i = 0; i < 3; ++i)
                        mf.beta[i] = R(0.5) * (R(met[(1 + i) * NC + iL]) + R(met[(1 + i) * NC + iR]));
                    for (int c = 0; c < 6; ++c)
                        mf.g[c] = R(0.5) * (R(met[(4 + c) * NC + iL]) + R(met[(4 + c) * NC + iR]));
                    R PL[8], PR[8], CL[8], CR[8];
                    for (int q = 0; q < 8; ++q) {
                        PL[q] = qp[q * (nd + 2) + f];       // q^+ of cell f-1
                        PR[q] = qm[q * (nd + 2) + f + 1];   // q^- of cell f
                        CL[q] = R(prim[q * NC + iL]);
                        CR[q] = R(prim[q * NC + iR]);
                    }
                    face_flux(mf, d, gamma, PL, PR, CL, CR, &Fh[8 * (size_t)f], &nfb);
                }
                // O7: out -= (F_{f+1} - F_f)/dx_d
                for (int s = 0; s < nd; ++s)
                    for (int c = 0; c < 8; ++c) {
                        R div = (Fh[8 * (size_t)(s + 1) + c] - Fh[8 * (size_t)s + c]) / R(dx[d]);
                        acc[c * NC + at(s)] -= div;
                    }
            }
#pragma omp critical
            {
                nfb_all += nfb;
                ops_all.add += t_ops.add; ops_all.mul += t_ops.mul; ops_all.div += t_ops.div; ops_all.sqrt += t_ops.sqrt;
                t_ops = {0, 0, 0, 0};
            }
        }
    }

    // O8 + O9: sources
#pragma omp parallel
    {
#pragma omp for schedule(static) collapse(2)
        for (int k = 0; k < G.n[2]; ++k)
            for (int j = 0; j < G.n[1]; ++j)
                for (int i = 0; i < G.n[0]; ++i) {
                    const size_t c0 = G.idx(i, j, k);
                    const size_t stride[3] = {1, (size_t)G.N[0], (size_t)G.N[0] * G.N[1]};
                    R dm[3][10];
                    for (int a = 0; a < 3; ++a)
                        for (int f = 0; f < 10; ++f) {
                            const double* m = met + f * NC + c0;
                            const long s = (long)stride[a];
                            // O8: grouped so that a constant field differentiates to exactly zero
                            dm[a][f] = (R(8.0) * (R(m[s]) - R(m[-s])) - (R(m[2 * s]) - R(m[-2 * s]))) / (R(12.0) * R(dx[a]));
                        }
                    Metric<R> mc;
                    mc.alp = R(met[c0]);
                    for (int a = 0; a < 3; ++a) mc.beta[a] = R(met[(1 + a) * NC + c0]);
                    for (int c = 0; c < 6; ++c) mc.g[c] = R(met[(4 + c) * NC + c0]);
                    R P[8], K[6], S[8];
                    for (int q = 0; q < 8; ++q) P[q] = R(prim[q * NC + c0]);
                    for (int c = 0; c < 6; ++c) K[c] = R(Kc[c * NC + c0]);
                    sources_point(P, mc, K, dm, gamma, S);
                    for (int c = 1; c <= 4; ++c) acc[c * NC + c0] += S[c];
                }
#pragma omp critical
        {
            ops_all.add += t_ops.add; ops_all.mul += t_ops.mul; ops_all.div += t_ops.div; ops_all.sqrt += t_ops.sqrt;
            t_ops = {0, 0, 0, 0};
        }
    }
    if constexpr (!std::is_same<R, double>::value) {
        for (int c = 0; c < 8; ++c)
            for (int k = 0; k < G.n[2]; ++k)
                for (int j = 0; j < G.n[1]; ++j)
                    for (int i = 0; i < G.n[0]; ++i) out[c * NC + G.idx(i, j, k)] = to_double(acc[c * NC + G.idx(i, j, k)]);
    }
    if (fallback_total) *fallback_total += nfb_all;
    t_ops = ops_all;   // left for the caller (counting instance only)
}

template <class R>
int rhs_all(const int n[3], int nbox, const double* prim, const double* met, const double* K, const double dx[3],
            int g, int recon, double gamma, double* out, unsigned long long* nfallback, OpCount* ops) {
    if (!n || !prim || !met || !K || !dx || !out) return 1;
    if (n[0] < 1 || n[1] < 1 || n[2] < 1 || nbox < 1) return 1;
    if (recon != RECON_MINMOD && recon != RECON_MC && recon != RECON_WENO5) return 1;
    if (g < (recon == RECON_WENO5 ? 3 : 2)) return 1;   // R29
    if (!(gamma > 1.0) || !(dx[0] > 0.0) || !(dx[1] > 0.0) || !(dx[2] > 0.0)) return 1;
    Grid G;
    for (int a = 0; a < 3; ++a) { G.n[a] = n[a]; G.N[a] = n[a] + 2 * g; }
    G.g = g;
    G.ncell = (size_t)G.N[0] * G.N[1] * G.N[2];
    unsigned long long nfb = 0;
    OpCount tot = {0, 0, 0, 0};
    for (int b = 0; b < nbox; ++b) {
        t_ops = {0, 0, 0, 0};
        rhs_box<R>(G, prim + (size_t)b * 8 * G.ncell, met + (size_t)b * 10 * G.ncell, K + (size_t)b * 6 * G.ncell, dx,
                   recon, gamma, out + (size_t)b * 8 * G.ncell, &nfb);
        tot.add += t_ops.add; tot.mul += t_ops.mul; tot.div += t_ops.div; tot.sqrt += t_ops.sqrt;
    }
    if (nfallback) *nfallback = nfb;
    if (ops) *ops = tot;
    return 0;
}

// ---- NEXT-1: ideal-gas con2prim and the method-of-lines loop ----------------------------
// con2prim (PAPER.md l.129 step 1, l.142-146; reading R22): 1-D solve in z = rho h W^2 on the undensitised
// conserved variables,
//   v^2(z) = [S^2 z^2 + (S.B)^2 (B^2 + 2 z)] / [(z + B^2)^2 z^2],   W = (1 - v^2)^(-1/2),   rho = D / W,
//   p(z) = (Gamma-1)/Gamma (z / W^2 - rho),
//   f(z) = z + B^2 - p - B^2 / (2 W^2) - (S.B)^2 / (2 z^2) - (tau + D) = 0,
// by Newton's method with the ANALYTIC derivative
//   (v^2)' = (N' Dn - N Dn') / Dn^2,  N = S^2 z^2 + (S.B)^2 (B^2 + 2z),  Dn = (z + B^2)^2 z^2,
//   p' = (Gamma-1)/Gamma [ (1 - v^2) - z (v^2)' + D (v^2)' / (2 sqrt(1 - v^2)) ],
//   f' = 1 - p' + (B^2/2) (v^2)' + (S.B)^2 / z^3,
// safeguarded by a bracket [zlo, zhi] with f(zlo) < 0 < f(zhi) (bisection step whenever Newton leaves it), stopped at
// |dz| < 1e-14 z.  (The CUDA path solves the same equation with a finite-difference slope; the two share the equation,
// not the iteration.)
int con2prim_point(const double U[8], const Metric<double>& m, double gamma, double P[8]) {
    const double sg = m.sqrtg;
    const double D = U[0] / sg, tau = U[4] / sg;
    const double Sl[3] = {U[1] / sg, U[2] / sg, U[3] / sg};
    const double B[3] = {U[5] / sg, U[6] / sg, U[7] / sg};
    double Su[3], Bl[3];
    for (int i = 0; i < 3; ++i) {
        Su[i] = m.gu[SYM[i][0]] * Sl[0] + m.gu[SYM[i][1]] * Sl[1] + m.gu[SYM[i][2]] * Sl[2];
        Bl[i] = lower(m, B, i);
    }
    const double S2 = Sl[0] * Su[0] + Sl[1] * Su[1] + Sl[2] * Su[2];
    const double B2 = Bl[0] * B[0] + Bl[1] * B[1] + Bl[2] * B[2];
    const double SB = Sl[0] * B[0] + Sl[1] * B[1] + Sl[2] * B[2];
    const double T = SB * SB, E = tau + D, cg = (gamma - 1.0) / gamma;
    // f and f' at z
    auto eval = [&](double z, double& fp) {
        const double N = S2 * z * z + T * (B2 + 2.0 * z);
        const double zb = z + B2, Dn = zb * zb * z * z;
        const double dN = 2.0 * S2 * z + 2.0 * T, dDn = 2.0 * z * zb * (2.0 * z + B2);
        double x = N / Dn, dx = (dN * Dn - N * dDn) / (Dn * Dn);
        if (x > 1.0 - 1e-15) { x = 1.0 - 1e-15; dx = 0.0; }
        const double w = std::sqrt(1.0 - x);            // 1/W
        const double p = cg * (z * (1.0 - x) - D * w);
        const double dp = cg * ((1.0 - x) - z * dx + D * dx / (2.0 * w));
        fp = 1.0 - dp + 0.5 * B2 * dx + T / (z * z * z);
        return z + B2 - p - 0.5 * B2 * (1.0 - x) - T / (2.0 * z * z) - E;
    };
    double fp;
    double zhi = std::fmax(2.0 * (E + 1.0), 1.0);
    for (int it = 0; it < 200 && eval(zhi, fp) < 0.0; ++it) zhi *= 2.0;
    double zlo = zhi;
    for (int it = 0; it < 400 && eval(zlo, fp) > 0.0; ++it) zlo *= 0.5;
    double z = 0.5 * (zlo + zhi);
    int status = 1;
    for (int it = 0; it < 200; ++it) {
        const double f = eval(z, fp);
        if (f > 0.0) zhi = z; else zlo = z;
        double zn = z - f / fp;
        if (!(zn > zlo && zn < zhi)) zn = 0.5 * (zlo + zhi);
        const double dz = std::fabs(zn - z);
        z = zn;
        if (dz < 1e-14 * z) { status = 0; break; }
    }
    const double N = S2 * z * z + T * (B2 + 2.0 * z), zb = z + B2;
    double x = N / (zb * zb * z * z);
    if (x > 1.0 - 1e-15) x = 1.0 - 1e-15;
    const double w = std::sqrt(1.0 - x);
    const double rho = D * w, p = cg * (z * (1.0 - x) - rho);
    P[0] = rho;
    for (int i = 0; i < 3; ++i) P[1 + i] = (Su[i] + SB * B[i] / z) / zb;
    P[4] = p / ((gamma - 1.0) * rho);
    for (int i = 0; i < 3; ++i) P[5 + i] = B[i];
    return status;
}

// Ghost fill of the 8 primitive fields of one box at the outer boundary (l.170, l.255, l.329): bc = 0 "copy" (von
// Neumann: the nearest interior cell), bc = 1 periodic.  Every ghost cell takes the interior cell whose index is the
// clamped / wrapped ghost index, direction by direction.
void fill_ghosts_box(const Grid& G, double* prim, int bc) {
    auto src = [&](int i, int n) { return bc == 1 ? ((i % n) + n) % n : (i < 0 ? 0 : (i >= n ? n - 1 : i)); };
    for (int q = 0; q < 8; ++q)
        for (int k = -G.g; k < G.n[2] + G.g; ++k)
            for (int j = -G.g; j < G.n[1] + G.g; ++j)
                for (int i = -G.g; i < G.n[0] + G.g; ++i) {
                    const int si = src(i, G.n[0]), sj = src(j, G.n[1]), sk = src(k, G.n[2]);
                    if (si != i || sj != j || sk != k) prim[q * G.ncell + G.idx(i, j, k)] = prim[q * G.ncell + G.idx(si, sj, sk)];
                }
}

// ---- NEXT-2: constrained transport for the cell-centred calB^i, reading R30 ------------------
// The paper evolves the magnetic field with constrained transport in every multi-dimensional test (l.287, l.299, l.315)
// and names the staggered face / edge locations it lives on (l.194-196), but prints no algorithm (ref [56] is not in the
// reference).  R30 takes the flux-CT scheme that can be stated from the induction equation alone: the HLLE fluxes of
// calB are minus / plus the electromotive force, F^j(calB^i) = eps_{ijk} E_k (d_t B = -curl E), i.e.
//     F^x(B^y) = -E_z   F^y(B^x) = +E_z      F^y(B^z) = -E_x   F^z(B^y) = +E_x      F^z(B^x) = -E_y   F^x(B^z) = +E_y.
// (1) the face fluxes are evaluated exactly as in the right-hand side (same reconstruction, face metric, HLLE), also on the
//     one layer of grid lines next to the block (transverse index -1 and n), which the edge averages below reach;
// (2) the EMF on a cell EDGE is the arithmetic mean of the four face fluxes that touch the edge, with those signs;
// (3) the flux of calB^i through a face is replaced by the mean of the two edge EMFs on that face, and d calB^i/dt is the
//     difference of those replaced fluxes -- a discrete curl of edge EMFs, so the vertex-centred divergence (at a vertex:
//     sum_d [mean of B^d over the four cells on the high side - mean over the four on the low side] / dx_d) of the update
//     vanishes to rounding wherever the eight cells around the vertex are updated.
// FB layout: [9][Nz][Ny][Nx] per box, FB[3 d + c] = F^d(calB^c) at the LOW d-face of the cell it is indexed by (face
// i-1/2 for d = x, ...); normal index 0..n, transverse indices -1..n; other entries untouched.  The three normal
// components F^d(calB^d) -- the purely dissipative part of the HLLE flux, which flux-CT drops -- are stored so that the
// pins can rebuild the plain right-hand side from FB.
void face_bflux_box(const Grid& G, const double* prim, const double* met, int recon, double gamma_d, double* FB) {
    const size_t NC = G.ncell;
    for (int d = 0; d < 3; ++d) {
        const int d1 = (d + 1) % 3, d2 = (d + 2) % 3;
        const int nd = G.n[d], n1 = G.n[d1] + 2, n2 = G.n[d2] + 2;
#pragma omp parallel
        {
            unsigned long long nfb = 0;
            std::vector<double> qm(8 * (size_t)(nd + 2)), qp(8 * (size_t)(nd + 2));
#pragma omp for schedule(static)
            for (long line = 0; line < (long)n1 * n2; ++line) {
                int ijk[3];
                ijk[d1] = (int)(line % n1) - 1;
                ijk[d2] = (int)(line / n1) - 1;
                auto at = [&](int s) {
                    int c3[3] = {ijk[0], ijk[1], ijk[2]};
                    c3[d] = s;
                    return G.idx(c3[0], c3[1], c3[2]);
                };
                for (int s = -1; s <= nd; ++s)
                    for (int q = 0; q < 8; ++q) {
                        const double* f = prim + q * NC;
                        const double a = (recon == RECON_WENO5) ? f[at(s - 2)] : 0.0;
                        const double e = (recon == RECON_WENO5) ? f[at(s + 2)] : 0.0;
                        recon_cell<double>(recon, a, f[at(s - 1)], f[at(s)], f[at(s + 1)], e, qm[q * (nd + 2) + s + 1],
                                           qp[q * (nd + 2) + s + 1]);
                    }
                for (int f = 0; f <= nd; ++f) {
                    const size_t iL = at(f - 1), iR = at(f);
                    Metric<double> mf;
                    mf.alp = 0.5 * (met[0 * NC + iL] + met[0 * NC + iR]);
                    for (int i = 0; i < 3; ++i) mf.beta[i] = 0.5 * (met[(1 + i) * NC + iL] + met[(1 + i) * NC + iR]);
                    for (int c = 0; c < 6; ++c) mf.g[c] = 0.5 * (met[(4 + c) * NC + iL] + met[(4 + c) * NC + iR]);
                    double PL[8], PR[8], CL[8], CR[8], Fh[8];
                    for (int q = 0; q < 8; ++q) {
                        PL[q] = qp[q * (nd + 2) + f];
                        PR[q] = qm[q * (nd + 2) + f + 1];
                        CL[q] = prim[q * NC + iL];
                        CR[q] = prim[q * NC + iR];
                    }
                    face_flux(mf, d, gamma_d, PL, PR, CL, CR, Fh, &nfb);
                    for (int c = 0; c < 3; ++c) FB[(3 * d + c) * NC + iR] = Fh[5 + c];
                }
            }
        }
    }
    t_ops = {0, 0, 0, 0};
}

// Steps (2) and (3): d calB^i / dt on the interior cells from the face fluxes FB.
void flux_ct_box(const Grid& G, const double* FB, const double dx[3], double* dB) {
    const size_t NC = G.ncell;
    const double* FxBy = FB + 1 * NC; const double* FxBz = FB + 2 * NC;
    const double* FyBx = FB + 3 * NC; const double* FyBz = FB + 5 * NC;
    const double* FzBx = FB + 6 * NC; const double* FzBy = FB + 7 * NC;
    // edge EMFs, indexed by the cell whose LOW-LOW edge it is: Ez(i,j,k) sits at (i-1/2, j-1/2, k), and so on
    auto Ez = [&](int i, int j, int k) {
        return 0.25 * (-FxBy[G.idx(i, j, k)] - FxBy[G.idx(i, j - 1, k)] + FyBx[G.idx(i, j, k)] + FyBx[G.idx(i - 1, j, k)]);
    };
    auto Ex = [&](int i, int j, int k) {
        return 0.25 * (-FyBz[G.idx(i, j, k)] - FyBz[G.idx(i, j, k - 1)] + FzBy[G.idx(i, j, k)] + FzBy[G.idx(i, j - 1, k)]);
    };
    auto Ey = [&](int i, int j, int k) {
        return 0.25 * (-FzBx[G.idx(i, j, k)] - FzBx[G.idx(i - 1, j, k)] + FxBz[G.idx(i, j, k)] + FxBz[G.idx(i, j, k - 1)]);
    };
#pragma omp parallel for schedule(static) collapse(2)
    for (int k = 0; k < G.n[2]; ++k)
        for (int j = 0; j < G.n[1]; ++j)
            for (int i = 0; i < G.n[0]; ++i) {
                // replaced fluxes on the six faces of the cell: mean of the two edge EMFs on the face, with the sign of
                // F^j(B^i) = eps_{ijk} E_k
                const double FyBx_lo = 0.5 * (Ez(i, j, k) + Ez(i + 1, j, k)), FyBx_hi = 0.5 * (Ez(i, j + 1, k) + Ez(i + 1, j + 1, k));
                const double FzBx_lo = -0.5 * (Ey(i, j, k) + Ey(i + 1, j, k)), FzBx_hi = -0.5 * (Ey(i, j, k + 1) + Ey(i + 1, j, k + 1));
                const double FxBy_lo = -0.5 * (Ez(i, j, k) + Ez(i, j + 1, k)), FxBy_hi = -0.5 * (Ez(i + 1, j, k) + Ez(i + 1, j + 1, k));
                const double FzBy_lo = 0.5 * (Ex(i, j, k) + Ex(i, j + 1, k)), FzBy_hi = 0.5 * (Ex(i, j, k + 1) + Ex(i, j + 1, k + 1));
                const double FxBz_lo = 0.5 * (Ey(i, j, k) + Ey(i, j, k + 1)), FxBz_hi = 0.5 * (Ey(i + 1, j, k) + Ey(i + 1, j, k + 1));
                const double FyBz_lo = -0.5 * (Ex(i, j, k) + Ex(i, j, k + 1)), FyBz_hi = -0.5 * (Ex(i, j + 1, k) + Ex(i, j + 1, k + 1));
                const size_t c = G.idx(i, j, k);
                dB[0 * NC + c] = -(FyBx_hi - FyBx_lo) / dx[1] - (FzBx_hi - FzBx_lo) / dx[2];
                dB[1 * NC + c] = -(FxBy_hi - FxBy_lo) / dx[0] - (FzBy_hi - FzBy_lo) / dx[2];
                dB[2 * NC + c] = -(FxBz_hi - FxBz_lo) / dx[0] - (FyBz_hi - FyBz_lo) / dx[1];
            }
}

// ---- NEXT-3: vertex-centred spacetime, readings R31 / R32 -----------------------------------
// "Spacetime geometry quantities are stored on vertices", "the spacetime metric ... is known at the cell
// vertices and is interpolated linearly to the face centers" (l.130), "the stress-energy tensor [is] stored as samples at
// the cell vertices ... we perform a 4th-order symmetric 3D interpolation from cell center values to calculate the fluid
// variables at cell vertices" (l.84, l.323).
// Vertex arrays: [field][Nz+1][Ny+1][Nx+1]; vertex (I, J, K) is the LOW corner of cell (I, J, K) (indices with ghosts), so
// cell (I, J, K) has the eight vertices (I..I+1, J..J+1, K..K+1) and its low d-face the four with the d index fixed.
// R31: face metric = arithmetic mean of the 4 vertices of the face (linear interpolation to the face centre); cell-centre
//      metric and K_ij = mean of the 8 vertices; d_a of a metric field at the cell centre = staggered 4th-order difference
//      [27 (m(i+1/2) - m(i-1/2)) - (m(i+3/2) - m(i-3/2))] / (24 dx_a) of the transverse 4-vertex means m(.) at the four
//      vertex planes around the cell, grouped so that a constant differentiates to exactly zero.  Everything else is the
//      right-hand side of rhs_box.
struct VGrid {
    Grid G;
    size_t nv;                // vertices per field
    size_t vidx(int i, int j, int k) const {   // vertex at the low corner of the cell with INTERIOR index (i, j, k)
        return (size_t)(i + G.g) + (size_t)(G.N[0] + 1) * ((size_t)(j + G.g) + (size_t)(G.N[1] + 1) * (size_t)(k + G.g));
    }
};

// mean of the 4 vertices of the low d-face of cell (i, j, k)
inline double face_mean(const VGrid& V, const double* f, int d, int i, int j, int k) {
    const int d1 = (d + 1) % 3, d2 = (d + 2) % 3;
    double sum = 0.0;
    for (int a = 0; a < 2; ++a)
        for (int b = 0; b < 2; ++b) {
            int c[3] = {i, j, k};
            c[d1] += a;
            c[d2] += b;
            sum += f[V.vidx(c[0], c[1], c[2])];
        }
    return 0.25 * sum;
}

void rhs_vertex_box(const VGrid& V, const double* prim, const double* metv, const double* Kv, const double dx[3], int recon,
                    double gamma, double* out, unsigned long long* fallback_total) {
    const Grid& G = V.G;
    const size_t NC = G.ncell, NV = V.nv;
    unsigned long long nfb_all = 0;
    for (int c = 0; c < 8; ++c)
        for (int k = 0; k < G.n[2]; ++k)
            for (int j = 0; j < G.n[1]; ++j)
                for (int i = 0; i < G.n[0]; ++i) out[c * NC + G.idx(i, j, k)] = 0.0;
    for (int d = 0; d < 3; ++d) {
        const int d1 = (d + 1) % 3, d2 = (d + 2) % 3;
        const int nd = G.n[d];
        const long nlines = (long)G.n[d1] * G.n[d2];
#pragma omp parallel
        {
            unsigned long long nfb = 0;
            std::vector<double> qm(8 * (size_t)(nd + 2)), qp(8 * (size_t)(nd + 2)), Fh(8 * (size_t)(nd + 1));
#pragma omp for schedule(static)
            for (long line = 0; line < nlines; ++line) {
                int ijk[3];
                ijk[d1] = (int)(line % G.n[d1]);
                ijk[d2] = (int)(line / G.n[d1]);
                auto cell = [&](int s, int c3[3]) { c3[0] = ijk[0]; c3[1] = ijk[1]; c3[2] = ijk[2]; c3[d] = s; };
                auto at = [&](int s) { int c3[3]; cell(s, c3); return G.idx(c3[0], c3[1], c3[2]); };
                for (int s = -1; s <= nd; ++s)
                    for (int q = 0; q < 8; ++q) {
                        const double* f = prim + q * NC;
                        const double a = (recon == RECON_WENO5) ? f[at(s - 2)] : 0.0;
                        const double e = (recon == RECON_WENO5) ? f[at(s + 2)] : 0.0;
                        recon_cell<double>(recon, a, f[at(s - 1)], f[at(s)], f[at(s + 1)], e, qm[q * (nd + 2) + s + 1],
                                           qp[q * (nd + 2) + s + 1]);
                    }
                for (int f = 0; f <= nd; ++f) {
                    const size_t iL = at(f - 1), iR = at(f);
                    int c3[3];
                    cell(f, c3);                                   // the face is the low d-face of cell f
                    Metric<double> mf;
                    mf.alp = face_mean(V, metv + 0 * NV, d, c3[0], c3[1], c3[2]);                       // R31
                    for (int i = 0; i < 3; ++i) mf.beta[i] = face_mean(V, metv + (1 + i) * NV, d, c3[0], c3[1], c3[2]);
                    for (int c = 0; c < 6; ++c) mf.g[c] = face_mean(V, metv + (4 + c) * NV, d, c3[0], c3[1], c3[2]);
                    double PL[8], PR[8], CL[8], CR[8];
                    for (int q = 0; q < 8; ++q) {
                        PL[q] = qp[q * (nd + 2) + f];
                        PR[q] = qm[q * (nd + 2) + f + 1];
                        CL[q] = prim[q * NC + iL];
                        CR[q] = prim[q * NC + iR];
                    }
                    face_flux(mf, d, gamma, PL, PR, CL, CR, &Fh[8 * (size_t)f], &nfb);
                }
                for (int s = 0; s < nd; ++s)
                    for (int c = 0; c < 8; ++c) out[c * NC + at(s)] -= (Fh[8 * (size_t)(s + 1) + c] - Fh[8 * (size_t)s + c]) / dx[d];
            }
#pragma omp critical
            nfb_all += nfb;
        }
    }
#pragma omp parallel for schedule(static) collapse(2)
    for (int k = 0; k < G.n[2]; ++k)
        for (int j = 0; j < G.n[1]; ++j)
            for (int i = 0; i < G.n[0]; ++i) {
                const size_t c0 = G.idx(i, j, k);
                double dm[3][10];
                Metric<double> mc;
                double mcv[10], K[6];
                for (int f = 0; f < 10; ++f) {
                    const double* mv = metv + f * NV;
                    // centre = mean of 8 vertices = mean of the low and the high x-face means
                    mcv[f] = 0.5 * (face_mean(V, mv, 0, i, j, k) + face_mean(V, mv, 0, i + 1, j, k));
                    for (int a = 0; a < 3; ++a) {
                        int lo2[3] = {i, j, k}, lo1[3] = {i, j, k}, hi1[3] = {i, j, k}, hi2[3] = {i, j, k};
                        lo2[a] -= 1; hi1[a] += 1; hi2[a] += 2;      // vertex planes a-3/2, a-1/2, a+1/2, a+3/2 around the centre
                        const double m_m2 = face_mean(V, mv, a, lo2[0], lo2[1], lo2[2]);
                        const double m_m1 = face_mean(V, mv, a, lo1[0], lo1[1], lo1[2]);
                        const double m_p1 = face_mean(V, mv, a, hi1[0], hi1[1], hi1[2]);
                        const double m_p2 = face_mean(V, mv, a, hi2[0], hi2[1], hi2[2]);
                        dm[a][f] = (27.0 * (m_p1 - m_m1) - (m_p2 - m_m2)) / (24.0 * dx[a]);
                    }
                }
                mc.alp = mcv[0];
                for (int a = 0; a < 3; ++a) mc.beta[a] = mcv[1 + a];
                for (int c = 0; c < 6; ++c) mc.g[c] = mcv[4 + c];
                for (int c = 0; c < 6; ++c)
                    K[c] = 0.5 * (face_mean(V, Kv + c * NV, 0, i, j, k) + face_mean(V, Kv + c * NV, 0, i + 1, j, k));
                double P[8], S[8];
                for (int q = 0; q < 8; ++q) P[q] = prim[q * NC + c0];
                sources_point(P, mc, K, dm, gamma, S);
                for (int c = 1; c <= 4; ++c) out[c * NC + c0] += S[c];
            }
    if (fallback_total) *fallback_total += nfb_all;
    t_ops = {0, 0, 0, 0};
}

// R32: T^{mu nu} (Eq. 5, l.80-84) at the vertices of the interior cells.  The 8 primitives are interpolated from the cell
// centres to the vertex with the tensor product of the symmetric 4-point midpoint rule (-1, 9, 9, -1)/16 (64 cells: "4th-
// order symmetric 3D interpolation", l.84), then Eq. (5) is evaluated with the vertex's own metric sample:
//   T^{mu nu} = rho h* u^mu u^nu + P* g^{mu nu} - b^mu b^nu,   u^0 = W/alpha, u^i = W (v^i - beta^i/alpha),
//   b^0 = W B^k v_k / alpha, b^i = B^i / W + alpha b^0 (v^i - beta^i/alpha)... with b^i = (B^i + alpha b^0 u^i)/W,
//   g^{00} = -1/alpha^2, g^{0i} = beta^i/alpha^2, g^{ij} = gamma^{ij} - beta^i beta^j/alpha^2.
// T[10][vertex] = T^{00}, T^{0x}, T^{0y}, T^{0z}, T^{xx}, T^{xy}, T^{xz}, T^{yy}, T^{yz}, T^{zz}; vertices (0..n) per
// direction (interior-cell corners); other entries untouched.  Needs 2 ghost cells.
void tmunu_point(const double P[8], Metric<double>& m, double gamma, double T[10]) {
    metric_complete(m);
    const double rho = P[0], eps = P[4];
    const double v[3] = {P[1], P[2], P[3]}, B[3] = {P[5], P[6], P[7]};
    double vl[3], Bl[3];
    for (int i = 0; i < 3; ++i) { vl[i] = lower(m, v, i); Bl[i] = lower(m, B, i); }
    const double v2 = vl[0] * v[0] + vl[1] * v[1] + vl[2] * v[2];
    const double W = 1.0 / std::sqrt(1.0 - v2);
    const double Bv = Bl[0] * v[0] + Bl[1] * v[1] + Bl[2] * v[2];
    const double B2 = Bl[0] * B[0] + Bl[1] * B[1] + Bl[2] * B[2];
    const double a = m.alp;
    double u[4], b[4];
    u[0] = W / a;
    for (int i = 0; i < 3; ++i) u[1 + i] = W * (v[i] - m.beta[i] / a);
    b[0] = W * Bv / a;
    for (int i = 0; i < 3; ++i) b[1 + i] = (B[i] + a * b[0] * u[1 + i]) / W;
    const double b2 = (B2 + (a * b[0]) * (a * b[0])) / (W * W);
    const double p = (gamma - 1.0) * rho * eps;
    const double rhohs = rho * (1.0 + eps) + p + b2, Ps = p + 0.5 * b2;
    double ginv[4][4];
    ginv[0][0] = -1.0 / (a * a);
    for (int i = 0; i < 3; ++i) ginv[0][1 + i] = ginv[1 + i][0] = m.beta[i] / (a * a);
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) ginv[1 + i][1 + j] = m.gu[SYM[i][j]] - m.beta[i] * m.beta[j] / (a * a);
    int n = 0;
    for (int mu = 0; mu < 4; ++mu)
        for (int nu = mu; nu < 4; ++nu) T[n++] = rhohs * u[mu] * u[nu] + Ps * ginv[mu][nu] - b[mu] * b[nu];
}

void tmunu_vertex_box(const VGrid& V, const double* prim, const double* metv, double gamma, double* T) {
    const Grid& G = V.G;
    const size_t NC = G.ncell, NV = V.nv;
    const double w[4] = {-1.0 / 16.0, 9.0 / 16.0, 9.0 / 16.0, -1.0 / 16.0};
#pragma omp parallel for schedule(static) collapse(2)
    for (int k = 0; k <= G.n[2]; ++k)
        for (int j = 0; j <= G.n[1]; ++j)
            for (int i = 0; i <= G.n[0]; ++i) {
                double P[8];
                for (int q = 0; q < 8; ++q) {
                    double sum = 0.0;
                    for (int c = 0; c < 4; ++c)
                        for (int b = 0; b < 4; ++b)
                            for (int a = 0; a < 4; ++a)
                                sum += w[c] * w[b] * w[a] * prim[q * NC + G.idx(i - 2 + a, j - 2 + b, k - 2 + c)];
                    P[q] = sum;
                }
                Metric<double> m;
                const size_t v0 = V.vidx(i, j, k);
                m.alp = metv[v0];
                for (int a = 0; a < 3; ++a) m.beta[a] = metv[(1 + a) * NV + v0];
                for (int c = 0; c < 6; ++c) m.g[c] = metv[(4 + c) * NV + v0];
                double T10[10];
                tmunu_point(P, m, gamma, T10);
                for (int c = 0; c < 10; ++c) T[c * NV + v0] = T10[c];
            }
}

}  // namespace

// =================================================== C ABI ===================================================
// All pointers are HOST pointers.  Array layout is the library's (include/grx.h): SoA, x fastest,
// ghosts included, [box][field][k][j][i].  Return 0 = ok, 1 = invalid argument.
extern "C" {

int oracle_valencia_rhs(const int n[3], int nbox, const double* prim, const double* metric, const double* K,
                        const double dx[3], int nghost, int recon, double gamma, double* out,
                        unsigned long long* nfallback) {
    return rhs_all<double>(n, nbox, prim, metric, K, dx, nghost, recon, gamma, out, nfallback, nullptr);
}

// adjudicator: same algorithm evaluated in long double (x87 80-bit), results rounded to double
int oracle_valencia_rhs_ld(const int n[3], int nbox, const double* prim, const double* metric, const double* K,
                           const double dx[3], int nghost, int recon, double gamma, double* out,
                           unsigned long long* nfallback) {
    return rhs_all<long double>(n, nbox, prim, metric, K, dx, nghost, recon, gamma, out, nfallback, nullptr);
}

// counting instance: ops[4] = {add/sub, mul, div, sqrt} executed by one whole call (compares, selects,
// sign flips, abs and loads/stores are free).  Each face is evaluated once.
int oracle_valencia_rhs_count(const int n[3], int nbox, const double* prim, const double* metric, const double* K,
                              const double dx[3], int nghost, int recon, double gamma, double* out,
                              unsigned long long ops[4]) {
    OpCount c;
    int rc = rhs_all<Counted>(n, nbox, prim, metric, K, dx, nghost, recon, gamma, out, nullptr, &c);
    if (rc == 0 && ops) { ops[0] = c.add; ops[1] = c.mul; ops[2] = c.div; ops[3] = c.sqrt; }
    return rc;
}

// O10: prim2con on ALL cells including ghosts, cell-centre metric (Eqs. 6-9)
int oracle_prim2con(const int n[3], int nbox, const double* prim, const double* metric, int nghost, double gamma,
                    double* cons) {
    if (!n || !prim || !metric || !cons || nbox < 1 || nghost < 0 || !(gamma > 1.0)) return 1;
    const size_t NC = (size_t)(n[0] + 2 * nghost) * (n[1] + 2 * nghost) * (n[2] + 2 * nghost);
    for (int b = 0; b < nbox; ++b) {
        const double* pb = prim + (size_t)b * 8 * NC;
        const double* mb = metric + (size_t)b * 10 * NC;
        double* cb = cons + (size_t)b * 8 * NC;
#pragma omp parallel for schedule(static)
        for (long c0 = 0; c0 < (long)NC; ++c0) {
            Metric<double> m;
            m.alp = mb[c0];
            for (int a = 0; a < 3; ++a) m.beta[a] = mb[(1 + a) * NC + c0];
            for (int c = 0; c < 6; ++c) m.g[c] = mb[(4 + c) * NC + c0];
            metric_complete(m);
            double P[8];
            for (int q = 0; q < 8; ++q) P[q] = pb[q * NC + c0];
            State<double> s;
            prim2con_point(P, m, gamma, s);
            for (int q = 0; q < 8; ++q) cb[q * NC + c0] = s.U[q];
        }
    }
    return 0;
}

// support (R22): con2prim on all cells; returns the number of cells whose solve did not converge
int oracle_con2prim(const int n[3], int nbox, const double* cons, const double* metric, int nghost, double gamma,
                    double* prim) {
    if (!n || !prim || !metric || !cons || nbox < 1 || nghost < 0 || !(gamma > 1.0)) return -1;
    const size_t NC = (size_t)(n[0] + 2 * nghost) * (n[1] + 2 * nghost) * (n[2] + 2 * nghost);
    int nfail = 0;
    for (int b = 0; b < nbox; ++b) {
        const double* cb = cons + (size_t)b * 8 * NC;
        const double* mb = metric + (size_t)b * 10 * NC;
        double* pb = prim + (size_t)b * 8 * NC;
#pragma omp parallel for schedule(static) reduction(+ : nfail)
        for (long c0 = 0; c0 < (long)NC; ++c0) {
            Metric<double> m;
            m.alp = mb[c0];
            for (int a = 0; a < 3; ++a) m.beta[a] = mb[(1 + a) * NC + c0];
            for (int c = 0; c < 6; ++c) m.g[c] = mb[(4 + c) * NC + c0];
            metric_complete(m);
            double U[8], P[8];
            for (int q = 0; q < 8; ++q) U[q] = cb[q * NC + c0];
            nfail += con2prim_point(U, m, gamma, P);
            for (int q = 0; q < 8; ++q) pb[q * NC + c0] = P[q];
        }
    }
    return nfail;
}

// NEXT-1: method of lines (l.125) around the right-hand side, `nsteps` steps of size dt on every box.
//   rk = 2: SSP-RK2 (Heun; reading R21)   U1 = U + dt L(P);  U <- 1/2 U + 1/2 (U1 + dt L(P1))
//   rk = 4: classical RK4 (l.255, l.335)   U <- U + dt/6 (k1 + 2 k2 + 2 k3 + k4),  k2 = L(P(U + dt/2 k1)), ...
// The evolved variables are the conserved ones on the interior cells; after every stage update the primitives follow by
// con2prim on the interior (step 1 of the paper's RHS evaluation, l.129) and their ghost zones are filled (bc = 0 copy,
// 1 periodic).  prim (in/out) must come with filled ghosts; cons (out, may be NULL) receives U on the interior (ghosts 0).
// Returns the number of con2prim failures (>= 0) or -1 for invalid arguments.
int oracle_face_bfluxes(const int n[3], int nbox, const double* prim, const double* metric, int nghost, int recon,
                        double gamma, double* FB);
int oracle_flux_ct(const int n[3], int nbox, const double* FB, const double dx[3], int nghost, double* dB);

// ct = 1: the calB components of every right-hand side are the flux-CT update (NEXT-2, R30) instead of the plain flux difference.
static int evolve_impl(const int n[3], int nbox, double* prim, const double* metric, const double* K, const double dx[3],
                       int nghost, int recon, double gamma, double dt, int nsteps, int rk, int bc, double* cons, int ct) {
    if (!n || !prim || !metric || !K || !dx || nbox < 1 || nsteps < 0 || (rk != 2 && rk != 4) || (bc != 0 && bc != 1)) return -1;
    if (!(gamma > 1.0) || nghost < (recon == RECON_WENO5 ? 3 : 2)) return -1;
    Grid G;
    G.g = nghost;
    G.ncell = 1;
    for (int a = 0; a < 3; ++a) { G.n[a] = n[a]; G.N[a] = n[a] + 2 * nghost; G.ncell *= (size_t)G.N[a]; }
    const size_t NC = G.ncell, NA = 8 * NC * (size_t)nbox;
    std::vector<double> U(NA, 0.0), U0(NA), L(NA), acc;
    if (oracle_prim2con(n, nbox, prim, metric, nghost, gamma, U.data())) return -1;
    int nfail = 0;
    // U_out = a U0 + b (U_in + dt L) on the interior, then prim = con2prim(U_out) there and ghost fill
    auto stage = [&](double a, const std::vector<double>& Ua, double b, const std::vector<double>& Ub, double h,
                     std::vector<double>& Uout) {
        for (int bx = 0; bx < nbox; ++bx) {
            const size_t off = (size_t)bx * 8 * NC;
            const double* mb = metric + (size_t)bx * 10 * NC;
            int nf = 0;
#pragma omp parallel for schedule(static) collapse(2) reduction(+ : nf)
            for (int k = 0; k < G.n[2]; ++k)
                for (int j = 0; j < G.n[1]; ++j)
                    for (int i = 0; i < G.n[0]; ++i) {
                        const size_t c0 = G.idx(i, j, k);
                        double Uc[8], P[8];
                        for (int q = 0; q < 8; ++q) {
                            const size_t o = off + q * NC + c0;
                            Uc[q] = a * Ua[o] + b * (Ub[o] + h * L[o]);
                            Uout[o] = Uc[q];
                        }
                        Metric<double> m;
                        m.alp = mb[c0];
                        for (int d = 0; d < 3; ++d) m.beta[d] = mb[(1 + d) * NC + c0];
                        for (int c = 0; c < 6; ++c) m.g[c] = mb[(4 + c) * NC + c0];
                        metric_complete(m);
                        nf += con2prim_point(Uc, m, gamma, P);
                        for (int q = 0; q < 8; ++q) prim[off + q * NC + c0] = P[q];
                    }
            nfail += nf;
            fill_ghosts_box(G, prim + off, bc);
        }
    };
    std::vector<double> FB, dB;
    if (ct) { FB.assign(9 * NC * (size_t)nbox, 0.0); dB.assign(3 * NC * (size_t)nbox, 0.0); }
    auto rhs = [&]() {
        if (rhs_all<double>(n, nbox, prim, metric, K, dx, nghost, recon, gamma, L.data(), nullptr, nullptr)) return 1;
        if (!ct) return 0;
        if (oracle_face_bfluxes(n, nbox, prim, metric, nghost, recon, gamma, FB.data())) return 1;
        if (oracle_flux_ct(n, nbox, FB.data(), dx, nghost, dB.data())) return 1;
        for (int bx = 0; bx < nbox; ++bx)
            for (int c = 0; c < 3; ++c)
                for (int k = 0; k < G.n[2]; ++k)
                    for (int j = 0; j < G.n[1]; ++j)
                        for (int i = 0; i < G.n[0]; ++i)
                            L[(size_t)bx * 8 * NC + (5 + c) * NC + G.idx(i, j, k)] = dB[(size_t)bx * 3 * NC + c * NC + G.idx(i, j, k)];
        return 0;
    };
    for (int s = 0; s < nsteps; ++s) {
        U0 = U;
        if (rk == 2) {
            if (rhs()) return -1;
            stage(0.0, U0, 1.0, U0, dt, U);          // U1 = U0 + dt L(P0)
            if (rhs()) return -1;
            stage(0.5, U0, 0.5, U, dt, U);           // U  = 1/2 U0 + 1/2 (U1 + dt L(P1))
        } else {
            acc = U0;                                 // acc = U0 + dt/6 (k1 + 2 k2 + 2 k3 + k4), built stage by stage
            const double w[4] = {1.0 / 6.0, 1.0 / 3.0, 1.0 / 3.0, 1.0 / 6.0}, hs[3] = {0.5, 0.5, 1.0};
            for (int st = 0; st < 4; ++st) {
                if (rhs()) return -1;
                for (int bx = 0; bx < nbox; ++bx)
                    for (int q = 0; q < 8; ++q)
                        for (int k = 0; k < G.n[2]; ++k)
                            for (int j = 0; j < G.n[1]; ++j)
                                for (int i = 0; i < G.n[0]; ++i) {
                                    const size_t o = (size_t)bx * 8 * NC + q * NC + G.idx(i, j, k);
                                    acc[o] += w[st] * dt * L[o];
                                }
                if (st < 3) stage(0.0, U0, 1.0, U0, hs[st] * dt, U);   // U = U0 + h dt k_st
                else { for (size_t o = 0; o < NA; ++o) L[o] = 0.0; stage(0.0, U0, 1.0, acc, 0.0, U); }
            }
        }
    }
    if (cons)
        for (size_t o = 0; o < NA; ++o) cons[o] = 0.0;
    if (cons)
        for (int bx = 0; bx < nbox; ++bx)
            for (int q = 0; q < 8; ++q)
                for (int k = 0; k < G.n[2]; ++k)
                    for (int j = 0; j < G.n[1]; ++j)
                        for (int i = 0; i < G.n[0]; ++i) {
                            const size_t o = (size_t)bx * 8 * NC + q * NC + G.idx(i, j, k);
                            cons[o] = U[o];
                        }
    return nfail;
}

int oracle_evolve(const int n[3], int nbox, double* prim, const double* metric, const double* K, const double dx[3],
                  int nghost, int recon, double gamma, double dt, int nsteps, int rk, int bc, double* cons) {
    return evolve_impl(n, nbox, prim, metric, K, dx, nghost, recon, gamma, dt, nsteps, rk, bc, cons, 0);
}

int oracle_evolve_ct(const int n[3], int nbox, double* prim, const double* metric, const double* K, const double dx[3],
                     int nghost, int recon, double gamma, double dt, int nsteps, int rk, int bc, double* cons) {
    return evolve_impl(n, nbox, prim, metric, K, dx, nghost, recon, gamma, dt, nsteps, rk, bc, cons, 1);
}

// ---- point-level entry points used by the pins (tests/test_oracle_pins*.py) -------------------------
void oracle_recon_cell(int recon, const double q[5], double* qm, double* qp) {
    recon_cell<double>(recon, q[0], q[1], q[2], q[3], q[4], *qm, *qp);
}

static void fill_metric(Metric<double>& m, const double met[10]) {
    m.alp = met[0];
    for (int a = 0; a < 3; ++a) m.beta[a] = met[1 + a];
    for (int c = 0; c < 6; ++c) m.g[c] = met[4 + c];
}

// U, F^d and the two characteristic speeds of one state in one metric (O4-O6)
void oracle_state_flux(const double P[8], const double met[10], int d, double gamma, double U[8], double F[8],
                       double lam[2]) {
    Metric<double> m;
    fill_metric(m, met);
    metric_complete(m);
    State<double> s;
    prim2con_point(P, m, gamma, s);
    for (int c = 0; c < 8; ++c) U[c] = s.U[c];
    flux_point(P, m, s, d, F);
    wavespeeds_point(P, m, s, d, gamma, lam[0], lam[1]);
}

// HLLE flux of one interface from already reconstructed states and an already averaged face metric (O3-O7)
void oracle_face_flux(const double PL[8], const double PR[8], const double CL[8], const double CR[8],
                      const double met_face[10], int d, double gamma, double Fh[8]) {
    Metric<double> m;
    fill_metric(m, met_face);
    face_flux(m, d, gamma, PL, PR, CL, CR, Fh, nullptr);
}

void oracle_hlle(const double UL[8], const double FL[8], const double lamL[2], const double UR[8],
                 const double FR[8], const double lamR[2], double Fh[8]) {
    hlle<double>(UL, FL, lamL[0], lamL[1], UR, FR, lamR[0], lamR[1], Fh);
}

// sources of one cell from point values and given metric derivatives dm[3][10] (O9)
void oracle_sources_point(const double P[8], const double met[10], const double K[6], const double dm[30],
                          double gamma, double S[8]) {
    Metric<double> m;
    fill_metric(m, met);
    double d3[3][10];
    for (int a = 0; a < 3; ++a)
        for (int f = 0; f < 10; ++f) d3[a][f] = dm[a * 10 + f];
    sources_point(P, m, K, d3, gamma, S);
}

// ---- point-level COUNTING entry point (tests/test_bench_model.py pins the operation count of every piece
// against a hand count, so that the roofline numerator is fixed by something other than this file's own total).
// piece: 0 recon_cell(recon)  1 face average of the 10 metric fields (O1)  2 metric_complete_face(d)
//        3 admissible  4 prim2con_point  5 flux_point(d)  6 wavespeeds_point(d)  7 hlle  8 metric_complete
//        9 one 4th-order derivative (O8)  10 sources_point  11 flux difference of one component (O7)
// ops[4] = {add/sub, mul, div, sqrt}.  The sample inputs are fixed, smooth and admissible; no arithmetic of the
// double instance is touched.
int oracle_count_piece(int piece, int d, int recon, unsigned long long ops[4]) {
    typedef Counted R;
    if (!ops || d < 0 || d > 2) return 1;
    R P[8] = {R(0.7), R(0.2), R(-0.1), R(0.3), R(1.3), R(0.4), R(-0.2), R(0.1)};
    R Q[8] = {R(0.6), R(0.1), R(-0.2), R(0.2), R(1.1), R(0.3), R(-0.1), R(0.2)};
    Metric<R> m;
    m.alp = R(0.9); m.beta[0] = R(0.02); m.beta[1] = R(-0.03); m.beta[2] = R(0.01);
    const double gv[6] = {1.2, 0.1, -0.05, 1.1, 0.07, 0.95};
    for (int c = 0; c < 6; ++c) m.g[c] = R(gv[c]);
    metric_complete(m);
    State<R> s, s2;
    prim2con_point(P, m, R(1.4), s);
    prim2con_point(Q, m, R(1.4), s2);
    R F[8], F2[8], lm, lp, lm2, lp2, out[8];
    flux_point(P, m, s, d, F); wavespeeds_point(P, m, s, d, R(1.4), lm, lp);
    flux_point(Q, m, s2, d, F2); wavespeeds_point(Q, m, s2, d, R(1.4), lm2, lp2);
    t_ops = {0, 0, 0, 0};
    switch (piece) {
        case 0: { R qm, qp; recon_cell<R>(recon, R(1.0), R(1.3), R(1.7), R(2.0), R(2.6), qm, qp); break; }
        case 1: { Metric<R> f; f.alp = R(0.5) * (m.alp + m.alp);
                  for (int i = 0; i < 3; ++i) f.beta[i] = R(0.5) * (m.beta[i] + m.beta[i]);
                  for (int c = 0; c < 6; ++c) f.g[c] = R(0.5) * (m.g[c] + m.g[c]);
                  break; }
        case 2: metric_complete_face(m, d); break;
        case 3: (void)admissible(P, m); break;
        case 4: prim2con_point(P, m, R(1.4), s); break;
        case 5: flux_point(P, m, s, d, F); break;
        case 6: wavespeeds_point(P, m, s, d, R(1.4), lm, lp); break;
        case 7: hlle<R>(s.U, F, lm, lp, s2.U, F2, lm2, lp2, out); break;
        case 8: metric_complete(m); break;
        case 9: { R v = (R(8.0) * (R(1.1) - R(0.9)) - (R(1.2) - R(0.8))) / (R(12.0) * R(0.1)); (void)v; break; }
        case 10: { R K[6], dm[3][10], S[8];
                   for (int c = 0; c < 6; ++c) K[c] = R(0.01 * (c + 1));
                   for (int a = 0; a < 3; ++a) for (int f = 0; f < 10; ++f) dm[a][f] = R(0.01 * (a + 1) * (f + 1));
                   sources_point(P, m, K, dm, R(1.4), S); break; }
        case 11: { R acc = R(0.0); R div = (F[0] - F2[0]) / R(0.1); acc -= div; (void)acc; break; }
        default: return 1;
    }
    ops[0] = t_ops.add; ops[1] = t_ops.mul; ops[2] = t_ops.div; ops[3] = t_ops.sqrt;
    t_ops = {0, 0, 0, 0};
    return 0;
}

// NEXT-2: face fluxes of calB (FB, [nbox][9][Nz][Ny][Nx]) and the flux-CT update (dB, [nbox][3][Nz][Ny][Nx], interior cells).
int oracle_face_bfluxes(const int n[3], int nbox, const double* prim, const double* metric, int nghost, int recon,
                        double gamma, double* FB) {
    if (!n || !prim || !metric || !FB || nbox < 1 || n[0] < 1 || n[1] < 1 || n[2] < 1) return 1;
    if (recon != RECON_MINMOD && recon != RECON_MC && recon != RECON_WENO5) return 1;
    if (nghost < (recon == RECON_WENO5 ? 3 : 2) || !(gamma > 1.0)) return 1;
    Grid G;
    for (int a = 0; a < 3; ++a) { G.n[a] = n[a]; G.N[a] = n[a] + 2 * nghost; }
    G.g = nghost;
    G.ncell = (size_t)G.N[0] * G.N[1] * G.N[2];
    for (int b = 0; b < nbox; ++b)
        face_bflux_box(G, prim + (size_t)b * 8 * G.ncell, metric + (size_t)b * 10 * G.ncell, recon, gamma,
                       FB + (size_t)b * 9 * G.ncell);
    return 0;
}

int oracle_flux_ct(const int n[3], int nbox, const double* FB, const double dx[3], int nghost, double* dB) {
    if (!n || !FB || !dx || !dB || nbox < 1 || n[0] < 1 || n[1] < 1 || n[2] < 1 || nghost < 1) return 1;
    Grid G;
    for (int a = 0; a < 3; ++a) { G.n[a] = n[a]; G.N[a] = n[a] + 2 * nghost; }
    G.g = nghost;
    G.ncell = (size_t)G.N[0] * G.N[1] * G.N[2];
    for (int b = 0; b < nbox; ++b) flux_ct_box(G, FB + (size_t)b * 9 * G.ncell, dx, dB + (size_t)b * 3 * G.ncell);
    return 0;
}

// NEXT-3: right-hand side with vertex-centred metric and K (metv [nbox][10][Nz+1][Ny+1][Nx+1], Kv [nbox][6][...]) and
// T^{mu nu} at the vertices of the interior cells (T [nbox][10][Nz+1][Ny+1][Nx+1]).
static bool make_vgrid(const int n[3], int nghost, VGrid& V) {
    if (!n || n[0] < 1 || n[1] < 1 || n[2] < 1 || nghost < 0) return false;
    for (int a = 0; a < 3; ++a) { V.G.n[a] = n[a]; V.G.N[a] = n[a] + 2 * nghost; }
    V.G.g = nghost;
    V.G.ncell = (size_t)V.G.N[0] * V.G.N[1] * V.G.N[2];
    V.nv = (size_t)(V.G.N[0] + 1) * (V.G.N[1] + 1) * (V.G.N[2] + 1);
    return true;
}

int oracle_valencia_rhs_vertex(const int n[3], int nbox, const double* prim, const double* metv, const double* Kv,
                               const double dx[3], int nghost, int recon, double gamma, double* out,
                               unsigned long long* nfallback) {
    VGrid V;
    if (!make_vgrid(n, nghost, V) || !prim || !metv || !Kv || !dx || !out || nbox < 1) return 1;
    if (recon != RECON_MINMOD && recon != RECON_MC && recon != RECON_WENO5) return 1;
    if (nghost < (recon == RECON_WENO5 ? 3 : 2)) return 1;
    if (!(gamma > 1.0) || !(dx[0] > 0.0) || !(dx[1] > 0.0) || !(dx[2] > 0.0)) return 1;
    unsigned long long nfb = 0;
    for (int b = 0; b < nbox; ++b)
        rhs_vertex_box(V, prim + (size_t)b * 8 * V.G.ncell, metv + (size_t)b * 10 * V.nv, Kv + (size_t)b * 6 * V.nv, dx, recon,
                       gamma, out + (size_t)b * 8 * V.G.ncell, &nfb);
    if (nfallback) *nfallback = nfb;
    return 0;
}

int oracle_tmunu_vertices(const int n[3], int nbox, const double* prim, const double* metv, int nghost, double gamma,
                          double* T) {
    VGrid V;
    if (!make_vgrid(n, nghost, V) || !prim || !metv || !T || nbox < 1 || nghost < 2 || !(gamma > 1.0)) return 1;
    for (int b = 0; b < nbox; ++b)
        tmunu_vertex_box(V, prim + (size_t)b * 8 * V.G.ncell, metv + (size_t)b * 10 * V.nv, gamma, T + (size_t)b * 10 * V.nv);
    return 0;
}

double oracle_weno_eps(void) { return WENO_EPS; }
double oracle_v2max(void) { return V2MAX; }

}  // extern "C"
