"""Pins P1-P15, P17, P18: the CPU oracle against what the paper and the mathematics fix.

None of these tests touches the CUDA path.  Each pin is chosen so that a plausible mistake in the
oracle (dropped term, wrong sign or index, transposed operand) fails at least one of them.
Citations: PAPER.md line numbers; readings R* and pins P* are listed in DESIGN.md.
"""
import numpy as np
import pytest

from paper_2210_17509_b200 import inputs
from util import MET_FLAT, SYM, interior, make_problem, permute_problem, relerr_per_component

RNG = np.random.default_rng(12345)


# --------------------------------------------------------------------------------------------------
# P1  minmod (TVD, l.134/l.255): linear data reproduced exactly; zero slope at extrema; bounded
# --------------------------------------------------------------------------------------------------
def test_p1_minmod(oracle):
    for _ in range(50):
        a, b = RNG.normal(size=2)
        q = a + b * np.arange(-2, 3)
        qm, qp = oracle.recon_cell("minmod", q)
        assert qm == pytest.approx(a - 0.5 * b, abs=1e-15) and qp == pytest.approx(a + 0.5 * b, abs=1e-15)
        qm, qp = oracle.recon_cell("mc", q)
        assert qm == pytest.approx(a - 0.5 * b, abs=1e-15) and qp == pytest.approx(a + 0.5 * b, abs=1e-15)
    for rec in ("minmod", "mc"):
        assert oracle.recon_cell(rec, [0, 1.0, 3.0, 2.0, 0]) == (3.0, 3.0)      # local maximum
        assert oracle.recon_cell(rec, [0, 1.0, -3.0, 2.0, 0]) == (-3.0, -3.0)   # local minimum
        assert oracle.recon_cell(rec, [0, 1.0, 1.0, 2.0, 0]) == (1.0, 1.0)      # flat on one side
    for _ in range(200):
        q = RNG.normal(size=5)
        for rec in ("minmod", "mc"):
            qm, qp = oracle.recon_cell(rec, q)
            assert min(q[1], q[2]) - 1e-15 <= qm <= max(q[1], q[2]) + 1e-15
            assert min(q[2], q[3]) - 1e-15 <= qp <= max(q[2], q[3]) + 1e-15
    # minmod picks the smaller one-sided slope, MC the limited central slope (textbook, Toro [31])
    assert oracle.recon_cell("minmod", [0, 0.0, 1.0, 4.0, 0]) == (0.5, 1.5)
    assert oracle.recon_cell("minmod", [0, 0.0, 3.0, 4.0, 0]) == (2.5, 3.5)
    assert oracle.recon_cell("minmod", [0, 0.0, -3.0, -4.0, 0]) == (-2.5, -3.5)
    assert oracle.recon_cell("mc", [0, 0.0, 1.0, 4.0, 0]) == (0.0, 2.0)       # min(2*1, 2*3, 0.5*4) = 2
    assert oracle.recon_cell("mc", [0, 0.0, 2.0, 4.0, 0]) == (1.0, 3.0)       # central slope 2


# --------------------------------------------------------------------------------------------------
# P2  WENO5 (Jiang-Shu, ref [32]): exact for cell averages of quadratics whatever the weights; exact
#     for linear point data; 5th order on smooth data (needs the right linear weights); ENO property
# --------------------------------------------------------------------------------------------------
def _cell_avg_poly(coef, i):
    # exact cell average over [i-1/2, i+1/2] of sum_k coef[k] x^k
    P = np.polynomial.Polynomial(coef).integ()
    return P(i + 0.5) - P(i - 0.5)


def test_p2_weno5_polynomials(oracle):
    for _ in range(50):
        coef = RNG.normal(size=3)
        q = [_cell_avg_poly(coef, i) for i in range(-2, 3)]
        qm, qp = oracle.recon_cell("weno5", q)
        P = np.polynomial.Polynomial(coef)
        assert qm == pytest.approx(P(-0.5), abs=2e-14) and qp == pytest.approx(P(0.5), abs=2e-14)
    q = 3.0 - 2.0 * np.arange(-2, 3)
    assert oracle.recon_cell("weno5", q) == pytest.approx((4.0, 2.0), abs=1e-15)
    c = 0.7
    assert oracle.recon_cell("weno5", [c] * 5) == pytest.approx((c, c), abs=1e-15)


def test_p2_weno5_fifth_order(oracle):
    # cell averages of sin(x) on [0, 2 pi); error of the face values at i+1/2 and i-1/2
    errs = []
    for n in (16, 32, 64, 128):
        h = 2 * np.pi / n
        xc = (np.arange(-2, n + 2) + 0.5) * h
        avg = (np.cos(xc - h / 2) - np.cos(xc + h / 2)) / h
        e = 0.0
        for i in range(2, n + 2):
            qm, qp = oracle.recon_cell("weno5", avg[i - 2:i + 3])
            e = max(e, abs(qp - np.sin(xc[i] + h / 2)), abs(qm - np.sin(xc[i] - h / 2)))
        errs.append(e)
    orders = [np.log2(errs[k] / errs[k + 1]) for k in range(3)]
    # critical points of sin lower the classical JS weights' order locally towards 3 on coarse grids;
    # the max-norm order must still approach 5 and the error at n=128 must be at the 1e-8 level
    assert errs[-1] < 5e-8, errs
    assert orders[-1] > 4.5, (errs, orders)


def test_p2_weno5_step(oracle):
    # a jump between cells +1 and +2: q^+ must come from the smooth side and stay (nearly) constant
    qm, qp = oracle.recon_cell("weno5", [1.0, 1.0, 1.0, 1.0, 5.0])
    assert qp == pytest.approx(1.0, abs=1e-12) and qm == pytest.approx(1.0, abs=1e-12)
    qm, qp = oracle.recon_cell("weno5", [5.0, 1.0, 1.0, 1.0, 1.0])
    assert qp == pytest.approx(1.0, abs=1e-12) and qm == pytest.approx(1.0, abs=1e-12)
    # mirror property: reversing the stencil swaps the two faces (pins q^- against q^+)
    for _ in range(50):
        q = RNG.normal(size=5)
        qm, qp = oracle.recon_cell("weno5", q)
        rm, rp = oracle.recon_cell("weno5", q[::-1].copy())
        assert (qm, qp) == pytest.approx((rp, rm), rel=1e-12, abs=1e-14)


def test_p2_weno5_small_magnitude_fields(oracle):
    # R4: eps_w = 1e-26 must not linearise the scheme for atmosphere-sized data (rho ~ 1e-10)
    assert oracle.weno_eps() == 1e-26
    q = np.array([1.0, 1.0, 1.0, 1.0, 5.0]) * 1e-10
    qm, qp = oracle.recon_cell("weno5", q)
    assert qp == pytest.approx(1e-10, rel=1e-9)


# --------------------------------------------------------------------------------------------------
# helpers: random admissible state / metric
# --------------------------------------------------------------------------------------------------
def rand_metric(offdiag=0.15, shift=0.1):
    A = np.eye(3) + offdiag * RNG.normal(size=(3, 3))
    g = A @ A.T
    met = np.empty(10)
    met[0] = RNG.uniform(0.6, 1.2)
    met[1:4] = shift * RNG.normal(size=3)
    met[4:] = [g[0, 0], g[0, 1], g[0, 2], g[1, 1], g[1, 2], g[2, 2]]
    return met, g


def rand_state(g, vmax=0.7):
    v = RNG.normal(size=3)
    v *= RNG.uniform(0.05, vmax) / np.sqrt(v @ g @ v)
    B = RNG.normal(size=3)
    return np.array([RNG.uniform(0.1, 2.0), *v, RNG.uniform(0.05, 3.0), *B])


# --------------------------------------------------------------------------------------------------
# P3  HLLE consistency F^(U,U) = F(U);  P4 upwinding and the Rankine-Hugoniot limits
# --------------------------------------------------------------------------------------------------
def test_p3_hlle_consistency(oracle):
    for d in range(3):
        for _ in range(20):
            met, g = rand_metric()
            P = rand_state(g)
            U, F, lam = oracle.state_flux(P, met, d, 5.0 / 3.0)
            Fh = oracle.face_flux(P, P, P, P, met, d, 5.0 / 3.0)
            assert np.allclose(Fh, F, rtol=0, atol=1e-13 * np.abs(F).max())


def test_p4_hlle_upwind_and_rankine_hugoniot(oracle):
    UL, UR, FL, FR = RNG.normal(size=(4, 8))
    # all speeds positive -> F_L ; all negative -> F_R (R9: 0 is included in the min/max)
    assert np.allclose(oracle.hlle(UL, FL, [0.2, 0.9], UR, FR, [0.1, 0.8]), FL, rtol=5e-16, atol=0)
    assert np.allclose(oracle.hlle(UL, FL, [-0.9, -0.2], UR, FR, [-0.8, -0.1]), FR, rtol=5e-16, atol=0)
    # isolated discontinuity moving with the fastest right-going speed: F_R - F_L = s (U_R - U_L), s = lam+
    lm, lp = -0.4, 0.7
    FRr = FL + lp * (UR - UL)
    assert np.allclose(oracle.hlle(UL, FL, [lm, 0.1], UR, FRr, [-0.2, lp]), FL, atol=1e-14)
    FRl = FL + lm * (UR - UL)
    assert np.allclose(oracle.hlle(UL, FL, [lm, 0.1], UR, FRl, [-0.2, lp]), FRl, atol=1e-14)
    # symmetric fan, equal fluxes: pure diffusion -lam/2 (U_R-U_L) on top of the mean flux
    Fh = oracle.hlle(UL, FL, [-0.5, 0.5], UR, FL, [-0.5, 0.5])
    assert np.allclose(Fh, FL - 0.25 * (UR - UL), atol=1e-14)


# --------------------------------------------------------------------------------------------------
# P6  Minkowski => special-relativistic MHD, written independently in flat-space vector form
# --------------------------------------------------------------------------------------------------
def srmhd_flat(P, d, gamma):
    rho, eps = P[0], P[4]
    v, B = P[1:4], P[5:8]
    v2 = v @ v
    W = 1 / np.sqrt(1 - v2)
    p = (gamma - 1) * rho * eps
    rhoh = rho + rho * eps + p
    Bv, B2 = B @ v, B @ B
    b2 = B2 / W ** 2 + Bv ** 2
    ptot = p + 0.5 * b2
    D = rho * W
    S = (rhoh * W ** 2 + B2) * v - Bv * B
    E = rhoh * W ** 2 - p + 0.5 * B2 * (1 + v2) - 0.5 * Bv ** 2   # total energy density
    tau = E - D
    U = np.array([D, *S, tau, *B])
    bvec = B / W + W * Bv * v
    FS = S * v[d] - bvec * B[d] / W
    FS[d] += ptot
    Ftau = S[d] - D * v[d]                                          # energy flux = momentum density - mass flux
    FB = B * v[d] - B[d] * v
    F = np.array([D * v[d], *FS, Ftau, *FB])
    return U, F


def test_p6_minkowski_is_srmhd(oracle):
    for d in range(3):
        for _ in range(30):
            P = rand_state(np.eye(3), vmax=0.95)
            U, F, lam = oracle.state_flux(P, MET_FLAT, d, 4.0 / 3.0)
            U0, F0 = srmhd_flat(P, d, 4.0 / 3.0)
            W2 = 1 / (1 - P[1:4] @ P[1:4])
            assert np.allclose(U, U0, rtol=0, atol=4e-15 * W2 * np.abs(U0).max())
            assert np.allclose(F, F0, rtol=0, atol=4e-15 * W2 * np.abs(U0).max())


def test_p6_wave_speeds_closed_forms(oracle):
    gamma = 5.0 / 3.0
    for d in range(3):
        # pure hydro, flow along d: relativistic addition of v and c_s
        P = np.zeros(8)
        P[0], P[4], P[1 + d] = 1.3, 0.9, 0.45
        p = (gamma - 1) * P[0] * P[4]
        cs = np.sqrt(gamma * p / (P[0] * (1 + P[4]) + p))
        _, _, lam = oracle.state_flux(P, MET_FLAT, d, gamma)
        v = P[1 + d]
        assert lam == pytest.approx([(v - cs) / (1 - v * cs), (v + cs) / (1 + v * cs)], abs=1e-15)
        # fluid at rest, field perpendicular to d: exact perpendicular fast magnetosonic speed
        P = np.zeros(8)
        P[0], P[4], P[5 + (d + 1) % 3] = 0.8, 1.1, 1.7
        p = (gamma - 1) * P[0] * P[4]
        rhoh = P[0] * (1 + P[4]) + p
        cs2, va2 = gamma * p / rhoh, 1.7 ** 2 / (rhoh + 1.7 ** 2)
        a = np.sqrt(cs2 + va2 - cs2 * va2)
        _, _, lam = oracle.state_flux(P, MET_FLAT, d, gamma)
        assert lam == pytest.approx([-a, a], abs=1e-15)
    # coordinate speed in a constant lapse/shift/scale metric: lam = alpha * lam_flat / a_d - beta^d
    met = np.array([0.7, 0.1, -0.2, 0.05, 4.0, 0, 0, 9.0, 0, 0.25])
    P = np.array([1.0, 0.1, 0.05, -0.3, 0.5, 0.3, -0.2, 0.4])
    scale = np.array([2.0, 3.0, 0.5])
    Pflat = P.copy()
    Pflat[1:4] *= scale
    Pflat[5:8] *= scale
    for d in range(3):
        _, _, lam = oracle.state_flux(P, met, d, gamma)
        _, _, lam0 = oracle.state_flux(Pflat, MET_FLAT, d, gamma)
        assert lam == pytest.approx(0.7 * lam0 / scale[d] - met[1 + d], abs=1e-14)


def test_wave_speeds_solve_dispersion_relation(oracle):
    # R8: lam+- are the roots of (1-a^2)(u^mu k_mu)^2 - a^2 g^{mu nu} k_mu k_nu = 0 with k = (-lam, e_d)
    gamma = 5.0 / 3.0
    for d in range(3):
        for _ in range(20):
            met, g = rand_metric()
            P = rand_state(g)
            _, _, lam = oracle.state_flux(P, met, d, gamma)
            alp, beta = met[0], met[1:4]
            gi = np.linalg.inv(g)
            v, B = P[1:4], P[5:8]
            v2 = v @ g @ v
            W = 1 / np.sqrt(1 - v2)
            p = (gamma - 1) * P[0] * P[4]
            rhoh = P[0] * (1 + P[4]) + p
            b2 = (B @ g @ B) / W ** 2 + (B @ g @ v) ** 2
            cs2, va2 = gamma * p / rhoh, b2 / (rhoh + b2)
            a2 = cs2 + va2 - cs2 * va2
            u = W * np.array([1 / alp, *(v - beta / alp)])
            ginv4 = np.empty((4, 4))
            ginv4[0, 0] = -1 / alp ** 2
            ginv4[0, 1:] = ginv4[1:, 0] = beta / alp ** 2
            ginv4[1:, 1:] = gi - np.outer(beta, beta) / alp ** 2
            for l in lam:
                k = np.zeros(4)
                k[0], k[1 + d] = -l, 1.0
                res = (1 - a2) * (u @ k) ** 2 - a2 * (k @ ginv4 @ k)
                assert abs(res) < 1e-12 * W ** 2


# --------------------------------------------------------------------------------------------------
# P5  uniform state on ANY constant metric (shift, off-diagonals) => RHS = 0 exactly
# --------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("recon", ["minmod", "mc", "weno5"])
def test_p5_uniform_state_zero_rhs(oracle, recon):
    for flat in (True, False):
        met, g = (MET_FLAT, np.eye(3)) if flat else rand_metric()
        P = rand_state(g)
        prob = make_problem((6, 5, 4), (0, 0, 0), (1, 1, 1), 5.0 / 3.0, lambda X, Y, Z: list(P),
                            lambda X, Y, Z: list(met))
        out, nfb = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, 3, recon, prob.gamma)
        assert nfb == 0
        assert np.all(interior(prob, out) == 0.0)
        g_ = prob.nghost
        ghost = out.copy()
        ghost[prob.interior] = np.nan
        assert np.all(np.isnan(ghost))       # R23: ghost cells of `out` are never written
        assert g_ == 3


# --------------------------------------------------------------------------------------------------
# smooth random problem on a general metric (shared by P7, P8, P18)
# --------------------------------------------------------------------------------------------------
def general_problem(n=(10, 8, 6)):
    return inputs.general_metric_box(n=n, seed=99)


# P7  axis permutation (x,y,z) -> (y,z,x) permutes the output
@pytest.mark.parametrize("recon", ["minmod", "weno5"])
def test_p7_axis_permutation(oracle, recon):
    prob = general_problem()
    out, _ = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, 3, recon, prob.gamma)
    p2, tr, old_of_new = permute_problem(prob)
    out2, _ = oracle.valencia_rhs(p2.prim, p2.metric, p2.K, p2.dx, 3, recon, p2.gamma)
    exp = tr(out)
    exp2 = exp.copy()
    for a in range(3):
        exp2[:, 1 + a] = exp[:, 1 + old_of_new[a]]
        exp2[:, 5 + a] = exp[:, 5 + old_of_new[a]]
    err = relerr_per_component(interior(p2, out2), interior(p2, exp2))
    assert err.max() < 5e-14, err


# P8  mirror x -> -x: dS_x and dB^x flip sign, everything else is even (pins q^- against q^+ on the grid)
@pytest.mark.parametrize("recon", ["minmod", "mc", "weno5"])
def test_p8_mirror(oracle, recon):
    prob = general_problem()
    out, _ = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, 3, recon, prob.gamma)
    flip = lambda a: np.ascontiguousarray(a[..., ::-1])   # noqa: E731
    prim, met, K = flip(prob.prim), flip(prob.metric), flip(prob.K)
    prim[:, 1] *= -1
    prim[:, 5] *= -1
    met[:, 1] *= -1
    met[:, 5] *= -1
    met[:, 6] *= -1
    K[:, 1] *= -1
    K[:, 2] *= -1
    out2, _ = oracle.valencia_rhs(prim, met, K, prob.dx, 3, recon, prob.gamma)
    exp = flip(out)
    exp[:, 1] *= -1
    exp[:, 5] *= -1
    err = relerr_per_component(interior(prob, out2), interior(prob, exp))
    assert err.max() < 2e-14, err


# P9  constant diagonal metric diag(a^2,b^2,c^2), constant lapse == Minkowski in rescaled coordinates
def test_p9_constant_diagonal_metric(oracle):
    base = inputs.sweep_boxes(8, 1)
    a = np.array([1.3, 0.8, 1.7])
    alp0 = 0.75
    met = np.zeros_like(base.metric)
    met[:, 0] = alp0
    met[:, 4], met[:, 7], met[:, 9] = a[0] ** 2, a[1] ** 2, a[2] ** 2
    K0 = np.zeros_like(base.K)
    out, _ = oracle.valencia_rhs(base.prim, met, K0, base.dx, 3, "weno5", base.gamma)
    # orthonormal-frame problem: v' = a v, B' = a B, dx' = a dx on Minkowski
    prim2 = base.prim.copy()
    for i in range(3):
        prim2[:, 1 + i] *= a[i]
        prim2[:, 5 + i] *= a[i]
    met2 = np.zeros_like(met)
    met2[:, 0] = met2[:, 4] = met2[:, 7] = met2[:, 9] = 1.0
    dx2 = tuple(base.dx[i] * a[i] for i in range(3))
    out2, _ = oracle.valencia_rhs(prim2, met2, K0, dx2, 3, "weno5", base.gamma)
    vol = alp0 * a.prod()
    exp = out2.copy()
    exp[:, 0] *= vol
    exp[:, 4] *= vol
    for i in range(3):
        exp[:, 1 + i] *= vol * a[i]
        exp[:, 5 + i] *= vol / a[i]
    err = relerr_per_component(interior(base, out), interior(base, exp))
    assert err.max() < 5e-14, err


# P10 sheared coordinates y' = y - s x on Balsara-1 data: exercises the off-diagonal metric exactly
@pytest.mark.parametrize("recon", ["minmod", "weno5"])
def test_p10_shear(oracle, recon):
    prob = inputs.balsara1()
    out, _ = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, 3, recon, prob.gamma)
    s = 0.37
    met = prob.metric.copy()
    met[:, 4] = 1 + s * s      # gamma_xx
    met[:, 5] = s              # gamma_xy
    prim = prob.prim.copy()
    prim[:, 6] = prob.prim[:, 6] - s * prob.prim[:, 5]     # B'^y = B^y - s B^x   (v = 0)
    out2, _ = oracle.valencia_rhs(prim, met, prob.K, prob.dx, 3, recon, prob.gamma)
    exp = out.copy()
    exp[:, 1] = out[:, 1] + s * out[:, 2]                   # S'_x = S_x + s S_y
    exp[:, 6] = out[:, 6] - s * out[:, 5]                   # calB'^y = calB^y - s calB^x
    diff = np.abs(interior(prob, out2) - interior(prob, exp)).max()
    assert diff < 2e-13, diff


# --------------------------------------------------------------------------------------------------
# P11 hydrostatic balance: static fluid, static metric => dS_j -> -sqrt(gamma)(alpha d_j p + rho h d_j alpha)
# --------------------------------------------------------------------------------------------------
def test_p11_hydrostatic_convergence(oracle):
    gamma = 2.0
    M = 1.4

    def fields(X, Y, Z):
        r2 = X * X + Y * Y + Z * Z
        s = np.sqrt(r2 + 9.0)            # softened so the coarse grids resolve the metric
        u = M / (2 * s)
        psi = 1 + u
        alp = (1 - u) / (1 + u)
        rho = 1.28e-3 * np.exp(-r2 / 36.0) + 1e-5
        p = 100.0 * rho * rho
        return r2, s, u, psi, alp, rho, p

    errs, resid = [], []
    for N in (16, 32, 64):
        def prim_fn(X, Y, Z):
            *_, rho, p = fields(X, Y, Z)
            return [rho, 0, 0, 0, p / ((gamma - 1) * rho), 0, 0, 0]

        def met_fn(X, Y, Z):
            r2, s, u, psi, alp, rho, p = fields(X, Y, Z)
            return [alp, 0, 0, 0, psi ** 4, 0, 0, psi ** 4, 0, psi ** 4]

        prob = make_problem((N, N, N), (-8, -8, -8), (8, 8, 8), gamma, prim_fn, met_fn)
        out, _ = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, 3, "weno5", gamma)
        o = interior(prob, out)[0]
        # analytic balance at the cell centres
        g = 3
        ax = -8 + (np.arange(N) + 0.5) * 16 / N
        X, Y, Z = ax[None, None, :], ax[None, :, None], ax[:, None, None]
        r2, s, u, psi, alp, rho, p = fields(X, Y, Z)
        rhoh = rho + 2 * p      # Gamma = 2: rho eps = p
        sg = psi ** 6
        h = 1e-5
        for j, (dxx, dyy, dzz) in enumerate(((h, 0, 0), (0, h, 0), (0, 0, h))):
            fp = fields(X + dxx, Y + dyy, Z + dzz)
            fm = fields(X - dxx, Y - dyy, Z - dzz)
            dp = (fp[6] - fm[6]) / (2 * h)
            da = (fp[4] - fm[4]) / (2 * h)
            exact = -sg * (alp * dp + rhoh * da)
            if j == 0:
                num, ref = np.abs(o[1] - exact).max(), np.abs(exact).max()
        errs.append(num / ref)
        assert np.abs(o[5:]).max() == 0.0                                     # dB = 0 exactly for B = 0
        # dD, dtau: only the HLLE diffusion of the (high-order small) reconstruction jumps survives
        resid.append((np.abs(o[0]).max(), np.abs(o[4]).max()))
    assert resid[1][0] < resid[0][0] / 8 and resid[2][0] < resid[1][0] / 8, resid
    assert resid[1][1] < resid[0][1] / 8 and resid[2][1] < resid[1][1] / 8, resid
    assert errs[0] > errs[1] > errs[2]
    # 2nd order asymptotically (2-point face average of the metric; cf. l.319 "convergence order ~2");
    # measured here: 1.5e-2, 4.5e-3, 1.6e-3 (4.4e-4 at N = 128)
    assert np.log2(errs[1] / errs[2]) > 1.4 and errs[0] / errs[2] > 8, errs
    assert errs[2] < 2e-2, errs


# --------------------------------------------------------------------------------------------------
# P12 FLRW slice: gamma_ij = a^2 delta_ij, K_ij = -a adot delta_ij, alpha = 1: d tau = -a^2 adot (3p + b^2/2)
#     (first law of thermodynamics; pins the sign convention of K_ij, R12)
# --------------------------------------------------------------------------------------------------
def test_p12_flrw(oracle):
    a, adot, gamma = 1.3, 0.21, 5.0 / 3.0
    rho, eps, Bx = 0.9, 0.6, 0.35
    prob = make_problem((5, 4, 4), (0, 0, 0), (1, 1, 1), gamma,
                        lambda X, Y, Z: [rho, 0, 0, 0, eps, Bx, 0, 0],
                        lambda X, Y, Z: [1, 0, 0, 0, a * a, 0, 0, a * a, 0, a * a],
                        lambda X, Y, Z: [-a * adot, 0, 0, -a * adot, 0, -a * adot])
    out, _ = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, 3, "weno5", gamma)
    o = interior(prob, out)[0]
    p = (gamma - 1) * rho * eps
    b2 = a * a * Bx * Bx
    assert np.allclose(o[4], -a * a * adot * (3 * p + 0.5 * b2), rtol=1e-14)
    for c in (0, 1, 2, 3, 5, 6, 7):
        assert np.abs(o[c]).max() < 1e-15


# P13 shearing shift beta^x = omega y on flat space: dS_y = omega S_x, dB^x = -omega B^y (linear data: exact)
def test_p13_shearing_shift(oracle):
    om, gamma = 0.3, 5.0 / 3.0
    P = np.array([1.1, 0.4, 0.0, 0.0, 0.7, 0.0, 0.2, 0.0])
    prob = make_problem((6, 6, 4), (-1, -1, 0), (1, 1, 1), gamma, lambda X, Y, Z: list(P),
                        lambda X, Y, Z: [1, om * Y, 0, 0, 1, 0, 0, 1, 0, 1])
    for recon in ("minmod", "weno5"):
        out, _ = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, 3, recon, gamma)
        o = interior(prob, out)[0]
        U, _, _ = oracle.state_flux(P, MET_FLAT, 0, gamma)
        assert np.allclose(o[2], om * U[1], rtol=1e-13)
        assert np.allclose(o[5], -om * U[6], rtol=1e-13)      # induction: d calB^x = -d_y(-calB^y vtilde^x)
        for c in (0, 1, 3, 4, 6, 7):
            assert np.abs(o[c]).max() < 2e-15, (c, np.abs(o[c]).max())


# P14 Rindler-like lapse alpha = 1 + g x, static uniform fluid: dS_x = -rho h g, everything else 0
def test_p14_rindler(oracle):
    gacc, gamma = 0.4, 5.0 / 3.0
    rho, eps = 0.9, 0.3
    prob = make_problem((6, 4, 4), (0, 0, 0), (1, 1, 1), gamma, lambda X, Y, Z: [rho, 0, 0, 0, eps, 0, 0, 0],
                        lambda X, Y, Z: [1 + gacc * X, 0, 0, 0, 1, 0, 0, 1, 0, 1])
    for recon in ("minmod", "weno5"):
        out, _ = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, 3, recon, gamma)
        o = interior(prob, out)[0]
        rhoh = rho * (1 + eps) + (gamma - 1) * rho * eps
        assert np.allclose(o[1], -rhoh * gacc, rtol=1e-13)
        for c in (0, 2, 3, 4, 5, 6, 7):
            assert np.abs(o[c]).max() < 1e-15


# --------------------------------------------------------------------------------------------------
# P15 the 3+1 sources against the paper's literal 4-D Eq. (13) (l.112) with exact Christoffel symbols
# --------------------------------------------------------------------------------------------------
def eq13_sources_4d(P, met, K, dm, gamma, dt_alp, dt_beta):
    """S_{S_j} = alpha sqrt(gamma) T^{mu nu}(d_mu g_{nu j} - Gamma^lam_{mu nu} g_{lam j}),
       S_tau   = alpha sqrt(gamma) alpha (T^{mu 0} d_mu ln alpha - T^{mu nu} Gamma^0_{mu nu})."""
    alp, beta = met[0], met[1:4]
    g = np.array([[met[4 + SYM[i][j]] for j in range(3)] for i in range(3)])
    Kij = np.array([[K[SYM[i][j]] for j in range(3)] for i in range(3)])
    dalp = np.array([dt_alp, dm[0][0], dm[1][0], dm[2][0]])                  # d_mu alpha
    dbeta = np.zeros((4, 3))                                                  # d_mu beta^i
    dbeta[0] = dt_beta
    for a in range(3):
        dbeta[1 + a] = dm[a][1:4]
    dg3 = np.zeros((4, 3, 3))                                                 # d_mu gamma_ij
    for a in range(3):
        dg3[1 + a] = [[dm[a][4 + SYM[i][j]] for j in range(3)] for i in range(3)]
    # ADM evolution equation: d_t gamma_ij = -2 alpha K_ij + L_beta gamma_ij
    lie = np.einsum("k,kij->ij", beta, dg3[1:]) + np.einsum("kj,ik->ij", g, dbeta[1:]) + np.einsum("ik,jk->ij", g, dbeta[1:])
    dg3[0] = -2 * alp * Kij + lie
    # 4-metric and its derivatives
    g4 = np.zeros((4, 4))
    bl = g @ beta
    g4[0, 0] = -alp ** 2 + beta @ bl
    g4[0, 1:] = g4[1:, 0] = bl
    g4[1:, 1:] = g
    dg4 = np.zeros((4, 4, 4))                                                 # dg4[mu, a, b] = d_mu g_ab
    for mu in range(4):
        dbl = dg3[mu] @ beta + g @ dbeta[mu]
        dg4[mu, 0, 0] = -2 * alp * dalp[mu] + dbl @ beta + bl @ dbeta[mu]
        dg4[mu, 0, 1:] = dg4[mu, 1:, 0] = dbl
        dg4[mu, 1:, 1:] = dg3[mu]
    gi4 = np.linalg.inv(g4)
    Gam = np.zeros((4, 4, 4))                                                 # Gam[l, m, n]
    for l in range(4):
        for m in range(4):
            for n in range(4):
                Gam[l, m, n] = 0.5 * sum(gi4[l, s] * (dg4[m, s, n] + dg4[n, s, m] - dg4[s, m, n]) for s in range(4))
    # fluid: u^mu, b^mu, T^{mu nu} (Eq. 5)
    rho, eps = P[0], P[4]
    v, B = P[1:4], P[5:8]
    W = 1 / np.sqrt(1 - v @ g @ v)
    u = W * np.array([1 / alp, *(v - beta / alp)])
    B4 = np.array([0.0, *B])
    ul = g4 @ u
    b = (B4 + (ul @ B4) * u) / W
    assert abs(u @ g4 @ u + 1) < 1e-12 and abs(b @ g4 @ u) < 1e-12
    b2 = b @ g4 @ b
    p = (gamma - 1) * rho * eps
    T = (rho * (1 + eps) + p + b2) * np.outer(u, u) + (p + 0.5 * b2) * gi4 - np.outer(b, b)
    sg = np.sqrt(np.linalg.det(g))
    S = np.zeros(8)
    for j in range(3):
        S[1 + j] = alp * sg * sum(T[m, n] * (dg4[m, n, 1 + j] - sum(Gam[l, m, n] * g4[l, 1 + j] for l in range(4)))
                                  for m in range(4) for n in range(4))
    S[4] = alp * sg * alp * (sum(T[m, 0] * dalp[m] / alp for m in range(4)) -
                             sum(T[m, n] * Gam[0, m, n] for m in range(4) for n in range(4)))
    return S


def test_p15_sources_vs_4d_equation_13(oracle):
    gamma = 5.0 / 3.0
    for trial in range(25):
        met, g = rand_metric(offdiag=0.2, shift=0.2)
        P = rand_state(g)
        K = 0.3 * RNG.normal(size=6)
        dm = 0.3 * RNG.normal(size=(3, 10))
        S = oracle.sources_point(P, met, K, dm, gamma)
        # the gauge time derivatives drop out of Eq. (13): any value must give the same sources
        S4 = eq13_sources_4d(P, met, K, dm, gamma, dt_alp=RNG.normal(), dt_beta=RNG.normal(size=3))
        assert S[0] == 0 and np.all(S[5:] == 0)
        assert np.allclose(S, S4, rtol=0, atol=1e-11 * np.abs(S4).max()), (trial, S, S4)


# --------------------------------------------------------------------------------------------------
# P17 prim2con: Eqs. (6)-(9) against the classical forms, and the con2prim round trip (R22)
# --------------------------------------------------------------------------------------------------
def test_p17_prim2con_classical_forms_and_roundtrip(oracle):
    prob = general_problem((7, 6, 5))
    cons = oracle.prim2con(prob.prim, prob.metric, 3, prob.gamma)
    P, m = prob.prim[0], prob.metric[0]
    g = [[m[4 + SYM[i][j]] for j in range(3)] for i in range(3)]
    v, B = P[1:4], P[5:8]
    vl = [sum(g[i][j] * v[j] for j in range(3)) for i in range(3)]
    Bl = [sum(g[i][j] * B[j] for j in range(3)) for i in range(3)]
    v2 = sum(vl[i] * v[i] for i in range(3))
    B2 = sum(Bl[i] * B[i] for i in range(3))
    Bv = sum(Bl[i] * v[i] for i in range(3))
    W = 1 / np.sqrt(1 - v2)
    det = (g[0][0] * (g[1][1] * g[2][2] - g[1][2] ** 2) - g[0][1] * (g[0][1] * g[2][2] - g[1][2] * g[0][2])
           + g[0][2] * (g[0][1] * g[1][2] - g[1][1] * g[0][2]))
    sg = np.sqrt(det)
    rho, eps = P[0], P[4]
    p = (prob.gamma - 1) * rho * eps
    rhoh = rho * (1 + eps) + p
    assert np.allclose(cons[0, 0], sg * rho * W, rtol=1e-14)
    for j in range(3):
        assert np.allclose(cons[0, 1 + j], sg * ((rhoh * W ** 2 + B2) * vl[j] - Bv * Bl[j]), rtol=1e-12, atol=1e-14)
        assert np.allclose(cons[0, 5 + j], sg * B[j], rtol=1e-15)
    tau = sg * (rho * W * (W - 1) + rho * eps * W ** 2 + p * (W ** 2 - 1) + 0.5 * (B2 * (1 + v2) - Bv ** 2))
    assert np.allclose(cons[0, 4], tau, rtol=1e-12)
    prim_back, nfail = oracle.con2prim(cons, prob.metric, 3, prob.gamma)
    assert nfail == 0
    assert np.allclose(prim_back, prob.prim, rtol=1e-10, atol=1e-12)


# --------------------------------------------------------------------------------------------------
# P18 the oracle's own rounding: long double instance vs double instance (must be << 1e-11)
# --------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name,recon", [("c1", "minmod"), ("c1", "weno5"), ("c2:small", "weno5"), ("c2:small", "minmod"),
                                         ("c3:small", "weno5"), ("c4:small", "weno5"), ("c5-32:small", "weno5"),
                                         ("gen", "weno5"), ("gen", "mc")])
def test_p18_double_vs_long_double(oracle, name, recon):
    prob = inputs.by_name(name)
    out, nfb = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, prob.nghost, recon, prob.gamma)
    ref, nfb2 = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, prob.nghost, recon, prob.gamma,
                                    variant="long double")
    assert nfb == nfb2
    err = relerr_per_component(interior(prob, out), interior(prob, ref))
    assert err.max() < 5e-13, err


def test_argument_validation(oracle):
    prob = inputs.balsara1()
    with pytest.raises(ValueError):
        oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, 2, "weno5", prob.gamma)     # R29
    with pytest.raises(ValueError):
        oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, 3, "weno5", 1.0)
    with pytest.raises(ValueError):
        oracle.valencia_rhs(prob.prim, prob.metric, prob.K, (0.1, 0.0, 0.1), 3, "weno5", prob.gamma)


def test_config2_fallback_count(oracle):
    """R5 is needed: WENO5 on the rotor overshoots v^2 >= 1 at 64 face sides; minmod at none."""
    prob = inputs.rotor()
    _, nfb = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, 3, "weno5", prob.gamma)
    assert nfb == 64
    _, nfb = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, 3, "minmod", prob.gamma)
    assert nfb == 0


def test_r5_admissibility_uses_the_face_metric(oracle):
    """R5 on a non-flat metric: v^2 = gamma_ij v^i v^j with the FACE metric decides, not the coordinate components.
    (a) gamma_xx = 4, v^x = 0.6: v^2 = 1.44 -> the side falls back to its donor cell, so the face flux is exactly the one
        computed from the donor's centre values; the same state is admissible (and gives another flux) on the flat metric.
    (b) gamma_xx = 0.25, v^x = 1.5: v^2 = 0.5625 -> admissible although the coordinate velocity exceeds 1: the flux is finite
        and is NOT the fallback's.
    (c) rho <= 0, eps <= 0 and NaN fail the test too."""
    gamma = 5.0 / 3.0
    CL = np.array([1.0, 0.1, 0.05, -0.02, 0.8, 0.3, 0.2, -0.1])
    CR = np.array([0.9, 0.12, 0.02, 0.01, 0.7, 0.3, 0.25, -0.05])
    flat = np.array([1.0, 0, 0, 0, 1, 0, 0, 1, 0, 1.0])
    g4 = flat.copy(); g4[4] = 4.0
    gq = flat.copy(); gq[4] = 0.25
    PL = CL.copy(); PL[1] = 0.6
    for d in range(3):
        # (a)
        assert np.array_equal(oracle.face_flux(PL, CR, CL, CR, g4, d, gamma), oracle.face_flux(CL, CR, CL, CR, g4, d, gamma))
        assert not np.array_equal(oracle.face_flux(PL, CR, CL, CR, flat, d, gamma), oracle.face_flux(CL, CR, CL, CR, flat, d, gamma))
        # the right side is checked independently of the left one
        PR = CR.copy(); PR[1] = -0.6
        assert np.array_equal(oracle.face_flux(CL, PR, CL, CR, g4, d, gamma), oracle.face_flux(CL, CR, CL, CR, g4, d, gamma))
        # (b)
        fast = CL.copy(); fast[1] = 1.5
        F = oracle.face_flux(fast, CR, CL, CR, gq, d, gamma)
        assert np.all(np.isfinite(F)) and not np.array_equal(F, oracle.face_flux(CL, CR, CL, CR, gq, d, gamma))
        # (c)
        for q, bad in ((0, 0.0), (0, -1.0), (4, 0.0), (4, -0.3), (2, np.nan)):
            P = CL.copy(); P[q] = bad
            assert np.array_equal(oracle.face_flux(P, CR, CL, CR, flat, d, gamma), oracle.face_flux(CL, CR, CL, CR, flat, d, gamma))
    # the bound itself: v^2 just below / at 1 - 1e-4 (V2MAX)
    for v, falls in ((np.sqrt(oracle.v2max()) * (1 - 1e-12), False), (np.sqrt(oracle.v2max()) * (1 + 1e-12), True)):
        P = CL.copy(); P[1:4] = (v, 0.0, 0.0)
        same = np.array_equal(oracle.face_flux(P, CR, CL, CR, flat, 0, gamma), oracle.face_flux(CL, CR, CL, CR, flat, 0, gamma))
        assert same == falls
