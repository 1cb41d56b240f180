"""Pins of the oracle's vertex-centred spacetime path (NEXT-3; readings R31 / R32).

R31, the right-hand side with the metric and K_ij sampled at the cell vertices (face = mean of 4 vertices, centre = mean of
8, staggered 4th-order derivative):
  V1  a metric that is LINEAR in the coordinates: 4- and 8-vertex means are exact at the face and cell centres and both
      derivative stencils are exact, so the vertex path must reproduce the (independently pinned) cell-centred path;
  V2  uniform state on a constant metric: exactly zero (P5 on the vertex path);
  V3  smooth metric: the two paths agree to second order in the cell size;
  V4  cyclic permutation of the axes permutes the result (vertex indexing treats the three directions alike);
  V5  the staggered derivative and the 4-vertex face mean are exact for a lapse that is cubic in one coordinate (closed
      form of dS_k for a fluid at rest).
R32, T^{mu nu} at the vertices from 4th-order interpolated primitives:
  W1  closed forms on Minkowski: fluid at rest, boosted fluid, magnetic field at rest;
  W2  the trace g_{mu nu} T^{mu nu} = -rho (1 + eps) + 3 p on random general metrics (the field part is traceless): every
      index placement of Eq. (5) and of the 3+1 inverse metric enters;
  W3  the interpolation is exact for tri-cubic polynomials and fourth-order accurate on smooth data.
"""
import numpy as np
import pytest

from paper_2210_17509_b200 import inputs
from util import SYM, permute_problem, relerr_per_component

G = inputs.NGHOST


def _axes(n, lo, hi, g, vertex):
    dx = [(hi[d] - lo[d]) / n[d] for d in range(3)]
    ax = []
    for d in range(3):
        i = np.arange(-g, n[d] + g + (1 if vertex else 0))
        ax.append(lo[d] + (i + (0.0 if vertex else 0.5)) * dx[d])
    X = ax[0][None, None, :]
    Y = ax[1][None, :, None]
    Z = ax[2][:, None, None]
    shape = (len(ax[2]), len(ax[1]), len(ax[0]))
    return tuple(np.broadcast_to(a, shape) for a in (X, Y, Z)), dx


def _fields(fn, n, lo, hi, g, vertex):
    (X, Y, Z), dx = _axes(n, lo, hi, g, vertex)
    vals = fn(X, Y, Z)
    return np.stack([np.broadcast_to(np.asarray(v, dtype=float), X.shape) for v in vals])[None].copy(), dx


def _prim_fn(X, Y, Z):
    s = np.sin(1.3 * X + 0.4) * np.cos(0.9 * Y - 0.2) + 0.5 * np.sin(0.7 * Z + X)
    c = np.cos(0.8 * X - 0.5 * Y + 0.3 * Z)
    rho = 1.0 + 0.3 * s
    eps = 0.8 + 0.3 * c
    return [rho, 0.2 * s, -0.15 * c, 0.1 * s * c, eps, 0.3 * c, 0.2 + 0.1 * s, -0.25 * s]


def _linear_metric(X, Y, Z):
    L = lambda a, b, c, d: a + b * X + c * Y + d * Z     # noqa: E731
    return [L(0.9, 0.02, -0.01, 0.015), L(0.02, 0.004, 0.003, -0.002), L(-0.01, 0.002, -0.004, 0.001),
            L(0.015, -0.003, 0.001, 0.002), L(1.2, 0.02, 0.01, -0.015), L(0.05, 0.004, -0.003, 0.002),
            L(-0.03, 0.001, 0.002, 0.003), L(1.1, -0.01, 0.02, 0.01), L(0.04, 0.002, 0.001, -0.002),
            L(0.95, 0.015, -0.01, 0.02)]


def _linear_K(X, Y, Z):
    return [0.03 + 0.002 * X, -0.01 + 0.001 * Y, 0.02 - 0.001 * Z, 0.01 + 0.002 * Z, -0.02 + 0.001 * X, 0.015 - 0.002 * Y]


def _smooth_metric(X, Y, Z):
    s = np.sin(0.9 * X + 0.3) * np.cos(0.7 * Y) + 0.4 * np.sin(0.5 * Z - X)
    c = np.cos(0.6 * X + 0.8 * Y - 0.4 * Z)
    psi4 = (1.1 + 0.05 * s) ** 4
    return [0.9 + 0.05 * c, 0.02 * s, -0.015 * c, 0.01 * s * c, psi4 * (1 + 0.05 * c), psi4 * 0.03 * s, psi4 * 0.02 * c,
            psi4 * (1 - 0.04 * s), psi4 * 0.025 * s * c, psi4 * (1 + 0.03 * s)]


def _smooth_K(X, Y, Z):
    s = np.sin(0.8 * X - 0.6 * Y + 0.2 * Z)
    return [0.03 * s, -0.01 * s, 0.02 * s, 0.01 * s, -0.02 * s, 0.015 * s]


def _both(n, lo, hi, metric_fn, K_fn, prim_fn=_prim_fn):
    prim, dx = _fields(prim_fn, n, lo, hi, G, False)
    met_c, _ = _fields(metric_fn, n, lo, hi, G, False)
    K_c, _ = _fields(K_fn, n, lo, hi, G, False)
    met_v, _ = _fields(metric_fn, n, lo, hi, G, True)
    K_v, _ = _fields(K_fn, n, lo, hi, G, True)
    return prim, met_c, K_c, met_v, K_v, dx


def _int(a):
    return a[..., G:-G, G:-G, G:-G]


@pytest.mark.parametrize("recon", ["minmod", "weno5"])
def test_V1_linear_metric_reproduces_the_cell_centred_path(oracle, recon):
    n, lo, hi = (10, 8, 7), (-1.0, -0.8, -0.7), (1.0, 0.8, 0.7)
    prim, met_c, K_c, met_v, K_v, dx = _both(n, lo, hi, _linear_metric, _linear_K)
    ref, nf = oracle.valencia_rhs(prim, met_c, K_c, dx, G, recon, 5.0 / 3.0)
    got, nf2 = oracle.valencia_rhs_vertex(prim, met_v, K_v, dx, G, recon, 5.0 / 3.0)
    assert nf == nf2
    assert relerr_per_component(_int(got), _int(ref)).max() < 2e-13
    assert np.all(np.isnan(got[..., 0])), "ghost cells of out are not written"


def test_V2_uniform_state_constant_metric_exact_zero(oracle):
    n = (6, 5, 4)
    pv = [0.7, 0.2, -0.1, 0.3, 1.3, 0.4, -0.2, 0.1]
    mv = [0.9, 0.02, -0.03, 0.01, 1.2, 0.1, -0.05, 1.1, 0.07, 0.95]
    prim, _, _, met_v, K_v, dx = _both(n, (0, 0, 0), (1, 1, 1), lambda X, Y, Z: mv, lambda X, Y, Z: [0.0] * 6,
                                       lambda X, Y, Z: pv)
    for recon in ("minmod", "mc", "weno5"):
        got, _ = oracle.valencia_rhs_vertex(prim, met_v, K_v, dx, G, recon, 1.4)
        assert np.abs(_int(got)).max() == 0.0


def test_V3_smooth_metric_second_order_agreement(oracle):
    errs = []
    for N in (8, 16, 32):
        n = (N, N, N)
        prim, met_c, K_c, met_v, K_v, dx = _both(n, (-1, -1, -1), (1, 1, 1), _smooth_metric, _smooth_K)
        ref, _ = oracle.valencia_rhs(prim, met_c, K_c, dx, G, "weno5", 5.0 / 3.0)
        got, _ = oracle.valencia_rhs_vertex(prim, met_v, K_v, dx, G, "weno5", 5.0 / 3.0)
        errs.append(np.abs(_int(got) - _int(ref)).max() / np.abs(_int(ref)).max())
    assert errs[0] / errs[1] > 3.4 and errs[1] / errs[2] > 3.7 and errs[2] < 2e-3, errs


def test_V4_axis_permutation_covariance(oracle):
    n, lo, hi = (9, 7, 6), (-0.9, -0.7, -0.6), (0.9, 0.7, 0.6)
    prim, met_c, K_c, met_v, K_v, dx = _both(n, lo, hi, _smooth_metric, _smooth_K)
    out, _ = oracle.valencia_rhs_vertex(prim, met_v, K_v, dx, G, "weno5", 5.0 / 3.0)
    # the permuted problem: cell arrays through util.permute_problem, vertex arrays by the same relabelling
    probc = inputs.Problem("v", n, 1, G, tuple(dx), 5.0 / 3.0, prim, met_c, K_c)
    p2, tr, old_of_new = permute_problem(probc)
    mv = tr(met_v)
    kv = tr(K_v)
    mv2, kv2 = mv.copy(), kv.copy()
    for a in range(3):
        mv2[:, 1 + a] = mv[:, 1 + old_of_new[a]]
        for b in range(a, 3):
            mv2[:, 4 + SYM[a][b]] = mv[:, 4 + SYM[old_of_new[a]][old_of_new[b]]]
            kv2[:, SYM[a][b]] = kv[:, SYM[old_of_new[a]][old_of_new[b]]]
    out2, _ = oracle.valencia_rhs_vertex(p2.prim, mv2, kv2, p2.dx, G, "weno5", 5.0 / 3.0)
    exp = tr(out)
    exp2 = exp.copy()
    for a in range(3):
        exp2[:, 1 + a] = exp[:, 1 + old_of_new[a]]
        exp2[:, 5 + a] = exp[:, 5 + old_of_new[a]]
    assert relerr_per_component(_int(out2), _int(exp2)).max() < 5e-14


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_V5_staggered_derivative_exact_for_cubics(oracle, axis):
    """Fluid at rest with uniform rho, eps and no field on gamma_ij = delta_ij, beta = 0, alpha = 1 + a1 t + a3 t^3 along one
    coordinate t.  Then F^k(S_k) = alpha_face p with the EXACT face lapse (the four vertices of a face share t), and the
    only source is S_{S_k} = -E d_k alpha with E = rho (1 + eps) (3+1 form of Eq. 13), so
        dS_k = -p (alpha(t + h/2) - alpha(t - h/2)) / h - rho (1 + eps) alpha'(t)
    holds to rounding exactly if the staggered stencil differentiates the cubic exactly (the centred stencil of the cell-
    centred path would too; the 2-point face average of that path would not)."""
    n, lo, hi = (8, 8, 8), (-1.0, -1.0, -1.0), (1.0, 1.0, 1.0)
    rho0, eps0 = 1.3, 0.6
    prim_fn = lambda X, Y, Z: [rho0, 0, 0, 0, eps0, 0, 0, 0]     # noqa: E731
    coord = lambda X, Y, Z: (X, Y, Z)[axis]                        # noqa: E731
    a3, a1 = 0.05, 0.1
    met_fn = lambda X, Y, Z: [1.0 + a1 * coord(X, Y, Z) + a3 * coord(X, Y, Z) ** 3, 0, 0, 0, 1, 0, 0, 1, 0, 1]     # noqa: E731
    prim, _, _, met_v, K_v, dx = _both(n, lo, hi, met_fn, lambda X, Y, Z: [0.0] * 6, prim_fn)
    got, _ = oracle.valencia_rhs_vertex(prim, met_v, K_v, dx, G, "weno5", 5.0 / 3.0)
    # fluid at rest, uniform p: F^k(S_k) = alpha_face p with alpha_face the EXACT face value (the 4 vertices of a face share
    # the coordinate), so dS_k = -p (alpha_{+} - alpha_{-})/dx - rho (1+eps) d_k alpha with the exact centre derivative
    (Xc, Yc, Zc), _ = _axes(n, lo, hi, G, False)
    x = (Xc, Yc, Zc)[axis]
    h = dx[axis]
    alpha = lambda t: 1.0 + a1 * t + a3 * t ** 3     # noqa: E731
    p0 = (5.0 / 3.0 - 1.0) * rho0 * eps0
    expect = -p0 * (alpha(x + h / 2) - alpha(x - h / 2)) / h - rho0 * (1 + eps0) * (a1 + 3 * a3 * x ** 2)
    assert np.abs(_int(got[0, 1 + axis]) - _int(expect)).max() < 1e-13
    other = [c for c in (1, 2, 3) if c != 1 + axis]
    assert np.abs(_int(got[0, other])).max() < 1e-14


# ------------------------------------------------------------------------------------------------ T^{mu nu}
def _tm(P, met, gamma, oracle):
    """T^{mu nu} at one vertex for uniform primitives P and vertex metric `met` (a 2^3-cell box is enough)."""
    n = (2, 2, 2)
    prim, _, _, met_v, _, _ = _both(n, (0, 0, 0), (1, 1, 1), lambda X, Y, Z: met, lambda X, Y, Z: [0.0] * 6,
                                    lambda X, Y, Z: P)
    T = oracle.tmunu_vertices(prim, met_v, G, gamma)
    return T[0, :, G + 1, G + 1, G + 1]


MINK = [1.0, 0, 0, 0, 1, 0, 0, 1, 0, 1]


def test_W1_closed_forms_on_minkowski(oracle):
    gamma = 5.0 / 3.0
    rho, eps = 1.7, 0.4
    p = (gamma - 1) * rho * eps
    T = _tm([rho, 0, 0, 0, eps, 0, 0, 0], MINK, gamma, oracle)           # fluid at rest
    assert np.allclose(T, [rho * (1 + eps), 0, 0, 0, p, 0, 0, p, 0, p], rtol=0, atol=5e-15)
    v = 0.6
    W2 = 1 / (1 - v * v)
    rhoh = rho * (1 + eps) + p
    T = _tm([rho, v, 0, 0, eps, 0, 0, 0], MINK, gamma, oracle)           # boosted along x
    assert np.allclose(T, [rhoh * W2 - p, rhoh * W2 * v, 0, 0, rhoh * W2 * v * v + p, 0, 0, p, 0, p], rtol=1e-14, atol=1e-14)
    Bx, By = 0.3, -0.4
    B2 = Bx * Bx + By * By
    T = _tm([rho, 0, 0, 0, eps, Bx, By, 0], MINK, gamma, oracle)         # magnetic field at rest: Maxwell stress
    exp = [rho * (1 + eps) + B2 / 2, 0, 0, 0, p + B2 / 2 - Bx * Bx, -Bx * By, 0, p + B2 / 2 - By * By, 0, p + B2 / 2]
    assert np.allclose(T, exp, rtol=0, atol=5e-15)


def test_W2_trace_on_general_metrics(oracle):
    rng = np.random.default_rng(11)
    gamma = 1.4
    for _ in range(20):
        A = np.eye(3) + 0.2 * rng.standard_normal((3, 3))
        g = A @ A.T
        alp = 0.6 + 0.5 * rng.random()
        beta = 0.2 * rng.standard_normal(3)
        met = [alp, *beta, g[0, 0], g[0, 1], g[0, 2], g[1, 1], g[1, 2], g[2, 2]]
        vdir = rng.standard_normal(3)
        vu = vdir * (0.7 * rng.random() / np.sqrt(vdir @ g @ vdir))
        rho, eps = 0.5 + rng.random(), 0.1 + rng.random()
        B = 0.5 * rng.standard_normal(3)
        T10 = _tm([rho, *vu, eps, *B], met, gamma, oracle)
        T = np.zeros((4, 4))
        it = iter(T10)
        for mu in range(4):
            for nu in range(mu, 4):
                T[mu, nu] = T[nu, mu] = next(it)
        g4 = np.zeros((4, 4))
        bl = g @ beta
        g4[0, 0] = -alp ** 2 + beta @ bl
        g4[0, 1:] = g4[1:, 0] = bl
        g4[1:, 1:] = g
        p = (gamma - 1) * rho * eps
        assert np.sum(g4 * T) == pytest.approx(-rho * (1 + eps) + 3 * p, rel=1e-12, abs=1e-12)
        # and the comoving energy density: u_mu u_nu T^{mu nu} = rho (1 + eps) + b^2 / 2  with b^2 = (B^2 + (alpha b^0)^2)/W^2
        vl = g @ vu
        W = 1 / np.sqrt(1 - vu @ vl)
        u_up = np.array([W / alp, *(W * (vu - beta / alp))])
        u_dn = g4 @ u_up
        Bv = B @ vl
        b2 = (B @ g @ B + (W * Bv) ** 2) / W ** 2
        assert u_dn @ T @ u_dn == pytest.approx(rho * (1 + eps) + b2 / 2, rel=1e-12)


def test_W3_interpolation_exact_for_tricubics_and_fourth_order(oracle):
    gamma = 5.0 / 3.0
    eps0 = 0.5
    poly = lambda X, Y, Z: 2.0 + 0.3 * X ** 3 - 0.2 * X * Y ** 2 + 0.1 * Y ** 3 * Z - 0.05 * Z ** 3 * X ** 2 + 0.4 * Z     # noqa: E731
    n, lo, hi = (6, 5, 4), (-1.0, -0.9, -0.8), (1.0, 0.9, 0.8)
    prim, _, _, met_v, _, dx = _both(n, lo, hi, lambda X, Y, Z: MINK, lambda X, Y, Z: [0.0] * 6,
                                     lambda X, Y, Z: [poly(X, Y, Z), 0, 0, 0, eps0, 0, 0, 0])
    T = oracle.tmunu_vertices(prim, met_v, G, gamma)
    (Xv, Yv, Zv), _ = _axes(n, lo, hi, G, True)
    sl = (slice(G, -G), slice(G, -G), slice(G, -G))          # vertices 0..n of the interior cells
    exact = poly(Xv, Yv, Zv)[sl] * (1 + eps0)                # T^{00} = rho (1 + eps) for a fluid at rest
    assert np.abs(T[0, 0][sl] - exact).max() < 2e-14 * np.abs(exact).max()
    assert np.all(np.isnan(T[0, 0, 0])) and np.all(np.isnan(T[0, 0, :, :, 1]))       # only those vertices are written
    errs = []
    for N in (8, 16, 32):
        n = (N, N, N)
        prim, _, _, met_v, _, dx = _both(n, (-1, -1, -1), (1, 1, 1), lambda X, Y, Z: MINK, lambda X, Y, Z: [0.0] * 6,
                                         lambda X, Y, Z: [1.0 + 0.3 * np.sin(2 * X + Y) * np.cos(1.5 * Z), 0, 0, 0, eps0, 0, 0, 0])
        T = oracle.tmunu_vertices(prim, met_v, G, gamma)
        (Xv, Yv, Zv), _ = _axes(n, (-1, -1, -1), (1, 1, 1), G, True)
        exact = (1.0 + 0.3 * np.sin(2 * Xv + Yv) * np.cos(1.5 * Zv))[sl] * (1 + eps0)
        errs.append(np.abs(T[0, 0][sl] - exact).max())
    assert errs[0] / errs[1] > 13 and errs[1] / errs[2] > 15, errs
