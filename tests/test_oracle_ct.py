"""Pins of the oracle's constrained transport (NEXT-2, reading R30: flux-CT of the cell-centred calB from the HLLE face
fluxes).  The paper names the ingredient ("constrained transport for the magnetic field";
l.194-196: face / edge staggering) but prints no formula, so the pins are what the mathematics fixes:

  T1  the face fluxes the CT step starts from are the right-hand side's own (their plain difference reproduces the
      independently pinned d calB/dt of oracle_valencia_rhs);
  T2  the update equals a separately written numpy statement of  d_t B = -curl <E>  with edge EMFs;
  T3  for ARBITRARY face fluxes the vertex-centred divergence of the update vanishes to rounding (the defining
      property of flux-CT; any wrong sign or index breaks it);
  T4  cyclic permutation of the axes permutes the update; and (T4b) the known behaviour on grid-aligned plane-parallel
      data: the arithmetic edge average halves the x-face dissipation (it does not reduce to the 1-D scheme);
  T5  smooth data: flux-CT and the plain flux difference agree to second order in the cell size;
  T6  evolution (oracle_evolve_ct, RK2 and RK4, periodic): the vertex-centred divergence of calB is constant in time to
      rounding, whatever it was initially, while the plain flux difference changes it.
"""
import numpy as np
import pytest

from paper_2210_17509_b200 import inputs


def _interior(a, g):
    return a[..., g:-g, g:-g, g:-g]


def test_T1_face_fluxes_are_the_right_hand_sides_own(oracle):
    prob = inputs.general_metric_box(n=(12, 9, 7), seed=31, nbox=2)
    g = prob.nghost
    for recon in ("minmod", "weno5"):
        ref, _ = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, g, recon, prob.gamma)
        FB = oracle.face_bfluxes(prob.prim, prob.metric, g, recon, prob.gamma)
        s = lambda a, d: np.roll(a, -1, axis={0: -1, 1: -2, 2: -3}[d])      # value at the high face of the cell
        for c in range(3):
            # all three directions, including the dissipative normal flux F^c(B^c) that flux-CT drops
            d = sum(-(s(FB[:, 3 * dd + c], dd) - FB[:, 3 * dd + c]) / prob.dx[dd] for dd in range(3))
            a, b = _interior(d, g), _interior(ref[:, 5 + c], g)
            assert np.abs(a - b).max() <= 1e-12 * max(np.abs(b).max(), 1e-300) + 1e-13 * np.abs(_interior(ref[:, 5:8], g)).max()


def _numpy_flux_ct(FB, dx, g):
    """d_t B = -curl <E>, written with whole-array shifts: E on edges from the four adjacent faces, then the EMF of a
    face = mean of its two edges, then the curl."""
    sh = lambda a, di, dj, dk: np.roll(np.roll(np.roll(a, -dk, -3), -dj, -2), -di, -1)   # a[i+di, j+dj, k+dk]
    FxBy, FxBz, FyBx, FyBz, FzBx, FzBy = (FB[:, c] for c in (1, 2, 3, 5, 6, 7))
    # minus / plus signs: E_z = -F^x(B^y) = +F^y(B^x), E_x = -F^y(B^z) = +F^z(B^y), E_y = -F^z(B^x) = +F^x(B^z)
    Ez = 0.25 * (FyBx + sh(FyBx, -1, 0, 0) - FxBy - sh(FxBy, 0, -1, 0))     # at (i-1/2, j-1/2, k)
    Ex = 0.25 * (FzBy + sh(FzBy, 0, -1, 0) - FyBz - sh(FyBz, 0, 0, -1))     # at (i, j-1/2, k-1/2)
    Ey = 0.25 * (FxBz + sh(FxBz, 0, 0, -1) - FzBx - sh(FzBx, -1, 0, 0))     # at (i-1/2, j, k-1/2)
    ax = lambda E: 0.5 * (E + sh(E, 1, 0, 0))      # mean over the two edges of a face that differ in x
    ay = lambda E: 0.5 * (E + sh(E, 0, 1, 0))
    az = lambda E: 0.5 * (E + sh(E, 0, 0, 1))
    ddx = lambda a: (sh(a, 1, 0, 0) - a) / dx[0]
    ddy = lambda a: (sh(a, 0, 1, 0) - a) / dx[1]
    ddz = lambda a: (sh(a, 0, 0, 1) - a) / dx[2]
    dBx = -(ddy(ax(Ez)) - ddz(ax(Ey)))
    dBy = -(ddz(ay(Ex)) - ddx(ay(Ez)))
    dBz = -(ddx(az(Ey)) - ddy(az(Ex)))
    return np.stack([dBx, dBy, dBz], axis=1)


def test_T2_flux_ct_equals_minus_curl_of_edge_emfs(oracle):
    rng = np.random.default_rng(5)
    g, n = 3, (9, 6, 5)
    FB = rng.standard_normal((2, 9, n[2] + 2 * g, n[1] + 2 * g, n[0] + 2 * g))
    dx = (0.1, 0.25, 0.4)
    got = oracle.flux_ct(FB, dx, g)
    ref = _numpy_flux_ct(FB, dx, g)
    assert np.all(np.isnan(got[:, :, 0])) and np.all(np.isnan(got[..., 0]))       # ghosts untouched
    assert np.abs(_interior(got, g) - _interior(ref, g)).max() < 1e-12


def test_T3_update_is_divergence_free_for_any_fluxes(oracle):
    """The divergence flux-CT preserves is the VERTEX-centred one: at the vertex shared by eight cells,
    div = sum_d [mean of B^d over the four cells on the high side - mean over the four on the low side] / dx_d.
    Its time derivative under the update vanishes to rounding whatever the face fluxes are."""
    rng = np.random.default_rng(6)
    g, n = 2, (10, 8, 7)
    FB = rng.standard_normal((1, 9, n[2] + 2 * g, n[1] + 2 * g, n[0] + 2 * g))
    dx = (0.3, 0.2, 0.5)
    dB = _interior(oracle.flux_ct(FB, dx, g), g)[0]          # [3][nz][ny][nx]
    lo, hi = slice(None, -1), slice(1, None)

    def vertex_diff(a, axis):
        """(mean over the 4 cells on the high side) - (mean over the 4 on the low side) along `axis` (0 = x)."""
        sl = {0: [(lo, lo), (lo, hi), (hi, lo), (hi, hi)]}
        tot = 0.0
        for s1, s2 in sl[0]:
            if axis == 0:
                tot = tot + a[s1, s2, hi] - a[s1, s2, lo]
            elif axis == 1:
                tot = tot + a[s1, hi, s2] - a[s1, lo, s2]
            else:
                tot = tot + a[hi, s1, s2] - a[lo, s1, s2]
        return 0.25 * tot

    div = sum(vertex_diff(dB[d], d) / dx[d] for d in range(3))
    scale = np.abs(dB).max() / min(dx)
    assert np.abs(div).max() < 1e-13 * scale
    # neither the update nor a single term of the divergence is trivially zero
    assert np.abs(dB).max() > 1.0 and np.abs(vertex_diff(dB[0], 0)).max() > 0.1


def test_T4_axis_permutation_covariance(oracle):
    """Cyclic relabelling of the axes (x,y,z) -> (y,z,x) of a general-metric box permutes the flux-CT update the same way:
    the three directions and the three edge orientations are treated alike."""
    from util import permute_problem
    prob = inputs.general_metric_box(n=(10, 8, 6), seed=98)
    g = prob.nghost
    out, _ = oracle.valencia_rhs_ct(prob.prim, prob.metric, prob.K, prob.dx, g, "weno5", prob.gamma)
    p2, tr, old_of_new = permute_problem(prob)
    out2, _ = oracle.valencia_rhs_ct(p2.prim, p2.metric, p2.K, p2.dx, g, "weno5", p2.gamma)
    exp = tr(out)
    exp2 = exp.copy()
    for a in range(3):
        exp2[:, 1 + a] = exp[:, 1 + old_of_new[a]]
        exp2[:, 5 + a] = exp[:, 5 + old_of_new[a]]
    a, b = _interior(out2, g), _interior(exp2, g)
    assert np.abs(a - b)[:, 5:8].max() < 1e-13 * np.abs(b[:, 5:8]).max()


def test_T4b_plane_parallel_flow_halves_the_face_dissipation(oracle):
    """What flux-CT does NOT do (and the test documents): on grid-aligned one-dimensional data the arithmetic edge average
    mixes the upwinded x-face flux with the undissipated y/z-face fluxes, so the transverse update is not the plain
    right-hand side; at t = 0 of Balsara-1 (v = 0: the physical fluxes vanish, only the HLLE dissipation is left) it is
    exactly half of it.  The normal component stays untouched."""
    prob = inputs.balsara1()
    g = prob.nghost
    plain, _ = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, g, "minmod", prob.gamma)
    ct, _ = oracle.valencia_rhs_ct(prob.prim, prob.metric, prob.K, prob.dx, g, "minmod", prob.gamma)
    a, b = _interior(ct, g), _interior(plain, g)
    assert np.array_equal(a[:, :5], b[:, :5])
    assert np.abs(b[:, 6]).max() > 1.0
    assert np.abs(a[:, 6] - 0.5 * b[:, 6]).max() <= 1e-13 * np.abs(b[:, 6]).max()
    assert np.abs(a[:, 5]).max() == 0.0 and np.abs(a[:, 7]).max() == 0.0


def test_T5_smooth_data_second_order_agreement(oracle):
    """The same smooth fields (config-5 recipe, one seed) at three resolutions: flux-CT differs from the plain flux
    difference by the O(h^2) error of its edge averages."""
    errs = []
    g = inputs.NGHOST
    for N in (32, 64, 128):
        prim, met, K, dx, gamma = inputs._smooth_box(N, 77, g)
        prim, met, K = prim[None], met[None], K[None]
        plain, _ = oracle.valencia_rhs(prim, met, K, dx, g, "weno5", gamma)
        ct, _ = oracle.valencia_rhs_ct(prim, met, K, dx, g, "weno5", gamma)
        errs.append(np.abs(_interior(ct, g)[:, 5:8] - _interior(plain, g)[:, 5:8]).max())
    assert errs[0] / errs[1] > 3.3 and errs[1] / errs[2] > 3.7 and errs[2] < 0.02 * 2.3, errs


def _vertex_divergence(B, dx):
    """Vertex-centred divergence of a cell-centred field B[3][nz][ny][nx] (periodic wrap): at every vertex, sum over d of
    [mean of B^d over the 4 cells on the high side - mean over the 4 on the low side] / dx_d."""
    div = 0.0
    for d in range(3):
        ax = {0: -1, 1: -2, 2: -3}[d]
        diff = B[d] - np.roll(B[d], 1, axis=ax)                # high cell - low cell across the vertex plane
        t1, t2 = [a for a in (-1, -2, -3) if a != ax]
        mean = 0.25 * (diff + np.roll(diff, 1, axis=t1) + np.roll(diff, 1, axis=t2) + np.roll(np.roll(diff, 1, axis=t1), 1, axis=t2))
        div = div + mean / dx[d]
    return div


@pytest.mark.parametrize("rk", [2, 4])
def test_T6_evolution_with_flux_ct_keeps_the_vertex_divergence(oracle, rk):
    """Method of lines with flux-CT (oracle_evolve_ct) on a periodic Minkowski block whose initial field is NOT divergence-
    free: every Runge-Kutta stage adds a discrete curl, so the vertex-centred divergence of calB stays what it was, to
    rounding; the plain flux difference changes it by orders of magnitude more.  D, S_i, tau and the sums of calB stay
    conserved."""
    from util import make_problem

    def prim(X, Y, Z):
        s = np.sin(2 * np.pi * X) * np.cos(2 * np.pi * Y) + 0.5 * np.sin(2 * np.pi * (Z + X))
        rho = 1.0 + 0.3 * s
        p = 1.0 + 0.2 * np.cos(2 * np.pi * (X - Y))
        return [rho, 0.2 + 0.1 * s, -0.1 + 0.05 * np.cos(2 * np.pi * Z), 0.15 * np.sin(2 * np.pi * Y), p / ((5.0 / 3.0 - 1) * rho),
                0.3 + 0.1 * np.sin(2 * np.pi * X), 0.2 * np.sin(2 * np.pi * (X + Y)), 0.1 * np.cos(2 * np.pi * (X - Z))]
    prob = make_problem((12, 12, 12), (0, 0, 0), (1, 1, 1), 5.0 / 3.0, prim, g=3, name="wave-divB")
    g = prob.nghost
    ii = prob.interior
    U0 = oracle.prim2con(prob.prim, prob.metric, g, prob.gamma)
    dt = 0.3 * prob.dx[0]
    out = {}
    for ct in (True, False):
        _, U, nfail = oracle.evolve(prob.prim, prob.metric, prob.K, prob.dx, g, "weno5", prob.gamma, dt, 3, rk=rk,
                                    bc="periodic", ct=ct)
        assert nfail == 0
        out[ct] = U
    d0 = _vertex_divergence(U0[ii][0, 5:8], prob.dx)
    d_ct = _vertex_divergence(out[True][ii][0, 5:8], prob.dx)
    d_plain = _vertex_divergence(out[False][ii][0, 5:8], prob.dx)
    scale = np.abs(U0[ii][0, 5:8]).max() / min(prob.dx)
    assert np.abs(d0).max() > 1e-2 * scale                      # the test field does have a divergence
    assert np.abs(d_ct - d0).max() < 1e-13 * scale
    assert np.abs(d_plain - d0).max() > 1e-6 * scale
    for c in range(8):
        s0, s1 = U0[ii][:, c].sum(), out[True][ii][:, c].sum()
        assert abs(s1 - s0) <= 1e-12 * np.abs(U0[ii][:, c]).sum(), c
    # the hydrodynamic part is driven by a different field history, but the two runs stay close over three steps
    assert np.abs(out[True][ii] - out[False][ii]).max() < 0.05
