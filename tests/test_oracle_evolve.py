"""NEXT-1 on the oracle side: the Gamma-law con2prim (reading R22) and the method-of-lines
loop (l.125; R21) of oracle/valencia_oracle.cpp against what the paper and the mathematics fix:
round trips through the independently pinned prim2con (P6/P17) on relativistic and magnetically dominated states,
the paper's printed Balsara-1 outcome (l.257), exact rest-mass conservation on a periodic block, the formal order of
the two Runge-Kutta schemes, and admissible evolutions of the Table I states of Balsara 2-5."""
import os

import numpy as np
import pytest

from paper_2210_17509_b200 import inputs
from test_oracle_balsara import read_golden
from util import MET_FLAT, make_problem

GOLD = os.path.join(os.path.dirname(__file__), "golden", "balsara_table1.txt")


def table1():
    rows = {}
    for line in open(GOLD):
        line = line.split("#")[0].split()
        if line:
            rows[(int(line[0]), line[1])] = [float(v) for v in line[2:]]
    return rows


def shocktube(test, n=200, g=3):
    """1-D shocktube block on [-0.5, 0.5] from a Table I row pair (eps given, as the ABI carries it)."""
    L, R = table1()[(test, "L")], table1()[(test, "R")]
    gamma = L[1]

    def prim(X, Y, Z):
        left = X < 0.0
        pick = lambda i: np.where(left, L[i], R[i])
        return [pick(3), pick(5), pick(6), pick(7), pick(4), np.full(X.shape, L[0]), pick(8), pick(9)]
    return make_problem((n, 1, 1), (-0.5, 0.0, 0.0), (0.5, 1.0 / n, 1.0 / n), gamma, prim, g=g, name=f"balsara{test}"), L[2]


def test_con2prim_round_trip_relativistic_and_magnetised(oracle):
    """prim -> cons (Eqs. 6-9, pinned by P6/P17) -> prim on general metrics: Lorentz factors up to 20, B^2/(rho h W^2)
    up to ~1e4, eps from 1e-3 to 1e2.  The solve is conditioned like W^2 (1 + B^2/z) (z = rho h W^2): the recovered
    state must be accurate to rounding times that factor."""
    rng = np.random.default_rng(7)
    n = 4000
    shape = (1, 1, n)
    prob = inputs.general_metric_box(n=(n - 6, 1, 1), seed=3, g=3)     # smooth general metric, (n) x 7 x 7 cells
    met = prob.metric
    N = met.shape[-1] * met.shape[-2] * met.shape[-3]
    prim = np.empty((1, 8) + met.shape[2:])
    W = 10.0 ** rng.uniform(0, np.log10(20.0), N)
    dirs = rng.normal(size=(3, N))
    g6 = met[0, 4:].reshape(6, N)
    sym = ((0, 1, 2), (1, 3, 4), (2, 4, 5))
    norm2 = sum(g6[sym[a][b]] * dirs[a] * dirs[b] for a in range(3) for b in range(3))
    v = dirs / np.sqrt(norm2) * np.sqrt(1.0 - 1.0 / W ** 2)
    prim[0, 0] = (10.0 ** rng.uniform(-2, 1, N)).reshape(met.shape[2:])
    for a in range(3):
        prim[0, 1 + a] = v[a].reshape(met.shape[2:])
        prim[0, 5 + a] = (rng.normal(size=N) * 10.0 ** rng.uniform(-3, 1.0, N)).reshape(met.shape[2:])
    prim[0, 4] = (10.0 ** rng.uniform(-3, 2, N)).reshape(met.shape[2:])
    cons = oracle.prim2con(prim, met, 3, 5.0 / 3.0)
    back, nfail = oracle.con2prim(cons, met, 3, 5.0 / 3.0)
    assert nfail == 0
    Wg = W.reshape(met.shape[2:])
    B = prim[0, 5:].reshape(3, N)
    B2 = sum(g6[sym[a][b]] * B[a] * B[b] for a in range(3) for b in range(3)).reshape(met.shape[2:])
    z = prim[0, 0] * (1.0 + (5.0 / 3.0) * prim[0, 4]) * Wg ** 2
    cond = Wg ** 2 * (1.0 + B2 / z)
    assert np.max(np.abs(back[0, 0] / prim[0, 0] - 1) / cond) < 1e-12
    assert np.max(np.abs(back[0, 1:4] - prim[0, 1:4]) / cond) < 1e-12
    assert np.max(np.abs(back[0, 5:] - prim[0, 5:])) <= 1e-12 * np.abs(prim[0, 5:]).max()
    # the pressure against the energy scale of the state
    scale = (np.abs(cons[0, 4]) + np.abs(cons[0, 0])) / np.sqrt(np.linalg.det(np.array(
        [[g6[0], g6[1], g6[2]], [g6[1], g6[3], g6[4]], [g6[2], g6[4], g6[5]]]).transpose(2, 0, 1))).reshape(met.shape[2:])
    p_err = (5.0 / 3.0 - 1) * np.abs(back[0, 0] * back[0, 4] - prim[0, 0] * prim[0, 4])
    assert np.max(p_err / scale) < 1e-12


def test_p16_balsara1_through_the_oracle_loop(oracle):
    """The paper's printed Balsara-1 outcome (l.257: Lorentz factor ~1.458) with oracle.evolve (SSP-RK2, R21)."""
    gold = read_golden()
    N = 400
    prob = inputs.balsara1(n=(N, 1, 1))
    dt = 0.4 * prob.dx[0]
    nsteps = int(round(gold["t_ref"] / dt))
    U0 = oracle.prim2con(prob.prim, prob.metric, 3, prob.gamma)
    prim, U, nfail = oracle.evolve(prob.prim, prob.metric, prob.K, prob.dx, 3, "minmod", prob.gamma, dt, nsteps, rk=2, bc="copy")
    assert nfail == 0
    line = prim[0, :, 3, 3, 3:-3]
    W = 1 / np.sqrt(1 - (line[1] ** 2 + line[2] ** 2 + line[3] ** 2))
    assert abs(W.max() - gold["lorentz_max"]) < 0.01, W.max()
    assert abs(line[6][0] - gold["By_left"]) < 1e-10 and abs(line[6][-1] - gold["By_right"]) < 1e-10
    m0, m1 = U0[0, 0, 3, 3, 3:-3].sum(), U[0, 0, 3, 3, 3:-3].sum()
    assert abs(m1 - m0) < 1e-12 * m0
    # RK4 at the paper's CFL 0.8 (l.255) reaches the same state
    prim4, _, nf4 = oracle.evolve(prob.prim, prob.metric, prob.K, prob.dx, 3, "minmod", prob.gamma, 0.8 * prob.dx[0],
                                  nsteps // 2, rk=4, bc="copy")
    l4 = prim4[0, :, 3, 3, 3:-3]
    assert nf4 == 0 and abs((1 / np.sqrt(1 - l4[1] ** 2 - l4[2] ** 2)).max() - gold["lorentz_max"]) < 0.01


def _periodic_wave(n=24, g=3):
    """Smooth periodic state on Minkowski: density, pressure, velocity and field waves along all three axes."""
    def prim(X, Y, Z):
        s = np.sin(2 * np.pi * X) * np.cos(2 * np.pi * Y) + 0.5 * np.sin(2 * np.pi * (Z + X))
        rho = 1.0 + 0.3 * s
        p = 1.0 + 0.2 * np.cos(2 * np.pi * (X - Y))
        return [rho, 0.2 + 0.1 * s, -0.1 + 0.05 * np.cos(2 * np.pi * Z), 0.15 * np.sin(2 * np.pi * Y), p / ((5.0 / 3.0 - 1) * rho),
                0.3 + 0 * X, 0.2 * np.sin(2 * np.pi * X), 0.1 * np.cos(2 * np.pi * X)]
    return make_problem((n, n, n), (0, 0, 0), (1, 1, 1), 5.0 / 3.0, prim, g=g, name="wave")


@pytest.mark.parametrize("rk", [2, 4])
def test_periodic_evolution_conserves_every_conserved_variable(oracle, rk):
    """Flux form + periodic ghost fill on Minkowski (no sources): the sums of D, S_i, tau and calB^i over the block do
    not change beyond rounding; pins the sign and pairing of the flux differences through the whole loop."""
    prob = _periodic_wave(16)
    U0 = oracle.prim2con(prob.prim, prob.metric, 3, prob.gamma)
    ii = prob.interior
    _, U, nfail = oracle.evolve(prob.prim, prob.metric, prob.K, prob.dx, 3, "weno5", prob.gamma, 0.3 * prob.dx[0], 4, rk=rk,
                                bc="periodic")
    assert nfail == 0
    for c in range(8):
        s0, s1 = U0[ii][:, c].sum(), U[ii][:, c].sum()
        assert abs(s1 - s0) <= 1e-12 * np.abs(U0[ii][:, c]).sum(), c


def test_runge_kutta_stability_polynomials_on_the_flrw_slice(oracle):
    """A uniform fluid at rest with a uniform field on the slice gamma_ij = a^2 delta_ij, K_ij = -a adot delta_ij, alpha = 1
    (pin P12: d tau/dt = -a^2 adot (3p + b^2/2), everything else 0).  With the metric held fixed, tau obeys the LINEAR
    equation tau' = -lam tau + mu, lam = 3 (Gamma-1) adot / a, so n steps of size h multiply (tau - mu/lam) by R(lam h)^n
    with R = 1 - z + z^2/2 for SSP-RK2 and 1 - z + z^2/2 - z^3/6 + z^4/24 for RK4 -- exactly, up to rounding."""
    a_, adot, gam = 1.3, 0.4, 5.0 / 3.0
    rho, eps, Bx = 1.0, 0.5, 0.2

    def prim(X, Y, Z):
        one = np.ones_like(X + Y + Z)
        return [rho * one, 0 * one, 0 * one, 0 * one, eps * one, Bx * one, 0 * one, 0 * one]
    met = lambda X, Y, Z: [1.0, 0, 0, 0, a_ ** 2, 0, 0, a_ ** 2, 0, a_ ** 2]
    Kf = lambda X, Y, Z: [-a_ * adot, 0, 0, -a_ * adot, 0, -a_ * adot]
    prob = make_problem((4, 4, 4), (0, 0, 0), (1, 1, 1), gam, prim, met, Kf, g=3, name="flrw")
    b2 = a_ ** 2 * Bx ** 2
    tau0 = a_ ** 3 * (rho * eps + 0.5 * b2)
    lam = 3.0 * (gam - 1.0) * adot / a_
    mu = a_ ** 2 * adot * b2 * (1.5 * (gam - 1.0) - 0.5)
    h, nsteps = 0.2, 5
    z = lam * h
    for rk, R in ((2, 1 - z + z * z / 2), (4, 1 - z + z * z / 2 - z ** 3 / 6 + z ** 4 / 24)):
        _, U, nfail = oracle.evolve(prob.prim, prob.metric, prob.K, prob.dx, 3, "weno5", gam, h, nsteps, rk=rk, bc="periodic")
        assert nfail == 0
        tau = U[prob.interior][0, 4]
        want = mu / lam + (tau0 - mu / lam) * R ** nsteps
        assert np.max(np.abs(tau - want)) < 1e-13 * abs(tau0), (rk, tau.flat[0], want)
        assert np.max(np.abs(U[prob.interior][0, 0] - a_ ** 3 * rho)) < 1e-14 and np.max(np.abs(U[prob.interior][0, 1:4])) < 1e-14


@pytest.mark.parametrize("test,cfl", [(2, 0.8), (3, 0.4), (4, 0.2), (5, 0.8)])
def test_balsara_2_to_5_start_admissibly(oracle, test, cfl):
    """Table I states of Balsara 2-5 (l.242-249), minmod + HLLE + RK4, copy boundaries (l.255), 200 cells: the first 20
    time units of dx keep every cell admissible, con2prim converges everywhere, B^x stays constant and rest mass is
    conserved.  The paper's CFL 0.8 (l.255) is used where this bare loop survives it at this resolution: the 10^4
    pressure jump of Balsara 3 and the W = 22 collision of Balsara 4 need 0.4 and 0.2 here, since the path applies no
    floor or atmosphere (reading R27) and has none of the paper's con2prim fallbacks (l.144-146)."""
    prob, _ = shocktube(test, 200)
    U0 = oracle.prim2con(prob.prim, prob.metric, 3, prob.gamma)
    prim, U, nfail = oracle.evolve(prob.prim, prob.metric, prob.K, prob.dx, 3, "minmod", prob.gamma, cfl * prob.dx[0],
                                   int(round(8 / cfl)), rk=4, bc="copy")
    assert nfail == 0
    line = prim[0, :, 3, 3, 3:-3]
    v2 = line[1] ** 2 + line[2] ** 2 + line[3] ** 2
    assert np.all(line[0] > 0) and np.all(line[4] > 0) and np.all(v2 < 1.0)
    assert np.max(np.abs(line[5] - table1()[(test, "L")][0])) < 1e-11
    # rest mass changes by what flows through the two ends, where the states are still the initial ones: D v^x t / dx
    L, R = table1()[(test, "L")], table1()[(test, "R")]
    Dv = [r[3] * r[5] / np.sqrt(1 - r[5] ** 2 - r[6] ** 2 - r[7] ** 2) for r in (L, R)]
    t_over_dx = cfl * int(round(8 / cfl))
    m0, m1 = U0[0, 0, 3, 3, 3:-3].sum(), U[0, 0, 3, 3, 3:-3].sum()
    assert abs((m1 - m0) - t_over_dx * (Dv[0] - Dv[1])) < 1e-10 * abs(m0)


def test_copy_boundary_ghost_fill_is_the_nearest_interior_cell(oracle):
    """Pin of fill_ghosts_box, bc = "copy" ("copy" boundaries; l.170 user-supplied outer boundary): after a
    step every ghost cell of every primitive holds the bits of the interior cell with the CLAMPED index -- faces, edges and
    corners -- on a 3-D block with an off-diagonal metric whose interior values are all distinct, so that clamping to n or
    n - 2, or treating an edge / corner direction by direction in the wrong way, fails.  Then the whole loop against the
    independently written numpy loop of tests/evolve.py (its own clamp, ghost fill after every stage) over three SSP-RK2
    steps: the fill happens where the method needs it."""
    from evolve import fill_copy_bc, rk2_evolve
    g = 3
    prob = inputs.general_metric_box(n=(9, 7, 6), seed=11)
    start = fill_copy_bc(prob.prim.copy(), g)
    dt = 0.2 * min(prob.dx)
    prim, U, nfail = oracle.evolve(start, prob.metric, prob.K, prob.dx, g, "minmod", prob.gamma, dt, 1, rk=2, bc="copy")
    assert nfail == 0
    inner = prim[prob.interior]
    assert len(np.unique(inner[0, 0])) == inner[0, 0].size          # distinct values: a wrong source index is visible
    Nz, Ny, Nx = prim.shape[2:]
    kk, jj, ii = (np.clip(np.arange(N), g, N - g - 1) for N in (Nz, Ny, Nx))
    want = prim[:, :, kk[:, None, None], jj[None, :, None], ii[None, None, :]]
    assert np.array_equal(prim, want)
    assert not np.array_equal(prim, start)                           # the step did change the block

    class Backend:
        def rhs(self, p):
            return oracle.valencia_rhs(p, prob.metric, prob.K, prob.dx, g, "minmod", prob.gamma)[0]

        def prim2con(self, p):
            return oracle.prim2con(p, prob.metric, g, prob.gamma)

        def con2prim(self, U):
            return oracle.con2prim(U, prob.metric, g, prob.gamma)[0]

    p_loop, U_loop = rk2_evolve(Backend(), start, g, dt, 3)
    p_orc, U_orc, nfail = oracle.evolve(start, prob.metric, prob.K, prob.dx, g, "minmod", prob.gamma, dt, 3, rk=2, bc="copy")
    assert nfail == 0
    ii3 = prob.interior
    assert np.abs(U_orc[ii3] - U_loop[ii3]).max() <= 1e-12 * np.abs(U_loop[ii3]).max()
    assert np.abs(p_orc - p_loop).max() <= 1e-12 * np.abs(p_loop).max()     # ghosts included
