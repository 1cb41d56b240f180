"""P16: short CPU evolution of the Balsara-1 shocktube with the oracle reproduces what the paper
prints (tests/golden/balsara1_paper.txt; Table I and l.255-257)."""
import os

import numpy as np

from evolve import rk2_evolve
from paper_2210_17509_b200 import inputs

GOLD = os.path.join(os.path.dirname(__file__), "golden", "balsara1_paper.txt")


def read_golden():
    vals = {}
    for line in open(GOLD):
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split("=")
            vals[k.strip()] = float(v)
    return vals


class OracleBackend:
    def __init__(self, orc, prob, recon):
        self.o, self.p, self.recon = orc, prob, recon

    def rhs(self, prim):
        return self.o.valencia_rhs(prim, self.p.metric, self.p.K, self.p.dx, self.p.nghost, self.recon, self.p.gamma)[0]

    def prim2con(self, prim):
        return self.o.prim2con(prim, self.p.metric, self.p.nghost, self.p.gamma)

    def con2prim(self, U):
        prim, nfail = self.o.con2prim(U, self.p.metric, self.p.nghost, self.p.gamma)
        assert nfail == 0
        return prim


def test_golden_matches_config1():
    gold = read_golden()
    prob = inputs.balsara1()
    P = prob.prim[0][:, 3, 3, :]
    assert prob.gamma == gold["gamma"]
    assert P[0, 3] == gold["rho_left"] and P[0, -4] == gold["rho_right"]
    assert P[4, 3] == gold["eps_left"] and abs(P[4, -4] - gold["eps_right"]) < 1e-15
    assert P[5, 3] == gold["Bx"] and P[6, 3] == gold["By_left"] and P[6, -4] == gold["By_right"]


def test_p16_balsara1_evolution(oracle):
    gold = read_golden()
    N = 400
    prob = inputs.balsara1(n=(N, 1, 1))
    dt = 0.4 * prob.dx[0]                       # R21
    nsteps = int(round(gold["t_ref"] / dt))
    be = OracleBackend(oracle, prob, "minmod")  # l.255: TVD minmod + HLLE
    U0 = be.prim2con(prob.prim)
    prim, U = rk2_evolve(be, prob.prim, prob.nghost, dt, nsteps)
    g = prob.nghost
    line = prim[0, :, g, g, g:-g]
    rho, vx, vy, eps, By = line[0], line[1], line[2], line[4], line[6]
    W = 1 / np.sqrt(1 - (line[1] ** 2 + line[2] ** 2 + line[3] ** 2))
    # the paper's printed maximum Lorentz factor (~1.458 at 1600 points; 1.46 at 400 points)
    assert abs(W.max() - gold["lorentz_max"]) < 0.01, W.max()
    # outer states untouched at t = 0.4, B^y goes from +1 to -1, density stays between the outer states
    assert abs(rho[0] - gold["rho_left"]) < 1e-10 and abs(rho[-1] - gold["rho_right"]) < 1e-10
    assert abs(By[0] - gold["By_left"]) < 1e-10 and abs(By[-1] - gold["By_right"]) < 1e-10
    # (the right-going fast rarefaction lowers rho slightly below the right state)
    assert rho.min() >= 0.9 * gold["rho_right"] and rho.max() <= gold["rho_left"] + 1e-3
    assert np.all(np.abs(line[5] - gold["Bx"]) < 1e-12)          # normal field stays constant in 1-D
    assert np.all(line[3] == 0) and np.all(line[7] == 0)         # no z-dynamics
    # rest mass is conserved to rounding while the waves are inside the domain
    m0 = U0[0, 0, g, g, g:-g].sum()
    m1 = U[0, 0, g, g, g:-g].sum()
    assert abs(m1 - m0) < 1e-12 * m0
    # five-wave structure of l.257: count the maximal runs where |d rho/dx| is significant
    drho = np.abs(np.diff(rho)) > 2e-4
    runs = np.flatnonzero(np.diff(np.concatenate(([0], drho.astype(int), [0]))) == 1)
    # merge runs closer than 6 cells
    merged = [runs[0]]
    ends = np.flatnonzero(np.diff(np.concatenate(([0], drho.astype(int), [0]))) == -1)
    last_end = ends[0]
    for s, e in zip(runs[1:], ends[1:]):
        if s - last_end > 6:
            merged.append(s)
        last_end = e
    # fast rarefaction | compound wave | contact | slow shock | (right fast rarefaction: tiny in rho)
    assert 4 <= len(merged) <= 5, (merged, len(merged))
    # flow is to the right between the left rarefaction and the right-going waves; v^y < 0 develops
    assert vx.max() > 0.3 and vy.min() < -0.5
