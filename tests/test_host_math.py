"""The CUDA path's point-wise arithmetic (csrc/grx_math.cuh), compiled for the host by
tests/host_math_harness.cpp and driven by a naive per-cell loop, against the oracle: checks the rearranged
formulas (common-denominator WENO5 weights, a^2 = (b^2 + Gamma p)/(rho h*), Eulerian-observer sources) on a CPU
box.  On the host the MUFU-seeded reciprocals are IEEE ones, so this pins the algebra, not the seeds; the
-m gpu tests pin the device code itself."""
import ctypes as C
import os
import subprocess

import numpy as np
import pytest

from paper_2210_17509_b200 import inputs
from util import relerr_per_component

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
DP = C.POINTER(C.c_double)


@pytest.fixture(scope="module")
def hm():
    src = os.path.join(HERE, "host_math_harness.cpp")
    out = os.path.join(ROOT, "build", "libhostmath.so")
    os.makedirs(os.path.dirname(out), exist_ok=True)
    hdr = os.path.join(ROOT, "paper_2210_17509_b200", "csrc", "grx_math.cuh")
    if not os.path.exists(out) or os.path.getmtime(out) < max(os.path.getmtime(src), os.path.getmtime(hdr)):
        subprocess.run(["g++", "-O2", "-march=native", "-std=c++17", "-shared", "-fPIC", "-Wno-unknown-pragmas", src,
                        "-o", out], check=True)
    return C.CDLL(out)


def _p(a):
    return a.ctypes.data_as(DP)


def host_rhs(hm, prob, recon, oracle):
    n = (C.c_int * 3)(*prob.n)
    out = np.full(prob.prim.shape, np.nan)
    nfb = C.c_ulonglong(0)
    dx = (C.c_double * 3)(*prob.dx)
    hm.hm_valencia_rhs(n, prob.nbox, _p(prob.prim), _p(prob.metric), _p(prob.K), dx, prob.nghost, oracle.RECON[recon],
                       C.c_double(prob.gamma), _p(out), C.byref(nfb))
    return out, nfb.value


@pytest.mark.parametrize("name", ["c1", "gen", "c2:small", "c3:small", "c4:small", "c5-32:small"])
def test_device_arithmetic_matches_oracle(hm, oracle, name):
    prob = inputs.by_name(name)
    for recon in prob.recons:
        ref, nfb_ref = oracle.valencia_rhs(prob.prim, prob.metric, prob.K, prob.dx, prob.nghost, recon, prob.gamma)
        got, nfb = host_rhs(hm, prob, recon, oracle)
        ii = prob.interior
        assert relerr_per_component(got[ii], ref[ii]).max() < 1e-12, (name, recon)
        assert nfb == nfb_ref


def test_weno5_rearrangement_pointwise(hm, oracle):
    rng = np.random.default_rng(3)
    for scale in (1.0, 1e-10, 1e6):
        for _ in range(300):
            q = scale * rng.normal(size=5)
            if rng.random() < 0.3:
                q[rng.integers(0, 5):] += scale * 10.0      # a jump inside the stencil
            qm, qp = C.c_double(), C.c_double()
            hm.hm_recon_cell(2, _p(q), C.byref(qm), C.byref(qp))
            rm, rp = oracle.recon_cell("weno5", q)
            tol = 4e-15 * np.abs(q).max()
            assert abs(qm.value - rm) <= tol and abs(qp.value - rp) <= tol
    for rec, code in (("minmod", 0), ("mc", 1)):
        for _ in range(300):
            q = rng.normal(size=5)
            qm, qp = C.c_double(), C.c_double()
            hm.hm_recon_cell(code, _p(q), C.byref(qm), C.byref(qp))
            assert (qm.value, qp.value) == pytest.approx(oracle.recon_cell(rec, q), abs=1e-15)


def test_prim2con_con2prim_pointwise(hm, oracle):
    rng = np.random.default_rng(4)
    hm.hm_con2prim.restype = C.c_int
    for _ in range(100):
        P = np.array([rng.uniform(0.1, 2), *rng.uniform(-0.4, 0.4, 3), rng.uniform(0.1, 3), *rng.uniform(-1, 1, 3)])
        met = np.array([0.9, 0.01, -0.02, 0.03, 1.3, 0.1, -0.05, 1.1, 0.02, 0.9])
        U = np.empty(8)
        hm.hm_prim2con(_p(P), _p(met), C.c_double(1.6), _p(U))
        Uo, _, _ = oracle.state_flux(P, met, 0, 1.6)
        assert np.abs(U - Uo).max() < 1e-14 * np.abs(Uo).max()
        back = np.empty(8)
        assert hm.hm_con2prim(_p(U), _p(met), C.c_double(1.6), _p(back)) == 0
        assert np.abs(back - P).max() < 1e-11


def test_con2prim_warm_start_agrees_with_the_bracketed_solve(hm):
    """The RK stage kernel starts the solve from the previous stage's primitives (con2prim_point_warm): from a state a few
    per cent away it converges to the bracketed solve's answer; a useless guess (negative, NaN, far off) falls back to it."""
    rng = np.random.default_rng(8)
    hm.hm_con2prim.restype = C.c_int
    hm.hm_con2prim_warm.restype = C.c_int
    hm.hm_con2prim_warm_steps.restype = C.c_int
    met = np.array([0.9, 0.01, -0.02, 0.03, 1.3, 0.1, -0.05, 1.1, 0.02, 0.9])
    ok_warm = 0
    for _ in range(200):
        P = np.array([rng.uniform(0.1, 2), *rng.uniform(-0.4, 0.4, 3), rng.uniform(0.1, 3), *rng.uniform(-1, 1, 3)])
        U, a, b = np.empty(8), np.empty(8), np.empty(8)
        hm.hm_prim2con(_p(P), _p(met), C.c_double(1.6), _p(U))
        assert hm.hm_con2prim(_p(U), _p(met), C.c_double(1.6), _p(a)) == 0
        Pold = P * (1 + 0.05 * rng.uniform(-1, 1, 8))
        assert hm.hm_con2prim_warm(_p(U), _p(met), C.c_double(1.6), _p(Pold), _p(b)) == 0
        assert np.abs(a - b).max() < 1e-12
        rhoh = Pold[0] * (1 + 1.6 * Pold[4])
        ok_warm += hm.hm_con2prim_warm_steps(_p(U), _p(met), C.c_double(1.6), C.c_double(rhoh)) == 0
        for bad in (np.full(8, np.nan), -P, P * 1e6):
            assert hm.hm_con2prim_warm(_p(U), _p(met), C.c_double(1.6), _p(bad), _p(b)) == 0
            assert np.abs(a - b).max() < 1e-12
    assert ok_warm >= 195          # the warm path itself converges (it is not the fallback doing the work)
