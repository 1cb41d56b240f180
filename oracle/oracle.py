"""ctypes binding of the CPU oracle (oracle/valencia_oracle.cpp).

TEST INFRASTRUCTURE: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this module.  It never imports the CUDA package.

Array convention (same as include/grx.h): numpy float64, C-contiguous, shape
[nbox, nfield, Nz, Ny, Nx] with N = n + 2*nghost (x fastest).
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

RECON = {"minmod": 0, "mc": 1, "weno5": 2}
_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        dp = C.POINTER(C.c_double)
        ip = C.POINTER(C.c_int)
        up = C.POINTER(C.c_ulonglong)
        for name in ("oracle_valencia_rhs", "oracle_valencia_rhs_ld"):
            f = getattr(L, name)
            f.argtypes = [ip, C.c_int, dp, dp, dp, dp, C.c_int, C.c_int, C.c_double, dp, up]
            f.restype = C.c_int
        L.oracle_valencia_rhs_count.argtypes = [ip, C.c_int, dp, dp, dp, dp, C.c_int, C.c_int, C.c_double, dp, up]
        L.oracle_valencia_rhs_count.restype = C.c_int
        L.oracle_prim2con.argtypes = [ip, C.c_int, dp, dp, C.c_int, C.c_double, dp]
        L.oracle_prim2con.restype = C.c_int
        L.oracle_con2prim.argtypes = [ip, C.c_int, dp, dp, C.c_int, C.c_double, dp]
        L.oracle_con2prim.restype = C.c_int
        L.oracle_evolve.argtypes = [ip, C.c_int, dp, dp, dp, dp, C.c_int, C.c_int, C.c_double, C.c_double, C.c_int, C.c_int,
                                    C.c_int, dp]
        L.oracle_evolve.restype = C.c_int
        L.oracle_evolve_ct.argtypes = L.oracle_evolve.argtypes
        L.oracle_evolve_ct.restype = C.c_int
        L.oracle_recon_cell.argtypes = [C.c_int, dp, dp, dp]
        L.oracle_recon_cell.restype = None
        L.oracle_state_flux.argtypes = [dp, dp, C.c_int, C.c_double, dp, dp, dp]
        L.oracle_state_flux.restype = None
        L.oracle_face_flux.argtypes = [dp, dp, dp, dp, dp, C.c_int, C.c_double, dp]
        L.oracle_face_flux.restype = None
        L.oracle_hlle.argtypes = [dp, dp, dp, dp, dp, dp, dp]
        L.oracle_hlle.restype = None
        L.oracle_sources_point.argtypes = [dp, dp, dp, dp, C.c_double, dp]
        L.oracle_sources_point.restype = None
        L.oracle_count_piece.argtypes = [C.c_int, C.c_int, C.c_int, up]
        L.oracle_count_piece.restype = C.c_int
        L.oracle_face_bfluxes.argtypes = [ip, C.c_int, dp, dp, C.c_int, C.c_int, C.c_double, dp]
        L.oracle_face_bfluxes.restype = C.c_int
        L.oracle_flux_ct.argtypes = [ip, C.c_int, dp, dp, C.c_int, dp]
        L.oracle_flux_ct.restype = C.c_int
        L.oracle_valencia_rhs_vertex.argtypes = [ip, C.c_int, dp, dp, dp, dp, C.c_int, C.c_int, C.c_double, dp, up]
        L.oracle_valencia_rhs_vertex.restype = C.c_int
        L.oracle_tmunu_vertices.argtypes = [ip, C.c_int, dp, dp, C.c_int, C.c_double, dp]
        L.oracle_tmunu_vertices.restype = C.c_int
        L.oracle_weno_eps.restype = C.c_double
        L.oracle_v2max.restype = C.c_double
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _arr(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


def _grid(prim, nghost):
    nbox, nf, Nz, Ny, Nx = prim.shape
    n = (C.c_int * 3)(Nx - 2 * nghost, Ny - 2 * nghost, Nz - 2 * nghost)
    return n, nbox


def valencia_rhs(prim, metric, K, dx, nghost, recon, gamma, variant="double", out=None):
    """d/dt of (D, S_x, S_y, S_z, tau, calB^x, calB^y, calB^z) on the interior cells.

    variant: "double" (the oracle), "long double" (adjudicator) or "count" (returns (out, ops)).
    Returns (out, nfallback) -- out has the shape of prim; its ghost cells are NaN.
    """
    prim, metric, K = _arr(prim), _arr(metric), _arr(K)
    assert prim.ndim == 5 and prim.shape[1] == 8 and metric.shape[1] == 10 and K.shape[1] == 6
    n, nbox = _grid(prim, nghost)
    if out is None:
        out = np.full(prim.shape, np.nan)
    dxa = (C.c_double * 3)(*dx)
    r = RECON[recon] if isinstance(recon, str) else int(recon)
    if variant == "count":
        ops = (C.c_ulonglong * 4)()
        rc = lib().oracle_valencia_rhs_count(n, nbox, _p(prim), _p(metric), _p(K), dxa, nghost, r, gamma, _p(out), ops)
        if rc:
            raise ValueError("oracle: invalid argument")
        return out, dict(add=ops[0], mul=ops[1], div=ops[2], sqrt=ops[3])
    nfb = C.c_ulonglong(0)
    fn = lib().oracle_valencia_rhs if variant == "double" else lib().oracle_valencia_rhs_ld
    rc = fn(n, nbox, _p(prim), _p(metric), _p(K), dxa, nghost, r, gamma, _p(out), C.byref(nfb))
    if rc:
        raise ValueError("oracle: invalid argument")
    return out, int(nfb.value)


def prim2con(prim, metric, nghost, gamma):
    prim, metric = _arr(prim), _arr(metric)
    n, nbox = _grid(prim, nghost)
    cons = np.empty_like(prim)
    if lib().oracle_prim2con(n, nbox, _p(prim), _p(metric), nghost, gamma, _p(cons)):
        raise ValueError("oracle: invalid argument")
    return cons


def con2prim(cons, metric, nghost, gamma):
    cons, metric = _arr(cons), _arr(metric)
    n, nbox = _grid(cons, nghost)
    prim = np.empty_like(cons)
    nfail = lib().oracle_con2prim(n, nbox, _p(cons), _p(metric), nghost, gamma, _p(prim))
    if nfail < 0:
        raise ValueError("oracle: invalid argument")
    return prim, nfail


def face_bfluxes(prim, metric, nghost, recon, gamma):
    """NEXT-2: HLLE fluxes of calB on the faces (normal index 0..n, transverse -1..n), FB[nbox, 9, Nz, Ny, Nx] indexed by
    the cell whose low face it is: FB[:, 3 d + c] = F^d(calB^c); NaN where not defined."""
    prim, metric = _arr(prim), _arr(metric)
    n, nbox = _grid(prim, nghost)
    FB = np.full((nbox, 9) + prim.shape[2:], np.nan)
    r = RECON[recon] if isinstance(recon, str) else int(recon)
    if lib().oracle_face_bfluxes(n, nbox, _p(prim), _p(metric), nghost, r, gamma, _p(FB)):
        raise ValueError("oracle: invalid argument")
    return FB


def flux_ct(FB, dx, nghost):
    """NEXT-2: d calB^i/dt on the interior cells from the face fluxes by flux-CT (reading R30); dB[nbox, 3, Nz, Ny, Nx],
    ghost cells NaN."""
    FB = _arr(FB)
    nbox, nf, Nz, Ny, Nx = FB.shape
    n = (C.c_int * 3)(Nx - 2 * nghost, Ny - 2 * nghost, Nz - 2 * nghost)
    dB = np.full((nbox, 3, Nz, Ny, Nx), np.nan)
    if lib().oracle_flux_ct(n, nbox, _p(FB), (C.c_double * 3)(*dx), nghost, _p(dB)):
        raise ValueError("oracle: invalid argument")
    return dB


def valencia_rhs_ct(prim, metric, K, dx, nghost, recon, gamma):
    """Right-hand side with the calB components replaced by the flux-CT update (NEXT-2)."""
    out, nfb = valencia_rhs(prim, metric, K, dx, nghost, recon, gamma)
    dB = flux_ct(face_bfluxes(prim, metric, nghost, recon, gamma), dx, nghost)
    out[:, 5:8] = dB
    return out, nfb


def valencia_rhs_vertex(prim, metric_v, K_v, dx, nghost, recon, gamma):
    """NEXT-3 (R31): the right-hand side with the metric and K_ij sampled at the cell VERTICES,
    metric_v[nbox, 10, Nz+1, Ny+1, Nx+1] (vertex (I,J,K) = low corner of cell (I,J,K)).  Returns (out, nfallback)."""
    prim, metric_v, K_v = _arr(prim), _arr(metric_v), _arr(K_v)
    n, nbox = _grid(prim, nghost)
    assert metric_v.shape == (nbox, 10) + tuple(s + 1 for s in prim.shape[2:]) and K_v.shape[1] == 6
    out = np.full(prim.shape, np.nan)
    nfb = C.c_ulonglong(0)
    r = RECON[recon] if isinstance(recon, str) else int(recon)
    if lib().oracle_valencia_rhs_vertex(n, nbox, _p(prim), _p(metric_v), _p(K_v), (C.c_double * 3)(*dx), nghost, r, gamma,
                                        _p(out), C.byref(nfb)):
        raise ValueError("oracle: invalid argument")
    return out, int(nfb.value)


def tmunu_vertices(prim, metric_v, nghost, gamma):
    """NEXT-3 (R32): T^{mu nu} (10 components) at the vertices of the interior cells; NaN elsewhere."""
    prim, metric_v = _arr(prim), _arr(metric_v)
    n, nbox = _grid(prim, nghost)
    T = np.full((nbox, 10) + metric_v.shape[2:], np.nan)
    if lib().oracle_tmunu_vertices(n, nbox, _p(prim), _p(metric_v), nghost, gamma, _p(T)):
        raise ValueError("oracle: invalid argument")
    return T


BC = {"copy": 0, "periodic": 1}


def evolve(prim, metric, K, dx, nghost, recon, gamma, dt, nsteps, rk=2, bc="copy", ct=False):
    """Method of lines around the right-hand side (oracle_evolve; ct=True: oracle_evolve_ct, the calB components of every
    right-hand side by flux-CT): returns (prim, cons, nfail) after `nsteps` steps; `prim` must come with filled ghosts and
    is not modified."""
    prim = np.array(prim, dtype=np.float64, order="C", copy=True)
    metric, K = _arr(metric), _arr(K)
    n, nbox = _grid(prim, nghost)
    cons = np.zeros_like(prim)
    dxa = (C.c_double * 3)(*dx)
    r = RECON[recon] if isinstance(recon, str) else int(recon)
    fn = lib().oracle_evolve_ct if ct else lib().oracle_evolve
    nfail = fn(n, nbox, _p(prim), _p(metric), _p(K), dxa, nghost, r, gamma, dt, int(nsteps), int(rk), BC[bc], _p(cons))
    if nfail < 0:
        raise ValueError("oracle: invalid argument")
    return prim, cons, nfail


def recon_cell(recon, q5):
    q = _arr(q5)
    qm, qp = C.c_double(), C.c_double()
    lib().oracle_recon_cell(RECON[recon], _p(q), C.byref(qm), C.byref(qp))
    return qm.value, qp.value


def state_flux(P, met, d, gamma):
    P, met = _arr(P), _arr(met)
    U, F, lam = np.empty(8), np.empty(8), np.empty(2)
    lib().oracle_state_flux(_p(P), _p(met), d, gamma, _p(U), _p(F), _p(lam))
    return U, F, lam


def face_flux(PL, PR, CL, CR, met_face, d, gamma):
    PL, PR, CL, CR, met_face = map(_arr, (PL, PR, CL, CR, met_face))
    Fh = np.empty(8)
    lib().oracle_face_flux(_p(PL), _p(PR), _p(CL), _p(CR), _p(met_face), d, gamma, _p(Fh))
    return Fh


def hlle(UL, FL, lamL, UR, FR, lamR):
    UL, FL, lamL, UR, FR, lamR = map(_arr, (UL, FL, lamL, UR, FR, lamR))
    Fh = np.empty(8)
    lib().oracle_hlle(_p(UL), _p(FL), _p(lamL), _p(UR), _p(FR), _p(lamR), _p(Fh))
    return Fh


def sources_point(P, met, K, dm, gamma):
    P, met, K, dm = _arr(P), _arr(met), _arr(K), _arr(dm).reshape(30)
    S = np.empty(8)
    lib().oracle_sources_point(_p(P), _p(met), _p(K), _p(dm), gamma, _p(S))
    return S


PIECES = {"recon_cell": 0, "face_average": 1, "metric_complete_face": 2, "admissible": 3, "prim2con_point": 4,
          "flux_point": 5, "wavespeeds_point": 6, "hlle": 7, "metric_complete": 8, "derivative": 9,
          "sources_point": 10, "flux_difference": 11}


def count_piece(piece, d=0, recon="weno5"):
    """Operations {add, mul, div, sqrt} the counting instance executes in ONE evaluation of a piece of the
    algorithm (oracle_count_piece); the hand counts in tests/test_bench_model.py pin these."""
    ops = (C.c_ulonglong * 4)()
    if lib().oracle_count_piece(PIECES[piece], int(d), RECON[recon], ops):
        raise ValueError("oracle: invalid argument")
    return dict(add=ops[0], mul=ops[1], div=ops[2], sqrt=ops[3])


def weno_eps():
    return lib().oracle_weno_eps()


def v2max():
    return lib().oracle_v2max()


def num_threads():
    """OpenMP threads the oracle will use (what bench.py reports as `cores`)."""
    env = os.environ.get("OMP_NUM_THREADS")
    if env:
        return int(env.split(",")[0])
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1
