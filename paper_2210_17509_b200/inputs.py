"""Seeded synthetic inputs shaped like the paper's tests; DESIGN.md "Input recipe".

This module serves BOTH the CUDA path and the CPU oracle.  It holds none of the method's
arithmetic: it only fills the primitive, metric and extrinsic-curvature arrays.  The single
physics-flavoured line is the change of thermodynamic variable p -> eps = p/((Gamma-1) rho)
(reading R1: the ABI carries eps; the configs are stated in p).

Layout produced (numpy float64, C-contiguous; same as include/grx.h):
    prim   [nbox, 8,  Nz, Ny, Nx]   rho, vx, vy, vz, eps, Bx, By, Bz
    metric [nbox, 10, Nz, Ny, Nx]   alp, betax, betay, betaz, gxx, gxy, gxz, gyy, gyz, gzz
    K      [nbox, 6,  Nz, Ny, Nx]   kxx, kxy, kxz, kyy, kyz, kzz
with N = n + 2*nghost and cell centres x_i = lo + (i + 1/2) dx, i = -nghost .. n+nghost-1.

These are analytic / seeded stand-ins for the paper's set-ups (Balsara-1 shocktube l.240-255,
magnetic rotor l.291-301, magnetised TOV star l.303-323, cylindrical explosion l.269-289 and
the periodic benchmark boxes l.325-345); the paper's parameter files, exact Riemann solutions
and TOV solver output are not used.
"""
from dataclasses import dataclass, field

import numpy as np

NGHOST = 3


@dataclass
class Problem:
    name: str
    n: tuple            # interior cells (nx, ny, nz)
    nbox: int
    nghost: int
    dx: tuple           # (dx, dy, dz)
    gamma: float
    prim: np.ndarray
    metric: np.ndarray
    K: np.ndarray
    recons: tuple = ("weno5",)
    meta: dict = field(default_factory=dict)

    @property
    def interior(self):
        g = self.nghost
        return (slice(None), slice(None), slice(g, -g), slice(g, -g), slice(g, -g))

    @property
    def cells(self):
        return self.n[0] * self.n[1] * self.n[2] * self.nbox


def _axes(n, lo, hi, g):
    dx = [(hi[d] - lo[d]) / n[d] for d in range(3)]
    ax = [lo[d] + (np.arange(-g, n[d] + g) + 0.5) * dx[d] for d in range(3)]
    # arrays are indexed [k, j, i]
    X = ax[0][None, None, :]
    Y = ax[1][None, :, None]
    Z = ax[2][:, None, None]
    return X, Y, Z, tuple(dx)


def _shape(n, g):
    return (n[2] + 2 * g, n[1] + 2 * g, n[0] + 2 * g)


def _minkowski(shape):
    met = np.zeros((10,) + shape)
    met[0] = 1.0
    met[4] = met[7] = met[9] = 1.0
    return met, np.zeros((6,) + shape)


def _pack(rho, v, p, B, gamma, shape):
    prim = np.empty((8,) + shape)
    prim[0] = rho
    for a in range(3):
        prim[1 + a] = v[a]
        prim[5 + a] = B[a]
    prim[4] = p / ((gamma - 1.0) * prim[0])   # R1
    return prim


def balsara1(n=(64, 4, 4), g=NGHOST):
    """Config 1: Balsara-1 shocktube block (Table I row 1), jump at x = 0.5."""
    gamma = 2.0
    nx = n[0]
    lo, hi = (0.0, 0.0, 0.0), (1.0, n[1] / nx, n[2] / nx)
    X, Y, Z, dx = _axes(n, lo, hi, g)
    shape = _shape(n, g)
    left = np.broadcast_to(X < 0.5, shape)
    rho = np.where(left, 1.0, 0.125)
    p = np.where(left, 1.0, 0.1)
    zero = np.zeros(shape)
    B = [np.full(shape, 0.5), np.where(left, 1.0, -1.0), zero]
    met, K = _minkowski(shape)
    prim = _pack(rho, [zero, zero, zero], p, B, gamma, shape)
    return Problem("C1-balsara1", tuple(n), 1, g, dx, gamma, prim[None], met[None], K[None], ("minmod", "weno5"))


def rotor(n=(256, 256, 1), g=NGHOST):
    """Config 2: magnetic-rotor-shaped block (l.293-299) with a linear taper 0.1 < r < 0.115."""
    gamma = 5.0 / 3.0
    lo, hi = (-0.5, -0.5, 0.0), (0.5, 0.5, n[2] / n[0])
    X, Y, Z, dx = _axes(n, lo, hi, g)
    shape = _shape(n, g)
    X, Y = np.broadcast_to(X, shape), np.broadcast_to(Y, shape)
    r = np.sqrt(X * X + Y * Y)
    f = np.clip((0.115 - r) / 0.015, 0.0, 1.0)
    rho = 1.0 + 9.0 * f
    omega = 9.95
    rs = np.where(r > 0.0, r, 1.0)
    scale = np.where(r <= 0.1, omega, f * omega * 0.1 / rs)
    v = [-scale * Y, scale * X, np.zeros(shape)]
    p = np.ones(shape)
    B = [np.ones(shape), np.zeros(shape), np.zeros(shape)]
    met, K = _minkowski(shape)
    prim = _pack(rho, v, p, B, gamma, shape)
    return Problem("C2-rotor", tuple(n), 1, g, dx, gamma, prim[None], met[None], K[None], ("weno5", "minmod"))


def star(n=(128, 128, 128), g=NGHOST, seed=20221031):
    """Config 3: static curved-spacetime star (shaped like the TOV test, l.303-315)."""
    gamma = 2.0
    lo, hi = (-20.0,) * 3, (20.0,) * 3
    X, Y, Z, dx = _axes(n, lo, hi, g)
    shape = _shape(n, g)
    r2 = np.broadcast_to(X * X + Y * Y + Z * Z, shape)
    M = 1.4
    s = np.sqrt(r2 + 1.0)
    u = M / (2.0 * s)
    psi = 1.0 + u
    met = np.zeros((10,) + shape)
    met[0] = (1.0 - u) / (1.0 + u)
    met[4] = met[7] = met[9] = psi ** 4
    K = np.zeros((6,) + shape)
    rho = np.maximum(1.28e-3 * np.exp(-r2 / 36.0), 1e-10)
    p = 100.0 * rho * rho
    rng = np.random.default_rng(seed)
    v = 1e-3 * (2.0 * rng.random((3,) + shape) - 1.0)
    Psi = np.exp(-r2 / 18.0)
    Bx = Psi * (X * Z / 9.0) / psi ** 6
    By = Psi * (Y * Z / 9.0) / psi ** 6
    Bz = Psi * (2.0 - (X * X + Y * Y) / 9.0) / psi ** 6
    ii = (slice(g, -g),) * 3
    amp = np.sqrt(Bx[ii] ** 2 + By[ii] ** 2 + Bz[ii] ** 2).max()
    c = 1e-6 / amp
    prim = _pack(rho, [v[0], v[1], v[2]], p, [c * Bx, c * By, c * Bz], gamma, shape)
    return Problem("C3-star", tuple(n), 1, g, dx, gamma, prim[None], met[None], K[None], ("weno5",), {"seed": seed})


def explosion(n=(256, 256, 256), g=NGHOST):
    """Config 4: cylindrical explosion (l.269-287) with a smooth tanh taper, axis along z."""
    gamma = 4.0 / 3.0
    lo, hi = (-6.0,) * 3, (6.0,) * 3
    X, Y, Z, dx = _axes(n, lo, hi, g)
    shape = _shape(n, g)
    R = np.broadcast_to(np.sqrt(X * X + Y * Y), shape)
    sig = 0.5 * (1.0 - np.tanh((R - 0.9) / 0.05))
    rho = np.exp(sig * np.log(1e-2) + (1.0 - sig) * np.log(1e-4))
    p = np.exp(sig * np.log(1.0) + (1.0 - sig) * np.log(3e-5))
    zero = np.zeros(shape)
    met, K = _minkowski(shape)
    prim = _pack(rho, [zero, zero, zero], p, [np.full(shape, 0.1), zero, zero], gamma, shape)
    return Problem("C4-explosion", tuple(n), 1, g, dx, gamma, prim[None], met[None], K[None], ("minmod", "weno5"))


def _fourier_field(rng, X, Y, Z, shape):
    """s(x) = sum_{m=1..4} a_m sin(2 pi k_m.x + phi_m), k_m in {0..3}^3 \\ 0, sum a_m = 1 => |s| <= 1."""
    ks = []
    while len(ks) < 4:
        k = rng.integers(0, 4, size=3)
        if k.any():
            ks.append(k)
    phi = rng.random(4) * 2.0 * np.pi
    a = rng.random(4)
    a = a / a.sum()
    s = np.zeros(shape)
    for m in range(4):
        ph = 2.0 * np.pi * (ks[m][0] * X + ks[m][1] * Y + ks[m][2] * Z) + phi[m]
        s += a[m] * np.sin(ph)
    return s


def _smooth_box(N, seed, g, general_metric=False):
    n = (N, N, N) if np.isscalar(N) else tuple(N)
    X, Y, Z, dx = _axes(n, (0.0,) * 3, (1.0,) * 3, g)
    shape = _shape(n, g)
    rng = np.random.default_rng(seed)
    s = lambda: _fourier_field(rng, X, Y, Z, shape)   # noqa: E731  (draw order = ABI order)
    gamma = 5.0 / 3.0
    rho = 0.55 + 0.45 * s()
    v = [(0.3 / np.sqrt(3.0)) * s() for _ in range(3)]
    p = 0.505 + 0.495 * s()
    B = [(0.5 / np.sqrt(3.0)) * s() for _ in range(3)]
    prim = _pack(rho, v, p, B, gamma, shape)
    met = np.zeros((10,) + shape)
    met[0] = 0.9 + 0.1 * s()
    for a in range(3):
        met[1 + a] = (0.05 / np.sqrt(3.0)) * s()
    psi4 = (1.1 + 0.1 * s()) ** 4
    if general_metric:
        # off-diagonal, still positive definite: psi^4 (delta_ij + 0.1 s_ij)
        for c in range(6):
            met[4 + c] = psi4 * ((1.0 if c in (0, 3, 5) else 0.0) + 0.1 * s())
    else:
        met[4] = met[7] = met[9] = psi4
    K = np.empty((6,) + shape)
    for c in range(6):
        K[c] = 0.05 * s()
    return prim, met, K, dx, gamma


def sweep_boxes(N, nbox, g=NGHOST):
    """Config 5: batch of `nbox` cubic N^3 boxes, seeded smooth random states on a perturbed
    conformally flat metric (+ a small K_ij so the K terms are exercised); seed = 1000 N + box."""
    prims, mets, Ks = [], [], []
    for b in range(nbox):
        prim, met, K, dx, gamma = _smooth_box(N, 1000 * N + b, g)
        prims.append(prim), mets.append(met), Ks.append(K)
    return Problem(f"C5-{N}^3x{nbox}", (N, N, N), nbox, g, dx, gamma, np.stack(prims), np.stack(mets), np.stack(Ks),
                   ("minmod", "weno5"))


def general_metric_box(n=(20, 12, 9), seed=7, g=NGHOST, nbox=1):
    """Extra unit config: off-diagonal gamma_ij, shift, K_ij, ragged non-cubic box (no BASELINE
    config has off-diagonal metric terms)."""
    prims, mets, Ks = [], [], []
    for b in range(nbox):
        prim, met, K, dx, gamma = _smooth_box(n, seed + b, g, general_metric=True)
        prims.append(prim), mets.append(met), Ks.append(K)
    return Problem("GEN-offdiag", tuple(n), nbox, g, dx, gamma, np.stack(prims), np.stack(mets), np.stack(Ks),
                   ("minmod", "mc", "weno5"))


SWEEP = ((32, 64), (64, 16), (128, 4), (256, 1))   # (N, nbox) of config 5


def by_name(name):
    """Problem factory for bench.py / tests: 'c1', 'c2', 'c3', 'c4', 'c5-<N>', 'gen' (+ optional ':small')."""
    small = name.endswith(":small")
    key = name.split(":")[0].lower()
    if key == "c1":
        return balsara1()
    if key == "c2":
        return rotor((64, 64, 1)) if small else rotor()
    if key == "c3":
        return star((32, 32, 32)) if small else star()
    if key == "c4":
        return explosion((48, 48, 16)) if small else explosion()
    if key.startswith("c5-"):
        N = int(key[3:])
        nbox = dict(SWEEP).get(N, 1)
        return sweep_boxes(N, 2 if small else nbox)
    if key == "gen":
        return general_metric_box()
    raise KeyError(name)
