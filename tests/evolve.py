"""Method-of-lines driver used by the evolution tests (support code, reading R21/R22): SSP-RK2
(Heun) with "copy" outflow boundaries on the primitives.  Generic over a backend
object with rhs(prim) -> dU, prim2con(prim) -> U, con2prim(U) -> prim working on numpy arrays of
shape [nbox, 8, Nz, Ny, Nx]."""
import numpy as np


def fill_copy_bc(a, g):
    """von Neumann 'copy' boundary: ghost cells take the nearest interior value (l.255)."""
    for ax in (2, 3, 4):
        n = a.shape[ax]
        lo = [slice(None)] * 5
        hi = [slice(None)] * 5
        src_lo = [slice(None)] * 5
        src_hi = [slice(None)] * 5
        lo[ax], src_lo[ax] = slice(0, g), slice(g, g + 1)
        hi[ax], src_hi[ax] = slice(n - g, n), slice(n - g - 1, n - g)
        a[tuple(lo)] = a[tuple(src_lo)]
        a[tuple(hi)] = a[tuple(src_hi)]
    return a


def rk2_evolve(backend, prim, g, dt, nsteps):
    """U1 = Un + dt L(Un);  Un+1 = 1/2 Un + 1/2 (U1 + dt L(U1)).  Returns (prim, U)."""
    prim = fill_copy_bc(prim.copy(), g)
    U = backend.prim2con(prim)
    ii = (slice(None), slice(None), slice(g, -g), slice(g, -g), slice(g, -g))
    for _ in range(nsteps):
        L0 = backend.rhs(prim)
        U1 = U.copy()
        U1[ii] = U[ii] + dt * L0[ii]
        p1 = fill_copy_bc(backend.con2prim(U1), g)
        U1 = backend.prim2con(p1)
        L1 = backend.rhs(p1)
        U2 = U.copy()
        U2[ii] = 0.5 * U[ii] + 0.5 * (U1[ii] + dt * L1[ii])
        prim = fill_copy_bc(backend.con2prim(U2), g)
        U = backend.prim2con(prim)
    return prim, U
