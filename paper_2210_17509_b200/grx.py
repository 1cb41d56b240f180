"""Thin binding of the C-ABI library (include/grx.h): argument marshalling only.

Every function takes torch CUDA float64 tensors (device memory and streams are PyTorch's; all
arithmetic happens in libgrx.so) in the library's layout [nbox, nfield, Nz, Ny, Nx], x fastest.
There is no CPU path: `lib()` raises if libgrx.so has not been built, and every call raises GrxError on a
non-zero return code.

    from paper_2210_17509_b200 import grx
    out = grx.valencia_rhs(prim, metric, K, dx, nghost=3, recon="weno5", gamma=5/3)
"""
import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgrx.so")

RECON = {"minmod": 0, "mc": 1, "weno5": 2}
VARIANT = {"auto": 0, "simple": 1, "ldg": 2, "tma": 3}
EXPORTS = (
    "grx_valencia_rhs", "grx_valencia_rhs_host", "grx_host_workspace_bytes", "grx_prim2con", "grx_con2prim", "grx_rk_axpy",
    "grx_step_rk", "grx_step_workspace_bytes", "grx_step_rk_ct", "grx_step_ct_workspace_bytes", "grx_valencia_rhs_ct", "grx_ct_workspace_bytes",
    "grx_valencia_rhs_ct_static", "grx_ct_static_max_bytes",
    "grx_valencia_rhs_vertex", "grx_tmunu_vertices", "grx_valencia_rhs_zrange", "grx_halo_z", "grx_halo_z_bytes", "grx_halo_z_pull", "grx_fill_ghosts", "grx_rk_stage", "grx_debug_set_fallback_counter", "grx_debug_fallback_count",
    "grx_set_variant", "grx_selftest_math", "grx_last_error", "grx_version",
    "grx_weno_eps", "grx_v2max",
)


class GrxError(RuntimeError):
    pass


class grx_grid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("nbox", C.c_int)]


_lib = None


def lib():
    """Loads libgrx.so (built by `python -m paper_2210_17509_b200.build`); raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise GrxError(f"{LIB_PATH} not found: build it with `python -m paper_2210_17509_b200.build` "
                           "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, dbl, i, sz = C.c_void_p, C.c_double, C.c_int, C.c_size_t
        gp = C.POINTER(grx_grid)
        d3 = C.POINTER(C.c_double)
        L.grx_valencia_rhs.argtypes = [gp, vp, vp, vp, d3, i, i, dbl, vp, vp]
        L.grx_valencia_rhs_host.argtypes = [gp, vp, vp, vp, d3, i, i, dbl, vp, vp, sz, vp]
        L.grx_host_workspace_bytes.argtypes = [gp, i]
        L.grx_prim2con.argtypes = [gp, vp, vp, i, dbl, vp, vp]
        L.grx_con2prim.argtypes = [gp, vp, vp, i, dbl, vp, vp, vp]
        L.grx_rk_axpy.argtypes = [gp, i, dbl, vp, dbl, dbl, vp, vp, vp]
        L.grx_step_workspace_bytes.argtypes = [gp, i, i]
        L.grx_step_rk.argtypes = [gp, vp, vp, vp, vp, d3, i, i, dbl, dbl, i, i, i, vp, sz, vp, vp]
        L.grx_step_rk_ct.argtypes = L.grx_step_rk.argtypes
        L.grx_step_ct_workspace_bytes.argtypes = [gp, i, i]
        L.grx_ct_workspace_bytes.argtypes = [gp, i]
        L.grx_valencia_rhs_ct.argtypes = [gp, vp, vp, vp, d3, i, i, dbl, vp, vp, sz, vp]
        L.grx_valencia_rhs_ct_static.argtypes = [gp, vp, vp, vp, d3, i, i, dbl, vp, vp]
        L.grx_ct_static_max_bytes.argtypes = []
        L.grx_valencia_rhs_zrange.argtypes = [gp, vp, vp, vp, d3, i, i, dbl, vp, i, i, vp]
        L.grx_halo_z_bytes.argtypes = [gp, i]
        L.grx_halo_z.argtypes = [gp, vp, i, i, i, vp, vp]
        L.grx_halo_z_pull.argtypes = [gp, vp, i, vp, vp, vp]
        L.grx_fill_ghosts.argtypes = [gp, vp, i, i, i, vp]
        L.grx_rk_stage.argtypes = [gp, i, dbl, vp, dbl, vp, dbl, vp, vp, vp, dbl, vp, dbl, vp, vp, vp]
        L.grx_valencia_rhs_vertex.argtypes = [gp, vp, vp, vp, d3, i, i, dbl, vp, vp]
        L.grx_tmunu_vertices.argtypes = [gp, vp, vp, i, dbl, vp, vp]
        L.grx_debug_set_fallback_counter.argtypes = [vp]
        L.grx_debug_fallback_count.argtypes = [C.POINTER(C.c_ulonglong), vp]
        L.grx_set_variant.argtypes = [i]
        L.grx_selftest_math.argtypes = [vp, vp, sz, vp]
        for name in EXPORTS:
            getattr(L, name).restype = C.c_int
        L.grx_host_workspace_bytes.restype = sz
        L.grx_step_workspace_bytes.restype = sz
        L.grx_step_ct_workspace_bytes.restype = sz
        L.grx_ct_workspace_bytes.restype = sz
        L.grx_ct_static_max_bytes.restype = sz
        L.grx_halo_z_bytes.restype = sz
        L.grx_last_error.restype = C.c_char_p
        L.grx_weno_eps.restype = dbl
        L.grx_v2max.restype = dbl
        _lib = L
    return _lib


def _check(rc):
    if rc != 0:
        raise GrxError(f"grx error {rc}: {lib().grx_last_error().decode()}")


def _stream(stream=None):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _dev(t, nfield=None):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise GrxError("expected a contiguous CUDA float64 tensor")
    if nfield is not None and (t.dim() != 5 or t.shape[1] != nfield):
        raise GrxError(f"expected shape [nbox, {nfield}, Nz, Ny, Nx], got {tuple(t.shape)}")
    return C.c_void_p(t.data_ptr())


def _grid(t, nghost):
    nbox, _, Nz, Ny, Nx = t.shape
    return grx_grid(Nx - 2 * nghost, Ny - 2 * nghost, Nz - 2 * nghost, nbox)


def valencia_rhs(prim, metric, K, dx, nghost, recon, gamma, out=None, stream=None):
    """grx_valencia_rhs: d/dt of (D, S_i, tau, calB^i) on the interior cells (asynchronous on the stream).
    `out` (same shape as prim) is allocated if not given; its ghost cells are left untouched."""
    import torch
    if out is None:
        out = torch.empty_like(prim)
    g = _grid(prim, nghost)
    if metric.shape[0] != prim.shape[0] or K.shape[0] != prim.shape[0] or metric.shape[2:] != prim.shape[2:] \
            or K.shape[2:] != prim.shape[2:] or out.shape != prim.shape:
        raise GrxError("prim, metric, K, out must share nbox and the spatial shape")
    r = RECON[recon] if isinstance(recon, str) else int(recon)
    dxa = (C.c_double * 3)(*[float(v) for v in dx])
    _check(lib().grx_valencia_rhs(C.byref(g), _dev(prim, 8), _dev(metric, 10), _dev(K, 6), dxa, int(nghost), r,
                                  float(gamma), _dev(out, 8), _stream(stream)))
    return out


def ct_workspace_bytes(shape, nghost):
    nbox, _, Nz, Ny, Nx = shape
    g = grx_grid(Nx - 2 * nghost, Ny - 2 * nghost, Nz - 2 * nghost, nbox)
    return lib().grx_ct_workspace_bytes(C.byref(g), int(nghost))


def valencia_rhs_ct(prim, metric, K, dx, nghost, recon, gamma, out=None, workspace=None, stream=None):
    """grx_valencia_rhs_ct (NEXT-2): the right-hand side with d calB^i/dt by flux-CT.  `workspace`: CUDA float64 tensor of
    at least ct_workspace_bytes(prim.shape, nghost) bytes (allocated if not given); on return it holds the six face-flux
    arrays [nbox, 6, Nz, Ny, Nx].  Returns (out, workspace)."""
    import torch
    if out is None:
        out = torch.empty_like(prim)
    if workspace is None:
        workspace = torch.empty((prim.shape[0], 6) + tuple(prim.shape[2:]), dtype=torch.float64, device=prim.device)
    g = _grid(prim, nghost)
    if metric.shape[0] != prim.shape[0] or K.shape[0] != prim.shape[0] or metric.shape[2:] != prim.shape[2:] \
            or K.shape[2:] != prim.shape[2:] or out.shape != prim.shape:
        raise GrxError("prim, metric, K, out must share nbox and the spatial shape")
    r = RECON[recon] if isinstance(recon, str) else int(recon)
    dxa = (C.c_double * 3)(*[float(v) for v in dx])
    _check(lib().grx_valencia_rhs_ct(C.byref(g), _dev(prim, 8), _dev(metric, 10), _dev(K, 6), dxa, int(nghost), r,
                                     float(gamma), _dev(out, 8), C.c_void_p(workspace.data_ptr()),
                                     workspace.numel() * workspace.element_size(), _stream(stream)))
    return out, workspace


def ct_static_max_bytes():
    """GRX_CT_STATIC_MAX_BYTES: the size of the library's built-in face-flux array (16 MiB)."""
    return lib().grx_ct_static_max_bytes()


def valencia_rhs_ct_static(prim, metric, K, dx, nghost, recon, gamma, out, stream=None):
    """grx_valencia_rhs_ct_static: valencia_rhs_ct for callers that cannot allocate device memory -- a code whose driver
    owns all of HBM, a callback that is handed field pointers only, a region where cudaMalloc's device-wide
    synchronisation is not acceptable.  The six face-flux arrays live in a fixed 16 MiB device array inside libgrx.so, so
    neither this wrapper nor the library allocates anything: `out` is required (same shape as prim), and the call is
    refused with GrxError when 6 * cells (ghosts included, all boxes) * 8 bytes exceeds ct_static_max_bytes().
    Make the first call on a device during start-up (it looks up the array's device address, once per device).  All calls
    on a device share the array: order them on one stream, overlapping calls corrupt each other.  Returns `out`."""
    g = _grid(prim, nghost)
    if metric.shape[0] != prim.shape[0] or K.shape[0] != prim.shape[0] or metric.shape[2:] != prim.shape[2:] \
            or K.shape[2:] != prim.shape[2:] or out.shape != prim.shape:
        raise GrxError("prim, metric, K, out must share nbox and the spatial shape")
    r = RECON[recon] if isinstance(recon, str) else int(recon)
    dxa = (C.c_double * 3)(*[float(v) for v in dx])
    _check(lib().grx_valencia_rhs_ct_static(C.byref(g), _dev(prim, 8), _dev(metric, 10), _dev(K, 6), dxa, int(nghost), r,
                                            float(gamma), _dev(out, 8), _stream(stream)))
    return out


def host_workspace_bytes(shape, nghost):
    nbox, _, Nz, Ny, Nx = shape
    g = grx_grid(Nx - 2 * nghost, Ny - 2 * nghost, Nz - 2 * nghost, nbox)
    return lib().grx_host_workspace_bytes(C.byref(g), int(nghost))


def valencia_rhs_host(prim, metric, K, dx, nghost, recon, gamma, out, workspace, stream=None):
    """grx_valencia_rhs_host: prim/metric/K/out are HOST tensors (float64, contiguous, ideally pinned);
    `workspace` is a CUDA tensor of at least host_workspace_bytes(prim.shape, nghost) bytes.  Asynchronous:
    `out` is valid after the stream is synchronised."""
    import torch
    for t in (prim, metric, K, out):
        if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
            raise GrxError("expected contiguous host float64 tensors")
    if not workspace.is_cuda:
        raise GrxError("workspace must be a CUDA tensor")
    g = _grid(prim, nghost)
    r = RECON[recon] if isinstance(recon, str) else int(recon)
    dxa = (C.c_double * 3)(*[float(v) for v in dx])
    _check(lib().grx_valencia_rhs_host(C.byref(g), C.c_void_p(prim.data_ptr()), C.c_void_p(metric.data_ptr()),
                                       C.c_void_p(K.data_ptr()), dxa, int(nghost), r, float(gamma),
                                       C.c_void_p(out.data_ptr()), C.c_void_p(workspace.data_ptr()),
                                       workspace.numel() * workspace.element_size(), _stream(stream)))
    return out


def prim2con(prim, metric, nghost, gamma, out=None, stream=None):
    import torch
    if out is None:
        out = torch.empty_like(prim)
    g = _grid(prim, nghost)
    _check(lib().grx_prim2con(C.byref(g), _dev(prim, 8), _dev(metric, 10), int(nghost), float(gamma), _dev(out, 8),
                              _stream(stream)))
    return out


def con2prim(cons, metric, nghost, gamma, out=None, nfail=None, stream=None):
    """Support code (R22).  nfail: optional CUDA int64 tensor of one element, incremented per failed cell."""
    import torch
    if out is None:
        out = torch.empty_like(cons)
    g = _grid(cons, nghost)
    nf = C.c_void_p(nfail.data_ptr()) if nfail is not None else C.c_void_p(0)
    _check(lib().grx_con2prim(C.byref(g), _dev(cons, 8), _dev(metric, 10), int(nghost), float(gamma), _dev(out, 8), nf,
                              _stream(stream)))
    return out


def rk_axpy(a, x, b, dt, rhs, y, nghost, stream=None):
    """y[int] = a*x[int] + b*(y[int] + dt*rhs[int])  (support code, R21)."""
    g = _grid(x, nghost)
    _check(lib().grx_rk_axpy(C.byref(g), int(nghost), float(a), _dev(x, 8), float(b), float(dt), _dev(rhs, 8),
                             _dev(y, 8), _stream(stream)))
    return y


BC = {"copy": 0, "periodic": 1}


def step_workspace_bytes(shape, nghost, rk):
    nbox, _, Nz, Ny, Nx = shape
    g = grx_grid(Nx - 2 * nghost, Ny - 2 * nghost, Nz - 2 * nghost, nbox)
    return lib().grx_step_workspace_bytes(C.byref(g), int(nghost), int(rk))


def step_rk(cons, prim, metric, K, dx, nghost, recon, gamma, dt, nsteps, rk=2, bc="copy", workspace=None, nfail=None,
            stream=None, ct=False):
    """grx_step_rk (ct=True: grx_step_rk_ct, constrained transport in every stage): `nsteps` device-resident method-of-lines
    steps (in place in cons and prim).  `workspace`: CUDA tensor of at least step_workspace_bytes(...) bytes (allocated if
    not given)."""
    import torch
    g = _grid(prim, nghost)
    need = step_workspace_bytes(prim.shape, nghost, rk)
    if ct:
        need = lib().grx_step_ct_workspace_bytes(C.byref(g), int(nghost), int(rk))
    if workspace is None:
        workspace = torch.empty(need // 8, dtype=torch.float64, device=prim.device)
    r = RECON[recon] if isinstance(recon, str) else int(recon)
    dxa = (C.c_double * 3)(*[float(v) for v in dx])
    nf = C.c_void_p(nfail.data_ptr()) if nfail is not None else C.c_void_p(0)
    fn = lib().grx_step_rk_ct if ct else lib().grx_step_rk
    _check(fn(C.byref(g), _dev(cons, 8), _dev(prim, 8), _dev(metric, 10), _dev(K, 6), dxa, int(nghost), r,
                             float(gamma), float(dt), int(rk), BC[bc] if isinstance(bc, str) else int(bc), int(nsteps),
                             C.c_void_p(workspace.data_ptr()), workspace.numel() * workspace.element_size(), nf,
                             _stream(stream)))
    return cons, prim


def valencia_rhs_zrange(prim, metric, K, dx, nghost, recon, gamma, out, k_begin, k_end, stream=None):
    """grx_valencia_rhs_zrange (NEXT-4): the right-hand side on the interior planes k_begin <= k < k_end of a single box."""
    g = _grid(prim, nghost)
    r = RECON[recon] if isinstance(recon, str) else int(recon)
    dxa = (C.c_double * 3)(*[float(v) for v in dx])
    _check(lib().grx_valencia_rhs_zrange(C.byref(g), _dev(prim, 8), _dev(metric, 10), _dev(K, 6), dxa, int(nghost), r,
                                         float(gamma), _dev(out, 8), int(k_begin), int(k_end), _stream(stream)))
    return out


def halo_z_bytes(shape, nghost):
    nbox, _, Nz, Ny, Nx = shape
    g = grx_grid(Nx - 2 * nghost, Ny - 2 * nghost, Nz - 2 * nghost, nbox)
    return lib().grx_halo_z_bytes(C.byref(g), int(nghost))


def halo_z(prim, nghost, side, unpack, buf, stream=None):
    """grx_halo_z (NEXT-4): pack the nghost lowest / highest interior planes of prim into buf, or unpack buf into the low /
    high z ghost planes."""
    g = _grid(prim, nghost)
    _check(lib().grx_halo_z(C.byref(g), _dev(prim, 8), int(nghost), int(side), int(bool(unpack)),
                            C.c_void_p(buf.data_ptr()), _stream(stream)))


def halo_z_pull(prim, nghost, below, above, stream=None):
    """grx_halo_z_pull (NEXT-4, peer-memory transport): fills the z ghost planes of prim straight from the prim arrays of the
    slabs below and above (same shape; this device or a peer with access enabled)."""
    g = _grid(prim, nghost)
    for t in (below, above):
        if tuple(t.shape) != tuple(prim.shape):
            raise GrxError("the neighbours' arrays must have the shape of prim")
    _check(lib().grx_halo_z_pull(C.byref(g), _dev(prim, 8), int(nghost), C.c_void_p(below.data_ptr()),
                                 C.c_void_p(above.data_ptr()), _stream(stream)))


def fill_ghosts(prim, nghost, bc="periodic", dirs=7, stream=None):
    g = _grid(prim, nghost)
    _check(lib().grx_fill_ghosts(C.byref(g), _dev(prim, 8), int(nghost), BC[bc] if isinstance(bc, str) else int(bc),
                                 int(dirs), _stream(stream)))


def rk_stage(nghost, a, Ua, b, Ub, h, L, Uout, metric, gamma, prim, acc=None, wdt=0.0, nfail=None, stream=None):
    """grx_rk_stage: Uout = a Ua + b (Ub + h L) on the interior, acc += wdt L, prim = con2prim(Uout)."""
    g = _grid(prim, nghost)
    nul = C.c_void_p(0)
    _check(lib().grx_rk_stage(C.byref(g), int(nghost), float(a), _dev(Ua, 8), float(b), _dev(Ub, 8), float(h), _dev(L, 8),
                              _dev(Uout, 8), _dev(acc, 8) if acc is not None else nul, float(wdt), _dev(metric, 10),
                              float(gamma), _dev(prim, 8), C.c_void_p(nfail.data_ptr()) if nfail is not None else nul,
                              _stream(stream)))


def _devv(t, nfield, prim):
    """A vertex array [nbox, nfield, Nz+1, Ny+1, Nx+1] that belongs to `prim`."""
    import torch
    want = (prim.shape[0], nfield) + tuple(s + 1 for s in prim.shape[2:])
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()) \
            or tuple(t.shape) != want:
        raise GrxError(f"expected a contiguous CUDA float64 vertex array of shape {want}")
    return C.c_void_p(t.data_ptr())


def valencia_rhs_vertex(prim, metric_v, K_v, dx, nghost, recon, gamma, out=None, stream=None):
    """grx_valencia_rhs_vertex (NEXT-3): the right-hand side with metric and K_ij sampled at the cell vertices."""
    import torch
    if out is None:
        out = torch.empty_like(prim)
    g = _grid(prim, nghost)
    r = RECON[recon] if isinstance(recon, str) else int(recon)
    dxa = (C.c_double * 3)(*[float(v) for v in dx])
    _check(lib().grx_valencia_rhs_vertex(C.byref(g), _dev(prim, 8), _devv(metric_v, 10, prim), _devv(K_v, 6, prim), dxa,
                                         int(nghost), r, float(gamma), _dev(out, 8), _stream(stream)))
    return out


def tmunu_vertices(prim, metric_v, nghost, gamma, out=None, stream=None):
    """grx_tmunu_vertices (NEXT-3): T^{mu nu} [nbox, 10, Nz+1, Ny+1, Nx+1] at the vertices of the interior cells."""
    import torch
    if out is None:
        out = torch.full((prim.shape[0], 10) + tuple(s + 1 for s in prim.shape[2:]), float("nan"), dtype=torch.float64,
                         device=prim.device)
    g = _grid(prim, nghost)
    _check(lib().grx_tmunu_vertices(C.byref(g), _dev(prim, 8), _devv(metric_v, 10, prim), int(nghost), float(gamma),
                                    _devv(out, 10, prim), _stream(stream)))
    return out


def set_fallback_counter(counter):
    """counter: CUDA int64 tensor of one element (caller-zeroed) or None to switch counting off."""
    _check(lib().grx_debug_set_fallback_counter(C.c_void_p(counter.data_ptr()) if counter is not None else C.c_void_p(0)))


def fallback_count(stream=None):
    """grx_debug_fallback_count: value of the counter registered with set_fallback_counter, after the work enqueued on the
    stream (synchronises it)."""
    n = C.c_ulonglong(0)
    _check(lib().grx_debug_fallback_count(C.byref(n), _stream(stream)))
    return int(n.value)


def set_variant(name):
    _check(lib().grx_set_variant(VARIANT[name] if isinstance(name, str) else int(name)))


def selftest_math(x):
    """Returns (1/x, 1/sqrt(x), sqrt(x)) computed with the kernels' division-free helpers."""
    import torch
    n = x.numel()
    y = torch.empty(3 * n, dtype=torch.float64, device=x.device)
    _check(lib().grx_selftest_math(_dev(x), _dev(y), n, _stream()))
    return y[:n], y[n:2 * n], y[2 * n:]


def version():
    return lib().grx_version()


def weno_eps():
    return lib().grx_weno_eps()


def v2max():
    return lib().grx_v2max()
