"""Helpers shared by the tests (no method arithmetic from either implementation)."""
import numpy as np

from paper_2210_17509_b200.inputs import Problem

MET_FLAT = np.array([1.0, 0, 0, 0, 1, 0, 0, 1, 0, 1.0])
SYM = ((0, 1, 2), (1, 3, 4), (2, 4, 5))


def make_problem(n, lo, hi, gamma, prim_fn, metric_fn=None, K_fn=None, g=3, name="test"):
    """Uniform block with analytic fields.  *_fn(X, Y, Z) return lists of arrays/scalars
    (8 prims with eps, 10 metric fields, 6 K fields)."""
    dx = [(hi[d] - lo[d]) / n[d] for d in range(3)]
    ax = [lo[d] + (np.arange(-g, n[d] + g) + 0.5) * dx[d] for d in range(3)]
    shape = (n[2] + 2 * g, n[1] + 2 * g, n[0] + 2 * g)
    X = np.broadcast_to(ax[0][None, None, :], shape)
    Y = np.broadcast_to(ax[1][None, :, None], shape)
    Z = np.broadcast_to(ax[2][:, None, None], shape)

    def fill(fn, nf, default):
        arr = np.empty((nf,) + shape)
        vals = default if fn is None else fn(X, Y, Z)
        for f in range(nf):
            arr[f] = vals[f]
        return arr

    prim = fill(prim_fn, 8, None)
    met = fill(metric_fn, 10, list(MET_FLAT))
    K = fill(K_fn, 6, [0.0] * 6)
    return Problem(name, tuple(n), 1, g, tuple(dx), gamma, prim[None].copy(), met[None].copy(), K[None].copy())


def interior(prob, arr):
    return arr[prob.interior]


def relerr_per_component(a, b):
    """max|a-b| / max|b| per component (axis 1); components that vanish identically in b are
    measured against the largest component (reading R25)."""
    ncomp = b.shape[1]
    mx = np.array([np.abs(b[:, c]).max() for c in range(ncomp)])
    scale = np.where(mx > 0, mx, mx.max())
    err = np.array([np.abs(a[:, c] - b[:, c]).max() for c in range(ncomp)])
    return err / scale


def permute_problem(prob):
    """Relabel axes (x,y,z) -> (y,z,x): new x-axis is the old z-axis, etc.  Returns the permuted
    problem; new component a equals old component PERM[a]."""
    # arrays are [box, f, k(z), j(y), i(x)].  New coordinates (x',y',z') = (y,z,x)?  We define the
    # new grid by x' = z_old ... concretely: new array[k',j',i'] = old array[k=i', j=k', i=j'],
    # i.e. old x index = new y index, old y = new z, old z = new x.
    def tr(a):
        # old axes (k,j,i) = (2,3,4) -> new (k',j',i') with i'=k_old, j'=i_old, k'=j_old
        return np.ascontiguousarray(np.transpose(a, (0, 1, 3, 4, 2)))

    # old direction index of new direction a: new x = old z (2), new y = old x (0), new z = old y (1)
    old_of_new = (2, 0, 1)
    prim = tr(prob.prim)
    met = tr(prob.metric)
    K = tr(prob.K)
    prim2 = prim.copy()
    met2 = met.copy()
    K2 = K.copy()
    for a in range(3):
        prim2[:, 1 + a] = prim[:, 1 + old_of_new[a]]
        prim2[:, 5 + a] = prim[:, 5 + old_of_new[a]]
        met2[:, 1 + a] = met[:, 1 + old_of_new[a]]
    for a in range(3):
        for b in range(a, 3):
            met2[:, 4 + SYM[a][b]] = met[:, 4 + SYM[old_of_new[a]][old_of_new[b]]]
            K2[:, SYM[a][b]] = K[:, SYM[old_of_new[a]][old_of_new[b]]]
    n = tuple(prob.n[old_of_new[a]] for a in range(3))
    dx = tuple(prob.dx[old_of_new[a]] for a in range(3))
    p2 = Problem(prob.name + "-perm", n, prob.nbox, prob.nghost, dx, prob.gamma, prim2, met2, K2)
    return p2, tr, old_of_new


def cut_block(prob, lo, n, box=None):
    """Sub-block of `n` interior cells starting at interior cell `lo`, with its ghost shell taken from the
    surrounding data (so even a 1x1x1 block has non-trivial neighbours)."""
    g = prob.nghost
    sl = (slice(None) if box is None else slice(box, box + 1), slice(None),
          slice(lo[2], lo[2] + n[2] + 2 * g), slice(lo[1], lo[1] + n[1] + 2 * g), slice(lo[0], lo[0] + n[0] + 2 * g))
    arrs = [np.ascontiguousarray(a[sl]) for a in (prob.prim, prob.metric, prob.K)]
    return Problem(f"{prob.name}-cut{tuple(n)}", tuple(n), arrs[0].shape[0], g, prob.dx, prob.gamma, *arrs)
