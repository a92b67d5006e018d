"""Shared test helpers (no method arithmetic)."""
import numpy as np

from oracle import ref

G = 3
I3 = (slice(G, -G),) * 3


def make_ref(w, **override):
    opts = dict(w.opts)
    opts.update(override)
    s = ref.RefSolver(w.nx, w.ny, w.nz, w.dx, ref.make_opts(**opts))
    s.set_metric(w.metric)
    s.set_prims(w.prims)
    if w.vecpot is not None:
        s.set_vecpot(w.vecpot)
    if w.mask is not None:
        s.set_mask(w.mask)
    return s


def interior(a):
    return a[I3]


def rel_field_err(a, b, scale=None):
    """max|a-b| / max|b| over interior cells (DESIGN.md parity norm)."""
    a, b = interior(a), interior(b)
    s = np.abs(b).max() if scale is None else scale
    return np.abs(a - b).max() / max(s, 1e-300)


def cons_errors(Ua, Ub):
    """Parity norm per conserved field; vectors are scaled by the vector's max magnitude."""
    out = {}
    out["D"] = rel_field_err(Ua[0], Ub[0])
    smax = max(np.abs(interior(Ub[r])).max() for r in (1, 2, 3))
    for r, nm in zip((1, 2, 3), ("Sx", "Sy", "Sz")):
        out[nm] = rel_field_err(Ua[r], Ub[r], smax)
    out["tau"] = rel_field_err(Ua[4], Ub[4])
    bmax = max(np.abs(interior(Ub[r])).max() for r in (5, 6, 7))
    for r, nm in zip((5, 6, 7), ("Bx", "By", "Bz")):
        out[nm] = rel_field_err(Ua[r], Ub[r], bmax)
    return out


def make_gpu(w, **override):
    """The CUDA library on the same workload (imports torch/CUDA lazily)."""
    from paper_2406_11669_b200 import binding
    opts = dict(w.opts)
    opts.update(override)
    s = binding.Solver(w.nx, w.ny, w.nz, w.dx, binding.make_opts(**opts))
    s.set_metric(w.metric)
    s.set_prims(w.prims)
    if w.vecpot is not None:
        s.set_vecpot(w.vecpot)
    if w.mask is not None:
        s.set_mask(w.mask)
    return s


def to_np(fields):
    return [f.cpu().numpy() for f in fields]
