"""ctypes binding of libgrmhd.so (include/grmhd.h): argument marshalling only.

Every numerical step of the path runs in the CUDA kernels of csrc/; this module owns device
memory through torch (workspace, outputs) and passes raw pointers.  There is no CPU
fallback: if the library is missing or no CUDA device is present the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

from . import build as _build

G = 3
OK, EINVAL, ENOMEM, ESTATE, ECUDA, ENUMERIC, ELIMIT = 0, -1, -2, -3, -4, -5, -6
_ERRNAME = {EINVAL: "GRMHD_EINVAL", ENOMEM: "GRMHD_ENOMEM", ESTATE: "GRMHD_ESTATE",
            ECUDA: "GRMHD_ECUDA", ENUMERIC: "GRMHD_ENUMERIC", ELIMIT: "GRMHD_ELIMIT"}
NOALLOC_MAX_STATES = 1 << 22   # GRMHD_NOALLOC_MAX_STATES of include/grmhd.h

EXPORTS = ["grmhd_workspace_bytes", "grmhd_create", "grmhd_destroy", "grmhd_set_metric",
           "grmhd_set_prims", "grmhd_set_vecpot", "grmhd_set_mask", "grmhd_step",
           "grmhd_step_until", "grmhd_get_prims", "grmhd_get_cons", "grmhd_get_vecpot", "grmhd_get_psi",
           "grmhd_set_option", "grmhd_get_stats", "grmhd_get_kernel_times", "grmhd_launch_count", "grmhd_last_error",
           "grmhd_prim2con_batch", "grmhd_con2prim_batch", "grmhd_con2prim1d_batch", "grmhd_dfma_peak",
           "grmhd_maxspeed_noalloc"]


class GrmhdOpts(C.Structure):
    _fields_ = [("gamma_ad", C.c_double), ("poly_k", C.c_double), ("poly_gamma", C.c_double),
                ("rho_atm", C.c_double), ("p_floor", C.c_double), ("w_max", C.c_double),
                ("c2p_tol", C.c_double), ("c2p_maxit", C.c_int), ("recon", C.c_int),
                ("ppm_flatten", C.c_int), ("riemann", C.c_int), ("rk", C.c_int),
                ("bc", C.c_int * 3)]


class GrmhdStats(C.Structure):
    _fields_ = [("t", C.c_double), ("dt", C.c_double), ("maxspeed", C.c_double * 3),
                ("steps", C.c_longlong), ("c2p_fail", C.c_longlong), ("p_fix", C.c_longlong),
                ("atmo", C.c_longlong), ("w_cap", C.c_longlong), ("c2p_maxiter", C.c_longlong),
                ("c2p_backup", C.c_longlong)]


class GrmhdError(RuntimeError):
    def __init__(self, what, code, detail=""):
        self.code = code
        super().__init__(f"{what} -> {_ERRNAME.get(code, code)} {detail}".strip())


def make_opts(gamma_ad=5.0 / 3.0, poly_k=1.0, poly_gamma=None, rho_atm=1e-10, p_floor=1e-12,
              w_max=100.0, c2p_tol=1e-12, c2p_maxit=100, recon=1, ppm_flatten=1, riemann=0,
              rk=3, bc=(0, 0, 0)) -> GrmhdOpts:
    o = GrmhdOpts()
    o.gamma_ad, o.poly_k = gamma_ad, poly_k
    o.poly_gamma = gamma_ad if poly_gamma is None else poly_gamma
    o.rho_atm, o.p_floor, o.w_max = rho_atm, p_floor, w_max
    o.c2p_tol, o.c2p_maxit = c2p_tol, c2p_maxit
    o.recon, o.ppm_flatten, o.riemann, o.rk = recon, ppm_flatten, riemann, rk
    for a in range(3):
        o.bc[a] = int(bc[a])
    return o


_lib = None


def lib():
    """Load (building if stale) the CUDA library.  Raises if it cannot be built/loaded."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.grmhd_workspace_bytes.restype = C.c_size_t
        L.grmhd_workspace_bytes.argtypes = [C.c_int] * 4 + [C.POINTER(GrmhdOpts)]
        L.grmhd_create.argtypes = [C.c_int] * 4 + [C.POINTER(C.c_double), C.POINTER(GrmhdOpts),
                                                    C.c_void_p, C.c_size_t, C.c_void_p,
                                                    C.POINTER(C.c_void_p)]
        for nm in ("grmhd_set_metric", "grmhd_set_prims", "grmhd_set_vecpot", "grmhd_get_prims",
                   "grmhd_get_cons", "grmhd_get_vecpot"):
            getattr(L, nm).argtypes = [C.c_void_p, C.POINTER(C.c_void_p)]
        L.grmhd_get_psi.argtypes = [C.c_void_p, C.c_void_p]
        L.grmhd_destroy.argtypes = [C.c_void_p]
        L.grmhd_set_mask.argtypes = [C.c_void_p, C.c_void_p]
        L.grmhd_step.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.grmhd_step_until.argtypes = [C.c_void_p, C.c_double, C.c_double, C.POINTER(C.c_int)]
        L.grmhd_set_option.argtypes = [C.c_void_p, C.c_char_p, C.c_double]
        L.grmhd_get_stats.argtypes = [C.c_void_p, C.POINTER(GrmhdStats)]
        L.grmhd_get_kernel_times.argtypes = [C.c_void_p, C.POINTER(C.c_double),
                                             C.POINTER(C.c_longlong)]
        L.grmhd_launch_count.argtypes = [C.c_void_p]
        L.grmhd_launch_count.restype = C.c_longlong
        L.grmhd_last_error.argtypes = [C.c_void_p]
        L.grmhd_last_error.restype = C.c_char_p
        L.grmhd_prim2con_batch.argtypes = [C.POINTER(C.c_void_p), C.POINTER(C.c_void_p),
                                           C.POINTER(C.c_void_p), C.c_longlong,
                                           C.POINTER(GrmhdOpts), C.c_void_p]
        L.grmhd_con2prim_batch.argtypes = [C.POINTER(C.c_void_p), C.POINTER(C.c_void_p),
                                           C.POINTER(C.c_void_p), C.c_void_p, C.c_void_p,
                                           C.c_longlong, C.POINTER(GrmhdOpts), C.c_void_p]
        L.grmhd_dfma_peak.argtypes = [C.c_void_p, C.c_longlong, C.c_int, C.c_void_p]
        L.grmhd_maxspeed_noalloc.argtypes = [C.POINTER(C.c_void_p), C.POINTER(C.c_void_p),
                                             C.c_longlong, C.POINTER(GrmhdOpts), C.c_void_p,
                                             C.c_void_p, C.c_char_p, C.c_size_t]
        _lib = L
    return _lib


def _require_cuda():
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2406_11669_b200: no CUDA device; there is no CPU fallback")


def _as_arg(a, keep):
    """Pointer of a torch tensor / numpy array (fp64, contiguous); None -> NULL."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        a = np.ascontiguousarray(a, dtype=np.float64)
        keep.append(a)
        return a.ctypes.data
    if not isinstance(a, torch.Tensor):
        raise TypeError("fields must be torch tensors or numpy arrays")
    if a.dtype != torch.float64 or not a.is_contiguous():
        a = a.to(torch.float64).contiguous()
    keep.append(a)
    return a.data_ptr()


def _ptrs(arrs, n, keep):
    assert len(arrs) == n, f"expected {n} fields"
    out = (C.c_void_p * n)()
    for i, a in enumerate(arrs):
        out[i] = _as_arg(a, keep)
    return out


def _out_ptrs(arrs, n, shape):
    """Pointers of OUTPUT buffers: the library writes straight into them, so a buffer that would
    need a converted copy (wrong dtype, not contiguous, wrong shape) is an error, not a silent
    write into a temporary."""
    assert len(arrs) == n, f"expected {n} fields"
    out = (C.c_void_p * n)()
    for i, a in enumerate(arrs):
        if isinstance(a, np.ndarray):
            ok = a.dtype == np.float64 and a.flags["C_CONTIGUOUS"] and a.flags["WRITEABLE"]
            ptr = a.ctypes.data
        elif isinstance(a, torch.Tensor):
            ok = a.dtype == torch.float64 and a.is_contiguous()
            ptr = a.data_ptr()
        else:
            raise TypeError("output fields must be torch tensors or numpy arrays")
        if not ok or tuple(a.shape) != tuple(shape):
            raise ValueError(f"output field {i}: need a contiguous fp64 buffer of shape {tuple(shape)}")
        out[i] = ptr
    return out


class Solver:
    """One handle of the C ABI.  Inputs: torch tensors (CUDA or pinned/pageable host) or
    numpy arrays, fp64, shapes (nz+6, ny+6, nx+6) / staggered (nz+7, ny+7, nx+7)."""

    def __init__(self, nx, ny, nz, dx, opts: GrmhdOpts, device="cuda:0", stream=None,
                 guard_bytes=0):
        """guard_bytes > 0 (tests): that many bytes of 0xA5 are kept on both sides of the
        workspace; `guards_intact()` tells whether any kernel wrote outside it."""
        _require_cuda()
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.opts = opts
        self.device = torch.device(device)
        self.cc_shape = (self.nz + 2 * G, self.ny + 2 * G, self.nx + 2 * G)
        self.st_shape = (self.nz + 2 * G + 1, self.ny + 2 * G + 1, self.nx + 2 * G + 1)
        L = lib()
        nbytes = L.grmhd_workspace_bytes(self.nx, self.ny, self.nz, G, C.byref(opts))
        if nbytes == 0:
            raise GrmhdError("grmhd_workspace_bytes", EINVAL)
        self.workspace_bytes = int(nbytes)
        gb = (int(guard_bytes) + 255) // 256 * 256
        with torch.cuda.device(self.device):
            self._ws = torch.empty(nbytes + 256 + 2 * gb, dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        base = (self._ws.data_ptr() + 255) // 256 * 256 + gb
        self._guard = None
        if gb:
            off = base - self._ws.data_ptr()
            self._guard = (self._ws[off - gb:off], self._ws[off + nbytes:off + nbytes + gb])
            for t in self._guard:
                t.fill_(0xA5)
        self.h = C.c_void_p()
        d = (C.c_double * 3)(*[float(x) for x in dx])
        rc = L.grmhd_create(self.nx, self.ny, self.nz, G, d, C.byref(opts), C.c_void_p(base),
                            C.c_size_t(nbytes), C.c_void_p(self.stream.cuda_stream),
                            C.byref(self.h))
        if rc != OK:
            raise GrmhdError("grmhd_create", rc)

    def guards_intact(self) -> bool:
        """True if the guard zones around the workspace still hold their pattern."""
        assert self._guard is not None, "create the Solver with guard_bytes > 0"
        self.stream.synchronize()
        return all(bool((t == 0xA5).all()) for t in self._guard)

    def close(self):
        if getattr(self, "h", None) is not None and self.h.value:
            lib().grmhd_destroy(self.h)
            self.h = C.c_void_p()
        self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _chk(self, rc, what):
        if rc != OK:
            msg = lib().grmhd_last_error(self.h)
            raise GrmhdError(what, rc, msg.decode() if msg else "")

    # ---- inputs
    def set_metric(self, fields):
        keep = []
        self._chk(lib().grmhd_set_metric(self.h, _ptrs(fields, 16, keep)), "grmhd_set_metric")
        self.stream.synchronize()  # host sources may be temporaries

    def set_prims(self, fields):
        keep = []
        self._chk(lib().grmhd_set_prims(self.h, _ptrs(fields, 8, keep)), "grmhd_set_prims")
        self.stream.synchronize()

    def set_vecpot(self, fields):
        keep = []
        self._chk(lib().grmhd_set_vecpot(self.h, _ptrs(fields, 3, keep)), "grmhd_set_vecpot")
        self.stream.synchronize()

    def set_mask(self, mask):
        if mask is None:
            self._chk(lib().grmhd_set_mask(self.h, None), "grmhd_set_mask")
            return
        if isinstance(mask, np.ndarray):
            m = np.ascontiguousarray(mask, dtype=np.uint8)
            ptr = m.ctypes.data
        else:
            m = mask.to(torch.uint8).contiguous()
            ptr = m.data_ptr()
        assert tuple(m.shape) == self.cc_shape
        self._chk(lib().grmhd_set_mask(self.h, C.c_void_p(ptr)), "grmhd_set_mask")
        self.stream.synchronize()

    def set_option(self, key, value):
        self._chk(lib().grmhd_set_option(self.h, key.encode(), float(value)), "grmhd_set_option")

    # ---- evolution
    def step(self, n, cfl):
        self._chk(lib().grmhd_step(self.h, int(n), float(cfl)), "grmhd_step")

    def step_until(self, t_end, cfl):
        n = C.c_int(0)
        self._chk(lib().grmhd_step_until(self.h, float(t_end), float(cfl), C.byref(n)),
                  "grmhd_step_until")
        return n.value

    # ---- outputs
    def _get(self, fn, what, n, shape, out, host):
        if out is None:
            if host:
                out = [torch.empty(shape, dtype=torch.float64).pin_memory() for _ in range(n)]
            else:
                out = [torch.empty(shape, dtype=torch.float64, device=self.device)
                       for _ in range(n)]
        self._chk(fn(self.h, _out_ptrs(out, n, shape)), what)
        return out

    def get_prims(self, out=None, host=False):
        return self._get(lib().grmhd_get_prims, "grmhd_get_prims", 8, self.cc_shape, out, host)

    def get_cons(self, out=None, host=False):
        return self._get(lib().grmhd_get_cons, "grmhd_get_cons", 8, self.cc_shape, out, host)

    def get_vecpot(self, out=None, host=False):
        return self._get(lib().grmhd_get_vecpot, "grmhd_get_vecpot", 3, self.st_shape, out, host)

    def get_psi(self):
        """Psi_mhd of the generalised Lorenz gauge on the vertices (staggered shape)."""
        out = torch.empty(self.st_shape, dtype=torch.float64, device=self.device)
        self._chk(lib().grmhd_get_psi(self.h, C.c_void_p(out.data_ptr())), "grmhd_get_psi")
        return out

    def stats(self) -> dict:
        s = GrmhdStats()
        rc = lib().grmhd_get_stats(self.h, C.byref(s))
        d = {k: getattr(s, k) for k, _ in GrmhdStats._fields_ if k != "maxspeed"}
        d["maxspeed"] = [s.maxspeed[i] for i in range(3)]
        d["rc"] = rc
        return d

    KERNEL_GROUPS = ("flux_x", "flux_y", "flux_z", "update", "bfield", "con2prim", "ghost_prims",
                     "dt", "sources")

    def kernel_times(self) -> dict:
        """{group: (summed ms, brackets)} since set_option("kernel_timing", 1)."""
        ms = (C.c_double * 9)()
        cnt = (C.c_longlong * 9)()
        self._chk(lib().grmhd_get_kernel_times(self.h, ms, cnt), "grmhd_get_kernel_times")
        return {k: (ms[i], cnt[i]) for i, k in enumerate(self.KERNEL_GROUPS)}

    def launch_count(self) -> int:
        return int(lib().grmhd_launch_count(self.h))


# ---- stand-alone batches (device tensors, structure of arrays) -------------------------
def prim2con_batch(prim, metric, opts: GrmhdOpts):
    """prim (8,n), metric (10,n) CUDA fp64 tensors -> cons (8,n)."""
    _require_cuda()
    n = prim.shape[1]
    cons = torch.empty((8, n), dtype=torch.float64, device=prim.device)
    keep = []
    rc = lib().grmhd_prim2con_batch(_ptrs(list(prim), 8, keep), _ptrs(list(metric), 10, keep),
                                    _ptrs(list(cons), 8, keep), n, C.byref(opts),
                                    C.c_void_p(torch.cuda.current_stream().cuda_stream))
    if rc != OK:
        raise GrmhdError("grmhd_prim2con_batch", rc)
    return cons


def con2prim_batch(cons, metric, opts: GrmhdOpts):
    """cons (8,n), metric (10,n) -> prim (5,n), status (n) int32, iters (n) int32."""
    _require_cuda()
    n = cons.shape[1]
    prim = torch.empty((5, n), dtype=torch.float64, device=cons.device)
    status = torch.empty(n, dtype=torch.int32, device=cons.device)
    iters = torch.empty(n, dtype=torch.int32, device=cons.device)
    keep = []
    rc = lib().grmhd_con2prim_batch(_ptrs(list(cons), 8, keep), _ptrs(list(metric), 10, keep),
                                    _ptrs(list(prim), 5, keep), C.c_void_p(status.data_ptr()),
                                    C.c_void_p(iters.data_ptr()), n, C.byref(opts),
                                    C.c_void_p(torch.cuda.current_stream().cuda_stream))
    if rc != OK:
        raise GrmhdError("grmhd_con2prim_batch", rc)
    return prim, status, iters


def con2prim1d_batch(cons, metric, opts: GrmhdOpts):
    """The 1-D backup scheme alone: cons (8,n), metric (10,n) -> prim (5,n), status, iters."""
    _require_cuda()
    n = cons.shape[1]
    prim = torch.empty((5, n), dtype=torch.float64, device=cons.device)
    status = torch.empty(n, dtype=torch.int32, device=cons.device)
    iters = torch.empty(n, dtype=torch.int32, device=cons.device)
    keep = []
    rc = lib().grmhd_con2prim1d_batch(_ptrs(list(cons), 8, keep), _ptrs(list(metric), 10, keep),
                                      _ptrs(list(prim), 5, keep), C.c_void_p(status.data_ptr()),
                                      C.c_void_p(iters.data_ptr()), n, C.byref(opts),
                                      C.c_void_p(torch.cuda.current_stream().cuda_stream))
    if rc != OK:
        raise GrmhdError("grmhd_con2prim1d_batch", rc)
    return prim, status, iters


def maxspeed_noalloc(prim, metric, opts: GrmhdOpts, out, stream=None):
    """grmhd_maxspeed_noalloc: max |lambda| along x, y, z over n plain states, with no allocation
    on the library's side (its scratch is a static device array; n <= NOALLOC_MAX_STATES).
    prim (8,n) and metric (10,n) contiguous CUDA fp64 tensors; `out` = the caller's CUDA fp64
    tensor of 3 elements (this wrapper allocates nothing on the device either).  Only enqueues on
    `stream` (default: torch's current stream).  Calls that overlap on the GPU race on the
    library's scratch array."""
    _require_cuda()
    for t, rows in ((prim, 8), (metric, 10)):
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64
                and t.dim() == 2 and t.shape[0] == rows and t.is_contiguous()):
            raise ValueError(f"need a contiguous CUDA fp64 tensor of shape ({rows}, n)")
    if not (isinstance(out, torch.Tensor) and out.is_cuda and out.dtype == torch.float64
            and out.numel() == 3 and out.is_contiguous()):
        raise ValueError("out: need a contiguous CUDA fp64 tensor of 3 elements")
    n = int(prim.shape[1])
    if metric.shape[1] != n:
        raise ValueError("prim and metric hold a different number of states")
    pp = (C.c_void_p * 8)(*[prim[r].data_ptr() for r in range(8)])
    mp = (C.c_void_p * 10)(*[metric[r].data_ptr() for r in range(10)])
    s = stream if stream is not None else torch.cuda.current_stream(prim.device)
    msg = C.create_string_buffer(256)
    with torch.cuda.device(prim.device):
        rc = lib().grmhd_maxspeed_noalloc(pp, mp, n, C.byref(opts), C.c_void_p(out.data_ptr()),
                                          C.c_void_p(s.cuda_stream), msg, len(msg))
    if rc != OK:
        raise GrmhdError("grmhd_maxspeed_noalloc", rc, msg.value.decode())
    return out


def dfma_peak(threads=148 * 2048, iters=4096, reps=5):
    """Measured FP64 FMA throughput in TFLOP/s (2 flops per DFMA), best of `reps`."""
    _require_cuda()
    out = torch.empty(threads, dtype=torch.float64, device="cuda")
    s = torch.cuda.current_stream()
    best = 0.0
    for _ in range(reps + 1):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(s)
        rc = lib().grmhd_dfma_peak(C.c_void_p(out.data_ptr()), threads, iters,
                                   C.c_void_p(s.cuda_stream))
        e1.record(s)
        e1.synchronize()
        if rc != OK:
            raise GrmhdError("grmhd_dfma_peak", rc)
        ms = e0.elapsed_time(e1)
        best = max(best, 2.0 * 16 * iters * threads / (ms * 1e-3) / 1e12)
    return best
