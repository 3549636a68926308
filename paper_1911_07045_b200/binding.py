"""Thin ctypes binding of csrc/liblq.so -- the same names as include/lq.h.

Argument marshalling only: every function forwards to the C ABI entry point of
the same name; no step of the method runs in Python.  Arrays may be numpy
arrays (host, ``LQ_HOST``) or CUDA torch tensors (``LQ_DEVICE``); they must be
contiguous, fp64 (uint8 for mask / kind / flags).  There is no CPU fallback:
if the library cannot be loaded or there is no B200, calls raise ``LqError``.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

LQ_OK, LQ_ERR_ARG, LQ_ERR_STATE, LQ_ERR_CUDA, LQ_ERR_NOMEM = 0, -1, -2, -3, -4
LQ_HOST, LQ_DEVICE = 0, 1
LQ_SITE_LC, LQ_SITE_OBJECT = 0, 1
LQ_ANCH_NONE, LQ_ANCH_ORIENTED, LQ_ANCH_DEGENERATE_PLANAR = 0, 1, 2

_LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "csrc", "liblq.so")
_lib = None

# every symbol include/lq.h declares (checked by tests/test_abi.py against the header)
SYMBOLS = ["lq_create", "lq_destroy", "lq_set_stream", "lq_set_sites", "lq_get_flags", "lq_set_Q", "lq_get_Q",
           "lq_get_velocity", "lq_set_field", "lq_set_chiral", "lq_set_cubic", "lq_analyze", "lq_energy", "lq_energy_terms", "lq_energy_terms_noalloc", "lq_forces", "lq_fire_minimize", "lq_descent_minimize", "lq_get_S0",
           "lq_set_option", "lq_get_info", "lq_last_error", "lq_version",
           "lq_create_slab", "lq_set_sites_ext", "lq_halo_bytes", "lq_halo_export", "lq_halo_import", "lq_slabs_exchange",
           "lq_slabs_fire_minimize", "lq_fire_begin", "lq_fire_step_local", "lq_fire_step_finish", "lq_fire_step_commit", "lq_fire_peek",
           "lq_fire_end"]
LQ_HALO_Q, LQ_HALO_STATE = 0, 1


class LqError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("lq error %d: %s" % (code, msg))
        self.code = code


class lq_fire_params(C.Structure):
    _fields_ = [("dt0", C.c_double), ("dtmax", C.c_double), ("alpha0", C.c_double), ("finc", C.c_double),
                ("fdec", C.c_double), ("falpha", C.c_double), ("Nmin", C.c_int), ("integrator", C.c_int),
                ("report_energy", C.c_int)]


class lq_fire_report(C.Structure):
    _fields_ = [("steps", C.c_long), ("converged", C.c_int), ("Fmax", C.c_double), ("Frms", C.c_double),
                ("P", C.c_double), ("dt", C.c_double), ("alpha", C.c_double), ("energy", C.c_double),
                ("launches", C.c_long), ("sweep_launches", C.c_long), ("gpu_ms", C.c_double)]


class lq_descent_params(C.Structure):
    _fields_ = [("eta", C.c_double), ("mu", C.c_double), ("report_energy", C.c_int)]


LQ_MIN_GD, LQ_MIN_NESTEROV = 0, 1


def lib_path() -> str:
    return _LIB_PATH


def load():
    """dlopen liblq.so and declare the prototypes.  Raises LqError if it is missing (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise LqError(LQ_ERR_CUDA, "CUDA library %s is not built (python -m paper_1911_07045_b200.build); "
                      "there is no CPU fallback" % _LIB_PATH)
    L = C.CDLL(_LIB_PATH)
    vp, dp, ip = C.c_void_p, C.POINTER(C.c_double), C.c_int
    L.lq_create.argtypes = [ip, ip, ip] + [C.c_double] * 6 + [C.POINTER(vp)]
    L.lq_destroy.argtypes = [vp]
    L.lq_destroy.restype = None
    L.lq_set_stream.argtypes = [vp, vp]
    L.lq_set_sites.argtypes = [vp, vp, vp, vp, vp, ip]
    L.lq_get_flags.argtypes = [vp, vp, ip]
    L.lq_set_Q.argtypes = [vp, vp, ip]
    L.lq_get_Q.argtypes = [vp, vp, ip]
    L.lq_get_velocity.argtypes = [vp, vp, ip]
    L.lq_energy.argtypes = [vp, dp]
    L.lq_energy_terms.argtypes = [vp, dp]
    L.lq_energy_terms_noalloc.argtypes = [vp, vp, ip]
    L.lq_forces.argtypes = [vp, vp, ip]
    L.lq_fire_minimize.argtypes = [vp, C.c_long, C.c_double, C.POINTER(lq_fire_params), C.POINTER(lq_fire_report)]
    L.lq_analyze.argtypes = [vp, C.c_double, vp, vp, vp, C.POINTER(C.c_long), ip]
    L.lq_set_chiral.argtypes = [vp, C.c_double]
    L.lq_set_cubic.argtypes = [vp, C.c_double]
    L.lq_set_field.argtypes = [vp, dp, C.c_double, dp, C.c_double]
    L.lq_descent_minimize.argtypes = [vp, ip, C.c_long, C.c_double, C.POINTER(lq_descent_params), C.POINTER(lq_fire_report)]
    L.lq_get_S0.argtypes = [vp, dp]
    L.lq_set_option.argtypes = [vp, C.c_char_p, C.c_double]
    L.lq_get_info.argtypes = [vp, C.c_char_p, dp]
    L.lq_create_slab.argtypes = [ip, ip, ip, ip, ip] + [C.c_double] * 6 + [C.POINTER(vp)]
    L.lq_set_sites_ext.argtypes = [vp, vp, vp, vp, vp, ip]
    L.lq_halo_bytes.argtypes = [vp, ip, C.POINTER(C.c_size_t)]
    L.lq_halo_export.argtypes = [vp, ip, ip, vp, ip]
    L.lq_halo_import.argtypes = [vp, ip, ip, vp, ip]
    L.lq_slabs_exchange.argtypes = [C.POINTER(vp), ip, ip]
    L.lq_slabs_fire_minimize.argtypes = [C.POINTER(vp), ip, C.c_long, C.c_double, C.POINTER(lq_fire_params),
                                         C.POINTER(lq_fire_report)]
    L.lq_fire_begin.argtypes = [vp, C.c_long, C.c_double, C.POINTER(lq_fire_params)]
    L.lq_fire_step_local.argtypes = [vp]
    L.lq_fire_step_finish.argtypes = [vp, vp, ip, C.POINTER(C.c_int)]
    L.lq_fire_step_commit.argtypes = [vp, vp, ip, ip]
    L.lq_fire_peek.argtypes = [vp, C.POINTER(lq_fire_report)]
    L.lq_fire_end.argtypes = [vp, C.POINTER(lq_fire_report)]
    L.lq_last_error.argtypes = [vp]
    L.lq_last_error.restype = C.c_char_p
    L.lq_version.restype = C.c_char_p
    for name in SYMBOLS:
        getattr(L, name)
    _lib = L
    return L


def _buf(a, dtype, count):
    """(pointer, where) of a numpy array or CUDA torch tensor; checks dtype, size, contiguity."""
    if a is None:
        return None, None
    if isinstance(a, np.ndarray):
        if a.dtype != dtype or not a.flags["C_CONTIGUOUS"] or a.size != count:
            raise LqError(LQ_ERR_ARG, "array must be C-contiguous %s with %d elements" % (np.dtype(dtype).name, count))
        return C.c_void_p(a.ctypes.data), LQ_HOST
    # torch tensor (duck-typed so that torch is not imported for host-only use)
    if hasattr(a, "data_ptr") and hasattr(a, "is_cuda"):
        import torch
        tdt = {np.dtype(np.float64): torch.float64, np.dtype(np.uint8): torch.uint8}[np.dtype(dtype)]
        if a.dtype != tdt or not a.is_contiguous() or a.numel() != count:
            raise LqError(LQ_ERR_ARG, "tensor must be contiguous %s with %d elements" % (tdt, count))
        if a.is_cuda:
            return C.c_void_p(a.data_ptr()), LQ_DEVICE
        return C.c_void_p(a.data_ptr()), LQ_HOST      # CPU (possibly pinned) tensor
    raise LqError(LQ_ERR_ARG, "unsupported buffer type %r" % type(a))


def _check(ctx, rc):
    if rc != LQ_OK:
        raise LqError(rc, load().lq_last_error(ctx).decode())


class lq_ctx:
    """Opaque handle; destroyed by lq_destroy or garbage collection."""

    def __init__(self, handle, dims):
        self.handle = handle
        self.Lx, self.Ly, self.Lz = dims
        self.N = dims[0] * dims[1] * dims[2]
        self.stream = 0                      # cudaStream_t handle last given to lq_set_stream (0 = legacy default)

    def __del__(self):
        try:
            lq_destroy(self)
        except Exception:
            pass


def lq_version() -> str:
    return load().lq_version().decode()


def lq_create(Lx, Ly, Lz, A, B, Cc, L1, L2=0.0, L3=0.0) -> lq_ctx:
    h = C.c_void_p()
    rc = load().lq_create(int(Lx), int(Ly), int(Lz), A, B, Cc, L1, L2, L3, C.byref(h))
    _check(None, rc)
    return lq_ctx(h, (int(Lx), int(Ly), int(Lz)))


def lq_destroy(ctx: lq_ctx) -> None:
    if ctx.handle is not None and _lib is not None:
        _lib.lq_destroy(ctx.handle)
    ctx.handle = None


def lq_set_stream(ctx, cuda_stream) -> None:
    """cuda_stream: integer handle (e.g. torch.cuda.current_stream().cuda_stream) or None."""
    _check(ctx.handle, load().lq_set_stream(ctx.handle, C.c_void_p(cuda_stream or 0)))
    ctx.stream = int(cuda_stream or 0)


def lq_set_sites(ctx, mask, anch_kind=None, W=None, axis=None) -> None:
    N = ctx.N
    pm, wm = _buf(mask, np.uint8, N)
    pk, wk = _buf(anch_kind, np.uint8, N)
    pw, ww = _buf(W, np.float64, N)
    pa, wa = _buf(axis, np.float64, 3 * N)
    wheres = {w for w in (wm, wk, ww, wa) if w is not None}
    if len(wheres) > 1:
        raise LqError(LQ_ERR_ARG, "lq_set_sites: all arrays must live in the same place")
    where = wheres.pop() if wheres else LQ_HOST
    _check(ctx.handle, load().lq_set_sites(ctx.handle, pm, pk, pw, pa, where))


def lq_get_flags(ctx, out=None):
    if out is None:
        out = np.empty(ctx.N, dtype=np.uint8)
    p, w = _buf(out, np.uint8, ctx.N)
    _check(ctx.handle, load().lq_get_flags(ctx.handle, p, w))
    return out


def lq_set_Q(ctx, q) -> None:
    p, w = _buf(q, np.float64, 5 * ctx.N)
    _check(ctx.handle, load().lq_set_Q(ctx.handle, p, w))


def _get5(fn, ctx, out):
    if out is None:
        out = np.empty((5, ctx.N), dtype=np.float64)
    p, w = _buf(out, np.float64, 5 * ctx.N)
    _check(ctx.handle, fn(ctx.handle, p, w))
    return out


def lq_get_Q(ctx, out=None):
    return _get5(load().lq_get_Q, ctx, out)


def lq_get_velocity(ctx, out=None):
    return _get5(load().lq_get_velocity, ctx, out)


def lq_forces(ctx, out=None):
    return _get5(load().lq_forces, ctx, out)


def lq_energy(ctx) -> float:
    e = C.c_double()
    _check(ctx.handle, load().lq_energy(ctx.handle, C.byref(e)))
    return e.value


def lq_energy_terms(ctx):
    t = (C.c_double * 3)()
    _check(ctx.handle, load().lq_energy_terms(ctx.handle, t))
    return np.array(t[:])


def lq_energy_terms_noalloc(ctx, out=None):
    """lq_energy_terms without any device allocation (static scratch inside the library; see include/lq.h for who
    needs that, the 65536-block size limit and the sharing rules).  ``out``: a 3-element fp64 numpy array (filled
    when the call returns) or CUDA torch tensor (filled in stream order, no synchronisation); None = a new numpy
    array.  Returns ``out``."""
    if out is None:
        out = np.empty(3, dtype=np.float64)
    ptr, where = _buf(out, np.float64, 3)
    _check(ctx.handle, load().lq_energy_terms_noalloc(ctx.handle, ptr, where))
    return out


def lq_get_S0(ctx) -> float:
    s = C.c_double()
    _check(ctx.handle, load().lq_get_S0(ctx.handle, C.byref(s)))
    return s.value


def lq_set_option(ctx, key: str, value: float) -> None:
    _check(ctx.handle, load().lq_set_option(ctx.handle, key.encode(), float(value)))


def lq_get_info(ctx, key: str) -> float:
    v = C.c_double()
    _check(ctx.handle, load().lq_get_info(ctx.handle, key.encode(), C.byref(v)))
    return v.value


def lq_fire_minimize(ctx, max_steps, force_tol, params: dict, report_energy=False) -> dict:
    """params: dict with dt0, dtmax, alpha0, finc, fdec, falpha, Nmin.  Returns the report as a dict."""
    fp = lq_fire_params(params["dt0"], params["dtmax"], params["alpha0"], params["finc"], params["fdec"],
                        params["falpha"], int(params["Nmin"]), int(params.get("integrator", 0)),
                        int(bool(report_energy)))
    rep = lq_fire_report()
    _check(ctx.handle, load().lq_fire_minimize(ctx.handle, int(max_steps), float(force_tol), C.byref(fp), C.byref(rep)))
    return {k: getattr(rep, k) for k, _ in lq_fire_report._fields_}


def lq_analyze(ctx, threshold=0.0, want_S=True, want_director=True, want_defect=True):
    """director / S / defect mask of the current Q into fresh host arrays.
    Returns dict(S [N], director [3][N], defect [N] uint8, n_defect)."""
    N = ctx.N
    S = np.empty(N, dtype=np.float64) if want_S else None
    d = np.empty((3, N), dtype=np.float64) if want_director else None
    m = np.empty(N, dtype=np.uint8) if want_defect else None
    cnt = C.c_long()

    def ptr(a):
        return None if a is None else C.c_void_p(a.ctypes.data)
    _check(ctx.handle, load().lq_analyze(ctx.handle, float(threshold), ptr(S), ptr(d), ptr(m), C.byref(cnt), LQ_HOST))
    return {"S": S, "director": d, "defect": m, "n_defect": cnt.value}


def lq_analyze_device(ctx, threshold, S=None, director=None, defect=None) -> int:
    """same, into caller-owned CUDA tensors (float64 [N], float64 [3][N], uint8 [N]; any may be None)"""
    cnt = C.c_long()

    def ptr(t):
        return None if t is None else C.c_void_p(t.data_ptr())
    _check(ctx.handle, load().lq_analyze(ctx.handle, float(threshold), ptr(S), ptr(director), ptr(defect), C.byref(cnt),
                                         LQ_DEVICE))
    return cnt.value


def lq_set_chiral(ctx, L4: float) -> None:
    """chiral distortion constant L4 of Eq. 10 (0 = off)"""
    _check(ctx.handle, load().lq_set_chiral(ctx.handle, float(L4)))


def lq_set_cubic(ctx, L6: float) -> None:
    """cubic distortion constant L6 of Eq. 10 (0 = off)"""
    _check(ctx.handle, load().lq_set_cubic(ctx.handle, float(L6)))


def lq_set_field(ctx, H=None, chi=0.0, E=None, eps=0.0) -> None:
    """uniform external fields of Eq. 13: H, E sequences of 3 floats (None = zero)"""
    def vec(v):
        return None if v is None else (C.c_double * 3)(*[float(t) for t in v])
    _check(ctx.handle, load().lq_set_field(ctx.handle, vec(H), float(chi), vec(E), float(eps)))


def lq_descent_minimize(ctx, method, max_steps, force_tol, eta, mu=0.0, report_energy=False) -> dict:
    """method: LQ_MIN_GD or LQ_MIN_NESTEROV; fixed step eta, momentum mu.  Returns the report as a dict."""
    dpar = lq_descent_params(float(eta), float(mu), int(bool(report_energy)))
    rep = lq_fire_report()
    _check(ctx.handle, load().lq_descent_minimize(ctx.handle, int(method), int(max_steps), float(force_tol),
                                                  C.byref(dpar), C.byref(rep)))
    return {k: getattr(rep, k) for k, _ in lq_fire_report._fields_}


def lq_last_error(ctx) -> str:
    return load().lq_last_error(ctx.handle if ctx else None).decode()


def create_from_config(c: dict) -> lq_ctx:
    """Convenience for tests / bench: context + sites + Q from a workloads.* config dict (host arrays)."""
    ctx = lq_create(c["Lx"], c["Ly"], c["Lz"], c["A"], c["B"], c["C"], c["L1"], c["L2"], c["L3"])
    if c.get("mask") is not None:
        lq_set_sites(ctx, c["mask"], c.get("kind"), c.get("W"), c.get("axis"))
    lq_set_Q(ctx, np.ascontiguousarray(c["q"]))
    return ctx


# ---------------------------------------------------------------- z-slab sub-domains (lq.h)

def _fire_params(params, report_energy=False):
    return lq_fire_params(params["dt0"], params["dtmax"], params["alpha0"], params["finc"], params["fdec"],
                          params["falpha"], int(params["Nmin"]), int(params.get("integrator", 0)), int(bool(report_energy)))


def _report(rep):
    return {k: getattr(rep, k) for k, _ in lq_fire_report._fields_}


def lq_create_slab(Lx, Ly, Lz_global, z0, nz, A, B, Cc, L1, L2=0.0, L3=0.0) -> lq_ctx:
    """sub-domain context for the planes [z0, z0 + nz) of a global Lx x Ly x Lz_global lattice"""
    h = C.c_void_p()
    _check(None, load().lq_create_slab(int(Lx), int(Ly), int(Lz_global), int(z0), int(nz), A, B, Cc, L1, L2, L3, C.byref(h)))
    ctx = lq_ctx(h, (int(Lx), int(Ly), int(nz)))
    ctx.z0, ctx.Lz_global = int(z0), int(Lz_global)
    return ctx


def lq_set_sites_ext(ctx, mask_ext, kind_ext=None, W_ext=None, axis_ext=None) -> None:
    """arrays cover the planes z0-3 .. z0+nz+2 of the global lattice: (nz + 6) * Ly * Lx sites"""
    n = (ctx.Lz + 6) * ctx.Ly * ctx.Lx
    pm, wm = _buf(mask_ext, np.uint8, n)
    pk, wk = _buf(kind_ext, np.uint8, n)
    pw, ww = _buf(W_ext, np.float64, n)
    pa, wa = _buf(axis_ext, np.float64, 3 * n)
    wheres = {w for w in (wm, wk, ww, wa) if w is not None}
    if len(wheres) != 1:
        raise LqError(LQ_ERR_ARG, "lq_set_sites_ext: all arrays must live in the same place")
    _check(ctx.handle, load().lq_set_sites_ext(ctx.handle, pm, pk, pw, pa, wheres.pop()))


def lq_halo_bytes(ctx, what) -> int:
    b = C.c_size_t()
    _check(ctx.handle, load().lq_halo_bytes(ctx.handle, int(what), C.byref(b)))
    return b.value


def _rawbuf(buf, nbytes):
    """(pointer, where) of a byte buffer: numpy array or torch tensor (any dtype) holding >= nbytes"""
    if isinstance(buf, np.ndarray):
        if not buf.flags["C_CONTIGUOUS"] or buf.nbytes < nbytes:
            raise LqError(LQ_ERR_ARG, "halo buffer too small or not contiguous")
        return C.c_void_p(buf.ctypes.data), LQ_HOST
    if hasattr(buf, "data_ptr"):
        if not buf.is_contiguous() or buf.numel() * buf.element_size() < nbytes:
            raise LqError(LQ_ERR_ARG, "halo buffer too small or not contiguous")
        return C.c_void_p(buf.data_ptr()), (LQ_DEVICE if buf.is_cuda else LQ_HOST)
    raise LqError(LQ_ERR_ARG, "unsupported buffer type %r" % type(buf))


def lq_halo_export(ctx, what, face, buf) -> None:
    p, w = _rawbuf(buf, lq_halo_bytes(ctx, what))
    _check(ctx.handle, load().lq_halo_export(ctx.handle, int(what), int(face), p, w))


def lq_halo_import(ctx, what, face, buf) -> None:
    p, w = _rawbuf(buf, lq_halo_bytes(ctx, what))
    _check(ctx.handle, load().lq_halo_import(ctx.handle, int(what), int(face), p, w))


def _handles(ctxs):
    return (C.c_void_p * len(ctxs))(*[c.handle for c in ctxs])


def lq_slabs_exchange(ctxs, what) -> None:
    _check(ctxs[0].handle, load().lq_slabs_exchange(_handles(ctxs), len(ctxs), int(what)))


def lq_slabs_fire_minimize(ctxs, max_steps, force_tol, params: dict, report_energy=False) -> dict:
    fp = _fire_params(params, report_energy)
    rep = lq_fire_report()
    _check(ctxs[0].handle, load().lq_slabs_fire_minimize(_handles(ctxs), len(ctxs), int(max_steps), float(force_tol),
                                                         C.byref(fp), C.byref(rep)))
    return _report(rep)


def lq_fire_begin(ctx, max_steps, force_tol, params: dict) -> None:
    fp = _fire_params(params)
    _check(ctx.handle, load().lq_fire_begin(ctx.handle, int(max_steps), float(force_tol), C.byref(fp)))


def lq_fire_step_local(ctx) -> None:
    """this slab's fused sweep of the next step"""
    _check(ctx.handle, load().lq_fire_step_local(ctx.handle))


def lq_fire_step_finish(ctx, tot6) -> bool:
    """fix-up launch (where the path has one) + this slab's reductions into tot6 (6 doubles: numpy array or CUDA
    tensor).  Returns True if the halo packages must be exchanged once more after the commit."""
    p, w = _buf(tot6, np.float64, 6)
    again = C.c_int()
    _check(ctx.handle, load().lq_fire_step_finish(ctx.handle, p, w, C.byref(again)))
    return bool(again.value)


def lq_fire_step_commit(ctx, rows) -> None:
    """rows: [nrank][6] doubles (numpy array or CUDA tensor), combined in rank order"""
    n = (rows.size if isinstance(rows, np.ndarray) else rows.numel()) // 6
    p, w = _buf(rows, np.float64, 6 * n)
    _check(ctx.handle, load().lq_fire_step_commit(ctx.handle, p, int(n), w))


def lq_fire_peek(ctx) -> dict:
    rep = lq_fire_report()
    _check(ctx.handle, load().lq_fire_peek(ctx.handle, C.byref(rep)))
    return _report(rep)


def lq_fire_end(ctx) -> dict:
    rep = lq_fire_report()
    _check(ctx.handle, load().lq_fire_end(ctx.handle, C.byref(rep)))
    return _report(rep)
