"""ctypes binding of oracle/lq_oracle.c (TEST INFRASTRUCTURE, not the product).

Builds ``oracle/liblq_oracle.so`` with gcc (``-O2 -fopenmp -ffp-contract=off``:
no FMA contraction, so the arithmetic is the one written in the C file) and
exposes it through numpy arrays.  This module holds no arithmetic of its own.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lq_oracle.c")
_LIB = os.path.join(_HERE, "liblq_oracle.so")
_lib = None


def oracle_lib_path() -> str:
    return _LIB


def build_oracle(force: bool = False) -> str:
    """Compile the oracle if the .so is missing or older than its source."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    tmp = _LIB + ".tmp%d" % os.getpid()
    cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", tmp, _SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _LIB)
    return _LIB


class _Problem(C.Structure):
    _fields_ = [("Lx", C.c_int), ("Ly", C.c_int), ("Lz", C.c_int),
                ("A", C.c_double), ("B", C.c_double), ("C", C.c_double),
                ("L1", C.c_double), ("L2", C.c_double), ("L3", C.c_double),
                ("mask", C.c_void_p), ("kind", C.c_void_p), ("W", C.c_void_p), ("axis", C.c_void_p),
                ("H", C.c_double * 3), ("chi", C.c_double), ("E", C.c_double * 3), ("eps", C.c_double),
                ("L4", C.c_double), ("L6", C.c_double)]


class _FireParams(C.Structure):
    _fields_ = [("dt0", C.c_double), ("dtmax", C.c_double), ("alpha0", C.c_double),
                ("finc", C.c_double), ("fdec", C.c_double), ("falpha", C.c_double),
                ("Nmin", C.c_int), ("integrator", C.c_int)]


class _FireReport(C.Structure):
    _fields_ = [("steps", C.c_long), ("converged", C.c_int), ("Fmax", C.c_double),
                ("Frms", C.c_double), ("P", C.c_double), ("dt", C.c_double),
                ("alpha", C.c_double), ("energy", C.c_double)]


def _load():
    global _lib
    if _lib is not None:
        return _lib
    build_oracle()
    L = C.CDLL(_LIB)
    dp = C.POINTER(C.c_double)
    PP = C.POINTER(_Problem)
    L.lqo_S0.restype = C.c_double
    L.lqo_S0.argtypes = [C.c_double] * 3
    L.lqo_q0.restype = C.c_double
    L.lqo_q0.argtypes = [C.c_double] * 3
    L.lqo_num_threads.restype = C.c_int
    L.lqo_set_num_threads.argtypes = [C.c_int]
    L.lqo_classify.argtypes = [PP, C.c_void_p]
    L.lqo_site_energy.restype = C.c_double
    L.lqo_site_energy.argtypes = [PP, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, dp]
    L.lqo_energy.restype = C.c_double
    L.lqo_energy.argtypes = [PP, C.c_void_p, C.c_int, dp]
    L.lqo_forces.argtypes = [PP, C.c_void_p, C.c_void_p, C.c_int]
    L.lqo_force_at.argtypes = [PP, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, dp]
    L.lqo_fire.restype = C.c_int
    L.lqo_fire.argtypes = [PP, C.c_void_p, C.c_void_p, C.c_long, C.c_double,
                           C.POINTER(_FireParams), C.POINTER(_FireReport), C.c_int, C.c_void_p, C.c_int]
    L.lqo_descent.restype = C.c_int
    L.lqo_descent.argtypes = [PP, C.c_void_p, C.c_int, C.c_long, C.c_double, C.c_double, C.c_double,
                              C.POINTER(_FireReport), C.c_int, C.c_void_p, C.c_int]
    _lib = L
    return L


def S0_of(A, B, Cc):
    return _load().lqo_S0(A, B, Cc)


def q0_of(A, B, Cc):
    return _load().lqo_q0(A, B, Cc)


def num_threads() -> int:
    return _load().lqo_num_threads()


def set_num_threads(n: int) -> None:
    _load().lqo_set_num_threads(int(n))


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class Oracle:
    """One lattice problem held as host numpy arrays; every method calls C."""

    def __init__(self, Lx, Ly, Lz, A, B, Cc, L1, L2=0.0, L3=0.0,
                 mask=None, kind=None, W=None, axis=None, H=(0.0, 0.0, 0.0), chi=0.0, E=(0.0, 0.0, 0.0), eps=0.0, L4=0.0, L6=0.0):
        self.lib = _load()
        self.shape = (int(Lx), int(Ly), int(Lz))
        self.N = int(Lx) * int(Ly) * int(Lz)
        N = self.N
        self.mask = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8).reshape(N)
        self.kind = None if kind is None else np.ascontiguousarray(kind, dtype=np.uint8).reshape(N)
        self.W = None if W is None else np.ascontiguousarray(W, dtype=np.float64).reshape(N)
        self.axis = None if axis is None else np.ascontiguousarray(axis, dtype=np.float64).reshape(3, N)
        if self.kind is not None and (self.W is None or self.axis is None):
            raise ValueError("kind given without W/axis")
        self.p = _Problem(int(Lx), int(Ly), int(Lz), A, B, Cc, L1, L2, L3,
                          _ptr(self.mask), _ptr(self.kind), _ptr(self.W), _ptr(self.axis),
                          (C.c_double * 3)(*[float(h) for h in H]), float(chi),
                          (C.c_double * 3)(*[float(e) for e in E]), float(eps), float(L4), float(L6))

    def _q(self, q):
        q = np.ascontiguousarray(q, dtype=np.float64)
        assert q.size == 5 * self.N
        return q.reshape(5, self.N)

    def classify(self):
        f = np.empty(self.N, dtype=np.uint8)
        self.lib.lqo_classify(C.byref(self.p), _ptr(f))
        return f

    def site_energy(self, q, x, y, z, variant=0):
        q = self._q(q)
        t = (C.c_double * 3)()
        e = self.lib.lqo_site_energy(C.byref(self.p), _ptr(q), x, y, z, variant, t)
        return e, np.array(t[:])

    def energy(self, q, variant=0, terms=False):
        q = self._q(q)
        t = (C.c_double * 3)()
        e = self.lib.lqo_energy(C.byref(self.p), _ptr(q), variant, t)
        return (e, np.array(t[:])) if terms else e

    def forces(self, q, variant=0):
        q = self._q(q)
        F = np.empty((5, self.N), dtype=np.float64)
        self.lib.lqo_forces(C.byref(self.p), _ptr(q), _ptr(F), variant)
        return F

    def force_at(self, q, x, y, z, variant=0):
        q = self._q(q)
        f = (C.c_double * 5)()
        self.lib.lqo_force_at(C.byref(self.p), _ptr(q), int(x), int(y), int(z), variant, f)
        return np.array(f[:])

    def fire(self, q, max_steps, force_tol, params, variant=1, trace=False, trace_energy=False,
             return_v=False):
        """Run FIRE from q (not modified).  Returns (q_final, report dict[, v][, trace])."""
        q = self._q(q).copy()
        fp = _FireParams(params["dt0"], params["dtmax"], params["alpha0"], params["finc"],
                         params["fdec"], params["falpha"], int(params["Nmin"]), int(params.get("integrator", 0)))
        rep = _FireReport()
        v = np.zeros((5, self.N), dtype=np.float64) if return_v else None
        tr = np.zeros((max(int(max_steps), 1), 8), dtype=np.float64) if trace else None
        rc = self.lib.lqo_fire(C.byref(self.p), _ptr(q), _ptr(v), int(max_steps), float(force_tol),
                               C.byref(fp), C.byref(rep), variant, _ptr(tr), int(bool(trace_energy)))
        if rc != 0:
            raise MemoryError("lqo_fire rc=%d" % rc)
        report = {k: getattr(rep, k) for k, _ in _FireReport._fields_}
        out = [q, report]
        if return_v:
            out.append(v)
        if trace:
            out.append(tr[: report["steps"]])
        return tuple(out)

    def descent(self, q, method, max_steps, force_tol, eta, mu=0.0, variant=1, trace=False, trace_energy=False):
        """Fixed-step gradient descent (method 0) or Nesterov's accelerated gradient (method 1) from q (not
        modified).  Returns (q_final, report dict[, trace])."""
        q = self._q(q).copy()
        rep = _FireReport()
        tr = np.zeros((max(int(max_steps), 1), 3), dtype=np.float64) if trace else None
        rc = self.lib.lqo_descent(C.byref(self.p), _ptr(q), int(method), int(max_steps), float(force_tol),
                                  float(eta), float(mu), C.byref(rep), variant, _ptr(tr), int(bool(trace_energy)))
        if rc != 0:
            raise MemoryError("lqo_descent rc=%d" % rc)
        report = {k: getattr(rep, k) for k, _ in _FireReport._fields_}
        return (q, report, tr[: report["steps"]]) if trace else (q, report)


def analyze(q, mask=None, threshold=0.0):
    """Director, degree of order and defect mask of a Q field, the plain definition:
    "The nematic director can be recovered as the eigenvector corresponding to the largest eigenvalue of Q, which
    equals S" (Eq. 2) and defects are "regions where the largest eigenvalue of Q falls below some
    threshold".  numpy.linalg.eigh per site (a library routine as the one step).
    q [5][N] (xx, xy, xz, yy, yz); mask [N] or None.  Returns S [N], n [3][N] (unit, sign: largest-|.| component
    positive, first such component on ties), defect [N] uint8 (S < threshold); object sites get S = 0, n = 0, 0."""
    q = np.ascontiguousarray(q, dtype=np.float64)
    N = q.size // 5
    q = q.reshape(5, N)
    Q = np.empty((N, 3, 3))
    Q[:, 0, 0], Q[:, 0, 1], Q[:, 0, 2] = q[0], q[1], q[2]
    Q[:, 1, 0], Q[:, 1, 1], Q[:, 1, 2] = q[1], q[3], q[4]
    Q[:, 2, 0], Q[:, 2, 1], Q[:, 2, 2] = q[2], q[4], -q[0] - q[3]
    w, v = np.linalg.eigh(Q)                     # ascending eigenvalues
    S = w[:, 2].copy()
    n = v[:, :, 2].T.copy()                      # [3][N]
    k = np.argmax(np.abs(n), axis=0)
    sgn = np.sign(n[k, np.arange(N)])
    sgn[sgn == 0] = 1.0
    n *= sgn
    defect = (S < threshold).astype(np.uint8)
    if mask is not None:
        obj = np.asarray(mask).reshape(N) != 0
        S[obj] = 0.0
        n[:, obj] = 0.0
        defect[obj] = 0
    return S, n, defect
