"""CPU ORACLE binding (TEST INFRASTRUCTURE -- not the product path).

ctypes wrapper around ``oracle/chfpe_ref.c`` (plain C, fp64, host only), the slow and obviously
correct restatement of the CHFPE hot path written from PAPER.md (see ``chfpe_ref.h`` for the
passages each function follows).  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package.  It shares no code with
``paper_2509_25840_b200`` and never imports it.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libchfpe_ref.so")


def build(force=False):
    """Compile the oracle with gcc (-O2, OpenMP on the outermost loops only)."""
    src = os.path.join(_HERE, "chfpe_ref.c")
    hdr = os.path.join(_HERE, "chfpe_ref.h")
    if (not force and os.path.exists(_SO)
            and os.path.getmtime(_SO) >= max(os.path.getmtime(src), os.path.getmtime(hdr))):
        return _SO
    tmp = _SO + ".tmp%d" % os.getpid()
    subprocess.check_call(["gcc", "-O2", "-std=gnu11", "-fPIC", "-shared", "-fopenmp",
                           "-ffp-contract=off", "-o", tmp, src, "-lm"])
    os.replace(tmp, _SO)
    return _SO


class Monomial(C.Structure):
    _fields_ = [("coef", C.c_double), ("expo", C.c_int32 * 3)]


class Desc(C.Structure):
    _fields_ = [("n_modes", C.c_int32), ("mass", C.c_double * 3),
                ("n_terms", C.c_int32), ("U", C.POINTER(Monomial)),
                ("V_LL", C.c_double * 3), ("V_SL", C.c_double * 3),
                ("zeta", C.c_double * 3), ("gamma", C.c_double * 3), ("beta", C.c_double),
                ("nq", C.c_int32 * 3), ("np", C.c_int32 * 3),
                ("qmin", C.c_double * 3), ("qmax", C.c_double * 3),
                ("pmin", C.c_double * 3), ("pmax", C.c_double * 3),
                ("depth", C.c_int32), ("scheme", C.c_int32), ("gauge", C.c_int32), ("batch", C.c_int32),
                ("closure", C.c_int32)]


class Observable(C.Structure):
    _fields_ = [("c0", C.c_double), ("lin_q", C.c_double * 3), ("quad", (C.c_double * 3) * 3),
                ("lin_p", C.c_double * 3)]


SCHEMES = {"central4": 0, "central2": 1, "compact6": 2}
CLOSURES = {"truncate": 0, "terminator": 1}
GAUGES = {"sqrt_eq": 0, "w": 1}

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        L = _lib
        dp = C.POINTER(C.c_double)
        L.chfpe_ref_create.argtypes = [C.POINTER(Desc), C.POINTER(C.c_void_p)]
        L.chfpe_ref_destroy.argtypes = [C.c_void_p]
        L.chfpe_ref_destroy.restype = None
        L.chfpe_ref_num_elements.argtypes = [C.c_void_p, C.POINTER(C.c_int32)]
        L.chfpe_ref_num_cells.argtypes = [C.c_void_p]
        L.chfpe_ref_num_cells.restype = C.c_int64
        L.chfpe_ref_element_index.argtypes = [C.c_void_p, C.c_int32, C.POINTER(C.c_int32)]
        L.chfpe_ref_neighbor.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
        L.chfpe_ref_deriv_axis.argtypes = [C.c_void_p, dp, C.c_int32, dp]
        L.chfpe_ref_rhs.argtypes = [C.c_void_p, dp, dp]
        L.chfpe_ref_rhs_deriv.argtypes = [C.c_void_p, dp, dp]
        L.chfpe_ref_rhs_at.argtypes = [C.c_void_p, dp, C.c_int32, C.c_int64, dp]
        L.chfpe_ref_equilibrate.argtypes = [C.c_void_p, C.c_int64, C.c_double, dp]
        L.chfpe_ref_step.argtypes = [C.c_void_p, C.c_int64, C.c_double]
        L.chfpe_ref_kick.argtypes = [C.c_void_p, C.POINTER(Observable)]
        L.chfpe_ref_expect.argtypes = [C.c_void_p, C.POINTER(Observable), dp]
        L.chfpe_ref_expect_element.argtypes = [C.c_void_p, C.c_int32, C.POINTER(Observable), dp]
        L.chfpe_ref_response_1d.argtypes = [C.c_void_p, C.POINTER(Observable), C.POINTER(Observable),
                                            C.c_int64, C.c_int64, C.c_double, dp]
        L.chfpe_ref_response_2d.argtypes = [C.c_void_p, C.POINTER(Observable), C.POINTER(Observable),
                                            C.POINTER(Observable), C.POINTER(C.c_int64), C.c_int32,
                                            C.POINTER(C.c_int64), C.c_int32, C.c_double, dp]
        L.chfpe_ref_response_3d.argtypes = [C.c_void_p] + [C.POINTER(Observable)] * 4 + \
            [C.POINTER(C.c_int64), C.c_int32] * 3 + [C.c_double, dp]
        L.chfpe_ref_export_state.argtypes = [C.c_void_p, dp]
        L.chfpe_ref_import_state.argtypes = [C.c_void_p, dp]
        L.chfpe_ref_scaled_norm2.argtypes = [C.c_void_p, dp]
        L.chfpe_ref_set_threads.argtypes = [C.c_int32]
    return _lib


def _vec3(vals, fill=0.0):
    v = list(vals) + [fill] * (3 - len(vals))
    return (C.c_double * 3)(*v)


def make_observable(c0=0.0, lin_q=(), quad=None, lin_p=()):
    o = Observable()
    o.c0 = c0
    for s, v in enumerate(lin_q):
        o.lin_q[s] = v
    for s, v in enumerate(lin_p):
        o.lin_p[s] = v
    if quad is not None:
        for a, row in enumerate(quad):
            for b, v in enumerate(row):
                o.quad[a][b] = v
    return o


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


class RefCHFPE:
    """One oracle instance.  ``cfg`` is the plain dict produced by ``chfpe_inputs.configs``."""

    def __init__(self, cfg):
        L = lib()
        M = cfg["n_modes"]
        d = Desc()
        d.n_modes = M
        d.mass = _vec3(cfg.get("mass", [1.0] * M), 1.0)
        terms = cfg["U"]
        self._terms = (Monomial * max(1, len(terms)))()
        for i, (coef, expo) in enumerate(terms):
            self._terms[i].coef = coef
            e = list(expo) + [0] * (3 - len(expo))
            self._terms[i].expo = (C.c_int32 * 3)(*e)
        d.n_terms = len(terms)
        d.U = C.cast(self._terms, C.POINTER(Monomial))
        d.V_LL = _vec3(cfg["V_LL"])
        d.V_SL = _vec3(cfg["V_SL"])
        d.zeta = _vec3(cfg["zeta"])
        d.gamma = _vec3(cfg["gamma"], 1.0)
        d.beta = cfg.get("beta", 1.0)
        d.nq = (C.c_int32 * 3)(*(list(cfg["nq"]) + [0] * (3 - M)))
        d.np = (C.c_int32 * 3)(*(list(cfg["np"]) + [0] * (3 - M)))
        d.qmin = _vec3(cfg["qmin"]); d.qmax = _vec3(cfg["qmax"])
        d.pmin = _vec3(cfg["pmin"]); d.pmax = _vec3(cfg["pmax"])
        d.depth = cfg["depth"]
        d.scheme = SCHEMES[cfg.get("scheme", "central4")]
        d.gauge = GAUGES[cfg.get("gauge", "sqrt_eq")]
        d.batch = 1
        d.closure = CLOSURES[cfg.get("closure", "truncate")]
        self._h = C.c_void_p()
        rc = L.chfpe_ref_create(C.byref(d), C.byref(self._h))
        if rc != 0:
            raise ValueError("chfpe_ref_create failed: %d" % rc)
        k = C.c_int32()
        L.chfpe_ref_num_elements(self._h, C.byref(k))
        self.K = k.value
        self.cells = L.chfpe_ref_num_cells(self._h)
        self.M = M
        self.shape = tuple(x for s in range(M) for x in (cfg["nq"][s], cfg["np"][s]))

    def close(self):
        if self._h:
            lib().chfpe_ref_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def element_index(self, k):
        n = (C.c_int32 * 3)()
        lib().chfpe_ref_element_index(self._h, k, n)
        return tuple(n[: self.M])

    def elements(self):
        return [self.element_index(k) for k in range(self.K)]

    def neighbor(self, k, s):
        up, dn = C.c_int32(), C.c_int32()
        lib().chfpe_ref_neighbor(self._h, k, s, C.byref(up), C.byref(dn))
        return up.value, dn.value

    def deriv_axis(self, f, axis):
        f = np.ascontiguousarray(f, dtype=np.float64).reshape(-1)
        out = np.empty_like(f)
        lib().chfpe_ref_deriv_axis(self._h, _dp(f), axis, _dp(out))
        return out.reshape(self.shape)

    def rhs(self, X, via_deriv=False):
        X = np.ascontiguousarray(X, dtype=np.float64).reshape(-1)
        assert X.size == self.K * self.cells
        F = np.empty_like(X)
        fn = lib().chfpe_ref_rhs_deriv if via_deriv else lib().chfpe_ref_rhs
        fn(self._h, _dp(X), _dp(F))
        return F.reshape((self.K,) + self.shape)

    def rhs_at(self, X, k, cell):
        X = np.ascontiguousarray(X, dtype=np.float64).reshape(-1)
        out = C.c_double()
        rc = lib().chfpe_ref_rhs_at(self._h, _dp(X), k, cell, C.byref(out))
        if rc != 0:
            raise ValueError("rhs_at failed")
        return out.value

    def equilibrate(self, n_steps=0, dt=0.0):
        r = C.c_double()
        lib().chfpe_ref_equilibrate(self._h, n_steps, dt, C.byref(r))
        return r.value

    def step(self, n_steps, dt):
        lib().chfpe_ref_step(self._h, n_steps, dt)

    def kick(self, obs):
        lib().chfpe_ref_kick(self._h, C.byref(obs))

    def expect(self, obs, element=0):
        out = C.c_double()
        lib().chfpe_ref_expect_element(self._h, element, C.byref(obs), C.byref(out))
        return out.value

    def response_1d(self, A, Cobs, n_samples, stride, dt):
        R = np.empty(n_samples)
        lib().chfpe_ref_response_1d(self._h, C.byref(A), C.byref(Cobs), n_samples, stride, dt, _dp(R))
        return R

    def response_2d(self, A, B, Cobs, t1_steps, t2_steps, dt):
        t1 = np.ascontiguousarray(t1_steps, dtype=np.int64)
        t2 = np.ascontiguousarray(t2_steps, dtype=np.int64)
        R = np.empty((len(t1), len(t2)))
        rc = lib().chfpe_ref_response_2d(self._h, C.byref(A), C.byref(B), C.byref(Cobs),
                                         t1.ctypes.data_as(C.POINTER(C.c_int64)), len(t1),
                                         t2.ctypes.data_as(C.POINTER(C.c_int64)), len(t2), dt, _dp(R))
        if rc != 0:
            raise ValueError("response_2d failed: %d" % rc)
        return R

    def response_3d(self, A, B, Cobs, D, t1_steps, t2_steps, t3_steps, dt):
        """Eq. (17), literal: R[k][j][l]."""
        ts = [np.ascontiguousarray(t, dtype=np.int64) for t in (t1_steps, t2_steps, t3_steps)]
        R = np.empty(tuple(len(t) for t in ts))
        args = []
        for t in ts:
            args += [t.ctypes.data_as(C.POINTER(C.c_int64)), len(t)]
        rc = lib().chfpe_ref_response_3d(self._h, C.byref(A), C.byref(B), C.byref(Cobs), C.byref(D), *args, dt, _dp(R))
        if rc != 0:
            raise ValueError("response_3d failed: %d" % rc)
        return R

    def export_state(self):
        X = np.empty(self.K * self.cells)
        lib().chfpe_ref_export_state(self._h, _dp(X))
        return X.reshape((self.K,) + self.shape)

    def import_state(self, X):
        X = np.ascontiguousarray(X, dtype=np.float64).reshape(-1)
        assert X.size == self.K * self.cells
        lib().chfpe_ref_import_state(self._h, _dp(X))

    def scaled_norm2(self):
        out = C.c_double()
        lib().chfpe_ref_scaled_norm2(self._h, C.byref(out))
        return out.value


def set_threads(n):
    return lib().chfpe_ref_set_threads(n)
