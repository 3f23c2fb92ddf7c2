"""ctypes binding of include/chfpe.h (same names, argument marshalling only)."""
import ctypes as C
import os

import numpy as np

from . import build as _build

EXPORTED_SYMBOLS = [
    "chfpe_workspace_bytes", "chfpe_create", "chfpe_destroy", "chfpe_num_elements", "chfpe_element_index",
    "chfpe_equilibrate", "chfpe_step", "chfpe_kick", "chfpe_expect", "chfpe_expect_element",
    "chfpe_response_1d", "chfpe_response_2d", "chfpe_response_3d", "chfpe_export_state", "chfpe_import_state", "chfpe_export_rhs",
    "chfpe_rk4_stage", "chfpe_stage_input", "chfpe_launch_count", "chfpe_profile_enable", "chfpe_profile_read", "chfpe_stage_kernel", "chfpe_spectrum_1d", "chfpe_spectrum_2d", "chfpe_spectrum_2d_static", "chfpe_last_error",
    "chfpe_hermite_workspace_bytes", "chfpe_hermite_create", "chfpe_hermite_destroy", "chfpe_hermite_num_elements",
    "chfpe_hermite_equilibrate", "chfpe_hermite_step", "chfpe_hermite_kick", "chfpe_hermite_expect",
    "chfpe_hermite_response_1d", "chfpe_hermite_response_2d", "chfpe_hermite_response_3d", "chfpe_hermite_export_state",
    "chfpe_hermite_import_state", "chfpe_hermite_export_rhs", "chfpe_hermite_launch_count", "chfpe_hermite_stage_kernel", "chfpe_hermite_last_error",
]


class ChfpeError(RuntimeError):
    pass


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
GAUGES = {"sqrt_eq": 0, "w": 1}
CLOSURES = {"truncate": 0, "terminator": 1}
_lib = None


def lib():
    """Load libchfpe.so (building it in-tree with nvcc if absent).  Raises if that is impossible."""
    global _lib
    if _lib is not None:
        return _lib
    try:
        so = _build.build()
    except FileNotFoundError as exc:   # no nvcc on this machine: a prebuilt library is acceptable only if it is not stale
        if not os.path.exists(_build.SO):
            raise ChfpeError("libchfpe.so is missing and nvcc is not available to build it: %s" % exc)
        if _build.stale():
            raise ChfpeError("libchfpe.so is older than its sources and nvcc is not available to rebuild it")
        so = _build.SO
    # any other failure (e.g. a compile error in freshly edited sources) propagates: never run a stale binary
    L = C.CDLL(so)
    vp, dp, i64p = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int64)
    op = C.POINTER(Observable)
    L.chfpe_workspace_bytes.argtypes = [C.POINTER(Desc), C.POINTER(C.c_size_t)]
    L.chfpe_create.argtypes = [C.POINTER(Desc), vp, C.c_size_t, vp, C.POINTER(vp)]
    L.chfpe_destroy.argtypes = [vp]
    L.chfpe_num_elements.argtypes = [vp, C.POINTER(C.c_int32)]
    L.chfpe_element_index.argtypes = [vp, C.c_int32, C.POINTER(C.c_int32)]
    L.chfpe_equilibrate.argtypes = [vp, C.c_int64, C.c_double, dp]
    L.chfpe_step.argtypes = [vp, C.c_int64, C.c_double]
    L.chfpe_kick.argtypes = [vp, op]
    L.chfpe_expect.argtypes = [vp, op, dp]
    L.chfpe_expect_element.argtypes = [vp, C.c_int32, C.c_int32, op, dp]
    L.chfpe_response_1d.argtypes = [vp, op, op, C.c_int64, C.c_int64, C.c_double, dp]
    L.chfpe_response_2d.argtypes = [vp, op, op, op, i64p, C.c_int32, i64p, C.c_int32, C.c_double, dp]
    L.chfpe_response_3d.argtypes = [vp, op, op, op, op, i64p, C.c_int32, i64p, C.c_int32, i64p, C.c_int32, C.c_double, dp]
    L.chfpe_export_state.argtypes = [vp, C.c_int32, vp, C.c_int]
    L.chfpe_import_state.argtypes = [vp, C.c_int32, vp, C.c_int]
    L.chfpe_export_rhs.argtypes = [vp, C.c_int32, vp, C.c_int]
    L.chfpe_launch_count.argtypes = [vp, C.POINTER(C.c_int64)]
    L.chfpe_rk4_stage.argtypes = [vp, C.c_int32, C.c_double]
    L.chfpe_stage_input.argtypes = [vp, C.c_int32, C.c_int32, C.POINTER(vp), C.POINTER(C.c_int64)]
    L.chfpe_profile_enable.argtypes = [vp, C.c_int]
    L.chfpe_profile_read.argtypes = [vp, dp, C.POINTER(C.c_int64)]
    L.chfpe_stage_kernel.argtypes = [vp, C.POINTER(C.c_int32)]
    L.chfpe_spectrum_1d.argtypes = [vp, vp, C.c_int64, C.c_double, vp, C.c_int32, vp]
    L.chfpe_spectrum_2d.argtypes = [vp, vp, C.c_int32, C.c_int32, C.c_double, C.c_double, vp, C.c_int32, vp, C.c_int32,
                                    C.c_int32, C.c_int32, vp, vp]
    L.chfpe_spectrum_2d_static.argtypes = [vp, vp, C.c_int32, C.c_int32, C.c_double, C.c_double, vp, C.c_int32, vp,
                                           C.c_int32, C.c_int32, C.c_int32, vp]
    L.chfpe_last_error.argtypes = [vp]
    L.chfpe_last_error.restype = C.c_char_p
    L.chfpe_hermite_workspace_bytes.argtypes = [C.POINTER(Desc), C.POINTER(C.c_size_t)]
    L.chfpe_hermite_create.argtypes = [C.POINTER(Desc), vp, C.c_size_t, vp, C.POINTER(vp)]
    L.chfpe_hermite_destroy.argtypes = [vp]
    L.chfpe_hermite_num_elements.argtypes = [vp, C.POINTER(C.c_int32)]
    L.chfpe_hermite_equilibrate.argtypes = [vp, C.c_int64, C.c_double, dp]
    L.chfpe_hermite_step.argtypes = [vp, C.c_int64, C.c_double]
    L.chfpe_hermite_kick.argtypes = [vp, op]
    L.chfpe_hermite_expect.argtypes = [vp, C.c_int32, op, dp]
    L.chfpe_hermite_response_1d.argtypes = [vp, op, op, C.c_int64, C.c_int64, C.c_double, dp]
    L.chfpe_hermite_response_2d.argtypes = [vp, op, op, op, i64p, C.c_int32, i64p, C.c_int32, C.c_double, dp]
    L.chfpe_hermite_response_3d.argtypes = [vp, op, op, op, op, i64p, C.c_int32, i64p, C.c_int32, i64p, C.c_int32,
                                            C.c_double, dp]
    L.chfpe_hermite_export_state.argtypes = [vp, C.c_int32, vp, C.c_int]
    L.chfpe_hermite_import_state.argtypes = [vp, C.c_int32, vp, C.c_int]
    L.chfpe_hermite_export_rhs.argtypes = [vp, C.c_int32, vp, C.c_int]
    L.chfpe_hermite_launch_count.argtypes = [vp, C.POINTER(C.c_int64)]
    L.chfpe_hermite_stage_kernel.argtypes = [vp, C.POINTER(C.c_int32)]
    L.chfpe_hermite_last_error.argtypes = [vp]
    L.chfpe_hermite_last_error.restype = C.c_char_p
    _lib = L
    return L


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


def make_desc(cfg, batch=1):
    """Fill a chfpe_desc from a plain parameter dict (chfpe_inputs.config).  Returns (desc, keepalive)."""
    M = cfg["n_modes"]
    d = Desc()
    d.n_modes = M
    d.mass = _vec3(cfg.get("mass", [1.0] * M), 1.0)
    terms = cfg["U"]
    arr = (Monomial * max(1, len(terms)))()
    for i, (coef, expo) in enumerate(terms):
        arr[i].coef = coef
        arr[i].expo = (C.c_int32 * 3)(*(list(expo) + [0] * (3 - len(expo))))
    d.n_terms = len(terms)
    d.U = C.cast(arr, C.POINTER(Monomial))
    d.V_LL = _vec3(cfg["V_LL"])
    d.V_SL = _vec3(cfg["V_SL"])
    d.zeta = _vec3(cfg["zeta"])
    d.gamma = _vec3(cfg["gamma"], 1.0)
    d.beta = cfg.get("beta", 1.0)
    d.nq = (C.c_int32 * 3)(*(list(cfg["nq"]) + [0] * (3 - M)))
    d.np = (C.c_int32 * 3)(*(list(cfg["np"]) + [0] * (3 - M)))
    d.qmin = _vec3(cfg["qmin"])
    d.qmax = _vec3(cfg["qmax"])
    d.pmin = _vec3(cfg["pmin"])
    d.pmax = _vec3(cfg["pmax"])
    d.depth = cfg["depth"]
    d.scheme = SCHEMES[cfg.get("scheme", "central4")]
    d.gauge = GAUGES[cfg.get("gauge", "sqrt_eq")]
    d.batch = batch
    d.closure = CLOSURES[cfg.get("closure", "truncate")]
    return d, arr


def workspace_bytes(cfg, batch=1):
    d, _keep = make_desc(cfg, batch)
    n = C.c_size_t()
    rc = lib().chfpe_workspace_bytes(C.byref(d), C.byref(n))
    if rc != 0:
        raise ChfpeError("chfpe_workspace_bytes: %d %s" % (rc, lib().chfpe_last_error(None).decode()))
    return n.value


class CHFPE:
    """One library handle.  The workspace is a torch uint8 CUDA tensor owned by this object."""

    def __init__(self, cfg, batch=1, device="cuda:0", stream=None, guard_bytes=0):
        import torch
        if not torch.cuda.is_available():
            raise ChfpeError("CUDA device required: the CHFPE path has no CPU fallback")
        L = lib()
        self._torch = torch
        self.device = torch.device(device)
        d, keep = make_desc(cfg, batch)
        nbytes = workspace_bytes(cfg, batch)
        with torch.cuda.device(self.device):
            # guard_bytes > 0 (tests): canary bytes on both sides of the workspace, checked by guards_intact()
            self._guard = int(guard_bytes)
            self.workspace = torch.full((nbytes + 256 + 2 * self._guard,), 0xA5, dtype=torch.uint8, device=self.device) \
                if self._guard else torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            base = self.workspace.data_ptr() + self._guard
            aligned = (base + 255) & ~255
            self._ws_lo, self._ws_hi = aligned - self.workspace.data_ptr(), aligned - self.workspace.data_ptr() + nbytes
            self._h = C.c_void_p()
            rc = L.chfpe_create(C.byref(d), C.c_void_p(aligned), nbytes, C.c_void_p(self.stream.cuda_stream),
                                C.byref(self._h))
        if rc != 0:
            raise ChfpeError("chfpe_create: %d %s" % (rc, L.chfpe_last_error(None).decode()))
        self.cfg = cfg
        self.batch = batch
        self.M = cfg["n_modes"]
        k = C.c_int32()
        L.chfpe_num_elements(self._h, C.byref(k))
        self.K = k.value
        self.shape = tuple(x for s in range(self.M) for x in (cfg["nq"][s], cfg["np"][s]))
        self.cells = int(np.prod(self.shape))

    def _ck(self, rc, what):
        if rc != 0:
            raise ChfpeError("%s: %d %s" % (what, rc, lib().chfpe_last_error(self._h).decode()))

    def guards_intact(self):
        """True if no byte outside [workspace, workspace + workspace_bytes) was written (needs guard_bytes > 0)."""
        self._torch.cuda.synchronize(self.device)
        w = self.workspace
        return bool((w[: self._ws_lo] == 0xA5).all().item() and (w[self._ws_hi:] == 0xA5).all().item())

    def close(self):
        if getattr(self, "_h", None):
            lib().chfpe_destroy(self._h)
            self._h = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def element_index(self, k):
        n = (C.c_int32 * 3)()
        self._ck(lib().chfpe_element_index(self._h, k, n), "chfpe_element_index")
        return tuple(n[: self.M])

    def elements(self):
        return [self.element_index(k) for k in range(self.K)]

    def equilibrate(self, n_steps=0, dt=0.0, residual=True):
        r = C.c_double()
        self._ck(lib().chfpe_equilibrate(self._h, n_steps, dt, C.byref(r) if residual else None), "chfpe_equilibrate")
        return r.value if residual else None

    def step(self, n_steps, dt):
        self._ck(lib().chfpe_step(self._h, n_steps, dt), "chfpe_step")

    def kick(self, obs):
        self._ck(lib().chfpe_kick(self._h, C.byref(obs)), "chfpe_kick")

    def expect(self, obs):
        out = np.empty(self.batch)
        self._ck(lib().chfpe_expect(self._h, C.byref(obs), out.ctypes.data_as(C.POINTER(C.c_double))), "chfpe_expect")
        return out

    def expect_element(self, obs, k, replica=0):
        out = C.c_double()
        self._ck(lib().chfpe_expect_element(self._h, replica, k, C.byref(obs), C.byref(out)), "chfpe_expect_element")
        return out.value

    def response_1d(self, A, Cobs, n_samples, stride, dt):
        """A may be None: no kick, continue the trajectory replica 0 holds."""
        R = np.empty(n_samples)
        self._ck(lib().chfpe_response_1d(self._h, C.byref(A) if A is not None else None, C.byref(Cobs),
                                         n_samples, stride, dt,
                                         R.ctypes.data_as(C.POINTER(C.c_double))), "chfpe_response_1d")
        return R

    def response_2d(self, A, B, Cobs, t1_steps, t2_steps, dt):
        t1 = np.ascontiguousarray(t1_steps, dtype=np.int64)
        t2 = np.ascontiguousarray(t2_steps, dtype=np.int64)
        R = np.empty((len(t1), len(t2)))
        self._ck(lib().chfpe_response_2d(self._h, C.byref(A), C.byref(B), C.byref(Cobs),
                                         t1.ctypes.data_as(C.POINTER(C.c_int64)), len(t1),
                                         t2.ctypes.data_as(C.POINTER(C.c_int64)), len(t2), dt,
                                         R.ctypes.data_as(C.POINTER(C.c_double))), "chfpe_response_2d")
        return R

    def response_3d(self, A, B, Cobs, D, t1_steps, t2_steps, t3_steps, dt):
        """R[k][j][l] of Eq. (17); needs batch >= 3."""
        ts = [np.ascontiguousarray(t, dtype=np.int64) for t in (t1_steps, t2_steps, t3_steps)]
        R = np.empty(tuple(len(t) for t in ts))
        args = []
        for t in ts:
            args += [t.ctypes.data_as(C.POINTER(C.c_int64)), len(t)]
        self._ck(lib().chfpe_response_3d(self._h, C.byref(A), C.byref(B), C.byref(Cobs), C.byref(D), *args, dt,
                                         R.ctypes.data_as(C.POINTER(C.c_double))), "chfpe_response_3d")
        return R

    def export_state(self, replica=0):
        X = np.empty((self.K,) + self.shape)
        self._ck(lib().chfpe_export_state(self._h, replica, C.c_void_p(X.ctypes.data), 0), "chfpe_export_state")
        return X

    def export_state_device(self, replica=0):
        t = self._torch.empty((self.K,) + self.shape, dtype=self._torch.float64, device=self.device)
        self._ck(lib().chfpe_export_state(self._h, replica, C.c_void_p(t.data_ptr()), 1), "chfpe_export_state")
        return t

    def import_state(self, X, replica=0):
        if hasattr(X, "data_ptr"):
            assert X.is_cuda and X.is_contiguous() and X.numel() == self.K * self.cells
            self._ck(lib().chfpe_import_state(self._h, replica, C.c_void_p(X.data_ptr()), 1), "chfpe_import_state")
            self.stream.synchronize()
            return
        X = np.ascontiguousarray(X, dtype=np.float64)
        assert X.size == self.K * self.cells
        self._ck(lib().chfpe_import_state(self._h, replica, C.c_void_p(X.ctypes.data), 0), "chfpe_import_state")

    def export_rhs(self, replica=0):
        F = np.empty((self.K,) + self.shape)
        self._ck(lib().chfpe_export_rhs(self._h, replica, C.c_void_p(F.ctypes.data), 0), "chfpe_export_rhs")
        return F

    def export_rhs_device(self, replica=0):
        t = self._torch.empty((self.K,) + self.shape, dtype=self._torch.float64, device=self.device)
        self._ck(lib().chfpe_export_rhs(self._h, replica, C.c_void_p(t.data_ptr()), 1), "chfpe_export_rhs")
        return t

    def rk4_stage(self, stage, dt):
        """Stage 0..3 of one RK4 step (chfpe_rk4_stage); four calls = step(1, dt) without the norm guard."""
        self._ck(lib().chfpe_rk4_stage(self._h, int(stage), float(dt)), "chfpe_rk4_stage")

    def stage_input(self, stage, replica=0):
        """Torch view [K, nq_1, plane] (float64, device memory inside the workspace, no copy) of the array that RK4
        stage `stage` reads, internal layout (chfpe_stage_input): index [k, i] is the q_1 plane i of element k."""
        dev, pd = C.c_void_p(), C.c_int64()
        self._ck(lib().chfpe_stage_input(self._h, replica, int(stage), C.byref(dev), C.byref(pd)), "chfpe_stage_input")
        off = dev.value - self.workspace.data_ptr()
        n = self.K * self.cells
        flat = self.workspace[off: off + 8 * n].view(self._torch.float64)
        return flat.view(self.K, self.shape[0], pd.value)

    def profile_enable(self, on=True):
        self._ck(lib().chfpe_profile_enable(self._h, 1 if on else 0), "chfpe_profile_enable")

    def profile_read(self):
        """(summed stage-kernel milliseconds, stage launches) since the last read; synchronises the stream."""
        ms, n = C.c_double(), C.c_int64()
        self._ck(lib().chfpe_profile_read(self._h, C.byref(ms), C.byref(n)), "chfpe_profile_read")
        return ms.value, n.value

    def stage_kernel(self):
        """'generic' | 'brick' | 'compact' | 'tma': the kernel family that runs the RK stage on this handle."""
        k = C.c_int32()
        self._ck(lib().chfpe_stage_kernel(self._h, C.byref(k)), "chfpe_stage_kernel")
        return ("generic", "brick", None, "compact", "tma")[k.value]

    def stage_kernel_name(self):
        """Name of the CUDA kernel family behind stage_kernel() (for benchmark records)."""
        return {"generic": "k_stage_generic", "brick": "k_stage_brick3",
                "compact": "COMPACT6 passes: k_compact_line / k_compact_qplane (q axes) + k_compact_pbrick (p axes)",
                "tma": "k_stage_tma"}[self.stage_kernel()]

    def launch_count(self):
        n = C.c_int64()
        self._ck(lib().chfpe_launch_count(self._h, C.byref(n)), "chfpe_launch_count")
        return n.value


def hermite_workspace_bytes(cfg, batch=1):
    d, _keep = make_desc(_hermite_cfg(cfg), batch)
    n = C.c_size_t()
    rc = lib().chfpe_hermite_workspace_bytes(C.byref(d), C.byref(n))
    if rc != 0:
        raise ChfpeError("chfpe_hermite_workspace_bytes: %d %s" % (rc, lib().chfpe_hermite_last_error(None).decode()))
    return n.value


def _hermite_cfg(cfg):
    cfg = dict(cfg)                                   # the momentum range is unused by the Hermite representation
    cfg.setdefault("pmin", [-1.0] * cfg["n_modes"])
    cfg.setdefault("pmax", [1.0] * cfg["n_modes"])
    return cfg


class Hermite:
    """One chfpe_hermite_* handle (row f1: Hermite functions in the momenta, cfg["np"] = functions per mode).
    State arrays have the shape (K, kp_1..kp_M, nq_1..nq_M).  The workspace is a torch uint8 CUDA tensor."""

    def __init__(self, cfg, batch=1, device="cuda:0", stream=None, guard_bytes=0):
        import torch
        if not torch.cuda.is_available():
            raise ChfpeError("CUDA device required: the CHFPE path has no CPU fallback")
        L = lib()
        self._torch = torch
        self.device = torch.device(device)
        cfg = _hermite_cfg(cfg)
        d, keep = make_desc(cfg, batch)
        nbytes = hermite_workspace_bytes(cfg, batch)
        with torch.cuda.device(self.device):
            # guard_bytes > 0 (tests): canary bytes on both sides of the workspace, checked by guards_intact()
            self._guard = int(guard_bytes)
            self.workspace = torch.full((nbytes + 256 + 2 * self._guard,), 0xA5, dtype=torch.uint8, device=self.device) \
                if self._guard else torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            aligned = (self.workspace.data_ptr() + self._guard + 255) & ~255
            self._ws_lo = aligned - self.workspace.data_ptr()
            self._ws_hi = self._ws_lo + nbytes
            self._h = C.c_void_p()
            rc = L.chfpe_hermite_create(C.byref(d), C.c_void_p(aligned), nbytes, C.c_void_p(self.stream.cuda_stream),
                                        C.byref(self._h))
        if rc != 0:
            raise ChfpeError("chfpe_hermite_create: %d %s" % (rc, L.chfpe_hermite_last_error(None).decode()))
        self.cfg, self.batch, self.M = cfg, batch, cfg["n_modes"]
        k = C.c_int32()
        L.chfpe_hermite_num_elements(self._h, C.byref(k))
        self.K = k.value
        self.shape = (self.K,) + tuple(cfg["np"][: self.M]) + tuple(cfg["nq"][: self.M])
        self.values = int(np.prod(self.shape))

    def _ck(self, rc, what):
        if rc != 0:
            raise ChfpeError("%s: %d %s" % (what, rc, lib().chfpe_hermite_last_error(self._h).decode()))

    def guards_intact(self):
        """True if no byte outside [workspace, workspace + workspace_bytes) was written (needs guard_bytes > 0)."""
        self._torch.cuda.synchronize(self.device)
        w = self.workspace
        return bool((w[: self._ws_lo] == 0xA5).all().item() and (w[self._ws_hi:] == 0xA5).all().item())

    def close(self):
        if getattr(self, "_h", None):
            lib().chfpe_hermite_destroy(self._h)
            self._h = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def equilibrate(self, n_steps=0, dt=0.0, residual=True):
        r = C.c_double()
        self._ck(lib().chfpe_hermite_equilibrate(self._h, n_steps, dt, C.byref(r) if residual else None),
                 "chfpe_hermite_equilibrate")
        return r.value if residual else None

    def step(self, n_steps, dt):
        self._ck(lib().chfpe_hermite_step(self._h, n_steps, dt), "chfpe_hermite_step")

    def kick(self, obs):
        self._ck(lib().chfpe_hermite_kick(self._h, C.byref(obs)), "chfpe_hermite_kick")

    def expect(self, obs, element=0):
        out = np.empty(self.batch)
        self._ck(lib().chfpe_hermite_expect(self._h, element, C.byref(obs), out.ctypes.data_as(C.POINTER(C.c_double))),
                 "chfpe_hermite_expect")
        return out

    def response_1d(self, A, Cobs, n_samples, stride, dt):
        R = np.empty(n_samples)
        self._ck(lib().chfpe_hermite_response_1d(self._h, C.byref(A) if A is not None else None, C.byref(Cobs),
                                                 n_samples, stride, dt, R.ctypes.data_as(C.POINTER(C.c_double))),
                 "chfpe_hermite_response_1d")
        return R

    def response_2d(self, A, B, Cobs, t1_steps, t2_steps, dt):
        t1 = np.ascontiguousarray(t1_steps, dtype=np.int64)
        t2 = np.ascontiguousarray(t2_steps, dtype=np.int64)
        R = np.empty((len(t1), len(t2)))
        self._ck(lib().chfpe_hermite_response_2d(self._h, C.byref(A), C.byref(B), C.byref(Cobs),
                                                 t1.ctypes.data_as(C.POINTER(C.c_int64)), len(t1),
                                                 t2.ctypes.data_as(C.POINTER(C.c_int64)), len(t2), dt,
                                                 R.ctypes.data_as(C.POINTER(C.c_double))), "chfpe_hermite_response_2d")
        return R

    def response_3d(self, A, B, Cobs, D, t1_steps, t2_steps, t3_steps, dt):
        """R[k][j][l] of Eq. (17); needs batch >= 3 (batch >= 2 for a single t2 sample)."""
        ts = [np.ascontiguousarray(t, dtype=np.int64) for t in (t1_steps, t2_steps, t3_steps)]
        R = np.empty(tuple(len(t) for t in ts))
        args = []
        for t in ts:
            args += [t.ctypes.data_as(C.POINTER(C.c_int64)), len(t)]
        self._ck(lib().chfpe_hermite_response_3d(self._h, C.byref(A), C.byref(B), C.byref(Cobs), C.byref(D), *args, dt,
                                                 R.ctypes.data_as(C.POINTER(C.c_double))), "chfpe_hermite_response_3d")
        return R

    def export_state(self, replica=0):
        X = np.empty(self.shape)
        self._ck(lib().chfpe_hermite_export_state(self._h, replica, C.c_void_p(X.ctypes.data), 0),
                 "chfpe_hermite_export_state")
        return X

    def export_state_device(self, replica=0):
        t = self._torch.empty(self.shape, dtype=self._torch.float64, device=self.device)
        self._ck(lib().chfpe_hermite_export_state(self._h, replica, C.c_void_p(t.data_ptr()), 1),
                 "chfpe_hermite_export_state")
        return t

    def import_state(self, X, replica=0):
        if hasattr(X, "data_ptr"):
            assert X.is_cuda and X.is_contiguous() and X.numel() == self.values
            self._ck(lib().chfpe_hermite_import_state(self._h, replica, C.c_void_p(X.data_ptr()), 1),
                     "chfpe_hermite_import_state")
            return
        X = np.ascontiguousarray(X, dtype=np.float64)
        assert X.size == self.values
        self._ck(lib().chfpe_hermite_import_state(self._h, replica, C.c_void_p(X.ctypes.data), 0),
                 "chfpe_hermite_import_state")

    def export_rhs(self, replica=0):
        F = np.empty(self.shape)
        self._ck(lib().chfpe_hermite_export_rhs(self._h, replica, C.c_void_p(F.ctypes.data), 0),
                 "chfpe_hermite_export_rhs")
        return F

    def export_rhs_device(self, replica=0):
        t = self._torch.empty(self.shape, dtype=self._torch.float64, device=self.device)
        self._ck(lib().chfpe_hermite_export_rhs(self._h, replica, C.c_void_p(t.data_ptr()), 1),
                 "chfpe_hermite_export_rhs")
        return t

    def launch_count(self):
        n = C.c_int64()
        self._ck(lib().chfpe_hermite_launch_count(self._h, C.byref(n)), "chfpe_hermite_launch_count")
        return n.value

    def stage_kernel(self):
        """'value' | 'column' | 'patch' | 'compact' | 'tma' | 'compact_tma': the kernel family that runs the RK stage."""
        k = C.c_int32()
        self._ck(lib().chfpe_hermite_stage_kernel(self._h, C.byref(k)), "chfpe_hermite_stage_kernel")
        return ("value", "column", "patch", "compact", "tma", "compact_tma")[k.value]

    def stage_kernel_name(self):
        """Name of the CUDA kernel family behind stage_kernel() (for benchmark records)."""
        return {"value": "k_hermite_stage", "column": "k_hermite_stage_col", "patch": "k_hermite_stage_patch",
                "compact": "RK stage = k_hermite_stage<DER=false> + one k_hermite_compact_line per mode",
                "tma": "k_hermite_stage_tma<CMP=false>",
                "compact_tma": "RK stage = k_hermite_stage_tma<CMP=true> (q_2, q_3 solves inside) + k_hermite_compact_line (q_1)"}[self.stage_kernel()]


def _dev(a):
    import torch
    if not torch.cuda.is_available():
        raise ChfpeError("no CUDA device: the spectra run in CUDA kernels only (no CPU fallback)")
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()


def spectrum_1d(R, dt, omega):
    """Eq. (19): I(w) = w Im int_0^T e^{iwt} R1(t) dt (trapezoid sum) at the frequencies `omega`; numpy in / out,
    computed by chfpe_spectrum_1d on the current CUDA stream."""
    import torch
    Rd, od = _dev(np.ravel(R)), _dev(np.ravel(omega))
    out = torch.empty(od.numel(), dtype=torch.float64, device=Rd.device)
    rc = lib().chfpe_spectrum_1d(C.c_void_p(torch.cuda.current_stream().cuda_stream), C.c_void_p(Rd.data_ptr()),
                                 Rd.numel(), float(dt), C.c_void_p(od.data_ptr()), od.numel(),
                                 C.c_void_p(out.data_ptr()))
    if rc != 0:
        raise ChfpeError("chfpe_spectrum_1d failed: %d" % rc)
    return out.cpu().numpy()


def spectrum_2d(R, dt1, dt2, omega1, omega2, sign1=-1, sign2=-1):
    """Eq. (20) (default signs) / Eq. (21) (sign1 = -1, sign2 = +1): I[a][b] = Im of the double half-line transform
    of R[k][j] (rows = first delay); numpy in / out, computed by chfpe_spectrum_2d on the current CUDA stream."""
    import torch
    R = np.asarray(R, dtype=np.float64)
    if R.ndim != 2:
        raise ValueError("R must be [n1][n2]")
    Rd, o1, o2 = _dev(R), _dev(np.ravel(omega1)), _dev(np.ravel(omega2))
    scratch = torch.empty(2 * R.shape[0] * o2.numel(), dtype=torch.float64, device=Rd.device)
    out = torch.empty((o1.numel(), o2.numel()), dtype=torch.float64, device=Rd.device)
    rc = lib().chfpe_spectrum_2d(C.c_void_p(torch.cuda.current_stream().cuda_stream), C.c_void_p(Rd.data_ptr()),
                                 R.shape[0], R.shape[1], float(dt1), float(dt2), C.c_void_p(o1.data_ptr()), o1.numel(),
                                 C.c_void_p(o2.data_ptr()), o2.numel(), int(sign1), int(sign2),
                                 C.c_void_p(scratch.data_ptr()), C.c_void_p(out.data_ptr()))
    if rc != 0:
        raise ChfpeError("chfpe_spectrum_2d failed: %d" % rc)
    return out.cpu().numpy()


SPECTRUM_STATIC_MAX = 65536   # CHFPE_SPECTRUM_STATIC_MAX of include/chfpe.h: n1 * n_omega2 of chfpe_spectrum_2d_static


def spectrum_2d_static_device(Rd, dt1, dt2, o1, o2, out, sign1=-1, sign2=-1):
    """chfpe_spectrum_2d_static on device tensors (float64, contiguous), result written into `out`
    [n_omega1][n_omega2]: the variant that allocates nothing (its scratch is a static device array inside the
    library).  Calls that overlap on the GPU race on that array; successive calls on one stream are safe."""
    import torch
    rc = lib().chfpe_spectrum_2d_static(C.c_void_p(torch.cuda.current_stream().cuda_stream), C.c_void_p(Rd.data_ptr()),
                                        Rd.shape[0], Rd.shape[1], float(dt1), float(dt2), C.c_void_p(o1.data_ptr()),
                                        o1.numel(), C.c_void_p(o2.data_ptr()), o2.numel(), int(sign1), int(sign2),
                                        C.c_void_p(out.data_ptr()))
    if rc != 0:
        raise ChfpeError("chfpe_spectrum_2d_static failed: %d" % rc)
    return out
