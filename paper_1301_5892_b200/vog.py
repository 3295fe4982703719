"""Thin ctypes binding of libvog (include/vog.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels; there is no CPU or PyTorch fallback --
if libvog.so is missing or cannot be loaded this module raises.  PyTorch is used by callers only
for device memory and streams: any object with a ``data_ptr()`` (a torch tensor) or a plain int
device address can be passed where the C API takes a ``*_dev`` pointer.
"""
import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libvog.so")

OK, EINVAL, ENOMEM, ECUDA, EUNSUPPORTED, ETOOLARGE = 0, -1, -2, -3, -4, -5
NOALLOC_MAX_NX = 4096
LAGRANGE, BSPLINE = 0, 1
SPLIT_XVX, SPLIT_VXV = 0, 1

EXPORTS = ("vog_plan", "vog_destroy", "vog_advect_x", "vog_advect_v", "vog_field", "vog_step",
           "vog_get_field", "vog_shift_x", "vog_shift_v", "vog_shift_v_to", "vog_run", "vog_run_host",
           "vog_run_host_async", "vog_launch_count", "vog_strerror", "vog_plan_tune", "vog_reset", "vog_diagnostics",
           "vog_shift_x_f64", "vog_shift_v_f64", "vog_advect_x_f64", "vog_advect_v_f64", "vog_field_f64",
           "vog_get_field_f64", "vog_step_f64", "vog_field_noalloc")


class vog_feq_t(ctypes.Structure):
    _fields_ = [("n", ctypes.c_int), ("amp", ctypes.c_double * 4), ("mu", ctypes.c_double * 4),
                ("c", ctypes.c_double * 4)]


class vog_params_t(ctypes.Structure):
    _fields_ = [("Nx", ctypes.c_int), ("Nv", ctypes.c_int), ("L", ctypes.c_double),
                ("vmin", ctypes.c_double), ("vmax", ctypes.c_double), ("kind", ctypes.c_int),
                ("order", ctypes.c_int), ("feq", vog_feq_t), ("split", ctypes.c_int)]


class VogError(RuntimeError):
    def __init__(self, status, where):
        self.status = status
        super().__init__("%s: %s (%d)" % (where, strerror(status), status))


_lib = None


def lib():
    """Load libvog.so; fail loudly if the CUDA extension is missing (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libvog.so not built: run `python -m paper_1301_5892_b200.build` "
                              "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        vp = ctypes.c_void_p
        L.vog_plan.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(vog_params_t), vp]
        L.vog_destroy.argtypes = [vp]
        L.vog_advect_x.argtypes = [vp, vp, ctypes.c_double]
        L.vog_advect_v.argtypes = [vp, vp, vp, ctypes.c_double]
        L.vog_field.argtypes = [vp, vp, vp]
        L.vog_step.argtypes = [vp, vp, ctypes.c_double, vp]
        L.vog_get_field.argtypes = [vp, vp]
        L.vog_shift_x.argtypes = [vp, vp, vp]
        L.vog_shift_v.argtypes = [vp, vp, vp]
        L.vog_shift_v_to.argtypes = [vp, vp, vp, vp]
        L.vog_run.argtypes = [vp, vp, ctypes.c_double, ctypes.c_int, vp, ctypes.c_int, vp]
        L.vog_run_host.argtypes = [vp, vp, ctypes.c_double, ctypes.c_int, vp, vp]
        L.vog_run_host_async.argtypes = [vp, vp, ctypes.c_double, ctypes.c_int, vp, vp]
        L.vog_launch_count.argtypes = [vp]
        L.vog_launch_count.restype = ctypes.c_longlong
        L.vog_strerror.argtypes = [ctypes.c_int]
        L.vog_strerror.restype = ctypes.c_char_p
        L.vog_plan_tune.argtypes = [vp, ctypes.c_int, ctypes.c_int]
        L.vog_reset.argtypes = [vp]
        L.vog_diagnostics.argtypes = [vp, vp, vp]
        L.vog_shift_x_f64.argtypes = [vp, vp, vp]
        L.vog_shift_v_f64.argtypes = [vp, vp, vp]
        L.vog_advect_x_f64.argtypes = [vp, vp, ctypes.c_double]
        L.vog_advect_v_f64.argtypes = [vp, vp, vp, ctypes.c_double]
        L.vog_field_f64.argtypes = [vp, vp, vp]
        L.vog_get_field_f64.argtypes = [vp, vp]
        L.vog_step_f64.argtypes = [vp, vp, ctypes.c_double, vp]
        L.vog_field_noalloc.argtypes = [vp, ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double,
                                        ctypes.c_double, vp, vp]
        for name in EXPORTS:
            if name not in ("vog_launch_count", "vog_strerror"):
                getattr(L, name).restype = ctypes.c_int
        _lib = L
    return _lib


def strerror(status):
    return lib().vog_strerror(int(status)).decode()


def _ptr(x):
    if x is None:
        return None
    if hasattr(x, "data_ptr"):
        return ctypes.c_void_p(x.data_ptr())
    if hasattr(x, "ctypes"):            # numpy array: host pointer (vog_run_host only)
        return ctypes.c_void_p(x.ctypes.data)
    return ctypes.c_void_p(int(x))


def make_params(Nx, Nv, L, vmin, vmax, kind=LAGRANGE, order=17, feq=(), split=SPLIT_XVX):
    p = vog_params_t()
    p.Nx, p.Nv, p.L, p.vmin, p.vmax = int(Nx), int(Nv), float(L), float(vmin), float(vmax)
    p.kind, p.order, p.split = int(kind), int(order), int(split)
    p.feq.n = len(feq)
    for g, (amp, mu, c) in enumerate(feq):
        if g < 4:
            p.feq.amp[g], p.feq.mu[g], p.feq.c[g] = float(amp), float(mu), float(c)
    return p


def field_noalloc(f, Nx, Nv, L, vmin, vmax, E, stream=None):
    """vog_field_noalloc (include/vog.h): the self-consistent field without a plan and without any allocation; scratch in
    a fixed device array shared by all calls (Nx <= NOALLOC_MAX_NX; overlapping calls race).  Returns nothing; raises
    VogError (ETOOLARGE beyond the limit)."""
    sp = None if stream is None else ctypes.c_void_p(int(getattr(stream, "cuda_stream", stream)))
    rc = lib().vog_field_noalloc(_ptr(f), int(Nx), int(Nv), float(L), float(vmin), float(vmax), _ptr(E), sp)
    if rc != OK:
        raise VogError(rc, "vog_field_noalloc")


class Plan:
    """vog_plan_t with the same-named calls as methods.  `stream` is a raw cudaStream_t (int) or
    a torch.cuda.Stream; None = the legacy default stream."""

    def __init__(self, Nx, Nv, L, vmin, vmax, kind=LAGRANGE, order=17, feq=(), split=SPLIT_XVX, stream=None):
        self.params = make_params(Nx, Nv, L, vmin, vmax, kind, order, feq, split)
        self.Nx, self.Nv = int(Nx), int(Nv)
        if stream is not None and hasattr(stream, "cuda_stream"):
            stream = stream.cuda_stream
        h = ctypes.c_void_p()
        rc = lib().vog_plan(ctypes.byref(h), ctypes.byref(self.params), ctypes.c_void_p(stream or 0))
        if rc != OK:
            raise VogError(rc, "vog_plan")
        self._h = h

    @classmethod
    def from_config(cls, cfg, stream=None, **over):
        kw = dict(Nx=cfg.Nx, Nv=cfg.Nv, L=cfg.L, vmin=cfg.vmin, vmax=cfg.vmax, kind=cfg.kind,
                  order=cfg.order, feq=tuple(cfg.feq), split=cfg.split, stream=stream)
        kw.update(over)
        return cls(**kw)

    def _ck(self, rc, where):
        if rc != OK:
            raise VogError(rc, where)

    def advect_x(self, f, dt):
        self._ck(lib().vog_advect_x(self._h, _ptr(f), float(dt)), "vog_advect_x")

    def advect_v(self, f, E, dt):
        self._ck(lib().vog_advect_v(self._h, _ptr(f), _ptr(E), float(dt)), "vog_advect_v")

    def field(self, f, E):
        self._ck(lib().vog_field(self._h, _ptr(f), _ptr(E)), "vog_field")

    def step(self, f, dt, E_ext=None):
        self._ck(lib().vog_step(self._h, _ptr(f), float(dt), _ptr(E_ext)), "vog_step")

    def diagnostics(self, f, diag):
        self._ck(lib().vog_diagnostics(self._h, _ptr(f), _ptr(diag)), "vog_diagnostics")

    def get_field(self, E):
        self._ck(lib().vog_get_field(self._h, _ptr(E)), "vog_get_field")

    def shift_x(self, f, beta):
        self._ck(lib().vog_shift_x(self._h, _ptr(f), _ptr(beta)), "vog_shift_x")

    def shift_v(self, f, beta):
        self._ck(lib().vog_shift_v(self._h, _ptr(f), _ptr(beta)), "vog_shift_v")

    def shift_v_to(self, src, dst, beta):
        self._ck(lib().vog_shift_v_to(self._h, _ptr(src), _ptr(dst), _ptr(beta)), "vog_shift_v_to")

    # double-precision mode (include/vog.h, NEXT-2): the same calls on fp64 arrays
    def shift_x_f64(self, f, beta):
        self._ck(lib().vog_shift_x_f64(self._h, _ptr(f), _ptr(beta)), "vog_shift_x_f64")

    def shift_v_f64(self, f, beta):
        self._ck(lib().vog_shift_v_f64(self._h, _ptr(f), _ptr(beta)), "vog_shift_v_f64")

    def advect_x_f64(self, f, dt):
        self._ck(lib().vog_advect_x_f64(self._h, _ptr(f), float(dt)), "vog_advect_x_f64")

    def advect_v_f64(self, f, E, dt):
        self._ck(lib().vog_advect_v_f64(self._h, _ptr(f), _ptr(E), float(dt)), "vog_advect_v_f64")

    def field_f64(self, f, E):
        self._ck(lib().vog_field_f64(self._h, _ptr(f), _ptr(E)), "vog_field_f64")

    def get_field_f64(self, E):
        self._ck(lib().vog_get_field_f64(self._h, _ptr(E)), "vog_get_field_f64")

    def step_f64(self, f, dt, E_ext=None):
        self._ck(lib().vog_step_f64(self._h, _ptr(f), float(dt), _ptr(E_ext)), "vog_step_f64")

    def run(self, f, dt, nsteps, E_ext_seq=None, merge=False, energy=None):
        self._ck(lib().vog_run(self._h, _ptr(f), float(dt), int(nsteps), _ptr(E_ext_seq), 1 if merge else 0,
                               _ptr(energy)), "vog_run")

    def run_host(self, f_host, dt, nsteps, E_ext_host=None, E_host=None):
        self._ck(lib().vog_run_host(self._h, _ptr(f_host), float(dt), int(nsteps), _ptr(E_ext_host),
                                    _ptr(E_host)), "vog_run_host")

    def run_host_async(self, f_host, dt, nsteps, E_ext_host=None, E_host=None):
        self._ck(lib().vog_run_host_async(self._h, _ptr(f_host), float(dt), int(nsteps), _ptr(E_ext_host),
                                          _ptr(E_host)), "vog_run_host_async")

    def launch_count(self):
        return int(lib().vog_launch_count(self._h))

    def reset(self):
        self._ck(lib().vog_reset(self._h), "vog_reset")

    def tune(self, which, value):
        self._ck(lib().vog_plan_tune(self._h, int(which), int(value)), "vog_plan_tune")

    def destroy(self):
        if self._h is not None and self._h.value:
            lib().vog_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
