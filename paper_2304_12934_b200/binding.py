"""Thin ctypes binding of include/tc.h -- argument marshalling only; every step runs in libtc.so's CUDA kernels.

Accepts torch tensors (CUDA, or CPU -- pinned or not) and numpy arrays (host).  There is no CPU fallback:
a missing library raises at import of this module.
"""
import ctypes, os
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.environ.get("TC_LIBTC", os.path.join(_HERE, "libtc.so"))
if not os.path.exists(_LIB_PATH):
    raise ImportError("libtc.so not built: run `python -m paper_2304_12934_b200.build` (no CPU fallback exists)")
lib = ctypes.CDLL(_LIB_PATH)

TC_OK, TC_EINVAL, TC_ENOMEM, TC_ECUDA, TC_EUNSUPPORTED = range(5)


class tc_geom(ctypes.Structure):
    _fields_ = [("n", ctypes.c_int), ("n_det", ctypes.c_int), ("n_angles", ctypes.c_int),
                ("angles", ctypes.POINTER(ctypes.c_float)), ("center", ctypes.c_float),
                ("oversamp", ctypes.c_float), ("kb_width", ctypes.c_int)]


class tc_prior(ctypes.Structure):
    _fields_ = [("p", ctypes.c_float), ("sigma", ctypes.c_float), ("c", ctypes.c_float),
                ("lam", ctypes.c_float), ("L", ctypes.c_float), ("nonneg", ctypes.c_int), ("grad_restart", ctypes.c_int),
                ("neighbours", ctypes.c_int), ("mm_step", ctypes.c_int)]


class tc_iter_log(ctypes.Structure):
    _fields_ = [("F", ctypes.c_double), ("data", ctypes.c_double), ("prior", ctypes.c_double),
                ("margin", ctypes.c_double), ("dot", ctypes.c_double), ("beta", ctypes.c_float), ("accepted", ctypes.c_int),
                ("restarted", ctypes.c_int), ("alpha", ctypes.c_float), ("ms", ctypes.c_float)]


class tc_sched_stats(ctypes.Structure):
    _fields_ = [("h2d_s", ctypes.c_double), ("compute_s", ctypes.c_double), ("d2h_s", ctypes.c_double),
                ("wall_s", ctypes.c_double), ("overlap", ctypes.c_double), ("h2d_bytes", ctypes.c_longlong),
                ("d2h_bytes", ctypes.c_longlong), ("n_slabs", ctypes.c_int), ("setup_s", ctypes.c_double), ("handover_s", ctypes.c_double)]


EXCHANGE_FN = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p)
ALLREDUCE_FN = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.POINTER(ctypes.c_double), ctypes.c_int)


class tc_comm(ctypes.Structure):
    _fields_ = [("ctx", ctypes.c_void_p), ("exchange", EXCHANGE_FN), ("allreduce", ALLREDUCE_FN),
                ("send_down", ctypes.c_void_p), ("send_up", ctypes.c_void_p), ("recv_down", ctypes.c_void_p), ("recv_up", ctypes.c_void_p)]


_vp, _ci = ctypes.c_void_p, ctypes.c_int
lib.tc_plan_create.argtypes = [ctypes.POINTER(tc_geom), _ci, ctypes.POINTER(_vp)]
lib.tc_plan_destroy.argtypes = [_vp]
lib.tc_radon.argtypes = [_vp, _vp, _ci, _vp, _vp]
lib.tc_backproject.argtypes = [_vp, _vp, _ci, _vp, _vp]
lib.tc_radon_static.argtypes = [_vp, _vp, _ci, _vp, _vp]
lib.tc_fbp.argtypes = [_vp, _vp, _ci, _ci, _vp, _vp]
lib.tc_mbir.argtypes = [_vp, _vp, _ci, ctypes.POINTER(tc_prior), _ci, _vp, ctypes.POINTER(tc_iter_log), _vp]
lib.tc_mbir_sharded.argtypes = [_vp, _vp, _ci, ctypes.POINTER(tc_prior), _ci, _vp, ctypes.POINTER(tc_iter_log), ctypes.POINTER(tc_comm), _vp]
lib.tc_power_iteration.argtypes = [_vp, _ci, ctypes.POINTER(ctypes.c_double)]
lib.tc_stage_fine_grid.argtypes = [_vp, _vp, _vp, _vp]
lib.tc_stage_gather.argtypes = [_vp, _vp, _vp]
lib.tc_stage_spread.argtypes = [_vp, _vp, _vp]
lib.tc_prior_eval.argtypes = [_vp, _ci, _ci, ctypes.POINTER(tc_prior), _vp, ctypes.POINTER(ctypes.c_double)]
lib.tc_radon1.argtypes = [_vp, _ci, _ci, ctypes.POINTER(ctypes.c_float), _ci, _ci, ctypes.c_float, _vp]
lib.tc_launch_count.argtypes = [_ci]
lib.tc_launch_count.restype = ctypes.c_longlong
lib.tc_last_sched_stats.argtypes = [_vp, ctypes.POINTER(tc_sched_stats)]
lib.tc_profile.argtypes = [_vp, _ci]
lib.tc_profile_read.argtypes = [_vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_longlong)]
lib.tc_preprocess.argtypes = [_vp, _vp, _vp, _ci, _ci, _ci, ctypes.c_float, _vp, _vp]
lib.tc_host_alloc.argtypes = [ctypes.c_size_t, ctypes.POINTER(_vp)]
lib.tc_host_free.argtypes = [_vp]
lib.tc_last_error.restype = ctypes.c_char_p
for _f in ("tc_plan_create", "tc_plan_destroy", "tc_radon", "tc_backproject", "tc_fbp", "tc_mbir", "tc_power_iteration",
           "tc_prior_eval", "tc_radon1", "tc_last_sched_stats", "tc_profile", "tc_profile_read", "tc_host_alloc", "tc_host_free", "tc_preprocess", "tc_mbir_sharded"):
    getattr(lib, _f).restype = _ci


class TcError(RuntimeError):
    def __init__(self, status):
        self.status = status
        super().__init__("tc status %d: %s" % (status, lib.tc_last_error().decode()))


def _check(st):
    if st != TC_OK:
        raise TcError(st)


def _ptr(a):
    """data pointer of a float32 C-contiguous torch tensor or numpy array."""
    if isinstance(a, np.ndarray):
        assert a.dtype == np.float32 and a.flags.c_contiguous
        return a.ctypes.data
    assert a.dtype.__str__() == "torch.float32" and a.is_contiguous()
    return a.data_ptr()


def _stream(a):
    if isinstance(a, np.ndarray) or not a.is_cuda:
        return None
    import torch
    return torch.cuda.current_stream(a.device).cuda_stream


def _like(a, shape):
    if isinstance(a, np.ndarray):
        return np.empty(shape, dtype=np.float32)
    import torch
    return torch.empty(shape, dtype=torch.float32, device=a.device, pin_memory=(not a.is_cuda and a.is_pinned()))


def prior_params(p=1.2, sigma=1 / 0.7, c=1e-4, lam=1.0, L=0.0, nonneg=False, grad_restart=False, neighbours=26, mm_step=False):
    return tc_prior(p, sigma, c, lam, L, 1 if nonneg else 0, 1 if grad_restart else 0, int(neighbours), 1 if mm_step else 0)


class Plan:
    """tc_plan_create / tc_plan_destroy; methods are the C calls of the same names."""

    def __init__(self, n, n_det, angles, center=-1.0, max_slab_slices=0, kb_width=6):
        ang = np.ascontiguousarray(np.asarray(angles, dtype=np.float32))
        self.n, self.n_det, self.n_angles = int(n), int(n_det), int(ang.size)
        g = tc_geom(self.n, self.n_det, self.n_angles, ang.ctypes.data_as(ctypes.POINTER(ctypes.c_float)),
                    float(center), 2.0, int(kb_width))
        self._h = _vp()
        _check(lib.tc_plan_create(ctypes.byref(g), int(max_slab_slices), ctypes.byref(self._h)))

    def close(self):
        if getattr(self, "_h", None) and lib is not None:
            lib.tc_plan_destroy(self._h)
            self._h = None

    __del__ = close

    def radon(self, volume, out=None):
        S = volume.shape[0]
        assert tuple(volume.shape) == (S, self.n, self.n)
        out = _like(volume, (S, self.n_angles, self.n_det)) if out is None else out
        _check(lib.tc_radon(self._h, _ptr(volume), S, _ptr(out), _stream(volume)))
        return out

    def radon_static(self, volume, out):
        """tc_radon_static: device tensors only, `out` preallocated by the caller (nothing is allocated on the way)."""
        _check(lib.tc_radon_static(self._h, _ptr(volume), int(volume.shape[0]), _ptr(out), _stream(volume)))
        return out

    def backproject(self, sinogram, out=None):
        S = sinogram.shape[0]
        assert tuple(sinogram.shape) == (S, self.n_angles, self.n_det)
        out = _like(sinogram, (S, self.n, self.n)) if out is None else out
        _check(lib.tc_backproject(self._h, _ptr(sinogram), S, _ptr(out), _stream(sinogram)))
        return out

    def fbp(self, sinogram, filter="ramp", out=None):
        S = sinogram.shape[0]
        assert tuple(sinogram.shape) == (S, self.n_angles, self.n_det)
        out = _like(sinogram, (S, self.n, self.n)) if out is None else out
        _check(lib.tc_fbp(self._h, _ptr(sinogram), S, {"ramp": 0, "hann": 1, "shepp-logan": 2, "butterworth": 3}[filter], _ptr(out), _stream(sinogram)))
        return out

    def mbir(self, sinogram, prior, iters, out=None):
        S = sinogram.shape[0]
        assert tuple(sinogram.shape) == (S, self.n_angles, self.n_det)
        out = _like(sinogram, (S, self.n, self.n)) if out is None else out
        log = (tc_iter_log * max(iters, 1))()
        _check(lib.tc_mbir(self._h, _ptr(sinogram), S, ctypes.byref(prior), int(iters), _ptr(out), log, _stream(sinogram)))
        recs = [dict(F=l.F, data=l.data, prior=l.prior, margin=l.margin, dot=l.dot, beta=l.beta, accepted=l.accepted, restarted=l.restarted, alpha=l.alpha, ms=l.ms)
                for l in log[:iters]]
        return out, recs

    def mbir_sharded(self, sinogram, prior, iters, comm, out=None):
        """tc_mbir_sharded on this rank's slices; `comm` has the attributes of shard.TorchComm (exchange(), allreduce(list) -> list,
        send_down / send_up / recv_down / recv_up: device tensors or None)."""
        S = sinogram.shape[0]
        assert sinogram.is_cuda and tuple(sinogram.shape) == (S, self.n_angles, self.n_det)
        out = _like(sinogram, (S, self.n, self.n)) if out is None else out
        log = (tc_iter_log * max(iters, 1))()
        errs = []

        def _ex(_ctx):
            try:
                comm.exchange(); return 0
            except Exception as e:                                   # an exception must not unwind through the C frames
                errs.append(e); return 1

        def _ar(_ctx, vals, n):
            try:
                res = comm.allreduce([vals[i] for i in range(n)])
                for i in range(n):
                    vals[i] = res[i]
                return 0
            except Exception as e:
                errs.append(e); return 1
        ptr = lambda t: None if t is None else t.data_ptr()
        c = tc_comm(None, EXCHANGE_FN(_ex), ALLREDUCE_FN(_ar), ptr(comm.send_down), ptr(comm.send_up), ptr(comm.recv_down), ptr(comm.recv_up))
        st = lib.tc_mbir_sharded(self._h, _ptr(sinogram), S, ctypes.byref(prior), int(iters), _ptr(out), log, ctypes.byref(c), _stream(sinogram))
        if errs:
            raise errs[0]
        _check(st)
        recs = [dict(F=l.F, data=l.data, prior=l.prior, margin=l.margin, dot=l.dot, beta=l.beta, accepted=l.accepted, restarted=l.restarted, alpha=l.alpha, ms=l.ms)
                for l in log[:iters]]
        return out, recs

    def power_iteration(self, iters=10):
        v = ctypes.c_double()
        _check(lib.tc_power_iteration(self._h, int(iters), ctypes.byref(v)))
        return v.value

    STAGES = ("fwd_rows", "fwd_cols", "fwd_gather", "adj_radial", "adj_spread", "adj_cols", "adj_rows", "fwd_radial")

    def profile(self, enable=True):
        _check(lib.tc_profile(self._h, 1 if enable else 0))

    def profile_read(self):
        ms = (ctypes.c_double * 8)(); cnt = (ctypes.c_longlong * 8)()
        _check(lib.tc_profile_read(self._h, ms, cnt))
        return {k: (ms[i], cnt[i]) for i, k in enumerate(self.STAGES)}

    # stage hooks (per-stage unit tests): numpy host arrays, complex64 in natural order
    def stage_fine_grid(self, re, im=None):
        re = np.ascontiguousarray(re, dtype=np.float32)
        im = None if im is None else np.ascontiguousarray(im, dtype=np.float32)
        out = np.empty((2 * self.n, 2 * self.n), dtype=np.complex64)
        _check(lib.tc_stage_fine_grid(self._h, re.ctypes.data, None if im is None else im.ctypes.data, out.ctypes.data))
        return out

    def stage_gather(self, grid):
        grid = np.ascontiguousarray(grid, dtype=np.complex64)
        out = np.empty((self.n_angles, self.n_det), dtype=np.complex64)
        _check(lib.tc_stage_gather(self._h, grid.ctypes.data, out.ctypes.data))
        return out

    def stage_spread(self, cpol):
        cpol = np.ascontiguousarray(cpol, dtype=np.complex64)
        out = np.empty((2 * self.n, 2 * self.n), dtype=np.complex64)
        _check(lib.tc_stage_spread(self._h, cpol.ctypes.data, out.ctypes.data))
        return out

    def sched_stats(self):
        s = tc_sched_stats()
        _check(lib.tc_last_sched_stats(self._h, ctypes.byref(s)))
        return {k: getattr(s, k) for k, _ in tc_sched_stats._fields_}


def prior_eval(volume, prior, want_grad=True):
    S, n, _ = volume.shape
    grad = _like(volume, tuple(volume.shape)) if want_grad else None
    val = ctypes.c_double()
    _check(lib.tc_prior_eval(_ptr(volume), S, n, ctypes.byref(prior), _ptr(grad) if want_grad else None, ctypes.byref(val)))
    return val.value, grad


def preprocess(proj, flat=None, dark=None, floor=1e-6):
    """tc_preprocess: proj (Na, S, Nd) intensities -> sinogram (S, Na, Nd) line integrals."""
    na, S, nd = proj.shape
    out = _like(proj, (S, na, nd))
    _check(lib.tc_preprocess(_ptr(proj), None if flat is None else _ptr(flat), None if dark is None else _ptr(dark), na, S, nd,
                             float(floor), _ptr(out), _stream(proj)))
    return out


def radon1(volume, angles, n_det, center):
    ang = np.ascontiguousarray(np.asarray(angles, dtype=np.float32))
    S, n, _ = volume.shape
    out = _like(volume, (S, ang.size, n_det))
    _check(lib.tc_radon1(_ptr(volume), S, n, ang.ctypes.data_as(ctypes.POINTER(ctypes.c_float)), ang.size, n_det, float(center), _ptr(out)))
    return out


class PinnedArray:
    """float32 numpy array on tc_host_alloc memory (exact size, page-locked); call free() when done with every view of it."""

    def __init__(self, shape):
        n = int(np.prod(shape))
        self._p = _vp()
        _check(lib.tc_host_alloc(n * 4, ctypes.byref(self._p)))
        self.array = np.frombuffer((ctypes.c_float * n).from_address(self._p.value), dtype=np.float32).reshape(shape)

    def free(self):
        if self._p:
            self.array = None
            lib.tc_host_free(self._p)
            self._p = None


def launch_count(reset=False):
    return lib.tc_launch_count(1 if reset else 0)
