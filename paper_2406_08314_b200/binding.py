"""Thin Python binding of libmsd_b200.so (include/msd.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of the library; PyTorch is used for device
memory and streams.  There is no CPU fallback: if the shared library is missing or cannot be
loaded, importing a symbol from here raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmsd_b200.so")

MSD_OK, MSD_EINVAL, MSD_ENOMEM, MSD_ECUDA, MSD_EUNSUPPORTED = 0, -1, -2, -3, -4
_CODES = {MSD_EINVAL: "MSD_EINVAL", MSD_ENOMEM: "MSD_ENOMEM", MSD_ECUDA: "MSD_ECUDA",
          MSD_EUNSUPPORTED: "MSD_EUNSUPPORTED"}

EXPORTS = ["msd_setup", "msd_setup_sharded", "msd_set_allreduce", "msd_setup_from_occ", "msd_overlap", "msd_force_bias", "msd_local_energy", "msd_greens",
           "msd_overlap_host", "msd_force_bias_host", "msd_local_energy_host",
           "msd_force_bias_energy", "msd_force_bias_energy_host",
           "msd_propagator_setup", "msd_propagate",
           "msd_get_info", "msd_get_packed", "msd_set_workspace_limit", "msd_set_option", "msd_launch_count",
           "msd_set_profiling", "msd_get_phase_ms", "msd_destroy", "msd_last_error",
           "msd_noalloc_setup", "msd_overlap_noalloc", "msd_force_bias_overlap", "msd_reference_cond"]
MSD_NOALLOC_SCRATCH_BYTES = 4 * 1024 * 1024
MSD_OPT_NO_SMEM_TILES = 1
MSD_OPT_NO_FUSED_S7 = 2
MSD_OPT_NO_3M = 3
MSD_OPT_COOP_MIN_ELEMS = 4
MSD_OPT_3M_MAX_COND = 5


class MSDError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__("%s (%d): %s" % (_CODES.get(code, "error"), code, msg))
        self.code = code


_lib = None


def load_library() -> C.CDLL:
    """Load libmsd_b200.so (built in-tree by paper_2406_08314_b200/build.py).  Fails loudly if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError("libmsd_b200.so not found at %s: run `python -m paper_2406_08314_b200.build` "
                          "(or __graft_entry__.build()); there is no CPU fallback" % LIB_PATH)
    lib = C.CDLL(LIB_PATH)
    vp, i32, i64, dbl = C.c_void_p, C.c_int, C.c_int64, C.c_double
    lib.msd_setup.restype = i32
    lib.msd_setup.argtypes = [C.POINTER(vp), i32, i32, i32, i32, i64, vp, vp, dbl, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.msd_setup_sharded.restype = i32
    lib.msd_setup_sharded.argtypes = [C.POINTER(vp), i32, i32, i32, i32, i64, vp, vp, dbl, vp, vp, vp, vp, vp, vp, vp, vp, vp,
                                      i32, i32, vp]
    lib.msd_set_allreduce.restype = i32
    lib.msd_set_allreduce.argtypes = [vp, vp, vp]
    lib.msd_setup_from_occ.restype = i32
    lib.msd_setup_from_occ.argtypes = [C.POINTER(vp), i32, i32, i32, i32, i64, vp, vp, dbl, vp, vp, vp, vp]
    for name in ("msd_overlap", "msd_force_bias", "msd_local_energy", "msd_greens", "msd_force_bias_energy",
                 "msd_overlap_host", "msd_force_bias_host", "msd_local_energy_host", "msd_force_bias_energy_host",
                 "msd_overlap_noalloc"):
        f = getattr(lib, name)
        f.restype = i32
        f.argtypes = [vp, i64, vp, vp, vp, vp, vp]
    lib.msd_reference_cond.restype = i32
    lib.msd_reference_cond.argtypes = [vp, i64, vp, vp, vp, vp]
    lib.msd_force_bias_overlap.restype = i32
    lib.msd_force_bias_overlap.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp]
    lib.msd_noalloc_setup.restype = i32
    lib.msd_noalloc_setup.argtypes = [vp, vp]
    lib.msd_propagator_setup.restype = i32
    lib.msd_propagator_setup.argtypes = [vp, dbl, i32, vp, vp, vp]
    lib.msd_propagate.restype = i32
    lib.msd_propagate.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp, vp]
    lib.msd_get_info.restype = i32
    lib.msd_get_info.argtypes = [vp, vp]
    lib.msd_get_packed.restype = i32
    lib.msd_get_packed.argtypes = [vp, vp, vp, vp, vp]
    lib.msd_set_workspace_limit.restype = i32
    lib.msd_set_workspace_limit.argtypes = [vp, i64]
    lib.msd_launch_count.restype = i64
    lib.msd_launch_count.argtypes = [vp]
    lib.msd_set_profiling.restype = i32
    lib.msd_set_profiling.argtypes = [vp, i32]
    lib.msd_get_phase_ms.restype = i32
    lib.msd_get_phase_ms.argtypes = [vp, vp, i32]
    lib.msd_set_option.restype = i32
    lib.msd_set_option.argtypes = [vp, i32, i64]
    lib.msd_destroy.restype = None
    lib.msd_destroy.argtypes = [vp]
    lib.msd_last_error.restype = C.c_char_p
    lib.msd_last_error.argtypes = [vp]
    _lib = lib
    return lib


def _np(a, dtype):
    return np.ascontiguousarray(a, dtype=dtype)


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _stream_ptr(stream) -> Optional[int]:
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    if isinstance(stream, int):
        return stream or None
    return stream.cuda_stream or None


class MSDTrial:
    """Owns an msd_ctx.  Methods mirror the C entry points of include/msd.h."""

    def __init__(self, handle: int, N: int, n_alpha: int, n_beta: int, n_chol: int, n_det: int):
        self._h = C.c_void_p(handle)
        self.N, self.n_alpha, self.n_beta, self.n_chol, self.n_det = N, n_alpha, n_beta, n_chol, n_det

    # -- lifetime ------------------------------------------------------------------------------
    def close(self):
        if self._h:
            load_library().msd_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc: int):
        err = getattr(self, "_allreduce_error", None)
        if err is not None:
            self._allreduce_error = None
            raise err
        if rc != MSD_OK:
            msg = load_library().msd_last_error(self._h)
            raise MSDError(rc, msg.decode() if msg else "")

    # -- hot calls -----------------------------------------------------------------------------
    def _walkers(self, phi_a, phi_b):
        import torch
        for phi, n in ((phi_a, self.n_alpha), (phi_b, self.n_beta)):
            if not (isinstance(phi, torch.Tensor) and phi.is_cuda and phi.dtype == torch.complex128
                    and phi.is_contiguous() and phi.dim() == 3 and phi.shape[1] == self.N and phi.shape[2] == n):
                raise ValueError("walkers must be contiguous CUDA complex128 tensors [n_w][N][n_sigma]")
        if phi_a.shape[0] != phi_b.shape[0]:
            raise ValueError("phi_a and phi_b disagree on n_w")
        return int(phi_a.shape[0])

    def _call(self, fn, phi_a, phi_b, out, flags, stream):
        import torch
        nw = self._walkers(phi_a, phi_b)
        if flags is not None and not (isinstance(flags, torch.Tensor) and flags.is_cuda and flags.dtype == torch.int32
                                      and flags.is_contiguous() and flags.numel() >= nw
                                      and flags.device == phi_a.device):
            raise ValueError("flags must be a contiguous CUDA int32 tensor of at least n_w elements on the walkers' device")
        shape = self._out_shape(fn, nw)
        if not (isinstance(out, torch.Tensor) and out.is_cuda and out.device == phi_a.device
                and out.dtype == torch.complex128 and out.is_contiguous() and tuple(out.shape) == shape):
            raise ValueError("out must be a contiguous CUDA complex128 tensor of shape %s on the walkers' device" % (shape,))
        rc = fn(self._h, nw, phi_a.data_ptr(), phi_b.data_ptr(), out.data_ptr(),
                flags.data_ptr() if flags is not None else None, _stream_ptr(stream))
        self._check(rc)
        return out

    def _out_shape(self, fn, nw):
        """Result shape of a hot call (include/msd.h), by entry-point name."""
        name = fn.__name__.replace("_host", "")
        return {"msd_overlap": (nw,), "msd_overlap_noalloc": (nw,), "msd_force_bias": (nw, self.n_chol), "msd_local_energy": (nw, 3),
                "msd_force_bias_energy": (nw, self.n_chol + 3), "msd_greens": (nw, 2, self.N, self.N)}[name]

    def overlap(self, phi_a, phi_b, out=None, flags=None, stream=None):
        import torch
        nw = self._walkers(phi_a, phi_b)
        out = torch.empty(nw, dtype=torch.complex128, device=phi_a.device) if out is None else out
        return self._call(load_library().msd_overlap, phi_a, phi_b, out, flags, stream)

    def noalloc_setup(self, stream=None):
        """Set-up for overlap_noalloc (include/msd.h: msd_noalloc_setup): once per context, may allocate."""
        self._check(load_library().msd_noalloc_setup(self._h, _stream_ptr(stream)))

    def overlap_noalloc(self, phi_a, phi_b, out, flags=None, stream=None):
        """msd_overlap_noalloc: the overlap with the workspace in the library's static device array; `out` (and `flags`)
        are the caller's -- nothing is allocated here either.  Batches beyond MSD_NOALLOC_SCRATCH_BYTES raise MSDError."""
        return self._call(load_library().msd_overlap_noalloc, phi_a, phi_b, out, flags, stream)

    def force_bias(self, phi_a, phi_b, out=None, flags=None, stream=None):
        import torch
        nw = self._walkers(phi_a, phi_b)
        out = torch.empty((nw, self.n_chol), dtype=torch.complex128, device=phi_a.device) if out is None else out
        return self._call(load_library().msd_force_bias, phi_a, phi_b, out, flags, stream)

    def reference_cond(self, phi_a, phi_b, stream=None):
        """msd_reference_cond: ||O0||_F ||O0^-1||_F per walker and spin, float64 [n_w][2] on the walkers' device."""
        import torch
        nw = self._walkers(phi_a, phi_b)
        out = torch.empty((nw, 2), dtype=torch.float64, device=phi_a.device)
        self._check(load_library().msd_reference_cond(self._h, nw, phi_a.data_ptr(), phi_b.data_ptr(), out.data_ptr(),
                                                      _stream_ptr(stream)))
        return out

    def force_bias_overlap(self, phi_a, phi_b, out=None, out_ovlp=None, flags=None, stream=None):
        """msd_force_bias_overlap: (fb [n_w][n_chol], ovlp [n_w]) of the same walkers from one determinant pass."""
        import torch
        nw = self._walkers(phi_a, phi_b)
        dev = phi_a.device
        out = torch.empty((nw, self.n_chol), dtype=torch.complex128, device=dev) if out is None else out
        out_ovlp = torch.empty(nw, dtype=torch.complex128, device=dev) if out_ovlp is None else out_ovlp
        if not (isinstance(out_ovlp, torch.Tensor) and out_ovlp.is_cuda and out_ovlp.device == dev
                and out_ovlp.dtype == torch.complex128 and out_ovlp.is_contiguous() and tuple(out_ovlp.shape) == (nw,)):
            raise ValueError("out_ovlp must be a contiguous CUDA complex128 tensor of shape (%d,) on the walkers' device" % nw)
        lib = load_library()

        def fn(h, n, a, b, o, f, st):
            return lib.msd_force_bias_overlap(h, n, a, b, o, out_ovlp.data_ptr(), f, st)
        fn.__name__ = "msd_force_bias"
        self._call(fn, phi_a, phi_b, out, flags, stream)
        return out, out_ovlp

    def local_energy(self, phi_a, phi_b, out=None, flags=None, stream=None):
        import torch
        nw = self._walkers(phi_a, phi_b)
        out = torch.empty((nw, 3), dtype=torch.complex128, device=phi_a.device) if out is None else out
        return self._call(load_library().msd_local_energy, phi_a, phi_b, out, flags, stream)

    def force_bias_energy(self, phi_a, phi_b, out=None, flags=None, stream=None):
        """Both outputs from one pass: returns out [n_w][n_chol + 3]; out[:, :n_chol] is the force bias,
        out[:, n_chol:] is (E, E1, E2)."""
        import torch
        nw = self._walkers(phi_a, phi_b)
        out = torch.empty((nw, self.n_chol + 3), dtype=torch.complex128, device=phi_a.device) if out is None else out
        return self._call(load_library().msd_force_bias_energy, phi_a, phi_b, out, flags, stream)

    def greens(self, phi_a, phi_b, out=None, flags=None, stream=None):
        import torch
        nw = self._walkers(phi_a, phi_b)
        out = torch.empty((nw, 2, self.N, self.N), dtype=torch.complex128, device=phi_a.device) if out is None else out
        return self._call(load_library().msd_greens, phi_a, phi_b, out, flags, stream)

    # -- one propagation step (Eq. 5, 7-12) -------------------------------------------------
    def propagator_setup(self, dt: float, n_taylor: int, h1, L, stream=None):
        h1 = _np(h1, np.float64); L = _np(L, np.float64)
        if h1.shape != (self.N, self.N) or L.shape != (self.n_chol, self.N, self.N):
            raise ValueError("h1 / L shapes disagree with the trial")
        self._check(load_library().msd_propagator_setup(self._h, float(dt), int(n_taylor), _ptr(h1), _ptr(L),
                                                        _stream_ptr(stream)))

    def propagate(self, phi_a, phi_b, x, weights=None, out=None, flags=None, stream=None):
        """In place on phi_a / phi_b (and weights); returns step_out [n_w][8] float64 (see include/msd.h)."""
        import torch
        nw = self._walkers(phi_a, phi_b)
        dev = phi_a.device

        def f64(t, shape, what):
            if not (isinstance(t, torch.Tensor) and t.is_cuda and t.device == dev and t.dtype == torch.float64
                    and t.is_contiguous() and tuple(t.shape) == shape):
                raise ValueError("%s must be a contiguous CUDA float64 tensor of shape %s" % (what, (shape,)))
            return t
        f64(x, (nw, self.n_chol), "x")
        if weights is not None:
            f64(weights, (nw,), "weights")
        out = torch.empty((nw, 8), dtype=torch.float64, device=dev) if out is None else f64(out, (nw, 8), "out")
        if flags is not None and not (flags.is_cuda and flags.dtype == torch.int32 and flags.is_contiguous()
                                      and flags.numel() >= nw):
            raise ValueError("flags must be a contiguous CUDA int32 tensor of at least n_w elements")
        rc = load_library().msd_propagate(self._h, nw, phi_a.data_ptr(), phi_b.data_ptr(), x.data_ptr(),
                                          weights.data_ptr() if weights is not None else None, out.data_ptr(),
                                          flags.data_ptr() if flags is not None else None, _stream_ptr(stream))
        self._check(rc)
        return out

    # -- HOST-buffer variants (numpy or CPU torch arrays in and out; copies happen inside the C call) ----
    def _call_host(self, fn, phi_a, phi_b, out, flags, stream):
        def host_ptr(a, dtype, shape=None):
            if hasattr(a, "data_ptr"):                 # CPU torch tensor (e.g. pinned)
                import torch
                want = {np.complex128: torch.complex128, np.int32: torch.int32}[dtype]
                if a.is_cuda or not a.is_contiguous() or a.dtype != want:
                    raise ValueError("host variants take contiguous CPU %s buffers" % np.dtype(dtype).name)
                ptr = a.data_ptr()
            elif isinstance(a, np.ndarray) and a.dtype == dtype and a.flags.c_contiguous:
                ptr = a.ctypes.data
            else:
                raise ValueError("host variants take contiguous %s arrays" % np.dtype(dtype).name)
            if shape is not None and tuple(a.shape) != tuple(shape):
                raise ValueError("buffer of shape %s expected, got %s" % (tuple(shape), tuple(a.shape)))
            return ptr
        nw = int(phi_a.shape[0])
        if tuple(phi_a.shape) != (nw, self.N, self.n_alpha) or tuple(phi_b.shape) != (nw, self.N, self.n_beta):
            raise ValueError("walkers must be [n_w][N][n_sigma]")
        host_ptr(out, np.complex128, self._out_shape(fn, nw))
        if flags is not None and int(np.prod(flags.shape)) < nw:
            raise ValueError("flags must hold at least n_w elements")
        rc = fn(self._h, nw, host_ptr(phi_a, np.complex128), host_ptr(phi_b, np.complex128),
                host_ptr(out, np.complex128), host_ptr(flags, np.int32) if flags is not None else None,
                _stream_ptr(stream))
        self._check(rc)
        return out

    def overlap_host(self, phi_a, phi_b, out=None, flags=None, stream=None):
        out = np.empty(phi_a.shape[0], dtype=np.complex128) if out is None else out
        return self._call_host(load_library().msd_overlap_host, phi_a, phi_b, out, flags, stream)

    def force_bias_host(self, phi_a, phi_b, out=None, flags=None, stream=None):
        out = np.empty((phi_a.shape[0], self.n_chol), dtype=np.complex128) if out is None else out
        return self._call_host(load_library().msd_force_bias_host, phi_a, phi_b, out, flags, stream)

    def local_energy_host(self, phi_a, phi_b, out=None, flags=None, stream=None):
        out = np.empty((phi_a.shape[0], 3), dtype=np.complex128) if out is None else out
        return self._call_host(load_library().msd_local_energy_host, phi_a, phi_b, out, flags, stream)

    def force_bias_energy_host(self, phi_a, phi_b, out=None, flags=None, stream=None):
        out = np.empty((phi_a.shape[0], self.n_chol + 3), dtype=np.complex128) if out is None else out
        return self._call_host(load_library().msd_force_bias_energy_host, phi_a, phi_b, out, flags, stream)

    # -- introspection -------------------------------------------------------------------------
    def info(self) -> dict:
        a = np.zeros(11, dtype=np.int64)
        self._check(load_library().msd_get_info(self._h, _ptr(a)))
        keys = ["n_o_alpha", "n_v_alpha", "n_o_beta", "n_v_beta", "n_buckets", "kmax_alpha", "kmax_beta", "walker_tile",
                "energy_supported", "shard_rank", "shard_world"]
        return dict(zip(keys, (int(v) for v in a)))

    def packed(self) -> dict:
        perm = np.zeros(self.n_det, dtype=np.int64)
        coef = np.zeros(self.n_det, dtype=np.float64)
        la = np.zeros(self.n_det, dtype=np.int32)
        lb = np.zeros(self.n_det, dtype=np.int32)
        self._check(load_library().msd_get_packed(self._h, _ptr(perm), _ptr(coef), _ptr(la), _ptr(lb)))
        return dict(perm=perm, coef=coef, level_a=la, level_b=lb)

    def set_workspace_limit(self, nbytes: int):
        self._check(load_library().msd_set_workspace_limit(self._h, int(nbytes)))

    def set_allreduce(self, fn):
        """Determinant sharding (include/msd.h msd_set_allreduce): fn(t) must sum the CUDA float64 tensor t over the ranks in
        place, enqueued on the current stream (the binding makes the call's stream current).  None removes the hook."""
        lib = load_library()
        if fn is None:
            self._allreduce_cb = None
            self._check(lib.msd_set_allreduce(self._h, None, None))
            return
        import torch

        class _View:                      # raw device memory as a tensor (no copy): __cuda_array_interface__
            def __init__(self, ptr, n):
                self.__cuda_array_interface__ = {"shape": (n,), "typestr": "<f8", "data": (ptr, False), "version": 2}

        def hook(_user, buf, n, stream):
            try:
                t = torch.as_tensor(_View(int(buf), int(n)), device=torch.device("cuda", torch.cuda.current_device()))
                ext = torch.cuda.ExternalStream(int(stream or 0))
                with torch.cuda.stream(ext):
                    fn(t)
                ext.synchronize()         # the kernels the library enqueues next must see the reduced sums
            except BaseException as e:            # an exception must not cross the C ABI
                self._allreduce_error = e
        self._allreduce_error = None
        self._allreduce_cb = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p)(hook)
        self._check(lib.msd_set_allreduce(self._h, C.cast(self._allreduce_cb, C.c_void_p), None))

    def set_option(self, option: int, value: int):
        self._check(load_library().msd_set_option(self._h, int(option), int(value)))

    def launch_count(self) -> int:
        return int(load_library().msd_launch_count(self._h))

    def set_profiling(self, on: bool):
        self._check(load_library().msd_set_profiling(self._h, 1 if on else 0))

    def phase_ms(self) -> dict:
        a = np.zeros(6, dtype=np.float32)
        self._check(load_library().msd_get_phase_ms(self._h, _ptr(a), 6))
        return dict(zip(["reference", "p1", "p2", "p3", "p4", "p5"], (float(v) for v in a)))


def msd_setup(N, n_alpha, n_beta, n_chol, n_det, h1, L, e0, occ_ref_a, occ_ref_b,
              exc_off_a, holes_a, parts_a, exc_off_b, holes_b, parts_b, ci, stream=None, shard=(0, 1)) -> MSDTrial:
    """include/msd.h msd_setup / msd_setup_sharded (shard = (rank, world)): host numpy arrays in, device-resident packed trial out."""
    lib = load_library()
    h1 = _np(h1, np.float64); L = _np(L, np.float64); ci = _np(ci, np.float64)
    ra = _np(occ_ref_a, np.int32); rb = _np(occ_ref_b, np.int32)
    oa = _np(exc_off_a, np.int64); ob = _np(exc_off_b, np.int64)
    ha = _np(holes_a, np.int32); pa = _np(parts_a, np.int32)
    hb = _np(holes_b, np.int32); pb = _np(parts_b, np.int32)
    if h1.shape != (N, N) or L.shape != (n_chol, N, N) or ci.shape != (n_det,):
        raise ValueError("h1 / L / ci shapes disagree with N, n_chol, n_det")
    if ra.shape != (n_alpha,) or rb.shape != (n_beta,) or oa.shape != (n_det + 1,) or ob.shape != (n_det + 1,):
        raise ValueError("occ_ref / exc_off shapes disagree with n_alpha, n_beta, n_det")
    if len(ha) != len(pa) or len(hb) != len(pb) or len(ha) != oa[-1] or len(hb) != ob[-1]:
        raise ValueError("holes / parts lengths disagree with exc_off")
    out = C.c_void_p()
    rc = lib.msd_setup_sharded(C.byref(out), N, n_alpha, n_beta, n_chol, n_det, _ptr(h1), _ptr(L), float(e0),
                               _ptr(ra), _ptr(rb), _ptr(oa), _ptr(ha), _ptr(pa), _ptr(ob), _ptr(hb), _ptr(pb), _ptr(ci),
                               int(shard[0]), int(shard[1]), _stream_ptr(stream))
    if rc != MSD_OK:
        msg = lib.msd_last_error(None)
        raise MSDError(rc, msg.decode() if msg else "")
    return MSDTrial(out.value, N, n_alpha, n_beta, n_chol, n_det)


def msd_setup_from_occ(N, n_alpha, n_beta, n_chol, n_det, h1, L, e0, occa, occb, ci, stream=None) -> MSDTrial:
    """include/msd.h msd_setup_from_occ: the paper's (coeff, occa, occb) format."""
    lib = load_library()
    h1 = _np(h1, np.float64); L = _np(L, np.float64); ci = _np(ci, np.float64)
    occa = _np(occa, np.int32); occb = _np(occb, np.int32)
    if occa.shape != (n_det, n_alpha) or occb.shape != (n_det, n_beta):
        raise ValueError("occa / occb shapes disagree with n_det, n_alpha, n_beta")
    if h1.shape != (N, N) or L.shape != (n_chol, N, N) or ci.shape != (n_det,):
        raise ValueError("h1 / L / ci shapes disagree with N, n_chol, n_det")
    out = C.c_void_p()
    rc = lib.msd_setup_from_occ(C.byref(out), N, n_alpha, n_beta, n_chol, n_det, _ptr(h1), _ptr(L), float(e0),
                                _ptr(occa), _ptr(occb), _ptr(ci), _stream_ptr(stream))
    if rc != MSD_OK:
        msg = lib.msd_last_error(None)
        raise MSDError(rc, msg.decode() if msg else "")
    return MSDTrial(out.value, N, n_alpha, n_beta, n_chol, n_det)


def msd_overlap(trial: MSDTrial, phi_a, phi_b, out=None, flags=None, stream=None):
    return trial.overlap(phi_a, phi_b, out, flags, stream)


def msd_force_bias(trial: MSDTrial, phi_a, phi_b, out=None, flags=None, stream=None):
    return trial.force_bias(phi_a, phi_b, out, flags, stream)


def msd_force_bias_energy(trial: MSDTrial, phi_a, phi_b, out=None, flags=None, stream=None):
    return trial.force_bias_energy(phi_a, phi_b, out, flags, stream)


def msd_force_bias_energy_host(trial: MSDTrial, phi_a, phi_b, out=None, flags=None, stream=None):
    return trial.force_bias_energy_host(phi_a, phi_b, out, flags, stream)


def msd_local_energy(trial: MSDTrial, phi_a, phi_b, out=None, flags=None, stream=None):
    return trial.local_energy(phi_a, phi_b, out, flags, stream)


def msd_greens(trial: MSDTrial, phi_a, phi_b, out=None, flags=None, stream=None):
    return trial.greens(phi_a, phi_b, out, flags, stream)


def msd_overlap_host(trial: MSDTrial, phi_a, phi_b, out=None, flags=None, stream=None):
    return trial.overlap_host(phi_a, phi_b, out, flags, stream)


def msd_force_bias_host(trial: MSDTrial, phi_a, phi_b, out=None, flags=None, stream=None):
    return trial.force_bias_host(phi_a, phi_b, out, flags, stream)


def msd_local_energy_host(trial: MSDTrial, phi_a, phi_b, out=None, flags=None, stream=None):
    return trial.local_energy_host(phi_a, phi_b, out, flags, stream)


def setup_from_inputs(inp, stream=None, shard=(0, 1)) -> MSDTrial:
    """Convenience for msd_inputs.MSDInputs (tests / bench); shard = (rank, world) for determinant sharding."""
    return msd_setup(inp.N, inp.n_alpha, inp.n_beta, inp.n_chol, inp.n_det, inp.h1, inp.L, inp.e0,
                     inp.occ_ref_a, inp.occ_ref_b, inp.exc_off_a, inp.holes_a, inp.parts_a,
                     inp.exc_off_b, inp.holes_b, inp.parts_b, inp.ci, stream=stream, shard=shard)


def dist_allreduce(group=None):
    """The hook for MSDTrial.set_allreduce under torch.distributed (NCCL over NVLink on GPUs): in-place SUM over the ranks."""
    import torch.distributed as dist

    def fn(t):
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return fn
