"""Thin ctypes binding of libmala_snap.so (include/mala_snap.h).  Argument marshalling only.

Every step of the path (binning, compute_ui, compute_zi, compute_bi, writer) runs in the CUDA kernels behind the
C ABI; PyTorch is used for device memory and streams only.  There is no CPU fallback: without the compiled
library or without a CUDA device the calls raise.
"""
import ctypes as C
import os

import numpy as np

dp_t = C.POINTER(C.c_double)
_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libmala_snap.so")
_lib = None

MALA_SNAP_OK = 0
MALA_SNAP_EINVAL = -1
MALA_SNAP_ECUDA = -2
MALA_SNAP_ENOMEM = -3

EXPORTS = ("mala_snap_create", "mala_snap_ncomp", "mala_snap_triples", "mala_bispectrum_grid", "mala_bispectrum_grid_host",
           "mala_gaussian_grid", "mala_gaussian_grid_static", "mala_mlp_create", "mala_mlp_widths", "mala_mlp_forward", "mala_mlp_destroy", "mala_bispectrum_ldos_grid", "mala_bispectrum_force_adjoint",
           "mala_snap_set_option", "mala_snap_last_stats", "mala_snap_kernel_times", "mala_snap_zi_kernel", "mala_snap_fp64_peak", "mala_snap_clebsch_gordan", "mala_snap_debug_utot",
           "mala_snap_destroy", "mala_last_error")


class MalaSnapError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libmala_snap error {code}: {msg}")
        self.code = code


def library_path():
    return _LIB_PATH


def load_library():
    """dlopen libmala_snap.so, building it with nvcc first if it is missing or stale.  Raises if that fails."""
    global _lib
    if _lib is not None:
        return _lib
    from . import build as _build
    try:
        path = _build.build()
    except Exception as e:  # no nvcc, or a compile error: never fall back to anything else
        if not os.path.exists(_LIB_PATH):
            raise RuntimeError(f"libmala_snap.so is missing and could not be built ({e}); "
                               "run `python -m paper_2411_19617_b200.build`") from e
        path = _LIB_PATH
    lib = C.CDLL(path)
    dp, ip, vp = C.POINTER(C.c_double), C.POINTER(C.c_int), C.c_void_p
    lib.mala_snap_create.restype = C.c_int
    lib.mala_snap_create.argtypes = [C.POINTER(vp), C.c_int, C.c_double, C.c_double, C.c_double, C.c_double, C.c_int, dp, dp]
    lib.mala_snap_ncomp.restype = C.c_int
    lib.mala_snap_ncomp.argtypes = [vp]
    lib.mala_snap_triples.restype = C.c_int
    lib.mala_snap_triples.argtypes = [vp, ip]
    grid_args = [vp, C.c_int, dp, ip, dp, dp, ip, ip, C.c_int, C.c_int, vp, vp]
    lib.mala_bispectrum_grid.restype = C.c_int
    lib.mala_bispectrum_grid.argtypes = grid_args
    lib.mala_bispectrum_grid_host.restype = C.c_int
    lib.mala_bispectrum_grid_host.argtypes = grid_args
    lib.mala_gaussian_grid.restype = C.c_int
    lib.mala_gaussian_grid.argtypes = [vp, C.c_double] + grid_args[1:]
    lib.mala_gaussian_grid_static.restype = C.c_int
    lib.mala_gaussian_grid_static.argtypes = [vp, C.c_double] + grid_args[1:]
    lib.mala_mlp_create.restype = C.c_int
    lib.mala_mlp_create.argtypes = [C.POINTER(vp), C.c_int, ip, C.POINTER(dp), C.POINTER(dp), C.c_int, C.c_int, dp, dp]
    lib.mala_mlp_widths.restype = C.c_int
    lib.mala_mlp_widths.argtypes = [vp, ip, ip]
    lib.mala_mlp_forward.restype = C.c_int
    lib.mala_mlp_forward.argtypes = [vp, C.c_longlong, vp, vp, vp]
    lib.mala_mlp_destroy.restype = None
    lib.mala_mlp_destroy.argtypes = [vp]
    lib.mala_bispectrum_ldos_grid.restype = C.c_int
    lib.mala_bispectrum_ldos_grid.argtypes = [vp, vp] + grid_args[1:]
    lib.mala_bispectrum_force_adjoint.restype = C.c_int
    lib.mala_bispectrum_force_adjoint.argtypes = grid_args[:10] + [vp, vp, vp]
    lib.mala_snap_debug_utot.restype = C.c_int
    lib.mala_snap_debug_utot.argtypes = grid_args
    lib.mala_snap_set_option.restype = C.c_int
    lib.mala_snap_set_option.argtypes = [vp, C.c_char_p, C.c_longlong]
    lib.mala_snap_last_stats.restype = C.c_int
    lib.mala_snap_last_stats.argtypes = [vp, C.POINTER(C.c_longlong)]
    lib.mala_snap_kernel_times.restype = C.c_int
    lib.mala_snap_kernel_times.argtypes = [vp, dp, C.POINTER(C.c_longlong)]
    lib.mala_snap_zi_kernel.restype = C.c_char_p
    lib.mala_snap_zi_kernel.argtypes = [vp]
    lib.mala_snap_fp64_peak.restype = C.c_int
    lib.mala_snap_fp64_peak.argtypes = [dp, dp, vp]
    lib.mala_snap_clebsch_gordan.restype = C.c_double
    lib.mala_snap_clebsch_gordan.argtypes = [C.c_int] * 6
    lib.mala_snap_destroy.restype = None
    lib.mala_snap_destroy.argtypes = [vp]
    lib.mala_last_error.restype = C.c_char_p
    lib.mala_last_error.argtypes = []
    _lib = lib
    return lib


def mala_last_error():
    return load_library().mala_last_error().decode()


def _check(rc):
    if rc != 0:
        raise MalaSnapError(rc, mala_last_error())


def mala_snap_clebsch_gordan(J1, M1, J2, M2, J, M):
    return load_library().mala_snap_clebsch_gordan(int(J1), int(M1), int(J2), int(M2), int(J), int(M))


def mala_snap_fp64_peak(stream=None):
    """(TFLOP/s, implied SM MHz) of the device's FP64 FMA pipe, measured by the library's register-only probe."""
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    t, f = C.c_double(0.0), C.c_double(0.0)
    _check(load_library().mala_snap_fp64_peak(C.byref(t), C.byref(f), C.c_void_p(s.cuda_stream)))
    return t.value, f.value


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int))


class MalaSnap:
    """One descriptor calculator (mala_snap_create ... mala_snap_destroy)."""

    def __init__(self, twojmax=10, rcutfac=4.67637, rfac0=0.99363, rmin0=0.0, wself=1.0, radelem=(0.5,), wj=(1.0,)):
        lib = load_library()
        self._lib = lib
        self._h = C.c_void_p()
        radelem = _d(radelem).ravel()
        wj = _d(wj).ravel()
        if radelem.shape != wj.shape:
            raise ValueError("radelem and wj must have the same length")
        _check(lib.mala_snap_create(C.byref(self._h), int(twojmax), float(rcutfac), float(rfac0), float(rmin0), float(wself),
                                    int(radelem.shape[0]), _dp(radelem), _dp(wj)))
        self.twojmax = int(twojmax)
        self.ncomp = lib.mala_snap_ncomp(self._h)
        self.ntypes = int(radelem.shape[0])

    # -- mala_snap_destroy
    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            self._lib.mala_snap_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # -- mala_snap_triples
    def triples(self):
        out = np.zeros((self.ncomp, 3), dtype=np.int32)
        _check(self._lib.mala_snap_triples(self._h, _ip(out)))
        return out

    def set_option(self, name, value):
        _check(self._lib.mala_snap_set_option(self._h, name.encode(), int(value)))

    def last_stats(self):
        st = (C.c_longlong * 8)()
        _check(self._lib.mala_snap_last_stats(self._h, st))
        keys = ("kernels", "chunks", "tiles", "ghosts", "cand_cap", "workspace_bytes", "points", "status")
        return dict(zip(keys, [int(x) for x in st]))

    def zi_kernel_name(self):
        return self._lib.mala_snap_zi_kernel(self._h).decode()

    def kernel_times(self):
        """{class: (ms, launches)} of the last call; needs set_option("timing", 1) before it."""
        ms = (C.c_double * 4)()
        n = (C.c_longlong * 4)()
        _check(self._lib.mala_snap_kernel_times(self._h, ms, n))
        return {k: (float(ms[i]), int(n[i])) for i, k in enumerate(("tile_bin", "compute_ui", "compute_zi_bi", "other"))}

    def _system(self, pos, types, box, origin, pbc, ngrid, z_begin, z_end):
        pos = _d(pos).reshape(-1, 3)
        types = _i(types).ravel()
        if types.shape[0] != pos.shape[0]:
            raise ValueError("pos and types disagree on the number of atoms")
        box = _d(box).reshape(9)
        origin = _d(origin).reshape(3)
        pbc = _i(pbc).reshape(3)
        ngrid = _i(ngrid).reshape(3)
        if z_end is None:
            z_end = int(ngrid[2])
        keep = (pos, types, box, origin, pbc, ngrid)
        args = [C.c_int(pos.shape[0]), _dp(pos), _ip(types), _dp(box), _dp(origin), _ip(pbc), _ip(ngrid), C.c_int(int(z_begin)),
                C.c_int(int(z_end))]
        npts = max(int(z_end) - int(z_begin), 0) * int(ngrid[1]) * int(ngrid[0])
        return args, keep, npts

    # -- mala_bispectrum_grid: result in device memory
    def bispectrum_grid(self, pos, types, box, origin=(0, 0, 0), pbc=(1, 1, 1), ngrid=(1, 1, 1), z_begin=0, z_end=None, out=None,
                        stream=None):
        import torch
        args, keep, npts = self._system(pos, types, box, origin, pbc, ngrid, z_begin, z_end)
        if out is None:
            out = torch.empty((npts, self.ncomp), dtype=torch.float64, device="cuda")
        if (not out.is_cuda) or out.dtype != torch.float64 or (not out.is_contiguous()) or out.numel() < npts * self.ncomp:
            raise ValueError("out must be a contiguous CUDA float64 tensor with at least npoints*ncomp elements")
        s = torch.cuda.current_stream() if stream is None else stream
        _check(self._lib.mala_bispectrum_grid(self._h, *args, C.c_void_p(out.data_ptr()), C.c_void_p(s.cuda_stream)))
        return out

    # -- mala_bispectrum_grid_host: result in (pinned) host memory, copies inside the call
    def bispectrum_grid_host(self, pos, types, box, origin=(0, 0, 0), pbc=(1, 1, 1), ngrid=(1, 1, 1), z_begin=0, z_end=None,
                             out=None, stream=None):
        import torch
        args, keep, npts = self._system(pos, types, box, origin, pbc, ngrid, z_begin, z_end)
        if out is None:
            out = torch.empty((npts, self.ncomp), dtype=torch.float64, pin_memory=True)
        if out.is_cuda or out.dtype != torch.float64 or (not out.is_contiguous()) or out.numel() < npts * self.ncomp:
            raise ValueError("out must be a contiguous CPU float64 tensor with at least npoints*ncomp elements")
        s = torch.cuda.current_stream() if stream is None else stream
        _check(self._lib.mala_bispectrum_grid_host(self._h, *args, C.c_void_p(out.data_ptr()), C.c_void_p(s.cuda_stream)))
        return out

    # -- mala_gaussian_grid: Gaussian descriptors [npoints, ntypes]
    def gaussian_grid(self, sigma, pos, types, box, origin=(0, 0, 0), pbc=(1, 1, 1), ngrid=(1, 1, 1), z_begin=0, z_end=None,
                      out=None, stream=None):
        import torch
        args, keep, npts = self._system(pos, types, box, origin, pbc, ngrid, z_begin, z_end)
        if out is None:
            out = torch.empty((npts, self.ntypes), dtype=torch.float64, device="cuda")
        if (not out.is_cuda) or out.dtype != torch.float64 or (not out.is_contiguous()) or out.numel() < npts * self.ntypes:
            raise ValueError("out must be a contiguous CUDA float64 tensor with at least npoints*ntypes elements")
        s = torch.cuda.current_stream() if stream is None else stream
        _check(self._lib.mala_gaussian_grid(self._h, C.c_double(float(sigma)), *args, C.c_void_p(out.data_ptr()),
                                            C.c_void_p(s.cuda_stream)))
        return out

    # -- mala_gaussian_grid_static: the same descriptors through the entry point that allocates no device memory
    def gaussian_grid_static(self, sigma, pos, types, box, origin=(0, 0, 0), pbc=(1, 1, 1), ngrid=(1, 1, 1), z_begin=0, z_end=None,
                             out=None, stream=None):
        import torch
        args, keep, npts = self._system(pos, types, box, origin, pbc, ngrid, z_begin, z_end)
        if out is None:   # the caller of the C entry point owns the output; here torch allocates it before the call
            out = torch.empty((npts, self.ntypes), dtype=torch.float64, device="cuda")
        if (not out.is_cuda) or out.dtype != torch.float64 or (not out.is_contiguous()) or out.numel() < npts * self.ntypes:
            raise ValueError("out must be a contiguous CUDA float64 tensor with at least npoints*ntypes elements")
        s = torch.cuda.current_stream() if stream is None else stream
        _check(self._lib.mala_gaussian_grid_static(self._h, C.c_double(float(sigma)), *args, C.c_void_p(out.data_ptr()),
                                                   C.c_void_p(s.cuda_stream)))
        return out

    # -- mala_bispectrum_force_adjoint: g[atom, k] += sum_points sum_j beta[point, j] dB_j(point)/dR_{atom,k}
    def force_adjoint(self, beta, pos, types, box, origin=(0, 0, 0), pbc=(1, 1, 1), ngrid=(1, 1, 1), z_begin=0, z_end=None, out=None,
                      stream=None):
        import torch
        args, keep, npts = self._system(pos, types, box, origin, pbc, ngrid, z_begin, z_end)
        natoms = keep[0].shape[0]
        if (not beta.is_cuda) or beta.dtype != torch.float64 or (not beta.is_contiguous()) or beta.numel() < npts * self.ncomp:
            raise ValueError("beta must be a contiguous CUDA float64 tensor with at least npoints*ncomp elements")
        if out is None:
            out = torch.zeros((natoms, 3), dtype=torch.float64, device="cuda")
        if (not out.is_cuda) or out.dtype != torch.float64 or (not out.is_contiguous()) or out.numel() < natoms * 3:
            raise ValueError("out must be a contiguous CUDA float64 tensor [natoms, 3]")
        s = torch.cuda.current_stream() if stream is None else stream
        _check(self._lib.mala_bispectrum_force_adjoint(self._h, *args, C.c_void_p(beta.data_ptr()), C.c_void_p(out.data_ptr()),
                                                       C.c_void_p(s.cuda_stream)))
        return out

    # -- mala_snap_debug_utot (test hook)
    def debug_utot(self, pos, types, box, origin=(0, 0, 0), pbc=(1, 1, 1), ngrid=(1, 1, 1), z_begin=0, z_end=None):
        import torch
        args, keep, npts = self._system(pos, types, box, origin, pbc, ngrid, z_begin, z_end)
        nelem = sum((J + 1) * (J // 2 + 1) for J in range(self.twojmax + 1))
        out = torch.zeros((npts, nelem, 2), dtype=torch.float64, device="cuda")
        s = torch.cuda.current_stream()
        rc = self._lib.mala_snap_debug_utot(self._h, *args, C.c_void_p(out.data_ptr()), C.c_void_p(s.cuda_stream))
        if rc < 0:
            _check(rc)
        assert rc == nelem
        return out


ACTIVATIONS = {"identity": 0, "relu": 1, "leaky_relu": 2, "sigmoid": 3}


class MalaMlp:
    """The descriptor -> LDOS network (mala_mlp_create ... mala_mlp_destroy): weights[l] is [w_{l+1}, w_l], biases[l] is [w_{l+1}]."""

    def __init__(self, weights, biases, act="leaky_relu", activate_last=True, in_shift=None, in_scale=None):
        lib = load_library()
        self._lib = lib
        self._h = C.c_void_p()
        ws = [_d(w) for w in weights]
        bs = [_d(b).ravel() for b in biases]
        if len(ws) != len(bs) or not ws:
            raise ValueError("weights and biases must be non-empty lists of the same length")
        sizes = [ws[0].shape[1]] + [w.shape[0] for w in ws]
        for l, (w, b) in enumerate(zip(ws, bs)):
            if w.ndim != 2 or w.shape[1] != sizes[l] or b.shape != (w.shape[0],):
                raise ValueError(f"layer {l}: shapes do not chain")
        sizes_a = _i(sizes)
        wp = (dp_t * len(ws))(*[_dp(w) for w in ws])
        bp = (dp_t * len(bs))(*[_dp(b) for b in bs])
        sh = None if in_shift is None else _d(in_shift).ravel()
        sc = None if in_scale is None else _d(in_scale).ravel()
        for v in (sh, sc):
            if v is not None and v.shape != (sizes[0],):
                raise ValueError("in_shift / in_scale must have w_0 entries")
        _check(lib.mala_mlp_create(C.byref(self._h), len(ws), _ip(sizes_a), wp, bp, int(ACTIVATIONS[act]), int(bool(activate_last)),
                                   None if sh is None else _dp(sh), None if sc is None else _dp(sc)))
        self.sizes = sizes
        self.w_in, self.w_out = sizes[0], sizes[-1]

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            self._lib.mala_mlp_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # -- mala_mlp_forward: x DEVICE [npoints, w_in] fp64 -> y DEVICE [npoints, w_out] fp32
    def forward(self, x, out=None, stream=None):
        import torch
        if (not x.is_cuda) or x.dtype != torch.float64 or (not x.is_contiguous()) or x.dim() != 2 or x.shape[1] != self.w_in:
            raise ValueError("x must be a contiguous CUDA float64 tensor [npoints, w_in]")
        n = x.shape[0]
        if out is None:
            out = torch.empty((n, self.w_out), dtype=torch.float32, device=x.device)
        if (not out.is_cuda) or out.dtype != torch.float32 or (not out.is_contiguous()) or out.numel() < n * self.w_out:
            raise ValueError("out must be a contiguous CUDA float32 tensor with at least npoints*w_out elements")
        s = torch.cuda.current_stream() if stream is None else stream
        _check(self._lib.mala_mlp_forward(self._h, C.c_longlong(n), C.c_void_p(x.data_ptr()), C.c_void_p(out.data_ptr()),
                                          C.c_void_p(s.cuda_stream)))
        return out


def bispectrum_ldos_grid(snap, net, pos, types, box, origin=(0, 0, 0), pbc=(1, 1, 1), ngrid=(1, 1, 1), z_begin=0, z_end=None, out=None,
                         stream=None):
    """mala_bispectrum_ldos_grid: LDOS [npoints, w_out] fp32 in device memory; the descriptors stay inside the library."""
    import torch
    args, keep, npts = snap._system(pos, types, box, origin, pbc, ngrid, z_begin, z_end)
    if out is None:
        out = torch.empty((npts, net.w_out), dtype=torch.float32, device="cuda")
    if (not out.is_cuda) or out.dtype != torch.float32 or (not out.is_contiguous()) or out.numel() < npts * net.w_out:
        raise ValueError("out must be a contiguous CUDA float32 tensor with at least npoints*w_out elements")
    s = torch.cuda.current_stream() if stream is None else stream
    _check(snap._lib.mala_bispectrum_ldos_grid(snap._h, net._h, *args, C.c_void_p(out.data_ptr()), C.c_void_p(s.cuda_stream)))
    return out


def bispectrum_for_workload(snap, w, out=None, host=False, z_begin=0, z_end=None):
    """Convenience: run a workloads.Workload through a MalaSnap built with w.snap_params()."""
    f = snap.bispectrum_grid_host if host else snap.bispectrum_grid
    return f(w.pos, w.types, w.box, w.origin, w.pbc, w.ngrid, z_begin, z_end, out=out)
