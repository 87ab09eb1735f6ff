"""Python binding of include/b200sht.h -- argument marshalling only; every step of the transforms runs in the CUDA
library.  PyTorch supplies device memory and the current CUDA stream, nothing else.

Layouts (see include/b200sht.h): flm[L, 2L-1] complex128 (column m+L-1); MW maps f[L, 2L-1] (MWSS [L+1, 2L], DH [2L, 2L-1],
GL [L, 2L-1]); HEALPix maps
f[12 nside^2] ring-ordered; SO(3) f[2N-1, L, 2L-1] = (gamma, beta, alpha); flmn[2N-1, L, 2L-1] = (n+N-1, l, m+L-1).
With reality=True maps are float64.
"""
import ctypes as C

import numpy as np
import torch

from . import _lib
from ._lib import SHT_DH, SHT_F32, SHT_F64, SHT_GL, SHT_HEALPIX, SHT_MW, SHT_MWSS, check, lib

MW, HEALPIX, MWSS, DH, GL = SHT_MW, SHT_HEALPIX, SHT_MWSS, SHT_DH, SHT_GL


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _dev(t, dtype, shape, what):
    if not (isinstance(t, torch.Tensor) and t.is_cuda):
        raise TypeError(f"{what} must be a CUDA tensor")
    if t.dtype != dtype or tuple(t.shape) != tuple(shape) or not t.is_contiguous():
        raise ValueError(f"{what}: expected contiguous {dtype} of shape {tuple(shape)}, got {t.dtype} {tuple(t.shape)}")
    return C.c_void_p(t.data_ptr())


def map_shape(L, sampling=MW, nside=0):
    """MW [L, 2L-1]; MWSS [L+1, 2L]; DH [2L, 2L-1]; GL [L, 2L-1]; HEALPix [12 nside^2] (ring-ordered)."""
    if sampling == HEALPIX:
        return (12 * nside * nside,)
    return {MW: (L, 2 * L - 1), MWSS: (L + 1, 2 * L), DH: (2 * L, 2 * L - 1), GL: (L, 2 * L - 1)}[sampling]


class Plan:
    """A transform plan (sht_plan): fixes the problem, owns one workspace tensor allocated through PyTorch."""

    def __init__(self, L, spin=0, sampling=MW, nside=0, reality=False, N=None, device="cuda:0", batch=1, dtype="f64",
                 fold=None, invsym=None, tile=None, adjoint=False, precompute=False, pair=None, graph=None, skip=None):
        """fold / invsym / tile map to the SHT_OPT_* creation flags (None = the library's automatic choice)."""
        self._h = C.c_void_p()
        opts = 0
        if fold is not None:
            opts |= _lib.SHT_OPT_FOLD_ON if fold else _lib.SHT_OPT_FOLD_OFF
        if invsym is not None:
            opts |= _lib.SHT_OPT_INVSYM if invsym else _lib.SHT_OPT_NO_INVSYM
        if tile is not None:
            opts |= {64: _lib.SHT_OPT_TILE64, 128: _lib.SHT_OPT_TILE128}[tile]
        if adjoint:
            opts |= _lib.SHT_OPT_ADJOINT
        if precompute:
            opts |= _lib.SHT_OPT_PRECOMPUTE
        if pair is not None and not pair:
            opts |= _lib.SHT_OPT_NO_PAIR
        if graph is not None:
            opts |= _lib.SHT_OPT_GRAPH if graph else _lib.SHT_OPT_NO_GRAPH
        if skip is not None and not skip:
            opts |= _lib.SHT_OPT_NO_SKIP
        self.L, self.spin, self.sampling, self.nside, self.reality, self.N = L, spin, sampling, nside, bool(reality), N
        self.batch = int(batch)
        if dtype not in ("f64", "f32"):
            raise ValueError("dtype must be 'f64' or 'f32'")
        self.dtype = dtype          # 'f32': complex64 / float32 arrays; fp32 hot kernels for spin 0, the fp64 kernels between fp32 arrays for spin != 0
        code = SHT_F32 if dtype == "f32" else SHT_F64
        self.device = torch.device(device)
        L_ = lib()
        with torch.cuda.device(self.device):
            if N is None:
                check(L_.sht_plan_s2_opts(C.byref(self._h), L, spin, sampling, nside, int(self.reality), code, self.batch, opts))
            else:
                check(L_.sht_plan_so3_opts(C.byref(self._h), L, N, code, opts))
            nbytes = L_.sht_plan_workspace_bytes(self._h)
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            check(L_.sht_plan_set_workspace(self._h, C.c_void_p(self.workspace.data_ptr()), nbytes, _stream()))
        self.coef_dtype = torch.complex64 if dtype == "f32" else torch.complex128
        if dtype == "f32":
            self.map_dtype = torch.float32 if self.reality else torch.complex64
        else:
            self.map_dtype = torch.float64 if self.reality else torch.complex128
        self.coef_shape = (L, 2 * L - 1) if N is None else (2 * N - 1, L, 2 * L - 1)
        self.map_shape = map_shape(L, sampling, nside) if N is None else (2 * N - 1, L, 2 * L - 1)
        if self.batch > 1:            # a batch of maps transformed together: leading [batch] axis on both sides
            self.coef_shape = (self.batch,) + self.coef_shape
            self.map_shape = (self.batch,) + self.map_shape

    def __del__(self):
        try:
            if self._h:
                lib().sht_plan_destroy(self._h)
                self._h = C.c_void_p()
        except Exception:
            pass

    # -- transforms (device tensors in, device tensors out) --
    def forward(self, f, out=None):
        out = torch.empty(self.coef_shape, dtype=self.coef_dtype, device=self.device) if out is None else out
        fn = lib().s2_forward_plan if self.N is None else lib().so3_forward_plan
        check(fn(self._h, _dev(f, self.map_dtype, self.map_shape, "f"), _dev(out, self.coef_dtype, self.coef_shape, "flm"), _stream()))
        return out

    def forward_iter(self, f, niter, out=None):
        """HEALPix forward with `niter` refinement iterations: flm <- flm + F (f - F^-1 flm)."""
        out = torch.empty(self.coef_shape, dtype=self.coef_dtype, device=self.device) if out is None else out
        check(lib().s2_forward_iter_plan(self._h, _dev(f, self.map_dtype, self.map_shape, "f"),
                                         _dev(out, self.coef_dtype, self.coef_shape, "flm"), int(niter), _stream()))
        return out

    def inverse(self, flm, out=None):
        out = torch.empty(self.map_shape, dtype=self.map_dtype, device=self.device) if out is None else out
        fn = lib().s2_inverse_plan if self.N is None else lib().so3_inverse_plan
        check(fn(self._h, _dev(flm, self.coef_dtype, self.coef_shape, "flm"), _dev(out, self.map_dtype, self.map_shape, "f"), _stream()))
        return out

    # -- adjoints (plans created with adjoint=True; Eq. 52 / 58) --
    def forward_adjoint(self, flm, out=None):
        """F^H: coefficients -> map (the conjugate transpose of forward)."""
        out = torch.empty(self.map_shape, dtype=self.map_dtype, device=self.device) if out is None else out
        fn = lib().s2_forward_adjoint_plan if self.N is None else lib().so3_forward_adjoint_plan
        check(fn(self._h, _dev(flm, self.coef_dtype, self.coef_shape, "flm"),
                                            _dev(out, self.map_dtype, self.map_shape, "f"), _stream()))
        return out

    def inverse_adjoint(self, f, out=None):
        """(F^-1)^H: map -> coefficients (the conjugate transpose of inverse)."""
        out = torch.empty(self.coef_shape, dtype=self.coef_dtype, device=self.device) if out is None else out
        fn = lib().s2_inverse_adjoint_plan if self.N is None else lib().so3_inverse_adjoint_plan
        check(fn(self._h, _dev(f, self.map_dtype, self.map_shape, "f"),
                                            _dev(out, self.coef_dtype, self.coef_shape, "flm"), _stream()))
        return out

    def theta_forward_adjoint(self, flm):
        """Conjugate transpose of theta_forward: flm -> W[2L-1, ntheta_q] (Eq. 62-63 without Q_Theta)."""
        out = torch.empty((2 * self.L - 1, self.ntheta(True)), dtype=torch.complex128, device=self.device)
        check(lib().s2_theta_forward_adjoint_plan(self._h, _dev(flm, torch.complex128, self.coef_shape, "flm"), C.c_void_p(out.data_ptr()), _stream()))
        return out

    def theta_inverse_adjoint(self, F):
        """Conjugate transpose of theta_inverse: F[2L-1, ntheta] -> flm (Eq. 67-68)."""
        shape = (2 * self.L - 1, self.ntheta(False))
        out = torch.empty(self.coef_shape, dtype=torch.complex128, device=self.device)
        check(lib().s2_theta_inverse_adjoint_plan(self._h, _dev(F, torch.complex128, shape, "F"), C.c_void_p(out.data_ptr()), _stream()))
        return out

    # -- ring shards (one transform over several GPUs) --
    def set_shard(self, rank, nranks):
        """Serve share `rank` of `nranks` of the kernel rings: forward returns a partial flm (sum over ranks = transform), inverse
        a map with only this shard's rings filled."""
        check(lib().sht_plan_set_shard(self._h, int(rank), int(nranks)))

    def shard_range(self, forward):
        a, n = C.c_int(), C.c_int()
        check(lib().sht_plan_shard_range(self._h, int(forward), C.byref(a), C.byref(n)))
        return a.value, a.value + n.value

    def ntheta(self, forward):
        return int(lib().sht_plan_ntheta(self._h, int(forward)))

    def theta_inverse(self, flm):
        """Hot path only (Eq. 33): flm -> F[2L-1, ntheta], row m+L-1."""
        out = torch.empty((2 * self.L - 1, self.ntheta(False)), dtype=torch.complex128, device=self.device)
        check(lib().s2_theta_inverse_plan(self._h, _dev(flm, torch.complex128, self.coef_shape, "flm"), C.c_void_p(out.data_ptr()), _stream()))
        return out

    def theta_forward(self, W):
        """Hot path only (Eq. 30): weighted W[2L-1, ntheta_q] (row m+L-1) -> flm."""
        shape = (2 * self.L - 1, self.ntheta(True))
        out = torch.empty(self.coef_shape, dtype=torch.complex128, device=self.device)
        check(lib().s2_theta_forward_plan(self._h, _dev(W, torch.complex128, shape, "W"), C.c_void_p(out.data_ptr()), _stream()))
        return out

    def enable_timing(self, on=True):
        check(lib().sht_plan_enable_timing(self._h, int(on)))

    def timings(self):
        """dict(hot, fft, staging, total) in ms for the last transform (synchronises)."""
        ms = (C.c_float * 4)()
        check(lib().sht_plan_timings(self._h, ms))
        return dict(hot=ms[0], fft=ms[1], staging=ms[2], total=ms[3])

    def stage_bytes(self):
        """dict(fft, staging): algorithmic bytes moved by the FFT / staging sections of the last timed transform."""
        b = (C.c_double * 3)()
        check(lib().sht_plan_stage_bytes(self._h, b))
        return dict(fft=b[1], staging=b[2])

    def dsteps(self, forward):
        return float(lib().sht_plan_dsteps(self._h, int(forward)))

    def skip_fraction(self, forward):
        """Share of the fused kernels' block-steps this plan skips (silent head of the polar tiles); 0 if every step runs."""
        return float(lib().sht_plan_skip_fraction(self._h, int(forward)))

    def flops(self, forward):
        """Algorithmic flop of the hot kernels of one transform (6 per d-step + 4 per order and map served)."""
        return float(lib().sht_plan_flops(self._h, int(forward)))


# -- the north-star calls (library-side plan cache; device tensors) --
def s2_forward(f, L, spin=0, sampling=MW, reality=False):
    nside = L // 2 if sampling == HEALPIX else 0
    dt = torch.float64 if reality else torch.complex128
    flm = torch.empty((L, 2 * L - 1), dtype=torch.complex128, device=f.device)
    with torch.cuda.device(f.device):
        check(lib().s2_forward(L, spin, sampling, int(reality), _dev(f, dt, map_shape(L, sampling, nside), "f"), C.c_void_p(flm.data_ptr()), _stream()))
    return flm


def s2_inverse(flm, L, spin=0, sampling=MW, reality=False):
    nside = L // 2 if sampling == HEALPIX else 0
    dt = torch.float64 if reality else torch.complex128
    f = torch.empty(map_shape(L, sampling, nside), dtype=dt, device=flm.device)
    with torch.cuda.device(flm.device):
        check(lib().s2_inverse(L, spin, sampling, int(reality), _dev(flm, torch.complex128, (L, 2 * L - 1), "flm"), C.c_void_p(f.data_ptr()), _stream()))
    return f


def so3_forward(f, L, N):
    shape = (2 * N - 1, L, 2 * L - 1)
    flmn = torch.empty(shape, dtype=torch.complex128, device=f.device)
    with torch.cuda.device(f.device):
        check(lib().so3_forward(L, N, _dev(f, torch.complex128, shape, "f"), C.c_void_p(flmn.data_ptr()), _stream()))
    return flmn


def so3_inverse(flmn, L, N):
    shape = (2 * N - 1, L, 2 * L - 1)
    f = torch.empty(shape, dtype=torch.complex128, device=flmn.device)
    with torch.cuda.device(flmn.device):
        check(lib().so3_inverse(L, N, _dev(flmn, torch.complex128, shape, "flmn"), C.c_void_p(f.data_ptr()), _stream()))
    return f


# -- end-to-end through HOST buffers (numpy arrays; copies happen inside the C call) --
def _host(a, dtype, shape, what):
    a = np.ascontiguousarray(a, dtype=dtype)
    if tuple(a.shape) != tuple(shape):
        raise ValueError(f"{what}: expected shape {tuple(shape)}, got {a.shape}")
    return a


def s2_forward_host(f, L, spin=0, sampling=MW, reality=False, out=None):
    nside = L // 2 if sampling == HEALPIX else 0
    f = _host(f, np.float64 if reality else np.complex128, map_shape(L, sampling, nside), "f")
    out = np.empty((L, 2 * L - 1), np.complex128) if out is None else out
    check(lib().s2_forward_host(L, spin, sampling, int(reality), f.ctypes.data, out.ctypes.data, _stream()))
    return out


def s2_inverse_host(flm, L, spin=0, sampling=MW, reality=False, out=None):
    nside = L // 2 if sampling == HEALPIX else 0
    flm = _host(flm, np.complex128, (L, 2 * L - 1), "flm")
    out = np.empty(map_shape(L, sampling, nside), np.float64 if reality else np.complex128) if out is None else out
    check(lib().s2_inverse_host(L, spin, sampling, int(reality), flm.ctypes.data, out.ctypes.data, _stream()))
    return out


def so3_forward_host(f, L, N, out=None):
    shape = (2 * N - 1, L, 2 * L - 1)
    f = _host(f, np.complex128, shape, "f")
    out = np.empty(shape, np.complex128) if out is None else out
    check(lib().so3_forward_host(L, N, f.ctypes.data, out.ctypes.data, _stream()))
    return out


def so3_inverse_host(flmn, L, N, out=None):
    shape = (2 * N - 1, L, 2 * L - 1)
    flmn = _host(flmn, np.complex128, shape, "flmn")
    out = np.empty(shape, np.complex128) if out is None else out
    check(lib().so3_inverse_host(L, N, flmn.ctypes.data, out.ctypes.data, _stream()))
    return out


def fp64_peak(iters=20000):
    """Measured FP64 FMA throughput of this GPU (register-only DFMA chains): (TFLOP/s, ms)."""
    tf, ms = C.c_double(), C.c_float()
    check(lib().sht_fp64_peak(iters, C.byref(tf), C.byref(ms), _stream()))
    return tf.value, ms.value


def peak(kind, iters=20000):
    """Measured instruction-chain peak: kind 'dfma' | 'dmma' | 'ffma' | 'ffma2' -> (TFLOP/s, ms)."""
    code = {"dfma": _lib.SHT_PEAK_DFMA, "dmma": _lib.SHT_PEAK_DMMA, "ffma": _lib.SHT_PEAK_FFMA, "ffma2": _lib.SHT_PEAK_FFMA2}[kind]
    tf, ms = C.c_double(), C.c_float()
    check(lib().sht_peak(code, iters, C.byref(tf), C.byref(ms), _stream()))
    return tf.value, ms.value


def launch_count(reset=False):
    return int(lib().sht_launch_count(int(reset)))


def cache_clear():
    check(lib().sht_cache_clear())


def theta_inverse_noalloc(flm, L, spin, theta, out=None):
    """Allocation-free theta step of the inverse transform (Eq. 33) on the rings `theta` (host sequence of colatitudes): flm[L, 2L-1]
    -> F[2L-1, len(theta)].  The library call allocates nothing (d-function table in a static device array of
    SHT_NOALLOC_SCRATCH_BYTES); pass `out` to keep this wrapper from allocating the result too.  Calls share the static table:
    do not overlap them on the GPU."""
    th = np.ascontiguousarray(np.asarray(theta, dtype=np.float64).ravel())
    nt = int(th.size)
    shape = (2 * L - 1, nt)
    if out is None:
        out = torch.empty(shape, dtype=torch.complex128, device=flm.device)
    err = C.create_string_buffer(512)
    rc = lib().s2_theta_inverse_noalloc(int(L), int(spin), nt, th.ctypes.data_as(C.POINTER(C.c_double)),
                                        _dev(flm, torch.complex128, (L, 2 * L - 1), "flm"), _dev(out, torch.complex128, shape, "F"),
                                        _stream(), err, len(err))
    if rc != 0:
        raise _lib.ShtError(f"{lib().sht_status_string(rc).decode()} [{err.value.decode()}]")
    return out
