"""Thin ctypes binding of include/ptycho_b200.h -- argument marshalling only.

Same names as the C ABI (`ptycho_init` -> `Ptycho.__init__`, `ptycho_iterate` -> `.iterate`,
`ptycho_fetch_*` -> `.fetch_*`, ...).  PyTorch is used for device memory (the workspace is a
torch CUDA tensor) and the stream; every step of the cycle runs in the library's kernels.
There is no CPU fallback: if `csrc/libptycho_b200.so` is missing or no CUDA device is present
this module raises.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
# Development only: PTYCHO_BUILD_ONLY_N=256 compiles one frame size into a separate file (a quarter of the build time);
# the product library always holds all four sizes.
_ONLY_N = os.environ.get("PTYCHO_BUILD_ONLY_N")
_TAG = os.environ.get("PTYCHO_BUILD_TAG", "")   # distinguishes development builds made with different PTYCHO_BUILD_DEFS
LIB_PATH = os.environ.get("PTYCHO_B200_LIB") or os.path.join(_CSRC, f"libptycho_dev{_ONLY_N}{_TAG}.so" if _ONLY_N else "libptycho_b200.so")
ALG = {"EPIE_MB": 0, "DM": 1, "LSQML": 2, "LSQML_PF": 3}
KCLASS = ["rows_fwd", "cols", "rows_inv", "update", "other", "mega"]   # ptycho_kclass
STATUS = ["OK", "EINVAL", "EBOUNDS", "EUNSUPPORTED", "ENOMEM", "ECUDA", "ESTATE"]
NVCC_FLAGS = ["--threads", "0", "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "-diag-suppress", "128"]


class PtychoError(RuntimeError):
    def __init__(self, status: int, msg: str = ""):
        self.status = STATUS[status] if 0 <= status < len(STATUS) else str(status)
        super().__init__(f"ptycho_b200: {self.status} {msg}".strip())


class Params(C.Structure):
    """ptycho_params (include/ptycho_b200.h)."""
    _fields_ = [("batch_size", C.c_int), ("probe_start", C.c_int), ("delta_blend", C.c_float),
                ("delta_obj", C.c_float), ("delta_probe", C.c_float), ("alpha_obj", C.c_float),
                ("alpha_probe", C.c_float), ("lsq_lambda", C.c_float), ("pbound", C.c_float),
                ("disable_dm", C.c_int), ("deterministic", C.c_int), ("dm_sweeps", C.c_int),
                ("batch_order", C.POINTER(C.c_int32)), ("shard_total_pos", C.c_int), ("n_foreign", C.c_int),
                ("foreign_pos", C.POINTER(C.c_int32)), ("subpixel_yx", C.POINTER(C.c_float))]


class ShardBufs(C.Structure):
    """ptycho_shard_bufs (include/ptycho_b200.h)."""
    _fields_ = [("c_canvas", C.c_void_p), ("probe_sums", C.c_void_p), ("sum_I", C.c_void_p), ("err_hist", C.c_void_p),
                ("row0", C.c_int), ("row1", C.c_int)]


def build(force: bool = False, verbose: bool = False) -> str:
    """nvcc the CUDA library in-tree for sm_100a (cross-compiles without a GPU)."""
    srcs = [os.path.join(_CSRC, f) for f in ("ptycho_api.cu", "kernels.cuh", "fft_core.cuh", "dm_mega.cuh", "dm_det.cuh")]
    srcs.append(os.path.join(os.path.dirname(_HERE), "include", "ptycho_b200.h"))
    if not force and os.path.exists(LIB_PATH) and all(os.path.getmtime(LIB_PATH) >= os.path.getmtime(s) for s in srcs):
        return LIB_PATH
    cmd = ["nvcc", *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), *([f"-DPTYCHO_ONLY_N={_ONLY_N}"] if _ONLY_N else []), *os.environ.get("PTYCHO_BUILD_DEFS", "").split(),
           srcs[0], "-o", LIB_PATH]
    subprocess.check_call(cmd, cwd=_CSRC)
    return LIB_PATH


_lib = None


def lib():
    """Load the C-ABI library (does not need a GPU; calls do)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise PtychoError(5, f"{LIB_PATH} not built; run `python -c 'import __graft_entry__ as g; g.build()'`")
        l = C.CDLL(LIB_PATH)
        l.ptycho_workspace_bytes.restype = C.c_size_t
        l.ptycho_workspace_bytes.argtypes = [C.c_int] * 5 + [C.c_int, C.c_int, C.POINTER(Params)]
        l.ptycho_init.argtypes = [C.POINTER(C.c_void_p), C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_int, C.c_int,
                                  C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.POINTER(Params), C.c_void_p,
                                  C.c_size_t, C.c_void_p]
        l.ptycho_iterate.argtypes = [C.c_void_p, C.c_int, C.c_int]
        for f in ("ptycho_fetch_object", "ptycho_fetch_probe", "ptycho_set_object", "ptycho_set_probe",
                  "ptycho_set_exit_waves"):
            getattr(l, f).argtypes = [C.c_void_p, C.c_void_p]
        l.ptycho_fetch_error.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.POINTER(C.c_int)]
        l.ptycho_fetch_steps.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.POINTER(C.c_int)]
        l.ptycho_fetch_exit_waves.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]
        l.ptycho_revised_waves.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]
        l.ptycho_eval_error.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        l.ptycho_profile.argtypes = [C.c_void_p, C.c_int]
        l.ptycho_profile_fetch.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
        l.ptycho_launch_count.restype = C.c_longlong
        l.ptycho_launch_count.argtypes = [C.c_void_p]
        l.ptycho_last_error.restype = C.c_char_p
        l.ptycho_last_error.argtypes = [C.c_void_p]
        l.ptycho_destroy.argtypes = [C.c_void_p]
        l.ptycho_append_frames.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p]
        l.ptycho_wait_frames.argtypes = [C.c_void_p]
        l.ptycho_orthogonalize_modes.argtypes = [C.c_void_p]
        l.ptycho_frames_present.argtypes = [C.c_void_p]
        l.ptycho_shard_buffers.argtypes = [C.c_void_p, C.POINTER(ShardBufs)]
        l.ptycho_shard_begin.argtypes = [C.c_void_p]
        l.ptycho_shard_end.argtypes = [C.c_void_p]
        l.ptycho_default_params.argtypes = [C.POINTER(Params)]
        l.ptycho_test_fft2.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p]
        l.ptycho_prepare_frames.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_float,
                                            C.c_float, C.c_int, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]
        _lib = l
    return _lib


def default_params(**over) -> Params:
    p = Params()
    lib().ptycho_default_params(C.byref(p))
    keep = None
    for k, v in over.items():
        if k == "batch_order":
            if v is not None:
                keep = np.ascontiguousarray(v, np.int32)
                p.batch_order = keep.ctypes.data_as(C.POINTER(C.c_int32))
        elif k == "subpixel_yx":
            if v is not None:
                p._keep_sub = np.ascontiguousarray(v, np.float32).reshape(-1, 2)
                p.subpixel_yx = p._keep_sub.ctypes.data_as(C.POINTER(C.c_float))
        elif k == "foreign_pos":
            if v is not None and len(v):
                p._keep_foreign = np.ascontiguousarray(v, np.int32).reshape(-1, 2)
                p.foreign_pos = p._keep_foreign.ctypes.data_as(C.POINTER(C.c_int32))
                p.n_foreign = p._keep_foreign.shape[0]
        else:
            if not hasattr(p, k):
                raise KeyError(k)
            setattr(p, k, v)
    p._keep = keep
    return p


def _ptr(a):
    """Host numpy array or torch tensor (host or device) -> raw pointer."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"]
        return C.c_void_p(a.ctypes.data)
    assert a.is_contiguous()
    return C.c_void_p(a.data_ptr())


def _c64(a):
    if isinstance(a, np.ndarray):
        return np.ascontiguousarray(a, np.complex64)
    return a.contiguous()


class Ptycho:
    """One reconstruction context (ptycho_ctx).  Arrays may be numpy (host) or torch (host/device)."""

    def __init__(self, obj, probe, pos, intensities, params: Params | None = None, stream=None, device="cuda:0", stream_dtype=None):
        """intensities = None with stream_dtype (np.uint16 / np.float32): a streaming context, frames come through append_frames."""
        import torch
        if not torch.cuda.is_available():
            raise PtychoError(5, "no CUDA device: the projection cycle has no CPU path")
        self._l = lib()
        self._torch = torch
        self.device = torch.device(device)
        obj, probe = _c64(obj), _c64(probe)
        if probe.ndim == 2:
            probe = probe[None]
        self.H, self.W = obj.shape
        self.K, self.n = probe.shape[0], probe.shape[-1]
        pos = np.ascontiguousarray(pos, np.int32) if isinstance(pos, np.ndarray) else pos.contiguous()
        self.J = pos.shape[0]
        dt = np.dtype(stream_dtype) if intensities is None else intensities.dtype
        self.itype = 1 if str(dt).endswith("uint16") else 0
        if self.itype == 0:
            assert str(dt).endswith("float32"), "intensities must be float32 or uint16"
        self._I = intensities if not isinstance(intensities, np.ndarray) else np.ascontiguousarray(intensities)
        on_host = 2 if intensities is None else (isinstance(self._I, np.ndarray) or not self._I.is_cuda)
        self.params = params if params is not None else default_params()
        need = self._l.ptycho_workspace_bytes(self.H, self.W, self.n, self.K, self.J, self.itype, int(on_host),
                                              C.byref(self.params))
        if need == 0:
            raise PtychoError(1, "invalid sizes")
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(need, dtype=torch.uint8, device=self.device)
            self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            h = C.c_void_p()
            st = self._l.ptycho_init(C.byref(h), _ptr(obj), self.H, self.W, _ptr(probe), self.K, self.n, _ptr(pos),
                                     self.J, _ptr(self._I), self.itype, C.byref(self.params),
                                     C.c_void_p(self.workspace.data_ptr()), need, C.c_void_p(self._stream.cuda_stream))
        if st != 0:
            raise PtychoError(st, "ptycho_init: " + lib().ptycho_last_error(None).decode())
        self._h = h

    # ---- the calls of the C ABI, same names -------------------------------------------------
    def append_frames(self, first_frame: int, intensities):
        intensities = intensities if not isinstance(intensities, np.ndarray) else np.ascontiguousarray(intensities)
        self._keep = intensities                                # must stay valid until wait_frames()
        self._check(self._l.ptycho_append_frames(self._h, int(first_frame), int(intensities.shape[0]), _ptr(intensities)))

    def orthogonalize_modes(self):
        self._check(self._l.ptycho_orthogonalize_modes(self._h))

    def shard_buffers(self) -> dict:
        """ptycho_shard_buffers as torch views of the workspace: c_canvas (H, W, 2) float32 (re, im), probe_sums (3 n^2,) float32,
        sum_I (1,) float64, err_hist float64, and the covered rows (row0, row1)."""
        b = ShardBufs()
        self._check(self._l.ptycho_shard_buffers(self._h, C.byref(b)))
        base, torch = self.workspace.data_ptr(), self._torch

        def view(ptr, nbytes, dtype):
            off = ptr - base
            assert 0 <= off and off + nbytes <= self.workspace.numel()
            return self.workspace[off:off + nbytes].view(dtype)
        return {"c_canvas": view(b.c_canvas, self.H * self.W * 8, torch.float32).view(self.H, self.W, 2),
                "probe_sums": view(b.probe_sums, 3 * self.n * self.n * 4, torch.float32),
                "sum_I": view(b.sum_I, 8, torch.float64), "err_hist": view(b.err_hist, 8 * 65536, torch.float64),
                "row0": b.row0, "row1": b.row1}

    def shard_begin(self):
        self._check(self._l.ptycho_shard_begin(self._h))

    def shard_end(self):
        self._check(self._l.ptycho_shard_end(self._h))

    def wait_frames(self):
        self._check(self._l.ptycho_wait_frames(self._h))

    def frames_present(self) -> int:
        return int(self._l.ptycho_frames_present(self._h))

    def _check(self, st):
        if st != 0:
            raise PtychoError(st, self._l.ptycho_last_error(self._h).decode())

    def iterate(self, alg: str | int, n_iters: int = 1):
        self._check(self._l.ptycho_iterate(self._h, ALG[alg] if isinstance(alg, str) else alg, n_iters))
        return self

    def _out(self, shape, out, dtype=np.complex64):
        return np.empty(shape, dtype) if out is None else out

    def fetch_object(self, out=None):
        out = self._out((self.H, self.W), out)
        self._check(self._l.ptycho_fetch_object(self._h, _ptr(out)))
        return out

    def fetch_probe(self, out=None):
        out = self._out((self.K, self.n, self.n), out)
        self._check(self._l.ptycho_fetch_probe(self._h, _ptr(out)))
        return out

    def fetch_error(self, cap: int = 65536):
        buf = np.zeros(cap, np.float64)
        n = C.c_int()
        self._check(self._l.ptycho_fetch_error(self._h, _ptr(buf), cap, C.byref(n)))
        return buf[: min(n.value, cap)]

    def fetch_steps(self, cap: int = 1 << 18):
        buf = np.zeros((cap, 2), np.float64)
        n = C.c_int()
        self._check(self._l.ptycho_fetch_steps(self._h, _ptr(buf), cap, C.byref(n)))
        return buf[: min(n.value, cap)]

    def fetch_exit_waves(self, idx=None, out=None):
        idx = np.arange(self.J, dtype=np.int32) if idx is None else np.ascontiguousarray(idx, np.int32)
        out = self._out((len(idx), self.K, self.n, self.n), out)
        self._check(self._l.ptycho_fetch_exit_waves(self._h, _ptr(idx), len(idx), _ptr(out)))
        return out

    def revised_waves(self, idx=None, out=None):
        idx = np.arange(self.J, dtype=np.int32) if idx is None else np.ascontiguousarray(idx, np.int32)
        out = self._out((len(idx), self.K, self.n, self.n), out)
        self._check(self._l.ptycho_revised_waves(self._h, _ptr(idx), len(idx), _ptr(out)))
        return out

    def set_object(self, obj):
        obj = _c64(obj)
        assert tuple(obj.shape) == (self.H, self.W)
        self._check(self._l.ptycho_set_object(self._h, _ptr(obj)))

    def set_probe(self, probe):
        probe = _c64(probe)
        assert probe.size == self.K * self.n * self.n if isinstance(probe, np.ndarray) else True
        self._check(self._l.ptycho_set_probe(self._h, _ptr(probe)))

    def set_exit_waves(self, psi):
        psi = _c64(psi)
        assert tuple(psi.shape) == (self.J, self.K, self.n, self.n)
        self._check(self._l.ptycho_set_exit_waves(self._h, _ptr(psi)))

    def eval_error(self) -> float:
        v = C.c_double()
        self._check(self._l.ptycho_eval_error(self._h, C.byref(v)))
        return v.value

    def profile(self, enable: bool = True):
        self._check(self._l.ptycho_profile(self._h, int(enable)))

    def profile_fetch(self) -> dict:
        """{class name: (total device ms, launches)} since the last profile(True)."""
        out = {}
        for i, name in enumerate(KCLASS):
            ms, n = C.c_double(), C.c_longlong()
            self._check(self._l.ptycho_profile_fetch(self._h, i, C.byref(ms), C.byref(n)))
            out[name] = (ms.value, n.value)
        return out

    def launch_count(self) -> int:
        return int(self._l.ptycho_launch_count(self._h))

    def synchronize(self):
        self._stream.synchronize()

    def destroy(self):
        if getattr(self, "_h", None):
            self._stream.synchronize()
            self._l.ptycho_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def prepare_frames(raw, center, n: int, threshold: float = 0.0, saturation: float = 0.0, out_dtype=np.uint16, out=None,
                   rot90: int = 0, frame_scale=None):
    """ptycho_prepare_frames: raw detector frames (F, det_h, det_w), uint16 or float32, numpy or torch CUDA ->
    FFT-order intensities (F, n, n) with masked pixels as the sentinel.  Marshalling only."""
    import torch
    is_t = isinstance(raw, torch.Tensor)
    itype = lambda dt: 1 if dt in (np.uint16, torch.uint16, np.dtype(np.uint16)) else 0
    if not is_t:
        raw = np.ascontiguousarray(raw)
        assert raw.dtype in (np.uint16, np.float32)
    f, dh, dw = raw.shape
    if out is None:
        out = (torch.empty((f, n, n), dtype=torch.uint16 if itype(out_dtype) else torch.float32, device=raw.device) if is_t
               else np.empty((f, n, n), np.uint16 if itype(out_dtype) else np.float32))
    stream = torch.cuda.current_stream().cuda_stream if torch.cuda.is_available() else 0
    if frame_scale is not None and not is_t:
        frame_scale = np.ascontiguousarray(frame_scale, np.float32)
    st = lib().ptycho_prepare_frames(_ptr(raw), itype(raw.dtype), f, dh, dw, int(center[0]), int(center[1]), int(n), float(threshold),
                                     float(saturation), int(rot90), _ptr(frame_scale), _ptr(out), itype(out.dtype), C.c_void_p(stream))
    if st != 0:
        raise PtychoError(st, "ptycho_prepare_frames")
    return out


def test_fft2(data, inverse: bool = False):
    """ptycho_test_fft2: batched in-place 2-D FFT of a torch CUDA complex64 tensor (count, n, n)."""
    import torch
    assert data.is_cuda and data.dtype == torch.complex64 and data.is_contiguous()
    st = lib().ptycho_test_fft2(C.c_void_p(data.data_ptr()), data.shape[-1], int(data.numel() // data.shape[-1] ** 2),
                                int(inverse), C.c_void_p(torch.cuda.current_stream().cuda_stream))
    if st != 0:
        raise PtychoError(st, "ptycho_test_fft2")
    return data


def fft2_noalloc(data, inverse: bool = False):
    """ptycho_fft2_noalloc: the same batched in-place 2-D FFT as test_fft2, with the kernels' scratch (the twiddle tables) in a
    static device array of the library: no cudaMalloc / cudaFree, no host-to-device copy, no synchronisation.  Asynchronous on
    torch's current stream.  n <= PTYCHO_NOALLOC_MAX_N = 512; calls that overlap on the GPU with different n race on the scratch."""
    import torch
    assert data.is_cuda and data.dtype == torch.complex64 and data.is_contiguous()
    l = lib()
    l.ptycho_fft2_noalloc.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p]
    with torch.cuda.device(data.device):
        st = l.ptycho_fft2_noalloc(C.c_void_p(data.data_ptr()), data.shape[-1], int(data.numel() // data.shape[-1] ** 2),
                                   int(inverse), C.c_void_p(torch.cuda.current_stream().cuda_stream))
    if st != 0:
        raise PtychoError(st, l.ptycho_last_error(None).decode())
    return data


def test_fft_rows(data, impl: int = 0):
    """ptycho_test_fft_rows: forward 1-D FFT of every row of a torch CUDA complex64 tensor (count, n, n), in place; impl 0 = the
    product's packed-fp32 line FFT, impl 1 = tensor-core DFT (n = 256).  Asynchronous on torch's current stream."""
    import torch
    assert data.is_cuda and data.dtype == torch.complex64 and data.is_contiguous()
    l = lib()
    l.ptycho_test_fft_rows.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p]
    with torch.cuda.device(data.device):
        st = l.ptycho_test_fft_rows(C.c_void_p(data.data_ptr()), data.shape[-1], int(data.numel() // data.shape[-1] ** 2), int(impl),
                                    C.c_void_p(torch.cuda.current_stream().cuda_stream))
    if st != 0:
        raise PtychoError(st, l.ptycho_last_error(None).decode())
    return data
