"""Thin Python binding of libqcldpc (include/qcldpc.h): argument marshalling only.

Every step of the decode runs in the CUDA kernels of csrc/qcldpc.cu; PyTorch is used for device memory and streams.
There is no CPU fallback: importing this module without csrc/libqcldpc.so raises, and so does every call on a box
without a CUDA device.
"""
from __future__ import annotations

import ctypes
import os
from typing import NamedTuple, Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
SO_PATH = os.path.join(_HERE, "csrc", "libqcldpc.so")

EXPORTED_SYMBOLS = (
    "qcldpc_code_create", "qcldpc_code_create_sparse", "qcldpc_code_destroy", "qcldpc_code_info", "qcldpc_workspace_bytes", "qcldpc_decode",
    "qcldpc_decode_ex",
    "qcldpc_host_workspace_bytes", "qcldpc_decode_host", "qcldpc_decode_host_ex", "qcldpc_last_launch_count", "qcldpc_status_string",
    "qcldpc_last_cuda_error", "qcldpc_profile_enable", "qcldpc_profile_collect",
    "qcldpc_llr_init", "qcldpc_pack_bits", "qcldpc_crc32_check", "qcldpc_iterations_issued", "qcldpc_last_loop_mode",
    "qcldpc_decode_static", "qcldpc_static_workspace_bytes",
)

if not os.path.exists(SO_PATH):
    raise ImportError(f"{SO_PATH} is missing: build it with `python -m paper_1702_07740_b200.build` "
                      "(there is no CPU fallback)")

_lib = ctypes.CDLL(SO_PATH)
_vp, _i, _sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_size_t
_lib.qcldpc_code_create.restype = _i
_lib.qcldpc_code_create.argtypes = [_vp, _i, _i, _i, ctypes.POINTER(_vp)]
_lib.qcldpc_code_create_sparse.restype = _i
_lib.qcldpc_code_create_sparse.argtypes = [_vp, _vp, _vp, ctypes.c_int64, _i, _i, _i, ctypes.POINTER(_vp)]
_lib.qcldpc_code_destroy.restype = None
_lib.qcldpc_code_destroy.argtypes = [_vp]
_lib.qcldpc_code_info.restype = _i
_lib.qcldpc_code_info.argtypes = [_vp, ctypes.POINTER(ctypes.c_int64), ctypes.POINTER(ctypes.c_int64),
                                  ctypes.POINTER(ctypes.c_int64)]
_lib.qcldpc_workspace_bytes.restype = _sz
_lib.qcldpc_workspace_bytes.argtypes = [_vp, _i]
_lib.qcldpc_host_workspace_bytes.restype = _sz
_lib.qcldpc_host_workspace_bytes.argtypes = [_vp, _i, _i]
_DECODE_ARGS = [_vp, _vp, _vp, _i, _i, _i, _vp, _vp, _vp, _vp, _vp, _sz, _vp]
_lib.qcldpc_decode.restype = _i
_lib.qcldpc_decode.argtypes = _DECODE_ARGS
_lib.qcldpc_decode_ex.restype = _i
_lib.qcldpc_decode_ex.argtypes = [_vp, _vp, _vp, _i, _i, _i, _i, _vp, _vp, _vp, _vp, _vp, _sz, _vp]
_lib.qcldpc_decode_host.restype = _i
_lib.qcldpc_decode_host.argtypes = _DECODE_ARGS
_lib.qcldpc_decode_host_ex.restype = _i
_lib.qcldpc_decode_host_ex.argtypes = _lib.qcldpc_decode_ex.argtypes
_lib.qcldpc_last_launch_count.restype = ctypes.c_int64
_lib.qcldpc_last_launch_count.argtypes = []
_lib.qcldpc_profile_enable.restype = _i
_lib.qcldpc_profile_enable.argtypes = [_i]
_lib.qcldpc_profile_collect.restype = _i
_lib.qcldpc_profile_collect.argtypes = [ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int64),
                                        ctypes.POINTER(ctypes.c_int64)]
_lib.qcldpc_llr_init.restype = _i
_lib.qcldpc_llr_init.argtypes = [_vp, _vp, _vp, _i, ctypes.c_int64, _i, _i, _vp, _vp]
_lib.qcldpc_pack_bits.restype = _i
_lib.qcldpc_pack_bits.argtypes = [_vp, _i, ctypes.c_int64, ctypes.c_int64, _vp, _vp]
_lib.qcldpc_crc32_check.restype = _i
_lib.qcldpc_crc32_check.argtypes = [_vp, _i, ctypes.c_int64, ctypes.c_int64, _vp, _vp, _vp]
_lib.qcldpc_iterations_issued.restype = _i
_lib.qcldpc_iterations_issued.argtypes = [_vp, _i, _vp, _vp, ctypes.POINTER(_i)]
_lib.qcldpc_last_loop_mode.restype = _i
_lib.qcldpc_last_loop_mode.argtypes = []
_lib.qcldpc_decode_static.restype = _i
_lib.qcldpc_decode_static.argtypes = [_vp, _vp, _vp, _i, _i, _i, _i, _vp, _vp, _vp, _vp, _vp]
_lib.qcldpc_static_workspace_bytes.restype = _sz
_lib.qcldpc_static_workspace_bytes.argtypes = []
_lib.qcldpc_status_string.restype = ctypes.c_char_p
_lib.qcldpc_status_string.argtypes = [_i]
_lib.qcldpc_last_cuda_error.restype = ctypes.c_char_p
_lib.qcldpc_last_cuda_error.argtypes = []


class QCLDPCError(RuntimeError):
    def __init__(self, status: int, where: str, with_detail: bool = False):
        self.status = status
        text = _lib.qcldpc_status_string(status).decode()
        detail = _lib.qcldpc_last_cuda_error().decode()
        super().__init__(f"{where}: {text} ({status})" +
                         (f": {detail}" if detail and (status == -4 or with_detail) else ""))


def _check(status: int, where: str) -> None:
    if status != 0:
        raise QCLDPCError(status, where)


def qcldpc_status_string(status: int) -> str:
    return _lib.qcldpc_status_string(status).decode()


def qcldpc_last_launch_count() -> int:
    return int(_lib.qcldpc_last_launch_count())


def qcldpc_last_loop_mode() -> int:
    """1: the last decode of this thread ran as one graph with the loop on the device; 0: one launch per iteration."""
    return int(_lib.qcldpc_last_loop_mode())


def qcldpc_static_workspace_bytes() -> int:
    """Bytes of the library's own device workspace (per GPU), the limit of QCLDPCCode.decode_static."""
    return int(_lib.qcldpc_static_workspace_bytes())


def qcldpc_profile_enable(stride: int) -> None:
    _check(_lib.qcldpc_profile_enable(int(stride)), "qcldpc_profile_enable")


def qcldpc_profile_collect():
    """{kind: (ms_sum, timed, launched)} for kind in ("pass", "cand")."""
    ms = (ctypes.c_double * 2)()
    timed = (ctypes.c_int64 * 2)()
    launched = (ctypes.c_int64 * 2)()
    _check(_lib.qcldpc_profile_collect(ms, timed, launched), "qcldpc_profile_collect")
    return {name: (ms[k], timed[k], launched[k]) for k, name in enumerate(("pass", "cand"))}


def _check_host_array(a, name, np_dtype, torch):
    """A HOST array the C ABI can read as it is: right dtype, C-contiguous, not a device tensor."""
    if isinstance(a, torch.Tensor):
        want = {np.float32: torch.float32, np.uint8: torch.uint8, np.int32: torch.int32}[np_dtype]
        if a.is_cuda or a.dtype != want or not a.is_contiguous():
            raise ValueError(f"{name}: need a contiguous host tensor of dtype {want}, got {a.dtype} on {a.device}")
    elif isinstance(a, np.ndarray):
        if a.dtype != np_dtype or not a.flags["C_CONTIGUOUS"]:
            raise ValueError(f"{name}: need a C-contiguous numpy array of dtype {np.dtype(np_dtype)}, got {a.dtype}")
    else:
        raise ValueError(f"{name}: need a numpy array or a host torch tensor")


def _check_outputs(out, F, n, torch, cuda: bool):
    """Caller-provided output buffers: shapes, dtypes, contiguity, residency."""
    spec = (("hard", (F, n), np.uint8), ("iters", (F,), np.int32), ("passed", (F,), np.uint8),
            ("posterior", (F, n), np.float32))
    for (name, shape, dt), a in zip(spec, out):
        if a is None:
            if name != "posterior":
                raise ValueError(f"out.{name} is missing")
            continue
        if tuple(a.shape) != shape:
            raise ValueError(f"out.{name}: shape {tuple(a.shape)}, need {shape}")
        if cuda:
            want = {np.float32: torch.float32, np.uint8: torch.uint8, np.int32: torch.int32}[dt]
            if not (isinstance(a, torch.Tensor) and a.is_cuda and a.dtype == want and a.is_contiguous()):
                raise ValueError(f"out.{name}: need a contiguous CUDA tensor of dtype {want}")
        else:
            _check_host_array(a, f"out.{name}", dt, torch)


class DecodeResult(NamedTuple):
    hard: "object"        # uint8  [F][n]
    iters: "object"       # int32  [F]
    passed: "object"      # uint8  [F]
    posterior: "object"   # float32 [F][n] or None


class QCLDPCCode:
    """Owns a qcldpc_code_t handle (qcldpc_code_create / qcldpc_code_destroy)."""

    def __init__(self, base_shifts: np.ndarray, Z: int):
        base = np.ascontiguousarray(base_shifts, dtype=np.int32)
        if base.ndim != 2:
            raise ValueError("base_shifts must be [mb][nb]")
        self.mb, self.nb = base.shape
        self.Z = int(Z)
        self._handle = _vp()
        _check(_lib.qcldpc_code_create(base.ctypes.data, self.mb, self.nb, self.Z, ctypes.byref(self._handle)),
               "qcldpc_code_create")
        self._read_info()
        self._device = self._current_device()

    @staticmethod
    def _current_device():
        """The CUDA device the handle's tables were allocated on (the one current at creation)."""
        import torch
        return torch.device("cuda", torch.cuda.current_device())

    def _require_device(self, dev):
        import torch
        dev = torch.device(dev)
        if dev.type != "cuda" or (dev.index if dev.index is not None else torch.cuda.current_device()) != self._device.index:
            raise ValueError(f"this code handle lives on {self._device}; got buffers on {dev}")

    def _read_info(self):
        n, m, e = ctypes.c_int64(), ctypes.c_int64(), ctypes.c_int64()
        _check(_lib.qcldpc_code_info(self._handle, ctypes.byref(n), ctypes.byref(m), ctypes.byref(e)),
               "qcldpc_code_info")
        self.n, self.m, self.active_base_edges = n.value, m.value, e.value

    @classmethod
    def from_sparse(cls, rows: np.ndarray, cols: np.ndarray, shifts: np.ndarray, mb: int, nb: int, Z: int):
        """qcldpc_code_create_sparse: the non-zero blocks (rows[k], cols[k]) with shift shifts[k]."""
        self = cls.__new__(cls)
        r = np.ascontiguousarray(rows, dtype=np.int32)
        c = np.ascontiguousarray(cols, dtype=np.int32)
        p = np.ascontiguousarray(shifts, dtype=np.int32)
        if not (r.ndim == c.ndim == p.ndim == 1 and len(r) == len(c) == len(p)):
            raise ValueError("rows, cols, shifts must be 1-D arrays of one length")
        self.mb, self.nb, self.Z = int(mb), int(nb), int(Z)
        self._handle = _vp()
        _check(_lib.qcldpc_code_create_sparse(r.ctypes.data, c.ctypes.data, p.ctypes.data, len(r), self.mb, self.nb,
                                              self.Z, ctypes.byref(self._handle)), "qcldpc_code_create_sparse")
        self._read_info()
        self._device = self._current_device()
        return self

    def __del__(self):
        h = getattr(self, "_handle", None)
        if h and _lib is not None:          # _lib is None while the interpreter shuts down
            _lib.qcldpc_code_destroy(h)
            self._handle = None

    # ---------------------------------------------------------------------------------------------- sizes
    def workspace_bytes(self, n_frames: int) -> int:
        return int(_lib.qcldpc_workspace_bytes(self._handle, int(n_frames)))

    def host_workspace_bytes(self, n_frames: int, want_posterior: bool) -> int:
        return int(_lib.qcldpc_host_workspace_bytes(self._handle, int(n_frames), int(bool(want_posterior))))

    def iterations_issued(self, n_frames: int, workspace, stream=None) -> int:
        """qcldpc_iterations_issued: iterations whose launches the last decode in `workspace` issued (waits)."""
        import torch
        st = stream if stream is not None else torch.cuda.current_stream(workspace.device)
        n = _i(0)
        with torch.cuda.device(workspace.device):
            _check(_lib.qcldpc_iterations_issued(self._handle, int(n_frames), workspace.data_ptr(), st.cuda_stream,
                                                 ctypes.byref(n)), "qcldpc_iterations_issued")
        return n.value

    # ---------------------------------------------------------------------------------------------- decode
    def decode(self, llr, syndrome, max_iter: int, early_stop: int, want_posterior: bool = True,
               workspace=None, out: Optional[DecodeResult] = None, stream=None,
               check_from_iter: int = 1) -> DecodeResult:
        """qcldpc_decode_ex on device tensors: llr float32 [F][n], syndrome uint8 [F][m] (torch, cuda, contiguous).

        Only enqueues work on `stream` (default: torch's current stream).  check_from_iter = 1 is qcldpc_decode."""
        import torch
        if not (llr.is_cuda and syndrome.is_cuda):
            raise ValueError("qcldpc_decode needs CUDA tensors (no CPU fallback)")
        if llr.dtype != torch.float32 or syndrome.dtype != torch.uint8:
            raise ValueError("llr must be float32 and syndrome uint8")
        llr = llr.contiguous()
        syndrome = syndrome.contiguous()
        if llr.dim() != 2 or llr.shape[1] != self.n or tuple(syndrome.shape) != (llr.shape[0], self.m):
            raise ValueError(f"shapes {tuple(llr.shape)} / {tuple(syndrome.shape)} do not match n={self.n}, m={self.m}")
        F = llr.shape[0]
        dev = llr.device
        self._require_device(dev)
        if syndrome.device != dev:
            raise ValueError("llr and syndrome must live on one device")
        st = stream if stream is not None else torch.cuda.current_stream(dev)
        need = self.workspace_bytes(F)
        own = []                                        # tensors allocated here and used on `st`
        if workspace is None:
            workspace = torch.empty(need, dtype=torch.uint8, device=dev)
            own.append(workspace)
        else:
            self._require_device(workspace.device)
        if out is None:
            out = DecodeResult(torch.empty((F, self.n), dtype=torch.uint8, device=dev),
                               torch.empty(F, dtype=torch.int32, device=dev),
                               torch.empty(F, dtype=torch.uint8, device=dev),
                               torch.empty((F, self.n), dtype=torch.float32, device=dev) if want_posterior else None)
            own.extend(t for t in out if t is not None)
        else:
            _check_outputs(out, F, self.n, torch, cuda=True)
        # the call only enqueues: tell the caching allocator that these blocks are in use on `st`, so that a block
        # dropped by the caller (the internal workspace on return) is not handed out again before the decode has run
        for t in own + [llr, syndrome]:
            t.record_stream(st)
        with torch.cuda.device(dev):
            rc = _lib.qcldpc_decode_ex(self._handle, llr.data_ptr(), syndrome.data_ptr(), F, int(max_iter),
                                       int(early_stop), int(check_from_iter), out.hard.data_ptr(),
                                       out.iters.data_ptr(), out.passed.data_ptr(),
                                       out.posterior.data_ptr() if out.posterior is not None else None,
                                       workspace.data_ptr(), workspace.numel(), st.cuda_stream)
        _check(rc, "qcldpc_decode_ex")
        return out

    def decode_static(self, llr, syndrome, max_iter: int, early_stop: int, out: DecodeResult, stream=None,
                      check_from_iter: int = 1) -> DecodeResult:
        """qcldpc_decode_static: the decode without any allocation, here or in the library.  The caller passes the
        inputs AND the outputs (`out`, torch CUDA tensors, contiguous; out.posterior may be None); the workspace is the
        library's own device array (qcldpc_static_workspace_bytes() per GPU, shared by every call on that GPU: calls
        that overlap on the GPU race on it).  Raises QCLDPCError (QCLDPC_ERR_WORKSPACE) if this code and batch need more
        than that.  Only enqueues plain launches on `stream` (default: torch's current stream)."""
        import torch
        _cuda_tensor(llr, "llr", torch.float32, torch)
        _cuda_tensor(syndrome, "syndrome", torch.uint8, torch)
        if llr.dim() != 2 or llr.shape[1] != self.n or tuple(syndrome.shape) != (llr.shape[0], self.m):
            raise ValueError(f"shapes {tuple(llr.shape)} / {tuple(syndrome.shape)} do not match n={self.n}, m={self.m}")
        F = llr.shape[0]
        dev = llr.device
        self._require_device(dev)
        if syndrome.device != dev:
            raise ValueError("llr and syndrome must live on one device")
        _check_outputs(out, F, self.n, torch, cuda=True)
        st = stream if stream is not None else torch.cuda.current_stream(dev)
        with torch.cuda.device(dev):
            rc = _lib.qcldpc_decode_static(self._handle, llr.data_ptr(), syndrome.data_ptr(), F, int(max_iter),
                                           int(early_stop), int(check_from_iter), out.hard.data_ptr(),
                                           out.iters.data_ptr(), out.passed.data_ptr(),
                                           out.posterior.data_ptr() if out.posterior is not None else None,
                                           st.cuda_stream)
        if rc != 0:
            raise QCLDPCError(rc, "qcldpc_decode_static", with_detail=True)   # (the sizes, for QCLDPC_ERR_WORKSPACE)
        return out

    def decode_host(self, llr: np.ndarray, syndrome: np.ndarray, max_iter: int, early_stop: int,
                    want_posterior: bool = False, workspace=None, out=None, stream=None, check_from_iter: int = 1):
        """qcldpc_decode_host_ex on HOST arrays (numpy or pinned torch CPU tensors; float32 / uint8, C-contiguous);
        returns host outputs.

        Host<->device copies happen inside the call; it returns after the stream has drained."""
        import torch

        def ptr(a):
            return a.data_ptr() if isinstance(a, torch.Tensor) else a.ctypes.data

        _check_host_array(llr, "llr", np.float32, torch)
        _check_host_array(syndrome, "syndrome", np.uint8, torch)
        F = llr.shape[0]
        if tuple(llr.shape) != (F, self.n) or tuple(syndrome.shape) != (F, self.m):
            raise ValueError("bad host shapes")
        need = self.host_workspace_bytes(F, want_posterior)
        if workspace is None:
            workspace = torch.empty(need, dtype=torch.uint8, device=self._device)
        self._require_device(workspace.device)
        if out is None:
            out = DecodeResult(np.empty((F, self.n), dtype=np.uint8), np.empty(F, dtype=np.int32),
                               np.empty(F, dtype=np.uint8),
                               np.empty((F, self.n), dtype=np.float32) if want_posterior else None)
        else:
            _check_outputs(out, F, self.n, torch, cuda=False)
        st = stream if stream is not None else torch.cuda.current_stream(workspace.device)
        with torch.cuda.device(workspace.device):
            rc = _lib.qcldpc_decode_host_ex(self._handle, ptr(llr), ptr(syndrome), F, int(max_iter), int(early_stop),
                                            int(check_from_iter), ptr(out.hard), ptr(out.iters), ptr(out.passed),
                                            ptr(out.posterior) if out.posterior is not None else None,
                                            workspace.data_ptr(), workspace.numel(), st.cuda_stream)
        _check(rc, "qcldpc_decode_host_ex")
        return out


def _cuda_tensor(t, name, dtype, torch):
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise ValueError(f"{name}: need a contiguous CUDA tensor of dtype {dtype}")
    return t


def llr_init(r, x, sigma2_z, dim: int = 1, norm_power: int = 2, out=None, stream=None):
    """qcldpc_llr_init (P:344 Step 1): Q = 2 R / sigma_N^2 on device tensors r, x float32 [F][n] (x may be None for
    dim = 0), sigma2_z float32 [F].  Returns Q float32 [F][n]; only enqueues on `stream`."""
    import torch
    _cuda_tensor(r, "r", torch.float32, torch)
    _cuda_tensor(sigma2_z, "sigma2_z", torch.float32, torch)
    if x is not None:
        _cuda_tensor(x, "x", torch.float32, torch)
        if x.shape != r.shape:
            raise ValueError("r and x must have one shape")
    if r.dim() != 2 or sigma2_z.numel() != r.shape[0]:
        raise ValueError("r must be [F][n] and sigma2_z [F]")
    if out is None:
        out = torch.empty_like(r)
    _cuda_tensor(out, "out", torch.float32, torch)
    st = stream if stream is not None else torch.cuda.current_stream(r.device)
    with torch.cuda.device(r.device):
        rc = _lib.qcldpc_llr_init(r.data_ptr(), x.data_ptr() if x is not None else None, sigma2_z.data_ptr(),
                                  r.shape[0], r.shape[1], int(dim), int(norm_power), out.data_ptr(), st.cuda_stream)
    _check(rc, "qcldpc_llr_init")
    return out


def pack_bits(hard, n_bits: int, out=None, stream=None):
    """qcldpc_pack_bits: the first n_bits of every row of hard (uint8 [F][n], one byte per bit) as bits, most
    significant first; returns uint8 [F][(n_bits + 7) // 8]."""
    import torch
    _cuda_tensor(hard, "hard", torch.uint8, torch)
    F, n = hard.shape
    if out is None:
        out = torch.empty((F, (int(n_bits) + 7) // 8), dtype=torch.uint8, device=hard.device)
    _cuda_tensor(out, "out", torch.uint8, torch)
    st = stream if stream is not None else torch.cuda.current_stream(hard.device)
    with torch.cuda.device(hard.device):
        rc = _lib.qcldpc_pack_bits(hard.data_ptr(), F, n, int(n_bits), out.data_ptr(), st.cuda_stream)
    _check(rc, "qcldpc_pack_bits")
    return out


def crc32_check(packed, k_bits: int, stream=None):
    """qcldpc_crc32_check on packed frames uint8 [F][>= k_bits / 8]: (crc uint32-as-int64 [F], ok uint8 [F])."""
    import torch
    _cuda_tensor(packed, "packed", torch.uint8, torch)
    F, stride = packed.shape
    crc = torch.empty(F, dtype=torch.int32, device=packed.device)
    ok = torch.empty(F, dtype=torch.uint8, device=packed.device)
    st = stream if stream is not None else torch.cuda.current_stream(packed.device)
    with torch.cuda.device(packed.device):
        rc = _lib.qcldpc_crc32_check(packed.data_ptr(), F, stride, int(k_bits), crc.data_ptr(), ok.data_ptr(),
                                     st.cuda_stream)
    _check(rc, "qcldpc_crc32_check")
    return crc.to(torch.int64) & 0xFFFFFFFF, ok


def raw_lib():
    """The ctypes handle (tests use it to probe argument checking)."""
    return _lib
