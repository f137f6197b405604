"""Thin Python binding of the C ABI in include/flexmoe.h (same names, argument marshalling only).

torch is used for device memory and streams; every step of the path runs in the CUDA kernels of
csrc/.  There is no CPU fallback: if libflexmoe.so is missing or no CUDA device is present the calls
raise.  This module never imports oracle/.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
_SO = os.path.join(_HERE, "libflexmoe.so")
_SOURCES = ["fxm_api.cu", "fxm_aux.cu", "fxm_route.cu", "fxm_simt.cu", "fxm_pair.cu", "fxm_decode.cu", "fxm_rank.cu"]
_HEADERS = [os.path.join(_CSRC, "fxm_internal.cuh"), os.path.join(_CSRC, "fxm_ptx.cuh"), os.path.join(_HERE, "..", "include", "flexmoe.h")]

IMPL_TCGEN05 = 0
IMPL_SIMT_DEBUG = 1
MAX_BUDGETS = 15

_STATUS = ["FXM_OK", "FXM_EINVAL", "FXM_ESHAPE", "FXM_EPERM", "FXM_EBUDGET", "FXM_ENOTNESTED",
           "FXM_EWORKSPACE", "FXM_ESTATE", "FXM_ECUDA", "FXM_ENOMEM", "FXM_ELIMIT"]


class FxmError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        self.name = _STATUS[code] if 0 <= code < len(_STATUS) else f"FXM_{code}"
        super().__init__(f"{where}: {self.name}")


def build(force: bool = False, verbose: bool = False) -> str:
    """nvcc-compile csrc/*.cu for sm_100a into paper_2606_27866_b200/libflexmoe.so (in-tree)."""
    srcs = [os.path.join(_CSRC, s) for s in _SOURCES]
    deps = srcs + _HEADERS
    if not force and os.path.exists(_SO) and all(os.path.getmtime(_SO) >= os.path.getmtime(p) for p in deps):
        return _SO
    cmd = ["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
           "-Xcompiler", "-fPIC", "-shared", "-o", _SO] + srcs
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    subprocess.check_call(cmd)
    return _SO


_lib = None


def lib():
    """Load the shared library; (re)build it first when it is missing or older than its sources and nvcc exists."""
    global _lib
    if _lib is not None:
        return _lib
    import shutil
    if not os.path.exists(_SO) or shutil.which("nvcc"):
        build()                       # a no-op when the .so is newer than every source and header
    L = ctypes.CDLL(_SO)
    vp, i32, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_size_t
    L.fxm_packed_bytes.argtypes = [i32, i32, i32, ctypes.POINTER(sz)]
    L.fxm_workspace_bytes.argtypes = [i32, i32, i32, i32, i32, ctypes.POINTER(sz)]
    L.fxm_pack.argtypes = [ctypes.POINTER(vp), i32, i32, i32, vp, vp, vp, vp, vp, vp]
    L.fxm_set_budget.argtypes = [vp, vp, vp]
    L.fxm_register_budgets.argtypes = [vp, i32, vp, i32, vp]
    L.fxm_select_budget.argtypes = [vp, i32]
    L.fxm_ratio_to_width.argtypes = [i32, i32, i32]
    L.fxm_ratio_to_width.restype = ctypes.c_int32
    L.fxm_moe_ffn.argtypes = [vp, vp, vp, vp, i32, i32, vp, vp, sz, vp]
    L.fxm_moe_ffn_shared.argtypes = [vp, vp, vp, vp, i32, i32, vp, vp, vp, sz, vp]
    L.fxm_moe_ffn_router.argtypes = [vp, vp, vp, i32, i32, vp, vp, vp, vp, vp, sz, vp]
    L.fxm_clipped_bytes.argtypes = [i32, i32, i32, vp, ctypes.POINTER(sz)]
    L.fxm_export_clipped.argtypes = [vp, vp, vp, sz, vp]
    L.fxm_parse_clipped_header.argtypes = [vp, sz, ctypes.POINTER(i32), ctypes.POINTER(i32), ctypes.POINTER(i32), vp]
    L.fxm_load_clipped.argtypes = [ctypes.POINTER(vp), i32, i32, i32, vp, vp, sz, vp]
    L.fxm_workspace_bytes_host.argtypes = [i32, i32, i32, i32, i32, ctypes.POINTER(sz)]
    L.fxm_moe_ffn_host.argtypes = [vp, vp, vp, vp, i32, i32, vp, vp, sz, vp]
    L.fxm_moe_ffn_host_pipelined.argtypes = [vp, vp, vp, vp, i32, i32, vp, vp, sz, vp]
    L.fxm_host_flush.argtypes = [vp, vp]
    L.fxm_saliency_workspace_bytes.argtypes = [i32, i32, i32, ctypes.POINTER(sz)]
    L.fxm_saliency.argtypes = [i32, i32, i32, vp, vp, vp, vp, vp, vp, i32, vp, vp, sz, vp]
    L.fxm_saliency_static.argtypes = [i32, i32, i32, vp, vp, vp, vp, vp, vp, i32, vp, vp]
    L.fxm_rank_channels.argtypes = [i32, i32, vp, vp, vp]
    L.fxm_sample_budget.argtypes = [vp, vp, vp, i32, vp, i32, vp, vp]
    L.fxm_action_cost.argtypes = [vp, vp, i32, vp, i32, vp, vp, vp]
    L.fxm_profile_begin.argtypes = [vp, i32]
    L.fxm_profile_end.argtypes = [vp, ctypes.POINTER(ctypes.c_float), ctypes.POINTER(i32)]
    L.fxm_route.argtypes = [vp, vp, i32, i32, vp, vp, vp, vp, vp, sz, vp]
    L.fxm_unpack_prefix.argtypes = [vp, i32, i32, vp, vp, vp, vp]
    L.fxm_debug_read_h.argtypes = [vp, vp, i32, i32, vp, vp, i32, vp]
    L.fxm_set_impl.argtypes = [vp, i32]
    L.fxm_set_tile_n.argtypes = [vp, i32]
    L.fxm_set_decode.argtypes = [vp, i32, i32]
    L.fxm_device_flags.argtypes = [vp, ctypes.POINTER(ctypes.c_uint32), vp]
    L.fxm_launches_per_ffn.argtypes = [vp]
    L.fxm_status_string.argtypes = [i32]
    L.fxm_status_string.restype = ctypes.c_char_p
    L.fxm_destroy.argtypes = [vp]
    L.fxm_destroy.restype = None
    _lib = L
    return L


EXPORTS = ["fxm_packed_bytes", "fxm_workspace_bytes", "fxm_pack", "fxm_set_budget", "fxm_register_budgets",
           "fxm_select_budget", "fxm_ratio_to_width", "fxm_moe_ffn", "fxm_moe_ffn_shared", "fxm_moe_ffn_router", "fxm_workspace_bytes_host",
           "fxm_moe_ffn_host", "fxm_moe_ffn_host_pipelined", "fxm_host_flush", "fxm_clipped_bytes", "fxm_export_clipped", "fxm_parse_clipped_header", "fxm_load_clipped",
           "fxm_saliency_workspace_bytes", "fxm_saliency", "fxm_saliency_static", "fxm_rank_channels", "fxm_sample_budget", "fxm_action_cost",
           "fxm_profile_begin", "fxm_profile_end", "fxm_route", "fxm_unpack_prefix",
           "fxm_debug_read_h", "fxm_set_impl", "fxm_set_tile_n", "fxm_set_decode", "fxm_device_flags", "fxm_launches_per_ffn",
           "fxm_status_string", "fxm_destroy"]


def _chk(code: int, where: str):
    if code != 0:
        raise FxmError(code, where)


def packed_bytes(E: int, d: int, I: int) -> int:
    n = ctypes.c_size_t()
    _chk(lib().fxm_packed_bytes(E, d, I, ctypes.byref(n)), "fxm_packed_bytes")
    return n.value


def workspace_bytes(E: int, d: int, I: int, T_max: int, k: int) -> int:
    n = ctypes.c_size_t()
    _chk(lib().fxm_workspace_bytes(E, d, I, T_max, k, ctypes.byref(n)), "fxm_workspace_bytes")
    return n.value


def workspace_bytes_host(E: int, d: int, I: int, T_max: int, k: int) -> int:
    n = ctypes.c_size_t()
    _chk(lib().fxm_workspace_bytes_host(E, d, I, T_max, k, ctypes.byref(n)), "fxm_workspace_bytes_host")
    return n.value


N_KERNELS = 5
KERNEL_NAMES = ("route", "gemm1_swiglu", "gemm2_scatter_add", "finalize", "decode_fused")
DECODE_DEFAULT_MAX_ASSIGNMENTS = 640
DECODE_DEFAULT_PREFETCH = 0


def saliency(W_gate, W_up, W_down, G_gate, G_up, G_down, stream=None):
    """Eq. 2 (fxm_saliency).  CUDA bf16 tensors: weights [E,I,d],[E,I,d],[E,d,I]; gradients [B,E,I,d],[B,E,I,d],[B,E,d,I]
    -> s [E,I] fp32."""
    import torch
    E, I, d = W_gate.shape
    B = G_gate.shape[0]
    for t in (W_gate, W_up, W_down, G_gate, G_up, G_down):
        assert t.is_cuda and t.dtype == torch.bfloat16 and t.is_contiguous()
    assert tuple(W_down.shape) == (E, d, I) and tuple(G_gate.shape) == (B, E, I, d) and tuple(G_down.shape) == (B, E, d, I)
    n = ctypes.c_size_t()
    _chk(lib().fxm_saliency_workspace_bytes(E, d, I, ctypes.byref(n)), "fxm_saliency_workspace_bytes")
    ws = torch.empty(n.value, dtype=torch.uint8, device=W_gate.device)
    s = torch.empty((E, I), dtype=torch.float32, device=W_gate.device)
    _chk(lib().fxm_saliency(E, d, I, W_gate.data_ptr(), W_up.data_ptr(), W_down.data_ptr(), G_gate.data_ptr(),
                            G_up.data_ptr(), G_down.data_ptr(), B, s.data_ptr(), ws.data_ptr(), ws.numel(),
                            _stream_ptr(stream)), "fxm_saliency")
    return s


SALIENCY_STATIC_BYTES = 8 << 20


def saliency_static(W_gate, W_up, W_down, G_gate, G_up, G_down, out, stream=None):
    """Eq. 2 through fxm_saliency_static: no workspace argument, nothing allocated (the scratch is a fixed 8 MB device array
    inside the library).  `out`: a preallocated CUDA fp32 [E,I] tensor.  Raises FXM_ELIMIT for shapes beyond the scratch."""
    import torch
    E, I, d = W_gate.shape
    B = G_gate.shape[0]
    for t in (W_gate, W_up, W_down, G_gate, G_up, G_down):
        assert t.is_cuda and t.dtype == torch.bfloat16 and t.is_contiguous()
    assert tuple(W_down.shape) == (E, d, I) and tuple(G_gate.shape) == (B, E, I, d) and tuple(G_down.shape) == (B, E, d, I)
    assert out.is_cuda and out.dtype == torch.float32 and out.is_contiguous() and tuple(out.shape) == (E, I)
    _chk(lib().fxm_saliency_static(E, d, I, W_gate.data_ptr(), W_up.data_ptr(), W_down.data_ptr(), G_gate.data_ptr(),
                                   G_up.data_ptr(), G_down.data_ptr(), B, out.data_ptr(), _stream_ptr(stream)),
         "fxm_saliency_static")
    return out


def rank_channels(s, stream=None):
    """Eq. 3's permutation (fxm_rank_channels): s [E,I] fp32 CUDA -> channel_rank [E,I] int32 CUDA."""
    import torch
    E, I = s.shape
    assert s.is_cuda and s.dtype == torch.float32 and s.is_contiguous()
    out = torch.empty((E, I), dtype=torch.int32, device=s.device)
    _chk(lib().fxm_rank_channels(E, I, s.data_ptr(), out.data_ptr(), _stream_ptr(stream)), "fxm_rank_channels")
    return out


def ratio_to_width(I: int, num: int, den: int) -> int:
    return int(lib().fxm_ratio_to_width(I, num, den))


def _stream_ptr(stream=None):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


def _i32_host(a):
    import numpy as np
    return np.ascontiguousarray(a, dtype=np.int32)


class Layer:
    """One packed MoE layer.  Owns (via torch) the packed weight blob and a workspace."""

    def __init__(self, handle, E, d, I, packed, clipped_widths=None):
        self._h = handle
        self.E, self.d, self.I = E, d, I
        self.packed = packed            # torch.uint8 tensor; must outlive the handle
        self.clipped_widths = clipped_widths   # None for a full layer, else the exported r[E]
        self._ws = None
        self._ws_key = None

    # -- (1) pack ---------------------------------------------------------------------------------
    @staticmethod
    def pack(W_gate, W_up, W_down, channel_rank=None, stream=None) -> "Layer":
        """W_gate/W_up [E,I,d], W_down [E,d,I]: CUDA bf16 tensors; channel_rank [E,I] int32 (host) or None."""
        import torch
        assert W_gate.is_cuda and W_gate.dtype == torch.bfloat16 and W_gate.is_contiguous()
        assert W_up.is_cuda and W_up.dtype == torch.bfloat16 and W_up.is_contiguous()
        assert W_down.is_cuda and W_down.dtype == torch.bfloat16 and W_down.is_contiguous()
        E, I, d = W_gate.shape
        assert tuple(W_up.shape) == (E, I, d) and tuple(W_down.shape) == (E, d, I)
        nbytes = packed_bytes(E, d, I)
        packed = torch.empty(nbytes + 1024, dtype=torch.uint8, device=W_gate.device)
        off = (-packed.data_ptr()) % 1024
        packed = packed[off:off + nbytes]
        rk = None
        rk_ptr = None
        if channel_rank is not None:
            rk = _i32_host(channel_rank)
            assert rk.shape == (E, I)
            rk_ptr = ctypes.c_void_p(rk.ctypes.data)
        h = ctypes.c_void_p()
        _chk(lib().fxm_pack(ctypes.byref(h), E, d, I, W_gate.data_ptr(), W_up.data_ptr(), W_down.data_ptr(), rk_ptr,
                            packed.data_ptr(), _stream_ptr(stream)), "fxm_pack")
        return Layer(h, E, d, I, packed)

    def __del__(self):
        try:
            if self._h:
                lib().fxm_destroy(self._h)
                self._h = None
        except Exception:
            pass

    # -- (2) budgets ------------------------------------------------------------------------------
    def set_budget(self, r, stream=None):
        r = _i32_host(r)
        assert r.shape == (self.E,)
        _chk(lib().fxm_set_budget(self._h, r.ctypes.data, _stream_ptr(stream)), "fxm_set_budget")

    def register_budgets(self, tables, require_nested=True, stream=None):
        t = _i32_host(tables)
        assert t.ndim == 2 and t.shape[1] == self.E
        _chk(lib().fxm_register_budgets(self._h, t.shape[0], t.ctypes.data, int(bool(require_nested)),
                                        _stream_ptr(stream)), "fxm_register_budgets")

    def sample_budget(self, alpha, gumbel, num, den, return_actions=False, stream=None):
        """Eq. 6-7 on the device (fxm_sample_budget): alpha, gumbel [E,K] fp32 CUDA (gumbel may be None)."""
        import torch
        num = _i32_host(num)
        K = num.shape[0]
        assert alpha.is_cuda and alpha.dtype == torch.float32 and alpha.is_contiguous() and tuple(alpha.shape) == (self.E, K)
        act = torch.empty(self.E, dtype=torch.int32, device=alpha.device) if return_actions else None
        _chk(lib().fxm_sample_budget(self._h, alpha.data_ptr(), gumbel.data_ptr() if gumbel is not None else None, K,
                                     num.ctypes.data, int(den), act.data_ptr() if act is not None else None,
                                     _stream_ptr(stream)), "fxm_sample_budget")
        return act

    def action_cost(self, alpha, num, den, counts, stream=None):
        """Eq. 10 on the device (fxm_action_cost) -> 1-element fp32 CUDA tensor."""
        import torch
        num = _i32_host(num)
        out = torch.empty(1, dtype=torch.float32, device=alpha.device)
        _chk(lib().fxm_action_cost(self._h, alpha.data_ptr(), num.shape[0], num.ctypes.data, int(den), counts.data_ptr(),
                                   out.data_ptr(), _stream_ptr(stream)), "fxm_action_cost")
        return out

    def select_budget(self, b: int):
        _chk(lib().fxm_select_budget(self._h, int(b)), "fxm_select_budget")

    def set_impl(self, impl: int):
        _chk(lib().fxm_set_impl(self._h, int(impl)), "fxm_set_impl")

    def set_tile_n(self, n: int):
        _chk(lib().fxm_set_tile_n(self._h, int(n)), "fxm_set_tile_n")

    def set_decode(self, max_assignments: int = DECODE_DEFAULT_MAX_ASSIGNMENTS, prefetch_tiles: int = DECODE_DEFAULT_PREFETCH):
        _chk(lib().fxm_set_decode(self._h, int(max_assignments), int(prefetch_tiles)), "fxm_set_decode")

    # -- workspace ----------------------------------------------------------------------------------
    def workspace(self, T: int, k: int):
        """A cached 1024-aligned torch buffer large enough for (T, k)."""
        import torch
        need = workspace_bytes(self.E, self.d, self.I, T, k)
        if self._ws is None or self._ws.numel() < need:
            raw = torch.empty(need + 1024, dtype=torch.uint8, device=self.packed.device)
            off = (-raw.data_ptr()) % 1024
            self._ws = raw[off:off + need]
        return self._ws

    # -- (3) forward --------------------------------------------------------------------------------
    def moe_ffn(self, x, topk_ids, topk_w, out=None, workspace=None, stream=None, y_shared=None):
        """x [T,d] bf16, topk_ids [T,k] int32, topk_w [T,k] fp32 (CUDA, contiguous) -> y [T,d] bf16.
        y_shared [T,d] bf16 (optional): the shared expert's output, added before the rounding (fxm_moe_ffn_shared)."""
        import torch
        T, d = x.shape
        k = topk_ids.shape[1]
        assert d == self.d and x.dtype == torch.bfloat16 and x.is_cuda and x.is_contiguous()
        assert topk_ids.dtype == torch.int32 and topk_ids.is_contiguous() and tuple(topk_ids.shape) == (T, k)
        assert topk_w.dtype == torch.float32 and topk_w.is_contiguous() and tuple(topk_w.shape) == (T, k)
        y = torch.empty((T, d), dtype=torch.bfloat16, device=x.device) if out is None else out
        ws = self.workspace(T, k) if workspace is None else workspace
        if y_shared is None:
            _chk(lib().fxm_moe_ffn(self._h, x.data_ptr(), topk_ids.data_ptr(), topk_w.data_ptr(), T, k, y.data_ptr(),
                                   ws.data_ptr(), ws.numel(), _stream_ptr(stream)), "fxm_moe_ffn")
        else:
            assert y_shared.dtype == torch.bfloat16 and y_shared.is_contiguous() and tuple(y_shared.shape) == (T, d)
            _chk(lib().fxm_moe_ffn_shared(self._h, x.data_ptr(), topk_ids.data_ptr(), topk_w.data_ptr(), T, k,
                                          y_shared.data_ptr(), y.data_ptr(), ws.data_ptr(), ws.numel(),
                                          _stream_ptr(stream)), "fxm_moe_ffn_shared")
        return y

    def moe_ffn_router(self, x, logits, k, y_shared=None, out=None, return_routing=False, workspace=None, stream=None):
        """Forward from router LOGITS [T,E] fp32 (fxm_moe_ffn_router): softmax -> top-k -> renormalise runs on the device
        in the route kernel.  -> y, or (y, topk_ids, topk_w) with return_routing."""
        import torch
        T, d = x.shape
        assert d == self.d and x.dtype == torch.bfloat16 and x.is_cuda and x.is_contiguous()
        assert logits.dtype == torch.float32 and logits.is_contiguous() and tuple(logits.shape) == (T, self.E)
        y = torch.empty((T, d), dtype=torch.bfloat16, device=x.device) if out is None else out
        ids = torch.empty((T, k), dtype=torch.int32, device=x.device) if return_routing else None
        w = torch.empty((T, k), dtype=torch.float32, device=x.device) if return_routing else None
        ws = self.workspace(T, k) if workspace is None else workspace
        _chk(lib().fxm_moe_ffn_router(self._h, x.data_ptr(), logits.data_ptr(), T, k,
                                      y_shared.data_ptr() if y_shared is not None else None, y.data_ptr(),
                                      ids.data_ptr() if ids is not None else None, w.data_ptr() if w is not None else None,
                                      ws.data_ptr(), ws.numel(), _stream_ptr(stream)), "fxm_moe_ffn_router")
        return (y, ids, w) if return_routing else y

    # -- offline clipping ----------------------------------------------------------------
    def export_clipped(self, r, stream=None):
        """-> torch.uint8 blob (device) holding only the retained prefix of every expert for the widths r[E]."""
        import torch
        r = _i32_host(r)
        assert r.shape == (self.E,)
        n = ctypes.c_size_t()
        _chk(lib().fxm_clipped_bytes(self.E, self.d, self.I, r.ctypes.data, ctypes.byref(n)), "fxm_clipped_bytes")
        raw = torch.empty(n.value + 1024, dtype=torch.uint8, device=self.packed.device)
        off = (-raw.data_ptr()) % 1024
        blob = raw[off:off + n.value]
        _chk(lib().fxm_export_clipped(self._h, r.ctypes.data, blob.data_ptr(), blob.numel(), _stream_ptr(stream)),
             "fxm_export_clipped")
        return blob

    @staticmethod
    def parse_clipped_header(host_bytes):
        """host_bytes: the first >= 2048 bytes of a blob (bytes / numpy uint8) -> (E, d, I, r[E])."""
        import numpy as np
        buf = np.frombuffer(bytes(host_bytes[:2048]), dtype=np.uint8).copy()
        E, d, I = ctypes.c_int(), ctypes.c_int(), ctypes.c_int()
        r = np.zeros(256, np.int32)
        _chk(lib().fxm_parse_clipped_header(buf.ctypes.data, buf.size, ctypes.byref(E), ctypes.byref(d), ctypes.byref(I),
                                            r.ctypes.data), "fxm_parse_clipped_header")
        return E.value, d.value, I.value, r[:E.value].copy()

    @staticmethod
    def load_clipped(blob, E, d, I, r, stream=None) -> "Layer":
        """blob: torch.uint8 CUDA tensor (1024-byte aligned) written by export_clipped, possibly after a round trip
        through host memory or a file."""
        r = _i32_host(r)
        h = ctypes.c_void_p()
        _chk(lib().fxm_load_clipped(ctypes.byref(h), E, d, I, r.ctypes.data, blob.data_ptr(), blob.numel(),
                                    _stream_ptr(stream)), "fxm_load_clipped")
        return Layer(h, E, d, I, blob, clipped_widths=r.copy())

    def workspace_host(self, T: int, k: int):
        import torch
        need = workspace_bytes_host(self.E, self.d, self.I, T, k)
        if getattr(self, "_wsh", None) is None or self._wsh.numel() < need:
            raw = torch.empty(need + 1024, dtype=torch.uint8, device=self.packed.device)
            off = (-raw.data_ptr()) % 1024
            self._wsh = raw[off:off + need]
        return self._wsh

    def moe_ffn_host(self, x_host, ids_host, w_host, y_host, stream=None, pipelined=False):
        """Host-buffer forward (fxm_moe_ffn_host): x_host/y_host [T,d] bf16, ids_host [T,k] int32, w_host [T,k]
        fp32 CPU tensors (pinned recommended).  Asynchronous; y_host is valid after the stream is synchronised.
        pipelined=True (fxm_moe_ffn_host_pipelined): y is copied back under the next call's kernels and is valid once the
        stream has passed a later host_flush()."""
        import torch
        T, d = x_host.shape
        k = ids_host.shape[1]
        for t in (x_host, ids_host, w_host, y_host):
            assert not t.is_cuda and t.is_contiguous()
        assert d == self.d and x_host.dtype == torch.bfloat16 and y_host.dtype == torch.bfloat16
        assert tuple(y_host.shape) == (T, d) and ids_host.dtype == torch.int32 and w_host.dtype == torch.float32
        assert tuple(ids_host.shape) == (T, k) and tuple(w_host.shape) == (T, k)
        ws = self.workspace_host(T, k)
        fn = lib().fxm_moe_ffn_host_pipelined if pipelined else lib().fxm_moe_ffn_host
        _chk(fn(self._h, x_host.data_ptr(), ids_host.data_ptr(), w_host.data_ptr(), T, k,
                y_host.data_ptr(), ws.data_ptr(), ws.numel(), _stream_ptr(stream)), "fxm_moe_ffn_host")
        return y_host

    def host_flush(self, stream=None):
        """fxm_host_flush: the stream waits for every pipelined y copy still in flight (host-only, no launch)."""
        _chk(lib().fxm_host_flush(self._h, _stream_ptr(stream)), "fxm_host_flush")

    # -- measurement surface ----------------------------------------------------------------------------
    def profile_begin(self, max_calls: int):
        _chk(lib().fxm_profile_begin(self._h, int(max_calls)), "fxm_profile_begin")

    def profile_end(self):
        """-> (dict kernel name -> summed ms over the recorded calls, number of calls)."""
        ms = (ctypes.c_float * N_KERNELS)()
        n = ctypes.c_int()
        _chk(lib().fxm_profile_end(self._h, ms, ctypes.byref(n)), "fxm_profile_end")
        return {KERNEL_NAMES[j]: float(ms[j]) for j in range(N_KERNELS)}, n.value

    # -- parity / debug surface -----------------------------------------------------------------------
    def route(self, topk_ids, stream=None):
        import torch
        T, k = topk_ids.shape
        assert topk_ids.dtype == torch.int32 and topk_ids.is_cuda and topk_ids.is_contiguous()
        dev = topk_ids.device
        counts = torch.empty(self.E, dtype=torch.int32, device=dev)
        offsets = torch.empty(self.E + 1, dtype=torch.int32, device=dev)
        perm = torch.empty(max(T * k, 1), dtype=torch.int32, device=dev)
        inv = torch.empty(max(T * k, 1), dtype=torch.int32, device=dev)
        ws = self.workspace(T, k)
        _chk(lib().fxm_route(self._h, topk_ids.data_ptr(), T, k, counts.data_ptr(), offsets.data_ptr(), perm.data_ptr(),
                             inv.data_ptr(), ws.data_ptr(), ws.numel(), _stream_ptr(stream)), "fxm_route")
        return counts, offsets, perm[:T * k], inv[:T * k]

    def unpack_prefix(self, e: int, r: int, stream=None):
        import torch
        dev = self.packed.device
        Wg = torch.empty((r, self.d), dtype=torch.bfloat16, device=dev)
        Wu = torch.empty((r, self.d), dtype=torch.bfloat16, device=dev)
        Wd = torch.empty((self.d, r), dtype=torch.bfloat16, device=dev)
        _chk(lib().fxm_unpack_prefix(self._h, e, r, Wg.data_ptr(), Wu.data_ptr(), Wd.data_ptr(), _stream_ptr(stream)),
             "fxm_unpack_prefix")
        return Wg, Wu, Wd

    def debug_read_h(self, topk_ids, raw=False, stream=None):
        import torch
        T, k = topk_ids.shape
        H = torch.zeros((T * k, self.I), dtype=torch.bfloat16, device=self.packed.device)
        ws = self.workspace(T, k)
        _chk(lib().fxm_debug_read_h(self._h, topk_ids.data_ptr(), T, k, ws.data_ptr(), H.data_ptr(), int(bool(raw)),
                                    _stream_ptr(stream)), "fxm_debug_read_h")
        return H

    def device_flags(self, stream=None) -> int:
        f = ctypes.c_uint32()
        _chk(lib().fxm_device_flags(self._h, ctypes.byref(f), _stream_ptr(stream)), "fxm_device_flags")
        return f.value

    def launches_per_ffn(self) -> int:
        return int(lib().fxm_launches_per_ffn(self._h))


# --------------------------------------------------------------------------------------- torch helpers
def bf16_from_bits(bits, device="cuda"):
    """numpy uint16 bf16 bit patterns -> torch.bfloat16 tensor on `device` (no arithmetic)."""
    import numpy as np
    import torch
    t = torch.from_numpy(np.ascontiguousarray(bits).view(np.int16))
    return t.to(device).view(torch.bfloat16)


def bf16_to_bits(t):
    """torch.bfloat16 tensor -> numpy uint16 bit patterns."""
    import numpy as np
    import torch
    return t.detach().contiguous().view(torch.int16).cpu().numpy().view(np.uint16)
