"""Thin ctypes binding of libdesigncp (include/designcp.h): argument marshalling only.

Every step of the hot path runs inside the library's CUDA kernels; torch is used here only to
hold device memory and to name the current stream.  There is NO CPU fallback: importing this
module raises if libdesigncp.so is missing, and every call raises on a non-OK status.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, Optional

import torch

_PKG = os.path.dirname(os.path.abspath(__file__))
# DCP_LIB names another build of the same library (A/B timing of two builds in one process each); default: in-tree
LIB_PATH = os.environ.get("DCP_LIB") or os.path.join(_PKG, "libdesigncp.so")

DCP_OK = 0
DCP_ERR_INVALID_ARG, DCP_ERR_UNSUPPORTED, DCP_ERR_WORKSPACE, DCP_ERR_CUDA = 1, 2, 3, 4
DCP_F32, DCP_BF16 = 0, 1
DCP_MONOLITHIC, DCP_ROW, DCP_GRID = 0, 1, 2
DCP_KERNEL_AUTO, DCP_KERNEL_GENERIC, DCP_KERNEL_MMA = 0, 1, 2

DECOMP = {"monolithic": DCP_MONOLITHIC, "row": DCP_ROW, "grid": DCP_GRID}
KERNEL = {"auto": DCP_KERNEL_AUTO, "generic": DCP_KERNEL_GENERIC, "mma": DCP_KERNEL_MMA}

EXPORTS = [
    "dcp_workspace_bytes", "dcp_pair_bias_attention", "dcp_atom_pair_bias_attention",
    "dcp_pair_bias_attention_host", "dcp_partial_states", "dcp_merge_states", "dcp_shard_range",
    "dcp_sparse_atom_workspace_bytes", "dcp_sparse_atom_attention", "dcp_knn", "dcp_knn_budget", "dcp_gather_pair_slice",
    "dcp_pair_transition_workspace_bytes", "dcp_pair_transition",
    "dcp_pairformer_stack_workspace_bytes", "dcp_pairformer_stack",
    "dcp_attention_stack_workspace_bytes", "dcp_attention_stack", "dcp_plan_units",
    "dcp_probe_l2_gather", "dcp_probe_scan",
    "dcp_attention_stack_cache_bytes", "dcp_attention_stack_cached_workspace_bytes", "dcp_attention_stack_cached",
    "dcp_pair_bias_attention_no_alloc",
    "dcp_event_create", "dcp_event_record", "dcp_event_elapsed_ms", "dcp_event_destroy",
    "dcp_kernel_supported", "dcp_last_launch_count", "dcp_status_string", "dcp_version",
    "dcp_no_alloc_scratch_bytes",
]


class DcpError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {status_string(status)}")


class dcp_weights(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in (
        "w_q", "w_k", "w_v", "w_g", "w_b", "w_o", "ln_z_gamma", "ln_z_beta", "ln_s_gamma", "ln_s_beta", "b_q")]
    _fields_ += [("ln_eps", C.c_float)]


class dcp_block_weights(C.Structure):
    _fields_ = [("attn", dcp_weights)] + [(n, C.c_void_p) for n in ("w1", "w2", "w3", "ln_gamma", "ln_beta")]
    _fields_ += [("ln_eps", C.c_float)]


class dcp_plan(C.Structure):
    _fields_ = [("parts", C.c_int), ("key_split", C.c_int), ("kernel", C.c_int),
                ("tile_q", C.c_int), ("tile_k", C.c_int), ("key_segments", C.c_int),
                ("ev_fused_begin", C.c_void_p), ("ev_fused_end", C.c_void_p)]


def _load() -> C.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is missing: build it with `python paper_2607_05439_b200/build.py` "
            "(there is no CPU fallback for the product path)")
    lib = C.CDLL(LIB_PATH)
    vp, i64, i32, sz = C.c_void_p, C.c_int64, C.c_int, C.c_size_t
    lib.dcp_workspace_bytes.argtypes = [i64, i32, i32, i32, i32, i32, i32, C.POINTER(dcp_plan), C.POINTER(sz)]
    layer_args = [vp, vp, i64, C.POINTER(dcp_weights), vp, i64, i32, i32, i32, i32, i32, i32,
                  C.POINTER(dcp_plan), vp, sz, vp]
    lib.dcp_pair_bias_attention.argtypes = layer_args
    lib.dcp_atom_pair_bias_attention.argtypes = layer_args
    lib.dcp_pair_bias_attention_host.argtypes = [vp, vp, C.POINTER(dcp_weights), vp, vp, vp, vp, i64, i32, i32, i32,
                                                 i32, i32, i32, C.POINTER(dcp_plan), vp, sz, vp]
    lib.dcp_partial_states.argtypes = [vp, vp, i64, C.POINTER(dcp_weights), i64, i32, i32, i32, i32, i32, i32,
                                       i64, i64, i64, i64, vp, vp, vp, vp, sz, vp]
    lib.dcp_merge_states.argtypes = [i32, i64, i32, i32, vp, vp, vp, vp, vp, vp, vp]
    lib.dcp_shard_range.argtypes = [i64, i32, i32, C.POINTER(i64), C.POINTER(i64)]
    lib.dcp_event_create.argtypes = [C.POINTER(vp)]
    lib.dcp_event_record.argtypes = [vp, vp]
    lib.dcp_event_elapsed_ms.argtypes = [vp, vp, C.POINTER(C.c_float)]
    lib.dcp_event_destroy.argtypes = [vp]
    for n in ("dcp_event_create", "dcp_event_record", "dcp_event_elapsed_ms", "dcp_event_destroy"):
        getattr(lib, n).restype = i32
    lib.dcp_kernel_supported.argtypes = [i32, i32, i32, i32, i32]
    lib.dcp_kernel_supported.restype = i32
    lib.dcp_last_launch_count.restype = i32
    lib.dcp_pair_bias_attention_no_alloc.argtypes = [vp, vp, i64, C.POINTER(dcp_weights), vp, i64, i32, i32, i32, i32, i32, i32,
                                                     C.POINTER(dcp_plan), vp]
    lib.dcp_no_alloc_scratch_bytes.argtypes = []
    lib.dcp_no_alloc_scratch_bytes.restype = sz
    lib.dcp_status_string.argtypes = [i32]
    lib.dcp_status_string.restype = C.c_char_p
    lib.dcp_version.restype = i32
    lib.dcp_sparse_atom_workspace_bytes.argtypes = [i64, i32, i32, i32, i32, C.POINTER(sz)]
    lib.dcp_sparse_atom_attention.argtypes = [vp, vp, vp, C.POINTER(dcp_weights), vp, i64, i32, i32, i32, i32, i32, i32,
                                              C.POINTER(dcp_plan), vp, sz, vp]
    lib.dcp_knn.argtypes = [vp, vp, i64, i32, vp]
    lib.dcp_gather_pair_slice.argtypes = [vp, i64, vp, vp, i64, i32, i32, i32, vp]
    lib.dcp_pair_transition_workspace_bytes.argtypes = [i32, i32, C.POINTER(sz)]
    lib.dcp_pair_transition.argtypes = [vp, vp, i64, i32, vp, vp, vp, vp, vp, C.c_float, i32, vp, sz, vp]
    lib.dcp_pairformer_stack_workspace_bytes.argtypes = [i64, i32, i32, i32, i32, i32, C.POINTER(sz)]
    lib.dcp_pairformer_stack.argtypes = [vp, vp, C.POINTER(dcp_block_weights), i32, i64, i32, i32, i32, i32, i32, vp, sz, vp]
    lib.dcp_attention_stack_workspace_bytes.argtypes = [i64, i32, i32, i32, i32, i32, C.POINTER(sz)]
    lib.dcp_attention_stack.argtypes = [vp, vp, i64, C.POINTER(dcp_weights), i32, i64, i32, i32, i32, i32, i32, vp, sz, vp]
    lib.dcp_knn_budget.argtypes = [vp, vp, vp, vp, i64, i32, i32, i32, vp]
    lib.dcp_plan_units.argtypes = [i64, i32, i32, i32, i32, i32, C.POINTER(dcp_plan), C.POINTER(i32), C.POINTER(i32), C.POINTER(i32)]
    lib.dcp_probe_l2_gather.argtypes = [vp, i64, i64, i32, vp, vp]
    lib.dcp_probe_scan.argtypes = [vp, i64, vp, vp]
    lib.dcp_attention_stack_cache_bytes.argtypes = [i64, i32, C.POINTER(sz)]
    lib.dcp_attention_stack_cached_workspace_bytes.argtypes = [i64, i32, i32, i32, i32, i32, C.POINTER(sz)]
    lib.dcp_attention_stack_cached.argtypes = [vp, vp, i64, C.POINTER(dcp_weights), i32, i64, i32, i32, i32, i32, i32, vp, sz, vp, sz, vp]
    for n in EXPORTS[:25]:
        getattr(lib, n).restype = i32
    return lib


_lib = _load()


def status_string(st: int) -> str:
    return _lib.dcp_status_string(int(st)).decode()


def version() -> int:
    return int(_lib.dcp_version())


def _check(st: int, where: str):
    if st != DCP_OK:
        raise DcpError(st, where)


def _dtype_code(t: torch.dtype) -> int:
    if t == torch.float32:
        return DCP_F32
    if t == torch.bfloat16:
        return DCP_BF16
    raise TypeError(f"libdesigncp stores f32 or bf16, not {t}")


def _ptr(t: Optional[torch.Tensor]):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream_ptr(stream=None):
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


def _weights_struct(w: Dict[str, torch.Tensor], eps: float, dtype: Optional[torch.dtype] = None) -> dcp_weights:
    ws = dcp_weights()
    for name in ("w_q", "w_k", "w_v", "w_g", "w_b", "w_o", "ln_z_gamma", "ln_z_beta"):
        t = w[name]
        assert t.is_cuda and t.is_contiguous(), name
        assert dtype is None or t.dtype == dtype, f"{name}: {t.dtype}, the activations are {dtype}"
        setattr(ws, name, t.data_ptr())
    for name in ("ln_s_gamma", "ln_s_beta", "b_q"):
        t = w.get(name)
        assert t is None or (t.is_cuda and t.is_contiguous() and (dtype is None or t.dtype == dtype)), name
        setattr(ws, name, None if t is None else t.data_ptr())
    ws.ln_eps = float(eps)
    return ws


def _plan(parts: int, key_split: int, kernel, events=None, tile=(0, 0), key_segments: int = 0) -> dcp_plan:
    k = KERNEL[kernel] if isinstance(kernel, str) else int(kernel)
    e0, e1 = (events if events is not None else (None, None))
    return dcp_plan(int(parts), int(key_split), k, int(tile[0]), int(tile[1]), int(key_segments), e0, e1)


class Event:
    """A timing-enabled cudaEvent_t owned through the C ABI (dcp_event_*)."""

    def __init__(self):
        h = C.c_void_p()
        _check(_lib.dcp_event_create(C.byref(h)), "dcp_event_create")
        self.handle = h

    def record(self, stream=None):
        _check(_lib.dcp_event_record(self.handle, _stream_ptr(stream)), "dcp_event_record")

    def elapsed_ms(self, end: "Event") -> float:
        ms = C.c_float()
        _check(_lib.dcp_event_elapsed_ms(self.handle, end.handle, C.byref(ms)), "dcp_event_elapsed_ms")
        return float(ms.value)

    def __del__(self):
        try:
            _lib.dcp_event_destroy(self.handle)
        except Exception:
            pass


def dcp_shard_range(n: int, parts: int, p: int):
    """Eq. 5, host only."""
    s, l = C.c_int64(), C.c_int64()
    _check(_lib.dcp_shard_range(n, parts, p, C.byref(s), C.byref(l)), "dcp_shard_range")
    return s.value, l.value


def dcp_workspace_bytes(I, c_s, H, c, c_z, dtype: torch.dtype, decomp="monolithic", parts=1, key_split=1,
                        kernel="auto", tile=(0, 0), key_segments=0) -> int:
    out = C.c_size_t()
    pl = _plan(parts, key_split, kernel, None, tile, key_segments)
    _check(_lib.dcp_workspace_bytes(I, c_s, H, c, c_z, _dtype_code(dtype), DECOMP[decomp], C.byref(pl),
                                    C.byref(out)), "dcp_workspace_bytes")
    return int(out.value)


def dcp_plan_units(I, H, c, c_z, dtype: torch.dtype, decomp="monolithic", parts=1, key_split=1, kernel="auto", tile=(0, 0),
                   key_segments=0):
    """(key_segments, tile_q, slots) a call with this plan uses (host only; no device needed)."""
    pl = _plan(parts, key_split, kernel, None, tile, key_segments)
    a, b, cc = C.c_int(), C.c_int(), C.c_int()
    _check(_lib.dcp_plan_units(int(I), H, c, c_z, _dtype_code(dtype), DECOMP[decomp], C.byref(pl), C.byref(a), C.byref(b),
                               C.byref(cc)), "dcp_plan_units")
    return a.value, b.value, cc.value


def dcp_probe_l2_gather(table, n_warps, gathers_per_warp, stream=None):
    """Measurement probe: random 256-byte-row gathers from `table` (uint8 [n_rows * 256], device).  Returns bytes moved."""
    assert table.is_cuda and table.dtype == torch.uint8 and table.numel() % 256 == 0
    sink = torch.zeros(1, dtype=torch.int32, device=table.device)
    _check(_lib.dcp_probe_l2_gather(_ptr(table), table.numel() // 256, int(n_warps), int(gathers_per_warp), _ptr(sink),
                                    _stream_ptr(stream)), "dcp_probe_l2_gather")
    return int(n_warps) * int(gathers_per_warp) * 512


def dcp_probe_scan(x, stream=None):
    """Measurement probe: the kNN candidate scan without selection over x [L, 3] fp32.  Returns L * L."""
    assert x.is_cuda and x.dtype == torch.float32 and x.is_contiguous()
    sink = torch.zeros(1, dtype=torch.int32, device=x.device)
    _check(_lib.dcp_probe_scan(_ptr(x), x.shape[0], _ptr(sink), _stream_ptr(stream)), "dcp_probe_scan")
    return x.shape[0] * x.shape[0]


def dcp_kernel_supported(kernel, dtype: torch.dtype, H: int, c: int, c_z: int) -> bool:
    k = KERNEL[kernel] if isinstance(kernel, str) else int(kernel)
    return bool(_lib.dcp_kernel_supported(k, _dtype_code(dtype), H, c, c_z))


def dcp_last_launch_count() -> int:
    return int(_lib.dcp_last_launch_count())


def _alloc_ws(nbytes: int, device, stream=None) -> torch.Tensor:
    """A temporary the kernels of `stream` use after the call returned: told to the caching allocator, so the block is
    not handed to another tensor while those kernels run."""
    t = torch.empty(max(nbytes, 256), dtype=torch.uint8, device=device)
    if stream is not None:
        t.record_stream(stream)
    return t


def dcp_pair_bias_attention(s, z, w, H, c, decomp="monolithic", parts=1, key_split=1, kernel="auto", eps=1e-5,
                            out=None, workspace=None, stream=None, atom=False, ldz=0, fused_events=None, tile=(0, 0),
                            key_segments=0):
    """out[I, c_s] = W_o (sigmoid(s W_g) (.) softmax(Q K^T/sqrt(c) + LN(z) W_b) V)  on the current CUDA device."""
    assert s.is_cuda and z.is_cuda and s.is_contiguous()
    I, c_s = s.shape
    c_z = z.shape[-1]
    dt = _dtype_code(s.dtype)
    assert z.dtype == s.dtype
    # z may be a view with a row pitch (ldz), but keys and channels are dense
    assert z.stride(-1) == 1 and z.stride(1) == c_z and (ldz or z.stride(0) == I * c_z), "z: inner dimensions not contiguous"
    if out is None:
        out = torch.empty(I, c_s, dtype=s.dtype, device=s.device)
    pl = _plan(parts, key_split, kernel,
               None if fused_events is None else (fused_events[0].handle, fused_events[1].handle), tile, key_segments)
    if workspace is None:
        workspace = _alloc_ws(dcp_workspace_bytes(I, c_s, H, c, c_z, s.dtype, decomp, parts, key_split, kernel, tile,
                                                  key_segments), s.device, stream)
    ws = _weights_struct(w, eps, s.dtype)
    fn = _lib.dcp_atom_pair_bias_attention if atom else _lib.dcp_pair_bias_attention
    st = fn(_ptr(s), _ptr(z), int(ldz), C.byref(ws), _ptr(out), I, c_s, H, c, c_z, dt, DECOMP[decomp], C.byref(pl),
            _ptr(workspace), workspace.numel(), _stream_ptr(stream))
    _check(st, "dcp_atom_pair_bias_attention" if atom else "dcp_pair_bias_attention")
    return out


def dcp_no_alloc_scratch_bytes() -> int:
    return int(_lib.dcp_no_alloc_scratch_bytes())


def dcp_pair_bias_attention_no_alloc(s, z, w, H, c, out, decomp="monolithic", parts=1, key_split=1, kernel="auto", eps=1e-5,
                                     stream=None, ldz=0):
    """dcp_pair_bias_attention with the workspace in the library's static device array: no allocation anywhere (the
    caller passes out); DcpError(DCP_ERR_SCRATCH_LIMIT) beyond dcp_no_alloc_scratch_bytes().  Calls that overlap on the
    GPU race on the shared array."""
    assert s.is_cuda and z.is_cuda and out.is_cuda and s.is_contiguous() and out.is_contiguous() and z.dtype == s.dtype
    I, c_s = s.shape
    c_z = z.shape[-1]
    assert z.stride(-1) == 1 and z.stride(1) == c_z and (ldz or z.stride(0) == I * c_z), "z: inner dimensions not contiguous"
    assert out.shape == s.shape and out.dtype == s.dtype
    pl = _plan(parts, key_split, kernel)
    ws = _weights_struct(w, eps, s.dtype)
    st = _lib.dcp_pair_bias_attention_no_alloc(_ptr(s), _ptr(z), int(ldz), C.byref(ws), _ptr(out), I, c_s, H, c, c_z,
                                               _dtype_code(s.dtype), DECOMP[decomp], C.byref(pl), _stream_ptr(stream))
    _check(st, "dcp_pair_bias_attention_no_alloc")
    return out


def dcp_atom_pair_bias_attention(a, p, w, H, c, **kw):
    """Atom-level dense variant (BASELINE.json config 4): (L, c_atom, c_atompair) for (I, c_s, c_z)."""
    return dcp_pair_bias_attention(a, p, w, H, c, atom=True, **kw)


def dcp_pair_transition(z, w1, w2, w3, ln_gamma, ln_beta, eps=1e-5, out=None, workspace=None, stream=None):
    """z_out = z + (SiLU(LN(z) W1) * (LN(z) W2)) W3 over the last axis of z (Eq. 6); out may be z (in place)."""
    assert z.is_cuda and z.is_contiguous()
    c_z = z.shape[-1]
    n_pairs = z.numel() // c_z
    if out is None:
        out = torch.empty_like(z)
    if workspace is None:
        n = C.c_size_t(0)
        _check(_lib.dcp_pair_transition_workspace_bytes(c_z, _dtype_code(z.dtype), C.byref(n)), "dcp_pair_transition_workspace_bytes")
        workspace = _alloc_ws(int(n.value), z.device, stream)
    st = _lib.dcp_pair_transition(_ptr(z), _ptr(out), n_pairs, c_z, _ptr(w1), _ptr(w2), _ptr(w3), _ptr(ln_gamma), _ptr(ln_beta),
                                  C.c_float(eps), _dtype_code(z.dtype), _ptr(workspace), workspace.numel(), _stream_ptr(stream))
    _check(st, "dcp_pair_transition")
    return out


def dcp_pairformer_stack(s, z, blocks, H, c, eps=1e-5, workspace=None, stream=None):
    """n_blocks non-triangular Pairformer blocks, IN PLACE on s [I, c_s] and z [I, I, c_z]:
    s += AttentionPairBias_b(s, z); z += Transition_b(z).  blocks: sequence of (attention weights dict, transition
    dict with w1, w2, w3, gamma, beta)."""
    assert s.is_cuda and z.is_cuda and s.is_contiguous() and z.is_contiguous()
    I, c_s, c_z = s.shape[0], s.shape[1], z.shape[-1]
    arr = (dcp_block_weights * len(blocks))()
    for b, (wa, wt) in enumerate(blocks):
        arr[b].attn = _weights_struct(wa, eps, s.dtype)
        for dst, src in (("w1", "w1"), ("w2", "w2"), ("w3", "w3"), ("ln_gamma", "gamma"), ("ln_beta", "beta")):
            t = wt[src]
            assert t.is_cuda and t.is_contiguous(), src
            setattr(arr[b], dst, t.data_ptr())
        arr[b].ln_eps = float(eps)
    if workspace is None:
        n = C.c_size_t(0)
        _check(_lib.dcp_pairformer_stack_workspace_bytes(I, c_s, H, c, c_z, _dtype_code(s.dtype), C.byref(n)),
               "dcp_pairformer_stack_workspace_bytes")
        workspace = _alloc_ws(int(n.value), s.device, stream)
    st = _lib.dcp_pairformer_stack(_ptr(s), _ptr(z), arr, len(blocks), I, c_s, H, c, c_z, _dtype_code(s.dtype), _ptr(workspace),
                                   workspace.numel(), _stream_ptr(stream))
    _check(st, "dcp_pairformer_stack")
    return s, z


def dcp_attention_stack(a, z, blocks, H, c, eps=1e-5, workspace=None, stream=None, ldz=0):
    """n sequential AttentionPairBias blocks with residual, IN PLACE on the latent a [I, c_token], against the read-only
    pair tensor z [I, I, c_z].  blocks: sequence of attention weight dicts (one per block)."""
    assert a.is_cuda and z.is_cuda and a.is_contiguous() and z.dtype == a.dtype
    I, c_s, c_z = a.shape[0], a.shape[1], z.shape[-1]
    assert z.stride(-1) == 1 and z.stride(1) == c_z and (ldz or z.stride(0) == I * c_z), "z: inner dimensions not contiguous"
    arr = (dcp_weights * len(blocks))()
    for b, w in enumerate(blocks):
        arr[b] = _weights_struct(w, eps, a.dtype)
    if workspace is None:
        n = C.c_size_t(0)
        _check(_lib.dcp_attention_stack_workspace_bytes(I, c_s, H, c, c_z, _dtype_code(a.dtype), C.byref(n)),
               "dcp_attention_stack_workspace_bytes")
        workspace = _alloc_ws(int(n.value), a.device, stream)
    st = _lib.dcp_attention_stack(_ptr(a), _ptr(z), int(ldz), arr, len(blocks), I, c_s, H, c, c_z, _dtype_code(a.dtype),
                                  _ptr(workspace), workspace.numel(), _stream_ptr(stream))
    _check(st, "dcp_attention_stack")
    return a


def dcp_attention_stack_cache_bytes(I, n_blocks) -> int:
    n = C.c_size_t(0)
    _check(_lib.dcp_attention_stack_cache_bytes(int(I), int(n_blocks), C.byref(n)), "dcp_attention_stack_cache_bytes")
    return int(n.value)


def dcp_attention_stack_cached(a, z, blocks, H, c, eps=1e-5, bias_cache=None, workspace=None, stream=None, ldz=0):
    """dcp_attention_stack with a bias cache: one pass over z writes every block's bias tiles (fp16), the blocks then
    stream 32 bytes per pair each.  bias_cache: device uint8 scratch of dcp_attention_stack_cache_bytes(I, n) bytes."""
    assert a.is_cuda and z.is_cuda and a.is_contiguous() and z.dtype == a.dtype
    I, c_s, c_z = a.shape[0], a.shape[1], z.shape[-1]
    assert z.stride(-1) == 1 and z.stride(1) == c_z and (ldz or z.stride(0) == I * c_z), "z: inner dimensions not contiguous"
    arr = (dcp_weights * len(blocks))()
    for b, w in enumerate(blocks):
        arr[b] = _weights_struct(w, eps, a.dtype)
    if bias_cache is None:
        bias_cache = _alloc_ws(dcp_attention_stack_cache_bytes(I, len(blocks)), a.device, stream)
    if workspace is None:
        n = C.c_size_t(0)
        _check(_lib.dcp_attention_stack_cached_workspace_bytes(I, c_s, H, c, c_z, _dtype_code(a.dtype), C.byref(n)),
               "dcp_attention_stack_cached_workspace_bytes")
        workspace = _alloc_ws(int(n.value), a.device, stream)
    st = _lib.dcp_attention_stack_cached(_ptr(a), _ptr(z), int(ldz), arr, len(blocks), I, c_s, H, c, c_z, _dtype_code(a.dtype),
                                         _ptr(bias_cache), bias_cache.numel(), _ptr(workspace), workspace.numel(),
                                         _stream_ptr(stream))
    _check(st, "dcp_attention_stack_cached")
    return a


def dcp_attention_stack_cached_workspace_bytes(I, c_s, H, c, c_z, dtype: torch.dtype) -> int:
    n = C.c_size_t(0)
    _check(_lib.dcp_attention_stack_cached_workspace_bytes(int(I), int(c_s), int(H), int(c), int(c_z), _dtype_code(dtype),
                                                           C.byref(n)), "dcp_attention_stack_cached_workspace_bytes")
    return int(n.value)


def dcp_attention_stack_workspace_bytes(I, c_s, H, c, c_z, dtype: torch.dtype) -> int:
    n = C.c_size_t(0)
    _check(_lib.dcp_attention_stack_workspace_bytes(int(I), int(c_s), int(H), int(c), int(c_z), _dtype_code(dtype), C.byref(n)),
           "dcp_attention_stack_workspace_bytes")
    return int(n.value)


def dcp_gather_pair_slice(p, idx, out=None, stream=None):
    """p_slice [L, k, c] = p[l, idx[l, j], :] from the dense pair tensor p [L, L, c] (zeros where idx < 0)."""
    assert p.is_cuda and idx.is_cuda and p.is_contiguous() and idx.is_contiguous() and idx.dtype == torch.int32
    L, k, c_p = p.shape[0], idx.shape[1], p.shape[2]
    if out is None:
        out = torch.empty(L, k, c_p, dtype=p.dtype, device=p.device)
    _check(_lib.dcp_gather_pair_slice(_ptr(p), 0, _ptr(idx), _ptr(out), L, k, c_p, _dtype_code(p.dtype), _stream_ptr(stream)),
           "dcp_gather_pair_slice")
    return out


def dcp_knn(x, k, out=None, stream=None):
    """idx [L, k] int32: the k nearest atoms of every atom of x [L, 3] fp32 (itself included), by (distance, index)."""
    assert x.is_cuda and x.dtype == torch.float32 and x.is_contiguous() and x.shape[1] == 3
    L = x.shape[0]
    if out is None:
        out = torch.empty(L, k, dtype=torch.int32, device=x.device)
    _check(_lib.dcp_knn(_ptr(x), _ptr(out), L, int(k), _stream_ptr(stream)), "dcp_knn")
    return out


def dcp_knn_budget(x, residue_id, chain_id, k, n_chains, n_seq=2, out=None, stream=None):
    """idx [L, k] int32: the structured neighbour budget of PAPER.md:303 (sequence-local atoms first, spatial fill,
    inter-chain quota when n_chains > 3).  residue_id, chain_id: [L] int32 device; n_chains: distinct chain ids."""
    assert x.is_cuda and x.dtype == torch.float32 and x.is_contiguous() and x.shape[1] == 3
    for t in (residue_id, chain_id):
        assert t.is_cuda and t.dtype == torch.int32 and t.is_contiguous() and t.shape[0] == x.shape[0]
    L = x.shape[0]
    if out is None:
        out = torch.empty(L, k, dtype=torch.int32, device=x.device)
    _check(_lib.dcp_knn_budget(_ptr(x), _ptr(residue_id), _ptr(chain_id), _ptr(out), L, int(k), int(n_seq), int(n_chains),
                               _stream_ptr(stream)), "dcp_knn_budget")
    return out


def dcp_sparse_atom_workspace_bytes(L, c_atom, H, c, dtype: torch.dtype) -> int:
    n = C.c_size_t(0)
    _check(_lib.dcp_sparse_atom_workspace_bytes(int(L), int(c_atom), int(H), int(c), _dtype_code(dtype), C.byref(n)),
           "dcp_sparse_atom_workspace_bytes")
    return int(n.value)


def dcp_sparse_atom_attention(a, p_slice, idx, w, H, c, eps=1e-5, out=None, workspace=None, stream=None,
                              fused_events=None):
    """Sparse k-neighbour atom attention: a [L, c_atom], p_slice [L, k, c_atompair],
    idx [L, k] int32 (negative = unused slot) -> out [L, c_atom]."""
    assert a.is_cuda and p_slice.is_cuda and idx.is_cuda and a.is_contiguous() and p_slice.is_contiguous()
    assert idx.dtype == torch.int32 and idx.is_contiguous() and p_slice.dtype == a.dtype
    L, c_atom = a.shape
    k, c_p = p_slice.shape[1], p_slice.shape[2]
    assert tuple(idx.shape) == (L, k) and p_slice.shape[0] == L
    if out is None:
        out = torch.empty(L, c_atom, dtype=a.dtype, device=a.device)
    if workspace is None:
        workspace = _alloc_ws(dcp_sparse_atom_workspace_bytes(L, c_atom, H, c, a.dtype), a.device, stream)
    ws = _weights_struct(w, eps, a.dtype)
    pl = _plan(1, 1, "auto", None if fused_events is None else (fused_events[0].handle, fused_events[1].handle))
    st = _lib.dcp_sparse_atom_attention(_ptr(a), _ptr(p_slice), _ptr(idx), C.byref(ws), _ptr(out), L, k, c_atom, H, c, c_p,
                                        _dtype_code(a.dtype), C.byref(pl), _ptr(workspace), workspace.numel(),
                                        _stream_ptr(stream))
    _check(st, "dcp_sparse_atom_attention")
    return out


def dcp_pair_bias_attention_host(s_host, z_host, w, H, c, out_host, s_dev, z_dev, out_dev, workspace,
                                 decomp="monolithic", parts=1, key_split=1, kernel="auto", eps=1e-5, stream=None):
    """End-to-end entry: HOST s, z, out (pinned tensors); device staging buffers supplied by the caller."""
    assert not s_host.is_cuda and not z_host.is_cuda and not out_host.is_cuda
    I, c_s = s_host.shape
    c_z = z_host.shape[-1]
    pl = _plan(parts, key_split, kernel)
    ws = _weights_struct(w, eps)
    st = _lib.dcp_pair_bias_attention_host(_ptr(s_host), _ptr(z_host), C.byref(ws), _ptr(out_host), _ptr(s_dev),
                                           _ptr(z_dev), _ptr(out_dev), I, c_s, H, c, c_z, _dtype_code(s_host.dtype),
                                           DECOMP[decomp], C.byref(pl), _ptr(workspace), workspace.numel(),
                                           _stream_ptr(stream))
    _check(st, "dcp_pair_bias_attention_host")
    return out_host


def dcp_partial_states(s, z, w, H, c, q0, q1, k0, k1, kernel="auto", eps=1e-5, stream=None):
    """Partial (m, l, acc) of query rows [q0,q1) against keys [k0,k1)."""
    I, c_s = s.shape
    c_z = z.shape[-1]
    R, D = q1 - q0, H * c
    m = torch.empty(max(R, 0), H, dtype=torch.float32, device=s.device)
    l = torch.empty_like(m)
    acc = torch.empty(max(R, 0), D, dtype=torch.float32, device=s.device)
    workspace = _alloc_ws(dcp_workspace_bytes(I, c_s, H, c, c_z, s.dtype), s.device, stream)
    ws = _weights_struct(w, eps, s.dtype)
    k = KERNEL[kernel] if isinstance(kernel, str) else int(kernel)
    st = _lib.dcp_partial_states(_ptr(s), _ptr(z), 0, C.byref(ws), I, c_s, H, c, c_z, _dtype_code(s.dtype), k,
                                 q0, q1, k0, k1, _ptr(m), _ptr(l), _ptr(acc), _ptr(workspace), workspace.numel(),
                                 _stream_ptr(stream))
    _check(st, "dcp_partial_states")
    return m, l, acc


def dcp_merge_states(m, l, acc, H, c, stream=None):
    """Left fold over partial states: m, l [n, rows, H], acc [n, rows, H*c] (fp32, device)."""
    n, rows = m.shape[0], m.shape[1]
    m_out = torch.empty(rows, H, dtype=torch.float32, device=m.device)
    l_out = torch.empty_like(m_out)
    acc_out = torch.empty(rows, H * c, dtype=torch.float32, device=m.device)
    m, l, acc = m.contiguous(), l.contiguous(), acc.contiguous()
    if stream is not None:
        for t in (m, l, acc):
            t.record_stream(stream)
    st = _lib.dcp_merge_states(n, rows, H, c, _ptr(m), _ptr(l), _ptr(acc), _ptr(m_out), _ptr(l_out), _ptr(acc_out),
                               _stream_ptr(stream))
    _check(st, "dcp_merge_states")
    return m_out, l_out, acc_out


def raw():
    """The ctypes library handle (tests call error paths with raw arguments)."""
    return _lib
