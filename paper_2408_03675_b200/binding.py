"""ctypes binding of libnacl_evict.so -- argument marshalling only.

Every step of the path (scoring, softmax statistics, column sum, selects, sampling keys,
compaction, gather) runs in the library's CUDA kernels; PyTorch supplies device memory and the
stream.  Function names mirror include/nacl_evict.h.  There is no CPU fallback: if the library is
missing or cannot be loaded, importing this module raises.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

from . import build as _build

NACL_DTYPE_F32, NACL_DTYPE_BF16 = 0, 1
FLAG_CAUSAL, FLAG_SAMPLE_SOFTMAX_OF_SCORE, FLAG_SAMPLE_UNIFORM, FLAG_SHARED_HEADS, FLAG_SCORE_CUDA_CORES = 1, 2, 4, 8, 0x100
FLAG_SCORE_TWO_LAUNCHES, FLAG_SELECT_GENERAL, FLAG_GATHER_SEPARATE = 0x200, 0x400, 0x800

EXPORTS = ("nacl_evict", "nacl_evict_f32", "nacl_evict_ex", "nacl_evict_host", "nacl_workspace_bytes",
           "nacl_release", "nacl_strerror", "nacl_last_cuda_error", "nacl_version",
           "nacl_profile_enable", "nacl_profile_read", "nacl_stage_name", "nacl_gumbel_keys", "nacl_evict_generation",
           "nacl_select_fallbacks", "nacl_evict_varlen", "nacl_evict_host_batch", "nacl_evict_batch", "nacl_evict_static", "nacl_proxy_lse",
           "nacl_last_select_launch")
N_STAGES = 7


class NaclParams(C.Structure):
    _fields_ = [
        ("struct_size", C.c_uint32), ("dtype", C.c_int32),
        ("K", C.c_void_p), ("V", C.c_void_p), ("Qproxy", C.c_void_p),
        ("batch", C.c_int32), ("L", C.c_int32), ("Hq", C.c_int32), ("Hkv", C.c_int32), ("d", C.c_int32), ("P", C.c_int32),
        ("budget_proxy", C.c_int32), ("budget_random", C.c_int32), ("n_sink", C.c_int32), ("n_recent", C.c_int32),
        ("seed", C.c_uint64), ("layer", C.c_int32), ("flags", C.c_uint32),
        ("out_K", C.c_void_p), ("out_V", C.c_void_p), ("out_idx", C.c_void_p),
        ("out_importance", C.c_void_p), ("out_lse", C.c_void_p),
        ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t), ("stream", C.c_void_p),
        ("lse_in", C.c_void_p),
        ("batch_offset", C.c_int32), ("head_offset", C.c_int32),
        ("protect_idx", C.c_void_p), ("n_protect", C.c_int32), ("reserved0", C.c_int32),
        ("kv_stride_batch", C.c_int64), ("kv_stride_head", C.c_int64), ("kv_stride_row", C.c_int64),
        ("out_stride_batch", C.c_int64), ("out_stride_head", C.c_int64), ("out_stride_row", C.c_int64),
        ("block_table", C.c_void_p), ("page_size", C.c_int32), ("table_stride", C.c_int32), ("n_pages", C.c_int32),
        ("reserved1", C.c_int32), ("kv_stride_page", C.c_int64),
    ]


class NaclGenParams(C.Structure):
    _fields_ = [
        ("struct_size", C.c_uint32), ("dtype", C.c_int32),
        ("K_cache", C.c_void_p), ("V_cache", C.c_void_p), ("q", C.c_void_p), ("pos_in", C.c_void_p),
        ("batch", C.c_int32), ("Hq", C.c_int32), ("Hkv", C.c_int32), ("d", C.c_int32), ("len", C.c_int32),
        ("cap_in", C.c_int32), ("cap_out", C.c_int32),
        ("budget_proxy", C.c_int32), ("budget_random", C.c_int32), ("n_sink", C.c_int32), ("n_recent", C.c_int32),
        ("seed", C.c_uint64), ("layer", C.c_int32), ("step", C.c_int32), ("flags", C.c_uint32),
        ("batch_offset", C.c_int32), ("head_offset", C.c_int32), ("reserved0", C.c_int32),
        ("K_out", C.c_void_p), ("V_out", C.c_void_p), ("pos_out", C.c_void_p), ("out_idx", C.c_void_p),
        ("out_importance", C.c_void_p), ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t), ("stream", C.c_void_p),
    ]


class NaclError(RuntimeError):
    def __init__(self, code: int, where: str):
        msg = _lib.nacl_strerror(code).decode()
        extra = f" (cudaError {_lib.nacl_last_cuda_error()})" if code == -6 else ""
        super().__init__(f"{where}: {msg}{extra} [code {code}]")
        self.code = code


def library_path() -> str:
    return _build.LIB


def _load() -> C.CDLL:
    path = _build.LIB
    if not os.path.exists(path) or _build.needs_build():
        path = _build.build()  # raises if nvcc is missing or the build fails: no fallback
    lib = C.CDLL(path)
    vp, i32, u64, u32 = C.c_void_p, C.c_int, C.c_uint64, C.c_uint32
    sig = [vp, vp, vp] + [i32] * 10 + [u64, i32, vp, vp, vp, vp]
    lib.nacl_evict.argtypes = sig
    lib.nacl_evict.restype = i32
    lib.nacl_evict_f32.argtypes = sig
    lib.nacl_evict_f32.restype = i32
    lib.nacl_evict_ex.argtypes = [C.POINTER(NaclParams)]
    lib.nacl_evict_ex.restype = i32
    lib.nacl_proxy_lse.argtypes = [C.POINTER(NaclParams)]
    lib.nacl_proxy_lse.restype = i32
    lib.nacl_evict_static.argtypes = [C.POINTER(NaclParams)]
    lib.nacl_evict_static.restype = i32
    lib.nacl_evict_batch.argtypes = [C.POINTER(NaclParams), i32]
    lib.nacl_evict_batch.restype = i32
    lib.nacl_evict_generation.argtypes = [C.POINTER(NaclGenParams)]
    lib.nacl_evict_generation.restype = i32
    lib.nacl_evict_host.argtypes = [vp, vp, vp, i32] + [i32] * 10 + [u64, i32, vp, vp, vp, i32]
    lib.nacl_evict_host.restype = i32
    lib.nacl_evict_host_batch.argtypes = [i32, vp, vp, vp, i32] + [i32] * 10 + [vp, vp, vp, vp, vp, i32]
    lib.nacl_evict_host_batch.restype = i32
    lib.nacl_workspace_bytes.argtypes = [i32] * 6
    lib.nacl_workspace_bytes.restype = C.c_size_t
    lib.nacl_release.argtypes = []
    lib.nacl_release.restype = None
    lib.nacl_last_select_launch.argtypes = [C.POINTER(i32)] * 3
    lib.nacl_last_select_launch.restype = None
    lib.nacl_select_fallbacks.argtypes = [i32]
    lib.nacl_select_fallbacks.restype = i32
    lib.nacl_evict_varlen.argtypes = [C.POINTER(NaclParams), C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.POINTER(C.c_int32), i32]
    lib.nacl_evict_varlen.restype = i32
    lib.nacl_strerror.argtypes = [i32]
    lib.nacl_strerror.restype = C.c_char_p
    lib.nacl_last_cuda_error.argtypes = []
    lib.nacl_last_cuda_error.restype = i32
    lib.nacl_version.argtypes = []
    lib.nacl_version.restype = i32
    lib.nacl_gumbel_keys.argtypes = [vp, vp, i32, i32, i32, u64, i32, u32, vp]
    lib.nacl_gumbel_keys.restype = i32
    lib.nacl_profile_enable.argtypes = [i32]
    lib.nacl_profile_enable.restype = i32
    lib.nacl_profile_read.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_int64), i32]
    lib.nacl_profile_read.restype = i32
    lib.nacl_stage_name.argtypes = [i32]
    lib.nacl_stage_name.restype = C.c_char_p
    return lib


_lib = _load()


def _dtype_tag(t: torch.Tensor) -> int:
    if t.dtype == torch.bfloat16:
        return NACL_DTYPE_BF16
    if t.dtype == torch.float32:
        return NACL_DTYPE_F32
    raise TypeError(f"nacl_evict takes bfloat16 or float32 tensors, got {t.dtype}")


def _shapes(K, V, Q):
    if K.dim() != 4 or Q.dim() != 4 or V.shape != K.shape:
        raise ValueError("expected K,V [batch,Hkv,L,d] and Qproxy [batch,Hq,P,d]")
    B, Hkv, L, d = K.shape
    B2, Hq, P, d2 = Q.shape
    if B2 != B or d2 != d or K.dtype != V.dtype or K.dtype != Q.dtype:
        raise ValueError("K/V/Qproxy batch, head_dim or dtype mismatch")
    if not Q.is_contiguous():
        raise ValueError("Qproxy must be contiguous")
    if K.stride() != V.stride() or K.stride(3) != 1:
        raise ValueError("K and V must share their strides and have contiguous rows (stride 1 along head_dim)")
    return B, Hkv, L, d, Hq, P


def _kv_strides(t):
    """(batch, head, row) element strides of a [batch, Hkv, L, d] view, or (0, 0, 0) when it is contiguous."""
    return (0, 0, 0) if t.is_contiguous() else (t.stride(0), t.stride(1), t.stride(2))


def nacl_version() -> int:
    return int(_lib.nacl_version())


def nacl_workspace_bytes(batch, L, Hq, Hkv, d, P) -> int:
    return int(_lib.nacl_workspace_bytes(batch, L, Hq, Hkv, d, P))


def nacl_select_fallbacks(reset: bool = True) -> int:
    rc = int(_lib.nacl_select_fallbacks(1 if reset else 0))
    if rc < 0:
        raise NaclError(rc, "nacl_select_fallbacks")
    return rc


def nacl_last_select_launch() -> dict:
    """Launch configuration of the selection kernel of the latest call issued from this thread (diagnostics)."""
    g, c, f = C.c_int32(0), C.c_int32(0), C.c_int32(0)
    _lib.nacl_last_select_launch(C.byref(g), C.byref(c), C.byref(f))
    return {"grid_ctas": g.value, "cluster_size": c.value, "fused_gather": bool(f.value)}


def nacl_release() -> None:
    _lib.nacl_release()


def nacl_profile_enable(on: bool) -> None:
    _lib.nacl_profile_enable(1 if on else 0)


def nacl_profile_read(reset: bool = True) -> dict:
    """{stage name: (device ms, launches)} accumulated since the last reset (include/nacl_evict.h)."""
    ms = (C.c_double * N_STAGES)()
    n = (C.c_int64 * N_STAGES)()
    rc = _lib.nacl_profile_read(ms, n, 1 if reset else 0)
    if rc != 0:
        raise NaclError(rc, "nacl_profile_read")
    return {_lib.nacl_stage_name(s).decode(): (float(ms[s]), int(n[s])) for s in range(N_STAGES)}


def nacl_gumbel_keys(importance: torch.Tensor, seed: int, layer: int, flags: int = 0, out: torch.Tensor | None = None,
                     stream=None) -> torch.Tensor:
    """Sampling keys of every position (include/nacl_evict.h nacl_gumbel_keys): importance [B,Hkv,L] fp32 on the GPU."""
    assert importance.is_cuda and importance.dtype == torch.float32 and importance.dim() == 3 and importance.is_contiguous()
    B, Hkv, L = importance.shape
    if out is None:
        out = torch.empty_like(importance)
    st = (stream or torch.cuda.current_stream(importance.device)).cuda_stream
    with torch.cuda.device(importance.device):
        rc = _lib.nacl_gumbel_keys(importance.data_ptr(), out.data_ptr(), B, Hkv, L, seed & 0xFFFFFFFFFFFFFFFF, layer, flags, st)
    if rc != 0:
        raise NaclError(rc, "nacl_gumbel_keys")
    return out


def nacl_evict(K, V, Qproxy, budget_proxy, budget_random, n_sink, n_recent, seed, layer,
               out_K=None, out_V=None, out_idx=None, stream=None):
    """include/nacl_evict.h `nacl_evict` / `nacl_evict_f32` on CUDA tensors.  Returns (out_K, out_V, out_idx)."""
    B, Hkv, L, d, Hq, P = _shapes(K, V, Qproxy)
    if not (K.is_contiguous() and V.is_contiguous()):
        raise ValueError("nacl_evict takes contiguous tensors (strided layouts: nacl_evict_ex)")
    if not K.is_cuda:
        raise ValueError("nacl_evict takes CUDA tensors (use nacl_evict_host for host buffers)")
    Cn = budget_proxy + budget_random
    if out_K is None:
        out_K = torch.empty((B, Hkv, max(Cn, 0), d), dtype=K.dtype, device=K.device)
    if out_V is None:
        out_V = torch.empty_like(out_K)
    if out_idx is None:
        out_idx = torch.empty((B, Hkv, max(Cn, 0)), dtype=torch.int32, device=K.device)
    st = (stream or torch.cuda.current_stream(K.device)).cuda_stream
    fn = _lib.nacl_evict if K.dtype == torch.bfloat16 else _lib.nacl_evict_f32
    _dtype_tag(K)
    with torch.cuda.device(K.device):
        rc = fn(K.data_ptr(), V.data_ptr(), Qproxy.data_ptr(), B, L, Hq, Hkv, d, P, budget_proxy, budget_random,
                n_sink, n_recent, seed, layer, out_K.data_ptr(), out_V.data_ptr(), out_idx.data_ptr(), st)
    if rc != 0:
        raise NaclError(rc, "nacl_evict")
    return out_K, out_V, out_idx


def _ex_params(K, V, Qproxy, budget_proxy, budget_random, n_sink, n_recent, seed, layer, flags=0,
               out_K=None, out_V=None, out_idx=None, want_importance=False, want_lse=False,
               workspace=None, stream=None, lse_in=None, batch_offset=0, head_offset=0, protect_idx=None):
    """Marshals one nacl_evict_ex call: (NaclParams, result dict).  The result dict keeps the output tensors alive."""
    B, Hkv, L, d, Hq, P = _shapes(K, V, Qproxy)
    if not K.is_cuda:
        raise ValueError("nacl_evict_ex takes CUDA tensors")
    dev = K.device
    Cn = budget_proxy + budget_random
    if out_K is None:
        out_K = torch.empty((B, Hkv, max(Cn, 0), d), dtype=K.dtype, device=dev)
    if out_V is None:
        out_V = torch.empty_like(out_K)
    if out_idx is None:
        out_idx = torch.empty((B, Hkv, max(Cn, 0)), dtype=torch.int32, device=dev)
    imp = torch.empty((B, Hkv, L), dtype=torch.float32, device=dev) if want_importance else None
    lse = torch.empty((B, Hq, P), dtype=torch.float32, device=dev) if want_lse else None
    p = NaclParams()
    p.struct_size = C.sizeof(NaclParams)
    p.dtype = _dtype_tag(K)
    p.K, p.V, p.Qproxy = K.data_ptr(), V.data_ptr(), Qproxy.data_ptr()
    p.batch, p.L, p.Hq, p.Hkv, p.d, p.P = B, L, Hq, Hkv, d, P
    p.budget_proxy, p.budget_random, p.n_sink, p.n_recent = budget_proxy, budget_random, n_sink, n_recent
    p.seed, p.layer, p.flags = seed, layer, flags
    p.batch_offset, p.head_offset = batch_offset, head_offset
    p.kv_stride_batch, p.kv_stride_head, p.kv_stride_row = _kv_strides(K)
    if out_K.stride() != out_V.stride() or (Cn > 0 and out_K.stride(3) != 1):
        raise ValueError("out_K and out_V must share their strides and have contiguous rows")
    p.out_stride_batch, p.out_stride_head, p.out_stride_row = _kv_strides(out_K) if Cn > 0 else (0, 0, 0)
    if Cn > 0 and out_K.data_ptr() == K.data_ptr():
        # in-place compaction: the output IS the [batch, Hkv, L, d] cache, not a dense [batch, Hkv, C, d] tensor
        p.out_stride_batch, p.out_stride_head, p.out_stride_row = out_K.stride(0), out_K.stride(1), out_K.stride(2)
        if K.is_contiguous():
            p.kv_stride_batch, p.kv_stride_head, p.kv_stride_row = K.stride(0), K.stride(1), K.stride(2)
    if protect_idx is not None:
        assert protect_idx.is_cuda and protect_idx.dtype == torch.int32 and protect_idx.is_contiguous() and protect_idx.dim() == 1
        p.protect_idx, p.n_protect = protect_idx.data_ptr(), protect_idx.numel()
    p.out_K, p.out_V, p.out_idx = out_K.data_ptr(), out_V.data_ptr(), out_idx.data_ptr()
    p.out_importance = imp.data_ptr() if imp is not None else None
    p.out_lse = lse.data_ptr() if lse is not None else None
    if workspace is not None:
        p.workspace, p.workspace_bytes = workspace.data_ptr(), workspace.numel() * workspace.element_size()
    p.stream = (stream or torch.cuda.current_stream(dev)).cuda_stream
    if lse_in is not None:
        assert lse_in.is_cuda and lse_in.dtype == torch.float32 and lse_in.is_contiguous() and lse_in.shape == (B, Hq, P)
        p.lse_in = lse_in.data_ptr()
    out = {"out_K": out_K, "out_V": out_V, "out_idx": out_idx}
    if imp is not None:
        out["importance"] = imp
    if lse is not None:
        out["lse"] = lse
    return p, out


def nacl_evict_ex(K, V, Qproxy, budget_proxy, budget_random, n_sink, n_recent, seed, layer, **kw):
    """include/nacl_evict.h `nacl_evict_ex`.  Keyword arguments: flags, out_K, out_V, out_idx, want_importance, want_lse,
    workspace, stream, lse_in ([B,Hq,P] fp32 row log-sum-exps: single-sweep path), batch_offset / head_offset (global
    indices of the call's first batch element / kv head: a shard of a larger problem draws what the unsharded call draws),
    protect_idx.  Returns a dict with out_K, out_V, out_idx and, if asked, importance [B,Hkv,L] fp32 and lse [B,Hq,P] fp32."""
    p, out = _ex_params(K, V, Qproxy, budget_proxy, budget_random, n_sink, n_recent, seed, layer, **kw)
    with torch.cuda.device(K.device):
        rc = _lib.nacl_evict_ex(C.byref(p))
    if rc != 0:
        raise NaclError(rc, "nacl_evict_ex")
    return out


def nacl_proxy_lse(K, Qproxy, flags=0, out=None, workspace=None, stream=None):
    """include/nacl_evict.h `nacl_proxy_lse`: the natural-log row normaliser of every proxy row, [B,Hq,P] fp32 -- one sweep
    over K.  Feed it to nacl_evict_ex(..., lse_in=) for the single-sweep eviction."""
    if K.dim() != 4 or Qproxy.dim() != 4 or not K.is_cuda or not Qproxy.is_contiguous() or K.dtype != Qproxy.dtype:
        raise ValueError("nacl_proxy_lse takes K [B,Hkv,L,d] and contiguous Qproxy [B,Hq,P,d] on the GPU, same dtype")
    B, Hkv, L, d = K.shape
    Hq, P = Qproxy.shape[1], Qproxy.shape[2]
    if out is None:
        out = torch.empty((B, Hq, P), dtype=torch.float32, device=K.device)
    p = NaclParams()
    p.struct_size = C.sizeof(NaclParams)
    p.dtype = _dtype_tag(K)
    p.K, p.Qproxy = K.data_ptr(), Qproxy.data_ptr()
    p.batch, p.L, p.Hq, p.Hkv, p.d, p.P = B, L, Hq, Hkv, d, P
    p.flags = flags
    p.kv_stride_batch, p.kv_stride_head, p.kv_stride_row = _kv_strides(K)
    p.out_lse = out.data_ptr()
    if workspace is not None:
        p.workspace, p.workspace_bytes = workspace.data_ptr(), workspace.numel() * workspace.element_size()
    p.stream = (stream or torch.cuda.current_stream(K.device)).cuda_stream
    with torch.cuda.device(K.device):
        rc = _lib.nacl_proxy_lse(C.byref(p))
    if rc != 0:
        raise NaclError(rc, "nacl_proxy_lse")
    return out


STATIC_SCRATCH_BYTES = 16 * 1024 * 1024  # NACL_STATIC_SCRATCH_BYTES of include/nacl_evict.h


def nacl_evict_static(K, V, Qproxy, budget_proxy, budget_random, n_sink, n_recent, seed, layer, **kw):
    """include/nacl_evict.h `nacl_evict_static`: nacl_evict_ex for callers that cannot allocate device memory (a server
    whose KV pool already owns the GPU, a decode loop that must not hit cudaMalloc's device-wide synchronisation, a guest
    of somebody else's allocator).  The kernels' scratch is a fixed STATIC_SCRATCH_BYTES array inside the library, so
    the C call allocates nothing; shapes that need more raise NaclError(-8).  Same keyword arguments as nacl_evict_ex
    except `workspace`; same results, bit for bit.  Pass out_K / out_V / out_idx (and do not ask for importance / lse)
    if this Python wrapper must not allocate either: tensors it is not given it creates with torch.empty.  All calls on
    one GPU share the array: keep them ordered on the GPU (one stream, or events), never concurrent."""
    if kw.get("workspace") is not None:
        raise ValueError("nacl_evict_static brings its own scratch: no workspace argument")
    p, out = _ex_params(K, V, Qproxy, budget_proxy, budget_random, n_sink, n_recent, seed, layer, **kw)
    with torch.cuda.device(K.device):
        rc = _lib.nacl_evict_static(C.byref(p))
    if rc != 0:
        raise NaclError(rc, "nacl_evict_static")
    return out


def nacl_evict_batch(calls):
    """include/nacl_evict.h `nacl_evict_batch`: `calls` is a list of dicts of nacl_evict_ex arguments (positional names
    K, V, Qproxy, budget_proxy, budget_random, n_sink, n_recent, seed, layer plus its keyword arguments), all on one
    stream.  The calls alternate between two internal streams; returns the list of result dicts."""
    if not calls:
        return []
    pos = ("K", "V", "Qproxy", "budget_proxy", "budget_random", "n_sink", "n_recent", "seed", "layer")
    arr = (NaclParams * len(calls))()
    outs = []
    for i, c in enumerate(calls):
        kw = {k: v for k, v in c.items() if k not in pos}
        p, out = _ex_params(*[c[k] for k in pos], **kw)
        arr[i] = p
        outs.append(out)
    with torch.cuda.device(calls[0]["K"].device):
        rc = _lib.nacl_evict_batch(arr, len(calls))
    if rc != 0:
        raise NaclError(rc, "nacl_evict_batch")
    return outs


def nacl_evict_paged(K_pool, V_pool, block_table, L, Qproxy, budget_proxy, budget_random, n_sink, n_recent, seed, layer,
                     flags=0, pool_layout="HND", want_importance=False, workspace=None, stream=None, batch_offset=0, head_offset=0):
    """include/nacl_evict.h `nacl_evict_ex` with a block table: K_pool / V_pool are page pools [n_pages, Hkv, page, d]
    ("HND") or [n_pages, page, Hkv, d] ("NHD"), block_table [B, pages_per_seq] int32 (device), L live keys per batch
    element.  Outputs are dense, as for nacl_evict_ex."""
    if pool_layout == "HND":
        n_pages, Hkv, ps, d = K_pool.shape
        st_page, st_head, st_row = K_pool.stride(0), K_pool.stride(1), K_pool.stride(2)
    else:
        n_pages, ps, Hkv, d = K_pool.shape
        st_page, st_row, st_head = K_pool.stride(0), K_pool.stride(1), K_pool.stride(2)
    if not (K_pool.is_cuda and V_pool.is_cuda and K_pool.stride() == V_pool.stride() and K_pool.stride(3) == 1):
        raise ValueError("nacl_evict_paged takes CUDA pools that share their strides and have contiguous rows")
    assert block_table.is_cuda and block_table.dtype == torch.int32 and block_table.dim() == 2 and block_table.stride(1) == 1
    B, Hq, P, _ = Qproxy.shape
    dev = K_pool.device
    Cn = budget_proxy + budget_random
    out_K = torch.empty((B, Hkv, max(Cn, 0), d), dtype=K_pool.dtype, device=dev)
    out_V = torch.empty_like(out_K)
    out_idx = torch.empty((B, Hkv, max(Cn, 0)), dtype=torch.int32, device=dev)
    imp = torch.empty((B, Hkv, L), dtype=torch.float32, device=dev) if want_importance else None
    p = NaclParams()
    p.struct_size = C.sizeof(NaclParams)
    p.dtype = _dtype_tag(K_pool)
    p.K, p.V, p.Qproxy = K_pool.data_ptr(), V_pool.data_ptr(), Qproxy.data_ptr()
    p.batch, p.L, p.Hq, p.Hkv, p.d, p.P = B, L, Hq, Hkv, d, P
    p.budget_proxy, p.budget_random, p.n_sink, p.n_recent = budget_proxy, budget_random, n_sink, n_recent
    p.seed, p.layer, p.flags = seed, layer, flags
    p.batch_offset, p.head_offset = batch_offset, head_offset
    p.kv_stride_head, p.kv_stride_row, p.kv_stride_page = st_head, st_row, st_page
    p.block_table, p.page_size, p.table_stride, p.n_pages = block_table.data_ptr(), ps, block_table.stride(0), n_pages
    p.out_K, p.out_V, p.out_idx = out_K.data_ptr(), out_V.data_ptr(), out_idx.data_ptr()
    p.out_importance = imp.data_ptr() if imp is not None else None
    if workspace is not None:
        p.workspace, p.workspace_bytes = workspace.data_ptr(), workspace.numel() * workspace.element_size()
    p.stream = (stream or torch.cuda.current_stream(dev)).cuda_stream
    with torch.cuda.device(dev):
        rc = _lib.nacl_evict_ex(C.byref(p))
    if rc != 0:
        raise NaclError(rc, "nacl_evict_ex (paged)")
    out = {"out_K": out_K, "out_V": out_V, "out_idx": out_idx}
    if imp is not None:
        out["importance"] = imp
    return out


def nacl_evict_varlen(K, V, Qproxy, seq_len, budget_proxy, budget_random, n_sink, n_recent, seed, layer, flags=0,
                      workspace=None, stream=None, batch_offset=0, head_offset=0):
    """include/nacl_evict.h `nacl_evict_varlen`: padded K/V [B,Hkv,L_max,d], Qproxy [B,Hq,P,d] (the last P positions of
    every prompt), per-element lengths and budgets (Python ints).  Returns out_K / out_V [B,Hkv,C_max,d] (rows past an
    element's own C untouched: zero here) and per element its packed index rows out_idx[b] [Hkv, C_b]."""
    B, Hkv, L, d, Hq, P = _shapes(K, V, Qproxy)
    if not K.is_cuda:
        raise ValueError("nacl_evict_varlen takes CUDA tensors")
    dev = K.device
    Cs = [int(a) + int(b) for a, b in zip(budget_proxy, budget_random)]
    C_max = max(Cs) if Cs else 0
    out_K = torch.zeros((B, Hkv, C_max, d), dtype=K.dtype, device=dev)
    out_V = torch.zeros_like(out_K)
    idx_flat = torch.zeros((B, Hkv * C_max), dtype=torch.int32, device=dev)
    p = NaclParams()
    p.struct_size = C.sizeof(NaclParams)
    p.dtype = _dtype_tag(K)
    p.K, p.V, p.Qproxy = K.data_ptr(), V.data_ptr(), Qproxy.data_ptr()
    p.batch, p.L, p.Hq, p.Hkv, p.d, p.P = B, L, Hq, Hkv, d, P
    p.n_sink, p.n_recent = n_sink, n_recent
    p.seed, p.layer, p.flags = seed, layer, flags
    p.batch_offset, p.head_offset = batch_offset, head_offset
    p.kv_stride_batch, p.kv_stride_head, p.kv_stride_row = _kv_strides(K)
    p.out_K, p.out_V, p.out_idx = out_K.data_ptr(), out_V.data_ptr(), idx_flat.data_ptr()
    if workspace is not None:
        p.workspace, p.workspace_bytes = workspace.data_ptr(), workspace.numel() * workspace.element_size()
    p.stream = (stream or torch.cuda.current_stream(dev)).cuda_stream
    arr = C.c_int32 * B
    with torch.cuda.device(dev):
        rc = _lib.nacl_evict_varlen(C.byref(p), arr(*[int(v) for v in seq_len]), arr(*[int(v) for v in budget_proxy]),
                                    arr(*[int(v) for v in budget_random]), C_max)
    if rc != 0:
        raise NaclError(rc, "nacl_evict_varlen")
    out_idx = [idx_flat[b, :Hkv * Cs[b]].view(Hkv, Cs[b]) for b in range(B)]
    return {"out_K": out_K, "out_V": out_V, "out_idx": out_idx, "C": Cs}


def nacl_evict_generation(K_cache, V_cache, q, length, budget_proxy, budget_random, n_sink, n_recent, seed, layer, step,
                          K_out, V_out, pos_in=None, pos_out=None, flags=0, want_idx=False, want_importance=False,
                          workspace=None, stream=None, batch_offset=0, head_offset=0):
    """include/nacl_evict.h `nacl_evict_generation`: caches [B,Hkv,cap,d] (contiguous), q [B,Hq,1,d]; the first `length`
    rows of every head are live.  Returns a dict (out_idx / importance when asked)."""
    B, Hkv, cap_in, d = K_cache.shape
    Hq = q.shape[1]
    for t in (K_cache, V_cache, q, K_out, V_out):
        if not (t.is_cuda and t.is_contiguous()):
            raise ValueError("nacl_evict_generation takes contiguous CUDA tensors")
    dev = K_cache.device
    Cn = budget_proxy + budget_random
    g = NaclGenParams()
    g.struct_size = C.sizeof(NaclGenParams)
    g.dtype = _dtype_tag(K_cache)
    g.K_cache, g.V_cache, g.q = K_cache.data_ptr(), V_cache.data_ptr(), q.data_ptr()
    g.batch, g.Hq, g.Hkv, g.d, g.len, g.cap_in, g.cap_out = B, Hq, Hkv, d, length, cap_in, K_out.shape[2]
    g.budget_proxy, g.budget_random, g.n_sink, g.n_recent = budget_proxy, budget_random, n_sink, n_recent
    g.seed, g.layer, g.step, g.flags = seed, layer, step, flags
    g.batch_offset, g.head_offset = batch_offset, head_offset
    g.K_out, g.V_out = K_out.data_ptr(), V_out.data_ptr()
    if pos_in is not None:
        assert pos_in.dtype == torch.int32 and pos_out.dtype == torch.int32 and pos_in.is_contiguous() and pos_out.is_contiguous()
        g.pos_in, g.pos_out = pos_in.data_ptr(), pos_out.data_ptr()
    idx = torch.empty((B, Hkv, max(Cn, 0)), dtype=torch.int32, device=dev) if want_idx else None
    imp = torch.empty((B, Hkv, length), dtype=torch.float32, device=dev) if want_importance else None
    g.out_idx = idx.data_ptr() if idx is not None else None
    g.out_importance = imp.data_ptr() if imp is not None else None
    if workspace is not None:
        g.workspace, g.workspace_bytes = workspace.data_ptr(), workspace.numel() * workspace.element_size()
    g.stream = (stream or torch.cuda.current_stream(dev)).cuda_stream
    with torch.cuda.device(dev):
        rc = _lib.nacl_evict_generation(C.byref(g))
    if rc != 0:
        raise NaclError(rc, "nacl_evict_generation")
    out = {}
    if idx is not None:
        out["out_idx"] = idx
    if imp is not None:
        out["importance"] = imp
    return out


def nacl_evict_host(K, V, Qproxy, budget_proxy, budget_random, n_sink, n_recent, seed, layer,
                    out_K=None, out_V=None, out_idx=None, device=-1):
    """include/nacl_evict.h `nacl_evict_host`: HOST tensors in, HOST tensors out (copies inside, synchronous)."""
    B, Hkv, L, d, Hq, P = _shapes(K, V, Qproxy)
    if not (K.is_contiguous() and V.is_contiguous()):
        raise ValueError("nacl_evict_host takes contiguous tensors")
    if K.is_cuda:
        raise ValueError("nacl_evict_host takes host tensors")
    Cn = budget_proxy + budget_random
    pin = K.is_pinned()
    if out_K is None:
        out_K = torch.empty((B, Hkv, max(Cn, 0), d), dtype=K.dtype, pin_memory=pin)
    if out_V is None:
        out_V = torch.empty_like(out_K, pin_memory=pin)
    if out_idx is None:
        out_idx = torch.empty((B, Hkv, max(Cn, 0)), dtype=torch.int32, pin_memory=pin)
    rc = _lib.nacl_evict_host(K.data_ptr(), V.data_ptr(), Qproxy.data_ptr(), _dtype_tag(K), B, L, Hq, Hkv, d, P,
                              budget_proxy, budget_random, n_sink, n_recent, seed, layer,
                              out_K.data_ptr(), out_V.data_ptr(), out_idx.data_ptr(), device)
    if rc != 0:
        raise NaclError(rc, "nacl_evict_host")
    return out_K, out_V, out_idx


def nacl_evict_host_batch(Ks, Vs, Qs, budget_proxy, budget_random, n_sink, n_recent, seeds, layers, out_Ks, out_Vs, out_idxs,
                          device=-1):
    """include/nacl_evict.h `nacl_evict_host_batch`: lists of HOST tensors of one shape (pinned memory makes the copies
    asynchronous), results into the given lists of host tensors; the copies of one problem overlap the next one's."""
    n = len(Ks)
    B, Hkv, L, d, Hq, P = _shapes(Ks[0], Vs[0], Qs[0])
    for t in list(Ks) + list(Vs) + list(Qs) + list(out_Ks) + list(out_Vs) + list(out_idxs):
        if t.is_cuda or not t.is_contiguous():
            raise ValueError("nacl_evict_host_batch takes contiguous host tensors")
    ptrs = lambda ts: (C.c_void_p * n)(*[t.data_ptr() for t in ts])
    rc = _lib.nacl_evict_host_batch(n, ptrs(Ks), ptrs(Vs), ptrs(Qs), _dtype_tag(Ks[0]), B, L, Hq, Hkv, d, P,
                                    budget_proxy, budget_random, n_sink, n_recent,
                                    (C.c_uint64 * n)(*[int(v) for v in seeds]), (C.c_int32 * n)(*[int(v) for v in layers]),
                                    ptrs(out_Ks), ptrs(out_Vs), ptrs(out_idxs), device)
    if rc != 0:
        raise NaclError(rc, "nacl_evict_host_batch")
    return out_Ks, out_Vs, out_idxs
