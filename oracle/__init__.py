"""ctypes front-end of the CPU oracle (oracle/nacl_oracle.c).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs.  The product package
(paper_2408_03675_b200) never imports this module and this module never imports
the product.  Arrays are numpy, host memory, contiguous; bf16 tensors are passed as
uint16 bit patterns (see `as_host_array`).
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

F32, BF16 = 0, 1
CAUSAL, SAMPLE_SOFTMAX_OF_SCORE, SAMPLE_UNIFORM = 1, 2, 4

_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        vp, i32, u64, u32 = C.c_void_p, C.c_int, C.c_uint64, C.c_uint
        L.nacl_oracle_philox4x32_10.argtypes = [vp, vp, vp]
        L.nacl_oracle_philox4x32_10.restype = None
        L.nacl_oracle_uniform.argtypes = [u64, i32, i32, i32, i32]
        L.nacl_oracle_uniform.restype = C.c_double
        L.nacl_oracle_gumbel_key.argtypes = [C.c_double, C.c_double, u32]
        L.nacl_oracle_gumbel_key.restype = C.c_float
        L.nacl_oracle_importance.argtypes = [vp, vp, i32, i32, i32, i32, i32, i32, i32, u32, vp, vp, i32]
        L.nacl_oracle_importance.restype = i32
        L.nacl_oracle_select.argtypes = [vp, i32, i32, i32, i32, i32, i32, i32, u64, i32, u32, vp, vp, vp]
        L.nacl_oracle_select.restype = i32
        L.nacl_oracle_select_ex.argtypes = [vp, i32, i32, i32, i32, i32, i32, i32, u64, i32, u32, vp, vp, vp, vp]
        L.nacl_oracle_select_ex.restype = i32
        L.nacl_oracle_gather.argtypes = [vp, vp, C.c_size_t, i32, i32, i32, i32, vp, vp, vp]
        L.nacl_oracle_gather.restype = i32
        L.nacl_oracle_evict.argtypes = [vp, vp, vp, i32] + [i32] * 10 + [u64, i32, u32, vp, vp, vp, vp, i32]
        L.nacl_oracle_evict.restype = i32
        L.nacl_oracle_threads.argtypes = [i32]
        L.nacl_oracle_threads.restype = i32
        _lib = L
    return _lib


class OracleError(RuntimeError):
    def __init__(self, code: int, where: str):
        super().__init__(f"{where} failed with code {code}")
        self.code = code


def _check(rc: int, where: str) -> None:
    if rc != 0:
        raise OracleError(rc, where)


def as_host_array(t) -> np.ndarray:
    """numpy view of a host tensor: fp32 stays fp32, torch.bfloat16 becomes uint16 bits."""
    if isinstance(t, np.ndarray):
        a = t
    else:  # torch tensor, kept out of the import list on purpose
        import torch

        t = t.detach().cpu().contiguous()
        a = t.view(torch.int16).numpy().view(np.uint16) if t.dtype == torch.bfloat16 else t.numpy()
    if a.dtype not in (np.float32, np.uint16):
        raise TypeError(f"oracle takes float32 or bf16-as-uint16, got {a.dtype}")
    return np.ascontiguousarray(a)


def _dtype_tag(a: np.ndarray) -> int:
    return F32 if a.dtype == np.float32 else BF16


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def threads(nthreads: int = 0) -> int:
    return int(lib().nacl_oracle_threads(nthreads))


def philox4x32_10(ctr, key) -> np.ndarray:
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().nacl_oracle_philox4x32_10(_ptr(c), _ptr(k), _ptr(out))
    return out


def uniform(seed: int, layer: int, b: int, hk: int, j: int) -> float:
    return float(lib().nacl_oracle_uniform(seed, layer, b, hk, j))


def gumbel_key(imp: float, u: float, flags: int = 0) -> float:
    return float(lib().nacl_oracle_gumbel_key(imp, u, flags))


def importance(K, Q, flags: int = 0, nthreads: int = 0, return_lse: bool = False):
    """K [B,Hkv,L,d], Q [B,Hq,P,d] -> imp [B,Hkv,L] fp64 (and lse [B,Hq,P] fp64)."""
    K, Q = as_host_array(K), as_host_array(Q)
    if K.dtype != Q.dtype:
        raise TypeError("K and Q must share a dtype")
    B, Hkv, L, d = K.shape
    B2, Hq, P, d2 = Q.shape
    if B2 != B or d2 != d:
        raise ValueError("K/Q shape mismatch")
    imp = np.empty((B, Hkv, L), dtype=np.float64)
    lse = np.empty((B, Hq, P), dtype=np.float64) if return_lse else None
    _check(lib().nacl_oracle_importance(_ptr(K), _ptr(Q), _dtype_tag(K), B, L, Hq, Hkv, d, P, flags,
                                        _ptr(imp), _ptr(lse), nthreads), "nacl_oracle_importance")
    return (imp, lse) if return_lse else imp


class _SelectOpts(C.Structure):
    _fields_ = [("batch_offset", C.c_int), ("head_offset", C.c_int), ("protect_idx", C.c_void_p), ("n_protect", C.c_int),
                ("shared_heads", C.c_int)]


def select(imp, budget_proxy: int, budget_random: int, n_sink: int, n_recent: int,
           seed: int, layer: int, flags: int = 0, return_parts: bool = False, return_keys: bool = False,
           batch_offset: int = 0, head_offset: int = 0, protect_idx=None, shared_heads: bool = False):
    """imp [B,Hkv,L] (any float dtype, widened exactly to fp64) -> idx [B,Hkv,C] int32 ascending.
    batch_offset / head_offset / protect_idx / shared_heads: nacl_oracle_select_opts (oracle/nacl_oracle.h)."""
    imp = np.ascontiguousarray(np.asarray(imp, dtype=np.float64))
    B, Hkv, L = imp.shape
    Cn = budget_proxy + budget_random
    idx = np.empty((B, Hkv, max(Cn, 0)), dtype=np.int32)
    part = np.empty_like(idx) if return_parts else None
    keys = np.empty((B, Hkv, L), dtype=np.float32) if return_keys else None
    prot = None if protect_idx is None else np.ascontiguousarray(np.asarray(protect_idx, dtype=np.int32))
    opts = _SelectOpts(batch_offset, head_offset, None if prot is None else prot.ctypes.data, 0 if prot is None else prot.size,
                       1 if shared_heads else 0)
    _check(lib().nacl_oracle_select_ex(_ptr(imp), B, L, Hkv, budget_proxy, budget_random, n_sink, n_recent,
                                       seed, layer, flags, C.byref(opts), _ptr(idx), _ptr(part), _ptr(keys)),
           "nacl_oracle_select_ex")
    out = (idx,)
    if return_parts:
        out += (part,)
    if return_keys:
        out += (keys,)
    return out if len(out) > 1 else idx


def gather(K, V, idx):
    K, V = as_host_array(K), as_host_array(V)
    idx = np.ascontiguousarray(np.asarray(idx, dtype=np.int32))
    B, Hkv, L, d = K.shape
    Cn = idx.shape[-1]
    oK = np.empty((B, Hkv, Cn, d), dtype=K.dtype)
    oV = np.empty((B, Hkv, Cn, d), dtype=V.dtype)
    _check(lib().nacl_oracle_gather(_ptr(K), _ptr(V), d * K.dtype.itemsize, B, L, Hkv, Cn, _ptr(idx),
                                    _ptr(oK), _ptr(oV)), "nacl_oracle_gather")
    return oK, oV


def evict(K, V, Q, budget_proxy: int, budget_random: int, n_sink: int, n_recent: int,
          seed: int, layer: int, flags: int = 0, nthreads: int = 0, return_importance: bool = False, **sel_opts):
    """Steps 1-8.  Returns (out_K, out_V, out_idx[, imp]).  sel_opts (batch_offset, head_offset, protect_idx,
    shared_heads): the three stages called one after the other with nacl_oracle_select_ex in the middle."""
    if sel_opts:
        imp = importance(K, Q, flags=flags & CAUSAL, nthreads=nthreads)
        idx = select(imp, budget_proxy, budget_random, n_sink, n_recent, seed, layer, flags, **sel_opts)
        oK, oV = gather(K, V, idx)
        return (oK, oV, idx, imp) if return_importance else (oK, oV, idx)
    K, V, Q = as_host_array(K), as_host_array(V), as_host_array(Q)
    B, Hkv, L, d = K.shape
    _, Hq, P, _ = Q.shape
    Cn = budget_proxy + budget_random
    oK = np.empty((B, Hkv, max(Cn, 0), d), dtype=K.dtype)
    oV = np.empty_like(oK)
    idx = np.empty((B, Hkv, max(Cn, 0)), dtype=np.int32)
    imp = np.empty((B, Hkv, L), dtype=np.float64) if return_importance else None
    _check(lib().nacl_oracle_evict(_ptr(K), _ptr(V), _ptr(Q), _dtype_tag(K), B, L, Hq, Hkv, d, P,
                                   budget_proxy, budget_random, n_sink, n_recent, seed, layer, flags,
                                   _ptr(oK), _ptr(oV), _ptr(idx), _ptr(imp), nthreads), "nacl_oracle_evict")
    return (oK, oV, idx, imp) if return_importance else (oK, oV, idx)
