"""CPU-side checks of the C ABI: the library loads, exports every symbol include/nacl_evict.h declares,
and its host-side validation (which never touches device memory) returns the documented codes."""
import ctypes as C
import os
import re

import pytest

from paper_2408_03675_b200 import build as nacl_build
from paper_2408_03675_b200 import CONFIGS

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    path = nacl_build.build()
    L = C.CDLL(path)
    L.nacl_strerror.restype = C.c_char_p
    L.nacl_workspace_bytes.restype = C.c_size_t
    return L


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "nacl_evict.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(nacl_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    names = declared_symbols()
    assert {"nacl_evict", "nacl_evict_f32", "nacl_evict_ex", "nacl_evict_host", "nacl_workspace_bytes"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/nacl_evict.h but not exported"


def test_version_and_strerror(lib):
    hdr = open(os.path.join(ROOT, "include", "nacl_evict.h")).read()
    assert lib.nacl_version() == int(re.search(r"#define NACL_VERSION (\d+)", hdr).group(1))
    for code in range(0, -9, -1):
        assert lib.nacl_strerror(code)
    assert b"unknown" in lib.nacl_strerror(-99)


def test_workspace_bytes_is_a_pure_function_of_shape(lib):
    for cfg in CONFIGS.values():
        w = lib.nacl_workspace_bytes(cfg.batch, cfg.L, cfg.Hq, cfg.Hkv, cfg.d, cfg.P)
        assert w == lib.nacl_workspace_bytes(cfg.batch, cfg.L, cfg.Hq, cfg.Hkv, cfg.d, cfg.P)
        # at least the importance vector (the sampling keys stay in shared memory for rows a cluster can hold)
        assert w >= 4 * cfg.batch * cfg.Hkv * cfg.L
        assert w < 64 << 20
    assert lib.nacl_workspace_bytes(1, 0, 4, 4, 64, 1) == 0
    assert lib.nacl_workspace_bytes(1, 128, 5, 4, 64, 1) == 0  # Hq % Hkv


def _call(lib, fn, K=0x1000, V=0x2000, Q=0x3000, batch=1, L=512, Hq=4, Hkv=4, d=64, P=16, bp=76, br=26, ns=4, nr=16,
          oK=0x4000, oV=0x5000, oidx=0x6000):
    f = getattr(lib, fn)
    f.argtypes = [C.c_void_p] * 3 + [C.c_int] * 10 + [C.c_uint64, C.c_int] + [C.c_void_p] * 4
    f.restype = C.c_int
    return f(K, V, Q, batch, L, Hq, Hkv, d, P, bp, br, ns, nr, 0, 0, oK, oV, oidx, None)


@pytest.mark.parametrize("fn", ["nacl_evict", "nacl_evict_f32"])
def test_validation_codes_without_touching_the_device(lib, fn):
    # fake (never dereferenced) pointers: every case below must be rejected on the host
    assert _call(lib, fn, K=None) == -1
    assert _call(lib, fn, oidx=None) == -1
    assert _call(lib, fn, Hq=6) == -2            # Hq % Hkv
    assert _call(lib, fn, P=600) == -2           # P > L
    assert _call(lib, fn, d=72) == -2            # d % 16
    assert _call(lib, fn, L=(1 << 24) + 1) == -2
    assert _call(lib, fn, bp=10) == -3           # budget_proxy < n_sink + n_recent
    assert _call(lib, fn, bp=500, br=13) == -3   # total > L
    assert _call(lib, fn, br=-1) == -3
    assert _call(lib, fn, ns=400, nr=200) == -3  # protected > L
    assert _call(lib, fn, K=0x1008) == -4        # misaligned


def test_ex_rejects_wrong_struct_and_unknown_flags(lib):
    from paper_2408_03675_b200.binding import NaclParams

    p = NaclParams()
    p.struct_size = 8
    lib.nacl_evict_ex.argtypes = [C.POINTER(NaclParams)]
    assert lib.nacl_evict_ex(C.byref(p)) == -7
    assert lib.nacl_evict_ex(None) == -1
    p.struct_size = C.sizeof(NaclParams)
    p.dtype = 1
    p.K, p.V, p.Qproxy, p.out_K, p.out_V, p.out_idx = 0x1000, 0x2000, 0x3000, 0x4000, 0x5000, 0x6000
    p.batch, p.L, p.Hq, p.Hkv, p.d, p.P = 1, 512, 4, 4, 64, 16
    p.budget_proxy, p.budget_random, p.n_sink, p.n_recent = 76, 26, 4, 16
    p.flags = 2 | 4  # both sampling variants at once
    assert lib.nacl_evict_ex(C.byref(p)) == -7
    p.flags = 0x8000
    assert lib.nacl_evict_ex(C.byref(p)) == -7
    p.flags = 0
    p.workspace, p.workspace_bytes = 0x10000, 16
    assert lib.nacl_evict_ex(C.byref(p)) == -5


def test_static_scratch_entry_point_validates_on_the_host(lib):
    """nacl_evict_static (the call for users who cannot allocate device memory) refuses what it cannot serve before it
    asks the CUDA runtime for anything: these checks need no GPU."""
    from paper_2408_03675_b200.binding import STATIC_SCRATCH_BYTES, NaclParams

    hdr = open(os.path.join(ROOT, "include", "nacl_evict.h")).read()
    m = re.search(r"#define NACL_STATIC_SCRATCH_BYTES \((\d+) \* (\d+) \* (\d+)\)", hdr)
    assert int(m.group(1)) * int(m.group(2)) * int(m.group(3)) == STATIC_SCRATCH_BYTES
    lib.nacl_evict_static.argtypes = [C.POINTER(NaclParams)]
    assert lib.nacl_evict_static(None) == -1
    p = NaclParams()
    p.struct_size = 8
    assert lib.nacl_evict_static(C.byref(p)) == -7
    p.struct_size = C.sizeof(NaclParams)
    p.dtype = 1
    p.K, p.V, p.Qproxy, p.out_K, p.out_V, p.out_idx = 0x1000, 0x2000, 0x3000, 0x4000, 0x5000, 0x6000
    p.batch, p.L, p.Hq, p.Hkv, p.d, p.P = 4, 32768, 16, 16, 128, 16
    p.budget_proxy, p.budget_random, p.n_sink, p.n_recent = 600, 200, 4, 16
    assert lib.nacl_workspace_bytes(4, 32768, 16, 16, 128, 16) > STATIC_SCRATCH_BYTES
    assert lib.nacl_evict_static(C.byref(p)) == -8       # more scratch than the library carries
    assert b"NACL_STATIC_SCRATCH_BYTES" in lib.nacl_strerror(-8)
    p.Hq = 15
    assert lib.nacl_evict_static(C.byref(p)) == -2       # a bad shape keeps its own code
    p.Hq, p.batch, p.L = 16, 1, 4096
    p.workspace, p.workspace_bytes = 0x10000, 1 << 24
    assert lib.nacl_evict_static(C.byref(p)) == -5       # it brings its own scratch: no caller workspace
    for cfg in CONFIGS.values():                         # every BASELINE.json shape fits
        assert lib.nacl_workspace_bytes(cfg.batch, cfg.L, cfg.Hq, cfg.Hkv, cfg.d, cfg.P) <= STATIC_SCRATCH_BYTES


def test_proxy_lse_validates_on_the_host(lib):
    from paper_2408_03675_b200.binding import NaclParams

    lib.nacl_proxy_lse.argtypes = [C.POINTER(NaclParams)]
    assert lib.nacl_proxy_lse(None) == -1
    p = NaclParams()
    p.struct_size = C.sizeof(NaclParams)
    p.dtype = 1
    p.K, p.Qproxy = 0x1000, 0x3000
    p.batch, p.L, p.Hq, p.Hkv, p.d, p.P = 1, 512, 4, 4, 64, 16
    assert lib.nacl_proxy_lse(C.byref(p)) == -1          # out_lse is what the call is for
    p.out_lse = 0x8000
    p.P = 600
    assert lib.nacl_proxy_lse(C.byref(p)) == -2          # P > L
    p.P = 16
    p.flags = 8                                          # a selection flag means nothing here
    assert lib.nacl_proxy_lse(C.byref(p)) == -7
    p.flags = 0
    p.lse_in = 0x9000
    assert lib.nacl_proxy_lse(C.byref(p)) == -7
    p.lse_in = None
    p.K = 0x1004
    assert lib.nacl_proxy_lse(C.byref(p)) == -4
    p.K, p.out_lse = 0x1000, 0x8002
    p.workspace, p.workspace_bytes = 0x10000, 1 << 24    # a workspace, so that no device is asked for one
    assert lib.nacl_proxy_lse(C.byref(p)) == -4          # misaligned out_lse


def test_paged_kv_validation_without_touching_the_device(lib):
    from paper_2408_03675_b200.binding import NaclParams

    lib.nacl_evict_ex.argtypes = [C.POINTER(NaclParams)]
    p = NaclParams()
    p.struct_size = C.sizeof(NaclParams)
    p.dtype = 1
    p.K, p.V, p.Qproxy, p.out_K, p.out_V, p.out_idx = 0x1000, 0x2000, 0x3000, 0x4000, 0x5000, 0x6000
    p.batch, p.L, p.Hq, p.Hkv, p.d, p.P = 2, 4096, 32, 8, 128, 16
    p.budget_proxy, p.budget_random, p.n_sink, p.n_recent = 600, 200, 4, 16
    p.page_size = 16                                  # paging fields without a table
    assert lib.nacl_evict_ex(C.byref(p)) == -7
    p.block_table, p.table_stride, p.n_pages = 0x7000, 256, 600
    p.page_size = 24                                  # not one of 8, 16, 32, 64, 128
    assert lib.nacl_evict_ex(C.byref(p)) == -2
    p.page_size, p.table_stride = 16, 255             # the table does not cover L
    assert lib.nacl_evict_ex(C.byref(p)) == -2
    p.table_stride = 256
    p.flags = 0x100                                   # only the tensor-core scoring kernel walks a block table
    assert lib.nacl_evict_ex(C.byref(p)) == -7
    p.flags, p.d = 0, 64
    assert lib.nacl_evict_ex(C.byref(p)) == -7
    p.d, p.block_table = 128, 0x7002                  # misaligned table
    assert lib.nacl_evict_ex(C.byref(p)) == -4


def test_in_place_needs_the_same_layout_on_both_sides(lib):
    from paper_2408_03675_b200.binding import NaclParams

    lib.nacl_evict_ex.argtypes = [C.POINTER(NaclParams)]
    p = NaclParams()
    p.struct_size = C.sizeof(NaclParams)
    p.dtype = 1
    p.K, p.V, p.Qproxy, p.out_idx = 0x100000, 0x900000, 0x3000, 0x6000
    p.out_K, p.out_V = p.K, p.V                       # in place ...
    p.batch, p.L, p.Hq, p.Hkv, p.d, p.P = 1, 4096, 8, 8, 128, 16
    p.budget_proxy, p.budget_random, p.n_sink, p.n_recent = 600, 200, 4, 16
    assert lib.nacl_evict_ex(C.byref(p)) == -7        # ... but the output strides default to a dense [B,Hkv,C,d] tensor
    p.out_V = 0xA00000                                # only one of the two aliased
    assert lib.nacl_evict_ex(C.byref(p)) == -7
    p.out_V = p.V
    p.kv_stride_batch = p.out_stride_batch = 8 * 4096 * 128
    p.kv_stride_head = p.out_stride_head = 4096 * 128
    p.kv_stride_row = p.out_stride_row = 128
    p.flags = 8                                       # one shared retained set: stand-alone gather, not in place
    assert lib.nacl_evict_ex(C.byref(p)) == -7


def test_batch_validation_without_touching_the_device(lib):
    from paper_2408_03675_b200.binding import NaclParams

    lib.nacl_evict_batch.argtypes = [C.POINTER(NaclParams), C.c_int]
    arr = (NaclParams * 2)()
    for q in arr:
        q.struct_size = C.sizeof(NaclParams)
    assert lib.nacl_evict_batch(None, 2) == -1
    assert lib.nacl_evict_batch(arr, 0) == 0
    assert lib.nacl_evict_batch(arr, -1) == -1
    arr[1].stream = 0x10                       # the calls of a batch share one stream
    assert lib.nacl_evict_batch(arr, 2) == -7
    arr[1].stream = None
    arr[1].struct_size = 8
    assert lib.nacl_evict_batch(arr, 2) == -7
    arr[1].struct_size = C.sizeof(NaclParams)
    assert lib.nacl_evict_batch(arr, 1) == -1  # a single call is nacl_evict_ex: K, V, Qproxy are NULL here


def test_varlen_validation_without_touching_the_device(lib):
    from paper_2408_03675_b200.binding import NaclParams

    i32x2 = C.c_int32 * 2
    lib.nacl_evict_varlen.argtypes = [C.POINTER(NaclParams), C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.c_int]
    p = NaclParams()
    p.struct_size = C.sizeof(NaclParams)
    p.dtype = 1
    p.K, p.V, p.Qproxy, p.out_K, p.out_V, p.out_idx = 0x1000, 0x2000, 0x3000, 0x4000, 0x5000, 0x6000
    p.batch, p.L, p.Hq, p.Hkv, p.d, p.P = 2, 512, 4, 4, 64, 16
    p.n_sink, p.n_recent = 4, 16
    lens, bp, br = i32x2(512, 300), i32x2(76, 40), i32x2(26, 10)
    assert lib.nacl_evict_varlen(None, lens, bp, br, 102) == -1
    assert lib.nacl_evict_varlen(C.byref(p), None, bp, br, 102) == -1
    assert lib.nacl_evict_varlen(C.byref(p), i32x2(512, 513), bp, br, 102) == -2  # longer than the padded length
    assert lib.nacl_evict_varlen(C.byref(p), i32x2(512, 0), bp, br, 102) == -2
    assert lib.nacl_evict_varlen(C.byref(p), lens, bp, br, 101) == -3             # an element's budget exceeds C_max
    # a LATER element that a batch-1 call would refuse is found before the first element is launched (here, without a
    # GPU, a launch would come back as -6): nothing is written on a validation error
    assert lib.nacl_evict_varlen(C.byref(p), i32x2(512, 15), bp, br, 102) == -2    # P = 16 proxy rows > 15 keys
    assert lib.nacl_evict_varlen(C.byref(p), i32x2(512, 18), i32x2(76, 18), i32x2(26, 0), 102) == -3   # protected 20 > 18 keys
    assert lib.nacl_evict_varlen(C.byref(p), lens, i32x2(76, 19), br, 102) == -3   # budget_proxy below the protected count
    assert lib.nacl_evict_varlen(C.byref(p), i32x2(512, 40), i32x2(76, 30), i32x2(26, 11), 102) == -3  # keeps more than it has
    p.lse_in = 0x7000
    assert lib.nacl_evict_varlen(C.byref(p), lens, bp, br, 102) == -7             # not offered for variable-length batches
    p.lse_in = None
    p.struct_size = 8
    assert lib.nacl_evict_varlen(C.byref(p), lens, bp, br, 102) == -7


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2408_03675_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "nacl_oracle" not in txt, f


def test_log_table_is_what_its_generator_writes():
    """csrc/logtab.inc (the constants behind the fp64 logarithm of the sampling keys) is reproducible: the tracked generator,
    which uses nothing but the standard library's arbitrary-precision decimal module, rewrites it bit for bit; and every
    entry agrees with libm (1/c and hi(ln c) to 1 ulp, hi + lo closer to ln c than a double can express)."""
    import math
    import subprocess
    import sys

    gen = os.path.join(ROOT, "paper_2408_03675_b200", "csrc", "gen_logtab.py")
    assert subprocess.run([sys.executable, gen, "--check"]).returncode == 0
    rows = re.findall(r"\{(\S+), (\S+), (\S+)\},", open(os.path.join(ROOT, "paper_2408_03675_b200", "csrc", "logtab.inc")).read())
    assert len(rows) == 92
    for i, (inv, hi, lo) in enumerate(rows):
        c = (90 + i) / 128.0
        inv, hi, lo = float.fromhex(inv), float.fromhex(hi), float.fromhex(lo)
        assert abs(inv - 1.0 / c) <= math.ulp(inv)
        assert abs(hi - math.log(c)) <= math.ulp(hi) if c != 1.0 else hi == 0.0
        assert abs(lo) <= math.ulp(hi) / 2 if c != 1.0 else lo == 0.0


def test_diagnostics_builds_are_refused_by_default(monkeypatch):
    """The -DNACL_* variants of the kernels (timing aids, some wrong by design) must not end up as the product library by
    accident: the build refuses them unless NACL_DIAGNOSTICS=1 is set."""
    monkeypatch.setenv("NACL_NVCC_EXTRA", "-DNACL_EPI_TRIVIAL")
    monkeypatch.delenv("NACL_DIAGNOSTICS", raising=False)
    with pytest.raises(RuntimeError, match="NACL_DIAGNOSTICS"):
        nacl_build.build(force=True)
    assert os.path.exists(nacl_build.LIB)  # the refused build left the product library alone
