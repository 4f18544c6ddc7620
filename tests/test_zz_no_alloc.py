"""nacl_evict_static: the eviction call for callers that cannot allocate device memory.

Some users of this library never get to call cudaMalloc after start-up: a serving engine whose KV-cache pool was given
the whole GPU, a decode loop that cannot afford the device-wide stall of cudaMalloc / cudaFree, a worker that lives
inside another program's allocator.  For them the library carries its kernels' scratch as a fixed 16 MiB array in its
own device image (include/nacl_evict.h, NACL_STATIC_SCRATCH_BYTES) and nacl_evict_static works in that array.

What is checked here, on a B200 (-m gpu):
  * its outputs equal those of the existing path (nacl_evict_ex with a workspace of the caller's) on calls that follow
    each other and differ in shape, so that each call finds the previous call's leftovers in the array -- index lists and
    compacted K/V bit for bit, importance within the 2e-3 relative tolerance of tests/parity.py;
  * once the kernels are loaded, a call with pre-allocated outputs leaves the driver's free-memory figure unchanged;
  * a shape whose scratch does not fit is refused with NACL_ERR_STATIC_LIMIT and nothing is written.

The file is named so that pytest collects it last: `pytest -x` stops at the first failure and a failure in here must
not hide the parity tests.  It passes alone in a fresh process (the first call does the per-device set-up) as well as
after the rest of the suite.
"""
import pytest
import torch

from paper_2408_03675_b200 import CONFIGS
from paper_2408_03675_b200.inputs import make_layer_inputs, make_random_inputs

from parity import ABS_TOL, REL_TOL

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def binding():
    from paper_2408_03675_b200 import binding as b  # raises if libnacl_evict.so is missing: no fallback

    assert torch.cuda.is_available()
    return b


def _existing_path(b, K, V, Q, Bp, Br, ns, nr, seed, layer, **kw):
    """The path the rest of the suite tests: nacl_evict_ex with a caller workspace (poisoned, as a reused one would be)."""
    B, Hkv, L, d = K.shape
    Hq, P = Q.shape[1], Q.shape[2]
    ws = torch.full((b.nacl_workspace_bytes(B, L, Hq, Hkv, d, P),), 0xA5, dtype=torch.uint8, device=K.device)
    return b.nacl_evict_ex(K, V, Q, Bp, Br, ns, nr, seed, layer, want_importance=True, workspace=ws, **kw)


def _same(got, want):
    assert torch.equal(got["out_idx"], want["out_idx"])
    assert torch.equal(got["out_K"].view(torch.uint8), want["out_K"].view(torch.uint8))
    assert torch.equal(got["out_V"].view(torch.uint8), want["out_V"].view(torch.uint8))
    g, w = got["importance"].double(), want["importance"].double()
    assert bool(((g - w).abs() <= REL_TOL * w.abs() + ABS_TOL).all())


def _cases():
    cfg = CONFIGS[2]  # 32 heads x 4096 keys, bf16: tensor-core path, one hand-over counter pair per head
    K, V, Q, _ = make_layer_inputs(cfg, layer=0, device="cuda")
    Bp, Br = cfg.budgets()
    big = (K, V, Q, Bp, Br, cfg.n_sink, cfg.n_recent, cfg.layer_seed(0), 0)
    # 4 heads, ragged length: its softmax partials land on the bytes that held the 32-head call's counters
    K2, V2, Q2 = make_random_inputs(2, 2049, 8, 2, 128, 32, dtype="bf16", seed=7, device="cuda")
    small = (K2, V2, Q2, 300, 100, 4, 32, 99, 5)
    # fp32: the CUDA-core kernels, another carve-up again
    K3, V3, Q3 = make_random_inputs(2, 333, 4, 2, 64, 5, dtype="f32", seed=11, device="cuda")
    generic = (K3, V3, Q3, 40, 13, 3, 7, 1234, 2)
    return big, small, generic


def test_static_scratch_call_equals_the_workspace_call_on_calls_in_a_row(binding):
    big, small, generic = _cases()
    want = [_existing_path(binding, *c) for c in (big, small, generic)]
    torch.cuda.synchronize()
    # back to back on one stream, no host synchronisation in between: big, small, big again, generic, small again
    order = [0, 1, 0, 2, 1]
    cases = (big, small, generic)
    got = [binding.nacl_evict_static(*cases[i], want_importance=True) for i in order]
    torch.cuda.synchronize()
    for i, g in zip(order, got):
        _same(g, want[i])
    # and the same call twice in a row is the same result twice (the array keeps nothing a call depends on)
    a = binding.nacl_evict_static(*big, want_importance=True)
    bb = binding.nacl_evict_static(*big, want_importance=True)
    torch.cuda.synchronize()
    _same(a, want[0])
    _same(bb, want[0])


def test_static_scratch_call_takes_no_device_memory(binding):
    big, small, _ = _cases()
    outs = []
    for c in (big, small):
        K, Cn = c[0], c[3] + c[4]
        oK = torch.empty((K.shape[0], K.shape[1], Cn, K.shape[3]), dtype=K.dtype, device="cuda")
        outs.append(dict(out_K=oK, out_V=torch.empty_like(oK),
                         out_idx=torch.empty(oK.shape[:3], dtype=torch.int32, device="cuda")))
    for c, o in zip((big, small), outs):  # loads the kernels and does the per-device set-up
        binding.nacl_evict_static(*c, **o)
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        for c, o in zip((big, small), outs):
            binding.nacl_evict_static(*c, **o)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after == free_before, f"device memory moved by {free_before - free_after} bytes"
    want = _existing_path(binding, *big)
    assert torch.equal(outs[0]["out_idx"], want["out_idx"])
    assert torch.equal(outs[0]["out_K"].view(torch.uint8), want["out_K"].view(torch.uint8))


def test_static_scratch_call_refuses_shapes_beyond_its_limit(binding):
    # 4 x 16 heads x 32768 keys want ~29 MiB of scratch: over the 16 MiB the library carries
    B, L, Hq, Hkv, d, P = 4, 32768, 16, 16, 128, 16
    assert binding.nacl_workspace_bytes(B, L, Hq, Hkv, d, P) > binding.STATIC_SCRATCH_BYTES
    K = torch.zeros((B, Hkv, L, d), dtype=torch.bfloat16, device="cuda")
    Q = torch.zeros((B, Hq, P, d), dtype=torch.bfloat16, device="cuda")
    oK = torch.full((B, Hkv, 64, d), 7.0, dtype=torch.bfloat16, device="cuda")
    oV = oK.clone()
    oidx = torch.full((B, Hkv, 64), -5, dtype=torch.int32, device="cuda")
    with pytest.raises(binding.NaclError) as ei:
        binding.nacl_evict_static(K, K, Q, 48, 16, 4, 16, 0, 0, out_K=oK, out_V=oV, out_idx=oidx)
    assert ei.value.code == -8 and "NACL_STATIC_SCRATCH_BYTES" in str(ei.value)
    torch.cuda.synchronize()
    assert bool((oidx == -5).all()) and bool((oK == 7.0).all()) and bool((oV == 7.0).all())
    # every configuration BASELINE.json names fits
    for cfg in CONFIGS.values():
        assert binding.nacl_workspace_bytes(cfg.batch, cfg.L, cfg.Hq, cfg.Hkv, cfg.d, cfg.P) <= binding.STATIC_SCRATCH_BYTES
    with pytest.raises(ValueError):
        binding.nacl_evict_static(K, K, Q, 48, 16, 4, 16, 0, 0, workspace=torch.empty(1, device="cuda"))
