"""Parity of the CUDA path (through the C ABI) against the fp64 CPU oracle, element by element,
on the same seeded inputs.  Protocol: tests/parity.py.  Needs a B200: run with -m gpu."""
import numpy as np
import pytest
import torch

import oracle
from paper_2408_03675_b200 import CONFIGS
from paper_2408_03675_b200.inputs import make_layer_inputs, make_random_inputs

from parity import full_parity

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def binding():
    from paper_2408_03675_b200 import binding as b  # raises if libnacl_evict.so is missing: no fallback

    assert torch.cuda.is_available()
    return b


@pytest.mark.parametrize("cid", [1, 2])
def test_baseline_configs_small(binding, cid):
    cfg = CONFIGS[cid]
    K, V, Q, planted = make_layer_inputs(cfg, layer=0)
    Bp, Br = cfg.budgets()
    r = full_parity(K, V, Q, Bp, Br, cfg.n_sink, cfg.n_recent, cfg.layer_seed(0), 0)
    # P11: planted heavy hitters are all kept
    for hk in range(cfg.Hkv):
        assert set(planted[0, hk].tolist()) <= set(r["idx_gpu"][0, hk].tolist())
    print(f"cfg{cid}: max rel err {r['max_rel_err']:.2e}, top-k swaps {r['topk_swaps']}, random diffs {r['random_diffs']}")


@pytest.mark.parametrize("cid,layer", [(3, 0), (4, 0), (4, 17), (5, 31)])
def test_baseline_configs_full_size(binding, cid, layer):
    """One whole layer of the 32-layer workloads at BASELINE.json's full sizes, in the launch configuration
    bench.py times (same entry point, same shapes); the oracle finishes a layer in seconds, so every output is
    compared, not a sample."""
    cfg = CONFIGS[cid]
    K, V, Q, planted = make_layer_inputs(cfg, layer=layer)
    Bp, Br = cfg.budgets()
    r = full_parity(K, V, Q, Bp, Br, cfg.n_sink, cfg.n_recent, cfg.layer_seed(layer), layer)
    for b in range(cfg.batch):
        for hk in range(cfg.Hkv):
            assert set(planted[b, hk].tolist()) <= set(r["idx_gpu"][b, hk].tolist())
    print(f"cfg{cid} layer {layer}: max rel err {r['max_rel_err']:.2e}, top-k swaps {r['topk_swaps']}, random diffs {r['random_diffs']}")


# (B, L, Hq, Hkv, d, P, dtype, Bp, Br, n_sink, n_recent): several tiles + ragged tails, GQA, both dtypes
RAGGED = [
    (2, 333, 4, 2, 64, 5, "f32", 40, 13, 3, 7),
    (1, 1000, 8, 2, 128, 16, "bf16", 150, 50, 4, 16),     # G*P = 64
    (2, 2049, 8, 2, 128, 32, "bf16", 300, 100, 4, 32),    # G*P = 128, one key past a tile
    (1, 4100, 32, 8, 128, 64, "bf16", 600, 200, 4, 64),   # G*P = 256
    (1, 777, 4, 4, 128, 16, "bf16", 100, 30, 0, 16),      # G*P = 16, no sinks
    (1, 129, 6, 2, 32, 3, "bf16", 20, 5, 1, 3),           # small d, odd G*P -> CUDA-core path
    (3, 515, 2, 1, 256, 7, "f32", 64, 16, 2, 7),          # d = 256
    (1, 5000, 16, 16, 128, 48, "bf16", 750, 250, 4, 48),  # G*P = 48
    (1, 1500, 8, 2, 128, 128, "bf16", 300, 75, 4, 128),   # G*P = 512: two 256-row blocks on the tensor-core path
    (2, 900, 6, 2, 128, 256, "bf16", 300, 45, 4, 256),    # G*P = 768: three row blocks, P = 256 proxy rows
]


@pytest.mark.parametrize("case", RAGGED, ids=lambda c: f"B{c[0]}_L{c[1]}_H{c[2]}-{c[3]}_d{c[4]}_P{c[5]}_{c[6]}")
def test_ragged_shapes(binding, case):
    B, L, Hq, Hkv, d, P, dt, Bp, Br, ns, nr = case
    K, V, Q = make_random_inputs(B, L, Hq, Hkv, d, P, dtype=dt, seed=L)
    full_parity(K, V, Q, Bp, Br, ns, nr, seed=12345, layer=3)


@pytest.mark.parametrize("dt,d", [("f32", 64), ("bf16", 128)])
def test_cuda_core_flag_matches_default_path(binding, dt, d):
    K, V, Q = make_random_inputs(1, 900, 8, 2, d, 16, dtype=dt, seed=5)
    full_parity(K, V, Q, 120, 40, 4, 16, seed=9, layer=1, flags=binding.FLAG_SCORE_CUDA_CORES, oracle_flags=0)


def test_edge_budgets(binding):
    K, V, Q = make_random_inputs(1, 300, 4, 2, 64, 4, dtype="f32", seed=1)
    L = 300
    # Br = 0: protected + pure top-k (north star); C = L: identity; all protected; nothing but protected
    full_parity(K, V, Q, 50, 0, 4, 4, seed=0, layer=0)
    r = full_parity(K, V, Q, 200, 100, 4, 4, seed=0, layer=0)
    np.testing.assert_array_equal(r["idx_gpu"][0, 0], np.arange(L))
    full_parity(K, V, Q, L, 0, 100, 200, seed=0, layer=0)
    full_parity(K, V, Q, 8, 0, 4, 4, seed=0, layer=0)
    full_parity(K, V, Q, 8, 292, 4, 4, seed=0, layer=0)
    full_parity(K, V, Q, 0, 1, 0, 0, seed=0, layer=0)
    full_parity(K, V, Q, 1, 0, 0, 0, seed=0, layer=0)
    # C = 0: empty outputs, no error
    res = binding.nacl_evict_ex(K.cuda(), V.cuda(), Q.cuda(), 0, 0, 0, 0, 0, 0)
    assert res["out_idx"].shape == (1, 2, 0)


def test_tiny_lengths(binding):
    for L, P in [(1, 1), (2, 2), (17, 1), (64, 64)]:
        K, V, Q = make_random_inputs(1, L, 2, 2, 64, P, dtype="f32", seed=L)
        full_parity(K, V, Q, max(1, L // 2), L // 4, 0, min(P, max(1, L // 2)), seed=7, layer=2)


def test_identical_keys_tie_to_lower_index(binding):
    # all keys equal -> uniform importance G*P/L (closed form): every top-k decision is a tie
    for dt, d in [("f32", 64), ("bf16", 128)]:
        K, V, Q = make_random_inputs(1, 1500, 4, 2, d, 8, dtype=dt, seed=3)
        K[:] = K[:, :, :1, :]
        r = full_parity(K, V, Q, 200, 0, 2, 8, seed=1, layer=0)
        np.testing.assert_array_equal(r["idx_gpu"][0, 0][:192], np.arange(192))
        full_parity(K, V, Q, 200, 77, 2, 8, seed=1, layer=0)


def test_zero_importance_and_huge_logits(binding):
    # one dominant key (huge norm along a query direction): importance underflows to 0 elsewhere (R13)
    K, V, Q = make_random_inputs(1, 700, 2, 2, 64, 4, dtype="f32", seed=11)
    Q[:] = Q[:, :, :1, :]
    K[0, :, 100] = 300.0 * Q[0, :, 0] / Q[0, :, 0].norm(dim=-1, keepdim=True)
    r = full_parity(K, V, Q, 50, 20, 2, 4, seed=1, layer=0)
    assert (r["imp_gpu"] == 0).sum() > 0
    # shift invariance: adding a vector to every key leaves the importance unchanged up to rounding
    K2, V2, Q2 = make_random_inputs(1, 600, 4, 4, 64, 8, dtype="f32", seed=12)
    full_parity(K2, V2, Q2, 90, 30, 4, 8, seed=2, layer=0)


@pytest.mark.parametrize("flag", ["uniform", "softmax_of_score"])
def test_sampling_variant_flags(binding, flag):
    f = binding.FLAG_SAMPLE_UNIFORM if flag == "uniform" else binding.FLAG_SAMPLE_SOFTMAX_OF_SCORE
    K, V, Q = make_random_inputs(1, 800, 4, 2, 128, 16, dtype="bf16", seed=21)
    full_parity(K, V, Q, 100, 60, 4, 16, seed=5, layer=4, flags=f)


def test_seed_layer_head_keying(binding):
    cfg = CONFIGS[1]
    K, V, Q, _ = make_layer_inputs(cfg, layer=0)
    Bp, Br = cfg.budgets()
    dev = "cuda:0"
    a = binding.nacl_evict(K.to(dev), V.to(dev), Q.to(dev), Bp, Br, cfg.n_sink, cfg.n_recent, 0, 0)[2]
    b = binding.nacl_evict(K.to(dev), V.to(dev), Q.to(dev), Bp, Br, cfg.n_sink, cfg.n_recent, 1, 0)[2]
    c = binding.nacl_evict(K.to(dev), V.to(dev), Q.to(dev), Bp, Br, cfg.n_sink, cfg.n_recent, 0, 1)[2]
    big = binding.nacl_evict(K.to(dev), V.to(dev), Q.to(dev), Bp, Br, cfg.n_sink, cfg.n_recent, (1 << 40) + 5, 0)[2]
    assert not torch.equal(a, b) and not torch.equal(a, c) and not torch.equal(a, big)
    ref = oracle.evict(K, V, Q, Bp, Br, cfg.n_sink, cfg.n_recent, (1 << 40) + 5, 0)[2]
    np.testing.assert_array_equal(big.cpu().numpy(), ref)


def test_host_entry_point_matches_device_entry_point(binding):
    cfg = CONFIGS[1]
    K, V, Q, _ = make_layer_inputs(cfg, layer=0)
    Bp, Br = cfg.budgets()
    oK, oV, idx = binding.nacl_evict_host(K.pin_memory(), V.pin_memory(), Q.pin_memory(), Bp, Br, cfg.n_sink, cfg.n_recent, 0, 0)
    dK, dV, didx = binding.nacl_evict(K.cuda(), V.cuda(), Q.cuda(), Bp, Br, cfg.n_sink, cfg.n_recent, 0, 0)
    assert torch.equal(idx, didx.cpu()) and torch.equal(oK, dK.cpu()) and torch.equal(oV, dV.cpu())


def test_caller_workspace_and_graph_capture(binding):
    cfg = CONFIGS[2]
    K, V, Q, _ = make_layer_inputs(cfg, layer=0)
    Bp, Br = cfg.budgets()
    Kd, Vd, Qd = K.cuda(), V.cuda(), Q.cuda()
    want = binding.nacl_evict(Kd, Vd, Qd, Bp, Br, cfg.n_sink, cfg.n_recent, 0, 0)
    ws = torch.empty(binding.nacl_workspace_bytes(cfg.batch, cfg.L, cfg.Hq, cfg.Hkv, cfg.d, cfg.P), dtype=torch.uint8, device="cuda")
    oK, oV, oi = torch.empty_like(want[0]), torch.empty_like(want[1]), torch.empty_like(want[2])
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        binding.nacl_evict_ex(Kd, Vd, Qd, Bp, Br, cfg.n_sink, cfg.n_recent, 0, 0, out_K=oK, out_V=oV, out_idx=oi, workspace=ws)  # warm
        s.synchronize()
        g = torch.cuda.CUDAGraph()
        oi.zero_()
        with torch.cuda.graph(g, stream=s):
            binding.nacl_evict_ex(Kd, Vd, Qd, Bp, Br, cfg.n_sink, cfg.n_recent, 0, 0, out_K=oK, out_V=oV, out_idx=oi, workspace=ws, stream=s)
        g.replay()
        s.synchronize()
    assert torch.equal(oi, want[2]) and torch.equal(oK, want[0]) and torch.equal(oV, want[1])


@pytest.mark.parametrize("flag_name", ["default", "FLAG_SAMPLE_SOFTMAX_OF_SCORE", "FLAG_SAMPLE_UNIFORM"])
def test_gumbel_keys_bitwise_against_the_oracle(binding, flag_name):
    """The sampling keys (Philox uniforms, two fp64 logarithms by the library's table-driven routine, one rounding to
    fp32: DESIGN.md R15) against the oracle's libm keys for 2^20 positions whose importances span 40 decades, including
    0 and fp32 subnormals.  Both logs are accurate to ~1 ulp of fp64, so a key can differ only where the fp64 sum falls
    within ~1e-16 (relative) of an fp32 rounding boundary: at most a few positions in 10^6, and never by more than 1 ulp."""
    flags = 0 if flag_name == "default" else getattr(binding, flag_name)
    B, Hkv, L = 2, 4, 131072
    rng = np.random.default_rng(7)
    imp = np.exp(rng.uniform(-92.0, 5.5, size=(B, Hkv, L))).astype(np.float32)
    imp[0, 0, :64] = 0.0
    imp[0, 1, :64] = np.float32(1e-42)          # subnormal
    imp[1, 2, :1024] = np.float32(1.0) + np.arange(1024, dtype=np.float32) * np.float32(2.0 ** -23)  # around ln = 0
    if flags == binding.FLAG_SAMPLE_SOFTMAX_OF_SCORE:
        imp = np.minimum(imp, np.float32(64.0))
    seed, layer = 0x1234_5678_9ABC_DEF0, 5
    keys_gpu = binding.nacl_gumbel_keys(torch.from_numpy(imp).cuda(), seed, layer, flags).cpu().numpy()
    # all non-protected positions are candidates when nothing is kept by the top-k: Bp = |Pi| = 0, Br = 1
    _, keys_ref = oracle.select(imp, 0, 1, 0, 0, seed, layer, flags & 0x7, return_keys=True)
    assert not np.isnan(keys_ref).any()
    a, b = keys_gpu.view(np.int32).astype(np.int64), keys_ref.view(np.int32).astype(np.int64)
    diff = a != b
    n_diff = int(diff.sum())
    assert n_diff <= 8, f"{n_diff} of {a.size} keys differ"
    if n_diff:
        assert np.abs(a[diff] - b[diff]).max() <= 1  # neighbouring floats (same sign: no key sits at +-0 here)
    print(f"{flag_name}: {n_diff} of {a.size} keys differ by 1 ulp")


@pytest.mark.parametrize("case", [(1, 4100, 32, 8, 128, 64, "bf16"), (2, 1500, 8, 4, 128, 16, "bf16"), (2, 700, 4, 2, 64, 5, "f32"),
                                  (1, 1100, 8, 2, 128, 128, "bf16")],
                         ids=["tc_GP256", "tc_GP32", "cuda_core_f32", "tc_GP512_row_blocks"])
def test_lse_in_single_sweep(binding, case):
    """SURVEY.md 8(f) f1 / the contract of the paper's Algorithm 2: with the row log-sum-exps
    supplied, one logit sweep gives the same importance (north-star tolerance) and, on it, exactly the oracle's selection."""
    from parity import check_scores, check_staged, check_structure, check_gather

    B, L, Hq, Hkv, d, P, dt = case
    K, V, Q = make_random_inputs(B, L, Hq, Hkv, d, P, dtype=dt, seed=L + 1)
    imp_ref, lse_ref = oracle.importance(K, Q, return_lse=True)
    Bp, Br, ns, nr = L // 6, L // 20, 4, P
    lse_in = torch.from_numpy(lse_ref.astype(np.float32)).cuda()
    res = binding.nacl_evict_ex(K.cuda(), V.cuda(), Q.cuda(), Bp, Br, ns, nr, 77, 2, want_importance=True, want_lse=True,
                                lse_in=lse_in)
    torch.cuda.synchronize()
    imp = res["importance"].cpu().numpy()
    idx = res["out_idx"].cpu().numpy()
    check_scores(imp, imp_ref, Hq // Hkv, P)
    check_structure(idx, L, Bp + Br, ns, nr)
    check_staged(idx, imp, Bp, Br, ns, nr, 77, 2)
    check_gather(K, V, res["out_K"].cpu(), res["out_V"].cpu(), idx)
    np.testing.assert_allclose(res["lse"].cpu().numpy(), lse_ref, rtol=1e-6, atol=1e-6)
    # and it agrees with the self-contained two-sweep call to the score tolerance
    res2 = binding.nacl_evict_ex(K.cuda(), V.cuda(), Q.cuda(), Bp, Br, ns, nr, 77, 2, want_importance=True)
    np.testing.assert_allclose(res2["importance"].cpu().numpy(), imp, rtol=2e-3, atol=1e-30)


@pytest.mark.parametrize("case", [(1, 4100, 32, 8, 128, 64, "bf16"), (2, 1000, 8, 2, 128, 48, "bf16"), (1, 300, 4, 4, 128, 16, "bf16"),
                                  (2, 333, 4, 2, 64, 5, "f32"), (1, 130, 6, 2, 32, 130, "bf16"), (1, 1300, 8, 2, 128, 128, "bf16")],
                         ids=["tc_GP256_ragged", "tc_GP192", "tc_GP16", "cuda_core_f32", "all_rows_proxy", "tc_GP512_row_blocks"])
def test_causal_flag(binding, case):
    """NACL_FLAG_CAUSAL (R1): proxy row i is prompt position L-P+i and attends keys j <= L-P+i only.  The last
    case makes every prompt row a proxy row: accumulated causal attention (the H2O one-shot case)."""
    B, L, Hq, Hkv, d, P, dt = case
    K, V, Q = make_random_inputs(B, L, Hq, Hkv, d, P, dtype=dt, seed=L + 3)
    nr = min(P, L // 2)
    Bp, Br = max(L // 6, 4 + nr), L // 20
    full_parity(K, V, Q, Bp, Br, 4, nr, seed=5, layer=1, flags=binding.FLAG_CAUSAL)


@pytest.mark.parametrize("case", [(1, 200000, 2, 1, 64, 8, "bf16"), (1, 330001, 1, 1, 64, 4, "bf16"), (2, 70000, 8, 2, 128, 32, "bf16")],
                         ids=["one_head_200k_cluster16", "row_too_long_for_a_cluster", "tc_70k_cluster8"])
def test_long_rows(binding, case):
    """Rows of 70k-330k keys: the largest cluster sizes of the select kernel and, past 16 x 20480 keys, the fallback
    with a separate keys kernel, a single-CTA select working out of global memory and the stand-alone gather."""
    B, L, Hq, Hkv, d, P, dt = case
    K, V, Q = make_random_inputs(B, L, Hq, Hkv, d, P, dtype=dt, seed=L % 1000)
    full_parity(K, V, Q, L // 8, L // 40, 4, P, seed=L, layer=7)
