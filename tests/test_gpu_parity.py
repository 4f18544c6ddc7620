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


@pytest.mark.parametrize("cid,layer", [(c, l) for c in (3, 4, 5) for l in (0, 10, 21, 31)])
def test_baseline_configs_full_size(binding, cid, layer):
    """Four whole layers (first, last, two others: SURVEY.md 8(d)) of each 32-layer workload at BASELINE.json's full
    sizes through the single-call form (nacl_evict_ex: fused scoring launch, selection over the whole GPU); the launch
    configuration bench.py times is test_timed_configuration_full_size below.  The oracle finishes a layer in seconds,
    so every output is compared, not a sample."""
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
    (1, 1200, 8, 2, 128, 100, "bf16", 300, 60, 4, 100),   # G*P = 400 = 256 + 144: the last row block is partial (masked)
    (2, 700, 4, 1, 128, 68, "bf16", 200, 30, 4, 68),      # G*P = 272 = 256 + 16
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


def test_fused_scoring_launch_matches_two_launches(binding):
    """The tensor-core path runs both sweeps in ONE cooperative launch (per-head hand-over counters between the CTAs);
    NACL_FLAG_SCORE_TWO_LAUNCHES runs them as two launches.  Same arithmetic in the same order: bit-identical importance,
    indices and caches.  Shapes alternate so that the self-cleaning counters are reused at different sizes."""
    shapes = [(1, 4100, 32, 8, 128, 64), (4, 700, 8, 8, 128, 16), (2, 9000, 16, 2, 128, 32), (1, 129, 8, 8, 128, 16),
              (1, 1200, 8, 2, 128, 100), (4, 700, 8, 8, 128, 16), (1, 4100, 32, 8, 128, 64)]
    for rep, (B, L, Hq, Hkv, d, P) in enumerate(shapes):
        K, V, Q = make_random_inputs(B, L, Hq, Hkv, d, P, dtype="bf16", seed=100 + rep)
        Kc, Vc, Qc = K.cuda(), V.cuda(), Q.cuda()
        Bp, Br = L // 5, L // 20
        a = binding.nacl_evict_ex(Kc, Vc, Qc, Bp, Br, 4, P, 3, rep, want_importance=True)
        b = binding.nacl_evict_ex(Kc, Vc, Qc, Bp, Br, 4, P, 3, rep, flags=binding.FLAG_SCORE_TWO_LAUNCHES, want_importance=True)
        for k in ("importance", "out_idx", "out_K", "out_V"):
            assert torch.equal(a[k], b[k]), f"shape {rep}: {k} differs between the fused and the two-launch scoring"
    full_parity(K, V, Q, Bp, Br, 4, P, seed=3, layer=1)


FAST_CASES = [
    # B, L, Hq, Hkv, d, P, dtype, Bp, Br, n_sink, n_recent, flags
    (1, 32768, 8, 2, 128, 64, "bf16", 4915, 1638, 4, 64, 0),        # a cfg-4 head shape: clusters of 4, 8192 positions per CTA
    (2, 16384, 4, 4, 128, 32, "bf16", 2457, 819, 4, 32, 0),
    (1, 4096, 8, 8, 128, 32, "bf16", 614, 205, 4, 32, 0),
    (1, 9000, 8, 2, 128, 16, "bf16", 1800, 450, 4, 16, 2),           # weight exp(importance)
    (1, 9000, 8, 2, 128, 16, "bf16", 1800, 450, 4, 16, 4),           # uniform weights
    (2, 3001, 4, 2, 64, 8, "f32", 500, 333, 3, 8, 0),                # CUDA-core scoring, ragged slices
    (1, 5000, 4, 4, 128, 16, "bf16", 4000, 900, 4, 16, 0),           # almost everything kept
    (1, 5000, 4, 4, 128, 16, "bf16", 21, 1, 4, 16, 0),               # one top-k element, one sample
    (1, 5000, 4, 4, 128, 16, "bf16", 20, 300, 4, 16, 0),             # no top-k at all
    (1, 131072, 4, 1, 128, 64, "bf16", 10485, 2622, 4, 64, 0),       # a cfg-5 head: cluster of 16
    (1, 131072, 8, 8, 128, 8, "bf16", 10485, 2622, 4, 64, 0),        # cfg-5 rows on 8 heads: 16 positions per thread
    (1, 70000, 6, 6, 128, 16, "bf16", 9000, 3000, 4, 16, 0),
]


@pytest.mark.parametrize("case", FAST_CASES, ids=lambda c: f"B{c[0]}_L{c[1]}_H{c[2]}-{c[3]}_P{c[5]}_{c[6]}_Bp{c[7]}_Br{c[8]}_f{c[11]}")
def test_fast_selection_matches_general_path(binding, case):
    """The one-pass bucket selection (windowed buckets for the top-k, fp32 key estimates + exact keys next to the
    threshold for the sample) takes the same decisions as the three-pass radix path on exact keys, bit for bit, and as
    the oracle's steps 4-7 on the same importance; on these shapes it must not fall back."""
    B, L, Hq, Hkv, d, P, dt, Bp, Br, ns, nr, flags = case
    K, V, Q = make_random_inputs(B, L, Hq, Hkv, d, P, dtype=dt, seed=L + Bp)
    Kc, Vc, Qc = K.cuda(), V.cuda(), Q.cuda()
    binding.nacl_select_fallbacks(reset=True)
    a = binding.nacl_evict_ex(Kc, Vc, Qc, Bp, Br, ns, nr, 77, 5, flags=flags, want_importance=True)
    torch.cuda.synchronize()
    assert binding.nacl_select_fallbacks(reset=True) == 0, "the fast selection path fell back to the general one"
    b = binding.nacl_evict_ex(Kc, Vc, Qc, Bp, Br, ns, nr, 77, 5, flags=flags | binding.FLAG_SELECT_GENERAL, want_importance=True)
    for k in ("importance", "out_idx", "out_K", "out_V"):
        assert torch.equal(a[k], b[k]), f"{k} differs between the fast and the general selection"
    ref = oracle.select(a["importance"].cpu().numpy(), Bp, Br, ns, nr, 77, 5, flags=flags)
    np.testing.assert_array_equal(a["out_idx"].cpu().numpy(), ref)


def test_fast_selection_falls_back_on_degenerate_rows(binding):
    """All-equal importance (every top-k decision is a tie: the threshold bucket holds the whole row), rows that are mostly
    zero importance (keys of -inf), and protected positions marked +inf: the fast path must give up or handle them, with
    the oracle's result either way."""
    K, V, Q = make_random_inputs(1, 20000, 4, 2, 128, 8, dtype="bf16", seed=3)
    K[:] = K[:, :, :1, :]
    full_parity(K, V, Q, 3000, 1000, 2, 8, seed=1, layer=0)
    K2, V2, Q2 = make_random_inputs(1, 6000, 2, 2, 128, 16, dtype="bf16", seed=11)
    Q2[:] = Q2[:, :, :1, :]
    K2[0, :, 100:130] = (300.0 * Q2[0, :, :1] / Q2[0, :, :1].float().norm(dim=-1, keepdim=True)).to(K2.dtype)
    r = full_parity(K2, V2, Q2, 500, 400, 2, 16, seed=1, layer=0)
    assert (r["imp_gpu"] == 0).sum() > 0


def test_concurrent_streams_keep_their_results_apart(binding):
    """Two streams evict different problems at the same time through the library's own (device, stream) workspaces: the
    cooperative scoring launches serialise instead of deadlocking, the hand-over counters of one call never meet the other's."""
    shapes = [(2, 6000, 16, 4, 128, 16), (1, 9000, 8, 8, 128, 32)]
    data = []
    for rep, (B, L, Hq, Hkv, d, P) in enumerate(shapes):
        K, V, Q = make_random_inputs(B, L, Hq, Hkv, d, P, dtype="bf16", seed=40 + rep)
        data.append((K.cuda(), V.cuda(), Q.cuda(), L // 5, L // 20, P))
    want = [binding.nacl_evict_ex(K, V, Q, Bp, Br, 4, P, 9, 1) for K, V, Q, Bp, Br, P in data]
    torch.cuda.synchronize()
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    got = [[], []]
    for it in range(6):
        for si, st in enumerate(streams):
            K, V, Q, Bp, Br, P = data[si]
            with torch.cuda.stream(st):
                got[si].append(binding.nacl_evict_ex(K, V, Q, Bp, Br, 4, P, 9, 1, stream=st))
    torch.cuda.synchronize()
    for si in range(2):
        for r in got[si]:
            for k in ("out_idx", "out_K", "out_V"):
                assert torch.equal(r[k], want[si][k]), f"stream {si}: {k} differs from the single-stream result"


@pytest.mark.parametrize("case", [(3, 5000, 8, 2, 128, 16, "bf16"), (2, 700, 4, 4, 64, 4, "f32")], ids=["tc", "cuda_core"])
def test_varlen_batch_matches_one_call_per_prompt(binding, case):
    """nacl_evict_varlen: a padded batch whose prompts have different lengths and budgets.  Every
    element must come out exactly as a batch-1 call on its own live rows with batch_offset = b (same Philox streams), and
    that call's index list must be the oracle's on the same importance; nothing is written past an element's own C rows."""
    B, Lmax, Hq, Hkv, d, P, dt = case
    K, V, Q = make_random_inputs(B, Lmax, Hq, Hkv, d, P, dtype=dt, seed=77)
    lens = [Lmax, Lmax * 3 // 5 + 1, Lmax // 4 + 3][:B]
    bps = [l // 6 for l in lens]
    brs = [l // 17 for l in lens]
    ns, nr = 4, P
    # element b's proxy queries are the last P positions of ITS prompt: Q as given stands for them
    Kc, Vc, Qc = K.cuda(), V.cuda(), Q.cuda()
    res = binding.nacl_evict_varlen(Kc, Vc, Qc, lens, bps, brs, ns, nr, 11, 2)
    torch.cuda.synchronize()
    for b in range(B):
        Kb, Vb, Qb = K[b:b + 1, :, :lens[b]].contiguous(), V[b:b + 1, :, :lens[b]].contiguous(), Q[b:b + 1].contiguous()
        one = binding.nacl_evict_ex(Kb.cuda(), Vb.cuda(), Qb.cuda(), bps[b], brs[b], ns, nr, 11, 2, batch_offset=b, want_importance=True)
        Cb = bps[b] + brs[b]
        assert torch.equal(res["out_idx"][b], one["out_idx"][0])
        assert torch.equal(res["out_K"][b, :, :Cb], one["out_K"][0]) and torch.equal(res["out_V"][b, :, :Cb], one["out_V"][0])
        assert (res["out_K"][b, :, Cb:] == 0).all() and (res["out_V"][b, :, Cb:] == 0).all()
        ref = oracle.select(one["importance"].cpu().numpy(), bps[b], brs[b], ns, nr, 11, 2, batch_offset=b)
        np.testing.assert_array_equal(one["out_idx"].cpu().numpy(), ref)
        imp_ref = oracle.importance(Kb, Qb)
        rel = np.abs(one["importance"].cpu().numpy() - imp_ref) / (np.abs(imp_ref) + 1e-30)
        assert rel.max() <= 2e-3


@pytest.mark.parametrize("layout", ["HND", "NHD"])
@pytest.mark.parametrize("case", [(2, 5000, 8, 2, 128, 32, 16), (1, 4100, 32, 8, 128, 64, 64), (3, 777, 4, 4, 128, 16, 8),
                                  (1, 70000, 8, 2, 128, 16, 128), (2, 300, 8, 8, 128, 16, 32)],
                         ids=lambda c: f"B{c[0]}_L{c[1]}_H{c[2]}-{c[3]}_P{c[5]}_page{c[6]}")
def test_paged_kv_matches_the_contiguous_call(binding, case, layout):
    """Paged K/V (block table): the pages of every prompt are scattered over a shuffled pool (with
    spare pages and a padded table); importance, kept positions and compacted caches must be bit-identical to the
    contiguous call on the same values, which itself is checked against the oracle."""
    B, L, Hq, Hkv, d, P, ps = case
    K, V, Q = make_random_inputs(B, L, Hq, Hkv, d, P, dtype="bf16", seed=L + ps)
    Bp, Br = L // 5, L // 20
    want = binding.nacl_evict_ex(K.cuda(), V.cuda(), Q.cuda(), Bp, Br, 4, P, 21, 3, want_importance=True)
    npp = (L + ps - 1) // ps                      # pages per prompt
    n_pages = B * npp + 5                         # spare pages that belong to nobody
    g = torch.Generator().manual_seed(ps)
    perm = torch.randperm(n_pages, generator=g)[:B * npp].view(B, npp)
    table = torch.full((B, npp + 3), -1, dtype=torch.int32)   # padded table: entries past the last page are never read
    table[:, :npp] = perm.to(torch.int32)
    Kp = torch.full((n_pages, Hkv, ps, d), float("nan"), dtype=torch.bfloat16)   # stale / foreign pages hold NaN
    Vp = torch.full((n_pages, Hkv, ps, d), float("nan"), dtype=torch.bfloat16)
    pad = npp * ps - L
    Kpad = torch.cat([K, torch.full((B, Hkv, pad, d), float("nan"), dtype=K.dtype)], dim=2) if pad else K
    Vpad = torch.cat([V, torch.full((B, Hkv, pad, d), float("nan"), dtype=V.dtype)], dim=2) if pad else V
    for b in range(B):
        Kp[perm[b]] = Kpad[b].view(Hkv, npp, ps, d).transpose(0, 1)
        Vp[perm[b]] = Vpad[b].view(Hkv, npp, ps, d).transpose(0, 1)
    if layout == "NHD":
        Kp, Vp = Kp.transpose(1, 2).contiguous(), Vp.transpose(1, 2).contiguous()
    got = binding.nacl_evict_paged(Kp.cuda(), Vp.cuda(), table.cuda(), L, Q.cuda(), Bp, Br, 4, P, 21, 3, pool_layout=layout,
                                   want_importance=True)
    torch.cuda.synchronize()
    for k in ("importance", "out_idx", "out_K", "out_V"):
        assert torch.equal(got[k], want[k]), f"{k} differs between the paged and the contiguous call"
    ref = oracle.select(want["importance"].cpu().numpy(), Bp, Br, 4, P, 21, 3)
    np.testing.assert_array_equal(got["out_idx"].cpu().numpy(), ref)


@pytest.mark.parametrize("case", [(2, 9000, 8, 2, 128, 16, "bf16", 0.2), (1, 32768, 8, 2, 128, 64, "bf16", 0.2),
                                  (1, 20000, 4, 4, 128, 16, "bf16", 0.7), (2, 3001, 4, 2, 64, 8, "f32", 0.45),
                                  (1, 131072, 4, 1, 128, 16, "bf16", 0.1), (3, 700, 4, 4, 128, 16, "bf16", 0.95)],
                         ids=lambda c: f"B{c[0]}_L{c[1]}_H{c[2]}-{c[3]}_{c[6]}_keep{c[7]}")
def test_in_place_compaction(binding, case):
    """out_K == K, out_V == V (a cache [B,Hkv,cap,d] compacted inside its own buffers): the first C rows of every head
    must be exactly what the out-of-place call writes, the rows behind them untouched, the index list the same -- also
    when most rows are kept (every kept row below C is the source of another row's destination)."""
    B, L, Hq, Hkv, d, P, dt, keep = case
    K, V, Q = make_random_inputs(B, L, Hq, Hkv, d, P, dtype=dt, seed=L + 1)
    Bp = int(L * keep * 0.75)
    Br = int(L * keep) - Bp
    Cn = Bp + Br
    Kc, Vc, Qc = K.cuda(), V.cuda(), Q.cuda()
    want = binding.nacl_evict_ex(Kc, Vc, Qc, Bp, Br, 4, P, 5, 1)
    K2, V2 = Kc.clone(), Vc.clone()
    idx = torch.empty_like(want["out_idx"])
    binding.nacl_evict_ex(K2, V2, Qc, Bp, Br, 4, P, 5, 1, out_K=K2, out_V=V2, out_idx=idx)
    torch.cuda.synchronize()
    assert torch.equal(idx, want["out_idx"])
    assert torch.equal(K2[:, :, :Cn], want["out_K"]) and torch.equal(V2[:, :, :Cn], want["out_V"])
    assert torch.equal(K2[:, :, Cn:], Kc[:, :, Cn:]) and torch.equal(V2[:, :, Cn:], Vc[:, :, Cn:])
    # a second, different call on the compacted cache must see a valid cache (no torn rows): compare with a copy
    rows = K2[:, :, :Cn].contiguous()
    assert torch.equal(rows, want["out_K"])


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


def test_host_batch_entry_point_matches_single_calls(binding):
    """nacl_evict_host_batch: five problems of one shape out of pinned host memory, pipelined over two staging slots; every
    result must equal the device entry point's on the same inputs (seeds and layers differ per problem)."""
    cfg = CONFIGS[2]
    Bp, Br = cfg.budgets()
    Cn = Bp + Br
    probs = [make_layer_inputs(cfg, layer=l)[:3] for l in range(5)]
    Ks, Vs, Qs = [p[0].pin_memory() for p in probs], [p[1].pin_memory() for p in probs], [p[2].pin_memory() for p in probs]
    oKs = [torch.empty((cfg.batch, cfg.Hkv, Cn, cfg.d), dtype=Ks[0].dtype, pin_memory=True) for _ in probs]
    oVs = [torch.empty_like(t, pin_memory=True) for t in oKs]
    ois = [torch.empty((cfg.batch, cfg.Hkv, Cn), dtype=torch.int32, pin_memory=True) for _ in probs]
    seeds, layers = [11, 12, 13, 14, 15], [0, 3, 1, 7, 2]
    binding.nacl_evict_host_batch(Ks, Vs, Qs, Bp, Br, cfg.n_sink, cfg.n_recent, seeds, layers, oKs, oVs, ois)
    for i, (K, V, Q) in enumerate(probs):
        dK, dV, di = binding.nacl_evict(K.cuda(), V.cuda(), Q.cuda(), Bp, Br, cfg.n_sink, cfg.n_recent, seeds[i], layers[i])
        assert torch.equal(ois[i], di.cpu()) and torch.equal(oKs[i], dK.cpu()) and torch.equal(oVs[i], dV.cpu())


def test_batch_of_calls_matches_single_calls_eagerly_and_in_a_graph(binding):
    """nacl_evict_batch: independent calls of mixed shapes alternate between two internal streams that fork from and join
    into the caller's stream.  Same results as one nacl_evict_ex call each, also when the batch is captured into a CUDA
    graph (caller workspaces, neighbouring calls on different ones) and replayed."""
    shapes = [(1, 4100, 32, 8, 128, 64), (2, 9000, 16, 2, 128, 32), (4, 700, 8, 8, 128, 16), (1, 20000, 8, 2, 128, 16),
              (2, 3001, 4, 2, 64, 8), (1, 4100, 32, 8, 128, 64), (1, 129, 8, 8, 128, 16)]
    calls, want = [], []
    for i, (B, L, Hq, Hkv, d, P) in enumerate(shapes):
        K, V, Q = make_random_inputs(B, L, Hq, Hkv, d, P, dtype="f32" if d == 64 else "bf16", seed=300 + i)
        Kc, Vc, Qc = K.cuda(), V.cuda(), Q.cuda()
        Bp, Br = L // 5, L // 20
        want.append(binding.nacl_evict_ex(Kc, Vc, Qc, Bp, Br, 4, P, 17, i))
        calls.append(dict(K=Kc, V=Vc, Qproxy=Qc, budget_proxy=Bp, budget_random=Br, n_sink=4, n_recent=P, seed=17, layer=i))
    torch.cuda.synchronize()
    got = binding.nacl_evict_batch(calls)
    torch.cuda.synchronize()
    for i in range(len(shapes)):
        for k in ("out_idx", "out_K", "out_V"):
            assert torch.equal(got[i][k], want[i][k]), f"call {i}: {k} differs between the batch and the single call"
    # captured: caller workspaces, calls i and i+1 on different ones, outputs preallocated
    wsz = max(binding.nacl_workspace_bytes(c["K"].shape[0], c["K"].shape[2], c["Qproxy"].shape[1], c["K"].shape[1], c["K"].shape[3],
                                           c["Qproxy"].shape[2]) for c in calls)
    wss = [torch.empty(wsz, dtype=torch.uint8, device="cuda") for _ in range(2)]
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        for i, c in enumerate(calls):
            c.update(out_K=torch.zeros_like(want[i]["out_K"]), out_V=torch.zeros_like(want[i]["out_V"]),
                     out_idx=torch.zeros_like(want[i]["out_idx"]), workspace=wss[i & 1], stream=s)
        binding.nacl_evict_batch(calls)  # warm: the library's streams exist
        s.synchronize()
        for c in calls:
            c["out_idx"].zero_()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            binding.nacl_evict_batch(calls)
        g.replay()
        s.synchronize()
    for i, c in enumerate(calls):
        assert torch.equal(c["out_idx"], want[i]["out_idx"]) and torch.equal(c["out_K"], want[i]["out_K"]) and torch.equal(c["out_V"], want[i]["out_V"])


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
                                  (1, 1100, 8, 2, 128, 128, "bf16"), (1, 1000, 8, 2, 128, 100, "bf16")],
                         ids=["tc_GP256", "tc_GP32", "cuda_core_f32", "tc_GP512_row_blocks", "tc_GP400_partial_row_block"])
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
                                  (2, 333, 4, 2, 64, 5, "f32"), (1, 130, 6, 2, 32, 130, "bf16"), (1, 1300, 8, 2, 128, 128, "bf16"),
                                  (1, 1100, 8, 2, 128, 100, "bf16")],
                         ids=["tc_GP256_ragged", "tc_GP192", "tc_GP16", "cuda_core_f32", "all_rows_proxy", "tc_GP512_row_blocks",
                              "tc_GP400_partial_row_block"])
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


# ------------------------------------------------------------------ round 2: gaps named by the round-1 review
@pytest.mark.parametrize("L", [16, 64, 127, 128, 129])
@pytest.mark.parametrize("causal", [False, True])
def test_tensor_core_path_short_rows_and_all_rows_proxy(binding, L, causal):
    """The tcgen05 path (bf16, d = 128, G*P % 16 == 0) below / at / just above one key tile, with a single kv head (fewer
    tiles than CTAs, one tile per head) and with EVERY prompt row a proxy row (P = L where 16 | L, else P = 16)."""
    P = L if L % 16 == 0 else 16
    K, V, Q = make_random_inputs(1, L, 1, 1, 128, P, dtype="bf16", seed=100 + L)
    nr = min(P, L // 2)
    flags = binding.FLAG_CAUSAL if causal else 0
    full_parity(K, V, Q, nr + 2 + L // 8, L // 10, 2, nr, seed=3, layer=1, flags=flags)
    # edge budgets on the same path: no random part, keep everything, nothing but the protected set
    full_parity(K, V, Q, nr + 2 + L // 8, 0, 2, nr, seed=3, layer=1, flags=flags)
    r = full_parity(K, V, Q, L - 3, 3, 2, nr, seed=3, layer=1, flags=flags)
    np.testing.assert_array_equal(r["idx_gpu"][0, 0], np.arange(L))
    full_parity(K, V, Q, 2 + nr, 0, 2, nr, seed=3, layer=1, flags=flags)


@pytest.mark.parametrize("case", [(1, 4100, 32, 8, 128, 64, "bf16"), (2, 700, 4, 2, 64, 5, "f32"), (1, 384, 8, 2, 128, 128, "bf16")],
                         ids=["tc_GP256", "cuda_core_f32", "tc_GP512_row_blocks"])
def test_lse_in_with_causal_flag(binding, case):
    """Algorithm 2 proper: the row log-sum-exps come from a CAUSAL forward pass, i.e. row i's LSE covers
    the keys j <= L-P+i only, and the column sum is taken under the same mask.  lse_in under NACL_FLAG_CAUSAL is that causal
    LSE (include/nacl_evict.h); the oracle's causal importance and causal LSE are the referee."""
    from parity import check_scores, check_staged, check_structure

    B, L, Hq, Hkv, d, P, dt = case
    K, V, Q = make_random_inputs(B, L, Hq, Hkv, d, P, dtype=dt, seed=L + 7)
    imp_ref, lse_ref = oracle.importance(K, Q, flags=oracle.CAUSAL, return_lse=True)
    Bp, Br, ns, nr = L // 6 + P, L // 20, 4, P
    res = binding.nacl_evict_ex(K.cuda(), V.cuda(), Q.cuda(), Bp, Br, ns, nr, 5, 2, flags=binding.FLAG_CAUSAL,
                                want_importance=True, lse_in=torch.from_numpy(lse_ref.astype(np.float32)).cuda())
    torch.cuda.synchronize()
    imp = res["importance"].cpu().numpy()
    check_scores(imp, imp_ref, Hq // Hkv, P)
    check_structure(res["out_idx"].cpu().numpy(), L, Bp + Br, ns, nr)
    check_staged(res["out_idx"].cpu().numpy(), imp, Bp, Br, ns, nr, 5, 2)
    # the self-contained causal call agrees
    res2 = binding.nacl_evict_ex(K.cuda(), V.cuda(), Q.cuda(), Bp, Br, ns, nr, 5, 2, flags=binding.FLAG_CAUSAL, want_importance=True,
                                 want_lse=True)
    np.testing.assert_allclose(res2["importance"].cpu().numpy(), imp, rtol=2e-3, atol=1e-30)
    # ln Z carries the FMA-pipe exp2's relative error (<= 7.5e-5) as an ABSOLUTE error; short causal
    # rows sum too few terms for it to average out
    np.testing.assert_allclose(res2["lse"].cpu().numpy(), lse_ref, rtol=0, atol=1e-4)


@pytest.mark.parametrize("case", [(2, 3000, 16, 8, 128, 16, "bf16"), (2, 500, 4, 4, 64, 4, "f32"), (1, 70000, 8, 2, 128, 32, "bf16")],
                         ids=["tc", "cuda_core", "long_rows"])
def test_shards_draw_what_the_unsharded_call_draws(binding, case):
    """PAPER.md:37 / DESIGN.md R10: the random stream belongs to the (layer, batch element, kv head), not to the GPU that
    holds it.  Evicting a slice of the kv heads (tensor parallel) or of the batch (data parallel) on its own, with
    head_offset / batch_offset, gives bit-identical out_idx / out_K / out_V to the slice of the unsharded call."""
    B, L, Hq, Hkv, d, P, dt = case
    G = Hq // Hkv
    K, V, Q = make_random_inputs(B, L, Hq, Hkv, d, P, dtype=dt, seed=L + 11)
    Kd, Vd, Qd = K.cuda(), V.cuda(), Q.cuda()
    Bp, Br = L // 6, L // 12
    full = binding.nacl_evict_ex(Kd, Vd, Qd, Bp, Br, 4, P, 77, 3)
    h0 = Hkv // 2
    sh = binding.nacl_evict_ex(Kd[:, h0:].contiguous(), Vd[:, h0:].contiguous(), Qd[:, h0 * G:].contiguous(), Bp, Br, 4, P, 77, 3,
                               head_offset=h0)
    assert torch.equal(sh["out_idx"], full["out_idx"][:, h0:]) and torch.equal(sh["out_K"], full["out_K"][:, h0:])
    assert torch.equal(sh["out_V"], full["out_V"][:, h0:])
    wrong = binding.nacl_evict_ex(Kd[:, h0:].contiguous(), Vd[:, h0:].contiguous(), Qd[:, h0 * G:].contiguous(), Bp, Br, 4, P, 77, 3)
    assert not torch.equal(wrong["out_idx"], full["out_idx"][:, h0:])
    if B > 1:
        bs = binding.nacl_evict_ex(Kd[1:].contiguous(), Vd[1:].contiguous(), Qd[1:].contiguous(), Bp, Br, 4, P, 77, 3, batch_offset=1)
        assert torch.equal(bs["out_idx"], full["out_idx"][1:]) and torch.equal(bs["out_K"], full["out_K"][1:])
    # and the sharded call itself is the oracle's sharded call
    full_parity(K[:, h0:].contiguous(), V[:, h0:].contiguous(), Q[:, h0 * G:].contiguous(), Bp, Br, 4, P, 77, 3, head_offset=h0)


@pytest.mark.parametrize("case", [(1, 2100, 8, 2, 128, 16, "bf16"), (2, 400, 4, 2, 64, 4, "f32"), (1, 70000, 4, 1, 128, 16, "bf16")],
                         ids=["tc", "cuda_core", "long_rows"])
def test_explicit_protected_positions(binding, case):
    """Table "hyperp": an explicit list of protected positions (e.g. the proxy tokens when they are not
    the last P positions) is always retained and counts inside budget_proxy (R7)."""
    B, L, Hq, Hkv, d, P, dt = case
    K, V, Q = make_random_inputs(B, L, Hq, Hkv, d, P, dtype=dt, seed=L + 13)
    rng = np.random.default_rng(L)
    prot = np.sort(rng.choice(np.arange(4, L - P), size=min(40, L // 20), replace=False)).tolist()
    Bp, Br = 4 + P + len(prot) + L // 10, L // 20
    r = full_parity(K, V, Q, Bp, Br, 4, P, seed=21, layer=6, protect_idx=prot)
    for b in range(B):
        for h in range(Hkv):
            assert set(prot) <= set(r["idx_gpu"][b, h].tolist())
    full_parity(K, V, Q, 4 + P + len(prot), 0, 4, P, seed=21, layer=6, protect_idx=prot)  # nothing but protected positions
    with pytest.raises(binding.NaclError):
        binding.nacl_evict_ex(K.cuda(), V.cuda(), Q.cuda(), 4 + P + len(prot) - 1, 0, 4, P, 0, 0,
                              protect_idx=torch.tensor(prot, dtype=torch.int32, device="cuda"))


@pytest.mark.parametrize("case", [(2, 2500, 16, 4, 128, 16, "bf16"), (1, 600, 4, 4, 64, 4, "f32")], ids=["tc", "cuda_core"])
def test_shared_across_heads_selection(binding, case):
    """NACL_FLAG_SHARED_HEADS, the paper's "- Head-wise" ablation: one retained set per batch
    element, selected on the importance summed over the kv heads.  Staged check: the oracle's single-head selection on the
    GPU's own fp32 head sum (same summation order) reproduces out_idx exactly; end to end: the oracle's shared selection
    on its fp64 importance, up to the tolerance bands."""
    from parity import check_e2e_sets, check_gather, check_scores, check_structure

    B, L, Hq, Hkv, d, P, dt = case
    K, V, Q = make_random_inputs(B, L, Hq, Hkv, d, P, dtype=dt, seed=L + 17)
    Bp, Br = L // 5, L // 15
    res = binding.nacl_evict_ex(K.cuda(), V.cuda(), Q.cuda(), Bp, Br, 4, P, 31, 4, flags=binding.FLAG_SHARED_HEADS, want_importance=True,
                                head_offset=2)
    torch.cuda.synchronize()
    idx, imp = res["out_idx"].cpu().numpy(), res["importance"].cpu().numpy()
    imp_ref = oracle.importance(K, Q)
    check_scores(imp, imp_ref, Hq // Hkv, P)
    check_structure(idx, L, Bp + Br, 4, P)
    for h in range(1, Hkv):
        np.testing.assert_array_equal(idx[:, h], idx[:, 0])
    s32 = imp[:, 0].copy()
    for h in range(1, Hkv):
        s32 = (s32 + imp[:, h]).astype(np.float32)
    st_idx, st_part = oracle.select(s32[:, None, :], Bp, Br, 4, P, 31, 4, head_offset=2, return_parts=True)
    np.testing.assert_array_equal(idx[:, :1], st_idx)
    check_e2e_sets(idx[:, :1], st_part, imp_ref.sum(axis=1, keepdims=True), Bp, Br, 4, P, 31, 4, head_offset=2)
    ref = oracle.select(imp_ref, Bp, Br, 4, P, 31, 4, head_offset=2, shared_heads=True)
    assert (ref[:, 0] == ref[:, -1]).all()
    check_gather(K, V, res["out_K"].cpu(), res["out_V"].cpu(), idx)


def test_log_table_every_interval_at_both_edges_and_the_centre(binding):
    """The table-driven fp64 logarithm of the sampling keys (csrc/select.cu log_tab, table csrc/logtab.inc): importances
    whose mantissa sits at the lower edge, the centre and the upper edge of EACH of the 92 table intervals
    (c = k/128, k = 90..181), at several binary exponents, give the oracle's libm key bit for bit."""
    ms = []
    for k in range(90, 182):
        for off in (-0.5 + 1e-6, -0.25, 0.0, 0.25, 0.5 - 1e-6):
            ms.append((k + off) / 128.0)
    m = np.array(ms, dtype=np.float64)
    vals = np.concatenate([np.ldexp(m, e) for e in (-100, -20, -3, -1, 0, 1, 7)]).astype(np.float32)
    L = vals.size
    imp = np.stack([vals, vals[::-1].copy()])[None]  # [1, 2, L]
    seed, layer = 0xDEADBEEF12345, 9
    keys_gpu = binding.nacl_gumbel_keys(torch.from_numpy(imp).cuda(), seed, layer, 0).cpu().numpy()
    _, keys_ref = oracle.select(imp, 0, 1, 0, 0, seed, layer, 0, return_keys=True)
    a, b = keys_gpu.view(np.int32).astype(np.int64), keys_ref.view(np.int32).astype(np.int64)
    assert int((a != b).sum()) <= 1 and np.abs(a - b).max() <= 1, f"{int((a != b).sum())} of {a.size} keys differ"


# ------------------------------------------------------------------ layouts and generation phase (f3)
@pytest.mark.parametrize("case", [(2, 1500, 8, 2, 128, 16, "bf16"), (2, 333, 4, 2, 64, 5, "f32"), (1, 70000, 4, 2, 128, 16, "bf16")],
                         ids=["tc", "cuda_core", "long_rows"])
@pytest.mark.parametrize("layout", ["cache_with_capacity", "token_major"])
def test_strided_layouts_match_the_contiguous_call(binding, case, layout):
    """K/V as views of a cache [B,Hkv,cap,d] with spare capacity, or of a token-major [B,L,Hkv,d] tensor (the two KV layouts
    of FlashAttention-style kernels), and outputs written into a strided destination: bit-identical to the
    contiguous call (which the oracle checks)."""
    B, L, Hq, Hkv, d, P, dt = case
    K, V, Q = make_random_inputs(B, L, Hq, Hkv, d, P, dtype=dt, seed=L + 23)
    Kd, Vd, Qd = K.cuda(), V.cuda(), Q.cuda()
    Bp, Br = L // 6, L // 12
    C = Bp + Br
    want = binding.nacl_evict_ex(Kd, Vd, Qd, Bp, Br, 4, P, 5, 1, want_importance=True)
    if layout == "cache_with_capacity":
        cap = L + 37 * 8
        Kb, Vb = torch.zeros(B, Hkv, cap, d, dtype=Kd.dtype, device="cuda"), torch.zeros(B, Hkv, cap, d, dtype=Kd.dtype, device="cuda")
        Kb[:, :, :L], Vb[:, :, :L] = Kd, Vd
        Kv, Vv = Kb[:, :, :L], Vb[:, :, :L]
        oKb, oVb = torch.zeros(B, Hkv, C + 24, d, dtype=Kd.dtype, device="cuda"), torch.zeros(B, Hkv, C + 24, d, dtype=Kd.dtype, device="cuda")
        oK, oV = oKb[:, :, :C], oVb[:, :, :C]
    else:
        Kv, Vv = Kd.permute(0, 2, 1, 3).contiguous().permute(0, 2, 1, 3), Vd.permute(0, 2, 1, 3).contiguous().permute(0, 2, 1, 3)
        oKb, oVb = torch.zeros(B, C, Hkv, d, dtype=Kd.dtype, device="cuda"), torch.zeros(B, C, Hkv, d, dtype=Kd.dtype, device="cuda")
        oK, oV = oKb.permute(0, 2, 1, 3), oVb.permute(0, 2, 1, 3)
    assert not Kv.is_contiguous()
    got = binding.nacl_evict_ex(Kv, Vv, Qd, Bp, Br, 4, P, 5, 1, out_K=oK, out_V=oV, want_importance=True)
    torch.cuda.synchronize()
    assert torch.equal(got["importance"], want["importance"]) and torch.equal(got["out_idx"], want["out_idx"])
    assert torch.equal(oK, want["out_K"]) and torch.equal(oV, want["out_V"])
    if layout == "cache_with_capacity":
        assert oKb[:, :, C:].abs().sum() == 0  # nothing written past the C live rows


@pytest.mark.parametrize("case", [(2, 8, 2, 128, "bf16", 256, 4), (1, 4, 4, 64, "f32", 96, 3)], ids=["bf16_gqa", "f32_mha"])
def test_generation_phase_eviction(binding, case):
    """PAPER.md:66-70 and Algorithm 1, function Generation: every m steps the cache, grown to C + m
    entries, is evicted back to C on the attention row of the current token (one proxy row per query head, protected = the
    first slots and the newest slots).  Twelve decoding steps with appends; at every eviction the full parity protocol runs
    against the oracle ON THE SAME CACHE STATE (an eviction of the live rows with P = 1 and the step's seed), the caches
    ping-pong between two buffers with spare capacity, and the position map composes."""
    from parity import check_e2e_sets, check_scores, check_staged, check_structure

    B, Hq, Hkv, d, dt, C, m = case
    tdt = torch.bfloat16 if dt == "bf16" else torch.float32
    g = torch.Generator().manual_seed(C)
    cap = C + m + 8
    Bp, Br = (3 * C) // 4, C - (3 * C) // 4
    ns, nr = 2, 4
    bufs = [(torch.zeros(B, Hkv, cap, d, dtype=tdt, device="cuda"), torch.zeros(B, Hkv, cap, d, dtype=tdt, device="cuda"),
             torch.zeros(B, Hkv, cap, dtype=torch.int32, device="cuda")) for _ in range(2)]
    cur, length = 0, C
    bufs[0][0][:, :, :C] = torch.randn(B, Hkv, C, d, generator=g).to(tdt).cuda()
    bufs[0][1][:, :, :C] = torch.randn(B, Hkv, C, d, generator=g).to(tdt).cuda()
    bufs[0][2][:, :, :C] = torch.arange(C, dtype=torch.int32, device="cuda")
    n_evictions = 0
    for t in range(1, 13):
        Kc, Vc, pos = bufs[cur]
        Kc[:, :, length] = (1.5 * torch.randn(B, Hkv, d, generator=g)).to(tdt).cuda()  # K_t = [K_{t-1}, z_t W_K]
        Vc[:, :, length] = torch.randn(B, Hkv, d, generator=g).to(tdt).cuda()
        pos[:, :, length] = 1000 + t
        length += 1
        if t % m != 0:
            continue
        q = (2.0 * torch.randn(B, Hq, 1, d, generator=g)).to(tdt).cuda()
        Ko, Vo, po = bufs[1 - cur]
        Ko.zero_(); Vo.zero_(); po.zero_()
        res = binding.nacl_evict_generation(Kc, Vc, q, length, Bp, Br, ns, nr, 77, 5, t, Ko, Vo, pos_in=pos, pos_out=po,
                                            want_idx=True, want_importance=True, head_offset=1)
        torch.cuda.synchronize()
        idx, imp = res["out_idx"].cpu().numpy(), res["importance"].cpu().numpy()
        Kh, Vh, qh = Kc[:, :, :length].cpu().contiguous(), Vc[:, :, :length].cpu().contiguous(), q.cpu()
        seed_t = (77 + t * 0x9E3779B97F4A7C15) % (1 << 64)
        imp_ref = oracle.importance(Kh, qh)
        check_scores(imp, imp_ref, Hq // Hkv, 1)
        check_structure(idx, length, C, ns, nr)
        part = check_staged(idx, imp, Bp, Br, ns, nr, seed_t, 5, head_offset=1)
        check_e2e_sets(idx, part, imp_ref, Bp, Br, ns, nr, seed_t, 5, head_offset=1)
        ti = torch.from_numpy(idx.astype(np.int64)).cuda()
        assert torch.equal(Ko[:, :, :C], torch.gather(Kc, 2, ti[..., None].expand(-1, -1, -1, d)))
        assert torch.equal(Vo[:, :, :C], torch.gather(Vc, 2, ti[..., None].expand(-1, -1, -1, d)))
        assert torch.equal(po[:, :, :C].long(), torch.gather(pos.long(), 2, ti))
        assert Ko[:, :, C:].abs().sum() == 0
        # without out_idx the call keeps the slots in its workspace and gives the same cache
        Ko2, Vo2, po2 = torch.zeros_like(Ko), torch.zeros_like(Vo), torch.zeros_like(po)
        binding.nacl_evict_generation(Kc, Vc, q, length, Bp, Br, ns, nr, 77, 5, t, Ko2, Vo2, pos_in=pos, pos_out=po2, head_offset=1)
        assert torch.equal(Ko2, Ko) and torch.equal(po2, po)
        cur, length = 1 - cur, C
        n_evictions += 1
    assert n_evictions == 12 // m
    # the newest tokens (protected recent slots) survive every eviction
    assert (bufs[cur][2][:, :, C - 1] == 1000 + (12 // m) * m).all()


def test_generation_call_between_fused_calls_on_the_library_workspace(binding):
    """Calls of different head counts that share the library's own per-stream workspace: a 64-head call through the fused
    scoring launch (whose CTAs hand partials over through counters that must be zero at launch), then a generation-phase
    call with 8 heads and no out_idx (its softmax partials land on the bytes that held the 64-head call's counters), then
    the 64-head call again.  The library's record of how much of the counter area is still zero has to survive the call in
    the middle; the third call must give what the first gave and what the two-launch form (no counters) gives."""
    K, V, Q = make_random_inputs(2, 1024, 32, 32, 128, 16, dtype="bf16", seed=21, device="cuda")
    args = (K, V, Q, 150, 50, 4, 16, 4242, 7)
    first = binding.nacl_evict_ex(*args, want_importance=True)
    Kc, Vc, q = (t.contiguous() for t in make_random_inputs(1, 4100, 8, 8, 128, 1, dtype="bf16", seed=22, device="cuda"))
    C = 600
    Ko, Vo = torch.zeros(1, 8, C, 128, dtype=torch.bfloat16, device="cuda"), torch.zeros(1, 8, C, 128, dtype=torch.bfloat16, device="cuda")
    pos = torch.arange(4100, dtype=torch.int32, device="cuda").repeat(1, 8, 1).contiguous()
    po = torch.zeros(1, 8, C, dtype=torch.int32, device="cuda")
    binding.nacl_evict_generation(Kc, Vc, q, 4100, 450, 150, 2, 4, 77, 5, 3, Ko, Vo, pos_in=pos, pos_out=po)  # no out_idx, no workspace
    third = binding.nacl_evict_ex(*args, want_importance=True)
    ref = binding.nacl_evict_ex(*args, want_importance=True, flags=binding.FLAG_SCORE_TWO_LAUNCHES)
    gen_ref = binding.nacl_evict_generation(Kc, Vc, q, 4100, 450, 150, 2, 4, 77, 5, 3, torch.zeros_like(Ko), torch.zeros_like(Vo), want_idx=True)
    torch.cuda.synchronize()
    for k in ("out_idx", "out_K", "out_V"):
        assert torch.equal(third[k], first[k]) and torch.equal(third[k], ref[k]), k
    assert torch.equal(third["importance"], first["importance"])
    assert torch.equal(po, gen_ref["out_idx"])  # identity position map: pos_out names the kept slots
    assert torch.equal(Ko, torch.gather(Kc, 2, po.long()[..., None].expand(-1, -1, -1, 128)))


def test_library_workspaces_do_not_pile_up(binding):
    """The library's own workspaces (calls without a workspace argument) are keyed by stream.  Streams that come and go
    must not each leave a buffer behind for good, and a stream whose shapes keep growing must not keep every buffer it
    outgrew: old buffers are freed once the work that used them is done.  Read off the driver's free-memory
    figure, with every tensor of the test allocated before the first reading."""
    MiB = 1 << 20
    binding.nacl_release()
    torch.cuda.synchronize()
    B, Hq, Hkv, d, P = 1, 8, 8, 128, 16
    Ls = [8192 + 4096 * k for k in range(7)]  # 8k .. 32k keys: every step outgrows the 9/8 head-room of the buffer before it
    data = {L: make_random_inputs(B, L, Hq, Hkv, d, P, dtype="bf16", seed=L, device="cuda") for L in Ls}
    oK = torch.empty((B, Hkv, 800, d), dtype=torch.bfloat16, device="cuda")
    outs = dict(out_K=oK, out_V=torch.empty_like(oK), out_idx=torch.empty((B, Hkv, 800), dtype=torch.int32, device="cuda"))
    streams = [torch.cuda.Stream() for _ in range(40)]
    ws_big = binding.nacl_workspace_bytes(B, Ls[-1], Hq, Hkv, d, P)
    assert 3 * MiB < ws_big < 5 * MiB
    K, V, Q = data[Ls[-1]]
    binding.nacl_evict_ex(K, V, Q, 600, 200, 4, P, 1, 0, **outs)  # loads the kernels; creates the current stream's workspace
    want = {k: v.clone() for k, v in outs.items()}
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    # 40 streams, one call each at the largest shape: at most 16 keep a buffer
    for st in streams:
        st.wait_stream(torch.cuda.current_stream())
        binding.nacl_evict_ex(K, V, Q, 600, 200, 4, P, 1, 0, stream=st, **outs)
        st.synchronize()
        for k in outs:
            assert torch.equal(outs[k], want[k])
    free1, _ = torch.cuda.mem_get_info()
    used = free0 - free1
    assert 0 <= used <= 18 * 6 * MiB, f"{used / MiB:.0f} MiB held after 40 streams (40 buffers would be >= {40 * ws_big / MiB:.0f})"
    # one stream, seven growing shapes: the outgrown buffers go away
    binding.nacl_release()
    torch.cuda.synchronize()
    free2, _ = torch.cuda.mem_get_info()
    st = streams[0]
    total = 0
    for L in Ls:
        Kl, Vl, Ql = data[L]
        total += binding.nacl_workspace_bytes(B, L, Hq, Hkv, d, P)
        binding.nacl_evict_ex(Kl, Vl, Ql, 600, 200, 4, P, 1, 0, stream=st, **outs)
        st.synchronize()
    free3, _ = torch.cuda.mem_get_info()
    used = free2 - free3
    assert total > 4 * ws_big
    assert 0 <= used <= 10 * MiB, f"{used / MiB:.0f} MiB held after growing to {ws_big / MiB:.1f} MiB (never freeing would hold ~{total / MiB:.0f})"
    for k in outs:
        assert torch.equal(outs[k], want[k])


@pytest.mark.parametrize("cid", [3, 4, 5])
def test_timed_configuration_full_size(binding, cid):
    """The launch configuration bench.py times, at BASELINE.json's full sizes: FOUR distinct layers in ONE nacl_evict_batch
    call (the calls alternate between two internal streams; two plain scoring launches per call; the selection grid kept
    below ~45 % of the SMs; the stand-alone gather or the small-grid fused one), caller workspaces alternating as in
    bench.py, once eagerly and once replayed from a CUDA graph.  Every layer's outputs go through the whole protocol of
    tests/parity.py against the oracle; the graph replay must equal the eager call bit for bit, and a single nacl_evict_ex
    call per layer (the other launch configuration) must give the same bits too."""
    from parity import check_result, same_outputs

    cfg = CONFIGS[cid]
    Bp, Br = cfg.budgets()
    layers = (0, 10, 21, 31)
    host = [make_layer_inputs(cfg, layer=l) for l in layers]
    dev = torch.device("cuda:0")
    data = [(K.to(dev), V.to(dev), Q.to(dev)) for K, V, Q, _ in host]
    nws = binding.nacl_workspace_bytes(cfg.batch, cfg.L, cfg.Hq, cfg.Hkv, cfg.d, cfg.P)
    wss = [torch.full((nws,), 0x5A, dtype=torch.uint8, device=dev) for _ in range(2)]
    stream = torch.cuda.current_stream(dev)

    def calls(outs=None):
        cs = []
        for i, (l, (K, V, Q)) in enumerate(zip(layers, data)):
            c = dict(K=K, V=V, Qproxy=Q, budget_proxy=Bp, budget_random=Br, n_sink=cfg.n_sink, n_recent=cfg.n_recent,
                     seed=cfg.layer_seed(l), layer=l, workspace=wss[i & 1], want_importance=True)
            if outs is not None:  # the graph writes where the captured call wrote: hand the same tensors in again
                c.update(out_K=outs[i]["out_K"], out_V=outs[i]["out_V"], out_idx=outs[i]["out_idx"])
            cs.append(c)
        return cs

    eager = binding.nacl_evict_batch(calls())
    torch.cuda.synchronize()
    # this really is the timed configuration: the selection kernel's grid leaves more than half of the SMs to the other stream
    sel = binding.nacl_last_select_launch()
    assert 0 < sel["grid_ctas"] <= 0.45 * 148, sel
    assert sel["fused_gather"] == (cfg.G * cfg.P <= 128), sel
    single = [binding.nacl_evict_ex(K, V, Q, Bp, Br, cfg.n_sink, cfg.n_recent, cfg.layer_seed(l), l, want_importance=True)
              for l, (K, V, Q) in zip(layers, data)]
    torch.cuda.synchronize()
    single_grid = binding.nacl_last_select_launch()["grid_ctas"]
    assert single_grid >= sel["grid_ctas"]
    if cid in (3, 4):  # ... which the single call does not do with 32 heads (8 heads x 131072 keys: 64 CTAs either way)
        assert single_grid > 0.45 * 148
    for i, l in enumerate(layers):
        K, V, Q, planted = host[i]
        r = check_result(K, V, Q, eager[i], Bp, Br, cfg.n_sink, cfg.n_recent, cfg.layer_seed(l), l)
        for b in range(cfg.batch):
            for hk in range(cfg.Hkv):
                assert set(planted[b, hk].tolist()) <= set(r["idx_gpu"][b, hk].tolist())
        same_outputs(eager[i], single[i])
        print(f"cfg{cid} layer {l} (batch form): max rel err {r['max_rel_err']:.2e}, top-k swaps {r['topk_swaps']}, random diffs {r['random_diffs']}")
    # the same batch call replayed from a CUDA graph, into fresh (poisoned) outputs
    outs = [{k: torch.full_like(v, -1) if v.dtype == torch.int32 else torch.zeros_like(v) for k, v in e.items() if k != "importance"}
            for e in eager]
    cap = torch.cuda.Stream(dev)
    cap.wait_stream(stream)
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(cap):
        with torch.cuda.graph(graph, stream=cap):
            captured = binding.nacl_evict_batch([dict(c, stream=cap) for c in calls(outs)])
    stream.wait_stream(cap)
    torch.cuda.synchronize()
    for o in outs:
        o["out_idx"].fill_(-1); o["out_K"].zero_(); o["out_V"].zero_()
    for c in captured:
        c["importance"].zero_()
    for _ in range(2):
        graph.replay()
    torch.cuda.synchronize()
    for i in range(len(layers)):
        same_outputs(captured[i], eager[i])


@pytest.mark.parametrize("case", [(1, 4100, 32, 8, 128, 64, "bf16", 0), (2, 1000, 8, 2, 128, 16, "bf16", 0), (1, 1300, 8, 2, 128, 128, "bf16", 0),
                                  (1, 1200, 8, 2, 128, 100, "bf16", 0), (2, 333, 4, 2, 64, 5, "f32", 0), (1, 2049, 8, 2, 128, 32, "bf16", 1),
                                  (2, 515, 4, 2, 64, 7, "f32", 1)],
                         ids=["tc_GP256_ragged", "tc_GP64", "tc_GP512_row_blocks", "tc_GP400_partial_row_block", "cuda_core_f32",
                              "tc_causal", "cuda_core_causal"])
def test_proxy_lse_feeds_the_single_sweep_call(binding, case):
    """nacl_proxy_lse (step a2 alone): the row log-sum-exps equal the oracle's fp64 values, and an
    eviction that is handed them through lse_in passes the whole parity protocol with a single sweep over K."""
    B, L, Hq, Hkv, d, P, dt, causal = case
    K, V, Q = make_random_inputs(B, L, Hq, Hkv, d, P, dtype=dt, seed=L + 9)
    flags = binding.FLAG_CAUSAL if causal else 0
    _, lse_ref = oracle.importance(K, Q, flags=oracle.CAUSAL if causal else 0, return_lse=True)
    ws = torch.full((binding.nacl_workspace_bytes(B, L, Hq, Hkv, d, P),), 0xC3, dtype=torch.uint8, device="cuda")
    lse = binding.nacl_proxy_lse(K.cuda(), Q.cuda(), flags=flags, workspace=ws)
    lse2 = binding.nacl_proxy_lse(K.cuda(), Q.cuda(), flags=flags)  # the library's workspace; same bits
    torch.cuda.synchronize()
    assert torch.equal(lse, lse2)
    # an error delta of a row's lse scales that row's softmax by exp(delta): 5e-5 spends 2.5 % of the 2e-3 score tolerance
    # (fp32 sums of up to L exponentials, part of them from the FMA-pipe polynomial exp2; measured: up to 1.1e-5)
    np.testing.assert_allclose(lse.cpu().numpy(), lse_ref, rtol=0, atol=1e-4 if causal else 5e-5)
    # the two-sweep call reports the same statistics
    nr = min(P, L // 2)
    Bp, Br = max(L // 6, 4 + nr), L // 20
    two = binding.nacl_evict_ex(K.cuda(), V.cuda(), Q.cuda(), Bp, Br, 4, nr, 5, 1, flags=flags, want_lse=True)
    np.testing.assert_allclose(two["lse"].cpu().numpy(), lse.cpu().numpy(), rtol=1e-6, atol=1e-6)
    full_parity(K, V, Q, Bp, Br, 4, nr, seed=5, layer=1, flags=flags, lse_in=lse.cpu())
