"""Pins for the oracle's steps 4-8: protected set, top-k, Gumbel-top-k sampling, merge, gather
(PAPER.md:134-163, 179-183, 63).  Referees: brute force written independently here,
printed examples (tests/golden), the Random123 known-answer vectors, exact
Plackett-Luce probabilities by enumeration, chi-square on sampling frequencies.
"""
import itertools
import math

import numpy as np
import pytest
from hypothesis import given, settings, strategies as st
from scipy import stats

import oracle
from conftest import read_golden


# ------------------------------------------------------------------ Philox / uniforms
def test_philox_known_answer_vectors():
    rows = read_golden("philox4x32_10_kat.txt")
    assert len(rows) == 3
    for line in rows:
        w = [int(x, 16) for x in line.split()]
        out = oracle.philox4x32_10(w[0:4], w[4:6])
        assert [int(x) for x in out] == w[6:10]


def test_uniform_mapping_and_keying():
    seed, layer, b, hk, j = 0x1234567890ABCDEF, 3, 1, 5, 77
    x0 = int(oracle.philox4x32_10([j, hk, b, layer], [seed & 0xFFFFFFFF, seed >> 32])[0])
    u = oracle.uniform(seed, layer, b, hk, j)
    assert u == ((x0 >> 9) + 0.5) * 2.0**-23
    assert np.float32(u) == u  # exactly representable in fp32 (23 bits + centring)
    assert 2.0**-24 <= u <= 1 - 2.0**-24
    # every coordinate of (seed, layer, batch, head, position) changes the draw
    base = oracle.uniform(seed, layer, b, hk, j)
    assert oracle.uniform(seed ^ 1, layer, b, hk, j) != base
    assert oracle.uniform(seed ^ (1 << 40), layer, b, hk, j) != base
    assert oracle.uniform(seed, layer + 1, b, hk, j) != base
    assert oracle.uniform(seed, layer, b + 1, hk, j) != base
    assert oracle.uniform(seed, layer, b, hk + 1, j) != base
    assert oracle.uniform(seed, layer, b, hk, j + 1) != base
    assert oracle.uniform(seed, layer, b, hk, j) == base


def test_uniforms_are_uniform():
    u = np.array([oracle.uniform(7, 0, 0, 0, j) for j in range(20000)])
    assert stats.kstest(u, "uniform").pvalue > 1e-4


def test_gumbel_key_edge_values():
    assert oracle.gumbel_key(0.0, 0.5) == -math.inf  # R13: zero importance is taken last
    k = oracle.gumbel_key(0.3, 0.25)
    assert k == np.float32(math.log(0.3) - math.log(-math.log(0.25)))
    assert oracle.gumbel_key(0.3, 0.25, oracle.SAMPLE_UNIFORM) == np.float32(-math.log(-math.log(0.25)))
    assert oracle.gumbel_key(0.3, 0.25, oracle.SAMPLE_SOFTMAX_OF_SCORE) == np.float32(0.3 - math.log(-math.log(0.25)))


# ------------------------------------------------------------------ top-k
def _brute_topk(scores, k, lo, hi):
    """independent restatement: repeatedly take the largest remaining, lowest index on ties"""
    chosen, avail = [], list(range(lo, hi))
    for _ in range(k):
        best = avail[0]
        for j in avail[1:]:
            if scores[j] > scores[best]:
                best = j
        chosen.append(best)
        avail.remove(best)
    return set(chosen)


def test_spec_topk_examples():
    for line in read_golden("spec_micro_examples.txt"):
        kind, data, expected, _ = [x.strip() for x in line.split("|")]
        if kind != "topk":
            continue
        f = dict(kv.split("=") for kv in data.split())
        s = np.array([float(x) for x in f["scores"].split(",")])
        idx = oracle.select(s[None, None], int(f["k"]), 0, 0, 0, seed=0, layer=0)
        assert idx[0, 0].tolist() == [int(x) for x in expected.split(",")]


@settings(max_examples=200, deadline=None)
@given(st.data())
def test_topk_matches_brute_force(data):
    L = data.draw(st.integers(1, 40))
    n_sink = data.draw(st.integers(0, L))
    n_recent = data.draw(st.integers(0, L - n_sink))
    free = L - n_sink - n_recent
    k1 = data.draw(st.integers(0, free))
    # few distinct values => many ties
    vals = data.draw(st.lists(st.sampled_from([0.0, 0.125, 0.25, 0.5, 1.0, 3.0]), min_size=L, max_size=L))
    s = np.array(vals)
    idx, part = oracle.select(s[None, None], n_sink + n_recent + k1, 0, n_sink, n_recent, seed=1, layer=0,
                              return_parts=True)
    got = set(idx[0, 0][part[0, 0] == 1].tolist())
    assert got == _brute_topk(s, k1, n_sink, L - n_recent)
    prot = set(range(n_sink)) | set(range(L - n_recent, L))
    assert set(idx[0, 0][part[0, 0] == 0].tolist()) == prot
    assert idx[0, 0].tolist() == sorted(got | prot)


def test_budget_random_zero_is_pure_topk_and_full_budget_is_identity():
    rng = np.random.default_rng(0)
    s = rng.random((2, 3, 64))
    a = oracle.select(s, 20, 0, 2, 4, seed=5, layer=1)
    b = oracle.select(s, 20, 0, 2, 4, seed=99, layer=7)  # no randomness involved
    np.testing.assert_array_equal(a, b)
    for bb in range(2):
        for h in range(3):
            want = sorted(_brute_topk(s[bb, h], 14, 2, 60) | {0, 1, 60, 61, 62, 63})
            assert a[bb, h].tolist() == want
    full = oracle.select(s, 40, 24, 2, 4, seed=5, layer=1)  # C = L
    assert np.all(full == np.arange(64))


def test_budget_errors():
    s = np.ones((1, 1, 10))
    for args in [(3, 0, 2, 2), (8, 3, 1, 1), (5, 0, 6, 6), (-1, 0, 0, 0), (4, -1, 0, 0)]:
        with pytest.raises(oracle.OracleError) as e:
            oracle.select(s, *args, seed=0, layer=0)
        assert e.value.code == -2
    with pytest.raises(oracle.OracleError):  # negative / NaN importance is not a sum of probabilities
        oracle.select(np.array([[[0.1, -0.2, 0.3]]]), 1, 0, 0, 0, seed=0, layer=0)
    with pytest.raises(oracle.OracleError):
        oracle.select(np.array([[[0.1, np.nan, 0.3]]]), 1, 0, 0, 0, seed=0, layer=0)


# ------------------------------------------------------------------ structure (P8)
@settings(max_examples=150, deadline=None)
@given(st.data())
def test_structure_properties(data):
    B = data.draw(st.integers(1, 2))
    H = data.draw(st.integers(1, 3))
    L = data.draw(st.integers(1, 60))
    n_sink = data.draw(st.integers(0, L))
    n_recent = data.draw(st.integers(0, L - n_sink))
    n_prot = n_sink + n_recent
    Bp = data.draw(st.integers(n_prot, L))
    Br = data.draw(st.integers(0, L - Bp))
    seed = data.draw(st.integers(0, 2**64 - 1))
    layer = data.draw(st.integers(0, 100))
    rng = np.random.default_rng(data.draw(st.integers(0, 1000)))
    s = rng.random((B, H, L)) * (rng.random((B, H, L)) > 0.2)  # some exact zeros
    idx, part, keys = oracle.select(s, Bp, Br, n_sink, n_recent, seed, layer, return_parts=True, return_keys=True)
    assert idx.shape == (B, H, Bp + Br)
    for b in range(B):
        for h in range(H):
            row, prt = idx[b, h], part[b, h]
            assert np.all(np.diff(row) > 0)  # strictly ascending => unique
            assert (prt == 0).sum() == n_prot and (prt == 1).sum() == Bp - n_prot and (prt == 2).sum() == Br
            prot = set(range(n_sink)) | set(range(L - n_recent, L))
            assert prot <= set(row.tolist())
            assert set(row[prt == 0].tolist()) == prot
            # random part = the Br largest keys among candidates (key desc, index asc), independent re-sort
            cand = [j for j in range(n_sink, L - n_recent) if j not in set(row[prt == 1].tolist())]
            assert np.all(~np.isnan(keys[b, h][cand])) and np.isnan(keys[b, h]).sum() == L - len(cand)
            order = sorted(cand, key=lambda j: (-keys[b, h][j], j))
            assert set(row[prt == 2].tolist()) == set(order[:Br])
    again = oracle.select(s, Bp, Br, n_sink, n_recent, seed, layer)
    np.testing.assert_array_equal(idx, again)  # determinism


# ------------------------------------------------------------------ sampling law (P7)
def _draws(s, Bp, Br, n_sink, n_recent, seeds, layer=0):
    out = np.empty((len(seeds), Br), dtype=np.int64)
    for n, seed in enumerate(seeds):
        idx, part = oracle.select(s[None, None], Bp, Br, n_sink, n_recent, int(seed), layer, return_parts=True)
        out[n] = idx[0, 0][part[0, 0] == 2]
    return out


def test_single_draw_frequencies_chi_square():
    """Br = 1: P(draw j) = imp_j / sum over candidates (north star: 'probability proportional
    to importance'); chi-square over 20000 seeds, df = 9."""
    rng = np.random.default_rng(42)
    L = 12
    s = rng.random(L) + 0.05
    Bp = 2  # no protection: the two largest go to top-k, 10 candidates remain
    top2 = set(np.argsort(-s)[:2].tolist())
    cand = [j for j in range(L) if j not in top2]
    draws = _draws(s, Bp, 1, 0, 0, np.arange(20000))[:, 0]
    assert set(draws.tolist()) <= set(cand)
    obs = np.array([(draws == j).sum() for j in cand])
    exp = s[cand] / s[cand].sum() * len(draws)
    assert stats.chisquare(obs, exp).pvalue > 1e-4


def test_spec_sampling_examples():
    for line in read_golden("spec_micro_examples.txt"):
        kind, data, expected, _ = [x.strip() for x in line.split("|")]
        f = dict(kv.split("=") for kv in data.split())
        if kind == "sample_all":
            s = np.array([float(x) for x in f["scores"].split(",")])
            idx = oracle.select(s[None, None], 0, int(f["k"]), 0, 0, seed=3, layer=0)
            assert idx[0, 0].tolist() == [int(x) for x in expected.split(",")]
        elif kind == "sample_freq":
            w = np.array([float(x) for x in f["weights"].split(",")])
            p, tol = [float(x) for x in expected.split()]
            draws = _draws(w, 0, 1, 0, 0, np.arange(10000))[:, 0]
            assert abs((draws == int(f["index"])).mean() - p) < tol


def _plackett_luce_set_probs(w, k):
    """exact probabilities of each unordered k-set under successive draws without replacement,
    renormalising after each draw -- by enumerating ordered draws."""
    n = len(w)
    probs = {}
    for perm in itertools.permutations(range(n), k):
        p, rest = 1.0, w.sum()
        for j in perm:
            p *= w[j] / rest
            rest -= w[j]
        key = tuple(sorted(perm))
        probs[key] = probs.get(key, 0.0) + p
    return probs


@pytest.mark.parametrize("k", [2, 3])
def test_without_replacement_law_matches_enumeration(k):
    """Gumbel-top-k == successive sampling without replacement (R5): total-variation
    distance of the empirical k-set distribution from the enumerated one < 0.02."""
    w = np.array([0.05, 0.4, 0.1, 0.25, 0.8, 0.15, 0.3])
    n = 30000
    draws = _draws(w, 0, k, 0, 0, np.arange(1000, 1000 + n), layer=2)
    exact = _plackett_luce_set_probs(w, k)
    counts = {}
    for row in draws:
        key = tuple(sorted(row.tolist()))
        counts[key] = counts.get(key, 0) + 1
    tv = 0.5 * sum(abs(counts.get(key, 0) / n - p) for key, p in exact.items())
    assert set(counts) <= set(exact)
    assert tv < 0.02
    # per-index inclusion probabilities too
    incl = np.zeros(len(w))
    for key, p in exact.items():
        for j in key:
            incl[j] += p
    emp = np.array([(draws == j).any(axis=1).mean() for j in range(len(w))])
    assert np.abs(emp - incl).max() < 0.015


def test_uniform_flag_draws_uniformly_and_zero_importance_goes_last():
    w = np.array([0.9, 0.05, 0.0, 0.05, 0.0, 0.3])
    draws = _draws(w, 0, 1, 0, 0, np.arange(6000))[:, 0]
    assert not np.isin(draws, [2, 4]).any()  # weight 0 is never drawn while others remain
    # all six must be returned when Br = 6, zeros included (taken last)
    assert oracle.select(w[None, None], 0, 6, 0, 0, seed=1, layer=0)[0, 0].tolist() == [0, 1, 2, 3, 4, 5]
    # five requested: exactly one of the zero-weight tokens is left out, the higher index (tie -> lower index wins)
    assert oracle.select(w[None, None], 0, 5, 0, 0, seed=1, layer=0)[0, 0].tolist() == [0, 1, 2, 3, 5]
    un = np.empty(12000, dtype=np.int64)
    for n in range(len(un)):
        idx = oracle.select(w[None, None], 0, 1, 0, 0, seed=n, layer=0, flags=oracle.SAMPLE_UNIFORM)
        un[n] = idx[0, 0, 0]
    obs = np.bincount(un, minlength=6)
    assert stats.chisquare(obs).pvalue > 1e-4


def test_head_layer_independence_and_paper_retention_formula():
    """P9: identical importance everywhere and Bp = n_prot => each head keeps a uniform random
    c-fraction, independently per head.  The fraction of tokens kept by >= 1 of h heads must
    follow the paper's 1-(1-C)^h (99.92% at C=20%, h=32)."""
    L, c = 4000, 0.2
    s = np.full((1, 32, L), 1.0 / L)
    idx = oracle.select(s, 0, int(c * L), 0, 0, seed=11, layer=0)
    kept = np.zeros((32, L), dtype=bool)
    for h in range(32):
        kept[h, idx[0, h]] = True
    assert not np.array_equal(idx[0, 0], idx[0, 1])
    for h in (1, 2, 4, 8):
        frac = kept[:h].any(axis=0).mean()
        want = 1 - (1 - c) ** h
        sigma = math.sqrt(want * (1 - want) / L)
        assert abs(frac - want) < 4 * sigma + 1e-3
    missing = L - kept.any(axis=0).sum()  # expectation L*(0.8^32) = 3.2
    assert missing <= 15
    # a different layer or batch element or seed redraws
    idx_l = oracle.select(s, 0, int(c * L), 0, 0, seed=11, layer=1)
    idx_s = oracle.select(s, 0, int(c * L), 0, 0, seed=12, layer=0)
    assert not np.array_equal(idx, idx_l) and not np.array_equal(idx, idx_s)
    s2 = np.full((2, 1, L), 1.0 / L)
    idx_b = oracle.select(s2, 0, int(c * L), 0, 0, seed=11, layer=0)
    assert not np.array_equal(idx_b[0], idx_b[1])
    np.testing.assert_array_equal(idx_b[0, 0], idx[0, 0])  # (b=0, hk=0) is the same stream


# ------------------------------------------------------------------ gather (P10)
def test_gather_is_a_bytewise_row_copy():
    rng = np.random.default_rng(3)
    for dt in (np.float32, np.uint16):
        K = rng.integers(0, 2**16, size=(2, 3, 17, 8)).astype(dt)
        V = rng.integers(0, 2**16, size=(2, 3, 17, 8)).astype(dt)
        idx = np.sort(rng.permuted(np.tile(np.arange(17), (2, 3, 1)), axis=-1)[..., :5], axis=-1).astype(np.int32)
        oK, oV = oracle.gather(K, V, idx)
        for b in range(2):
            for h in range(3):
                np.testing.assert_array_equal(oK[b, h], K[b, h, idx[b, h]])
                np.testing.assert_array_equal(oV[b, h], V[b, h, idx[b, h]])
    with pytest.raises(oracle.OracleError):
        oracle.gather(K, V, np.full((2, 3, 1), 17, dtype=np.int32))


# ------------------------------------------------------------------ options of nacl_oracle_select_ex
def test_offsets_make_a_shard_draw_what_the_unsharded_call_draws():
    """PAPER.md:37 ties the random stream to the head and the layer (R10: counter = (position, kv head, batch, layer)):
    a slice of the heads or of the batch, told where it starts, reproduces the slice of the unsharded result; without
    the offsets it does not (the draws differ)."""
    rng = np.random.default_rng(3)
    imp = rng.random((3, 4, 200))
    full, parts = oracle.select(imp, 30, 25, 2, 5, seed=11, layer=2, return_parts=True)
    for h0, h1 in [(0, 2), (2, 4), (1, 4)]:
        np.testing.assert_array_equal(oracle.select(imp[:, h0:h1], 30, 25, 2, 5, 11, 2, head_offset=h0), full[:, h0:h1])
    for b0 in (1, 2):
        np.testing.assert_array_equal(oracle.select(imp[b0:], 30, 25, 2, 5, 11, 2, batch_offset=b0), full[b0:])
    assert not np.array_equal(oracle.select(imp[:, 2:4], 30, 25, 2, 5, 11, 2), full[:, 2:4])
    # the top-k part never depends on the offsets
    sl, sp = oracle.select(imp[:, 2:4], 30, 25, 2, 5, 11, 2, return_parts=True)
    for b in range(3):
        for h in range(2):
            assert set(sl[b, h][sp[b, h] == 1]) == set(full[b, 2 + h][parts[b, 2 + h] == 1])


def test_explicit_protected_positions_reduce_to_infinite_importance():
    """Table "hyperp": protected proxy tokens are kept by default and count inside the proxy budget
    (R7).  Protecting a position is the same as giving it an importance above every other one and taking the same
    top-Bp: the base routine on the modified scores is the referee."""
    rng = np.random.default_rng(5)
    for _ in range(20):
        L = int(rng.integers(30, 120))
        imp = rng.random((2, 2, L))
        ns, nr = int(rng.integers(0, 4)), int(rng.integers(0, 6))
        free = np.arange(ns, L - nr)
        prot = np.sort(rng.choice(free, size=int(rng.integers(1, 6)), replace=False))
        Bp = ns + nr + len(prot) + int(rng.integers(0, 8))
        Br = int(rng.integers(0, min(10, L - Bp) + 1))
        idx, part = oracle.select(imp, Bp, Br, ns, nr, 4, 1, protect_idx=prot, return_parts=True)
        big = imp.copy()
        big[..., prot] = 1e30
        ref = oracle.select(big, Bp, Br, ns, nr, 4, 1)
        np.testing.assert_array_equal(idx, ref)
        for b in range(2):
            for h in range(2):
                assert set(prot.tolist()) <= set(idx[b, h][part[b, h] == 0].tolist())
    with pytest.raises(oracle.OracleError):
        oracle.select(imp, ns + nr + 1, 0, ns, nr, 0, 0, protect_idx=prot[:3] if len(prot) >= 3 else np.array([ns, ns + 1, ns + 2]))
    with pytest.raises(oracle.OracleError):
        oracle.select(imp, Bp + 3, 0, ns, nr, 0, 0, protect_idx=[free[1], free[0]])  # not ascending


def test_shared_heads_is_one_selection_on_the_head_summed_importance():
    """The "- Head-wise" ablation: every head of a batch element keeps the same positions,
    those a single-head call selects on the sum of the heads' importances."""
    rng = np.random.default_rng(8)
    imp = rng.random((2, 4, 150))
    idx = oracle.select(imp, 20, 15, 2, 4, 9, 3, shared_heads=True, head_offset=4)
    summed = imp[:, 0] + imp[:, 1] + imp[:, 2] + imp[:, 3]
    ref = oracle.select(summed[:, None, :], 20, 15, 2, 4, 9, 3, head_offset=4)
    for h in range(4):
        np.testing.assert_array_equal(idx[:, h], ref[:, 0])
