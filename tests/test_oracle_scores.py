"""Pins for the oracle's steps 1-3 (logits, row softmax, column sum): PAPER.md:59, 124.

Each test checks oracle/ against something other than itself: printed worked examples
(tests/golden), closed forms, invariants, special cases that reduce to a torch library
routine (torch.softmax / torch.logsumexp in fp64 as referee).
"""
import math

import numpy as np
import pytest
import torch

import oracle
from conftest import read_golden
from paper_2408_03675_b200.inputs import make_random_inputs


def _parse_mat(s):
    return np.array([[float(x) for x in row.split(",")] for row in s.split(";")], dtype=np.float32)


def _imp_single(Q, K):
    """Q [P,d], K [L,d] -> imp [L] through the oracle (B=Hq=Hkv=1)."""
    return oracle.importance(K[None, None], Q[None, None])[0, 0]


def test_spec_micro_examples_importance():
    for line in read_golden("spec_micro_examples.txt"):
        kind, data, expected, _cite = [x.strip() for x in line.split("|")]
        if kind not in ("logit_diff", "importance"):
            continue
        fields = dict(kv.split("=") for kv in data.split())
        Q, K = _parse_mat(fields["Q"]), _parse_mat(fields["K"])
        imp = _imp_single(Q, K)
        if kind == "logit_diff":
            assert math.log(imp[0] / imp[1]) == pytest.approx(float(expected), abs=1e-12)
        else:
            np.testing.assert_allclose(imp, [float(x) for x in expected.split(",")], rtol=0, atol=1e-15)


def _torch_referee(K, Q, causal=False):
    """Library referee: softmax(QK^T/sqrt(d)) in fp64, summed over rows and the GQA group."""
    K, Q = K.double(), Q.double()
    B, Hkv, L, d = K.shape
    _, Hq, P, _ = Q.shape
    G = Hq // Hkv
    Kx = K.repeat_interleave(G, dim=1)  # query head hq reads kv head hq // G
    S = torch.einsum("bhpd,bhld->bhpl", Q, Kx) / math.sqrt(d)
    if causal:
        pos = torch.arange(L - P, L)[:, None]
        S = S.masked_fill(torch.arange(L)[None, :] > pos, float("-inf"))
    prob = torch.softmax(S, dim=-1)
    imp = prob.view(B, Hkv, G * P, L).sum(dim=2)
    return imp.numpy(), torch.logsumexp(S, dim=-1).numpy()


@pytest.mark.parametrize("shape", [
    # B, L, Hq, Hkv, d, P
    (1, 53, 1, 1, 8, 37),     # ragged 37x53
    (2, 130, 4, 2, 16, 5),    # GQA, G=2
    (1, 257, 8, 2, 64, 3),    # G=4
    (3, 64, 3, 3, 4, 64),     # P == L (all rows as proxies: one-shot H2O case)
])
@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_importance_matches_torch_softmax_referee(shape, dtype):
    B, L, Hq, Hkv, d, P = shape
    K, _V, Q = make_random_inputs(B, L, Hq, Hkv, d, P, dtype=dtype, seed=sum(shape), scale=1.5)
    imp, lse = oracle.importance(K, Q, return_lse=True)
    ref_imp, ref_lse = _torch_referee(K, Q)
    np.testing.assert_allclose(imp, ref_imp, rtol=1e-11, atol=1e-300)
    np.testing.assert_allclose(lse, ref_lse, rtol=1e-12, atol=1e-12)


def test_causal_flag_matches_masked_referee():
    K, _V, Q = make_random_inputs(2, 40, 4, 2, 8, 7, seed=3)
    imp = oracle.importance(K, Q, flags=oracle.CAUSAL)
    ref_imp, _ = _torch_referee(K, Q, causal=True)
    np.testing.assert_allclose(imp, ref_imp, rtol=1e-11, atol=1e-300)
    # the last key is visible to the last proxy row only
    assert np.all(imp[..., -1] <= 2.0 + 1e-12)  # G=2 groups, one row each


def test_mass_invariant():
    """Columns sum to P per query head, i.e. G*P per kv head (north star)."""
    for (B, L, Hq, Hkv, d, P) in [(1, 512, 4, 4, 64, 16), (2, 300, 8, 2, 32, 9)]:
        K, _V, Q = make_random_inputs(B, L, Hq, Hkv, d, P, seed=L)
        imp = oracle.importance(K, Q)
        G = Hq // Hkv
        np.testing.assert_allclose(imp.sum(-1), G * P, rtol=1e-12)


def test_identical_keys_give_uniform_importance():
    """All keys equal => every softmax row is uniform => imp_j = G*P/L exactly-ish."""
    B, L, Hq, Hkv, d, P = 1, 97, 4, 2, 16, 6
    _K, _V, Q = make_random_inputs(B, L, Hq, Hkv, d, P, seed=1)
    k = torch.randn(d)
    K = k.expand(B, Hkv, L, d).contiguous()
    imp = oracle.importance(K, Q)
    np.testing.assert_allclose(imp, (Hq // Hkv) * P / L, rtol=1e-13)


def test_adding_a_vector_to_every_key_leaves_importance_unchanged():
    """k_j -> k_j + v shifts each logit row by the constant q.v/sqrt(d): softmax invariant
    (SPEC.md:222).  Large |v| also exercises the max-subtraction."""
    B, L, Hq, Hkv, d, P = 1, 80, 2, 1, 8, 5
    K, _V, Q = make_random_inputs(B, L, Hq, Hkv, d, P, seed=5)
    K = torch.round(K * 1024) / 1024  # multiples of 2^-10, so that K + 64 is exact in fp32
    v = torch.full((d,), 64.0)
    imp0 = oracle.importance(K, Q)
    imp1 = oracle.importance((K + v).contiguous(), Q)
    np.testing.assert_allclose(imp1, imp0, rtol=1e-9)


def test_single_proxy_row_is_that_rows_softmax():
    """P = 1 (MSRNN case)."""
    K, _V, Q = make_random_inputs(1, 33, 1, 1, 16, 1, seed=9)
    imp = oracle.importance(K, Q)[0, 0]
    s = (K[0, 0].double() @ Q[0, 0, 0].double()) / math.sqrt(16)
    np.testing.assert_allclose(imp, torch.softmax(s, 0).numpy(), rtol=1e-12)


def test_dominant_key_takes_all_mass():
    B, L, Hq, Hkv, d, P = 1, 50, 2, 2, 4, 3
    Q = torch.ones(B, Hq, P, d)
    K = torch.zeros(B, Hkv, L, d)
    K[:, :, 17] = 100.0  # logit 200 above the rest
    imp = oracle.importance(K, Q)
    np.testing.assert_allclose(imp[..., 17], P, rtol=1e-12)
    assert np.all(np.delete(imp, 17, axis=-1) < 1e-80)


def test_bf16_inputs_are_widened_exactly():
    """bf16 bit patterns must be read as the upper half of an fp32."""
    K, _V, Q = make_random_inputs(1, 20, 2, 2, 8, 2, dtype="bf16", seed=2)
    imp_bf16 = oracle.importance(K, Q)
    imp_f32 = oracle.importance(K.float(), Q.float())
    np.testing.assert_array_equal(imp_bf16, imp_f32)


def test_paper_closed_forms():
    for line in read_golden("paper_closed_forms.txt"):
        kind, data, expected, _cite = [x.strip() for x in line.split("|")]
        if kind == "kv_bytes":
            f = {k: int(v) for k, v in (kv.split("=") for kv in data.split())}
            assert 2 * f["layers"] * f["heads"] * f["head_dim"] * f["batch"] * f["seq"] * f["bytes"] == int(expected)
            assert int(expected) == 64 * 2**30
        elif kind == "retention_per_layer":
            f = {k: float(v) for k, v in (kv.split("=") for kv in data.split())}
            assert round(1 - (1 - f["C"]) ** f["h"], 4) == float(expected)
        elif kind == "retention_all_layers_gt":
            f = {k: float(v) for k, v in (kv.split("=") for kv in data.split())}
            assert 1 - ((1 - f["C"]) ** f["h"]) ** f["l"] > float(expected)
        elif kind == "hyperp_row":
            total, a, b, c = [float(x) for x in data.split()]
            assert a + b + c == total


def test_argument_errors():
    K, _V, Q = make_random_inputs(1, 8, 3, 2, 4, 2)  # Hq % Hkv != 0
    with pytest.raises(oracle.OracleError):
        oracle.importance(K, Q)
    K, _V, Q = make_random_inputs(1, 4, 1, 1, 4, 5)  # P > L
    with pytest.raises(oracle.OracleError):
        oracle.importance(K, Q)
