"""Pins for the float64 oracle (oracle/): each test checks it against something OTHER than itself --
a hand-derived example, closed forms, library routines, finite differences, brute-force loops,
invariants -- chosen so that a dropped term, wrong sign/index or transposed operand fails one of them.
CPU only (`-m "not gpu"`).
"""
import math
import os

import numpy as np
import pytest

from oracle import streamkl_algorithms as alg
from oracle import streamkl_oracle as orc

GOLD = os.path.join(os.path.dirname(__file__), "golden")
rng0 = np.random.default_rng(1234)


def _rand(NQ, NK, d1, d2, seed=0, scale=1.0):
    r = np.random.default_rng(seed)
    return (scale * r.standard_normal((NQ, d1)), r.standard_normal((NK, d1)),
            r.standard_normal((NQ, d2)), r.standard_normal((NK, d2)), 0.5 + r.random(NQ))


# ------------------------------------------------------------------ worked example (golden file)
def test_worked_example_golden():
    gold = {}
    for line in open(os.path.join(GOLD, "worked_example.txt")):
        if line.strip() and not line.startswith("#"):
            k, v = line.split()
            gold[k] = float(v)
    Q1 = np.array([[1.0]]); Q2 = np.array([[1.0]])
    K1 = np.array([[math.log(3.0)], [0.0]]); K2 = np.zeros((2, 1))
    o = orc.attention_kl_head(Q1, K1, Q2, K2, 1.0, 1.0, False, g=np.ones(1))
    assert o["lse1"][0] == pytest.approx(gold["lse1"], abs=1e-14)
    assert o["lse2"][0] == pytest.approx(gold["lse2"], abs=1e-14)
    assert o["kl"][0] == pytest.approx(gold["kl"], abs=1e-14)
    assert o["dQ1"][0, 0] == pytest.approx(gold["dQ1"], abs=1e-14)
    assert o["dQ2"][0, 0] == pytest.approx(gold["dQ2"], abs=1e-14)
    np.testing.assert_allclose(o["dK1"][:, 0], [gold["dK1_0"], gold["dK1_1"]], atol=1e-14)
    np.testing.assert_allclose(o["dK2"][:, 0], [gold["dK2_0"], gold["dK2_1"]], atol=1e-14)


# ------------------------------------------------------------------ closed forms
@pytest.mark.parametrize("causal", [False, True])
def test_identical_logits_give_zero(causal):
    # same logits through different factorisations: Q2 = 2*Q1, K2 = K1, c2 = c1/2 ; and zero-padded d2 > d1
    Q1, K1, _, _, g = _rand(9, 13, 4, 4, seed=1)
    o = orc.attention_kl_head(Q1, K1, 2 * Q1, K1, 0.7, 0.35, causal, g=g)
    assert np.abs(o["kl"]).max() < 1e-14
    np.testing.assert_allclose(o["lse1"], o["lse2"], atol=1e-13)
    for k in ("dQ1", "dK1", "dQ2", "dK2"):
        assert np.abs(o[k]).max() < 1e-13, k
    Q2 = np.concatenate([Q1, np.zeros((9, 3))], axis=1); K2 = np.concatenate([K1, rng0.standard_normal((13, 3))], axis=1)
    o = orc.attention_kl_head(Q1, K1, Q2, K2, 0.7, 0.7, causal, g=g)
    assert np.abs(o["kl"]).max() < 1e-14


@pytest.mark.parametrize("causal", [False, True])
def test_p2_uniform_and_p1_uniform(causal):
    # DESIGN.md R18.  nV = visible keys of the row.
    NQ, NK = 7, 11
    Q1, K1, Q2, K2, _ = _rand(NQ, NK, 5, 3, seed=2)
    nV = np.array([NK if not causal else i + (NK - NQ) + 1 for i in range(NQ)], dtype=float)
    # P2 uniform (Q2 = 0): KL = log nV - H(P1), lse2 = log nV
    o = orc.attention_kl_head(Q1, K1, 0 * Q2, K2, 0.4, 0.9, causal)
    H1 = np.empty(NQ)
    for i in range(NQ):
        n = int(nV[i]); s = 0.4 * (K1[:n] @ Q1[i]); p = np.exp(s - s.max()); p /= p.sum()
        H1[i] = -(p * np.log(p)).sum()
    np.testing.assert_allclose(o["kl"], np.log(nV) - H1, atol=1e-13)
    np.testing.assert_allclose(o["lse2"], np.log(nV), atol=1e-13)
    # P1 uniform (Q1 = 0): KL = lse2 - mean_V(s2) - log nV, lse1 = log nV
    o = orc.attention_kl_head(0 * Q1, K1, Q2, K2, 0.4, 0.9, causal)
    mean_s2 = np.array([(0.9 * (K2[: int(nV[i])] @ Q2[i])).mean() for i in range(NQ)])
    np.testing.assert_allclose(o["kl"], o["lse2"] - mean_s2 - np.log(nV), atol=1e-13)
    np.testing.assert_allclose(o["lse1"], np.log(nV), atol=1e-13)


def test_single_key_and_causal_row0():
    Q1, K1, Q2, K2, g = _rand(4, 1, 3, 2, seed=3)
    o = orc.attention_kl_head(Q1, K1, Q2, K2, 0.5, 0.8, False, g=g)
    assert np.abs(o["kl"]).max() == 0.0
    np.testing.assert_allclose(o["lse1"], 0.5 * (Q1 @ K1.T)[:, 0], atol=1e-15)
    np.testing.assert_allclose(o["lse2"], 0.8 * (Q2 @ K2.T)[:, 0], atol=1e-15)
    for k in ("dQ1", "dK1", "dQ2", "dK2"):
        assert np.abs(o[k]).max() < 1e-15
    Q1, K1, Q2, K2, g = _rand(6, 6, 3, 2, seed=4)
    o = orc.attention_kl_head(Q1, K1, Q2, K2, 0.5, 0.8, True, g=g)
    assert o["kl"][0] == 0.0 and o["lse1"][0] == pytest.approx(0.5 * Q1[0] @ K1[0], abs=1e-15)


def test_two_keys_bernoulli():
    Q1, K1, Q2, K2, _ = _rand(5, 2, 3, 3, seed=5)
    o = orc.attention_kl_head(Q1, K1, Q2, K2, 0.6, 1.1, False)
    s1 = 0.6 * Q1 @ K1.T; s2 = 1.1 * Q2 @ K2.T
    p = 1 / (1 + np.exp(-(s1[:, 0] - s1[:, 1]))); q = 1 / (1 + np.exp(-(s2[:, 0] - s2[:, 1])))
    kl = p * np.log(p / q) + (1 - p) * np.log((1 - p) / (1 - q))
    np.testing.assert_allclose(o["kl"], kl, atol=1e-14)


def test_causal_alignment_bottom_right():
    # R5: NQ < NK causal == non-causal run of each row on its own prefix of i + (NK-NQ) + 1 keys
    Q1, K1, Q2, K2, _ = _rand(4, 9, 3, 2, seed=6)
    o = orc.attention_kl_head(Q1, K1, Q2, K2, 0.5, 0.5, True)
    for i in range(4):
        n = i + 5 + 1
        oi = orc.attention_kl_head(Q1[i:i + 1], K1[:n], Q2[i:i + 1], K2[:n], 0.5, 0.5, False)
        assert o["kl"][i] == pytest.approx(oi["kl"][0], abs=1e-14)
        assert o["lse1"][i] == pytest.approx(oi["lse1"][0], abs=1e-14)
    with pytest.raises(ValueError):
        orc.attention_kl_head(K1, Q1, K2, Q2, 0.5, 0.5, True)  # NQ > NK causal rejected


# ------------------------------------------------------------------ library routines
@pytest.mark.parametrize("causal", [False, True])
def test_against_scipy(causal):
    from scipy.special import logsumexp, rel_entr, softmax
    NQ, NK = 6, 10
    Q1, K1, Q2, K2, _ = _rand(NQ, NK, 4, 7, seed=7)
    o = orc.attention_kl_head(Q1, K1, Q2, K2, 0.5, 0.3, causal)
    for i in range(NQ):
        n = NK if not causal else i + (NK - NQ) + 1
        s1 = 0.5 * K1[:n] @ Q1[i]; s2 = 0.3 * K2[:n] @ Q2[i]
        assert o["lse1"][i] == pytest.approx(logsumexp(s1), abs=1e-13)
        assert o["lse2"][i] == pytest.approx(logsumexp(s2), abs=1e-13)
        assert o["kl"][i] == pytest.approx(rel_entr(softmax(s1), softmax(s2)).sum(), abs=1e-13)


@pytest.mark.parametrize("causal", [False, True])
@pytest.mark.parametrize("shape", [(5, 7, 4, 3), (8, 8, 2, 6), (3, 40, 16, 8)])
def test_gradients_against_torch_autograd(causal, shape):
    import torch
    NQ, NK, d1, d2 = shape
    Q1, K1, Q2, K2, g = _rand(NQ, NK, d1, d2, seed=8)
    g = g * np.where(np.arange(NQ) % 2 == 0, 1.0, -1.3)  # mixed-sign upstream gradient
    c1, c2 = 0.45, 0.8
    t = [torch.tensor(a, dtype=torch.float64, requires_grad=True) for a in (Q1, K1, Q2, K2)]
    s1 = c1 * t[0] @ t[1].T; s2 = c2 * t[2] @ t[3].T
    if causal:
        mask = torch.arange(NK)[None, :] > torch.arange(NQ)[:, None] + (NK - NQ)
        s1 = s1.masked_fill(mask, float("-inf")); s2 = s2.masked_fill(mask, float("-inf"))
    lp1 = torch.log_softmax(s1, dim=-1); lp2 = torch.log_softmax(s2, dim=-1)
    if causal:  # -inf log-probs at masked entries would make 0*(-inf - -inf) = nan in kl_div
        lp1 = lp1.masked_fill(mask, -1e3); lp2 = lp2.masked_fill(mask, -1e3)  # exp(-1e3) == 0 exactly in float64
    kl = torch.nn.functional.kl_div(lp2, lp1, reduction="none", log_target=True).sum(-1)
    (kl * torch.tensor(g)).sum().backward()
    o = orc.attention_kl_head(Q1, K1, Q2, K2, c1, c2, causal, g=g)
    np.testing.assert_allclose(o["kl"], kl.detach().numpy(), atol=1e-13)
    for name, tt in zip(("dQ1", "dK1", "dQ2", "dK2"), t):
        np.testing.assert_allclose(o[name], tt.grad.numpy(), atol=1e-12, err_msg=name)


# ------------------------------------------------------------------ finite differences
@pytest.mark.parametrize("causal", [False, True])
def test_gradients_against_finite_differences(causal):
    NQ, NK, d1, d2 = 5, 7, 4, 3
    Q1, K1, Q2, K2, g = _rand(NQ, NK, d1, d2, seed=9)
    c1, c2 = 0.5, 0.7
    base = [Q1, K1, Q2, K2]

    def loss(args):
        return float((g * orc.attention_kl_head(*args, c1, c2, causal)["kl"]).sum())

    o = orc.attention_kl_head(Q1, K1, Q2, K2, c1, c2, causal, g=g)
    h = 1e-6
    for idx, name in enumerate(("dQ1", "dK1", "dQ2", "dK2")):
        num = np.zeros_like(base[idx])
        for e in np.ndindex(base[idx].shape):
            ap = [a.copy() for a in base]; am = [a.copy() for a in base]
            ap[idx][e] += h; am[idx][e] -= h
            num[e] = (loss(ap) - loss(am)) / (2 * h)
        np.testing.assert_allclose(o[name], num, atol=2e-8, err_msg=name)


# ------------------------------------------------------------------ brute force, scalar loops
def _brute(Q1, K1, Q2, K2, c1, c2, causal, g):
    NQ, NK = len(Q1), len(K1)
    kl = [0.0] * NQ; l1s = [0.0] * NQ; l2s = [0.0] * NQ
    dQ1 = np.zeros_like(Q1); dK1 = np.zeros_like(K1); dQ2 = np.zeros_like(Q2); dK2 = np.zeros_like(K2)
    for i in range(NQ):
        vis = [j for j in range(NK) if (not causal) or j <= i + NK - NQ]
        s1 = {j: c1 * sum(Q1[i][k] * K1[j][k] for k in range(Q1.shape[1])) for j in vis}
        s2 = {j: c2 * sum(Q2[i][k] * K2[j][k] for k in range(Q2.shape[1])) for j in vis}
        z1 = sum(math.exp(v) for v in s1.values()); z2 = sum(math.exp(v) for v in s2.values())
        p1 = {j: math.exp(s1[j]) / z1 for j in vis}; p2 = {j: math.exp(s2[j]) / z2 for j in vis}
        kl[i] = sum(p1[j] * math.log(p1[j] / p2[j]) for j in vis)
        l1s[i] = math.log(z1); l2s[i] = math.log(z2)
        for j in vis:
            ds2 = g[i] * (p2[j] - p1[j])
            ds1 = g[i] * p1[j] * (math.log(p1[j] / p2[j]) - kl[i])
            for k in range(Q2.shape[1]):
                dQ2[i][k] += c2 * ds2 * K2[j][k]; dK2[j][k] += c2 * ds2 * Q2[i][k]
            for k in range(Q1.shape[1]):
                dQ1[i][k] += c1 * ds1 * K1[j][k]; dK1[j][k] += c1 * ds1 * Q1[i][k]
    return np.array(kl), np.array(l1s), np.array(l2s), dQ1, dK1, dQ2, dK2


@pytest.mark.parametrize("causal", [False, True])
@pytest.mark.parametrize("shape", [(1, 1, 1, 1), (3, 5, 2, 3), (8, 8, 3, 2), (2, 7, 1, 4)])
def test_against_scalar_brute_force(causal, shape):
    NQ, NK, d1, d2 = shape
    Q1, K1, Q2, K2, g = _rand(NQ, NK, d1, d2, seed=10)
    o = orc.attention_kl_head(Q1, K1, Q2, K2, 0.9, 0.6, causal, g=g)
    kl, l1, l2, dQ1, dK1, dQ2, dK2 = _brute(Q1, K1, Q2, K2, 0.9, 0.6, causal, g)
    for a, b, n in ((o["kl"], kl, "kl"), (o["lse1"], l1, "lse1"), (o["lse2"], l2, "lse2"), (o["dQ1"], dQ1, "dQ1"),
                    (o["dK1"], dK1, "dK1"), (o["dQ2"], dQ2, "dQ2"), (o["dK2"], dK2, "dK2")):
        np.testing.assert_allclose(a, b, atol=1e-13, err_msg=n)


# ------------------------------------------------------------------ invariants
@pytest.mark.parametrize("causal", [False, True])
def test_invariants(causal):
    NQ, NK, d1, d2 = 12, 17, 6, 5
    Q1, K1, Q2, K2, g = _rand(NQ, NK, d1, d2, seed=11, scale=2.0)
    c1, c2 = 0.4, 0.45
    o = orc.attention_kl_head(Q1, K1, Q2, K2, c1, c2, causal, g=g)
    assert (o["kl"] >= -1e-15).all()                        # Gibbs
    # sum_j dS_t[i,j] = 0 per row  =>  dQ_t unchanged when a constant vector is added to every key
    v1 = rng0.standard_normal(d1); v2 = rng0.standard_normal(d2)
    o2 = orc.attention_kl_head(Q1, K1 + v1, Q2, K2 + v2, c1, c2, causal, g=g)
    np.testing.assert_allclose(o2["kl"], o["kl"], atol=1e-12)
    np.testing.assert_allclose(o2["dQ1"], o["dQ1"] , atol=1e-12)
    np.testing.assert_allclose(o2["dQ2"], o["dQ2"], atol=1e-12)
    # ... and  sum_j dS_t[i,j] K-independent identity: q-weighted column sums  sum_j dK_t[j,:] = sum_i (sum_j dS[i,j]) q_i = 0
    np.testing.assert_allclose(o["dK1"].sum(0), 0, atol=1e-12)
    np.testing.assert_allclose(o["dK2"].sum(0), 0, atol=1e-12)
    # orthogonal rotation of (Q_t, K_t) leaves scalars unchanged and rotates the gradients
    R1, _ = np.linalg.qr(rng0.standard_normal((d1, d1))); R2, _ = np.linalg.qr(rng0.standard_normal((d2, d2)))
    o3 = orc.attention_kl_head(Q1 @ R1, K1 @ R1, Q2 @ R2, K2 @ R2, c1, c2, causal, g=g)
    np.testing.assert_allclose(o3["kl"], o["kl"], atol=1e-12)
    np.testing.assert_allclose(o3["dQ1"], o["dQ1"] @ R1, atol=1e-12)
    np.testing.assert_allclose(o3["dK2"], o["dK2"] @ R2, atol=1e-12)
    if not causal:  # permuting keys permutes dK rows only
        perm = rng0.permutation(NK)
        o4 = orc.attention_kl_head(Q1, K1[perm], Q2, K2[perm], c1, c2, False, g=g)
        np.testing.assert_allclose(o4["kl"], o["kl"], atol=1e-12)
        np.testing.assert_allclose(o4["dK1"], o["dK1"][perm], atol=1e-12)
        np.testing.assert_allclose(o4["dQ2"], o["dQ2"], atol=1e-12)
    # row grouping (the only blocking the oracle does) does not change anything
    o5 = orc.attention_kl_head(Q1, K1, Q2, K2, c1, c2, causal, g=g, row_block=5)
    for k in o:
        np.testing.assert_allclose(o5[k], o[k], atol=1e-13, err_msg=k)
    # Eq.8 / Alg.3 row term: KL + lse1 - lse2 = acc/l1 = E_P1[s1 - s2]
    rows = np.arange(NQ)
    vis = orc.visible_mask(rows, NQ, NK, causal)
    S1 = c1 * Q1 @ K1.T; S2 = c2 * Q2 @ K2.T
    P1 = np.where(vis, np.exp(S1 - o["lse1"][:, None]), 0)
    np.testing.assert_allclose(o["kl"] + o["lse1"] - o["lse2"], (P1 * (S1 - S2)).sum(1), atol=1e-12)


# ------------------------------------------------------------------ Algorithms 1-3 (literal) == definition, all block sizes
@pytest.mark.parametrize("causal", [False, True])
@pytest.mark.parametrize("BQ,BK", [(1, 1), (4, 3), (16, 16), (5, 64), (64, 7), (3, 1)])
def test_algorithms_literal_equal_definition(causal, BQ, BK):
    NQ, NK, d1, d2 = 19, 23, 5, 3
    Q1, K1, Q2, K2, g = _rand(NQ, NK, d1, d2, seed=12, scale=3.0)
    K1[5] *= 6.0  # a big running-max jump mid-stream (stresses the alpha1 rescale of acc, Eq.9-10)
    c1, c2 = 0.7, 0.5
    o = orc.attention_kl_head(Q1, K1, Q2, K2, c1, c2, causal, g=g)
    kl, l1, l2 = alg.algorithm1_forward(Q1, K1, Q2, K2, c1, c2, causal, BQ, BK)
    np.testing.assert_allclose(kl, o["kl"], atol=1e-12)
    np.testing.assert_allclose(l1, o["lse1"], atol=1e-12)
    np.testing.assert_allclose(l2, o["lse2"], atol=1e-12)
    np.testing.assert_allclose(alg.algorithm2_dQ2(Q1, K1, Q2, K2, c1, c2, causal, l1, l2, g, BQ, BK), o["dQ2"], atol=1e-12)
    np.testing.assert_allclose(alg.algorithm3_dQ1(Q1, K1, Q2, K2, c1, c2, causal, l1, l2, kl, g, BQ, BK), o["dQ1"], atol=1e-12)
    dK1, dK2 = alg.transposed_dK(Q1, K1, Q2, K2, c1, c2, causal, l1, l2, kl, g, BQ, BK)
    np.testing.assert_allclose(dK1, o["dK1"], atol=1e-12)
    np.testing.assert_allclose(dK2, o["dK2"], atol=1e-12)


@pytest.mark.parametrize("causal", [False, True])
@pytest.mark.parametrize("W", [2, 3, 5])
def test_splitk_merge_eq11(causal, W):
    NQ, NK = 6, 29
    Q1, K1, Q2, K2, _ = _rand(NQ, NK, 4, 4, seed=13, scale=2.0)
    o = orc.attention_kl_head(Q1, K1, Q2, K2, 0.5, 0.5, causal)
    CK = -(-NK // W)
    parts = [alg.algorithm1_forward(Q1, K1, Q2, K2, 0.5, 0.5, causal, 4, 5, key_range=(w * CK, min(NK, (w + 1) * CK)), finalize=False)
             for w in range(W)]
    tot = parts[0]
    for p in parts[1:]:
        tot = alg.merge_partials(tot, p)
    kl, l1, l2 = alg.finalize_stats(*tot)
    np.testing.assert_allclose(kl, o["kl"], atol=1e-12)
    np.testing.assert_allclose(l1, o["lse1"], atol=1e-12)
    np.testing.assert_allclose(l2, o["lse2"], atol=1e-12)


def test_batched_wrapper_matches_per_head():
    r = np.random.default_rng(14)
    Q1 = r.standard_normal((2, 3, 5, 4)); K1 = r.standard_normal((2, 3, 6, 4))
    Q2 = r.standard_normal((2, 3, 5, 2)); K2 = r.standard_normal((2, 3, 6, 2)); g = r.random((2, 3, 5))
    o = orc.attention_kl(Q1, K1, Q2, K2, 0.5, 0.7, True, g=g)
    o12 = orc.attention_kl_head(Q1[1, 2], K1[1, 2], Q2[1, 2], K2[1, 2], 0.5, 0.7, True, g=g[1, 2])
    for k in o12:
        np.testing.assert_array_equal(o[k][1, 2], o12[k])


# ------------------------------------------------------------------ student ReLU activation (R23)
@pytest.mark.parametrize("causal", [False, True])
def test_relu_student_against_torch_autograd(causal):
    """softmax(relu(c2 Q2 K2^T)) built from torch float64 primitives + autograd pins the forward values and all four gradients."""
    import torch

    NQ, NK, d1, d2 = 7, 11, 5, 4
    Q1, K1, Q2, K2, g = _rand(NQ, NK, d1, d2, seed=21)
    c1, c2 = 0.6, 0.8
    o = orc.attention_kl_head(Q1, K1, Q2, K2, c1, c2, causal, g=g, act2="relu")
    t = [torch.tensor(a, dtype=torch.float64, requires_grad=True) for a in (Q1, K1, Q2, K2)]
    S1 = c1 * t[0] @ t[1].T
    S2 = torch.relu(c2 * t[2] @ t[3].T)
    if causal:
        m = torch.arange(NK)[None, :] <= (torch.arange(NQ)[:, None] + NK - NQ)
        S1 = S1.masked_fill(~m, -math.inf); S2 = S2.masked_fill(~m, -math.inf)
    lp1 = torch.log_softmax(S1, -1); lp2 = torch.log_softmax(S2, -1)
    lse2 = torch.logsumexp(S2, -1).detach().numpy()
    if causal:  # -inf log-probs at masked entries would make 0*(-inf - -inf) = nan in kl_div
        lp1 = lp1.masked_fill(~m, -1e3); lp2 = lp2.masked_fill(~m, -1e3)  # exp(-1e3) == 0 exactly in float64
    kl = torch.nn.functional.kl_div(lp2, lp1, reduction="none", log_target=True).sum(-1)
    (kl * torch.tensor(g)).sum().backward()
    np.testing.assert_allclose(o["kl"], kl.detach().numpy(), atol=1e-12)
    np.testing.assert_allclose(o["lse2"], lse2, atol=1e-12)
    for k, x in zip(("dQ1", "dK1", "dQ2", "dK2"), t):
        np.testing.assert_allclose(o[k], x.grad.numpy(), atol=1e-11, err_msg=k)


def test_relu_student_closed_forms():
    """(a) every raw student logit <= 0  =>  relu makes P2 uniform: lse2 = log nV, KL = log nV - H(P1), student gradients vanish
    identically (the gate is 0 everywhere);  (b) every raw student logit > 0  =>  identical to the plain softmax student."""
    Q1, K1, _, _, g = _rand(6, 9, 4, 3, seed=22)
    r = np.random.default_rng(23)
    Q2 = np.abs(r.standard_normal((6, 3))); K2 = -np.abs(r.standard_normal((9, 3)))        # <q2,k2> < 0 always
    o = orc.attention_kl_head(Q1, K1, Q2, K2, 0.5, 0.9, False, g=g, act2="relu")
    np.testing.assert_allclose(o["lse2"], math.log(9.0), atol=1e-13)
    S1 = 0.5 * Q1 @ K1.T
    P1 = np.exp(S1 - S1.max(1, keepdims=True)); P1 /= P1.sum(1, keepdims=True)
    np.testing.assert_allclose(o["kl"], math.log(9.0) + (P1 * np.log(P1)).sum(1), atol=1e-12)
    assert np.abs(o["dQ2"]).max() == 0.0 and np.abs(o["dK2"]).max() == 0.0
    K2p = np.abs(K2)                                                                          # <q2,k2> > 0 always
    a = orc.attention_kl_head(Q1, K1, Q2, K2p, 0.5, 0.9, True, g=g, act2="relu")
    b = orc.attention_kl_head(Q1, K1, Q2, K2p, 0.5, 0.9, True, g=g)
    for k in a:
        np.testing.assert_allclose(a[k], b[k], atol=1e-14, err_msg=k)


def test_relu_student_finite_differences():
    """Central differences on sum_i g_i KL_i (kinks have measure zero for random inputs; h is far below the smallest |raw s2|)."""
    NQ, NK, d1, d2 = 5, 7, 4, 3
    Q1, K1, Q2, K2, g = _rand(NQ, NK, d1, d2, seed=24)
    c1, c2 = 0.7, 1.1
    assert np.abs(c2 * Q2 @ K2.T).min() > 1e-4
    o = orc.attention_kl_head(Q1, K1, Q2, K2, c1, c2, True, g=g, act2="relu")
    f = lambda a, b, c, d: float((g * orc.attention_kl_head(a, b, c, d, c1, c2, True, act2="relu")["kl"]).sum())
    h = 1e-6
    args = [Q1, K1, Q2, K2]
    for idx, name in enumerate(("dQ1", "dK1", "dQ2", "dK2")):
        num = np.zeros_like(args[idx])
        for i in np.ndindex(*args[idx].shape):
            ap = [x.copy() for x in args]; am = [x.copy() for x in args]
            ap[idx][i] += h; am[idx][i] -= h
            num[i] = (f(*ap) - f(*am)) / (2 * h)
        np.testing.assert_allclose(o[name], num, atol=2e-8, err_msg=name)
