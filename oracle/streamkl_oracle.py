"""CPU float64 ORACLE for StreamKL's result -- TEST INFRASTRUCTURE, not the product.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs may import this file.  It shares no code with `paper_2606_20005_b200/` (the CUDA path) and
imports nothing from it; the only common module is `workloads.py` (seeded inputs, no arithmetic).

What it computes.  StreamKL is EXACT (Eq.5-8 are algebraic identities), so the
oracle is the plain DEFINITION written out, materialising full rows of P1 and P2 -- precisely what
the method avoids -- in float64, with numpy library primitives (`@`, `exp`, `log`, `max`, `sum`) as
steps and no tiling/fusion/reordering beyond processing independent query rows in groups to bound
memory (rows never interact in the forward; dK is a plain sum over rows).

Per (b,h) and query row i  (readings R1,R2,R4,R5 of DESIGN.md):
  s_t[j]  = c_t * sum_k Q_t[i,k] K_t[j,k]                  t in {1,2}            (:49, :57)
  V_i     = all keys, or causal {j : j <= i + (NK-NQ)}     (bottom-right aligned; :214)
  lse_t   = log sum_{j in V_i} exp(s_t[j])                 (max-shifted)         (:76-79)
  logP_t  = s_t - lse_t ;  P_t = exp(logP_t)
  KL_i    = sum_{j in V_i} P1[j] * (logP1[j] - logP2[j])                         (Eq.1, :59)
  dS2     = g_i * (P2 - P1)                                                      (Eq.2, :64; Alg.2 :228)
  dS1     = g_i * P1 * ((logP1 - logP2) - KL_i)                                  (Eq.3, :69; Alg.3 :277)
  dQ_t    = c_t * dS_t @ K_t ;  dK_t = c_t * dS_t^T @ Q_t                        (:64, :69; chain rule on c_t)
Masked entries contribute 0 everywhere.  Outputs stay float64; nothing is rounded on this side.

Student activation ("Generalizability beyond Softmax": "the ReLU variant used in the indexer training of
DeepSeek-V3.2"; the paper gives no formula -- reading R23 of DESIGN.md).  With `act2="relu"` the student's logit passes through
ReLU BEFORE its softmax, s2[j] = relu(c2 <Q2[i], K2[j]>), exactly as that indexer scores a key (one indexer head, unit weight) and
is then trained with KL(P1 || softmax(s2)).  Everything above is unchanged with this s2; the chain rule adds relu'(.) = 1[c2 <q,k> > 0]
to the student's logit gradient:  dS2 = g_i (P2 - P1) * 1[raw s2 > 0]  (0 at the kink).  The teacher's gradient is Eq.3 verbatim.

Pins (tests/test_oracle_pins.py, `-m "not gpu"`): hand-derived worked example (tests/golden/),
closed forms (identical logits, P2 uniform, P1 uniform, NK=1, NK=2 Bernoulli), scipy
logsumexp/rel_entr, torch float64 autograd through log_softmax, central finite differences,
scalar brute force on N<=8, invariants (KL>=0, column sums of dK = 0, key-shift invariance).
Nothing here is "parity unpinned".
"""
from __future__ import annotations

import numpy as np

__all__ = ["visible_mask", "attention_kl_rows", "attention_kl_head", "attention_kl"]


def visible_mask(rows: np.ndarray, NQ: int, NK: int, causal: bool) -> np.ndarray:
    """Boolean [len(rows), NK]: True where key j is visible to query row i (R5: j <= i + NK - NQ)."""
    if not causal:
        return np.ones((len(rows), NK), dtype=bool)
    if NQ > NK:
        raise ValueError("causal with NQ > NK leaves rows with empty support (DESIGN.md R5)")
    j = np.arange(NK)[None, :]
    return j <= (np.asarray(rows)[:, None] + (NK - NQ))


def attention_kl_rows(Q1, K1, Q2, K2, c1, c2, causal, rows, g=None, teacher=True, act2=None):
    """Definition for a group of query rows of one head.

    Q_t [NQ,d_t], K_t [NK,d_t] float64.  rows: int array of query indices.
    Returns dict(kl, lse1, lse2 [R]); with g ([NQ] upstream gradient) also
    dQ2 [R,d2], dK2_part [NK,d2] (this group's contribution), and if teacher: dQ1, dK1_part.
    """
    rows = np.asarray(rows, dtype=np.int64)
    NQ, NK = Q1.shape[0], K1.shape[0]
    vis = visible_mask(rows, NQ, NK, causal)
    S1 = c1 * (Q1[rows] @ K1.T)  # [R,NK]  logits of distribution 1
    S2 = c2 * (Q2[rows] @ K2.T)
    if act2 not in (None, "relu"):
        raise ValueError("act2 must be None or 'relu'")
    if act2 == "relu":  # R23: the student's logit is relu(c2 q.k); its derivative gates dS2 below
        relu_grad = (S2 > 0.0).astype(np.float64)
        S2 = np.maximum(S2, 0.0)
    neg = -np.inf
    S1m = np.where(vis, S1, neg)
    S2m = np.where(vis, S2, neg)
    m1 = S1m.max(axis=1, keepdims=True)
    m2 = S2m.max(axis=1, keepdims=True)
    lse1 = m1 + np.log(np.exp(S1m - m1).sum(axis=1, keepdims=True))
    lse2 = m2 + np.log(np.exp(S2m - m2).sum(axis=1, keepdims=True))
    logP1 = np.where(vis, S1 - lse1, 0.0)  # finite placeholders at masked entries; weights there are 0
    logP2 = np.where(vis, S2 - lse2, 0.0)
    P1 = np.where(vis, np.exp(logP1), 0.0)
    P2 = np.where(vis, np.exp(logP2), 0.0)
    r = logP1 - logP2
    kl = (P1 * r).sum(axis=1)  # Eq.1
    out = {"kl": kl, "lse1": lse1[:, 0], "lse2": lse2[:, 0]}
    if g is None:
        return out
    gi = np.asarray(g, dtype=np.float64)[rows][:, None]
    dS2 = gi * (P2 - P1)  # Eq.2
    if act2 == "relu":
        dS2 = dS2 * relu_grad
    out["dQ2"] = c2 * (dS2 @ K2)
    out["dK2_part"] = c2 * (dS2.T @ Q2[rows])
    if teacher:
        dS1 = gi * P1 * (r - kl[:, None])  # Eq.3
        out["dQ1"] = c1 * (dS1 @ K1)
        out["dK1_part"] = c1 * (dS1.T @ Q1[rows])
    return out


def attention_kl_head(Q1, K1, Q2, K2, c1, c2, causal, g=None, teacher=True, row_block=None, act2=None):
    """Whole head: every query row, dK summed over all rows.  Inputs any float dtype; computed in float64."""
    Q1 = np.asarray(Q1, dtype=np.float64)
    K1 = np.asarray(K1, dtype=np.float64)
    Q2 = np.asarray(Q2, dtype=np.float64)
    K2 = np.asarray(K2, dtype=np.float64)
    NQ, NK = Q1.shape[0], K1.shape[0]
    if row_block is None:
        # bound the materialised [R,NK] float64 matrices (about 8 live at once) to ~2 GB
        row_block = int(max(1, min(NQ, (1 << 28) // (8 * max(NK, 1)))))
    res = {"kl": np.empty(NQ), "lse1": np.empty(NQ), "lse2": np.empty(NQ)}
    if g is not None:
        res["dQ2"] = np.empty((NQ, Q2.shape[1]))
        res["dK2"] = np.zeros((NK, K2.shape[1]))
        if teacher:
            res["dQ1"] = np.empty((NQ, Q1.shape[1]))
            res["dK1"] = np.zeros((NK, K1.shape[1]))
    for r0 in range(0, NQ, row_block):
        rows = np.arange(r0, min(NQ, r0 + row_block))
        part = attention_kl_rows(Q1, K1, Q2, K2, c1, c2, causal, rows, g, teacher, act2)
        for k in ("kl", "lse1", "lse2"):
            res[k][rows] = part[k]
        if g is not None:
            res["dQ2"][rows] = part["dQ2"]
            res["dK2"] += part["dK2_part"]
            if teacher:
                res["dQ1"][rows] = part["dQ1"]
                res["dK1"] += part["dK1_part"]
    return res


def attention_kl(Q1, K1, Q2, K2, c1, c2, causal, g=None, teacher=True, act2=None):
    """Batched [..., N, d] wrapper: loops over the leading (batch, head) axes, heads are independent."""
    Q1 = np.asarray(Q1)
    lead = Q1.shape[:-2]
    n = int(np.prod(lead)) if lead else 1
    Q1r = Q1.reshape((n,) + Q1.shape[-2:])
    K1r = np.asarray(K1).reshape((n,) + np.asarray(K1).shape[-2:])
    Q2r = np.asarray(Q2).reshape((n,) + np.asarray(Q2).shape[-2:])
    K2r = np.asarray(K2).reshape((n,) + np.asarray(K2).shape[-2:])
    gr = None if g is None else np.asarray(g).reshape(n, -1)
    outs = [
        attention_kl_head(Q1r[i], K1r[i], Q2r[i], K2r[i], c1, c2, causal, None if gr is None else gr[i], teacher, act2=act2)
        for i in range(n)
    ]
    return {k: np.stack([o[k] for o in outs]).reshape(lead + outs[0][k].shape) for k in outs[0]}
