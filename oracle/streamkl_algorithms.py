"""Literal float64 transcriptions of the paper's Algorithms 1-3 and Eq.11 -- TEST INFRASTRUCTURE.

Same rules as `streamkl_oracle.py`: only tests/smoke/bench-cpu-baseline may import this, it shares
no code with the CUDA path.  Where `streamkl_oracle.py` writes out the DEFINITION, this file follows
the paper's STREAMING algorithms step by step, in the paper's order and notation, for arbitrary
block sizes (B_Q, B_K), including B_K=1, B_K=N_K and non-dividing sizes.  Tests check
"algorithm == definition" for every block size: that pins the rescaling logic (Eq.9-10) and the
recompute formulas (Alg.2/3, Eq.12) independently of any GPU.

Readings applied: R1 scale c_t on the logits; R5 causal j <= i + NK - NQ; R7 when the
new running maximum is still -inf the correction factor is taken as exp(0-0) (FlashAttention
convention) so (-inf)-(-inf) never forms; R8 the difference S1-S2 is taken from the RAW logits and
P~ is zeroed at masked entries; R9 acc and l1 scale by alpha1 only, l2 by alpha2 only; R10 loop order
loop -> LSE -> KL -> write; R11 split-K partials carry (m2,l2) too.
"""
from __future__ import annotations

import numpy as np


def _vis(i0, i1, j0, j1, NQ, NK, causal):
    if not causal:
        return np.ones((i1 - i0, j1 - j0), dtype=bool)
    ii = np.arange(i0, i1)[:, None]
    jj = np.arange(j0, j1)[None, :]
    return jj <= ii + (NK - NQ)


def algorithm1_forward(Q1, K1, Q2, K2, c1, c2, causal, BQ, BK, key_range=None, finalize=True):
    """Algorithm 1.  Returns (KL, LSE1, LSE2) or, with finalize=False, the raw
    running statistics (m1,l1,m2,l2,acc) over `key_range=(lo,hi)` -- a split-K partial (:238)."""
    Q1, K1, Q2, K2 = (np.asarray(a, dtype=np.float64) for a in (Q1, K1, Q2, K2))
    NQ, NK = Q1.shape[0], K1.shape[0]
    lo, hi = (0, NK) if key_range is None else key_range
    m1 = np.full(NQ, -np.inf)
    m2 = np.full(NQ, -np.inf)
    l1 = np.zeros(NQ)
    l2 = np.zeros(NQ)
    acc = np.zeros(NQ)
    for i0 in range(0, NQ, BQ):  # line 2: for 1 <= i <= T_Q in parallel
        i1 = min(NQ, i0 + BQ)
        Q1i, Q2i = Q1[i0:i1], Q2[i0:i1]  # line 3
        m1i, m2i = m1[i0:i1].copy(), m2[i0:i1].copy()  # line 4 (already -inf / 0)
        l1i, l2i, acci = l1[i0:i1].copy(), l2[i0:i1].copy(), acc[i0:i1].copy()
        for j0 in range(lo, hi, BK):  # line 5
            j1 = min(hi, j0 + BK)
            if causal and j0 > (i1 - 1) + (NK - NQ):
                break  # :214 early exit past the causal frontier
            S1 = c1 * (Q1i @ K1[j0:j1].T)  # line 7
            S2 = c2 * (Q2i @ K2[j0:j1].T)
            vis = _vis(i0, i1, j0, j1, NQ, NK, causal)
            S1m = np.where(vis, S1, -np.inf)
            S2m = np.where(vis, S2, -np.inf)
            m1n = np.maximum(m1i, S1m.max(axis=1))  # line 8
            m2n = np.maximum(m2i, S2m.max(axis=1))
            ref1 = np.where(np.isfinite(m1n), m1n, 0.0)  # R7
            ref2 = np.where(np.isfinite(m2n), m2n, 0.0)
            a1 = np.exp(m1i - ref1)  # line 9 (m^(0) = -inf gives alpha = 0 on the first tile)
            a2 = np.exp(m2i - ref2)
            P1t = np.exp(S1m - ref1[:, None])  # line 10; masked entries are exp(-inf) = 0
            P2t = np.exp(S2m - ref2[:, None])
            l1i = a1 * l1i + P1t.sum(axis=1)  # line 11
            l2i = a2 * l2i + P2t.sum(axis=1)
            acci = a1 * acci + (P1t * (S1 - S2)).sum(axis=1)  # line 12, R8: raw-logit difference
            m1i, m2i = m1n, m2n
        m1[i0:i1], m2[i0:i1], l1[i0:i1], l2[i0:i1], acc[i0:i1] = m1i, m2i, l1i, l2i, acci
    if not finalize:
        return m1, l1, m2, l2, acc
    return finalize_stats(m1, l1, m2, l2, acc)


def finalize_stats(m1, l1, m2, l2, acc):
    """Lines 13-15: LSE_t = m_t + log l_t ; KL = acc/l1 + LSE2 - LSE1 (Eq.8)."""
    LSE1 = m1 + np.log(l1)
    LSE2 = m2 + np.log(l2)
    return acc / l1 + LSE2 - LSE1, LSE1, LSE2


def merge_partials(a, b):
    """Eq.11 for two partials (m1,l1,m2,l2,acc); (m2,l2) merged the same way (R11)."""
    m1a, l1a, m2a, l2a, acca = a
    m1b, l1b, m2b, l2b, accb = b
    m1 = np.maximum(m1a, m1b)
    m2 = np.maximum(m2a, m2b)
    r1 = np.where(np.isfinite(m1), m1, 0.0)
    r2 = np.where(np.isfinite(m2), m2, 0.0)
    ea, eb = np.exp(m1a - r1), np.exp(m1b - r1)
    fa, fb = np.exp(m2a - r2), np.exp(m2b - r2)
    return m1, l1a * ea + l1b * eb, m2, l2a * fa + l2b * fb, acca * ea + accb * eb


def algorithm2_dQ2(Q1, K1, Q2, K2, c1, c2, causal, LSE1, LSE2, dL, BQ, BK):
    """Algorithm 2: dQ2 by recomputation, P_t = exp(S_t - LSE_t), dS2 = dL*(P2-P1)."""
    Q1, K1, Q2, K2 = (np.asarray(a, dtype=np.float64) for a in (Q1, K1, Q2, K2))
    NQ, NK = Q1.shape[0], K1.shape[0]
    dQ2 = np.zeros_like(Q2)
    for i0 in range(0, NQ, BQ):
        i1 = min(NQ, i0 + BQ)
        accq = np.zeros((i1 - i0, Q2.shape[1]))  # line 3
        for j0 in range(0, NK, BK):
            j1 = min(NK, j0 + BK)
            if causal and j0 > (i1 - 1) + (NK - NQ):
                break
            S1 = c1 * (Q1[i0:i1] @ K1[j0:j1].T)  # line 6
            S2 = c2 * (Q2[i0:i1] @ K2[j0:j1].T)
            vis = _vis(i0, i1, j0, j1, NQ, NK, causal)
            P1 = np.exp(np.where(vis, S1, -np.inf) - LSE1[i0:i1, None])  # line 7; masked -> 0
            P2 = np.exp(np.where(vis, S2, -np.inf) - LSE2[i0:i1, None])
            dS2 = dL[i0:i1, None] * (P2 - P1)  # line 8
            accq += c2 * (dS2 @ K2[j0:j1])  # line 9 (+ chain-rule factor c2, R1)
        dQ2[i0:i1] = accq  # line 11
    return dQ2


def algorithm3_dQ1(Q1, K1, Q2, K2, c1, c2, causal, LSE1, LSE2, L, dL, BQ, BK):
    """Algorithm 3: delta = LSE1-LSE2, r = (S1-S2)-delta (Eq.12), dS1 = dL*P1*(r-L)."""
    Q1, K1, Q2, K2 = (np.asarray(a, dtype=np.float64) for a in (Q1, K1, Q2, K2))
    NQ, NK = Q1.shape[0], K1.shape[0]
    dQ1 = np.zeros_like(Q1)
    delta = LSE1 - LSE2  # line 3
    for i0 in range(0, NQ, BQ):
        i1 = min(NQ, i0 + BQ)
        accq = np.zeros((i1 - i0, Q1.shape[1]))
        for j0 in range(0, NK, BK):
            j1 = min(NK, j0 + BK)
            if causal and j0 > (i1 - 1) + (NK - NQ):
                break
            S1 = c1 * (Q1[i0:i1] @ K1[j0:j1].T)
            S2 = c2 * (Q2[i0:i1] @ K2[j0:j1].T)
            vis = _vis(i0, i1, j0, j1, NQ, NK, causal)
            P1 = np.exp(np.where(vis, S1, -np.inf) - LSE1[i0:i1, None])  # line 8; masked -> 0
            r = (S1 - S2) - delta[i0:i1, None]  # line 9
            dS1 = dL[i0:i1, None] * P1 * (r - L[i0:i1, None])  # line 10
            accq += c1 * (dS1 @ K1[j0:j1])  # line 11
        dQ1[i0:i1] = accq
    return dQ1


def transposed_dK(Q1, K1, Q2, K2, c1, c2, causal, LSE1, LSE2, L, dL, BQ, BK):
    """The K-tile-owner loops the paper describes in prose: each block owns K tile j,
    iterates over all query tiles and accumulates dK2_j = sum_i dS2^T Q2_i and dK1_j = sum_i dS1^T Q1_i."""
    Q1, K1, Q2, K2 = (np.asarray(a, dtype=np.float64) for a in (Q1, K1, Q2, K2))
    NQ, NK = Q1.shape[0], K1.shape[0]
    dK1, dK2 = np.zeros_like(K1), np.zeros_like(K2)
    delta = LSE1 - LSE2
    for j0 in range(0, NK, BK):
        j1 = min(NK, j0 + BK)
        a1 = np.zeros((j1 - j0, K1.shape[1]))
        a2 = np.zeros((j1 - j0, K2.shape[1]))
        for i0 in range(0, NQ, BQ):
            i1 = min(NQ, i0 + BQ)
            if causal and j0 > (i1 - 1) + (NK - NQ):
                continue  # whole tile pair masked
            S1 = c1 * (Q1[i0:i1] @ K1[j0:j1].T)
            S2 = c2 * (Q2[i0:i1] @ K2[j0:j1].T)
            vis = _vis(i0, i1, j0, j1, NQ, NK, causal)
            P1 = np.exp(np.where(vis, S1, -np.inf) - LSE1[i0:i1, None])
            P2 = np.exp(np.where(vis, S2, -np.inf) - LSE2[i0:i1, None])
            dS2 = dL[i0:i1, None] * (P2 - P1)
            dS1 = dL[i0:i1, None] * P1 * ((S1 - S2) - delta[i0:i1, None] - L[i0:i1, None])
            a2 += c2 * (dS2.T @ Q2[i0:i1])
            a1 += c1 * (dS1.T @ Q1[i0:i1])
        dK1[j0:j1], dK2[j0:j1] = a1, a2
    return dK1, dK2
