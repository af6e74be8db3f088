"""ORACLE (test infrastructure, not product): RoPE and causal GQA attention in fp64, plain numpy.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
Shares no code with paper_2606_19667_b200/.

What the path computes (BASELINE.json north_star; PAPER.md:13, :31 "prefill … dominates latency", :33 APC
reuses cached blocks so only the uncached suffix is prefilled):
  RoPE (reading c4, paper silent; split-half "rotate_half" convention of the Llama/Qwen shapes in the configs):
     theta_i = p * theta^(-2i/D), i in [0, D/2)
     x'_i       = x_i cos(theta_i) - x_{i+D/2} sin(theta_i)
     x'_{i+D/2} = x_{i+D/2} cos(theta_i) + x_i sin(theta_i)          p = 0-based absolute token index
  attention for request r, head h, row at absolute position p:
     s_j = (q'_p . k'_j) / sqrt(D), 0 <= j <= p ;  P_j = exp(s_j - max)/sum ;  o = sum_j P_j v_j ; kv head = h // g
The definition is written out directly (a matmul is the only library step); no tiling, no online softmax,
no intermediate rounding.  Inputs are bf16 values converted exactly to fp64.
Pins: tests/test_oracle_attention.py (p=0 identity, norm preservation, shift invariance, rows of P sum to 1,
row 0 == v_0, constant V, Q=0 -> running mean, pure-Python loop brute force, torch SDPA fp64 special case,
suffix(c) rows == full(n) rows).
"""
from __future__ import annotations

import numpy as np


def rope(x: np.ndarray, positions: np.ndarray, theta: float) -> np.ndarray:
    """x: fp64 [T, H, D]; positions: int [T] absolute token index.  Returns fp64 [T, H, D]."""
    T, H, D = x.shape
    half = D // 2
    i = np.arange(half, dtype=np.float64)
    inv_freq = theta ** (-2.0 * i / D)                              # [D/2]
    ang = positions.astype(np.float64)[:, None] * inv_freq[None, :]  # [T, D/2]
    c, s = np.cos(ang)[:, None, :], np.sin(ang)[:, None, :]
    x1, x2 = x[..., :half], x[..., half:]
    return np.concatenate([x1 * c - x2 * s, x2 * c + x1 * s], axis=-1)


def softmax_rows(s: np.ndarray) -> np.ndarray:
    m = s.max(axis=-1, keepdims=True)
    e = np.exp(s - m)
    return e / e.sum(axis=-1, keepdims=True)


def attention_rows(q_r: np.ndarray, k_r: np.ndarray, v: np.ndarray, row_pos: np.ndarray,
                   return_probs: bool = False):
    """Causal GQA attention for a set of query rows.

    q_r  fp64 [S, Hq, D]   roped queries of the rows at absolute positions row_pos [S]
    k_r  fp64 [n, Hkv, D]  roped keys of ALL prompt positions 0..n-1 ; v fp64 [n, Hkv, D]
    Row i attends keys j <= row_pos[i].  Returns fp64 [S, Hq, D] (and P [Hq, S, n] if asked).
    """
    S, Hq, D = q_r.shape
    n, Hkv, _ = k_r.shape
    g = Hq // Hkv
    out = np.empty((S, Hq, D), dtype=np.float64)
    probs = np.zeros((Hq, S, n), dtype=np.float64) if return_probs else None
    j = np.arange(n)[None, :]
    allowed = j <= np.asarray(row_pos)[:, None]                     # [S, n]
    for h in range(Hq):
        kv = h // g
        s = (q_r[:, h, :] @ k_r[:, kv, :].T) / np.sqrt(float(D))    # [S, n]
        s = np.where(allowed, s, -np.inf)
        P = softmax_rows(s)
        out[:, h, :] = P @ v[:, kv, :]
        if return_probs:
            probs[h] = P
    return (out, probs) if return_probs else out


def attention_full(q: np.ndarray, k: np.ndarray, v: np.ndarray, theta: float) -> np.ndarray:
    """full(n): all n rows, c = 0.  q [n,Hq,D], k,v [n,Hkv,D] pre-RoPE fp64."""
    pos = np.arange(q.shape[0])
    return attention_rows(rope(q, pos, theta), rope(k, pos, theta), v, pos)


class PagedPool:
    """Oracle-side fp64 'pool' addressed through block tables (the oracle's own model of the paged KV pool).
    slot(p) = block_table[p // 16] * 16 + p % 16."""

    def __init__(self, num_blocks: int, Hkv: int, D: int):
        self.K = np.zeros((num_blocks * 16, Hkv, D), dtype=np.float64)
        self.V = np.zeros((num_blocks * 16, Hkv, D), dtype=np.float64)

    def slots(self, table, lo, hi):
        p = np.arange(lo, hi)
        return np.asarray(table)[p // 16] * 16 + p % 16

    def append(self, table, c, k_suffix, v_suffix, theta):
        """write RoPE'd K and plain V of suffix positions c..n-1."""
        s = k_suffix.shape[0]
        sl = self.slots(table, c, c + s)
        self.K[sl] = rope(k_suffix, np.arange(c, c + s), theta)
        self.V[sl] = v_suffix

    def gather(self, table, n):
        sl = self.slots(table, 0, n)
        return self.K[sl], self.V[sl]


def attention_suffix(pool: PagedPool, table, c: int, q_suffix, k_suffix, v_suffix, theta: float):
    """suffix(c): rows c..n-1 of a prompt whose first c positions are cached in `pool` (written there by
    earlier requests), exactly the a7+a8 steps: append the suffix K/V, then attend over prefix + suffix."""
    s = q_suffix.shape[0]
    n = c + s
    pool.append(table, c, k_suffix, v_suffix, theta)
    K, V = pool.gather(table, n)
    pos = np.arange(c, n)
    return attention_rows(rope(q_suffix, pos, theta), K, V, pos)


def attention_rows_loops(q, k, v, theta, rows, g):
    """Pure-Python restatement for tiny inputs (independent of the numpy vector code above): lists of floats,
    math.cos/sin/exp, explicit loops.  q [n][Hq][D], k,v [n][Hkv][D] python lists; returns {(p,h): [D]}."""
    import math
    n, Hq, D = len(q), len(q[0]), len(q[0][0])
    half = D // 2

    def rot(x, p):
        y = [0.0] * D
        for i in range(half):
            a = p * theta ** (-2.0 * i / D)
            y[i] = x[i] * math.cos(a) - x[i + half] * math.sin(a)
            y[i + half] = x[i + half] * math.cos(a) + x[i] * math.sin(a)
        return y

    res = {}
    for p in rows:
        for h in range(Hq):
            qq = rot(q[p][h], p)
            sc = []
            for j in range(p + 1):
                kk = rot(k[j][h // g], j)
                sc.append(sum(a * b for a, b in zip(qq, kk)) / math.sqrt(D))
            mx = max(sc)
            e = [math.exp(x - mx) for x in sc]
            z = sum(e)
            res[(p, h)] = [sum(e[j] / z * v[j][h // g][d] for j in range(p + 1)) for d in range(D)]
    return res
