"""Test-only helpers that are independent of both the oracle and the CUDA path."""
from __future__ import annotations

import itertools

import numpy as np


def dense_h(base_shifts: np.ndarray, Z: int) -> np.ndarray:
    """Dense H from the PRINTED lifting rule: block (R,C) with shift p is the ZxZ identity with each row
    cyclically shifted right by p (np.roll along columns); -1 is the zero block."""
    mb, nb = base_shifts.shape
    H = np.zeros((mb * Z, nb * Z), dtype=np.uint8)
    eye = np.eye(Z, dtype=np.uint8)
    for R in range(mb):
        for C in range(nb):
            p = int(base_shifts[R, C])
            if p >= 0:
                H[R * Z:(R + 1) * Z, C * Z:(C + 1) * Z] = np.roll(eye, p, axis=1)
    return H


def all_words(n: int) -> np.ndarray:
    """All 2^n binary words, uint8 [2^n][n]."""
    idx = np.arange(1 << n, dtype=np.uint32)
    return ((idx[:, None] >> np.arange(n, dtype=np.uint32)[None, :]) & 1).astype(np.uint8)


def bitwise_map_llr(H: np.ndarray, s: np.ndarray, Q: np.ndarray) -> np.ndarray:
    """Exact a-posteriori LLR of every bit given H x = s and channel LLRs Q (ln P0/P1), by enumeration:
    L_v = ln sum_{x: Hx=s, x_v=0} e^{l(x)} - ln sum_{x: Hx=s, x_v=1} e^{l(x)},  l(x) = sum_{v: x_v=0} Q_v."""
    n = H.shape[1]
    X = all_words(n)
    ok = ((X.astype(np.int64) @ H.T.astype(np.int64)) % 2 == s[None, :]).all(axis=1)
    X = X[ok]
    ell = ((1 - X.astype(np.float64)) * Q[None, :].astype(np.float64)).sum(axis=1)
    out = np.empty(n)
    for v in range(n):
        a = ell[X[:, v] == 0]
        b = ell[X[:, v] == 1]
        la = np.logaddexp.reduce(a) if a.size else -np.inf
        lb = np.logaddexp.reduce(b) if b.size else -np.inf
        out[v] = la - lb
    return out


def block_ml_word(H: np.ndarray, s: np.ndarray, Q: np.ndarray):
    """The word maximising l(x) among H x = s, and its l(x)."""
    n = H.shape[1]
    X = all_words(n)
    ok = ((X.astype(np.int64) @ H.T.astype(np.int64)) % 2 == s[None, :]).all(axis=1)
    X = X[ok]
    ell = ((1 - X.astype(np.float64)) * Q[None, :].astype(np.float64)).sum(axis=1)
    k = int(np.argmax(ell))
    return X[k], float(ell[k])


def random_tree_code(rng: np.random.Generator, n_target: int, max_check_deg: int = 4):
    """A cycle-free Tanner graph (Z=1 base matrix, entries 0 / -1) with every check degree >= 2:
    grow by attaching a new check to an existing variable plus 1..max_check_deg-1 NEW variables."""
    n = 1
    rows = []
    while n < n_target:
        k_new = int(rng.integers(1, max_check_deg))
        k_new = min(k_new, n_target - n)
        anchor = int(rng.integers(0, n))
        rows.append([anchor] + list(range(n, n + k_new)))
        n += k_new
    base = np.full((len(rows), n), -1, dtype=np.int32)
    for r, vs in enumerate(rows):
        base[r, vs] = 0
    return base


def tanh_rule_bp_dense(H: np.ndarray, Q: np.ndarray, s: np.ndarray, n_iter: int, msg_max: float):
    """Independent dense-matrix flooding BP using the tanh-product form  m_cv = 2 atanh( prod tanh(L_v'c / 2) )
    (a different formula from the oracle's Phi-sum form; equal in exact arithmetic).  Returns posteriors float64 [n]."""
    m, n = H.shape
    Hb = H.astype(bool)
    Lvc = np.where(Hb, Q[None, :].astype(np.float64), 0.0)
    Lv = Q.astype(np.float64).copy()
    for _ in range(n_iter):
        T = np.where(Hb, np.tanh(Lvc / 2.0), 1.0)
        M = np.zeros((m, n))
        for c in range(m):
            vs = np.nonzero(Hb[c])[0]
            for v in vs:
                others = [u for u in vs if u != v]
                p = np.prod(T[c, others]) * (-1.0 if s[c] else 1.0)
                p = np.clip(p, -1.0, 1.0)
                with np.errstate(divide="ignore"):
                    val = 2.0 * np.arctanh(p)
                M[c, v] = np.clip(val, -msg_max, msg_max)
        Lv = Q + M.sum(axis=0)
        Lvc = np.where(Hb, Lv[None, :] - M, 0.0)
    return Lv


def tie_cases():
    """Inputs whose posterior L_v is EXACTLY zero in any IEEE arithmetic, so that Step 4 ("0 if L_v >= 0") is
    decided by the tie rule alone.  Each case: (base, Z, llr [n], syndrome [m], max_iter, variables that tie).
      zero column        a variable without any check: L_v = Q_v = +0.0 or -0.0 (max_iter = 0 takes the decisions of
                         Step 1, max_iter > 0 those of Step 4);
      clamped checks     a variable whose only neighbours are two checks of degree 1: the exclusion set of a degree-1
                         check is empty, S = 0, |m_cv| = Phi(0) = inf clamped to 30 (reading S2), sign (-1)^{s_c}; with
                         Q_v = -/+60 the posterior is -60 + 30 + 30 = 0 (s = 0) or 60 - 30 - 30 = 0 (s = 1): all terms
                         dyadic multiples, exact in float and double in any summation order."""
    cases = []
    one_check = np.array([[-1, 0, 0]], dtype=np.int32)               # column 0 is empty
    for q0 in (0.0, -0.0):
        for it in (0, 3):
            cases.append((one_check, 1, np.array([q0, 1.0, -2.0], np.float32), np.zeros(1, np.uint8), it, [0]))
    two_leaves = np.array([[0], [0]], dtype=np.int32)                # one variable, two degree-1 checks
    for Z in (1, 5):
        cases.append((two_leaves, Z, np.full(Z, -60.0, np.float32), np.zeros(2 * Z, np.uint8), 2, list(range(Z))))
        cases.append((two_leaves, Z, np.full(Z, 60.0, np.float32), np.ones(2 * Z, np.uint8), 2, list(range(Z))))
    return cases
