"""TEST INFRASTRUCTURE (CPU oracle; only tests/, smoke() and bench.py's cpu_baseline leg may import it).

Subdomain recovery for a CSR Hamiltonian whose rows arrive in arbitrary order WITHOUT labels (SURVEY.md 8(a) step A0
"group rows so each subdomain's basis functions are contiguous", 8(f)-4 "locality recovery for unhinted CSR"; the paper
only states the structure that makes it possible: the basis functions of a subdomain overlap each other, so the diagonal
blocks are dense, and they overlap the neighbouring subdomains' functions).  The paper gives no
algorithm for this, so the algorithm is DESIGN.md reading #18, followed here step by step, in exact integer arithmetic, with
python sets and one library step (the common-neighbour counts c_ij are the entries of A A^T for the 0/1 pattern matrix A, taken
from scipy's sparse product; `counts="sets"` computes them by set intersection instead, for the pin that checks the two agree):

  N(i) = column set of row i.
  1. for every row i and every j in N(i), j != i:  c_ij = |N(i) & N(j)|,  u_ij = |N(i)| + |N(j)| - c_ij   (Jaccard c/u).
     (c*, u*) = the largest fraction of the row;  S(i) = {i} + {j : 5 c_ij u* >= 4 c* u_ij}   (within 80 % of the best match);
     S(i) = {i} if the row has no other column or c* = 0.  If any |S(i)| > 192 the matrix has no recoverable structure: fail.
  2. V(i) = {j in S(i) : 2 |S(i) & S(j)| >= max(|S(i)|, |S(j)|)}            (a pair is kept only if their candidate sets agree)
  3. root(i) = the smallest row index reachable from i along edges i -> j in V(i) (fixed point of L[i] = min(i, min_j L[j])).
  4. the roots in ascending order are numbered 0, 1, ...; label(i) = number of root(i).

Pins (tests/test_oracle_pins.py, P10): the planted partition of the synthetic generator under a random symmetric permutation is
returned exactly (z = 0: rows of a subdomain have identical column sets, Jaccard exactly 1, a closed form; z > 0: statistical
separation); a diagonal matrix gives M singletons; the labels do not depend on the order of the rows' entries.
"""
from __future__ import annotations

import numpy as np

CAP = 192   # largest candidate set (the largest tile is 128 rows)


def recover_subdomains(row_ptr: np.ndarray, col_idx: np.ndarray, counts: str = "product"):
    """Returns (labels int32[M], n_groups) or (None, 0) if a candidate set exceeds CAP."""
    M = len(row_ptr) - 1
    N = [frozenset(int(c) for c in col_idx[row_ptr[i]:row_ptr[i + 1]]) for i in range(M)]
    P = None
    if counts == "product":
        import scipy.sparse as sp
        A = sp.csr_matrix((np.ones(len(col_idx), np.int64), np.asarray(col_idx, np.int64), np.asarray(row_ptr, np.int64)), shape=(M, M))
        P = (A @ A.T).toarray()          # P[i, j] = |N(i) & N(j)|
    S = []
    for i in range(M):
        frac = {}
        for j in N[i]:
            if j == i:
                continue
            c = int(P[i, j]) if P is not None else len(N[i] & N[j])
            frac[j] = (c, len(N[i]) + len(N[j]) - c)
        best = None
        for (c, u) in frac.values():
            if best is None or c * best[1] > best[0] * u:
                best = (c, u)
        s = {i}
        if best is not None and best[0] > 0:
            for j, (c, u) in frac.items():
                if 5 * c * best[1] >= 4 * best[0] * u:
                    s.add(j)
        if len(s) > CAP:
            return None, 0
        S.append(frozenset(s))
    V = [[j for j in S[i] if 2 * len(S[i] & S[j]) >= max(len(S[i]), len(S[j]))] for i in range(M)]
    L = list(range(M))
    changed = True
    while changed:
        changed = False
        for i in range(M):
            m = min([L[i]] + [L[j] for j in V[i]])
            if m < L[i]:
                L[i] = m
                changed = True
    roots = sorted(i for i in range(M) if L[i] == i)
    number = {r: k for k, r in enumerate(roots)}
    return np.array([number[L[i]] for i in range(M)], dtype=np.int32), len(roots)
