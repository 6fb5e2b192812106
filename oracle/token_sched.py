"""Token Scheduler -- ORACLE, TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).

Follows PAPER.md §3.3 step by step, in the paper's order and notation (plain numpy / Python loops, integers
only; nothing blocked, packed or fused):

  * problem (§3.3.2): 2T tokens with binary routing-path matrices r_i of size (L, E) are split into
    two batches T_1, T_2 of exactly T tokens; the batch-level path R_b combines its tokens' paths (Eq. 4) and the
    objective counts the activated experts of both batches (Eq. 5).  Eq. 4 prints an element-wise AND, but the
    objective "counts the total number of activated experts in a batch" and Eq. 7's text uses OR:
    reading R14 takes OR -- `batch_path`.
  * similarity (§3.3.3, Eq. 6): S_ij = 1 - d_ij / (L*E), d_ij = Hamming distance of r_i and r_j --
    `hamming_matrix`, `similarity_matrix`.
  * balanced K-means with K = 2: random centroid selection (the two tokens drawn are an INPUT here);
    assign each token to the centroid it is most similar to; when a cluster exceeds T, adjust until both hold
    exactly T; new centroid = the token of the cluster with the highest average similarity to the others;
    repeat until convergence or an iteration limit -- `schedule`.

The appendix the paper refers to for the exact K-means procedure is not part of PAPER.md, so the
points it would settle are DESIGN.md readings R26-R29:
  R26  "adjustments when a cluster exceeds T": the tokens with the weakest preference for the over-full cluster
       move to the other one, i.e. cluster 0 = the T tokens with the largest margin S[i,c0] - S[i,c1].
  R27  ties (equal margin; equal average similarity) go to the lower token index.
  R28  convergence = both centroids unchanged by the update (the next assignment would repeat).
  R29  a centroid is a token (a medoid), as the update rule says; "average similarity to the others" excludes
       the token itself (S_ii = 1 adds the same constant to every candidate, so the argmax is unaffected).
Fidelity of R26-R29 to the authors' code: parity unpinned (no code, no appendix).  Everything the text does fix
is pinned in tests/test_oracle_token_sched.py (Fig. 4's example, Eq. 5 by brute force, Eq. 6 closed forms).
"""
from __future__ import annotations

from dataclasses import dataclass
from itertools import combinations

import numpy as np


def hamming_matrix(r: np.ndarray) -> np.ndarray:
    """d_ij of Eq. 6: r is [N, L, E] (or [N, L*E]) of 0/1; returns int64 [N, N]."""
    r = np.asarray(r).reshape(len(r), -1) != 0
    n = r.shape[0]
    d = np.zeros((n, n), np.int64)
    for i in range(n):
        d[i, :] = (r != r[i]).sum(axis=1)       # number of (layer, expert) entries where r_i and r_j differ
    return d


def similarity_matrix(r: np.ndarray) -> np.ndarray:
    """S_ij = 1 - d_ij / (L * E)   (Eq. 6)."""
    r = np.asarray(r)
    le = int(np.prod(r.shape[1:]))
    return 1.0 - hamming_matrix(r) / float(le)


def batch_path(r: np.ndarray, members) -> np.ndarray:
    """Batch-level routing path R of Eq. 4 for the token set `members` (OR over tokens, reading R14)."""
    r = np.asarray(r).reshape(len(r), -1)
    out = np.zeros(r.shape[1], np.uint8)
    for i in members:
        out |= (r[i] != 0).astype(np.uint8)
    return out


def batch_accuracy(r_batch: np.ndarray, r_batch_hat: np.ndarray) -> float:
    """B_acc of Eq. 7: the mean over the L layers of
        #{j : R_batch[i,j] = 1 and R^_batch[i,j] = 1} / #{j : R_batch[i,j] = 1},
    R_batch the true and R^_batch the predicted batch-level routing path, both binary (L, E) (each the OR of its
    tokens' paths, P:L239 -- `batch_path`).  Plain loops in the paper's index order.  A layer in which the true path
    activates no expert has no defined ratio; it is left out of the mean (cannot happen with top-k >= 1 routing)."""
    R = np.asarray(r_batch) != 0
    Rh = np.asarray(r_batch_hat) != 0
    assert R.shape == Rh.shape and R.ndim == 2
    L, E = R.shape
    total, layers = 0.0, 0
    for i in range(L):
        num = den = 0
        for j in range(E):
            if R[i, j]:
                den += 1
                if Rh[i, j]:
                    num += 1
        if den:
            total += num / den
            layers += 1
    return total / layers if layers else float("nan")


def objective(r: np.ndarray, batch_of) -> int:
    """Eq. 5: activated experts summed over layers, experts and the two batches."""
    batch_of = np.asarray(batch_of)
    return int(sum(int(batch_path(r, np.flatnonzero(batch_of == b)).sum()) for b in (0, 1)))


def brute_force_optimum(r: np.ndarray) -> int:
    """min of Eq. 5 over every balanced split (only for tiny N)."""
    n = len(r)
    assert n % 2 == 0 and n <= 14
    best = None
    for t1 in combinations(range(n), n // 2):
        if 0 not in t1:          # the two batches are interchangeable
            continue
        b = np.ones(n, np.int64)
        b[list(t1)] = 0
        v = objective(r, b)
        best = v if best is None else min(best, v)
    return int(best)


def assign_balanced(d: np.ndarray, c0: int, c1: int) -> np.ndarray:
    """One assignment step (P:L173 + R26/R27): cluster 0 = the T tokens with the largest S[i,c0] - S[i,c1]
    (= largest d[i,c1] - d[i,c0]; the common factor 1/(L*E) does not change the order), ties -> lower index."""
    n = d.shape[0]
    margin = [int(d[i, c1] - d[i, c0]) for i in range(n)]
    order = sorted(range(n), key=lambda i: (-margin[i], i))
    batch_of = np.ones(n, np.int64)
    batch_of[order[: n // 2]] = 0
    return batch_of


def medoid(d: np.ndarray, members) -> int:
    """The token of the cluster with the highest average similarity to the others (R27/R29) = the one
    with the smallest summed distance to the cluster; ties -> lower index."""
    members = np.sort(np.asarray(members, np.int64))
    sums = d[np.ix_(members, members)].sum(axis=1)      # d_ii = 0, so "the others" needs no special case
    return int(members[int(np.argmin(sums))])            # argmin returns the first minimum = the lowest index


@dataclass
class Schedule:
    batch_of: np.ndarray      # int32 [2T] in {0, 1}
    perm: np.ndarray          # int32 [2T]: tokens of T_1 ascending, then tokens of T_2 ascending ("Reindex")
    centroids: tuple          # final (c0, c1)
    iters: int                # assignment+update rounds executed
    converged: bool
    objective: int            # Eq. 5 of the result
    objective_before: int     # Eq. 5 of the input batching: tokens [0, T) and [T, 2T)


def schedule(r: np.ndarray, c0: int, c1: int, max_iter: int = 16) -> Schedule:
    """Balanced 2-means over the Hamming similarity of routing paths, from the drawn centroids (c0, c1)."""
    r = np.asarray(r)
    n = len(r)
    assert n % 2 == 0 and n >= 2 and 0 <= c0 < n and 0 <= c1 < n and c0 != c1 and max_iter >= 1
    d = hamming_matrix(r)
    converged = False
    iters = 0
    batch_of = None
    for _ in range(max_iter):
        batch_of = assign_balanced(d, c0, c1)
        n0 = medoid(d, np.flatnonzero(batch_of == 0))
        n1 = medoid(d, np.flatnonzero(batch_of == 1))
        iters += 1
        if (n0, n1) == (c0, c1):
            converged = True
            break
        c0, c1 = n0, n1
    perm = np.concatenate([np.flatnonzero(batch_of == 0), np.flatnonzero(batch_of == 1)]).astype(np.int32)
    before = np.concatenate([np.zeros(n // 2, np.int64), np.ones(n // 2, np.int64)])
    return Schedule(batch_of.astype(np.int32), perm, (int(c0), int(c1)), iters, converged, objective(r, batch_of),
                    objective(r, before))
