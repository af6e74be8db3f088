"""ORACLE (test infrastructure, not product): the ordering arms the paper compares with (Table 4).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
Shares no code with paper_2606_19667_b200/.

The paper names the arms but does not define them beyond a phrase; the readings ("strategy arms"):
  sorted     "APC+Sorted": lexicographic sorting — "a canonical, query-independent order": ascending
             document id.
  recency    "a recency heuristic": documents served most recently first.  last_served[d] = index (seq)
             of the last finished request whose order contained d; never-served documents last; ties keep retrieval rank.
  exhaustive "an exhaustive oracle": of all k! orders the one with the most blocks actually
             matched by the prefix cache (a peek lookup on the real block index); first maximiser in lexicographic
             order of retrieval-rank indices.  (The trie-objective optimum is KnowledgeTree.brute_force_permutations.)
"""
from __future__ import annotations

from itertools import permutations


def order_sorted(D):
    return sorted(D)


class RecencyOrder:
    def __init__(self):
        self.last_served = {}
        self.seq = 0

    def observe(self, order):
        self.seq += 1
        for d in order:
            self.last_served[d] = self.seq

    def order(self, D):
        # stable sort: descending last-served index, never-served (0) last, ties in retrieval rank
        return sorted(D, key=lambda d: -self.last_served.get(d, 0))


def order_exhaustive(D, cached_tokens_of):
    """cached_tokens_of(order) -> tokens the prefix cache would match for that order (peek, no state change)."""
    best, best_c = list(D), -1
    for perm in permutations(range(len(D))):
        O = [D[i] for i in perm]
        c = cached_tokens_of(O)
        if c > best_c:
            best, best_c = O, c
    return best, best_c
