"""ORACLE (test infrastructure, not product): CacheWeaver knowledge tree + greedy ordering, plain Python.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It shares no code with paper_2606_19667_b200/ and never imports it.

Follows PAPER.md step by step:
  * knowledge tree (trie of recently served document orders)        PAPER.md:57  (§3.2)
  * Algorithm 1 "Cache-Aware Evidence Ordering"
  * objective l(O,T), Eq. (1): reusable cached prefix depth          PAPER.md:61 (garbled), :100-104
  * exhaustive oracle ordering over k! permutations
Readings where the paper is silent (listed in DESIGN.md):
  isCached(node)  <=>  seq - node.last_seq < H   (recency of service)
  "for each d in R" scans R in retrieval rank and takes the first hit (D is given in retrieval rank, :66).
Pins: tests/test_oracle_ordering.py (Figure 2 and Figure 1 worked examples, fallback, permutation/tail
properties, probe bound k(k+1)/2, greedy == brute force when no branch ambiguity, two brute forces agree).
"""
from __future__ import annotations

from itertools import permutations


class Node:
    __slots__ = ("doc", "children", "last_seq")

    def __init__(self, doc):
        self.doc = doc
        self.children = {}
        self.last_seq = 0


class KnowledgeTree:
    def __init__(self, recency_window: int):
        self.H = int(recency_window)
        self.root = Node(None)
        self.seq = 0
        self.probes = 0            # child lookups done by the last order() call

    # PAPER.md:57 "after a request finishes, its ordered document sequence is inserted"
    def observe(self, order):
        self.seq += 1
        node = self.root
        for d in order:
            c = node.children.get(d)
            if c is None:
                c = Node(d)
                node.children[d] = c
            c.last_seq = self.seq
            node = c

    # PAPER.md:61 "a node is cached when its KV blocks are predicted resident"; :19 "by recency of service"
    def is_cached(self, node) -> bool:
        return self.seq - node.last_seq < self.H

    # Algorithm 1
    def order(self, D):
        if len(set(D)) != len(D):
            raise ValueError("D is a set (PAPER.md:61): duplicate document id")
        O, R, node = [], list(D), self.root          # line 1
        self.probes = 0
        while R:                                     # line 2
            found = False                            # line 3
            for d in R:                              # line 4 (retrieval rank)
                self.probes += 1
                c = node.children.get(d)             # line 5
                if c is not None and self.is_cached(c):   # line 6
                    O.append(d)                      # line 7
                    R.remove(d)
                    node = c                         # line 8
                    found = True
                    break
            if not found:                            # line 11
                O.extend(R)                          # line 12: remaining R in retrieval-rank order
                break                                # line 13
        depth = self.ell(O)
        return O, depth                              # line 16

    # l(O,T): largest m with root->O[0]->...->O[m-1] present and every node on it cached
    def ell(self, O) -> int:
        node, m = self.root, 0
        for d in O:
            c = node.children.get(d)
            if c is None or not self.is_cached(c):
                break
            node, m = c, m + 1
        return m

    # exhaustive oracle ordering: k! candidate orders; tail keeps retrieval rank (:104).
    # Tie-break: first maximiser in lexicographic order of retrieval-rank indices.
    def brute_force_permutations(self, D):
        best, best_l = list(D), -1
        for perm in permutations(range(len(D))):
            O = [D[i] for i in perm]
            l = self.ell(O)
            tail = perm[l:]
            if list(tail) != sorted(tail):           # documents past the reused prefix keep retrieval rank
                continue
            if l > best_l:
                best, best_l = O, l
        return best, best_l

    # same optimum by DFS over cached trie children restricted to D (usable for k = 10, 20)
    def brute_force_dfs(self, D):
        Dset = list(D)

        def dfs(node, remaining):
            best = 0
            for d in remaining:
                c = node.children.get(d)
                if c is not None and self.is_cached(c):
                    best = max(best, 1 + dfs(c, [x for x in remaining if x != d]))
            return best

        return dfs(self.root, Dset)

    def count_nodes(self) -> int:
        def rec(n):
            return 1 + sum(rec(c) for c in n.children.values())
        return rec(self.root) - 1

    def prune(self):
        """Drop nodes outside the recency window (result-invariant; PAPER.md:108 O(Hk) space)."""
        def rec(n):
            for d in [d for d, c in n.children.items() if not self.is_cached(c)]:
                del n.children[d]
            for c in n.children.values():
                rec(c)
        rec(self.root)
