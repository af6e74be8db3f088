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

Cache-state feedback ("when the trie predicts a long reusable prefix but
[the request behaves like] a cold request, the supposed cached path is probably gone, so we mark it stale and stop
relying on it"; "When serving engines expose direct cache-state signals, the middleware can use them to
align the knowledge tree with actual residency").  The paper gives no data structure for "stale"; the reading
(DESIGN.md §2):
  * every node carries stale_epoch (0 = never marked).  mark_stale(O, a) sets stale_epoch = seq on the node reached by
    O[0..a] (depth a + 1): the prefix O[0..a-1] was resident, the prefix O[0..a] was not.
  * blocks are chained to their prefix and released deepest-first, so when a node's blocks are gone the blocks of
    everything below it are gone too: a node is USABLE iff it is cached by recency AND it was served after the latest
    stale mark on itself or on any node above it on the walk (last_seq > max stale_epoch along the path).
    observe() re-stamps the served path, which makes exactly that path usable again.
  * feedback(O, predicted, actual): the engine's signal replaces the paper's TTFT heuristic — actual = number of
    leading documents of O the prefix cache really matched; if predicted > actual, mark_stale(O, actual).
  * order_resident(D, resident): Algorithm 1 whose line 6 additionally asks the engine (a peek on the real block
    index) whether the prefix O + [d] is resident; a recency-cached child that is not resident is marked stale and the
    scan of R goes on.
With no stale mark anywhere order() and ell() are exactly the functions pinned above.
Pins: tests/test_oracle_residency.py (hand-worked epochs; rows req5a_resident / req5a_after_feedback of the SURVEY.md
§8(c7) block-table scenario; predicted == actual for order_resident; never more hits than the exhaustive arm).
"""
from __future__ import annotations

from itertools import permutations


class Node:
    __slots__ = ("doc", "children", "last_seq", "stale_epoch")

    def __init__(self, doc):
        self.doc = doc
        self.children = {}
        self.last_seq = 0
        self.stale_epoch = 0


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

    # usable: cached by recency and served after the latest stale mark on itself or above it (floor) — see the header
    def usable(self, node, floor: int) -> bool:
        return self.is_cached(node) and node.last_seq > max(floor, node.stale_epoch)

    # Algorithm 1.  resident (optional, NEXT-1): callable(list of documents) -> bool, the engine's answer
    # to "are all full blocks of this document prefix resident"; None = the paper's minimal path (trie only).
    def order(self, D, resident=None):
        if len(set(D)) != len(D):
            raise ValueError("D is a set (PAPER.md:61): duplicate document id")
        O, R, node, floor = [], list(D), self.root, 0   # line 1
        self.probes = 0
        while R:                                     # line 2
            found = False                            # line 3
            for d in R:                              # line 4 (retrieval rank)
                self.probes += 1
                c = node.children.get(d)             # line 5
                if c is not None and self.usable(c, floor):   # line 6
                    if resident is not None and not resident(O + [d]):
                        c.stale_epoch = self.seq     # predicted resident, really gone: stop relying on it
                        continue
                    O.append(d)                      # line 7
                    R.remove(d)
                    node = c                         # line 8
                    floor = max(floor, c.stale_epoch)
                    found = True
                    break
            if not found:                            # line 11
                O.extend(R)                          # line 12: remaining R in retrieval-rank order
                break                                # line 13
        depth = self.ell(O)
        return O, depth                              # line 16

    def order_resident(self, D, resident):
        return self.order(D, resident)

    # l(O,T): largest m with root->O[0]->...->O[m-1] present and every node on it cached (and usable)
    def ell(self, O) -> int:
        node, m, floor = self.root, 0, 0
        for d in O:
            c = node.children.get(d)
            if c is None or not self.usable(c, floor):
                break
            node, m, floor = c, m + 1, max(floor, c.stale_epoch)
        return m

    # NEXT-1: the prefix O[0..a-1] was resident, O[0..a] was not -> the node at depth a+1 is marked stale
    def mark_stale(self, O, a: int):
        node = self.root
        for d in O[: a + 1]:
            node = node.children.get(d)
            if node is None:
                return
        node.stale_epoch = self.seq

    def feedback(self, O, predicted: int, actual: int):
        if predicted > actual:
            self.mark_stale(O, actual)

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

        def dfs(node, remaining, floor):
            best = 0
            for d in remaining:
                c = node.children.get(d)
                if c is not None and self.usable(c, floor):
                    best = max(best, 1 + dfs(c, [x for x in remaining if x != d], max(floor, c.stale_epoch)))
            return best

        return dfs(self.root, Dset, 0)

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
