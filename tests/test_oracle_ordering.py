"""Pins for oracle/ordering.py against what the paper fixes (no GPU)."""
import itertools
import random

import pytest

from conftest import golden
from oracle.ordering import KnowledgeTree


def test_figure2_worked_example():
    # PAPER.md:123
    g = golden("figure2_ordering.txt")
    T = KnowledgeTree(recency_window=8)
    T.observe(["A", "E"])                 # another branch (gray)
    T.observe(["Z", "B", "C"])            # another branch
    T.observe(g["cached_path"].split())   # the cached path root->A->B->C->D
    O, depth = T.order(g["candidates"].split())
    assert O == g["expected_order"].split()
    assert depth == int(g["expected_prefix_docs"])


def test_figure2_evicted_nodes_are_not_followed():
    # "gray nodes are evicted": an old path falls out of the recency window and must not be used
    T = KnowledgeTree(recency_window=2)
    T.observe(["F", "A"])                 # will be stale
    T.observe(["A", "B", "C", "D"])
    T.observe(["A", "B", "C", "D"])
    T.observe(["A", "B"])
    O, depth = T.order(["A", "B", "C", "F", "D"])
    assert (O, depth) == (["A", "B", "C", "D", "F"], 4)


def test_figure1_alignment():
    # PAPER.md:37
    g = golden("figure1_alignment.txt")
    T = KnowledgeTree(recency_window=4)
    T.observe(g["request1_order"].split())
    D2 = g["request2_retrieval"].split()
    assert T.ell(D2) == int(g["retrieval_order_prefix_docs"])
    O, depth = T.order(D2)
    assert depth == int(g["reordered_prefix_docs"])
    assert O == ["d1", "d2", "d3", "d4", "x9"]


def test_fallback_empty_trie_is_identity():
    # PAPER.md:143 "an empty trie or a missing cached continuation returns retrieval order"
    T = KnowledgeTree(4)
    assert T.order([5, 3, 9]) == ([5, 3, 9], 0)
    T.observe([1, 2])
    assert T.order([5, 3, 9]) == ([5, 3, 9], 0)
    assert T.order([]) == ([], 0)


def test_recency_window_hand_worked():
    # H=2, insert [A,B], [C], [D] => A no longer cached => order([B,A]) = [B,A]
    T = KnowledgeTree(2)
    T.observe(["A", "B"]); T.observe(["C"]); T.observe(["D"])
    assert T.order(["B", "A"]) == (["B", "A"], 0)
    T2 = KnowledgeTree(3)
    T2.observe(["A", "B"]); T2.observe(["C"]); T2.observe(["D"])
    assert T2.order(["B", "A"]) == (["A", "B"], 2)


def test_duplicate_ids_rejected():
    with pytest.raises(ValueError):
        KnowledgeTree(2).order([1, 1])


def _random_tree(rng, n_docs, k, n_obs, H):
    T = KnowledgeTree(H)
    for _ in range(n_obs):
        T.observe(rng.sample(range(n_docs), rng.randint(1, k)))
    return T


def _ambiguous(T, D):
    """does the greedy walk visit a node with >= 2 cached children still in R?"""
    node, R = T.root, list(D)
    while True:
        cand = [d for d in R if d in node.children and T.is_cached(node.children[d])]
        if len(cand) >= 2:
            return True
        if not cand:
            return False
        R.remove(cand[0]); node = node.children[cand[0]]


@pytest.mark.parametrize("seed", range(40))
def test_properties_and_bruteforce(seed):
    rng = random.Random(seed)
    k = rng.randint(1, 6)
    n_docs = rng.randint(k, 9)
    T = _random_tree(rng, n_docs, k, rng.randint(0, 12), rng.randint(1, 6))
    D = rng.sample(range(n_docs), k)
    O, depth = T.order(D)
    # permutation property
    assert sorted(O) == sorted(D)
    # tail keeps retrieval rank
    tail_idx = [D.index(d) for d in O[depth:]]
    assert tail_idx == sorted(tail_idx)
    # probe bound k(k+1)/2
    assert T.probes <= k * (k + 1) // 2
    # depth is l(O,T)
    assert depth == T.ell(O)
    # brute force: k! permutations == trie DFS; greedy <= optimum, == when no branch ambiguity
    bo, bl = T.brute_force_permutations(D)
    assert bl == T.brute_force_dfs(D)
    assert sorted(bo) == sorted(D) and T.ell(bo) == bl
    assert depth <= bl
    if not _ambiguous(T, D):
        assert depth == bl
    # independent restatement of the objective: max over ALL k! orders of the cached-path depth
    def ell_plain(o):
        node, m = T.root, 0
        for d in o:
            if d in node.children and T.seq - node.children[d].last_seq < T.H:
                node = node.children[d]; m += 1
            else:
                break
        return m
    assert bl == max(ell_plain(p) for p in itertools.permutations(D))


def test_oracle_search_size_k5():
    # PAPER.md:147 "5! = 120 candidate orders per request"
    assert len(list(itertools.permutations(range(5)))) == 120


def test_branch_ambiguity_greedy_can_be_suboptimal():
    # sub-optimality only with two cached children retrievable at one node
    T = KnowledgeTree(8)
    T.observe(["A", "B", "C"]); T.observe(["A", "C"])
    O, depth = T.order(["C", "B", "A"])      # at node A both B and C are cached; rank scan takes C first
    assert (O, depth) == (["A", "C", "B"], 2)
    assert T.brute_force_permutations(["C", "B", "A"])[1] == 3


def test_tree_space_bound_after_prune():
    # PAPER.md:108 O(Hk) space
    rng = random.Random(1)
    H, k = 5, 4
    T = KnowledgeTree(H)
    for _ in range(200):
        T.observe(rng.sample(range(50), k))
        T.prune()
        assert T.count_nodes() <= H * k
    before = T.order(list(range(10)))
    T.prune()
    assert T.order(list(range(10))) == before
