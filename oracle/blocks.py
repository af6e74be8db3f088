"""ORACLE (test infrastructure, not product): chained block hashing and the paged-KV block manager model.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
Shares no code with paper_2606_19667_b200/.

PAPER.md:33 "each block is hashed together with its prefix history, so reuse is inherently prefix-sensitive.
Once an early block differs, later blocks no longer line up with the cached chain"; PAPER.md:39 block size 16;
PAPER.md:129 residency is controlled "through internal block eviction".

Plain definition used for the match: m = the largest number of leading FULL 16-token blocks
of the prompt such that a resident registered block exists whose ENTIRE token prefix (position 0 through the
end of that block) is identical, capped at floor((n-1)/16).  This model matches by comparing token prefixes
directly (a dict keyed by the raw bytes of the whole prefix: equality is byte equality) — never by hash.
The hash chain is computed separately so the chain values can be compared bit-exactly.

Readings where the paper is silent: FNV-1a-64 over parent(8 LE bytes) ‖ 16 tokens
(4 LE bytes each); LRU free list, pop head, release in reverse block order to the tail; eager registration.
Pins: tests/test_oracle_blocks.py (FNV-1a textbook vectors, hand-worked chain values, prefix sensitivity,
the hand-worked block-table scenario of SURVEY.md §8(c7), invariants under random op sequences); extend():
tests/test_oracle_extend.py (hand-worked tables, growth == one-shot lookup in tables and registrations, invariants).
"""
from __future__ import annotations

from collections import OrderedDict

import numpy as np

BS = 16
FNV_OFFSET = 0xCBF29CE484222325
FNV_PRIME = 0x100000001B3
MASK64 = (1 << 64) - 1


def fnv1a64(data: bytes) -> int:
    h = FNV_OFFSET
    for b in data:
        h ^= b
        h = (h * FNV_PRIME) & MASK64
    return h


def chain_hashes(tokens, salt: int = 0):
    """h_i = FNV1a64( LE64(h_{i-1}) ‖ LE32(tokens[16i]) … LE32(tokens[16i+15]) ), h_{-1} = salt; i < floor(n/16)."""
    tokens = np.ascontiguousarray(tokens, dtype="<i4")
    out, parent = [], salt & MASK64
    for i in range(len(tokens) // BS):
        msg = parent.to_bytes(8, "little") + tokens[i * BS:(i + 1) * BS].tobytes()
        parent = fnv1a64(msg)
        out.append(parent)
    return out


class NoSpace(Exception):
    pass


class BlockManager:
    """Exact policy of SURVEY.md §8(c3), with prefix identity instead of hashes."""

    def __init__(self, num_blocks: int, eager_register: bool = True):
        self.NB = num_blocks
        self.eager = eager_register
        self.ref = [0] * num_blocks
        self.key_of = [None] * num_blocks          # registered prefix bytes of the block, or None
        self.index = {}                            # prefix bytes -> block id
        self.free = OrderedDict((b, None) for b in range(num_blocks))   # head = first key
        self.reqs = {}
        self.tokens_of = {}                        # request -> its token sequence so far (extend() appends to it)
        self.next_req = 1
        self.evictions = 0
        self.hit_blocks = 0
        self.miss_blocks = 0

    def _prefix_keys(self, tokens, upto_blocks):
        raw = np.ascontiguousarray(tokens, dtype="<i4").tobytes()
        return [raw[: (i + 1) * BS * 4] for i in range(upto_blocks)]

    def match(self, tokens):
        """peek: number of leading full blocks whose whole prefix is resident, capped at floor((n-1)/16)."""
        n = len(tokens)
        cap = (n - 1) // BS
        keys = self._prefix_keys(tokens, cap)
        m = 0
        while m < cap and keys[m] in self.index:
            m += 1
        return m

    def resident_prefix(self, tokens) -> bool:
        """NEXT-1 peek: are ALL full blocks of this token sequence resident (no cap: the sequence is a document prefix
        of a longer prompt).  Plain definition again: every leading full block's whole prefix is registered."""
        return all(k in self.index for k in self._prefix_keys(tokens, len(tokens) // BS))

    def lookup(self, tokens):
        n = len(tokens)
        if n <= 0:
            raise ValueError("n <= 0")
        nblk = -(-n // BS)
        nfull = n // BS
        keys = self._prefix_keys(tokens, nfull)
        cap = (n - 1) // BS
        m = 0
        while m < cap and keys[m] in self.index:                                   # (1)
            m += 1
        matched = [self.index[keys[i]] for i in range(m)]
        need = nblk - m                                                            # (2)
        available = len(self.free) - sum(1 for b in matched if self.ref[b] == 0)
        if need > available:
            raise NoSpace()
        table = []
        for b in matched:                                                          # (3)
            if self.ref[b] == 0:
                del self.free[b]
            self.ref[b] += 1
            table.append(b)
        for i in range(m, nblk):                                                   # (4)
            b, _ = self.free.popitem(last=False)
            if self.key_of[b] is not None:
                del self.index[self.key_of[b]]
                self.key_of[b] = None
                self.evictions += 1
            self.ref[b] = 1
            table.append(b)
        req = self.next_req
        self.next_req += 1
        self.reqs[req] = (table, keys, m, nfull)
        self.tokens_of[req] = np.ascontiguousarray(tokens, dtype="<i4").copy()
        if self.eager:
            self._register(table, keys, m, nfull)                                  # (5)
        self.hit_blocks += m
        self.miss_blocks += nblk - m
        return req, table, m * BS

    def _register(self, table, keys, m, nfull):
        for i in range(m, nfull):
            if keys[i] not in self.index:
                self.index[keys[i]] = table[i]
                self.key_of[table[i]] = keys[i]

    def extend(self, req, new_tokens):
        """NEXT-4 (PAPER.md:253-283 continuous batching / decode): the live request grows by new_tokens
        (a chunk of a chunked prefill, or generated tokens).  Blocks for the longer sequence are popped from the LRU head
        exactly like in lookup step (4) (NoSpace leaves everything unchanged); with eager registration every block the new
        tokens COMPLETE is registered under its whole token prefix (step (5)) — the formerly partial last block included.
        Returns the request's block table."""
        table, keys, m, nfull = self.reqs[req]
        tokens = np.concatenate([self.tokens_of[req], np.ascontiguousarray(new_tokens, dtype="<i4")])
        n = len(tokens)
        need = -(-n // BS) - len(table)
        if need > len(self.free):
            raise NoSpace()
        table = list(table)
        for _ in range(need):
            b, _ = self.free.popitem(last=False)
            if self.key_of[b] is not None:
                del self.index[self.key_of[b]]
                self.key_of[b] = None
                self.evictions += 1
            self.ref[b] = 1
            table.append(b)
        new_nfull = n // BS
        keys = self._prefix_keys(tokens, new_nfull)
        self.reqs[req] = (table, keys, m, new_nfull)
        self.tokens_of[req] = tokens
        if self.eager:
            self._register(table, keys, nfull, new_nfull)
        self.miss_blocks += need
        return table

    def release(self, req):
        self.tokens_of.pop(req, None)
        table, keys, m, nfull = self.reqs.pop(req)
        if not self.eager:
            self._register(table, keys, m, nfull)
        for i in range(len(table) - 1, -1, -1):        # reverse order: deepest blocks evicted first
            b = table[i]
            self.ref[b] -= 1
            if self.ref[b] == 0:
                self.free[b] = None                    # tail

    def free_list(self):
        return list(self.free.keys())

    def check_invariants(self):
        live = [0] * self.NB
        for table, *_ in self.reqs.values():
            assert len(set(table)) == len(table), "block id twice in one table"
            for b in table:
                live[b] += 1
        assert live == self.ref, "refcounts inconsistent with live requests"
        for b in range(self.NB):
            assert (self.ref[b] == 0) == (b in self.free), "block neither pinned nor exactly once free"
        assert len(self.index) == sum(1 for k in self.key_of if k is not None)
        for k, b in self.index.items():
            assert self.key_of[b] == k, "index <-> has_hash bijection broken"


def matched_docs(doc_ends, n_cached: int, n_tokens: int) -> int:
    """Leading documents of a prompt that count as served from the cache (the `actual` of the feedback rule; SURVEY.md 8(f)
    NEXT-1, "the trie predicts a long reusable prefix ... the supposed cached path is probably gone",
    :314).  Reading: doc_ends[j] is the prompt position just past the segment of the j-th document; a document
    counts when every FULL 16-token block up to its end was matched — the block it shares with what follows cannot match
    unless the next segment matches too — and "matched" is measured against what a lookup can ever return: it never
    matches the block that holds the last prompt token (c3: m <= floor((n-1)/16)), so a document that ends in that block is
    not punished for it (a prompt of block-aligned documents and no query would otherwise lose its last document every
    time).  Plain count, no state.  Pins: tests/test_oracle_residency.py (hand-worked ragged segment ends; the
    no-query case)."""
    cap = (n_tokens - 1) // BS * BS
    m = 0
    for end in doc_ends:
        if min(end // BS * BS, cap) > n_cached:
            break
        m += 1
    return m
