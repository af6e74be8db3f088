// Host state of the prefix-cached prefill path: knowledge tree + greedy ordering and the
// paged-KV block manager with chained block hashes and LRU eviction (DESIGN.md c2, c3).
// Product code; shares nothing with oracle/.
#include "cw_internal.h"

#include <algorithm>
#include <climits>
#include <cstring>
#include <random>

namespace cw {

// ------------------------------------------------------------------------------------------------ trie ----
const TrieNode* KnowledgeTree::child(uint64_t parent, int64_t doc) const {
    auto it = map_.find(TrieKey{parent, doc});
    return it == map_.end() ? nullptr : &it->second;
}

// Algorithm 1.  R is kept as an index list in retrieval rank; "for each d in R" scans it in that order and takes
// the first cached child (DESIGN.md reading: D is given in retrieval rank).
int KnowledgeTree::order(const int64_t* D, int k, int64_t* O,
                         const std::function<bool(const int64_t* O, int m, int64_t d)>* resident) {
    std::vector<int64_t> R(D, D + k);                 // line 1: O <- [], R <- D, node <- root
    uint64_t node = 0;
    int64_t floor = 0;
    int n_out = 0;
    probes_ = 0;
    while (!R.empty()) {                              // line 2
        bool found = false;                           // line 3
        for (size_t i = 0; i < R.size(); ++i) {       // line 4
            ++probes_;
            auto it = map_.find(TrieKey{node, R[i]}); // line 5
            if (it == map_.end() || !usable(&it->second, floor)) continue;   // line 6
            if (resident && !(*resident)(O, n_out, R[i])) {
                it->second.stale_epoch = seq_;        // predicted resident, really gone: stop relying on it
                ++marks_;
                continue;
            }
            O[n_out++] = R[i];                        // line 7: append d to O, remove d from R
            R.erase(R.begin() + (long)i);
            node = it->second.id;                     // line 8
            floor = std::max(floor, it->second.stale_epoch);
            found = true;
            break;
        }
        if (!found) {                                 // lines 11-13: remaining R in retrieval-rank order
            for (int64_t d : R) O[n_out++] = d;
            break;
        }
    }
    return predict(O, k);
}

int KnowledgeTree::predict(const int64_t* O, int k) const {
    uint64_t node = 0;
    int64_t floor = 0;
    int m = 0;
    for (; m < k; ++m) {
        const TrieNode* c = child(node, O[m]);
        if (!c || !usable(c, floor)) break;
        node = c->id;
        floor = std::max(floor, c->stale_epoch);
    }
    return m;
}

void KnowledgeTree::mark_stale(const int64_t* O, int k, int a) {
    if (a < 0 || a >= k) return;
    uint64_t node = 0;
    for (int i = 0; i <= a; ++i) {
        auto it = map_.find(TrieKey{node, O[i]});
        if (it == map_.end()) return;
        if (i == a) {
            it->second.stale_epoch = seq_;
            ++marks_;
        }
        node = it->second.id;
    }
}

void KnowledgeTree::observe(const int64_t* O, int k) {
    ++seq_;
    uint64_t node = 0;
    for (int i = 0; i < k; ++i) {
        TrieKey key{node, O[i]};
        auto it = map_.find(key);
        if (it == map_.end()) it = map_.emplace(key, TrieNode{next_id_++, seq_, 0}).first;
        it->second.last_seq = seq_;
        node = it->second.id;
    }
    if (seq_ - last_prune_ >= std::max<int64_t>(H_, 16)) prune();
}

void KnowledgeTree::prune() {
    last_prune_ = seq_;
    for (auto it = map_.begin(); it != map_.end();) {
        if (seq_ - it->second.last_seq >= H_) it = map_.erase(it);
        else ++it;
    }
}

// --------------------------------------------------------------------------------------- block manager ----
static inline uint64_t fnv1a_step(uint64_t h, uint8_t byte) { return (h ^ byte) * 0x100000001B3ull; }

BlockManager::BlockManager(int32_t num_blocks, bool eager, uint64_t salt, int32_t key_bits)
    : NB_(num_blocks), eager_(eager), salt_(salt), key_mask_(key_bits <= 0 || key_bits >= 64 ? ~0ull : (1ull << key_bits) - 1), ref_(num_blocks, 0), prev_(num_blocks + 1), next_(num_blocks + 1),
      has_hash_(num_blocks, 0), hash_(num_blocks, 0), verify_(num_blocks, 0), free_count_(num_blocks) {
    std::random_device rd;
    vsalt_ = ((uint64_t)rd() << 32) ^ (uint64_t)rd() ^ 0xA0761D6478BD642Full;
    // circular list with sentinel NB: head = next_[NB], tail = prev_[NB]; initial order 0,1,...,NB-1
    for (int32_t b = 0; b <= NB_; ++b) {
        next_[b] = (b + 1) % (NB_ + 1);
        prev_[b] = (b + NB_) % (NB_ + 1);
    }
    index_.reserve((size_t)num_blocks * 2);
}

void BlockManager::unlink(int32_t b) {
    next_[prev_[b]] = next_[b];
    prev_[next_[b]] = prev_[b];
    --free_count_;
}

void BlockManager::push_tail(int32_t b) {
    int32_t t = prev_[NB_];
    next_[t] = b; prev_[b] = t; next_[b] = NB_; prev_[NB_] = b;
    ++free_count_;
}

static inline uint64_t block_hash(uint64_t parent, const int32_t* tokens) {
    uint64_t h = 0xCBF29CE484222325ull;
    for (int b = 0; b < 8; ++b) h = fnv1a_step(h, (uint8_t)(parent >> (8 * b)));
    for (int t = 0; t < CW_BLOCK_SIZE; ++t) {
        uint32_t tok = (uint32_t)tokens[t];
        for (int b = 0; b < 4; ++b) h = fnv1a_step(h, (uint8_t)(tok >> (8 * b)));
    }
    return h;
}

// verification chain: multiply-xorshift mixing of the parent value and the 16 tokens (unrelated to FNV-1a)
static inline uint64_t verify_hash(uint64_t parent, const int32_t* tokens) {
    uint64_t x = parent ^ 0x9E3779B97F4A7C15ull;
    for (int t = 0; t < CW_BLOCK_SIZE; ++t) {
        x = (x ^ (uint32_t)tokens[t]) * 0xFF51AFD7ED558CCDull;
        x ^= x >> 32;
    }
    x *= 0xC4CEB9FE1A85EC53ull;
    return x ^ (x >> 29);
}

// h_i = FNV1a64(LE64(h_{i-1}) || LE32(tok[16i]) ... LE32(tok[16i+15])), h_{-1} = salt  (DESIGN.md c2)
void BlockManager::chain(const int32_t* tokens, int32_t n, std::vector<uint64_t>& out) const {
    int32_t nfull = n / CW_BLOCK_SIZE;
    out.resize((size_t)nfull);
    uint64_t parent = salt_;
    for (int32_t i = 0; i < nfull; ++i) out[(size_t)i] = parent = block_hash(parent, tokens + (size_t)i * CW_BLOCK_SIZE);
}

void BlockManager::chains(const int32_t* tokens, int32_t n, std::vector<uint64_t>& h, std::vector<uint64_t>& v) const {
    int32_t nfull = n / CW_BLOCK_SIZE;
    h.resize((size_t)nfull);
    v.resize((size_t)nfull);
    uint64_t parent = salt_, vparent = vsalt_;
    for (int32_t i = 0; i < nfull; ++i) {
        h[(size_t)i] = parent = block_hash(parent, tokens + (size_t)i * CW_BLOCK_SIZE);
        v[(size_t)i] = vparent = verify_hash(vparent, tokens + (size_t)i * CW_BLOCK_SIZE);
    }
}

int32_t BlockManager::find_block(uint64_t h, uint64_t v) const {
    auto it = index_.find(key(h));
    return it != index_.end() && verify_[(size_t)it->second] == v ? it->second : -1;
}

bool BlockManager::probe_extend(Probe& p, const int32_t* tokens, int32_t n) const {
    Probe q = p;
    for (int32_t i = 0; i < n; ++i) {
        q.pending[q.n_pending++] = tokens[i];
        if (q.n_pending == CW_BLOCK_SIZE) {
            q.parent = block_hash(q.parent, q.pending);
            q.vparent = verify_hash(q.vparent, q.pending);
            if (find_block(q.parent, q.vparent) < 0) return false;
            q.n_pending = 0;
        }
    }
    p = q;
    return true;
}

int32_t BlockManager::match(const std::vector<uint64_t>& ch, const std::vector<uint64_t>& vc, int32_t n) const {
    int32_t cap = (n - 1) / CW_BLOCK_SIZE, m = 0;
    while (m < cap && find_block(ch[(size_t)m], vc[(size_t)m]) >= 0) ++m;
    return m;
}

void BlockManager::reg(const Request& r, int32_t nfull) {
    for (int32_t i = r.m; i < nfull; ++i) {
        auto ins = index_.emplace(key(r.chain[(size_t)i]), r.table[(size_t)i]);
        if (ins.second) {          // else: the same content is registered already, or a colliding block is (never cached)
            has_hash_[(size_t)r.table[(size_t)i]] = 1;
            hash_[(size_t)r.table[(size_t)i]] = key(r.chain[(size_t)i]);
            verify_[(size_t)r.table[(size_t)i]] = r.verify[(size_t)i];
        }
    }
}

int BlockManager::lookup(const int32_t* tokens, int32_t n, int64_t* req, int32_t* table, int32_t* n_cached) {
    Request r;
    chains(tokens, n, r.chain, r.verify);
    int32_t nblk = (n + CW_BLOCK_SIZE - 1) / CW_BLOCK_SIZE, nfull = n / CW_BLOCK_SIZE;
    r.n = n;
    std::memcpy(r.tail, tokens + (size_t)nfull * CW_BLOCK_SIZE, sizeof(int32_t) * (size_t)(n - nfull * CW_BLOCK_SIZE));
    r.m = match(r.chain, r.verify, n);                                          // (1)
    r.n_done = r.m * CW_BLOCK_SIZE;
    r.table.resize((size_t)nblk);
    int32_t matched_free = 0;
    for (int32_t i = 0; i < r.m; ++i) {
        int32_t b = index_.find(key(r.chain[(size_t)i]))->second;
        r.table[(size_t)i] = b;
        if (ref_[(size_t)b] == 0) ++matched_free;
    }
    if (nblk - r.m > free_count_ - matched_free) return CW_ERR_NO_SPACE;        // (2) nothing changed so far
    for (int32_t i = 0; i < r.m; ++i) {                                         // (3) pin the hit blocks
        int32_t b = r.table[(size_t)i];
        if (ref_[(size_t)b] == 0) unlink(b);
        ++ref_[(size_t)b];
    }
    for (int32_t i = r.m; i < nblk; ++i) {                                      // (4) pop head, evict its hash
        int32_t b = next_[NB_];
        unlink(b);
        if (has_hash_[(size_t)b]) {
            index_.erase(hash_[(size_t)b]);
            has_hash_[(size_t)b] = 0;
            ++evictions;
        }
        ref_[(size_t)b] = 1;
        r.table[(size_t)i] = b;
    }
    if (eager_) reg(r, nfull);                                                  // (5)
    std::memcpy(table, r.table.data(), sizeof(int32_t) * (size_t)nblk);
    *n_cached = r.m * CW_BLOCK_SIZE;
    *req = next_req_++;
    ++requests; hit_blocks += r.m; miss_blocks += nblk - r.m;
    const int64_t c = (int64_t)r.m * CW_BLOCK_SIZE;
    prompt_tokens += n; suffix_tokens += n - c; attn_pairs += (int64_t)n * (n + 1) / 2 - c * (c + 1) / 2;
    reqs_.emplace(*req, std::move(r));
    return CW_OK;
}

// NEXT-4: blocks for the longer sequence are popped from the LRU head like in lookup step (4); every
// block the new tokens complete is hashed (chained to the request's last full block) and, with eager registration,
// entered into the index (step (5)) — the formerly partial last block included.
int BlockManager::extend(int64_t req, const int32_t* tokens, int32_t n_new, int32_t* table_out, int32_t cap, int32_t* n_blocks) {
    auto it = reqs_.find(req);
    if (it == reqs_.end()) return CW_ERR_BAD_HANDLE;
    Request& r = it->second;
    const int64_t n_total = (int64_t)r.n + n_new;
    if (n_total > INT32_MAX) return CW_ERR_INVALID;
    const int32_t nblk = (int32_t)((n_total + CW_BLOCK_SIZE - 1) / CW_BLOCK_SIZE);
    const int32_t need = nblk - (int32_t)r.table.size();
    if (nblk > cap) return CW_ERR_INVALID;
    if (need > free_count_) return CW_ERR_NO_SPACE;
    for (int32_t i = 0; i < need; ++i) {
        int32_t b = next_[NB_];
        unlink(b);
        if (has_hash_[(size_t)b]) {
            index_.erase(hash_[(size_t)b]);
            has_hash_[(size_t)b] = 0;
            ++evictions;
        }
        ref_[(size_t)b] = 1;
        r.table.push_back(b);
    }
    const int32_t old_full = (int32_t)r.chain.size();
    int32_t n_tail = r.n - old_full * CW_BLOCK_SIZE;
    uint64_t parent = old_full ? r.chain.back() : salt_, vparent = old_full ? r.verify.back() : vsalt_;
    for (int32_t i = 0; i < n_new; ++i) {
        r.tail[n_tail++] = tokens[i];
        if (n_tail == CW_BLOCK_SIZE) {
            parent = block_hash(parent, r.tail);
            vparent = verify_hash(vparent, r.tail);
            r.chain.push_back(parent);
            r.verify.push_back(vparent);
            n_tail = 0;
        }
    }
    suffix_tokens += n_new; attn_pairs += n_total * (n_total + 1) / 2 - (int64_t)r.n * (r.n + 1) / 2;
    r.n = (int32_t)n_total;
    if (eager_) {
        const int32_t m_keep = r.m;
        r.m = old_full;                       // reg() registers blocks [m, nfull): only the newly completed ones
        reg(r, (int32_t)r.chain.size());
        r.m = m_keep;
    }
    miss_blocks += need;
    std::memcpy(table_out, r.table.data(), sizeof(int32_t) * r.table.size());
    *n_blocks = nblk;
    return CW_OK;
}

int BlockManager::release(int64_t req) {
    auto it = reqs_.find(req);
    if (it == reqs_.end()) return CW_ERR_BAD_HANDLE;
    Request& r = it->second;
    if (!eager_) reg(r, (int32_t)r.chain.size());     // lazy registration: everything the request completed, at release
    for (int32_t i = (int32_t)r.table.size() - 1; i >= 0; --i) {               // reverse: deepest evicted first
        int32_t b = r.table[(size_t)i];
        if (--ref_[(size_t)b] == 0) push_tail(b);
    }
    reqs_.erase(it);
    return CW_OK;
}

int32_t BlockManager::free_list(int32_t* out, int32_t cap) const {
    int32_t n = 0;
    for (int32_t b = next_[NB_]; b != NB_; b = next_[b]) {
        if (n < cap) out[n] = b;
        ++n;
    }
    return n;
}

}  // namespace cw
