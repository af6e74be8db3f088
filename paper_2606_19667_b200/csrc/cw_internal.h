// Internal declarations shared by the host state (host.cpp), the kernels (*.cu) and the C ABI (api.cu).
// Product code: nothing here is shared with oracle/.
#pragma once
#include <algorithm>
#include <cstdint>
#include <functional>
#include <string>
#include <unordered_map>
#include <vector>

#include "cacheweaver.h"

namespace cw {

// ---- knowledge tree (§3.2) -------------------------------------------------------------------
// Flat representation: one hash map keyed by (parent node id, doc id).  A path stamps every node on it with
// the same seq, so last_seq(child) <= last_seq(parent): a stale parent has only stale children and nodes can
// be pruned individually (result-invariant, "bounded by the recency window").
struct TrieKey {
    uint64_t parent;
    int64_t doc;
    bool operator==(const TrieKey& o) const { return parent == o.parent && doc == o.doc; }
};
struct TrieKeyHash {
    size_t operator()(const TrieKey& k) const {
        uint64_t x = k.parent * 0x9E3779B97F4A7C15ull ^ (uint64_t)k.doc * 0xC2B2AE3D27D4EB4Full;
        x ^= x >> 29;
        return (size_t)(x * 0xBF58476D1CE4E5B9ull);
    }
};
struct TrieNode {
    uint64_t id;
    int64_t last_seq;
    int64_t stale_epoch;    // seq at which the engine reported this prefix as not resident (0 = never); DESIGN.md §2 NEXT-1
};

class KnowledgeTree {
  public:
    explicit KnowledgeTree(int64_t window) : H_(window) {}
    // Algorithm 1.  Returns depth l(O,T).  `resident` (optional, NEXT-1): asked for every recency-cached
    // child whether the document prefix O[0..m-1] + d is really resident (m = documents placed so far); a child that is
    // not is marked stale and the scan goes on.
    int order(const int64_t* D, int k, int64_t* O, const std::function<bool(const int64_t* O, int m, int64_t d)>* resident = nullptr);
    int predict(const int64_t* O, int k) const;
    void observe(const int64_t* O, int k);
    // the prefix O[0..a-1] was resident, O[0..a] was not: the node at depth a+1 is marked stale (no-op if it does not exist)
    void mark_stale(const int64_t* O, int k, int a);
    int64_t nodes() const { return (int64_t)map_.size(); }
    int64_t probes() const { return probes_; }
    int64_t seq() const { return seq_; }
    int64_t stale_marks() const { return marks_; }

  private:
    const TrieNode* child(uint64_t parent, int64_t doc) const;
    bool cached(const TrieNode* n) const { return seq_ - n->last_seq < H_; }
    // usable: cached by recency and served after the latest stale mark on itself or above it on the walk (floor)
    bool usable(const TrieNode* n, int64_t floor) const { return cached(n) && n->last_seq > std::max(floor, n->stale_epoch); }
    void prune();
    std::unordered_map<TrieKey, TrieNode, TrieKeyHash> map_;
    int64_t H_;
    int64_t seq_ = 0;
    int64_t last_prune_ = 0;
    uint64_t next_id_ = 1;  // 0 = root
    int64_t probes_ = 0;
    int64_t marks_ = 0;     // nodes marked stale so far
};

// ---- paged KV block manager (reading c3) --------------------------------
struct Request {
    std::vector<int32_t> table;
    std::vector<uint64_t> chain;
    std::vector<uint64_t> verify;  // second, secretly salted chain over the same blocks (collision check, see BlockManager)
    int32_t m;      // matched (cached) blocks
    int32_t n;      // sequence length in tokens (prompt + what cw_extend appended)
    int32_t n_done; // tokens whose K/V are (being) written to the pool: m*16 at lookup, advanced by cw_prefill_requests
    int32_t tail[CW_BLOCK_SIZE];   // tokens of the trailing partial block (n % 16 of them): cw_extend completes it
};

class BlockManager {
  public:
    BlockManager(int32_t num_blocks, bool eager, uint64_t salt, int32_t key_bits = 64);
    void chain(const int32_t* tokens, int32_t n, std::vector<uint64_t>& out) const;
    // Both chains of a token sequence: `h` is the FNV-1a-64 chain that keys the prefix index (reading c2), `v` an
    // independent 64-bit chain (multiply-xorshift mixing) salted with a per-context random secret.  An index entry only
    // matches when BOTH agree, so serving another prompt's KV needs a simultaneous collision of two unrelated functions, one of
    // them keyed with a value the prompt author cannot know; a colliding newcomer is simply never cached.
    void chains(const int32_t* tokens, int32_t n, std::vector<uint64_t>& h, std::vector<uint64_t>& v) const;
    int32_t match(const std::vector<uint64_t>& h, const std::vector<uint64_t>& v, int32_t n) const;
    // NEXT-1 peek, incremental over a growing document prefix: state = (hash of the last full block, tokens of the
    // pending partial block).  extend() appends tokens; it returns false and leaves the state unchanged unless every
    // full block completed by them is resident.
    struct Probe {
        uint64_t parent, vparent;
        int32_t pending[CW_BLOCK_SIZE];
        int32_t n_pending;
    };
    Probe probe_begin() const { return Probe{salt_, vsalt_, {0}, 0}; }
    bool probe_extend(Probe& p, const int32_t* tokens, int32_t n) const;
    // returns CW_OK / CW_ERR_NO_SPACE
    int lookup(const int32_t* tokens, int32_t n, int64_t* req, int32_t* table, int32_t* n_cached);
    int release(int64_t req);
    // NEXT-4: the live request grows by n_new tokens (chunked prefill / generated tokens).  CW_ERR_NO_SPACE: unchanged.
    int extend(int64_t req, const int32_t* tokens, int32_t n_new, int32_t* table_out, int32_t cap, int32_t* n_blocks);
    Request* find_mut(int64_t req) {
        auto it = reqs_.find(req);
        return it == reqs_.end() ? nullptr : &it->second;
    }
    const Request* find(int64_t req) const {
        auto it = reqs_.find(req);
        return it == reqs_.end() ? nullptr : &it->second;
    }
    int32_t free_list(int32_t* out, int32_t cap) const;
    int64_t requests = 0, hit_blocks = 0, miss_blocks = 0, evictions = 0;
    int64_t prompt_tokens = 0, suffix_tokens = 0, attn_pairs = 0;   // attn_pairs: (row, key) pairs the suffixes attend to
    int32_t free_count() const { return free_count_; }

  private:
    void unlink(int32_t b);
    void push_tail(int32_t b);
    void reg(const Request& r, int32_t nfull);
    int32_t find_block(uint64_t h, uint64_t v) const;   // block registered under (h, v), or -1
    int32_t NB_;
    bool eager_;
    uint64_t salt_, vsalt_, key_mask_;
    uint64_t key(uint64_t h) const { return h & key_mask_; }
    std::vector<int32_t> ref_, prev_, next_;   // list nodes 0..NB-1, sentinel = NB
    std::vector<uint8_t> has_hash_;
    std::vector<uint64_t> hash_, verify_;
    std::unordered_map<uint64_t, int32_t> index_;
    std::unordered_map<int64_t, Request> reqs_;
    int64_t next_req_ = 1;
    int32_t free_count_;
};

}  // namespace cw

struct cw_ctx {
    cw_config cfg;
    cw::KnowledgeTree* tree;
    cw::BlockManager* blocks;
    std::string last_error;
    bool host_only;
    int num_sms;
    // comparison arms (cw_order_arm): index of the last cw_observe call whose order contained the document
    std::unordered_map<int64_t, int64_t> last_served;
    // predicted-vs-actual prefix statistics, accumulated by cw_admit_batch / cw_feedback
    int64_t pred_docs = 0, actual_docs = 0, over_pred_docs = 0;
    // cw_prefill_host pipeline: copy streams and per-chunk events (created on first use, destroyed with the context)
    void* copy_in_stream = nullptr;
    void* copy_out_stream = nullptr;
    std::vector<void*> events;
    // cw_prefill_requests: ring of pinned host slots the wave descriptors are staged in (grown on demand); the event marks
    // the H2D copy that last read the slot
    struct Staging {
        void* host = nullptr;
        size_t cap = 0;
        void* event = nullptr;
    };
    // cw_prefill_requests: side stream the schedule kernel runs on beside cw_append_kv, and its fork / join events
    void* sched_stream = nullptr;
    void* sched_fork = nullptr;
    void* sched_join = nullptr;
    static constexpr int kStagingSlots = 4;
    Staging staging[kStagingSlots];
    int staging_next = 0;
};

// kernel launchers (defined in the .cu files); return cudaError_t as int
namespace cw {
int launch_append_kv(const cw_config& cfg, const void* q, const void* k, const void* v, void* q_roped,
                     const int32_t* cu, const int32_t* ncached, const int32_t* tables, int32_t max_blocks,
                     int32_t B, int32_t T, int num_sms, void* stream);
int launch_gather_kv(const cw_config& cfg, const int32_t* table, int32_t n, void* k_out, void* v_out, int num_sms, void* stream);
// attention: the item list (8 ints per item + an 8-int header) is built on the device by a schedule kernel launched in
// front of the attention kernel; attn_work_ints is the scratch size for a batch of B requests / T suffix rows
int64_t attn_max_items(const cw_config& cfg, int32_t B, int32_t T);
int64_t attn_work_ints(const cw_config& cfg, int32_t B, int32_t T);
int launch_prefill_attn(const cw_config& cfg, const void* q_roped, void* out, const int32_t* d_cu, const int32_t* d_nc,
                        const int32_t* d_kv_len, const int32_t* tables, int32_t max_blocks, int32_t B, int32_t T,
                        int32_t max_q_len, int32_t max_kv_len, int32_t* d_work, int num_sms, void* stream);
// its two launches separately: descriptors -> item list (needs no q_roped / KV), then the attention kernel over that list
int launch_attn_schedule(const cw_config& cfg, const int32_t* d_cu, const int32_t* d_nc, const int32_t* d_kv_len,
                         const int32_t* tables, int32_t max_blocks, int32_t B, int32_t T, int32_t max_q_len,
                         int32_t max_kv_len, int32_t* d_work, void* stream);
int launch_attn_run(const cw_config& cfg, const void* q_roped, void* out, const int32_t* tables, int32_t max_blocks,
                    int32_t B, int32_t T, int32_t* d_work, int num_sms, void* stream);
// the same with the work list in the library's own static device array (no caller scratch; at most CW_STATIC_WORK_INTS ints);
// d_status (device int32[4], may be null) receives the work header
int launch_prefill_attn_static(const cw_config& cfg, const void* q_roped, void* out, const int32_t* d_cu,
                               const int32_t* d_nc, const int32_t* d_kv_len, const int32_t* tables, int32_t max_blocks,
                               int32_t B, int32_t T, int32_t max_q_len, int32_t max_kv_len, int32_t* d_status, int num_sms,
                               void* stream);
}  // namespace cw
