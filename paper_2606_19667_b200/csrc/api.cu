// C ABI of libcacheweaver.so (include/cacheweaver.h): argument checking, error mapping and glue only.
#include <cuda_runtime.h>

#include <algorithm>
#include <climits>
#include <cmath>
#include <cstring>
#include <new>
#include <unordered_set>

#include "cw_internal.h"

namespace {

int fail(cw_ctx* ctx, int code, const char* msg) {
    if (ctx) ctx->last_error = msg;
    return code;
}
int cuda_fail(cw_ctx* ctx, int cuda_err, const char* where) {
    ctx->last_error = std::string(where) + ": " + cudaGetErrorString((cudaError_t)cuda_err);
    return CW_ERR_CUDA;
}
bool bad_cfg(const cw_config* c) {
    return !c || c->block_size != CW_BLOCK_SIZE || c->num_blocks <= 0 || c->num_q_heads <= 0 || c->num_kv_heads <= 0 ||
           c->num_q_heads % c->num_kv_heads != 0 || (c->head_dim != 64 && c->head_dim != 128) || c->recency_window <= 0 ||
           c->num_q_heads / c->num_kv_heads > 128;
}
inline int64_t align256(int64_t x) { return (x + 255) / 256 * 256; }
// Leading documents served from the cache (cacheweaver.h: cw_matched_docs).  end(j) = prompt position just past document j.
template <class EndFn>
int32_t count_matched_docs(EndFn end, int32_t k, int64_t n_cached, int64_t n_tokens) {
    const int64_t cap = (n_tokens - 1) / CW_BLOCK_SIZE * CW_BLOCK_SIZE;   // a lookup never matches the last token's block
    int32_t m = 0;
    while (m < k && std::min<int64_t>((int64_t)end(m) / CW_BLOCK_SIZE * CW_BLOCK_SIZE, cap) <= n_cached) ++m;
    return m;
}
bool bad_doc_ends(const int32_t* ends, int32_t k, int32_t n_cached, int32_t n_tokens) {
    if (k < 0 || (k > 0 && !ends) || n_tokens <= 0 || n_cached < 0 || n_cached > n_tokens) return true;
    for (int32_t j = 0; j < k; ++j)
        if (ends[j] <= 0 || ends[j] > n_tokens || (j > 0 && ends[j] < ends[j - 1])) return true;
    return false;
}

}  // namespace

extern "C" {

const char* cw_strerror(int code) {
    switch (code) {
        case CW_OK: return "ok";
        case CW_ERR_INVALID: return "invalid argument";
        case CW_ERR_NO_SPACE: return "not enough evictable KV blocks";
        case CW_ERR_BAD_HANDLE: return "unknown request handle";
        case CW_ERR_CUDA: return "CUDA error";
        default: return "unknown error code";
    }
}

const char* cw_last_error(cw_ctx* ctx) { return ctx ? ctx->last_error.c_str() : ""; }

int64_t cw_pool_bytes(const cw_config* c) {
    if (bad_cfg(c)) return CW_ERR_INVALID;
    return (int64_t)c->num_blocks * c->num_kv_heads * CW_BLOCK_SIZE * c->head_dim * 2;
}

int64_t cw_pool_offset(const cw_config* c, int32_t block, int32_t kv_head, int32_t t, int32_t d) {
    if (bad_cfg(c) || block < 0 || block >= c->num_blocks || kv_head < 0 || kv_head >= c->num_kv_heads || t < 0 ||
        t >= CW_BLOCK_SIZE || d < 0 || d >= c->head_dim)
        return CW_ERR_INVALID;
    const int64_t D = c->head_dim;
    return ((int64_t)block * c->num_kv_heads + kv_head) * (CW_BLOCK_SIZE * D) + (t / 8) * (8 * D) + (d / 64) * 512 +
           (t % 8) * 64 + ((((d % 64) / 8) ^ (t % 8)) * 8) + d % 8;
}

int64_t cw_q_roped_offset(const cw_config* c, int32_t s, int32_t tok, int32_t head, int32_t d) {
    if (bad_cfg(c) || s <= 0 || tok < 0 || tok >= s || head < 0 || head >= c->num_q_heads || d < 0 || d >= c->head_dim)
        return CW_ERR_INVALID;
    const int64_t D = c->head_dim, g = c->num_q_heads / c->num_kv_heads, tpt = 128 / g;
    const int64_t kvh = head / g, hh = head % g, t = tok / tpt, row = (tok % tpt) * g + hh;
    const int64_t rows_valid = std::min<int64_t>(tpt, s - t * tpt) * g;
    return kvh * s * g * D + t * (tpt * g) * D + (d / 64) * rows_valid * 64 + row * 64 + ((((d % 64) / 8) ^ (row % 8)) * 8) + d % 8;
}

int cw_create(const cw_config* cfg, cw_ctx** out) {
    if (!out || bad_cfg(cfg)) return CW_ERR_INVALID;
    const bool host_only = !cfg->k_pool && !cfg->v_pool && !cfg->rope_table;
    if (!host_only && (!cfg->k_pool || !cfg->v_pool || !cfg->rope_table || cfg->max_position <= 0 || !(cfg->rope_theta > 0)))
        return CW_ERR_INVALID;
    cw_ctx* ctx = new (std::nothrow) cw_ctx();
    if (!ctx) return CW_ERR_INVALID;
    ctx->cfg = *cfg;
    ctx->host_only = host_only;
    ctx->num_sms = 148;
    ctx->tree = new cw::KnowledgeTree(cfg->recency_window);
    ctx->blocks = new cw::BlockManager(cfg->num_blocks, cfg->eager_register != 0, cfg->hash_salt, cfg->index_key_bits);
    if (!host_only) {
        cudaError_t e = cudaSetDevice(cfg->device);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&ctx->num_sms, cudaDevAttrMultiProcessorCount, cfg->device);
        if (e == cudaSuccess) {
            // RoPE table (DESIGN.md c4): angle = p * theta^(-2i/D) evaluated in fp64, {cos, sin} rounded once to fp32
            const int half = cfg->head_dim / 2;
            std::vector<float> tab((size_t)cfg->max_position * half * 2);
            std::vector<double> inv((size_t)half);
            for (int i = 0; i < half; ++i) inv[(size_t)i] = std::pow(cfg->rope_theta, -2.0 * i / cfg->head_dim);
            for (int64_t p = 0; p < cfg->max_position; ++p)
                for (int i = 0; i < half; ++i) {
                    const double a = (double)p * inv[(size_t)i];
                    tab[((size_t)p * half + i) * 2] = (float)std::cos(a);
                    tab[((size_t)p * half + i) * 2 + 1] = (float)std::sin(a);
                }
            e = cudaMemcpy(cfg->rope_table, tab.data(), tab.size() * sizeof(float), cudaMemcpyHostToDevice);
        }
        if (e != cudaSuccess) {
            cw_destroy(ctx);
            return CW_ERR_CUDA;
        }
    }
    *out = ctx;
    return CW_OK;
}

void cw_destroy(cw_ctx* ctx) {
    if (!ctx) return;
    for (void* e : ctx->events) cudaEventDestroy(static_cast<cudaEvent_t>(e));
    for (auto& st : ctx->staging) {
        if (st.event) cudaEventDestroy(static_cast<cudaEvent_t>(st.event));
        if (st.host) cudaFreeHost(st.host);
    }
    if (ctx->sched_fork) cudaEventDestroy(static_cast<cudaEvent_t>(ctx->sched_fork));
    if (ctx->sched_join) cudaEventDestroy(static_cast<cudaEvent_t>(ctx->sched_join));
    if (ctx->sched_stream) cudaStreamDestroy(static_cast<cudaStream_t>(ctx->sched_stream));
    if (ctx->copy_in_stream) cudaStreamDestroy(static_cast<cudaStream_t>(ctx->copy_in_stream));
    if (ctx->copy_out_stream) cudaStreamDestroy(static_cast<cudaStream_t>(ctx->copy_out_stream));
    delete ctx->tree;
    delete ctx->blocks;
    delete ctx;
}

int cw_stats(cw_ctx* ctx, cw_stats_t* o) {
    if (!ctx || !o) return CW_ERR_INVALID;
    o->requests = ctx->blocks->requests;
    o->hit_blocks = ctx->blocks->hit_blocks;
    o->miss_blocks = ctx->blocks->miss_blocks;
    o->evictions = ctx->blocks->evictions;
    o->trie_nodes = ctx->tree->nodes();
    o->order_probes = ctx->tree->probes();
    o->free_blocks = ctx->blocks->free_count();
    o->seq = ctx->tree->seq();
    o->predicted_prefix_docs = ctx->pred_docs;
    o->actual_prefix_docs = ctx->actual_docs;
    o->over_predicted_docs = ctx->over_pred_docs;
    o->stale_marks = ctx->tree->stale_marks();
    const cw_config& c = ctx->cfg;
    o->prompt_tokens = ctx->blocks->prompt_tokens;
    o->suffix_tokens = ctx->blocks->suffix_tokens;
    o->attn_flops = 4 * (int64_t)c.num_q_heads * c.head_dim * ctx->blocks->attn_pairs;
    o->append_bytes = ctx->blocks->suffix_tokens * (2 * (int64_t)c.num_q_heads * c.head_dim * 2 + 4 * (int64_t)c.num_kv_heads * c.head_dim * 2 + 4);
    return CW_OK;
}

// ---- ordering ---------------------------------------------------------------------------------------------
static bool has_duplicates(const int64_t* ids, int32_t k) {
    if (k <= 16) {
        for (int i = 0; i < k; ++i)
            for (int j = i + 1; j < k; ++j)
                if (ids[i] == ids[j]) return true;
        return false;
    }
    std::unordered_set<int64_t> s(ids, ids + k);
    return (int32_t)s.size() != k;
}

int cw_order(cw_ctx* ctx, const int64_t* doc_ids, int32_t k, int64_t* out_order, int32_t* out_pred) {
    if (!ctx || k < 0 || (k > 0 && (!doc_ids || !out_order))) return fail(ctx, CW_ERR_INVALID, "cw_order: bad argument");
    if (has_duplicates(doc_ids, k)) return fail(ctx, CW_ERR_INVALID, "cw_order: duplicate document id");
    int depth = ctx->tree->order(doc_ids, k, out_order);
    if (out_pred) *out_pred = depth;
    return CW_OK;
}

int cw_predict(cw_ctx* ctx, const int64_t* order, int32_t k, int32_t* out_prefix_docs) {
    if (!ctx || k < 0 || (k > 0 && !order) || !out_prefix_docs) return fail(ctx, CW_ERR_INVALID, "cw_predict: bad argument");
    *out_prefix_docs = ctx->tree->predict(order, k);
    return CW_OK;
}

int cw_observe(cw_ctx* ctx, const int64_t* ordered, int32_t k) {
    if (!ctx || k < 0 || (k > 0 && !ordered)) return fail(ctx, CW_ERR_INVALID, "cw_observe: bad argument");
    if (has_duplicates(ordered, k)) return fail(ctx, CW_ERR_INVALID, "cw_observe: duplicate document id");
    ctx->tree->observe(ordered, k);
    for (int i = 0; i < k; ++i) ctx->last_served[ordered[i]] = ctx->tree->seq();
    return CW_OK;
}

int cw_mark_stale(cw_ctx* ctx, const int64_t* order, int32_t k, int32_t resident_docs) {
    if (!ctx || k < 0 || (k > 0 && !order) || resident_docs < 0) return fail(ctx, CW_ERR_INVALID, "cw_mark_stale: bad argument");
    ctx->tree->mark_stale(order, k, resident_docs);
    return CW_OK;
}

int cw_feedback(cw_ctx* ctx, const int64_t* order, int32_t k, int32_t predicted_docs, int32_t actual_docs) {
    if (!ctx || k < 0 || (k > 0 && !order) || predicted_docs < 0 || actual_docs < 0)
        return fail(ctx, CW_ERR_INVALID, "cw_feedback: bad argument");
    if (predicted_docs > actual_docs) ctx->tree->mark_stale(order, k, actual_docs);
    ctx->pred_docs += predicted_docs;
    ctx->actual_docs += actual_docs;
    ctx->over_pred_docs += std::max(0, predicted_docs - actual_docs);
    return CW_OK;
}

int cw_matched_docs(cw_ctx* ctx, const int32_t* doc_ends, int32_t k, int32_t n_cached, int32_t n_tokens, int32_t* out_docs) {
    if (!ctx || !out_docs || bad_doc_ends(doc_ends, k, n_cached, n_tokens))
        return fail(ctx, CW_ERR_INVALID, "cw_matched_docs: bad argument (doc_ends must be positive, non-decreasing, <= n_tokens)");
    *out_docs = count_matched_docs([&](int32_t j) { return doc_ends[j]; }, k, n_cached, n_tokens);
    return CW_OK;
}

int cw_feedback_tokens(cw_ctx* ctx, const int64_t* order, int32_t k, int32_t predicted_docs, const int32_t* doc_ends,
                       int32_t n_cached, int32_t n_tokens, int32_t* out_actual_docs) {
    int32_t actual = 0;
    if (!ctx || (k > 0 && !order) || predicted_docs < 0 || predicted_docs > k)
        return fail(ctx, CW_ERR_INVALID, "cw_feedback_tokens: bad argument");
    const int rc = cw_matched_docs(ctx, doc_ends, k, n_cached, n_tokens, &actual);
    if (rc != CW_OK) return rc;
    if (out_actual_docs) *out_actual_docs = actual;
    return cw_feedback(ctx, order, k, predicted_docs, actual);
}

int cw_order_arm(cw_ctx* ctx, int32_t arm, const int64_t* doc_ids, int32_t k, const int32_t* doc_tokens, int32_t num_docs,
                 int32_t doc_len, const int32_t* query_tokens, int32_t q_len, int64_t* out_order, int32_t* out_pred) {
    if (!ctx || k < 0 || (k > 0 && (!doc_ids || !out_order)) || arm < CW_ARM_RETRIEVAL || arm > CW_ARM_GREEDY_RESIDENT)
        return fail(ctx, CW_ERR_INVALID, "cw_order_arm: bad argument");
    if (has_duplicates(doc_ids, k)) return fail(ctx, CW_ERR_INVALID, "cw_order_arm: duplicate document id");
    if (arm == CW_ARM_GREEDY || arm == CW_ARM_GREEDY_FEEDBACK) {
        ctx->tree->order(doc_ids, k, out_order);
    } else if (arm == CW_ARM_GREEDY_RESIDENT) {
        if (doc_len < 0 || (k > 0 && !doc_tokens))
            return fail(ctx, CW_ERR_INVALID, "cw_order_arm: the residency-aware arm needs the document tokens");
        for (int i = 0; i < k; ++i)
            if (doc_ids[i] < 0 || doc_ids[i] >= num_docs) return fail(ctx, CW_ERR_INVALID, "cw_order_arm: doc id out of range");
        // peek on the real block index, incremental over the confirmed document prefix
        cw::BlockManager::Probe probe = ctx->blocks->probe_begin();
        const std::function<bool(const int64_t*, int, int64_t)> resident = [&](const int64_t*, int, int64_t d) {
            return ctx->blocks->probe_extend(probe, doc_tokens + (size_t)d * doc_len, doc_len);
        };
        ctx->tree->order(doc_ids, k, out_order, &resident);
    } else if (arm == CW_ARM_RETRIEVAL) {
        std::memcpy(out_order, doc_ids, sizeof(int64_t) * (size_t)k);
    } else if (arm == CW_ARM_SORTED) {
        std::memcpy(out_order, doc_ids, sizeof(int64_t) * (size_t)k);
        std::sort(out_order, out_order + k);
    } else if (arm == CW_ARM_RECENCY) {
        std::memcpy(out_order, doc_ids, sizeof(int64_t) * (size_t)k);
        auto served = [&](int64_t d) {
            auto it = ctx->last_served.find(d);
            return it == ctx->last_served.end() ? (int64_t)0 : it->second;
        };
        std::stable_sort(out_order, out_order + k, [&](int64_t a, int64_t b) { return served(a) > served(b); });
    } else {
        if (k > 8 || doc_len < 0 || q_len < 0 || (k > 0 && !doc_tokens) || (q_len > 0 && !query_tokens))
            return fail(ctx, CW_ERR_INVALID, "cw_order_arm: exhaustive search needs k <= 8 and the tokens");
        for (int i = 0; i < k; ++i)
            if (doc_ids[i] < 0 || doc_ids[i] >= num_docs) return fail(ctx, CW_ERR_INVALID, "cw_order_arm: doc id out of range");
        const int32_t n = k * doc_len + q_len;
        if (n <= 0) return fail(ctx, CW_ERR_INVALID, "cw_order_arm: empty prompt");
        std::vector<int32_t> tokens((size_t)n);
        if (q_len) std::memcpy(tokens.data() + (size_t)k * doc_len, query_tokens, sizeof(int32_t) * (size_t)q_len);
        std::vector<int> perm((size_t)k);
        for (int i = 0; i < k; ++i) perm[(size_t)i] = i;
        std::vector<uint64_t> chain, vchain;
        int32_t best = -1;
        do {   // permutations in lexicographic order of retrieval-rank indices; keep the first maximiser
            for (int i = 0; i < k; ++i)
                std::memcpy(tokens.data() + (size_t)i * doc_len, doc_tokens + (size_t)doc_ids[perm[(size_t)i]] * doc_len,
                            sizeof(int32_t) * (size_t)doc_len);
            ctx->blocks->chains(tokens.data(), n, chain, vchain);
            const int32_t m = ctx->blocks->match(chain, vchain, n);
            if (m > best) {
                best = m;
                for (int i = 0; i < k; ++i) out_order[i] = doc_ids[perm[(size_t)i]];
            }
        } while (std::next_permutation(perm.begin(), perm.end()));
    }
    if (out_pred) *out_pred = ctx->tree->predict(out_order, k);
    return CW_OK;
}

// ---- prefix cache -----------------------------------------------------------------------------------------
int cw_hash_chain(cw_ctx* ctx, const int32_t* tokens, int32_t n, uint64_t* out_chain) {
    if (!ctx || n < 0 || (n > 0 && !tokens) || (n >= CW_BLOCK_SIZE && !out_chain))
        return fail(ctx, CW_ERR_INVALID, "cw_hash_chain: bad argument");
    std::vector<uint64_t> ch;
    ctx->blocks->chain(tokens, n, ch);
    if (!ch.empty()) std::memcpy(out_chain, ch.data(), ch.size() * sizeof(uint64_t));
    return CW_OK;
}

int cw_lookup(cw_ctx* ctx, const int32_t* tokens, int32_t n, int32_t peek_only, int64_t* out_req,
              int32_t* out_block_table, int32_t* out_n_cached) {
    if (!ctx || !tokens || n <= 0 || !out_n_cached) return fail(ctx, CW_ERR_INVALID, "cw_lookup: bad argument");
    if (peek_only) {
        std::vector<uint64_t> ch;
        std::vector<uint64_t> vc;
        ctx->blocks->chains(tokens, n, ch, vc);
        *out_n_cached = ctx->blocks->match(ch, vc, n) * CW_BLOCK_SIZE;
        return CW_OK;
    }
    if (!out_req || !out_block_table) return fail(ctx, CW_ERR_INVALID, "cw_lookup: null output");
    return ctx->blocks->lookup(tokens, n, out_req, out_block_table, out_n_cached);
}

int cw_release(cw_ctx* ctx, int64_t req) {
    if (!ctx) return CW_ERR_INVALID;
    return ctx->blocks->release(req);
}

int cw_extend(cw_ctx* ctx, int64_t req, const int32_t* new_tokens, int32_t n_new, int32_t* out_block_table, int32_t cap,
              int32_t* out_n_blocks) {
    if (!ctx || n_new < 0 || (n_new > 0 && !new_tokens) || !out_block_table || !out_n_blocks || cap < 0)
        return fail(ctx, CW_ERR_INVALID, "cw_extend: bad argument");
    int rc = ctx->blocks->extend(req, new_tokens, n_new, out_block_table, cap, out_n_blocks);
    if (rc == CW_ERR_INVALID) return fail(ctx, rc, "cw_extend: block table capacity too small (or sequence too long)");
    return rc;
}

int cw_reset(cw_ctx* ctx) {
    if (!ctx) return CW_ERR_INVALID;
    delete ctx->tree;
    delete ctx->blocks;
    ctx->tree = new cw::KnowledgeTree(ctx->cfg.recency_window);
    ctx->blocks = new cw::BlockManager(ctx->cfg.num_blocks, ctx->cfg.eager_register != 0, ctx->cfg.hash_salt,
                                       ctx->cfg.index_key_bits);
    ctx->last_served.clear();
    ctx->last_error.clear();
    ctx->pred_docs = ctx->actual_docs = ctx->over_pred_docs = 0;
    return CW_OK;
}

int cw_admit_batch(cw_ctx* ctx, const int64_t* doc_ids, int32_t B, int32_t k, int32_t reorder, const int32_t* doc_tokens,
                   int32_t num_docs, int32_t doc_len, const int32_t* query_tokens, int32_t q_len, int64_t* out_orders,
                   int32_t* out_pred, int64_t* out_reqs, int32_t* out_tables, int32_t max_blocks, int32_t* out_nc,
                   int32_t* out_cu, int32_t* out_admitted) {
    if (!ctx || B < 0 || k < 0 || doc_len < 0 || q_len < 0 || num_docs < 0 || !out_admitted || !out_cu)
        return fail(ctx, CW_ERR_INVALID, "cw_admit_batch: bad argument");
    *out_admitted = 0;
    out_cu[0] = 0;
    if (B == 0) return CW_OK;
    const int64_t n64 = (int64_t)k * doc_len + q_len;
    if (n64 <= 0 || n64 > INT32_MAX || (n64 + CW_BLOCK_SIZE - 1) / CW_BLOCK_SIZE > max_blocks)
        return fail(ctx, CW_ERR_INVALID, "cw_admit_batch: prompt length / max_blocks");
    if ((k > 0 && (!doc_ids || !doc_tokens || !out_orders)) || (q_len > 0 && !query_tokens) || !out_pred || !out_reqs ||
        !out_tables || !out_nc)
        return fail(ctx, CW_ERR_INVALID, "cw_admit_batch: null pointer");
    const int32_t n = (int32_t)n64, nblk = (n + CW_BLOCK_SIZE - 1) / CW_BLOCK_SIZE;
    if (reorder < CW_ARM_RETRIEVAL || reorder > CW_ARM_GREEDY_RESIDENT || (reorder == CW_ARM_EXHAUSTIVE && k > 8))
        return fail(ctx, CW_ERR_INVALID, "cw_admit_batch: unknown ordering arm (or exhaustive with k > 8)");
    // every row is validated BEFORE anything is admitted: an invalid argument leaves the state untouched
    for (int32_t r = 0; r < B; ++r) {
        const int64_t* D = doc_ids + (size_t)r * k;
        for (int i = 0; i < k; ++i)
            if (D[i] < 0 || D[i] >= num_docs) return fail(ctx, CW_ERR_INVALID, "cw_admit_batch: doc id out of range");
        if (has_duplicates(D, k)) return fail(ctx, CW_ERR_INVALID, "cw_admit_batch: duplicate document id");
    }
    std::vector<int32_t> tokens((size_t)n);
    for (int32_t r = 0; r < B; ++r) {
        const int64_t* D = doc_ids + (size_t)r * k;
        int64_t* O = out_orders + (size_t)r * k;
        {
            const int rc = cw_order_arm(ctx, reorder, D, k, doc_tokens, num_docs, doc_len,
                                        q_len ? query_tokens + (size_t)r * q_len : nullptr, q_len, O, out_pred + r);
            if (rc != CW_OK) return rc;
        }
        for (int i = 0; i < k; ++i)
            std::memcpy(tokens.data() + (size_t)i * doc_len, doc_tokens + (size_t)O[i] * doc_len, sizeof(int32_t) * (size_t)doc_len);
        if (q_len) std::memcpy(tokens.data() + (size_t)k * doc_len, query_tokens + (size_t)r * q_len, sizeof(int32_t) * (size_t)q_len);
        int32_t* table = out_tables + (size_t)r * max_blocks;
        int rc = ctx->blocks->lookup(tokens.data(), n, out_reqs + r, table, out_nc + r);
        if (rc == CW_ERR_NO_SPACE) return CW_OK;
        if (rc != CW_OK) return rc;
        for (int32_t i = nblk; i < max_blocks; ++i) table[i] = 0;
        {   // predicted vs actual prefix: documents all of whose full 16-token blocks are inside the cached tokens
            const int32_t actual = count_matched_docs([&](int32_t j) { return (int64_t)(j + 1) * doc_len; }, k, out_nc[r], n);
            if (reorder == CW_ARM_GREEDY_FEEDBACK || reorder == CW_ARM_GREEDY_RESIDENT) {
                cw_feedback(ctx, O, k, out_pred[r], actual);
            } else {
                ctx->pred_docs += out_pred[r];
                ctx->actual_docs += actual;
                ctx->over_pred_docs += std::max(0, out_pred[r] - actual);
            }
        }
        ctx->tree->observe(O, k);
        for (int i = 0; i < k; ++i) ctx->last_served[O[i]] = ctx->tree->seq();
        out_cu[r + 1] = out_cu[r] + (n - out_nc[r]);
        *out_admitted = r + 1;
    }
    return CW_OK;
}

int cw_release_batch(cw_ctx* ctx, const int64_t* reqs, int32_t B) {
    if (!ctx || B < 0 || (B > 0 && !reqs)) return fail(ctx, CW_ERR_INVALID, "cw_release_batch: bad argument");
    for (int32_t i = 0; i < B; ++i) {
        int rc = ctx->blocks->release(reqs[i]);
        if (rc != CW_OK) return rc;
    }
    return CW_OK;
}

int cw_free_list(cw_ctx* ctx, int32_t* out, int32_t cap, int32_t* out_len) {
    if (!ctx || !out_len || cap < 0 || (cap > 0 && !out)) return fail(ctx, CW_ERR_INVALID, "cw_free_list: bad argument");
    *out_len = ctx->blocks->free_list(out, cap);
    return CW_OK;
}

// ---- device work ------------------------------------------------------------------------------------------
int cw_append_kv(cw_ctx* ctx, const void* q, const void* k, const void* v, void* q_roped, const int32_t* d_cu,
                 const int32_t* d_nc, const int32_t* d_tables, int32_t max_blocks, int32_t B, int32_t T, void* stream) {
    if (!ctx || ctx->host_only) return fail(ctx, CW_ERR_INVALID, "cw_append_kv: host-only context");
    if (B < 0 || T < 0 || max_blocks <= 0) return fail(ctx, CW_ERR_INVALID, "cw_append_kv: bad sizes");
    if (T == 0 || B == 0) return CW_OK;
    if (!q || !k || !v || !q_roped || !d_cu || !d_nc || !d_tables || q == q_roped)
        return fail(ctx, CW_ERR_INVALID, "cw_append_kv: null or aliased pointer");
    int e = cw::launch_append_kv(ctx->cfg, q, k, v, q_roped, d_cu, d_nc, d_tables, max_blocks, B, T, ctx->num_sms, stream);
    return e ? cuda_fail(ctx, e, "cw_append_kv") : CW_OK;
}

int cw_gather_kv(cw_ctx* ctx, const int32_t* d_table, int32_t n, void* k_out, void* v_out, void* stream) {
    if (!ctx || ctx->host_only) return fail(ctx, CW_ERR_INVALID, "cw_gather_kv: host-only context");
    if (n < 0) return fail(ctx, CW_ERR_INVALID, "cw_gather_kv: bad size");
    if (n == 0) return CW_OK;
    if (!d_table || !k_out || !v_out) return fail(ctx, CW_ERR_INVALID, "cw_gather_kv: null pointer");
    int e = cw::launch_gather_kv(ctx->cfg, d_table, n, k_out, v_out, ctx->num_sms, stream);
    return e ? cuda_fail(ctx, e, "cw_gather_kv") : CW_OK;
}

int64_t cw_attn_work_ints(cw_ctx* ctx, int32_t B, int32_t T) {
    if (!ctx || B < 0 || T < 0) return CW_ERR_INVALID;
    return cw::attn_work_ints(ctx->cfg, B, T);
}

int cw_prefill_attn(cw_ctx* ctx, const void* q_roped, void* out, const int32_t* d_cu, const int32_t* d_nc,
                    const int32_t* d_kv_len, const int32_t* d_tables, int32_t max_blocks, int32_t B, int32_t T,
                    int32_t max_q_len, int32_t max_kv_len, int32_t* d_work, void* stream) {
    if (!ctx || ctx->host_only) return fail(ctx, CW_ERR_INVALID, "cw_prefill_attn: host-only context");
    if (B < 0 || T < 0 || max_blocks <= 0 || max_q_len < 0 || max_kv_len < 0)
        return fail(ctx, CW_ERR_INVALID, "cw_prefill_attn: bad sizes");
    if (T == 0 || B == 0) return CW_OK;
    if (!q_roped || !out || !d_cu || !d_nc || !d_tables || !d_work)
        return fail(ctx, CW_ERR_INVALID, "cw_prefill_attn: null pointer");
    if (max_q_len > T || (int64_t)max_kv_len > (int64_t)max_blocks * CW_BLOCK_SIZE || max_kv_len > ctx->cfg.max_position)
        return fail(ctx, CW_ERR_INVALID, "cw_prefill_attn: max_q_len / max_kv_len exceed T, the block table or max_position");
    int le = cw::launch_prefill_attn(ctx->cfg, q_roped, out, d_cu, d_nc, d_kv_len, d_tables, max_blocks, B, T, max_q_len,
                                     max_kv_len, d_work, ctx->num_sms, stream);
    return le ? cuda_fail(ctx, le, "cw_prefill_attn") : CW_OK;
}

// The two launches of cw_prefill_attn one by one (cacheweaver.h): same checks, same kernels.
int cw_attn_schedule(cw_ctx* ctx, const int32_t* d_cu, const int32_t* d_nc, const int32_t* d_kv_len, const int32_t* d_tables,
                     int32_t max_blocks, int32_t B, int32_t T, int32_t max_q_len, int32_t max_kv_len, int32_t* d_work,
                     void* stream) {
    if (!ctx || ctx->host_only) return fail(ctx, CW_ERR_INVALID, "cw_attn_schedule: host-only context");
    if (B < 0 || T < 0 || max_blocks <= 0 || max_q_len < 0 || max_kv_len < 0)
        return fail(ctx, CW_ERR_INVALID, "cw_attn_schedule: bad sizes");
    if (T == 0 || B == 0) return CW_OK;
    if (!d_cu || !d_nc || !d_tables || !d_work) return fail(ctx, CW_ERR_INVALID, "cw_attn_schedule: null pointer");
    if (max_q_len > T || (int64_t)max_kv_len > (int64_t)max_blocks * CW_BLOCK_SIZE || max_kv_len > ctx->cfg.max_position)
        return fail(ctx, CW_ERR_INVALID, "cw_attn_schedule: max_q_len / max_kv_len exceed T, the block table or max_position");
    int le = cw::launch_attn_schedule(ctx->cfg, d_cu, d_nc, d_kv_len, d_tables, max_blocks, B, T, max_q_len, max_kv_len,
                                      d_work, stream);
    return le ? cuda_fail(ctx, le, "cw_attn_schedule") : CW_OK;
}

int cw_attn_run(cw_ctx* ctx, const void* q_roped, void* out, const int32_t* d_tables, int32_t max_blocks, int32_t B,
                int32_t T, int32_t* d_work, void* stream) {
    if (!ctx || ctx->host_only) return fail(ctx, CW_ERR_INVALID, "cw_attn_run: host-only context");
    if (B < 0 || T < 0 || max_blocks <= 0) return fail(ctx, CW_ERR_INVALID, "cw_attn_run: bad sizes");
    if (T == 0 || B == 0) return CW_OK;
    if (!q_roped || !out || !d_tables || !d_work) return fail(ctx, CW_ERR_INVALID, "cw_attn_run: null pointer");
    int le = cw::launch_attn_run(ctx->cfg, q_roped, out, d_tables, max_blocks, B, T, d_work, ctx->num_sms, stream);
    return le ? cuda_fail(ctx, le, "cw_attn_run") : CW_OK;
}

// cw_prefill_attn with the work list in the library's static device array: for callers that cannot allocate device memory
// (cacheweaver.h).  Nothing here or below allocates; a batch that needs more than CW_STATIC_WORK_INTS ints is refused.
int cw_prefill_attn_static(cw_ctx* ctx, const void* q_roped, void* out, const int32_t* d_cu, const int32_t* d_nc,
                           const int32_t* d_kv_len, const int32_t* d_tables, int32_t max_blocks, int32_t B, int32_t T,
                           int32_t max_q_len, int32_t max_kv_len, int32_t* d_status, void* stream) {
    if (!ctx || ctx->host_only) return fail(ctx, CW_ERR_INVALID, "cw_prefill_attn_static: host-only context");
    if (B < 0 || T < 0 || max_blocks <= 0 || max_q_len < 0 || max_kv_len < 0)
        return fail(ctx, CW_ERR_INVALID, "cw_prefill_attn_static: bad sizes");
    if (cw::attn_work_ints(ctx->cfg, B, T) > (int64_t)CW_STATIC_WORK_INTS)
        return fail(ctx, CW_ERR_INVALID,
                    "cw_prefill_attn_static: the batch exceeds the static work list (cw_attn_work_ints(B, T) > "
                    "CW_STATIC_WORK_INTS = 524288): split the wave or pass your own scratch to cw_prefill_attn");
    if (T == 0 || B == 0) return CW_OK;
    if (!q_roped || !out || !d_cu || !d_nc || !d_tables)
        return fail(ctx, CW_ERR_INVALID, "cw_prefill_attn_static: null pointer");
    if (max_q_len > T || (int64_t)max_kv_len > (int64_t)max_blocks * CW_BLOCK_SIZE || max_kv_len > ctx->cfg.max_position)
        return fail(ctx, CW_ERR_INVALID,
                    "cw_prefill_attn_static: max_q_len / max_kv_len exceed T, the block table or max_position");
    int le = cw::launch_prefill_attn_static(ctx->cfg, q_roped, out, d_cu, d_nc, d_kv_len, d_tables, max_blocks, B, T,
                                            max_q_len, max_kv_len, d_status, ctx->num_sms, stream);
    return le ? cuda_fail(ctx, le, "cw_prefill_attn_static") : CW_OK;
}

// ---- one call per wave: descriptors from the request handles, one staged H2D copy, three launches ----------
namespace {
// cw_prefill_requests: waves with at least this many suffix rows run the schedule kernel on a side stream beside
// cw_append_kv (below it the two event calls cost the host more than the ~20 us the GPU saves)
constexpr int32_t kSideScheduleMinRows = 4096;
struct ReqWsLayout {
    int64_t cu, nc, tables, work, total;
};
ReqWsLayout req_ws_layout(const cw_config& c, int32_t B, int32_t T, int32_t max_blocks) {
    ReqWsLayout w{};
    int64_t o = 0;
    w.cu = o; o += ((int64_t)B + 1) * 4;                 // cu, nc and the tables are contiguous: one H2D copy
    w.nc = o; o += (int64_t)B * 4;
    w.tables = o; o += (int64_t)B * max_blocks * 4;
    o = align256(o);
    w.work = o; o += align256(cw::attn_work_ints(c, B, T) * 4);
    w.total = o;
    return w;
}
}  // namespace

int64_t cw_prefill_requests_ws_bytes(cw_ctx* ctx, int32_t B, int32_t T, int32_t max_blocks) {
    if (!ctx || B < 0 || T < 0 || max_blocks <= 0) return CW_ERR_INVALID;
    return req_ws_layout(ctx->cfg, B, T, max_blocks).total;
}

int64_t cw_prefill_requests_work_offset(cw_ctx* ctx, int32_t B, int32_t max_blocks) {
    if (!ctx || B < 0 || max_blocks <= 0) return CW_ERR_INVALID;
    return req_ws_layout(ctx->cfg, B, 0, max_blocks).work;
}

int cw_prefill_requests(cw_ctx* ctx, const int64_t* reqs, int32_t B, const void* q, const void* k, const void* v,
                        void* q_roped, void* out, int32_t T, int32_t max_blocks, void* d_ws, void* stream) {
    if (!ctx || ctx->host_only) return fail(ctx, CW_ERR_INVALID, "cw_prefill_requests: host-only context");
    if (B < 0 || T < 0 || max_blocks <= 0) return fail(ctx, CW_ERR_INVALID, "cw_prefill_requests: bad sizes");
    if (B == 0) return T == 0 ? CW_OK : fail(ctx, CW_ERR_INVALID, "cw_prefill_requests: T != 0 for an empty batch");
    if (!reqs || !q || !k || !v || !q_roped || !out || !d_ws || q == q_roped)
        return fail(ctx, CW_ERR_INVALID, "cw_prefill_requests: null or aliased pointer");
    const ReqWsLayout w = req_ws_layout(ctx->cfg, B, T, max_blocks);
    // descriptors of the wave, written into a pinned staging slot (cu | nc | tables, contiguous like in d_ws)
    const size_t desc_bytes = (size_t)w.tables + (size_t)B * max_blocks * 4;
    cw_ctx::Staging& st = ctx->staging[ctx->staging_next];
    ctx->staging_next = (ctx->staging_next + 1) % cw_ctx::kStagingSlots;
    cudaError_t e = cudaSuccess;
    if (st.event) e = cudaEventSynchronize(static_cast<cudaEvent_t>(st.event));   // the copy that last read this slot
    if (e == cudaSuccess && st.cap < desc_bytes) {
        if (st.host) cudaFreeHost(st.host);
        st.host = nullptr;
        st.cap = 0;
        const size_t cap = std::max<size_t>(desc_bytes * 2, 1 << 16);
        e = cudaMallocHost(&st.host, cap);
        if (e == cudaSuccess) st.cap = cap;
    }
    if (e == cudaSuccess && !st.event) {
        cudaEvent_t ev;
        e = cudaEventCreateWithFlags(&ev, cudaEventDisableTiming);
        if (e == cudaSuccess) st.event = ev;
    }
    if (e != cudaSuccess) return cuda_fail(ctx, (int)e, "cw_prefill_requests (staging)");
    int32_t* cu = reinterpret_cast<int32_t*>(static_cast<char*>(st.host) + w.cu);
    int32_t* nc = reinterpret_cast<int32_t*>(static_cast<char*>(st.host) + w.nc);
    int32_t* tables = reinterpret_cast<int32_t*>(static_cast<char*>(st.host) + w.tables);
    cu[0] = 0;
    int32_t max_q = 0, max_kv = 0;
    std::unordered_set<int64_t> seen;
    seen.reserve((size_t)B * 2);
    for (int32_t r = 0; r < B; ++r) {
        const cw::Request* rq = ctx->blocks->find(reqs[r]);
        if (!rq) return fail(ctx, CW_ERR_BAD_HANDLE, "cw_prefill_requests: unknown request handle");
        if (!seen.insert(reqs[r]).second)       // its rows would be counted (and written) twice
            return fail(ctx, CW_ERR_INVALID, "cw_prefill_requests: a request handle is listed twice");
        const int32_t nblk = (int32_t)rq->table.size(), c = rq->n_done, s = rq->n - c;
        if (nblk > max_blocks) return fail(ctx, CW_ERR_INVALID, "cw_prefill_requests: max_blocks too small for a request");
        if (rq->n > ctx->cfg.max_position) return fail(ctx, CW_ERR_INVALID, "cw_prefill_requests: prompt longer than max_position");
        nc[r] = c;
        cu[r + 1] = cu[r] + s;
        std::memcpy(tables + (size_t)r * max_blocks, rq->table.data(), sizeof(int32_t) * (size_t)nblk);
        std::memset(tables + (size_t)r * max_blocks + nblk, 0, sizeof(int32_t) * (size_t)(max_blocks - nblk));
        max_q = std::max(max_q, s);
        max_kv = std::max(max_kv, rq->n);
    }
    if (cu[B] != T) return fail(ctx, CW_ERR_INVALID, "cw_prefill_requests: T does not match the requests' pending tokens");
    auto s = static_cast<cudaStream_t>(stream);
    char* ws = static_cast<char*>(d_ws);
    e = cudaMemcpyAsync(ws, st.host, desc_bytes, cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaEventRecord(static_cast<cudaEvent_t>(st.event), s);
    if (e != cudaSuccess) return cuda_fail(ctx, (int)e, "cw_prefill_requests (descriptor copy)");
    const int32_t* d_cu = reinterpret_cast<const int32_t*>(ws + w.cu);
    const int32_t* d_nc = reinterpret_cast<const int32_t*>(ws + w.nc);
    const int32_t* d_tables = reinterpret_cast<const int32_t*>(ws + w.tables);
    int32_t* d_work = reinterpret_cast<int32_t*>(ws + w.work);
    int rc;
    if (T >= kSideScheduleMinRows) {
        // The schedule kernel needs only the descriptors: it runs on a side stream BESIDE cw_append_kv (one CTA next to an
        // HBM-bound kernel) instead of between it and the attention kernel.  fork: behind the descriptor copy (and behind
        // everything earlier on `stream`, so the previous call's attention kernel is done with a shared d_ws); join: in
        // front of the attention kernel.
        if (!ctx->sched_stream) {
            cudaStream_t ss;
            cudaEvent_t ef, ej;
            if ((e = cudaStreamCreateWithFlags(&ss, cudaStreamNonBlocking)) != cudaSuccess ||
                (e = cudaEventCreateWithFlags(&ef, cudaEventDisableTiming)) != cudaSuccess ||
                (e = cudaEventCreateWithFlags(&ej, cudaEventDisableTiming)) != cudaSuccess)
                return cuda_fail(ctx, (int)e, "cw_prefill_requests (side stream)");
            ctx->sched_stream = ss;
            ctx->sched_fork = ef;
            ctx->sched_join = ej;
        }
        auto ss = static_cast<cudaStream_t>(ctx->sched_stream);
        auto ef = static_cast<cudaEvent_t>(ctx->sched_fork), ej = static_cast<cudaEvent_t>(ctx->sched_join);
        if ((e = cudaEventRecord(ef, s)) != cudaSuccess || (e = cudaStreamWaitEvent(ss, ef, 0)) != cudaSuccess)
            return cuda_fail(ctx, (int)e, "cw_prefill_requests (fork)");
        rc = cw_attn_schedule(ctx, d_cu, d_nc, nullptr, d_tables, max_blocks, B, T, max_q, max_kv, d_work, ss);
        // the join is enqueued whatever happened in between: the side stream must never be left un-joined
        e = cudaEventRecord(ej, ss);
        const int rc2 = cw_append_kv(ctx, q, k, v, q_roped, d_cu, d_nc, d_tables, max_blocks, B, T, stream);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(s, ej, 0);
        if (rc != CW_OK) return rc;
        if (rc2 != CW_OK) return rc2;
        if (e != cudaSuccess) return cuda_fail(ctx, (int)e, "cw_prefill_requests (join)");
        rc = cw_attn_run(ctx, q_roped, out, d_tables, max_blocks, B, T, d_work, stream);
    } else {
        rc = cw_append_kv(ctx, q, k, v, q_roped, d_cu, d_nc, d_tables, max_blocks, B, T, stream);
        if (rc != CW_OK) return rc;
        rc = cw_prefill_attn(ctx, q_roped, out, d_cu, d_nc, nullptr, d_tables, max_blocks, B, T, max_q, max_kv, d_work, stream);
    }
    if (rc != CW_OK) return rc;
    // Only now, with the copy and both kernels enqueued, do the handles move on: everything up to n is (being) written and
    // the next call starts there.  After a failure above they are unchanged, so the same call can be repeated (writing a
    // row's K/V twice is harmless).
    for (int32_t r = 0; r < B; ++r) ctx->blocks->find_mut(reqs[r])->n_done = ctx->blocks->find(reqs[r])->n;
    return CW_OK;
}

// ---- host-buffer entry point ------------------------------------------------------------------------------
namespace {
constexpr int kHostChunks = 16;   // cw_prefill_host pipelines the batch in up to this many request chunks
struct WsLayout {
    int64_t q, k, v, qr, out, cu, nc, tables, work, total;
};
WsLayout ws_layout(const cw_config& c, int32_t B, int32_t T, int32_t max_blocks) {
    WsLayout w{};
    const int64_t qb = (int64_t)T * c.num_q_heads * c.head_dim * 2, kb = (int64_t)T * c.num_kv_heads * c.head_dim * 2;
    int64_t o = 0;
    w.q = o; o += align256(qb);
    w.k = o; o += align256(kb);
    w.v = o; o += align256(kb);
    w.qr = o; o += align256(qb);
    w.out = o; o += align256(qb);
    w.cu = o; o += align256((int64_t)(B + 1 + kHostChunks) * 4);      // chunk-local prefix sums: (B_c + 1) ints per chunk
    w.nc = o; o += align256((int64_t)B * 4);
    w.tables = o; o += align256((int64_t)B * max_blocks * 4);
    // upper bound on tiles: every request may add one ragged tile per kv head
    w.work = o; o += align256(cw::attn_work_ints(c, B, T) * 4) + (align256(32) + 256) * kHostChunks;   // one list (+ header) per chunk
    w.total = o;
    return w;
}
}  // namespace

int64_t cw_prefill_host_ws_bytes(cw_ctx* ctx, int32_t B, int32_t T, int32_t max_blocks) {
    if (!ctx || B < 0 || T < 0 || max_blocks <= 0) return CW_ERR_INVALID;
    return ws_layout(ctx->cfg, B, T, max_blocks).total;
}

int cw_prefill_host(cw_ctx* ctx, const void* h_q, const void* h_k, const void* h_v, void* h_out,
                    const int32_t* h_cu, const int32_t* h_nc, const int32_t* h_tables, int32_t max_blocks, int32_t B,
                    int32_t T, void* d_ws, void* stream) {
    if (!ctx || ctx->host_only) return fail(ctx, CW_ERR_INVALID, "cw_prefill_host: host-only context");
    if (B < 0 || T < 0 || max_blocks <= 0) return fail(ctx, CW_ERR_INVALID, "cw_prefill_host: bad sizes");
    if (T == 0 || B == 0) return CW_OK;
    if (!h_q || !h_k || !h_v || !h_out || !h_cu || !h_nc || !h_tables || !d_ws)
        return fail(ctx, CW_ERR_INVALID, "cw_prefill_host: null pointer");
    if (h_cu[0] != 0 || h_cu[B] != T) return fail(ctx, CW_ERR_INVALID, "cw_prefill_host: cu_seqlens_q does not span T");
    int32_t max_q = 0, max_kv = 0;
    for (int r = 0; r < B; ++r) {
        const int s = h_cu[r + 1] - h_cu[r];
        if (s < 0 || h_nc[r] < 0 || (int64_t)h_nc[r] + s > (int64_t)max_blocks * CW_BLOCK_SIZE ||
            h_nc[r] + s > ctx->cfg.max_position)
            return fail(ctx, CW_ERR_INVALID, "cw_prefill_host: bad request descriptor");
        max_q = std::max(max_q, s);
        max_kv = std::max(max_kv, h_nc[r] + s);
    }
    const cw_config& c = ctx->cfg;
    const WsLayout w = ws_layout(c, B, T, max_blocks);
    auto s = static_cast<cudaStream_t>(stream);
    char* ws = static_cast<char*>(d_ws);
    cudaError_t e = cudaSuccess;
    // The batch is cut into request chunks of about equal token count and pipelined over three streams: H2D of chunk i+1
    // (copy-in stream), RoPE + scatter and attention of chunk i (caller's stream, in request order: later requests may read
    // blocks written by earlier ones of the same batch), D2H of chunk i-1 (copy-out stream).  PCIe is full duplex, so the
    // end-to-end time approaches max(H2D, D2H) instead of their sum.
    if (!ctx->copy_in_stream) {
        cudaStream_t a = nullptr, b = nullptr;
        e = cudaStreamCreateWithFlags(&a, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&b, cudaStreamNonBlocking);
        if (e != cudaSuccess) return cuda_fail(ctx, (int)e, "cw_prefill_host (streams)");
        ctx->copy_in_stream = a;
        ctx->copy_out_stream = b;
        for (int i = 0; i < 2 * kHostChunks + 1; ++i) {
            cudaEvent_t ev;
            e = cudaEventCreateWithFlags(&ev, cudaEventDisableTiming);
            if (e != cudaSuccess) return cuda_fail(ctx, (int)e, "cw_prefill_host (events)");
            ctx->events.push_back(ev);
        }
    }
    auto s_in = static_cast<cudaStream_t>(ctx->copy_in_stream), s_out = static_cast<cudaStream_t>(ctx->copy_out_stream);
    auto ev = [&](int i) { return static_cast<cudaEvent_t>(ctx->events[(size_t)i]); };
    // chunk boundaries (request indices) and chunk-local prefix sums
    const int nch = std::min<int>(kHostChunks, B);
    std::vector<int32_t> first((size_t)nch + 1, B), cu_local;
    first[0] = 0;
    for (int k = 1, r = 0; k < nch; ++k) {
        const int64_t target = (int64_t)T * k / nch;
        while (r < B && h_cu[r] < target) ++r;
        first[(size_t)k] = std::max(r, first[(size_t)k - 1]);
    }
    std::vector<int64_t> cu_off((size_t)nch);
    for (int k = 0; k < nch; ++k) {
        cu_off[(size_t)k] = (int64_t)cu_local.size();
        for (int r = first[(size_t)k]; r <= first[(size_t)k + 1]; ++r) cu_local.push_back(h_cu[r] - h_cu[first[(size_t)k]]);
    }
    // descriptors first (small), on the caller's stream; copies of activations wait for everything queued before us
    e = cudaMemcpyAsync(ws + w.cu, cu_local.data(), cu_local.size() * 4, cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(ws + w.nc, h_nc, (size_t)B * 4, cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(ws + w.tables, h_tables, (size_t)B * max_blocks * 4, cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaEventRecord(ev(2 * kHostChunks), s);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(s_in, ev(2 * kHostChunks), 0);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(s_out, ev(2 * kHostChunks), 0);
    if (e != cudaSuccess) return cuda_fail(ctx, (int)e, "cw_prefill_host (descriptors)");
    const size_t qrow = (size_t)c.num_q_heads * c.head_dim * 2, krow = (size_t)c.num_kv_heads * c.head_dim * 2;
    int64_t work_off = 0;
    for (int k = 0; k < nch; ++k) {
        const int r0 = first[(size_t)k], r1 = first[(size_t)k + 1], Bc = r1 - r0;
        const int64_t t0 = h_cu[r0], Tc = h_cu[r1] - t0;
        if (Bc == 0 || Tc == 0) continue;
        e = cudaMemcpyAsync(ws + w.q + t0 * qrow, (const char*)h_q + t0 * qrow, Tc * qrow, cudaMemcpyHostToDevice, s_in);
        if (e == cudaSuccess) e = cudaMemcpyAsync(ws + w.k + t0 * krow, (const char*)h_k + t0 * krow, Tc * krow, cudaMemcpyHostToDevice, s_in);
        if (e == cudaSuccess) e = cudaMemcpyAsync(ws + w.v + t0 * krow, (const char*)h_v + t0 * krow, Tc * krow, cudaMemcpyHostToDevice, s_in);
        if (e == cudaSuccess) e = cudaEventRecord(ev(k), s_in);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(s, ev(k), 0);
        if (e != cudaSuccess) return cuda_fail(ctx, (int)e, "cw_prefill_host (H2D)");
        const int32_t* d_cu = (const int32_t*)(ws + w.cu) + cu_off[(size_t)k];
        const int32_t* d_nc = (const int32_t*)(ws + w.nc) + r0;
        const int32_t* d_tab = (const int32_t*)(ws + w.tables) + (size_t)r0 * max_blocks;
        int rc = cw_append_kv(ctx, ws + w.q + t0 * qrow, ws + w.k + t0 * krow, ws + w.v + t0 * krow, ws + w.qr + t0 * qrow, d_cu, d_nc,
                              d_tab, max_blocks, Bc, (int32_t)Tc, stream);
        if (rc != CW_OK) return rc;
        int32_t* d_work = (int32_t*)(ws + w.work) + work_off;
        rc = cw_prefill_attn(ctx, ws + w.qr + t0 * qrow, ws + w.out + t0 * qrow, d_cu, d_nc, nullptr, d_tab, max_blocks, Bc,
                             (int32_t)Tc, std::min<int32_t>(max_q, (int32_t)Tc), max_kv, d_work, stream);
        if (rc != CW_OK) return rc;
        work_off += (cw::attn_work_ints(c, Bc, (int32_t)Tc) + 63) / 64 * 64;
        e = cudaEventRecord(ev(kHostChunks + k), s);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(s_out, ev(kHostChunks + k), 0);
        if (e == cudaSuccess) e = cudaMemcpyAsync((char*)h_out + t0 * qrow, ws + w.out + t0 * qrow, Tc * qrow, cudaMemcpyDeviceToHost, s_out);
        if (e != cudaSuccess) return cuda_fail(ctx, (int)e, "cw_prefill_host (D2H)");
    }
    e = cudaStreamSynchronize(s_out);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) return cuda_fail(ctx, (int)e, "cw_prefill_host (sync)");
    return CW_OK;
}

}  // extern "C"
