/* cacheweaver.h — C ABI of the B200-native prefix-cached prefill path of CacheWeaver
 * (arxiv/paper_2606_19667).  Citations are PAPER.md:<line> (+ section / algorithm) and DESIGN.md readings.
 *
 * The path:  cw_order -> cw_observe -> cw_lookup -> cw_append_kv -> cw_prefill_attn -> cw_release
 *
 * Conventions
 *   - every function returns int: CW_OK (0) or a negative CW_ERR_*; no exception crosses the ABI.
 *   - "host" / "device" is stated for every pointer.  The library allocates NO device memory: the caller
 *     (PyTorch in the binding) owns pools, tables, activations and the stream; `stream` is a cudaStream_t
 *     passed as void*.  All kernel launches are asynchronous on that stream.
 *   - out_* arrays are caller-allocated; request handles are library-owned until cw_release.
 *   - a context is not thread-safe: one context per caller thread.
 *   - block size is 16 tokens ("the token block size is 16 tokens").
 */
#ifndef CACHEWEAVER_H
#define CACHEWEAVER_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CW_BLOCK_SIZE 16

enum {
    CW_OK = 0,
    CW_ERR_INVALID = -1,     /* null pointer, k < 0, duplicate doc id, n <= 0, bad head config, bad sizes   */
    CW_ERR_NO_SPACE = -2,    /* not enough evictable blocks; library state is unchanged                     */
    CW_ERR_BAD_HANDLE = -3,  /* unknown / already released request handle                                   */
    CW_ERR_CUDA = -4         /* CUDA runtime / launch error; text via cw_last_error                         */
};

typedef struct cw_ctx cw_ctx; /* opaque, created by cw_create, freed by cw_destroy */

typedef struct {
    int32_t block_size;      /* must be 16                                                    */
    int32_t num_blocks;      /* NB: blocks in the paged KV pool                                             */
    int32_t num_q_heads;     /* Hq                                                                          */
    int32_t num_kv_heads;    /* Hkv, Hq % Hkv == 0 (GQA group g = Hq/Hkv)                                   */
    int32_t head_dim;        /* D in {64, 128}                                                              */
    int32_t max_position;    /* rows of the RoPE table = largest prompt length accepted                     */
    double  rope_theta;      /* RoPE base (reading c4)                                            */
    int32_t recency_window;  /* H: isCached(node) <=> seq - last_seq < H           */
    int32_t eager_register;  /* 1: new full blocks enter the prefix index inside cw_lookup; 0: at release    */
    uint64_t hash_salt;      /* parent hash of block 0 (reading c2)                               */
    void*   k_pool;          /* device, caller-owned, cw_pool_bytes() bytes, bf16, layout: see cw_pool_offset */
    void*   v_pool;          /* device, caller-owned, same size/layout                                      */
    void*   rope_table;      /* device, caller-owned, max_position*(D/2)*2 fp32 {cos,sin}; FILLED by cw_create.
                                may be NULL together with k_pool/v_pool for a host-only context (no kernels) */
    int32_t device;          /* CUDA device ordinal (ignored for a host-only context)                       */
    int32_t index_key_bits;  /* 0 or >= 64: the prefix index is keyed by the whole 64-bit chain hash; 1..63: by its low bits only.
                                Every index entry is also checked against a second 64-bit chain salted with a per-context random
                                secret, so serving another prompt's KV takes a simultaneous collision of two independent 64-bit
                                hashes, one of them secretly salted (a colliding block is simply not cached).  This is a
                                probabilistic safeguard built from non-cryptographic mixing, not a proof against an adversary who
                                can observe hits.  Small values make key collisions frequent (used by the tests of that property). */
} cw_config;

typedef struct {
    int64_t requests;        /* successful non-peek lookups                                                 */
    int64_t hit_blocks;      /* sum of m over those lookups                                                 */
    int64_t miss_blocks;     /* sum of ceil(n/16) - m                                                       */
    int64_t evictions;       /* hashed blocks whose index entry was dropped by allocation                   */
    int64_t trie_nodes;      /* live trie nodes (root excluded)                                             */
    int64_t order_probes;    /* child probes of the last cw_order call (<= k(k+1)/2)          */
    int64_t free_blocks;     /* current length of the LRU free list                                         */
    int64_t seq;             /* number of cw_observe calls so far                                           */
    /* predicted vs actual reusable prefix ("the trie can predict reuse for a path whose blocks were already
     * evicted"), summed over the requests admitted by cw_admit_batch and the calls of cw_feedback since cw_create/cw_reset: */
    int64_t predicted_prefix_docs;   /* sum of l(O,T)                                                        */
    int64_t actual_prefix_docs;      /* sum of the leading documents served from the cache (cw_matched_docs) */
    int64_t over_predicted_docs;     /* sum of max(0, predicted - actual)                                    */
    int64_t stale_marks;             /* trie nodes marked stale (cw_mark_stale, cw_feedback, the residency-aware arm)  */
    /* work the admitted requests ask of the device, summed over successful cw_lookup / cw_extend calls since cw_create / cw_reset
     * (only the uncached suffix is prefilled): */
    int64_t prompt_tokens;           /* sum of n                                                              */
    int64_t suffix_tokens;           /* sum of n - n_cached (+ the tokens appended by cw_extend)              */
    int64_t attn_flops;              /* sum of 4*Hq*D*[n(n+1)/2 - c(c+1)/2]: algorithmic flops of cw_prefill_attn */
    int64_t append_bytes;            /* suffix_tokens * (2*Hq*D*2 + 4*Hkv*D*2 + 4): algorithmic bytes of cw_append_kv */
} cw_stats_t;

/* ---- lifetime ---------------------------------------------------------------------------------------- */
/* Validates cfg, builds host state (trie, index, LRU list 0..NB-1), and — unless host-only — computes the
 * RoPE {cos,sin} table in fp64 on the host, rounds to fp32 and copies it to cfg->rope_table (synchronous). */
int  cw_create(const cw_config* cfg, cw_ctx** out);
void cw_destroy(cw_ctx* ctx);
const char* cw_strerror(int code);
const char* cw_last_error(cw_ctx* ctx);  /* text of the last CW_ERR_CUDA / CW_ERR_INVALID on this context */
int  cw_stats(cw_ctx* ctx, cw_stats_t* out);
/* bytes of ONE pool tensor (K or V): NB * Hkv * 16 * D * 2 */
int64_t cw_pool_bytes(const cw_config* cfg);
/* element offset (in bf16 elements) inside a pool tensor of element (block, kv_head, token-in-block t, dim d).
 * The in-block layout is the tcgen05 "canonical 128B-swizzled" tile so one (block, kv head) run of 16*D*2 bytes
 * is moved by ONE bulk copy and consumed by the MMA without re-layout:
 *   off = ((block*Hkv + kv_head) * 16*D) + (t/8)*(8*D) + (d/64)*512 + (t%8)*64 + ((((d%64)/8) ^ (t%8))*8) + d%8 */
int64_t cw_pool_offset(const cw_config* cfg, int32_t block, int32_t kv_head, int32_t t, int32_t d);

/* element offset (bf16 elements, relative to the request's first element q_begin*Hq*D) of (suffix token tok, query
 * head, dim d) inside q_roped, for a request with s suffix tokens.  q_roped is the intermediate between cw_append_kv
 * and cw_prefill_attn and is stored TILE-PACKED so that the attention kernel loads a Q tile with one bulk copy per
 * 64-dim half and feeds it to the MMA without re-layout.  With g = Hq/Hkv, tpt = 128/g tokens per tile:
 *   kvh = head/g, t = tok/tpt, row = (tok%tpt)*g + head%g, rows = min(tpt, s - t*tpt)*g
 *   off = kvh*s*g*D + t*(tpt*g)*D + (d/64)*rows*64 + row*64 + ((((d%64)/8) ^ (row%8))*8) + d%8
 * i.e. a permutation of the request's own [s, Hq, D] slice. */
int64_t cw_q_roped_offset(const cw_config* cfg, int32_t s, int32_t tok, int32_t head, int32_t d);

/* ---- ordering, host (PAPER.md:57 knowledge tree; Algorithm 1) ------------------------- */
/* Algorithm 1: doc_ids[k] in retrieval rank (host, distinct) -> out_order[k] (host); *out_pred_prefix_docs =
 * l(O,T), the depth of the cached trie path followed.  k == 0 is OK (empty order).
 * Pure: does not modify the tree.  Duplicate ids -> CW_ERR_INVALID (D is a set). */
int cw_order(cw_ctx* ctx, const int64_t* doc_ids, int32_t k, int64_t* out_order, int32_t* out_pred_prefix_docs);
/* l(O,T) of a given order without reordering it (retrieval-order arm). */
int cw_predict(cw_ctx* ctx, const int64_t* order, int32_t k, int32_t* out_prefix_docs);
/* "After a request finishes, its ordered document sequence is inserted": seq += 1, create the
 * path, stamp last_seq on every node of it; nodes outside the recency window are pruned lazily. */
int cw_observe(cw_ctx* ctx, const int64_t* ordered_doc_ids, int32_t k);

/* Ordering arms the paper compares with (Table 4; readings in DESIGN.md §2):
 *   CW_ARM_RETRIEVAL  the retrieval order as given
 *   CW_ARM_GREEDY     Algorithm 1 (cw_order)
 *   CW_ARM_SORTED     ascending document id ("lexicographic sorting", a canonical query-independent order)
 *   CW_ARM_RECENCY    documents served most recently first (index of the last cw_observe call containing the document,
 *                     descending; never-served documents last; ties keep retrieval rank)
 *   CW_ARM_EXHAUSTIVE of all k! orders (k <= 8) the one whose prompt matches the most resident blocks (peek lookups on
 *                     the real block index); first maximiser in lexicographic order of retrieval-rank indices.  Needs the
 *                     tokens: doc_tokens [num_docs, doc_len], query_tokens [q_len] (HOST; may be NULL for the other arms).
 * out_order[k] (host); *out_pred_prefix_docs = l(O,T) of the chosen order (may be NULL).  Pure: no state change (except
 * CW_ARM_GREEDY_RESIDENT, below).
 *   CW_ARM_GREEDY_FEEDBACK  Algorithm 1; inside cw_admit_batch the engine's answer is fed back after every lookup
 *                     (cw_feedback): NEXT-1, PAPER.md:129-141 with the direct cache-state signal instead of TTFT
 *   CW_ARM_GREEDY_RESIDENT  Algorithm 1 whose line 6 also asks the block index whether the prefix O + [d] is resident
 *                     (an incremental peek: every full 16-token block completed by the documents placed so far plus d);
 *                     a recency-cached child that is not resident is marked stale and the scan goes on.  Needs doc_tokens.
 *                     NOT pure: it marks trie nodes stale (it never changes the block manager).  PAPER.md:314. */
enum { CW_ARM_RETRIEVAL = 0, CW_ARM_GREEDY = 1, CW_ARM_SORTED = 2, CW_ARM_RECENCY = 3, CW_ARM_EXHAUSTIVE = 4,
       CW_ARM_GREEDY_FEEDBACK = 5, CW_ARM_GREEDY_RESIDENT = 6 };
int cw_order_arm(cw_ctx* ctx, int32_t arm, const int64_t* doc_ids, int32_t k, const int32_t* doc_tokens, int32_t num_docs,
                 int32_t doc_len, const int32_t* query_tokens, int32_t q_len, int64_t* out_order, int32_t* out_pred_prefix_docs);

/* Cache-state feedback ("when the trie predicts a long reusable prefix but the
 * observed TTFT stays close to a cold request, the supposed cached path is probably gone, so we mark it stale and stop
 * relying on it"; here the engine's own answer replaces the TTFT heuristic).  Reading:
 *   cw_mark_stale: the document prefix order[0..resident_docs-1] was resident, order[0..resident_docs] was not: the trie
 *     node at depth resident_docs+1 on that path gets stale_epoch = seq (no-op if the path does not exist).  A node is
 *     usable iff it is recency-cached AND it was served after the latest stale mark on itself or on any node above it
 *     on the walk — blocks are chained to their prefix and released deepest-first, so what hangs below an evicted
 *     prefix is gone as well.  cw_observe re-stamps the served path, which makes exactly that path usable again.
 *   cw_feedback(order, predicted, actual): if predicted > actual -> cw_mark_stale(order, actual); both also feed the
 *     predicted-vs-actual counters of cw_stats.  Call it after cw_lookup and before cw_observe. */
int cw_mark_stale(cw_ctx* ctx, const int64_t* order, int32_t k, int32_t resident_docs);
int cw_feedback(cw_ctx* ctx, const int64_t* order, int32_t k, int32_t predicted_docs, int32_t actual_docs);
/* The same from the engine's raw answer, so that the caller does no arithmetic of the method:
 *   cw_matched_docs: *out_docs = number of leading documents of a prompt served from the cache, given doc_ends[k] (HOST;
 *     doc_ends[j] = prompt position just past the segment of the j-th document: positive, non-decreasing, <= n_tokens — any
 *     layout: headers, ragged documents), the lookup's n_cached and the prompt length n_tokens.  Reading: a
 *     document counts when every FULL 16-token block up to its end lies inside the cached tokens (the block it shares with
 *     the next segment cannot match on its own), measured against what cw_lookup can return at most, 16*floor((n-1)/16): a
 *     document ending in the block of the last prompt token is not punished for the cap.  Pure.
 *   cw_feedback_tokens = cw_matched_docs + cw_feedback(order, predicted_docs, that count); *out_actual_docs (may be NULL)
 *     receives the count.  cw_admit_batch applies the same rule with doc_ends[j] = (j+1)*doc_len. */
int cw_matched_docs(cw_ctx* ctx, const int32_t* doc_ends, int32_t k, int32_t n_cached, int32_t n_tokens, int32_t* out_docs);
int cw_feedback_tokens(cw_ctx* ctx, const int64_t* order, int32_t k, int32_t predicted_docs, const int32_t* doc_ends,
                       int32_t n_cached, int32_t n_tokens, int32_t* out_actual_docs);

/* ---- prefix cache, host (PAPER.md:33 chained block hashes; PAPER.md:129 block eviction) -------------- */
/* chain[i] = FNV1a64(LE64(chain[i-1]) || 16 x LE32(token)), chain[-1] = hash_salt, i < floor(n/16). */
int cw_hash_chain(cw_ctx* ctx, const int32_t* tokens, int32_t n, uint64_t* out_chain);
/* Longest resident prefix + pin + allocate + evict + register (reading c3).
 *   tokens[n] host.  m = leading chain hashes found in the index, capped at floor((n-1)/16).
 *   peek_only = 1: only *out_n_cached = 16*m is written; no state change, out_req/out_block_table untouched.
 *   else: out_block_table[ceil(n/16)] (host) receives the block ids, *out_req the handle, *out_n_cached = 16*m.
 *   CW_ERR_NO_SPACE leaves every piece of state unchanged. */
int cw_lookup(cw_ctx* ctx, const int32_t* tokens, int32_t n, int32_t peek_only,
              int64_t* out_req, int32_t* out_block_table, int32_t* out_n_cached);
/* Unpin; blocks whose refcount reaches 0 go to the LRU tail in REVERSE block order. */
int cw_release(cw_ctx* ctx, int64_t req);
/* NEXT-4 (PAPER.md:253-283 continuous batching): the live request `req` grows by new_tokens[n_new]
 * (host) — the next chunk of a chunked prefill, or generated tokens.  Blocks for the longer sequence are popped from the
 * LRU head as in cw_lookup (CW_ERR_NO_SPACE leaves everything unchanged); with eager registration every block the new
 * tokens complete is hashed, chained to the request's last full block, and entered into the prefix index (the formerly
 * partial last block included).  out_block_table[cap] (host) receives the whole table, *out_n_blocks its length.
 * The K/V of the new tokens are written by the next cw_append_kv / cw_prefill_requests of this request, whose n_cached
 * is the number of tokens already in the pool (no longer a multiple of 16). */
int cw_extend(cw_ctx* ctx, int64_t req, const int32_t* new_tokens, int32_t n_new, int32_t* out_block_table, int32_t cap,
              int32_t* out_n_blocks);
/* Back to the state right after cw_create: empty knowledge tree, empty prefix index, LRU list 0..NB-1, no live
 * requests, statistics zeroed.  Pools and the RoPE table are untouched (old KV is unreachable: nothing is indexed). */
int cw_reset(cw_ctx* ctx);
/* Admission of a wave in ONE call: steps a1..a6 (+a2) for requests r = 0..B-1, in order (DESIGN.md reading
 * "requests of a batch are admitted sequentially on the host"):
 *     O_r = cw_order_arm(arm = reorder, doc_ids[r])      (0 = retrieval order, 1 = Algorithm 1, 2.. = the other arms;
 *                                                          arms 5 and 6 also call cw_feedback after the lookup)
 *     tokens = doc_tokens[O_r[0]] || ... || doc_tokens[O_r[k-1]] || query_tokens[r];   (prompt assembly)
 *     (req, table, n_cached) = cw_lookup(tokens);  cw_observe(O_r)
 * All pointers HOST.  doc_ids [B,k] in retrieval rank; doc_tokens [num_docs, doc_len]; query_tokens [B, q_len];
 * out_orders [B,k]; out_pred_prefix_docs [B]; out_reqs [B]; out_block_tables [B, max_blocks] (unused tail entries
 * are set to 0; max_blocks >= ceil((k*doc_len+q_len)/16)); out_n_cached [B]; out_cu_seqlens_q [B+1] (prefix sums of
 * the suffix lengths n - n_cached).  Admission stops at the first request that does not fit (CW_ERR_NO_SPACE; that
 * request and all later ones leave the state unchanged); *out_admitted = number admitted, return value CW_OK unless
 * an argument is invalid (doc id outside [0,num_docs), duplicate ids, unknown arm, ...): every row is checked before
 * the first request is admitted, so CW_ERR_INVALID leaves the state unchanged (*out_admitted = 0). */
int cw_admit_batch(cw_ctx* ctx, const int64_t* doc_ids, int32_t B, int32_t k, int32_t reorder,
                   const int32_t* doc_tokens, int32_t num_docs, int32_t doc_len,
                   const int32_t* query_tokens, int32_t q_len,
                   int64_t* out_orders, int32_t* out_pred_prefix_docs, int64_t* out_reqs,
                   int32_t* out_block_tables, int32_t max_blocks, int32_t* out_n_cached,
                   int32_t* out_cu_seqlens_q, int32_t* out_admitted);
/* cw_release for reqs[0..B-1] in order; stops at the first bad handle. */
int cw_release_batch(cw_ctx* ctx, const int64_t* reqs, int32_t B);
/* Copy the LRU free list head->tail into out[cap] (host); returns its length via *out_len (testing aid). */
int cw_free_list(cw_ctx* ctx, int32_t* out, int32_t cap, int32_t* out_len);

/* ---- device work (async on `stream`) ----------------------------------------------------------------- */
/* Batch of B requests; request r owns suffix rows cu_seqlens_q[r]..cu_seqlens_q[r+1]-1 (T rows in total),
 * row i of request r sits at absolute prompt position n_cached[r] + i; n_cached[r] = tokens of the request already in
 * the pool (16 * matched blocks after cw_lookup; any value for a later chunk of a chunked prefill or a decode row,
 * SURVEY.md 8(f) NEXT-4).  All d_* pointers are DEVICE int32.
 * d_block_tables is [B, max_blocks_per_req] row-major.
 *
 * cw_append_kv — fused RoPE + KV scatter (kernel 1):  for each suffix token at position p
 *     q_roped = RoPE(q, p);  pool_K[slot(p)] = RoPE(k, p);  pool_V[slot(p)] = v;
 *     slot(p) = (block_table[p/16], p%16)          (DESIGN.md c4 split-half RoPE)
 *   q [T,Hq,D], k,v [T,Hkv,D]: device bf16, row-major contiguous.  q_roped: device bf16, T*Hq*D elements, request r
 *   owns the slice starting at cu_seqlens_q[r]*Hq*D, laid out as cw_q_roped_offset() says; it must NOT alias q
 *   (q is read through the non-coherent path).  The descriptors are on the device, so they cannot be rejected by this call:
 *   a token whose position is >= max_position or >= 16*max_blocks_per_req, or whose table entry is not in [0, NB), is
 *   SKIPPED (nothing of it is written: no clamped rotation, no store outside the pool), and so is a row that does not lie
 *   inside its request's slice of [0, T) (non-monotone cu_seqlens_q); cw_prefill_attn flags a request that is too long or a
 *   table entry outside the pool in its work header.  The pools must have been
 *   zero-filled once by the caller (stale slots of a partially filled block must hold finite values). */
int cw_append_kv(cw_ctx* ctx, const void* q, const void* k, const void* v, void* q_roped,
                 const int32_t* d_cu_seqlens_q, const int32_t* d_n_cached, const int32_t* d_block_tables,
                 int32_t max_blocks_per_req, int32_t B, int32_t T, void* stream);

/* cw_prefill_attn — varlen paged causal GQA attention of the suffix rows (kernel 2):
 *     o[row p, head h] = sum_{j<=p} softmax_j(q'_p . k'_j / sqrt(D)) v_j, kv head = h / g, keys j read from the
 *     pool through the block table (cached prefix j < n_cached and the blocks just written by cw_append_kv).
 *   Fully asynchronous: every descriptor is a DEVICE pointer and nothing is read on the host.  The call enqueues a
 *   one-CTA schedule kernel (request descriptors -> list of work items, longest request first) and the persistent
 *   attention kernel (one CTA per SM) on `stream`.
 *   d_kv_len [B]: device, kv_len[r] = n_cached[r] + suffix length; may be NULL (it is redundant and only cross-checked).
 *   max_q_len / max_kv_len: upper bounds on the suffix length / kv length of any request of the batch (host values;
 *   max_kv_len <= 16 * max_blocks_per_req and <= max_position).
 *   d_work: DEVICE int32 scratch of cw_attn_work_ints(ctx, B, T) ints, caller-owned, written by this call.  After the
 *   stream has run the call: d_work[1] != 0 is an error.  Bit 0: a request descriptor was invalid (negative lengths,
 *   lengths beyond the stated maxima, kv_len mismatch) and that request produced no output; bit 2: one of the first
 *   ceil(kv_len/16) block table entries of a request was outside [0, NB) — that request produced no output either and no
 *   memory outside the pool was touched (cw_append_kv had skipped the tokens of such an entry; with B > 2048 the whole
 *   batch is dropped).  d_work[2] counts the
 *   softmax chunks that left the speculative path (statistics); d_work[3] is the number of work items.
 *   q_roped: as written by cw_append_kv (tile-packed); out [T,Hq,D] device bf16 row-major.
 *   (SURVEY.md 8(b) lists this signature without d_work; the scratch is passed in because the library allocates no
 *   device memory.) */
int64_t cw_attn_work_ints(cw_ctx* ctx, int32_t B, int32_t T);
int cw_prefill_attn(cw_ctx* ctx, const void* q_roped, void* out,
                    const int32_t* d_cu_seqlens_q, const int32_t* d_n_cached, const int32_t* d_kv_len,
                    const int32_t* d_block_tables, int32_t max_blocks_per_req, int32_t B, int32_t T,
                    int32_t max_q_len, int32_t max_kv_len, int32_t* d_work, void* stream);

/* The two launches of cw_prefill_attn, separately.  cw_attn_schedule (descriptors -> work list in d_work) reads neither
 * q_roped nor the pools, so it can be enqueued in front of cw_append_kv or, on a second stream, beside it; cw_attn_run (the
 * attention kernel over that list) must come after both.  cw_prefill_attn(...) == cw_attn_schedule(...) + cw_attn_run(...)
 * on one stream; arguments and error behaviour as described there.  B and T of the two calls must be equal. */
int cw_attn_schedule(cw_ctx* ctx, const int32_t* d_cu_seqlens_q, const int32_t* d_n_cached, const int32_t* d_kv_len,
                     const int32_t* d_block_tables, int32_t max_blocks_per_req, int32_t B, int32_t T,
                     int32_t max_q_len, int32_t max_kv_len, int32_t* d_work, void* stream);
int cw_attn_run(cw_ctx* ctx, const void* q_roped, void* out, const int32_t* d_block_tables, int32_t max_blocks_per_req,
                int32_t B, int32_t T, int32_t* d_work, void* stream);

/* cw_prefill_attn_static — cw_prefill_attn for callers that cannot hand over the d_work scratch because they cannot
 * allocate device memory: code that runs inside somebody else's process and is given only the tensors of the operation (an
 * inference server's custom-op slot, a plugin), code inside a region where touching the allocator is forbidden (after the
 * warm-up of a latency-critical serving loop, inside someone else's memory-pool lock), or a plain C caller that links no
 * allocator at all.  The work list lives in a fixed array of CW_STATIC_WORK_INTS ints (2 MiB) that is part of the library
 * image: every GPU the process uses through this library holds those 2 MiB from the moment the library's CUDA module is
 * loaded there until the process exits.  The call itself allocates and frees nothing (no cudaMalloc / cudaFree, no library
 * routine that allocates).
 *   Arguments as for cw_prefill_attn, without d_work.  d_status: DEVICE int32[4], caller-owned OUTPUT, may be NULL; after
 *   the stream has run the call it holds the first four ints of the work header (see cw_prefill_attn: [1] error flags,
 *   [2] exact-path fallbacks, [3] number of work items).
 *   Limit: cw_attn_work_ints(ctx, B, T) <= CW_STATIC_WORK_INTS, i.e. (T / (2*(128/g)) + B) * Hkv <= 65535 work items with
 *   g = Hq/Hkv (config 2 of BASELINE.json needs about 10 k; a 64-request wave of the 8B shape fits up to ~520 k suffix tokens).  A
 *   larger batch is rejected with CW_ERR_INVALID ("... exceeds the static work list ...") before anything is launched;
 *   split the wave or use cw_prefill_attn.
 *   Set-up: the first call on a device looks up the array's device address (cudaGetSymbolAddress) and keeps it; the
 *   context's device (cfg.device) must be the current device of the calling thread, else CW_ERR_CUDA.  Make that first call
 *   per device before any stream capture begins.
 *   Sharing: there is ONE array per device, shared by every context and every call, and it keeps what the last call left
 *   in it.  Each call rewrites all it reads (the schedule kernel resets the claim counter and the statistics and writes
 *   the item count before the attention kernel starts), so consecutive calls on one stream are safe.  Two calls that can
 *   run on the GPU at the same time (different streams without an event between them, two host threads) race on the
 *   array and produce garbage: order them, or give all but one of them a d_work of their own through cw_prefill_attn. */
#define CW_STATIC_WORK_INTS (8 * 65536)
int cw_prefill_attn_static(cw_ctx* ctx, const void* q_roped, void* out,
                           const int32_t* d_cu_seqlens_q, const int32_t* d_n_cached, const int32_t* d_kv_len,
                           const int32_t* d_block_tables, int32_t max_blocks_per_req, int32_t B, int32_t T,
                           int32_t max_q_len, int32_t max_kv_len, int32_t* d_status, void* stream);

/* cw_prefill_requests — steps a7 + a8 for a wave of admitted requests in ONE call: the descriptors (cu_seqlens_q,
 * n_cached, block tables) are taken from the request handles reqs[0..B-1] (HOST, as returned by cw_lookup /
 * cw_admit_batch, in batch order; a request's rows are its tokens not yet written to the pool: the uncached suffix after
 * cw_lookup, the appended tokens after cw_extend — prefill suffixes, prefill chunks and decode rows can share a call), written to a library-owned pinned staging slot, copied to d_ws with one
 * asynchronous H2D copy, and cw_append_kv + cw_prefill_attn are enqueued on `stream` (for waves of >= 4096 rows the schedule
 * kernel runs on a library-owned side stream beside cw_append_kv, forked from and joined back into `stream` with events:
 * for the caller everything is still ordered on `stream`).  The call does not wait for the
 * device, with one bound: the staging ring has 4 slots, so a call blocks on the host until the descriptor copy of the
 * fourth-last call has completed (only a caller that runs more than four waves ahead of the GPU ever waits).
 *   The handles advance (their rows count as written) only when the copy and both kernels were enqueued successfully: after
 *   any error the same call can be repeated.  A handle listed twice -> CW_ERR_INVALID.
 *   q [T,Hq,D], k, v [T,Hkv,D], q_roped, out: device bf16 as in cw_append_kv / cw_prefill_attn; T must equal the sum
 *   of the requests' suffix lengths.  max_blocks_per_req >= the largest block-table length of the wave.
 *   d_ws: device scratch of cw_prefill_requests_ws_bytes() bytes, caller-owned (descriptors at offset 0: cu [B+1],
 *   n_cached [B], tables [B, max_blocks_per_req]; then the attention work list, 256-byte aligned).  The work list of
 *   the call starts at byte offset cw_prefill_requests_work_offset(); its header reads as described at cw_prefill_attn). */
int64_t cw_prefill_requests_ws_bytes(cw_ctx* ctx, int32_t B, int32_t T, int32_t max_blocks_per_req);
int64_t cw_prefill_requests_work_offset(cw_ctx* ctx, int32_t B, int32_t max_blocks_per_req);
int cw_prefill_requests(cw_ctx* ctx, const int64_t* reqs, int32_t B, const void* q, const void* k, const void* v,
                        void* q_roped, void* out, int32_t T, int32_t max_blocks_per_req, void* d_ws, void* stream);

/* cw_gather_kv — export: pool -> plain row-major k_out, v_out [n, Hkv, D] bf16 (device) for one block table
 * (device int32 [ceil(n/16)]).  Used by tests and by callers that want the cached KV in a plain layout. */
int cw_gather_kv(cw_ctx* ctx, const int32_t* d_block_table, int32_t n, void* k_out, void* v_out, void* stream);

/* cw_prefill_host — the same path with HOST buffers (end-to-end entry point).  The batch is cut into up to 16 request
 * chunks of about equal token count and pipelined: H2D of chunk i+1 (library-owned copy stream), cw_append_kv +
 * cw_prefill_attn of chunk i (on `stream`, in request order), D2H of chunk i-1 (second copy stream); all of it is
 * enqueued without blocking, then the call waits until everything has completed (`stream` and the copy streams).  q, k, v, out are staged in the
 * caller-owned device workspace `d_ws` (cw_prefill_host_ws_bytes bytes).  Host buffers should be pinned (pageable
 * memory works but serialises the copies).  h_block_tables is [B, max_blocks_per_req].  The two copy streams and their
 * events are created on first use and destroyed by cw_destroy. */
int64_t cw_prefill_host_ws_bytes(cw_ctx* ctx, int32_t B, int32_t T, int32_t max_blocks_per_req);
int cw_prefill_host(cw_ctx* ctx, const void* h_q, const void* h_k, const void* h_v, void* h_out,
                    const int32_t* h_cu_seqlens_q, const int32_t* h_n_cached, const int32_t* h_block_tables,
                    int32_t max_blocks_per_req, int32_t B, int32_t T, void* d_ws, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* CACHEWEAVER_H */
