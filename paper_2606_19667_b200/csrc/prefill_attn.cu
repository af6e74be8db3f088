// Kernel 2: varlen paged causal GQA flash-attention prefill (cw_prefill_attn).  sm_100a, tcgen05 + TMEM + bulk TMA.
//
//   o[row p, head h] = sum_{j<=p} softmax_j(q'_p . k'_j / sqrt(D)) v_j ,  kv head = h / g
//
// Work item = (request r, kv head, 2 consecutive Q tiles).  A Q tile holds tpt = 128/g suffix tokens x the g query
// heads that share the kv head, packed into the M dimension (row = token*g + head), so one K/V tile read feeds all g
// heads and both Q tiles (M = 256 per CTA), and a short query-only suffix still fills the MMA.
//
// Persistent CTAs (one per SM, 512 threads = 4 warpgroups) claiming items from a host-built list with an atomic counter,
// warp-specialised, mbarrier pipelines only; registers are re-balanced with setmaxnreg (softmax 192, epilogue 64, MMA+loader 64):
//   warps 0-3   softmax + lazy rescale of Q tile 0 (thread i owns TMEM lane i = packed row i)
//   warps 4-7   the same for Q tile 1 — the two groups ping-pong: while one does exp on S_w, the tensor core runs the
//               other tile's PV and next QK^T
//   warps 8-11  epilogue of both tiles: O_w / l_w -> bf16 -> global, so the softmax groups go straight on to the next item
//   warp  12    MMA issuer: S_w = Q_w K^T (SS) and O_w += P_w V (TS: P is read from TMEM, where the softmax group wrote
//               it as bf16 over the first half of S_w); owns TMEM alloc/dealloc (512 columns: S0 S1 O0 O1)
//   warp  13    loader: Q tiles (q_roped is stored tile-packed and pre-swizzled by cw_append_kv: one bulk copy per
//              64-dim half tile) and K/V tiles (one bulk copy per 16-token pool block per operand, gathered through
//              the block table; pool blocks are pre-swizzled in the UMMA canonical layout) into a multi-stage ring
// Softmax is online in fp32 with exp2 and a lazy rescale: O/l are only rescaled when the running max grows by more
// than 2^8 (exact: the final normalisation uses the same reference max for O and l).
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include <algorithm>

#include "cw_internal.h"
#include "ptx_sm100.cuh"

namespace cw {

namespace {

constexpr int kTileM = 128;          // MMA M (TMEM lanes); a Q tile uses the first tpt*g of them
constexpr int kTileN = 128;          // keys per KV tile (8 pool blocks)
constexpr int kThreads = 512;
constexpr int kWorkInts = 8;         // ints per work item
constexpr float kRescaleThreshold = 8.0f;   // log2 units
constexpr float kSpecLimit = 65536.f;       // bound on a row sum taken against a stale reference maximum

template <int D>
struct Smem {
    static constexpr int kQBytes = kTileM * D * 2;            // one Q tile
    static constexpr int kKVBytes = kTileN * D * 2;           // one K or V tile
    static constexpr int kStages = D == 128 ? 5 : 8;          // K/V ring slots (a K tile or a V tile each)
    static constexpr int kQ = 0;
    static constexpr int kRing = kQ + 2 * kQBytes;
    static constexpr int kBar = kRing + kStages * kKVBytes;   // mbarriers (8 B each), then the TMEM slot
    static constexpr int kL = kBar + 512;                     // l_sum hand-off softmax -> epilogue: float [2][128]
    static constexpr int kSched = kL + 1024;                  // item ring: kSchedSlots x 8 ints, filled by the loader warp
    static constexpr int kTotal = kSched + 128;
};

// barrier slots (ring FULL[s] at BAR_RING + s, EMPTY[s] at BAR_RING + kStages + s)
enum { BAR_Q_FULL = 0, BAR_Q_EMPTY = 2, BAR_S_FULL = 4, BAR_P_FULL = 6, BAR_PV_DONE = 8, BAR_O_EMPTY = 10, BAR_L_FULL = 12,
       BAR_L_EMPTY = 14, BAR_SCHED_FULL = 16, BAR_SCHED_EMPTY = 20, BAR_RING = 24 };
constexpr int kSchedSlots = 4;
constexpr int kSchedConsumers = 13;  // warps that read every item: MMA (1) + softmax (8) + epilogue (4)

// Work item, 8 ints: {pos0, ntok0, ntok1, tok0 | r, kvh, q_off16, 0}.  The first int4 is all the softmax and MMA warps need.
//   pos0: absolute position of the first token; ntok0/1: tokens of Q tile 0/1; tok0: index of the first token in [0,T);
//   q_off16: offset of Q tile 0 inside q_roped in 16-byte units.
struct Item {
    int pos0, ntok0, ntok1, tok0, r, kvh, q_off16;
};
// volatile: the prefetch of the next item must stay where it is written (ptxas otherwise sinks it next to its first use)
__device__ __forceinline__ int4 ld_item_half(const int4* p) {
    int4 v;
    asm volatile("ld.global.nc.v4.s32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
    return v;
}
__device__ __forceinline__ Item load_item(const int4* __restrict__ work, int idx) {
    const int4 a = ld_item_half(work + 2 * idx), b = ld_item_half(work + 2 * idx + 1);
    return Item{a.x, a.y, a.z, a.w, b.x, b.y, b.z};
}

// exp2 on the FMA pipe for a share of the scores (the MUFU unit, 16 exp2 / clk / SM, is the softmax bottleneck):
// 2^x = 2^round(x) * 2^f, f = x - round(x) in [-0.5, 0.5]; 2^f by a degree-3 polynomial (max rel. error 7.8e-5, P is
// rounded to bf16 = 3.9e-3 afterwards); round(x) through the 1.5*2^23 magic constant, spliced into the exponent field.
#ifndef CW_POLY_PERIOD
#define CW_POLY_PERIOD 8
#define CW_POLY_COUNT 1
#endif
constexpr int kPolyPeriod = CW_POLY_PERIOD;   // of every kPolyPeriod score pairs ...
constexpr int kPolyCount = CW_POLY_COUNT;     // ... this many use the polynomial
__device__ __forceinline__ float2 exp2_poly2(float2 x) {
    const float kMagic = 12582912.f;
    x.x = fmaxf(x.x, -125.f);
    x.y = fmaxf(x.y, -125.f);
    const float2 t = __fadd2_rn(x, make_float2(kMagic, kMagic));
    const float2 r = __fadd2_rn(t, make_float2(-kMagic, -kMagic));
    const float2 f = __fadd2_rn(x, make_float2(-r.x, -r.y));
    float2 p = __ffma2_rn(make_float2(0.05508868396282196f, 0.05508868396282196f), f,
                          make_float2(0.24260404706001282f, 0.24260404706001282f));
    p = __ffma2_rn(p, f, make_float2(0.6932762265205383f, 0.6932762265205383f));
    p = __ffma2_rn(p, f, make_float2(0.9999289512634277f, 0.9999289512634277f));
    p.x = __int_as_float(__float_as_int(p.x) + (__float_as_int(t.x) << 23));
    p.y = __int_as_float(__float_as_int(p.y) + (__float_as_int(t.y) << 23));
    return p;
}

__device__ __forceinline__ int tiles_for(int nkv) { return (nkv + kTileN - 1) / kTileN; }

}  // namespace

#ifdef CW_PROF   // experiments only: cycle counters per CTA
__device__ unsigned long long cw_prof_buf[256][8];
#endif

template <int D>
__global__ void __launch_bounds__(kThreads, 1) prefill_attn_kernel(
    const __nv_bfloat16* __restrict__ q_roped, __nv_bfloat16* __restrict__ out,
    const __nv_bfloat16* __restrict__ k_pool, const __nv_bfloat16* __restrict__ v_pool,
    const int32_t* __restrict__ tables, int max_blocks, int4* __restrict__ work, int num_items,
    int Hq, int Hkv, float scale_log2) {
    using L = Smem<D>;
    constexpr int NS = L::kStages;
    extern __shared__ __align__(1024) uint8_t smem[];
    const uint32_t sbase = ptx::smem_u32(smem);
    const uint32_t bars = sbase + L::kBar;
    auto bar = [&](int i) { return bars + 8u * (uint32_t)i; };
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + L::kBar + 8 * (BAR_RING + 2 * NS));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = Hq / Hkv;
    const int tpt = kTileM / g;          // tokens per Q tile
    const int R = tpt * g;               // rows of a full Q tile

    // Dynamic schedule: work[0].x is a counter (zeroed by the host with the list upload), items follow from work + 2.
    // The loader warp claims items with atomicAdd and publishes each descriptor through a small smem ring; every other
    // warp reads item #n from slot n % kSchedSlots (an item with ntok0 == 0 ends the stream).
    const int4* items = work + 2;
    auto get_item = [&](uint32_t n, bool full) {
        const uint32_t slot = n % kSchedSlots;
        ptx::mbar_wait(bar(BAR_SCHED_FULL + slot), (n / kSchedSlots) & 1u);
        const int4* p = reinterpret_cast<const int4*>(smem + L::kSched + slot * 32);
        const int4 a = p[0];
        int4 b = make_int4(0, 0, 0, 0);
        if (full) b = p[1];
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(bar(BAR_SCHED_EMPTY + slot));
        return Item{a.x, a.y, a.z, a.w, b.x, b.y, b.z};
    };

    if (threadIdx.x == 0) {
        for (int w = 0; w < 2; ++w) {
            ptx::mbar_init(bar(BAR_Q_FULL + w), 1);
            ptx::mbar_init(bar(BAR_Q_EMPTY + w), 1);
            ptx::mbar_init(bar(BAR_S_FULL + w), 1);
            ptx::mbar_init(bar(BAR_P_FULL + w), 128);
            ptx::mbar_init(bar(BAR_PV_DONE + w), 1);
            ptx::mbar_init(bar(BAR_O_EMPTY + w), 128);
            ptx::mbar_init(bar(BAR_L_FULL + w), 128);
            ptx::mbar_init(bar(BAR_L_EMPTY + w), 128);
        }
        for (int s = 0; s < kSchedSlots; ++s) {
            ptx::mbar_init(bar(BAR_SCHED_FULL + s), 1);
            ptx::mbar_init(bar(BAR_SCHED_EMPTY + s), kSchedConsumers);
        }
        for (int s = 0; s < 2 * NS; ++s) ptx::mbar_init(bar(BAR_RING + s), 1);
        ptx::fence_mbar_init();
    }
    if (warp == 12) ptx::tmem_alloc(ptx::smem_u32(tmem_slot), 512);
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    if (warp >= 12) {
        ptx::setmaxnreg_dec<64>();
        if (warp == 13) {
            // ================================ loader ================================
            // Ring order per item: K(0) V(0) K(1) V(1) ...; the item's two Q tiles are loaded after K(0), V(0) so that
            // the MMA warp can chain QK(0) of this item right behind the last PV of the previous one.
            constexpr uint32_t kBlockBytes = 16 * D * 2;
            uint32_t it = 0, qcnt0 = 0, qcnt1 = 0, n_item = 0;
            int* counter = reinterpret_cast<int*>(work);
            auto claim = [&]() {                          // lane 0 holds the claimed index
                int i = 0;
                if (lane == 0) i = atomicAdd(counter, 1);
                return i;
            };
            auto publish = [&](const Item& x, uint32_t n) {
                const uint32_t slot = n % kSchedSlots;
                ptx::mbar_wait(bar(BAR_SCHED_EMPTY + slot), ((n / kSchedSlots) & 1u) ^ 1u);
                if (lane == 0) {
                    int4* p = reinterpret_cast<int4*>(smem + L::kSched + slot * 32);
                    p[0] = make_int4(x.pos0, x.ntok0, x.ntok1, x.tok0);
                    p[1] = make_int4(x.r, x.kvh, x.q_off16, 0);
                    ptx::mbar_arrive(bar(BAR_SCHED_FULL + slot));      // release: the stores above are visible to waiters
                }
                __syncwarp();
            };
            const Item kEnd{0, 0, 0, 0, 0, 0, 0};
            int idx = __shfl_sync(0xffffffffu, claim(), 0);
            Item w = idx < num_items ? load_item(items, idx) : kEnd;
            publish(w, 0);
            int idx_next = __shfl_sync(0xffffffffu, claim(), 0);
            for (; w.ntok0 > 0; ++n_item) {
                // next item: descriptor load and the claim after it are issued now and consumed after this item's first loads
                const bool has_next = idx_next < num_items;
                Item nxt = kEnd;
                if (has_next) nxt = load_item(items, idx_next);
                const int claimed = claim();
                const int rows0 = w.ntok0 * g, rows1 = w.ntok1 * g;
                const int nkv = w.pos0 + w.ntok0 + w.ntok1;
                const int nt = tiles_for(nkv);
                const int32_t* table = tables + (size_t)w.r * max_blocks;
                auto load_ids = [&](int j) {
                    const int left = nkv - j * kTileN;
                    const int nb = left >= kTileN ? 8 : (left + 15) >> 4;
                    return lane < nb ? __ldg(table + j * 8 + lane) : 0;
                };
                auto load_kv = [&](int j, int blk) {
                    const int left = nkv - j * kTileN;
                    const int nblk = left >= kTileN ? 8 : (left + 15) >> 4;
                    const size_t src_off = ((size_t)blk * Hkv + w.kvh) * (16 * D);
#pragma unroll
                    for (int kv = 0; kv < 2; ++kv) {
                        const uint32_t s = it % NS, ph = (it / NS) & 1u;
                        ptx::mbar_wait(bar(BAR_RING + NS + s), ph ^ 1u);
#ifdef CW_EXP_NOLOAD   // timing experiment only (wrong results): K/V tiles are loaded for the first ring fill, then faked
                        if (it >= NS) {
                            if (lane == 0) ptx::mbar_arrive(bar(BAR_RING + s));
                            ++it;
                            continue;
                        }
#endif
                        if (lane == 0) ptx::mbar_arrive_expect_tx(bar(BAR_RING + s), kBlockBytes * (uint32_t)nblk);
                        __syncwarp();
                        if (lane < nblk)
                            ptx::bulk_g2s(sbase + L::kRing + s * L::kKVBytes + lane * kBlockBytes,
                                          (kv == 0 ? k_pool : v_pool) + src_off, kBlockBytes, bar(BAR_RING + s));
                        ++it;
                    }
                };
                int blk = load_ids(0);
                int blk_next = nt > 1 ? load_ids(1) : 0;
                load_kv(0, blk);
                // Q tiles: each buffer is free once the previous item's last QK^T of that tile has completed
                const char* src = reinterpret_cast<const char*>(q_roped) + (size_t)w.q_off16 * 16;
                ptx::mbar_wait(bar(BAR_Q_EMPTY + 0), (qcnt0 & 1u) ^ 1u);
                ++qcnt0;
                if (lane == 0) {
                    ptx::mbar_arrive_expect_tx(bar(BAR_Q_FULL + 0), (uint32_t)(rows0 * D * 2));
#pragma unroll
                    for (int h = 0; h < D / 64; ++h)
                        ptx::bulk_g2s(sbase + L::kQ + h * (kTileM * 128), src + (size_t)h * rows0 * 128,
                                      (uint32_t)rows0 * 128u, bar(BAR_Q_FULL + 0));
                }
                if (rows1) {
                    ptx::mbar_wait(bar(BAR_Q_EMPTY + 1), (qcnt1 & 1u) ^ 1u);
                    ++qcnt1;
                    if (lane == 0) {
                        const char* src1 = src + (size_t)R * D * 2;      // tile 0 is full whenever tile 1 exists
                        ptx::mbar_arrive_expect_tx(bar(BAR_Q_FULL + 1), (uint32_t)(rows1 * D * 2));
#pragma unroll
                        for (int h = 0; h < D / 64; ++h)
                            ptx::bulk_g2s(sbase + L::kQ + L::kQBytes + h * (kTileM * 128), src1 + (size_t)h * rows1 * 128,
                                          (uint32_t)rows1 * 128u, bar(BAR_Q_FULL + 1));
                    }
                }
                publish(nxt, n_item + 1);
                idx_next = __shfl_sync(0xffffffffu, claimed, 0);
                if (has_next && lane == 0)   // pull the next item's Q tiles into L2 while this item computes
                    ptx::bulk_prefetch_l2(reinterpret_cast<const char*>(q_roped) + (size_t)nxt.q_off16 * 16,
                                          (uint32_t)((nxt.ntok0 + nxt.ntok1) * g * D * 2));
                for (int j = 1; j < nt; ++j) {
                    blk = blk_next;
                    blk_next = j + 1 < nt ? load_ids(j + 1) : 0;
                    load_kv(j, blk);
                }
                w = nxt;
            }
        } else if (warp == 12) {
            // ================================ MMA issuer ================================
            // The whole warp runs the control flow (so addresses and descriptors stay in uniform registers); one elected
            // lane issues the MMAs and commits.  The items of this CTA form one continuous stream: QK^T(0) of the next
            // item is issued right behind the last PV of the current one, so the ping-pong never drains between items.
            constexpr uint32_t kIdescQK = ptx::umma_idesc_bf16(kTileM, kTileN, 0, 0);
            constexpr uint32_t kIdescPV = ptx::umma_idesc_bf16(kTileM, D, 0, 1);
            constexpr uint32_t kGroupStride = (D / 64) * 1024;        // bytes between 8-key groups of a K/V tile
            uint32_t it = 0, cnt0 = 0, cnt1 = 0, oitem0 = 0, oitem1 = 0, qf0 = 0, qf1 = 0;
            const uint64_t qdesc0 = ptx::umma_desc_sw128(sbase + L::kQ, 16, 1024);
            const uint64_t kdesc0 = ptx::umma_desc_sw128(sbase + L::kRing, 16, kGroupStride);
            const uint64_t vdesc0 = ptx::umma_desc_sw128(sbase + L::kRing, 1024, kGroupStride);
            auto slot_of = [&](uint32_t i) { return i % NS; };
            auto wait_full = [&](uint32_t i) { ptx::mbar_wait(bar(BAR_RING + slot_of(i)), (i / NS) & 1u); };
            auto release = [&](uint32_t i) { ptx::umma_commit(bar(BAR_RING + NS + slot_of(i))); };
            // S_w = Q_w K^T; `last`: no further QK^T of this item reads Q_w, so its buffer is handed back to the loader
            auto issue_qk = [&](int w, uint32_t slot, bool last) {
                const uint64_t qd = qdesc0 + (uint64_t)((w * L::kQBytes) >> 4), kd = kdesc0 + (uint64_t)((slot * L::kKVBytes) >> 4);
                const uint32_t ts = tmem + (uint32_t)w * 128u;
#ifndef CW_EXP_NOQK
#pragma unroll
                for (int ks = 0; ks < D / 16; ++ks)
                    ptx::umma_ss(ts, qd + (uint64_t)(((ks >> 2) * (kTileM * 128) + (ks & 3) * 32) >> 4),
                                 kd + (uint64_t)(((ks >> 2) * 1024 + (ks & 3) * 32) >> 4), kIdescQK, ks > 0);
#endif
                ptx::umma_commit(bar(BAR_S_FULL + w));
                if (last) ptx::umma_commit(bar(BAR_Q_EMPTY + w));
            };
            auto issue_pv = [&](int w, uint32_t slot, int ksteps, bool first) {
                const uint64_t vd = vdesc0 + (uint64_t)((slot * L::kKVBytes) >> 4);
                const uint32_t to = tmem + 256u + (uint32_t)w * 128u, tp = tmem + (uint32_t)w * 128u;
#ifdef CW_EXP_NOPV
                ksteps = 0;
#endif
                if (ksteps == 8) {
#pragma unroll
                    for (int ks = 0; ks < 8; ++ks)
                        ptx::umma_ts(to, tp + (uint32_t)ks * 8u, vd + (uint64_t)((ks * 2 * kGroupStride) >> 4), kIdescPV,
                                     (!first || ks > 0) ? 1u : 0u);
                } else {
                    for (int ks = 0; ks < ksteps; ++ks)
                        ptx::umma_ts(to, tp + (uint32_t)ks * 8u, vd + (uint64_t)((ks * 2 * kGroupStride) >> 4), kIdescPV,
                                     (!first || ks > 0) ? 1u : 0u);
                }
                ptx::umma_commit(bar(BAR_PV_DONE + w));
            };
            // first QK^T of an item's tiles (K(0) sits at ring index i0); called once up front and then from inside the
            // last iteration of the previous item
            auto open_tile = [&](int w, const Item& x, uint32_t i0) {
                const int ntok = w ? x.ntok1 : x.ntok0;
                if (ntok == 0) return;
                uint32_t& qf = w ? qf1 : qf0;
                ptx::mbar_wait(bar(BAR_Q_FULL + w), qf & 1u);
                ++qf;
                ptx::tc_fence_after();
                const int n_w = tiles_for(x.pos0 + w * tpt + ntok);
                if (ptx::elect_one()) issue_qk(w, slot_of(i0), n_w == 1);
                __syncwarp();
            };
            uint32_t n_item = 0;
            Item w = get_item(0, false);
            if (w.ntok0 > 0) {
                wait_full(0);
                open_tile(0, w, 0);
                open_tile(1, w, 0);
                if (ptx::elect_one()) release(0);
                __syncwarp();
            }
            for (; w.ntok0 > 0; ++n_item) {
                Item nxt{0, 0, 0, 0, 0, 0, 0};
                bool has_next = false;
                const int nkv0 = w.pos0 + w.ntok0, nkv1 = nkv0 + w.ntok1;
                const int n0 = tiles_for(nkv0), n1 = w.ntok1 ? tiles_for(nkv1) : 0;
                const int nt = n1 ? n1 : n0;
                const int nkv = w.ntok1 ? nkv1 : nkv0;
                for (int j = 0; j < nt; ++j) {
                    const uint32_t iv = it + 2 * j + 1, ikn = it + 2 * j + 2;   // ikn: K(j+1), or K(0) of the next item
                    const bool last_iter = j + 1 == nt;
                    if (last_iter) {
                        nxt = get_item(n_item + 1, false);
                        has_next = nxt.ntok0 > 0;
                    }
                    const int left = nkv - j * kTileN;
                    const int ksteps = left >= kTileN ? 8 : (left + 15) >> 4;   // skip 16-key steps with no valid key
                    wait_full(iv);
                    if (!last_iter || has_next) wait_full(ikn);
                    // ---- Q tile 0: O0 += P0 V(j), then S0 = Q0 K(j+1)^T ----
                    if (j < n0) {
                        ptx::mbar_wait(bar(BAR_P_FULL + 0), cnt0 & 1u);
                        if (j == 0) ptx::mbar_wait(bar(BAR_O_EMPTY + 0), (oitem0 & 1u) ^ 1u);
                        ptx::tc_fence_after();
                        if (ptx::elect_one()) {
                            issue_pv(0, slot_of(iv), ksteps, j == 0);
                            if (j + 1 < n0) issue_qk(0, slot_of(ikn), j + 2 == n0);
                        }
                        __syncwarp();
                        ++cnt0;
                    }
                    if (last_iter && has_next) open_tile(0, nxt, ikn);
                    // ---- Q tile 1 ----
                    if (j < n1) {
                        ptx::mbar_wait(bar(BAR_P_FULL + 1), cnt1 & 1u);
                        if (j == 0) ptx::mbar_wait(bar(BAR_O_EMPTY + 1), (oitem1 & 1u) ^ 1u);
                        ptx::tc_fence_after();
                        if (ptx::elect_one()) {
                            issue_pv(1, slot_of(iv), ksteps, j == 0);
                            if (j + 1 < n1) issue_qk(1, slot_of(ikn), j + 2 == n1);
                        }
                        __syncwarp();
                        ++cnt1;
                    }
                    if (last_iter && has_next) open_tile(1, nxt, ikn);
                    if (ptx::elect_one()) {
                        release(iv);
                        if (!last_iter || has_next) release(ikn);
                    }
                    __syncwarp();
                }
                it += 2u * (uint32_t)nt;
                oitem0 += 1;
                oitem1 += n1 ? 1u : 0u;
                w = nxt;
            }
        }
        __syncwarp();
    } else if (warp >= 8) {
        // ================================ epilogue (warps 8-11): O_w / l_w -> bf16 -> global ================================
        ptx::setmaxnreg_dec<64>();
        const int row = threadIdx.x & 127;                 // TMEM lane == packed row within a tile
        const uint32_t lane_base = ((uint32_t)((warp & 3) * 32)) << 16;
        const int tdiv = row / g, hh = row - tdiv * g;
        uint32_t cnt[2] = {0, 0}, litem[2] = {0, 0};
        for (uint32_t n_item = 0;; ++n_item) {
            const Item w = get_item(n_item, true);
            if (w.ntok0 == 0) break;
#pragma unroll
            for (int t = 0; t < 2; ++t) {
                const int ntok = t ? w.ntok1 : w.ntok0;
                if (ntok == 0) continue;
                cnt[t] += (uint32_t)tiles_for(w.pos0 + t * tpt + ntok);
                const bool row_valid = row < ntok * g;
                ptx::mbar_wait(bar(BAR_L_FULL + t), litem[t] & 1u);
                const float inv_l = 1.f / ptx::ld_shared_f32(sbase + L::kL + (t * 128 + row) * 4);
                ptx::mbar_arrive(bar(BAR_L_EMPTY + t));
                ++litem[t];
                ptx::mbar_wait(bar(BAR_PV_DONE + t), (cnt[t] - 1u) & 1u);
                ptx::tc_fence_after();
                const uint32_t tO = tmem + 256u + (uint32_t)t * 128u + lane_base;
                __nv_bfloat16* orow = out + ((size_t)(w.tok0 + t * tpt + tdiv) * Hq + (size_t)w.kvh * g + hh) * D;
#pragma unroll
                for (int i = 0; i < D / 32; ++i) {
                    uint32_t o[32];
                    ptx::tmem_ld32(tO + i * 32, o);
                    ptx::tmem_ld_wait();
                    if (row_valid) {
#pragma unroll
                        for (int e = 0; e < 32; e += 8) {
                            uint4 pk;
                            pk.x = ptx::pack_bf16x2(__uint_as_float(o[e]) * inv_l, __uint_as_float(o[e + 1]) * inv_l);
                            pk.y = ptx::pack_bf16x2(__uint_as_float(o[e + 2]) * inv_l, __uint_as_float(o[e + 3]) * inv_l);
                            pk.z = ptx::pack_bf16x2(__uint_as_float(o[e + 4]) * inv_l, __uint_as_float(o[e + 5]) * inv_l);
                            pk.w = ptx::pack_bf16x2(__uint_as_float(o[e + 6]) * inv_l, __uint_as_float(o[e + 7]) * inv_l);
                            *reinterpret_cast<uint4*>(orow + i * 32 + e) = pk;
                        }
                    }
                }
                ptx::tc_fence_before();
                ptx::mbar_arrive(bar(BAR_O_EMPTY + t));
            }
        }
    } else {
        // ================================ softmax + lazy rescale (warps 0-7) ================================
        ptx::setmaxnreg_inc<192>();
        const int wg = warp >> 2;                          // Q tile of this group
        const int row = threadIdx.x & 127;                 // TMEM lane == packed row within the tile
        const uint32_t lane_base = ((uint32_t)((warp & 3) * 32)) << 16;
        const uint32_t tS = tmem + (uint32_t)wg * 128u + lane_base;
        const uint32_t tO = tmem + 256u + (uint32_t)wg * 128u + lane_base;
        const int tl = wg * tpt + row / g;                 // token of this row inside the item
        uint32_t cnt = 0, litem = 0;
        for (uint32_t n_item = 0;; ++n_item) {
            const Item w = get_item(n_item, false);
            if (w.ntok0 == 0) break;
            const int ntok = wg ? w.ntok1 : w.ntok0;
            if (ntok == 0) continue;
            const int limit = w.pos0 + tl;                 // last visible key (inclusive); rows past the tile end are never stored
            const bool row_valid = row < ntok * g;         // rows past the tile end hold stale Q: they must not steer the warp
            const int n_tiles = tiles_for(w.pos0 + wg * tpt + ntok);

            float m_ref = -INFINITY, l_sum = 0.f;
            for (int j = 0; j < n_tiles; ++j, ++cnt) {
#ifdef CW_PROF
                const long long pt0 = clock64();
#endif
                ptx::mbar_wait(bar(BAR_S_FULL + wg), cnt & 1u);
                ptx::tc_fence_after();
#ifdef CW_PROF
                const long long pt1 = clock64();
#endif
#ifdef CW_EXP_NOSOFTMAX   // timing experiment only (wrong results): the softmax group only hands the tile back
                l_sum = 1.f;
                ptx::tc_fence_before();
                ptx::mbar_arrive(bar(BAR_P_FULL + wg));
                continue;
#endif
                // Speculative path for j > 0: skip the max pass and take exp2 against the current reference maximum; the row
                // sum then bounds every P entry (P <= sum <= 2^16 is exact in fp32/bf16 — softmax does not depend on the
                // reference).  If any row of the warp exceeds the bound (or holds a NaN), the warp redoes the tile the
                // exact way: tile maximum, lazy rescale.  S stays intact in TMEM until P is stored, so it is re-read.
                uint32_t sv[4][32];
                float alpha = 1.f;
                bool grow = false;
                bool spec = j > 0;
                for (;;) {
#pragma unroll
                    for (int i = 0; i < 4; ++i) ptx::tmem_ld32(tS + i * 32, sv[i]);
                    ptx::tmem_ld_wait();

                    const int kbase = j * kTileN;
                    if (kbase + kTileN - 1 > limit) {
#pragma unroll
                        for (int i = 0; i < 4; ++i)
#pragma unroll
                            for (int e = 0; e < 32; ++e)
                                if (kbase + i * 32 + e > limit) sv[i][e] = 0xFF800000u;   // -inf
                    }
                    if (!spec) {
                        float tm[4];
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            float a = fmaxf(__uint_as_float(sv[i][0]), __uint_as_float(sv[i][1]));
                            float b = fmaxf(__uint_as_float(sv[i][2]), __uint_as_float(sv[i][3]));
#pragma unroll
                            for (int e = 4; e < 32; e += 4) {
                                a = fmaxf(a, fmaxf(__uint_as_float(sv[i][e]), __uint_as_float(sv[i][e + 1])));
                                b = fmaxf(b, fmaxf(__uint_as_float(sv[i][e + 2]), __uint_as_float(sv[i][e + 3])));
                            }
                            tm[i] = fmaxf(a, b);
                        }
                        const float tmax = fmaxf(fmaxf(tm[0], tm[1]), fmaxf(tm[2], tm[3]));
                        // lazy rescale decision (per row); the TMEM round trip below is made warp-uniform
                        grow = (tmax - m_ref) * scale_log2 > kRescaleThreshold;   // true on the first tile (m_ref = -inf)
                        if (grow) {
                            alpha = ptx::ex2((m_ref - tmax) * scale_log2);        // 0 on the first tile
                            m_ref = tmax;
                        }
                    }
                    const float mneg = -m_ref * scale_log2;
                    const float2 sc2 = make_float2(scale_log2, scale_log2), mn2 = make_float2(mneg, mneg);
                    float2 ps[4] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
#pragma unroll
                    for (int i = 0; i < 4; ++i)
#pragma unroll
                        for (int e = 0; e < 32; e += 2) {
                            // packed fp32x2 FMA / ADD (sm_100): one instruction per pair of scores
                            const float2 x = __ffma2_rn(make_float2(__uint_as_float(sv[i][e]), __uint_as_float(sv[i][e + 1])), sc2, mn2);
                            float2 p;
                            if (((e >> 1) % kPolyPeriod) < kPolyCount) p = exp2_poly2(x);        // FMA pipe
                            else p = make_float2(ptx::ex2(x.x), ptx::ex2(x.y));                  // MUFU (16 / clk / SM)
                            ps[(e >> 1) & 3] = __fadd2_rn(ps[(e >> 1) & 3], p);
                            sv[i >> 1][(i & 1) * 16 + (e >> 1)] = ptx::pack_bf16x2(p.x, p.y);   // packed P: 64 registers
                        }
                    const float psum = ((ps[0].x + ps[0].y) + (ps[1].x + ps[1].y)) + ((ps[2].x + ps[2].y) + (ps[3].x + ps[3].y));
                    if (spec && __any_sync(0xffffffffu, row_valid && !(psum <= kSpecLimit))) {
                        spec = false;
                        continue;
                    }
                    l_sum = l_sum * alpha + psum;
                    break;
                }

                if (j > 0 && __any_sync(0xffffffffu, grow)) {
                    // O_w holds the sum up to tile j-1: S_FULL(j) was committed after PV(j-1), so it is complete
                    ptx::mbar_wait(bar(BAR_PV_DONE + wg), (cnt - 1u) & 1u);
                    ptx::tc_fence_after();
#pragma unroll
                    for (int i = 0; i < D / 32; ++i) {
                        uint32_t o[32];
                        ptx::tmem_ld32(tO + i * 32, o);
                        ptx::tmem_ld_wait();
#pragma unroll
                        for (int e = 0; e < 32; ++e) o[e] = __float_as_uint(__uint_as_float(o[e]) * alpha);
                        ptx::tmem_st32(tO + i * 32, o);
                    }
                }
                // P (bf16, two keys per 32-bit column) over the first 64 columns of S_w: A operand of the PV MMA
                ptx::tmem_st32(tS, sv[0]);
                ptx::tmem_st32(tS + 32, sv[1]);
                ptx::tmem_st_wait();
                ptx::tc_fence_before();
                ptx::mbar_arrive(bar(BAR_P_FULL + wg));
#ifdef CW_PROF
                if (threadIdx.x == 0) {
                    cw_prof_buf[blockIdx.x][1] += pt1 - pt0;            // wait for S
                    cw_prof_buf[blockIdx.x][2] += clock64() - pt1;      // softmax compute until P_FULL arrive
                    cw_prof_buf[blockIdx.x][7] += 1;
                }
#endif
            }
            // hand the row sum to the epilogue group and go on to the next item
            ptx::mbar_wait(bar(BAR_L_EMPTY + wg), (litem & 1u) ^ 1u);
            ptx::st_shared_f32(sbase + L::kL + (wg * 128 + row) * 4, l_sum);
            ptx::mbar_arrive(bar(BAR_L_FULL + wg));
            ++litem;
        }
    }

    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 12) {
        ptx::tc_fence_after();
        ptx::tmem_dealloc(tmem, 512);
    }
}

// ---- host side: item list and launch ------------------------------------------------------------------------
// Items per request: ceil(s / (2*tpt)) * Hkv.
int64_t attn_count_tiles(const cw_config& cfg, const int32_t* h_cu, int32_t B) {
    const int g = cfg.num_q_heads / cfg.num_kv_heads;
    const int tpt = kTileM / g;
    int64_t n = 0;
    for (int r = 0; r < B; ++r) {
        const int64_t s = h_cu[r + 1] - h_cu[r];
        n += (s + 2 * tpt - 1) / (2 * tpt) * cfg.num_kv_heads;
    }
    return n;
}

int64_t attn_work_ints(const cw_config& cfg, const int32_t* h_cu, int32_t B) {
    return kWorkInts * (attn_count_tiles(cfg, h_cu, B) + 1);   // + header (work counter)
}

// Item order: requests by descending work (longest first, so the tail of the launch is made of short items); inside
// a request kv-head major, tile pairs by descending kv length.  CTA b takes items b, b+G, b+2G, ...: the CTAs work
// on neighbouring items of the same (request, kv head) at the same time and share its K/V blocks through L2.
int64_t attn_build_schedule(const cw_config& cfg, const int32_t* h_cu, const int32_t* h_nc, int32_t B,
                            std::vector<int32_t>& work) {
    const int g = cfg.num_q_heads / cfg.num_kv_heads, D = cfg.head_dim, Hq = cfg.num_q_heads;
    const int tpt = kTileM / g, R = tpt * g;
    std::vector<int32_t> reqs((size_t)B);
    for (int r = 0; r < B; ++r) reqs[(size_t)r] = r;
    auto work_of = [&](int r) {
        const int64_t s = h_cu[r + 1] - h_cu[r], c = h_nc[r];
        return s * (2 * c + s);                      // ~ number of (row, key) pairs
    };
    std::stable_sort(reqs.begin(), reqs.end(), [&](int a, int b) { return work_of(a) > work_of(b); });
    work.assign(kWorkInts, 0);                        // header: work[0] = claim counter, zeroed with every upload
    for (int r : reqs) {
        const int s = h_cu[r + 1] - h_cu[r];
        const int npair = (s + 2 * tpt - 1) / (2 * tpt);
        for (int kvh = 0; kvh < cfg.num_kv_heads; ++kvh)
            for (int t = npair - 1; t >= 0; --t) {
                const int tok0 = t * 2 * tpt;
                const int ntok0 = std::min(tpt, s - tok0), ntok1 = std::max(0, std::min(tpt, s - tok0 - tpt));
                const int64_t q_off = ((int64_t)h_cu[r] * Hq + (int64_t)kvh * s * g) * D + (int64_t)t * 2 * R * D;   // elements
                const int32_t item[kWorkInts] = {h_nc[r] + tok0, ntok0, ntok1, h_cu[r] + tok0, r, kvh, (int32_t)(q_off / 8), 0};
                work.insert(work.end(), item, item + kWorkInts);
            }
    }
    return (int64_t)work.size() / kWorkInts - 1;
}

int launch_prefill_attn(const cw_config& cfg, const void* q_roped, void* out, const int32_t* tables, int32_t max_blocks,
                        int32_t* d_work, int64_t num_items, int num_sms, void* stream) {
    if (num_items == 0) return 0;
    auto s = static_cast<cudaStream_t>(stream);
    const float scale_log2 = 1.4426950408889634f / sqrtf((float)cfg.head_dim);
    const unsigned grid = (unsigned)std::min<int64_t>(num_items, num_sms);
    cudaError_t e;
#define CW_LAUNCH_ATTN(DD)                                                                                          \
    do {                                                                                                            \
        e = cudaFuncSetAttribute(prefill_attn_kernel<DD>, cudaFuncAttributeMaxDynamicSharedMemorySize,              \
                                 Smem<DD>::kTotal);                                                                 \
        if (e != cudaSuccess) return (int)e;                                                                        \
        prefill_attn_kernel<DD><<<grid, kThreads, Smem<DD>::kTotal, s>>>(                                           \
            (const __nv_bfloat16*)q_roped, (__nv_bfloat16*)out, (const __nv_bfloat16*)cfg.k_pool,                   \
            (const __nv_bfloat16*)cfg.v_pool, tables, max_blocks, (int4*)d_work, (int)num_items,              \
            cfg.num_q_heads, cfg.num_kv_heads, scale_log2);                                                         \
    } while (0)
    if (cfg.head_dim == 128) CW_LAUNCH_ATTN(128); else CW_LAUNCH_ATTN(64);
#undef CW_LAUNCH_ATTN
    return (int)cudaGetLastError();
}

}  // namespace cw

#ifdef CW_PROF
extern "C" int cw_debug_prof(unsigned long long* out) {
    cudaDeviceSynchronize();
    int e = (int)cudaMemcpyFromSymbol(out, cw::cw_prof_buf, sizeof(cw::cw_prof_buf));
    static unsigned long long zeros[256][8];
    cudaMemcpyToSymbol(cw::cw_prof_buf, zeros, sizeof(zeros));
    return e;
}
#endif
