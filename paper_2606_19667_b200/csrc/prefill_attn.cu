// Kernel 2: varlen paged causal GQA flash-attention prefill (cw_prefill_attn).  sm_100a, tcgen05 + TMEM + bulk TMA.
//
//   o[row p, head h] = sum_{j<=p} softmax_j(q'_p . k'_j / sqrt(D)) v_j ,  kv head = h / g
//
// Work item = (request r, kv head, 2 consecutive Q tiles).  A Q tile holds tpt = 128/g suffix tokens x the g query
// heads that share the kv head, packed into the M dimension (row = token*g + head), so one K/V read feeds all g
// heads and both Q tiles (M = 256 per CTA), and a short query-only suffix still fills the MMA.
//
// The KV sequence is walked in CHUNKS of 64 keys (4 pool blocks).  Each Q tile owns 128 TMEM columns holding TWO
// S buffers of 64 fp32 columns; P (bf16) overwrites the first 32 columns of the buffer it was computed from.  The MMA
// warp keeps S = Q K^T two chunks ahead of O += P V for each tile, so the softmax of chunk j finds S(j+1) ready and the
// tensor pipe — not the softmax -> PV -> QK^T chain of one buffer — is what bounds a step.
//
// Persistent CTAs (one per SM, 512 threads = 4 warpgroups) claiming items from a list with an atomic counter,
// warp-specialised, mbarrier pipelines only:
//   warps 0-3   softmax of Q tile 0 (thread i owns TMEM lane i = packed row i)
//   warps 4-7   the same for Q tile 1
//   warps 8-11  epilogue of both tiles: O_w / l_w -> packed bf16 in registers, accumulator handed back, 32-byte stores; the
//               softmax groups go straight on to the next item
//   warps 12,14 MMA issuers of Q tile 0 / 1 (one elected lane each): S_w[b] = Q_w K(j)^T (SS, N = 64) and O_w += P_w[b] V(j)
//               (TS: P is read from TMEM); the chunk streams of consecutive items are chained (the first two QK^T of the
//               next item are issued behind the last PVs of the current one); interior chunks take a straight-line step;
//               warp 12 owns TMEM alloc/dealloc (512 columns: S0a S0b S1a S1b O0 O1)
//   warp  13    loader: Q tiles (q_roped is stored tile-packed and pre-swizzled by cw_append_kv: one bulk copy per
//               64-dim half tile) and K/V chunks (one bulk copy per 16-token pool block per operand, gathered through
//               the block table; pool blocks are pre-swizzled in the UMMA canonical layout) into a multi-stage ring
// Softmax is online in fp32 with exp2 and a lazy rescale: O/l are only rescaled when the running max grows by more
// than 2^8 (exact: the final normalisation uses the same reference max for O and l).
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <type_traits>

#include "cw_internal.h"
#include "ptx_sm100.cuh"

// Scratch of cw_prefill_attn_static (end of this file): the work list in memory that ships with the library.
// Some callers have nowhere to take the d_work scratch from: a plugin running inside a host application that owns all
// device memory and hands out only the tensors of the op, a caller inside a region where the allocator must not be
// touched (a serving loop that forbids allocation after warm-up), a C caller without any allocator of its own.  For them
// the item list lives in this fixed array.  It is part of the loaded module, so every GPU on which the library creates a
// CUDA context carries its 2 MiB until the process ends; nothing is ever allocated or freed for it.
static __device__ __align__(256) int32_t g_static_work[CW_STATIC_WORK_INTS];

namespace cw {

namespace {

constexpr int kTileM = 128;          // MMA M (TMEM lanes); a Q tile uses the first tpt*g of them
constexpr int kChunk = 64;           // keys per KV chunk (4 pool blocks)
constexpr int kThreads = 512;
constexpr int kRegsSoftmax = 136, kRegsOther = 120;   // 256 threads each: 256 * (136 + 120) = 65536 registers
constexpr int kWorkInts = 8;         // ints per work item
constexpr int kMaxDevices = 64;      // device ordinals with per-device launcher state (attribute flags, static work list)
constexpr float kRescaleThreshold = 8.0f;   // log2 units
constexpr float kSpecLimit = 65536.f;       // bound on a row sum taken against a stale reference maximum

template <int D>
struct Smem {
    static constexpr int kQBytes = kTileM * D * 2;            // one Q tile
    static constexpr int kKVBytes = kChunk * D * 2;           // one K or V chunk
    static constexpr int kStages = D == 128 ? 10 : 16;        // K/V ring slots (a K chunk or a V chunk each)
    static constexpr int kQ = 0;
    static constexpr int kRing = kQ + 2 * kQBytes;
    static constexpr int kBar = kRing + kStages * kKVBytes;   // mbarriers (8 B each), then the TMEM slot
    static constexpr int kL = kBar + 512;                     // l_sum hand-off softmax -> epilogue: float [2][128]
    static constexpr int kSched = kL + 1024;                  // item ring: kSchedSlots x 8 ints, filled by the loader warp
    static constexpr int kTotal = kSched + 128;
};

// barrier slots; S_FULL / P_FULL are indexed [tile * 2 + buffer]; ring FULL[s] at BAR_RING + s, EMPTY[s] at
// BAR_RING + kStages + s (K chunks sit in the even slots, V chunks in the odd ones; one release per Q tile)
enum { BAR_Q_FULL = 0, BAR_Q_EMPTY = 2, BAR_S_FULL = 4, BAR_P_FULL = 8, BAR_O_FULL = 12, BAR_O_EMPTY = 14,
       BAR_L_FULL = 16, BAR_L_EMPTY = 18, BAR_SCHED_FULL = 20, BAR_SCHED_EMPTY = 24, BAR_RING = 28 };
constexpr int kSchedSlots = 4;
constexpr int kSchedConsumers = 14;  // warps that read every item: MMA (2) + softmax (8) + epilogue (4)

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

// exp2 on the FMA pipe for a share of the scores (the MUFU unit, 16 exp2 / clk / SM, would otherwise be as busy as the
// tensor pipe): 2^x = 2^round(x) * 2^f, f = x - round(x) in [-0.5, 0.5]; 2^f by a degree-3 polynomial (max rel. error
// 7.8e-5, P is rounded to bf16 = 3.9e-3 afterwards); round(x) through the 1.5*2^23 magic constant, spliced into the
// exponent field.  x is clamped to [-125, 126]: the low side flushes to ~0, the high side (only reachable on the
// speculative path, where x is taken against a stale maximum) saturates at 2^126 so that the row sum trips kSpecLimit.
constexpr int kPolyPeriod = 8;   // of every kPolyPeriod score pairs ...
constexpr int kPolyCount = 1;    // ... this many use the polynomial
__device__ __forceinline__ float2 exp2_poly2(float2 x) {
    const float kMagic = 12582912.f;
    x.x = fminf(fmaxf(x.x, -125.f), 126.f);
    x.y = fminf(fmaxf(x.y, -125.f), 126.f);
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

__device__ __forceinline__ int chunks_for(int nkv) { return (nkv + kChunk - 1) / kChunk; }
// pool blocks of chunk j that hold keys below nkv (0..4)
__device__ __forceinline__ int blocks_in_chunk(int nkv, int j) {
    const int left = nkv - j * kChunk;
    return left >= kChunk ? kChunk / 16 : (left + 15) >> 4;
}

}  // namespace

template <int D>
__global__ void __launch_bounds__(kThreads, 1) prefill_attn_kernel(
    const __nv_bfloat16* __restrict__ q_roped, __nv_bfloat16* __restrict__ out,
    const __nv_bfloat16* __restrict__ k_pool, const __nv_bfloat16* __restrict__ v_pool,
    const int32_t* __restrict__ tables, int max_blocks, int4* __restrict__ work, int Hq, int Hkv, float scale_log2) {
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

    // Dynamic schedule (written by attn_schedule_kernel): work[0] = {claim counter, error flags, fallbacks, number of items},
    // items follow from work + 2.
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
            ptx::mbar_init(bar(BAR_O_FULL + w), 1);
            ptx::mbar_init(bar(BAR_O_EMPTY + w), 128);
            ptx::mbar_init(bar(BAR_L_FULL + w), 128);
            ptx::mbar_init(bar(BAR_L_EMPTY + w), 128);
        }
        for (int i = 0; i < 4; ++i) {
            ptx::mbar_init(bar(BAR_S_FULL + i), 1);
            ptx::mbar_init(bar(BAR_P_FULL + i), 4);          // one arrival per softmax warp
        }
        for (int s = 0; s < kSchedSlots; ++s) {
            ptx::mbar_init(bar(BAR_SCHED_FULL + s), 1);
            ptx::mbar_init(bar(BAR_SCHED_EMPTY + s), kSchedConsumers);
        }
        for (int s = 0; s < NS; ++s) {
            ptx::mbar_init(bar(BAR_RING + s), 1);
            ptx::mbar_init(bar(BAR_RING + NS + s), 2);       // one release per Q tile (MMA warp)
        }
        ptx::fence_mbar_init();
    }
    if (warp == 12) ptx::tmem_alloc(ptx::smem_u32(tmem_slot), 512);
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    // Register re-balance: each setmaxnreg sits at the head of its role's code (ptxas applies the limit to the code that
    // follows it in program order) and is executed by all four warps of the warpgroup.
    if (warp >= 12) {
      ptx::setmaxnreg_dec<kRegsOther>();
      if (warp == 13) {
        // ================================ loader ================================
        // Ring order per item: K(0) V(0) K(1) V(1) ...; the item's two Q tiles are loaded after K(0), V(0).
        constexpr uint32_t kBlockBytes = 16 * D * 2;
        uint32_t it = 0, qcnt0 = 0, qcnt1 = 0, n_item = 0;
        int* counter = reinterpret_cast<int*>(work);
        const int num_items = __ldg(reinterpret_cast<const int*>(work) + 3);
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
            const int nt = chunks_for(nkv);
            const int32_t* table = tables + (size_t)w.r * max_blocks;
            auto load_ids = [&](int j) {
                return lane < blocks_in_chunk(nkv, j) ? __ldg(table + j * (kChunk / 16) + lane) : 0;
            };
            auto load_kv = [&](int j, int blk) {
                const int nblk = blocks_in_chunk(nkv, j);
                const size_t src_off = ((size_t)blk * Hkv + w.kvh) * (16 * D);
#pragma unroll
                for (int kv = 0; kv < 2; ++kv) {
                    const uint32_t s = it % NS, ph = (it / NS) & 1u;
                    ptx::mbar_wait(bar(BAR_RING + NS + s), ph ^ 1u);
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
      } else if (warp == 12 || warp == 14) {
        // ================================ MMA issuers: warp 12 -> Q tile 0, warp 14 -> Q tile 1 ================================
        // One issuing warp per Q tile (a single warp cannot issue the 24 MMAs of a 64-key step fast enough).  Both walk the
        // same stream of KV chunks — all chunks of all items of this CTA, global index gq / gp — with S = Q K^T two chunks
        // ahead of O += P V; the first two QK^T of the next item are issued behind the last PVs of the current one.  A chunk
        // the tile does not read (tile 0 can be one chunk shorter than tile 1; tile 1 can be absent) is only handed back to
        // the loader.  The whole warp runs the control flow (operands stay in uniform registers); one elected lane issues.
        auto mma_role = [&](auto wtag) {
            constexpr int W = decltype(wtag)::value;
            if (!ptx::elect_one()) return;          // ONE thread runs the whole role: every operand is trivially uniform
            constexpr uint32_t kIdescQK = ptx::umma_idesc_bf16(kTileM, 0, 0, 0);      // N is added per chunk
            constexpr uint32_t kIdescPV = ptx::umma_idesc_bf16(kTileM, D, 0, 1);
            constexpr uint32_t kGroupStride = (D / 64) * 1024;        // bytes between 8-key groups of a K/V chunk
            const uint64_t qdesc = ptx::umma_desc_sw128(sbase + L::kQ + W * L::kQBytes, 16, 1024);
            const uint64_t kdesc0 = ptx::umma_desc_sw128(sbase + L::kRing, 16, kGroupStride);
            const uint64_t vdesc0 = ptx::umma_desc_sw128(sbase + L::kRing, 1024, kGroupStride);
            const uint32_t tS = tmem + W * 128u, tO = tmem + 256u + W * 128u;
            struct Geo {                             // of an item, for this tile: chunks it reads, its kv length, chunks of the item
                int n, nkv, nt;
            };
            auto geo_of = [&](const Item& x) {
                Geo gg;
                const int nkv0 = x.pos0 + x.ntok0, nkv1 = nkv0 + x.ntok1;
                gg.nt = x.ntok0 ? chunks_for(nkv1) : 0;
                gg.nkv = W == 0 ? nkv0 : (x.ntok1 ? nkv1 : 0);
                gg.n = (W == 0 && x.ntok0 == 0) ? 0 : chunks_for(gg.nkv);
                return gg;
            };
            uint32_t gq = 0, gp = 0;                 // stream chunks passed by the QK^T cursor / the PV cursor
            uint32_t sc = 0, pc = 0;                 // chunks of this tile issued as QK^T / PV: S buffer = & 1, phase = >> 1
            uint32_t kslot = 0, kph = 0;             // ring slot (even) and phase of the K chunk at the QK^T cursor
            uint32_t vslot = 1, vph = 0;             // ring slot (odd) and phase of the V chunk at the PV cursor
            uint32_t qf = 0, oi = 0, n_item = 0;
            auto fetch = [&](uint32_t n) {              // single-thread version of get_item
                const uint32_t slot = n % kSchedSlots;
                ptx::mbar_wait(bar(BAR_SCHED_FULL + slot), (n / kSchedSlots) & 1u);
                const int4 a = *reinterpret_cast<const int4*>(smem + L::kSched + slot * 32);
                ptx::mbar_arrive(bar(BAR_SCHED_EMPTY + slot));
                return Item{a.x, a.y, a.z, a.w, 0, 0, 0};
            };
            Geo gc = geo_of(fetch(0)), gn = gc;
            bool q_on_next = false;                  // QK^T cursor: chunk qj of the current / the next item
            int qj = 0;
            // pass the chunk at the QK^T cursor: S_w[sc & 1] = Q_w K^T if the tile reads it; false at the end of what is known
            auto qk_step = [&]() {
                if (!q_on_next && qj == gc.nt) {
                    q_on_next = true;
                    qj = 0;
                }
                if (q_on_next && qj >= gn.nt) return false;
                const int n_x = q_on_next ? gn.n : gc.n, nkv_x = q_on_next ? gn.nkv : gc.nkv;
                ptx::mbar_wait(bar(BAR_RING + kslot), kph);
                if (qj < n_x) {
                    if (qj == 0) {
                        ptx::mbar_wait(bar(BAR_Q_FULL + W), qf & 1u);
                        ++qf;
                    }
                    ptx::tc_fence_after();
                    const uint32_t b = sc & 1u;
                    const uint32_t idesc = kIdescQK | ((uint32_t)(blocks_in_chunk(nkv_x, qj) * 2) << 17);   // N = 16 * blocks
                    ptx::umma_ss_qk<D>(tS + b * 64u, qdesc, kdesc0 + (uint64_t)((kslot * L::kKVBytes) >> 4), idesc);
                    ptx::umma_commit(bar(BAR_S_FULL + W * 2 + (int)b));
                    ptx::umma_commit(bar(BAR_RING + NS + kslot));
                    if (qj + 1 == n_x) ptx::umma_commit(bar(BAR_Q_EMPTY + W));          // last read of Q_w: hand the buffer back
                    ++sc;
                } else {
                    ptx::mbar_arrive(bar(BAR_RING + NS + kslot));
                }
                kslot += 2;
                if (kslot >= (uint32_t)NS) {
                    kslot -= NS;
                    kph ^= 1u;
                }
                ++qj;
                ++gq;
                return true;
            };
            while (gc.nt > 0) {
                gn = geo_of(fetch(n_item + 1));
                while (gq - gp < 2u && qk_step()) {}
                for (int j = 0; j < gc.nt; ++j) {
                    // Steady state (the interior chunks of an item: both cursors inside the item, Q K^T exactly two full chunks
                    // ahead, nothing to open or close): one straight-line step — the issuing thread is the serial resource of a
                    // tile (~5 clk per dependent instruction), so the general path below, which re-derives every case, would make
                    // it the bottleneck of the whole kernel.
                    if (j > 0 && !q_on_next && qj == j + 2 && qj + 1 < gc.n && gq - gp == 2u && (qj + 1) * kChunk <= gc.nkv) {
                        const uint32_t b = pc & 1u;                                   // == sc & 1: S(j+2) replaces P(j)
                        ptx::mbar_wait(bar(BAR_RING + vslot), vph);
                        ptx::mbar_wait(bar(BAR_P_FULL + W * 2 + (int)b), (pc >> 1) & 1u);
                        ptx::mbar_wait(bar(BAR_RING + kslot), kph);
                        ptx::tc_fence_after();
                        ptx::umma_ts_pv4<D>(tO, tS + b * 64u, vdesc0 + (uint64_t)((vslot * L::kKVBytes) >> 4), kIdescPV, 1u);
                        ptx::umma_commit(bar(BAR_RING + NS + vslot));
                        ptx::umma_ss_qk<D>(tS + b * 64u, qdesc, kdesc0 + (uint64_t)((kslot * L::kKVBytes) >> 4),
                                           kIdescQK | ((uint32_t)(kChunk / 8) << 17));
                        ptx::umma_commit(bar(BAR_S_FULL + W * 2 + (int)b));
                        ptx::umma_commit(bar(BAR_RING + NS + kslot));
                        ++pc;
                        ++sc;
                        ++gp;
                        ++gq;
                        ++qj;
                        vslot += 2;
                        if (vslot >= (uint32_t)NS) {
                            vslot -= NS;
                            vph ^= 1u;
                        }
                        kslot += 2;
                        if (kslot >= (uint32_t)NS) {
                            kslot -= NS;
                            kph ^= 1u;
                        }
                        continue;
                    }
                    // ---- O_w (+)= P_w[pc & 1] V(j) ----
                    ptx::mbar_wait(bar(BAR_RING + vslot), vph);
                    if (j < gc.n) {
                        const uint32_t b = pc & 1u;
                        ptx::mbar_wait(bar(BAR_P_FULL + W * 2 + (int)b), (pc >> 1) & 1u);
                        if (j == 0) {
                            ptx::mbar_wait(bar(BAR_O_EMPTY + W), (oi & 1u) ^ 1u);
                            ++oi;
                        }
                        ptx::tc_fence_after();
                        const int ksteps = blocks_in_chunk(gc.nkv, j);            // 16-key steps that hold a visible key
                        const uint64_t vd = vdesc0 + (uint64_t)((vslot * L::kKVBytes) >> 4);
                        if (ksteps == kChunk / 16) {
                            ptx::umma_ts_pv4<D>(tO, tS + b * 64u, vd, kIdescPV, j > 0 ? 1u : 0u);
                        } else {
                            for (int ks = 0; ks < ksteps; ++ks)
                                ptx::umma_ts(tO, tS + b * 64u + (uint32_t)ks * 8u, vd + (uint64_t)((ks * 2 * kGroupStride) >> 4),
                                             kIdescPV, (j > 0 || ks > 0) ? 1u : 0u);
                        }
                        ptx::umma_commit(bar(BAR_RING + NS + vslot));              // V slot free; also "PV done" for the lazy rescale
                        if (j + 1 == gc.n) ptx::umma_commit(bar(BAR_O_FULL + W));       // O_w complete: the epilogue may read it
                        ++pc;
                    } else {
                        ptx::mbar_arrive(bar(BAR_RING + NS + vslot));
                    }
                    vslot += 2;
                    if (vslot >= (uint32_t)NS) {
                        vslot -= NS;
                        vph ^= 1u;
                    }
                    ++gp;
                    // ---- S_w = Q_w K^T two chunks ahead ----
                    while (gq - gp < 2u && qk_step()) {}
                }
                // the cursor has moved into the next item whenever that item has a chunk for it; otherwise (stream end or a
                // cursor parked at the end of this item) it restarts at chunk 0 of the new current item
                if (q_on_next) q_on_next = false; else qj = 0;
                gc = gn;
                ++n_item;
            }
        };
        if (warp == 12) mma_role(std::integral_constant<int, 0>{}); else mma_role(std::integral_constant<int, 1>{});
        __syncwarp();
      }
    } else if (warp >= 8) {
        // ================================ epilogue (warps 8-11): O_w / l_w -> bf16 -> global ================================
        ptx::setmaxnreg_dec<kRegsOther>();
        const int row = threadIdx.x & 127;                 // TMEM lane == packed row within a tile
        const uint32_t lane_base = ((uint32_t)((warp & 3) * 32)) << 16;
        const int tdiv = row / g, hh = row - tdiv * g;
        uint32_t litem[2] = {0, 0};
        for (uint32_t n_item = 0;; ++n_item) {
            const Item w = get_item(n_item, true);
            if (w.ntok0 == 0) break;
#pragma unroll
            for (int t = 0; t < 2; ++t) {
                const int ntok = t ? w.ntok1 : w.ntok0;
                if (ntok == 0) continue;
                const bool row_valid = row < ntok * g;
                ptx::mbar_wait(bar(BAR_L_FULL + t), litem[t] & 1u);
                const float inv_l = 1.f / ptx::ld_shared_f32(sbase + L::kL + (t * 128 + row) * 4);
                ptx::mbar_arrive(bar(BAR_L_EMPTY + t));
                ptx::mbar_wait(bar(BAR_O_FULL + t), litem[t] & 1u);
                ++litem[t];
                ptx::tc_fence_after();
                const uint32_t tO = tmem + 256u + (uint32_t)t * 128u + lane_base;
                __nv_bfloat16* orow = out + ((size_t)(w.tok0 + t * tpt + tdiv) * Hq + (size_t)w.kvh * g + hh) * D;
                // O -> registers as packed bf16 (D/2 registers); the accumulator is handed back to the MMA warp as soon as it has
                // been READ — the global stores, which are what takes time here, run while the next item's P V accumulates
                uint32_t pk[D / 2];
#pragma unroll
                for (int i = 0; i < D / 32; ++i) {
                    uint32_t o[32];
                    ptx::tmem_ld32(tO + i * 32, o);
                    ptx::tmem_ld_wait();
#pragma unroll
                    for (int x = 0; x < 16; ++x)
                        pk[i * 16 + x] = ptx::pack_bf16x2(__uint_as_float(o[2 * x]) * inv_l, __uint_as_float(o[2 * x + 1]) * inv_l);
                }
                ptx::tc_fence_before();
                ptx::mbar_arrive(bar(BAR_O_EMPTY + t));
                if (row_valid) {
                    // one thread owns one row: 32-byte stores (a whole sector each; a 16-byte store touches the same number of
                    // sectors for half the bytes)
#pragma unroll
                    for (int e = 0; e < D / 2; e += 8) {
                        const uint32_t v8[8] = {pk[e], pk[e + 1], pk[e + 2], pk[e + 3], pk[e + 4], pk[e + 5], pk[e + 6], pk[e + 7]};
                        ptx::st_global_v8(orow + 2 * e, v8);
                    }
                }
            }
        }
    } else {
        // ================================ softmax + lazy rescale (warps 0-7) ================================
        ptx::setmaxnreg_inc<kRegsSoftmax>();
        const int wg = warp >> 2;                          // Q tile of this group
        const int row = threadIdx.x & 127;                 // TMEM lane == packed row within the tile
        const uint32_t lane_base = ((uint32_t)((warp & 3) * 32)) << 16;
        const uint32_t tSw = tmem + (uint32_t)wg * 128u + lane_base;
        const uint32_t tO = tmem + 256u + (uint32_t)wg * 128u + lane_base;
        const int tl = wg * tpt + row / g;                 // token of this row inside the item
        int* fallbacks = reinterpret_cast<int*>(work) + 2; // work header: [0] claim counter, [2] exact-path fallbacks (statistics)
        uint32_t c = 0, g0 = 0, litem = 0;                 // c: chunks of this tile so far (S buffer c & 1, phase c >> 1);
                                                           // g0: index of this item's chunk 0 in the CTA's chunk stream
        for (uint32_t n_item = 0;; ++n_item) {
            const Item w = get_item(n_item, false);
            if (w.ntok0 == 0) break;
            const uint32_t g_item = g0;
            g0 += (uint32_t)chunks_for(w.pos0 + w.ntok0 + w.ntok1);
            const int ntok = wg ? w.ntok1 : w.ntok0;
            if (ntok == 0) continue;
            const int limit = w.pos0 + tl;                 // last visible key (inclusive); rows past the tile end are never stored
            const bool row_valid = row < ntok * g;         // rows past the tile end hold stale Q: they must not steer the warp
            const int n_chunks = chunks_for(w.pos0 + wg * tpt + ntok);
            const int first_limit = w.pos0 + wg * tpt;     // smallest `limit` of the tile: chunks ending above it need the mask

            float m_ref = -INFINITY, l_sum = 0.f;
            for (int j = 0; j < n_chunks; ++j, ++c) {
                const uint32_t b = c & 1u;
                const uint32_t tS = tSw + b * 64u;
                ptx::mbar_wait(bar(BAR_S_FULL + wg * 2 + (int)b), (c >> 1) & 1u);
                ptx::tc_fence_after();
                // Speculative path for j > 0: skip the max pass and take exp2 against the current reference maximum; the row
                // sum then bounds every P entry (P <= sum <= 2^16 is exact in fp32/bf16 — softmax does not depend on the
                // reference).  If any row of the warp exceeds the bound (or holds a NaN), the warp redoes the chunk the
                // exact way: chunk maximum, lazy rescale.  S stays intact in TMEM until P is stored, so it is re-read.
                uint32_t sv[2][32];
                const int rel = limit - j * kChunk;                            // last visible column of this chunk for this row
                const bool need_mask = j * kChunk + kChunk - 1 > first_limit;  // uniform over the tile
                auto load_scores = [&]() {
                    ptx::tmem_ld32(tS, sv[0]);
                    ptx::tmem_ld32(tS + 32, sv[1]);
                    ptx::tmem_ld_wait();
                    if (need_mask) {
#pragma unroll
                        for (int i = 0; i < 2; ++i)
#pragma unroll
                            for (int e = 0; e < 32; ++e)
                                if (i * 32 + e > rel) sv[i][e] = 0xFF800000u;   // -inf
                    }
                };
                // P = exp2(S * scale - m_ref * scale) -> bf16 pairs in sv[0][0..31]; returns the row sum (fp32, before rounding)
                auto exp_pack = [&]() {
                    const float mneg = -m_ref * scale_log2;
                    const float2 sc2 = make_float2(scale_log2, scale_log2), mn2 = make_float2(mneg, mneg);
                    float2 ps[4] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
#pragma unroll
                    for (int i = 0; i < 2; ++i)
#pragma unroll
                        for (int e = 0; e < 32; e += 2) {
                            // packed fp32x2 FMA / ADD (sm_100): one instruction per pair of scores
                            const float2 x = __ffma2_rn(make_float2(__uint_as_float(sv[i][e]), __uint_as_float(sv[i][e + 1])), sc2, mn2);
                            float2 p;
                            if (((e >> 1) % kPolyPeriod) < kPolyCount) p = exp2_poly2(x);        // FMA pipe
                            else p = make_float2(ptx::ex2(x.x), ptx::ex2(x.y));                  // MUFU (16 / clk / SM)
                            ps[(e >> 1) & 3] = __fadd2_rn(ps[(e >> 1) & 3], p);
                            sv[0][i * 16 + (e >> 1)] = ptx::pack_bf16x2(p.x, p.y);             // packed P: 32 registers
                        }
                    return ((ps[0].x + ps[0].y) + (ps[1].x + ps[1].y)) + ((ps[2].x + ps[2].y) + (ps[3].x + ps[3].y));
                };
                load_scores();
                float psum = 0.f, alpha = 1.f;
                bool exact = j == 0, grow = false;
                if (!exact) {
                    psum = exp_pack();
                    if (__any_sync(0xffffffffu, row_valid && !(psum <= kSpecLimit))) {
                        exact = true;
                        if (lane == 0) atomicAdd(fallbacks, 1);
                        load_scores();
                    }
                }
                if (exact) {
                    float tm[2];
#pragma unroll
                    for (int i = 0; i < 2; ++i) {
                        float a = fmaxf(__uint_as_float(sv[i][0]), __uint_as_float(sv[i][1]));
                        float bb = fmaxf(__uint_as_float(sv[i][2]), __uint_as_float(sv[i][3]));
#pragma unroll
                        for (int e = 4; e < 32; e += 4) {
                            a = fmaxf(a, fmaxf(__uint_as_float(sv[i][e]), __uint_as_float(sv[i][e + 1])));
                            bb = fmaxf(bb, fmaxf(__uint_as_float(sv[i][e + 2]), __uint_as_float(sv[i][e + 3])));
                        }
                        tm[i] = fmaxf(a, bb);
                    }
                    const float tmax = fmaxf(tm[0], tm[1]);
                    // lazy rescale decision (per row); the TMEM round trip below is made warp-uniform
                    grow = (tmax - m_ref) * scale_log2 > kRescaleThreshold;   // true on the first chunk (m_ref = -inf)
                    if (grow) {
                        alpha = ptx::ex2((m_ref - tmax) * scale_log2);        // 0 on the first chunk
                        m_ref = tmax;
                    }
                    psum = exp_pack();
                    if (j > 0 && __any_sync(0xffffffffu, grow)) {
                        // O_w must hold the sum up to chunk j-1: wait for the release of the ring slot of V(j-1), which each
                        // MMA warp commits behind its PV(j-1) (the slot's previous release is long past: no aliasing)
                        const uint32_t vi = 2u * (g_item + (uint32_t)j - 1u) + 1u;
                        ptx::mbar_wait(bar(BAR_RING + NS + (int)(vi % NS)), (vi / NS) & 1u);
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
                }
                l_sum = l_sum * alpha + psum;
                // P (bf16, two keys per 32-bit column) over the first 32 columns of this S buffer: A operand of the PV MMA
                ptx::tmem_st32(tS, sv[0]);
                ptx::tmem_st_wait();
                ptx::tc_fence_before();
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(bar(BAR_P_FULL + wg * 2 + (int)b));
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

// ---- schedule kernel: the item list is built on the device, so cw_prefill_attn never reads a descriptor on the host ----
// One CTA.  Request r has s = cu[r+1] - cu[r] suffix rows at positions nc[r] .. nc[r] + s - 1 and gives
// ceil(s / (2 tpt)) * Hkv items.  Item order: requests by descending work s * (2 nc + s) (ties by index: longest first,
// so the tail of the launch is made of short items); inside a request kv-head major, tile pairs by descending kv length.
// CTA b takes items b, b+G, b+2G, ...: the CTAs work on neighbouring items of the same (request, kv head) at the same
// time and share its K/V blocks through L2.
// n_cached[r] is the number of tokens of request r already in the pool: a multiple of 16 after cw_lookup, any value for a
// chunk of a chunked prefill or a decode row.
// work header (ints): [0] claim counter, [1] error flags (bit 0: a request descriptor was invalid and contributes no
// item; bit 1: item list overflow; bit 2: a block table entry outside the pool, request dropped), [2] exact-path fallbacks of the speculative softmax (statistics), [3] number of items; items from int 8 on.
constexpr int kSchedMaxSmemReqs = 2048;      // requests whose (suffix, cached, offset) fit the schedule kernel's shared memory

__global__ void __launch_bounds__(1024) attn_schedule_kernel(
    const int32_t* __restrict__ cu, const int32_t* __restrict__ nc, const int32_t* __restrict__ kv_len,
    const int32_t* __restrict__ tables, int num_blocks, int B, int T,
    int Hq, int Hkv, int D, int max_blocks, int max_position, int max_q_len, int max_kv_len, int32_t* __restrict__ work,
    int64_t max_items) {
    const int g = Hq / Hkv, tpt = kTileM / g, R = tpt * g;
    __shared__ int s_err, s_total;
    __shared__ int s_s[kSchedMaxSmemReqs], s_c[kSchedMaxSmemReqs], s_off[kSchedMaxSmemReqs];
    const bool in_smem = B <= kSchedMaxSmemReqs;
    if (threadIdx.x == 0) {
        s_err = 0;
        s_total = 0;
    }
    __syncthreads();
    // suffix length of request r (0 and the error flag if its descriptor is invalid) and its cached length
    auto suffix = [&](int r, int& c) {
        const int lo = cu[r], hi = cu[r + 1];
        c = nc[r];
        const int64_t s = (int64_t)hi - lo;
        const bool ok = lo >= 0 && s >= 0 && hi <= T && c >= 0 && s <= max_q_len &&
                        (int64_t)c + s <= max_kv_len && (int64_t)c + s <= (int64_t)max_blocks * CW_BLOCK_SIZE &&
                        (int64_t)c + s <= max_position && (kv_len == nullptr || kv_len[r] == c + s);
        return ok ? (int)s : -1;
    };
    auto get = [&](int r, int& c) {           // validated (s, c) of request r
        if (in_smem) {
            c = s_c[r];
            return s_s[r];
        }
        const int s = suffix(r, c);
        return s < 0 ? 0 : s;
    };
    for (int r = threadIdx.x; r < B; r += blockDim.x) {
        int c;
        int s = suffix(r, c);
        if (s < 0) {
            atomicOr(&s_err, 1);
            s = 0;
        }
        if (in_smem) {
            s_s[r] = s;
            s_c[r] = c;
        }
    }
    __syncthreads();
    // The block tables are device data nobody has checked, and the attention kernel's loader follows them into the pools:
    // every entry a request will read (blocks 0 .. ceil(kv_len/16) - 1) must name a pool block.  One warp per request, lanes
    // over its entries (coalesced, all loads of a lane independent).  A request with a bad entry is dropped (error bit 2,
    // no items, no output); a batch too large for the shared-memory copy of the lengths is dropped as a whole.
    for (int r = threadIdx.x >> 5; r < B; r += blockDim.x >> 5) {
        int c;
        const int s = get(r, c);
        const int nblk = s > 0 ? (c + s + CW_BLOCK_SIZE - 1) / CW_BLOCK_SIZE : 0;
        const int32_t* row = tables + (size_t)r * max_blocks;
        bool bad = false;
        for (int i = threadIdx.x & 31; i < nblk; i += 32) bad |= (unsigned)row[i] >= (unsigned)num_blocks;
        if (__any_sync(0xffffffffu, bad) && (threadIdx.x & 31) == 0) {
            atomicOr(&s_err, 4);
            if (in_smem) s_s[r] = 0;
        }
    }
    __syncthreads();
    const bool drop_all = !in_smem && (s_err & 4);
    // rank sort + exclusive prefix sum of the item counts in one pass over the other requests
    for (int r = threadIdx.x; r < B; r += blockDim.x) {
        int c;
        const int s = get(r, c);
        const int64_t key = (int64_t)s * (2 * (int64_t)c + s);      // ~ number of (row, key) pairs
        const int items = (s + 2 * tpt - 1) / (2 * tpt) * Hkv;
        int64_t off = 0;
        for (int q = 0; q < B; ++q) {
            int cq;
            const int sq = get(q, cq);
            const int64_t kq = (int64_t)sq * (2 * (int64_t)cq + sq);
            if (kq > key || (kq == key && q < r)) off += (sq + 2 * tpt - 1) / (2 * tpt) * Hkv;
        }
        if (off + items > max_items) {                                // cannot happen for the bound the host computes from B, T
            atomicOr(&s_err, 2);
            off = -1;
        } else {
            atomicAdd(&s_total, items);
        }
        if (in_smem) {
            s_off[r] = (int)off;
        } else if (off >= 0) {                                        // large batches: the owning thread writes its items
            int4* dst = reinterpret_cast<int4*>(work) + 2 + 2 * off;
            const int npair = (s + 2 * tpt - 1) / (2 * tpt);
            for (int i = 0; i < npair * Hkv; ++i) {
                const int kvh = i / npair, t = npair - 1 - i % npair;
                const int tok0 = t * 2 * tpt;
                const int64_t q_off = ((int64_t)cu[r] * Hq + (int64_t)kvh * s * g) * D + (int64_t)t * 2 * R * D;   // elements
                dst[2 * i] = make_int4(c + tok0, min(tpt, s - tok0), max(0, min(tpt, s - tok0 - tpt)), cu[r] + tok0);
                dst[2 * i + 1] = make_int4(r, kvh, (int)(q_off / 8), 0);
            }
        }
    }
    __syncthreads();
    if (in_smem) {
        // one warp per request, lanes over its items
        const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
        for (int r = warp; r < B; r += blockDim.x / 32) {
            const int s = s_s[r], c = s_c[r], off = s_off[r];
            if (off < 0) continue;
            const int q_begin = cu[r];
            int4* dst = reinterpret_cast<int4*>(work) + 2 + 2 * (int64_t)off;
            const int npair = (s + 2 * tpt - 1) / (2 * tpt);
            for (int i = lane; i < npair * Hkv; i += 32) {
                const int kvh = i / npair, t = npair - 1 - i % npair;
                const int tok0 = t * 2 * tpt;
                const int64_t q_off = ((int64_t)q_begin * Hq + (int64_t)kvh * s * g) * D + (int64_t)t * 2 * R * D;   // elements
                dst[2 * i] = make_int4(c + tok0, min(tpt, s - tok0), max(0, min(tpt, s - tok0 - tpt)), q_begin + tok0);
                dst[2 * i + 1] = make_int4(r, kvh, (int)(q_off / 8), 0);
            }
        }
    }
    if (threadIdx.x == 0) {
        work[0] = 0;
        work[1] = s_err;
        work[2] = 0;
        work[3] = drop_all ? 0 : s_total;
    }
}

// upper bound on the number of items of a batch with B requests and T suffix rows in total (every request may add one
// ragged tile pair per kv head)
int64_t attn_max_items(const cw_config& cfg, int32_t B, int32_t T) {
    const int g = cfg.num_q_heads / cfg.num_kv_heads;
    const int tpt2 = 2 * (kTileM / g);
    return ((int64_t)T / tpt2 + B) * cfg.num_kv_heads;
}

int64_t attn_work_ints(const cw_config& cfg, int32_t B, int32_t T) {
    return kWorkInts * (attn_max_items(cfg, B, T) + 1);   // + header
}

// The two launches of cw_prefill_attn can be enqueued apart: the schedule kernel needs only the descriptors, so a caller
// may run it in front of (or, on another stream, beside) cw_append_kv and keep it off the append -> attention chain.
int launch_attn_schedule(const cw_config& cfg, const int32_t* d_cu, const int32_t* d_nc, const int32_t* d_kv_len,
                         const int32_t* tables, int32_t max_blocks, int32_t B, int32_t T, int32_t max_q_len,
                         int32_t max_kv_len, int32_t* d_work, void* stream) {
    const int64_t max_items = attn_max_items(cfg, B, T);
    if (max_items == 0) return 0;
    attn_schedule_kernel<<<1, 1024, 0, static_cast<cudaStream_t>(stream)>>>(
        d_cu, d_nc, d_kv_len, tables, cfg.num_blocks, B, T, cfg.num_q_heads, cfg.num_kv_heads, cfg.head_dim, max_blocks,
        cfg.max_position, max_q_len, max_kv_len, d_work, max_items);
    return (int)cudaGetLastError();
}

int launch_prefill_attn(const cw_config& cfg, const void* q_roped, void* out, const int32_t* d_cu, const int32_t* d_nc,
                        const int32_t* d_kv_len, const int32_t* tables, int32_t max_blocks, int32_t B, int32_t T,
                        int32_t max_q_len, int32_t max_kv_len, int32_t* d_work, int num_sms, void* stream) {
    const int le = launch_attn_schedule(cfg, d_cu, d_nc, d_kv_len, tables, max_blocks, B, T, max_q_len, max_kv_len, d_work,
                                        stream);
    return le ? le : launch_attn_run(cfg, q_roped, out, tables, max_blocks, B, T, d_work, num_sms, stream);
}

int launch_attn_run(const cw_config& cfg, const void* q_roped, void* out, const int32_t* tables, int32_t max_blocks,
                    int32_t B, int32_t T, int32_t* d_work, int num_sms, void* stream) {
    auto s = static_cast<cudaStream_t>(stream);
    const int64_t max_items = attn_max_items(cfg, B, T);
    if (max_items == 0) return 0;
    cudaError_t e = cudaSuccess;
    const float scale_log2 = 1.4426950408889634f / sqrtf((float)cfg.head_dim);
    const unsigned grid = (unsigned)std::min<int64_t>(max_items, num_sms);
    // The dynamic shared memory opt-in is a per-device attribute of the kernel: one flag per device ordinal (a process may
    // hold contexts on several GPUs).  Two host threads racing on a flag both set the attribute, which is harmless.
    int dev = 0;
    e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return (int)e;
#define CW_LAUNCH_ATTN(DD)                                                                                          \
    do {                                                                                                            \
        static std::atomic<bool> attr_set[kMaxDevices];                                                             \
        if (dev < 0 || dev >= kMaxDevices || !attr_set[dev].load(std::memory_order_acquire)) {                      \
            e = cudaFuncSetAttribute(prefill_attn_kernel<DD>, cudaFuncAttributeMaxDynamicSharedMemorySize,          \
                                     Smem<DD>::kTotal);                                                             \
            if (e != cudaSuccess) return (int)e;                                                                    \
            if (dev >= 0 && dev < kMaxDevices) attr_set[dev].store(true, std::memory_order_release);                \
        }                                                                                                           \
        prefill_attn_kernel<DD><<<grid, kThreads, Smem<DD>::kTotal, s>>>(                                           \
            (const __nv_bfloat16*)q_roped, (__nv_bfloat16*)out, (const __nv_bfloat16*)cfg.k_pool,                   \
            (const __nv_bfloat16*)cfg.v_pool, tables, max_blocks, (int4*)d_work, cfg.num_q_heads,                   \
            cfg.num_kv_heads, scale_log2);                                                                          \
    } while (0)
    if (cfg.head_dim == 128) CW_LAUNCH_ATTN(128); else CW_LAUNCH_ATTN(64);
#undef CW_LAUNCH_ATTN
    return (int)cudaGetLastError();
}

// ---- cw_prefill_attn_static: the same two kernels with the work list in g_static_work (top of this file) ----
namespace {
// Device address of g_static_work per device ordinal.  `g_static_work` in HOST code is only a handle for the runtime's
// symbol table, not an address a kernel may use: the address is asked for with cudaGetSymbolAddress while that device is
// current, once per device.  A benign race between two host threads resolves the same value twice.
int32_t* g_static_work_ptr[kMaxDevices] = {};
}  // namespace

int launch_prefill_attn_static(const cw_config& cfg, const void* q_roped, void* out, const int32_t* d_cu,
                               const int32_t* d_nc, const int32_t* d_kv_len, const int32_t* tables, int32_t max_blocks,
                               int32_t B, int32_t T, int32_t max_q_len, int32_t max_kv_len, int32_t* d_status, int num_sms,
                               void* stream) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return (int)e;
    if (dev != cfg.device || dev < 0 || dev >= kMaxDevices) return (int)cudaErrorInvalidDevice;
    int32_t* work = g_static_work_ptr[dev];
    if (!work) {                                        // set-up: first call on this device
        e = cudaGetSymbolAddress((void**)&work, g_static_work);
        if (e != cudaSuccess) return (int)e;
        g_static_work_ptr[dev] = work;
    }
    // Nothing in the array has to be cleared from the host: the schedule kernel rewrites the whole header (claim counter
    // and fallback counter to zero, error flags, item count) and every item below the count it writes; items above it
    // are leftovers of earlier calls and are never read.
    int le = launch_prefill_attn(cfg, q_roped, out, d_cu, d_nc, d_kv_len, tables, max_blocks, B, T, max_q_len, max_kv_len,
                                 work, num_sms, stream);
    if (le) return le;
    if (d_status && attn_max_items(cfg, B, T) > 0)      // header -> caller's 4 ints, behind the attention kernel on the stream
        return (int)cudaMemcpyAsync(d_status, work, 4 * sizeof(int32_t), cudaMemcpyDeviceToDevice,
                                    static_cast<cudaStream_t>(stream));
    return 0;
}

}  // namespace cw
