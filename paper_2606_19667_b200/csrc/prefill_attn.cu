// Kernel 2: varlen paged causal GQA flash-attention prefill (cw_prefill_attn).  sm_100a, tcgen05 + TMEM + bulk TMA.
//
//   o[row p, head h] = sum_{j<=p} softmax_j(q'_p . k'_j / sqrt(D)) v_j ,  kv head = h / g
//
// Work item ("tile") = (request r, kv head, 128 packed rows).  The g query heads that share a KV head are packed
// into the M dimension: packed row i <-> (suffix token i / g, head kvh*g + i % g), so one K/V tile read feeds all g
// heads and short suffixes (query-only after a long cache hit) still fill M = 128.
//
// CTA = 192 threads, warp-specialised, mbarrier pipelines only (no __syncthreads in the main loop):
//   warps 0-3  softmax / correction / epilogue: thread i owns TMEM lane i = packed row i
//   warp  4    loader: one bulk copy (UBLKCP) per 16-token pool block per operand, gathered through the block table;
//              pool blocks are stored pre-swizzled in the UMMA canonical layout (cw_pool_offset), so no re-layout
//   warp  5    MMA issuer: S = Q K^T (SS, K-major/K-major) into a double-buffered S in TMEM, O += P V (A = P from
//              smem K-major, B = V MN-major), accumulators in TMEM; also owns TMEM alloc/dealloc
// Softmax is online in fp32 with exp2 and a lazy rescale: O/l are only rescaled when the running max grows by
// more than 2^8 (exact: the final normalisation uses the same reference max for O and l).
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include <algorithm>

#include "cw_internal.h"
#include "ptx_sm100.cuh"

namespace cw {

namespace {

constexpr int kTileM = 128;          // packed query rows per tile
constexpr int kTileN = 128;          // keys per KV tile (8 pool blocks)
constexpr int kStages = 2;           // K and V ring depth
constexpr int kThreads = 192;
constexpr float kRescaleThreshold = 8.0f;   // log2 units

template <int D>
struct Smem {
    static constexpr int kQBytes = kTileM * D * 2;
    static constexpr int kKVBytes = kTileN * D * 2;          // one K or V tile
    static constexpr int kPBytes = kTileM * kTileN * 2;
    static constexpr int kQ = 0;
    static constexpr int kK = kQ + kQBytes;
    static constexpr int kV = kK + kStages * kKVBytes;
    static constexpr int kP = kV + kStages * kKVBytes;
    static constexpr int kBar = kP + kPBytes;                 // mbarriers (8 B each)
    static constexpr int kTotal = kBar + 256;
};

// barrier slots
enum { BAR_Q_FULL = 0, BAR_K_FULL = 1, BAR_K_EMPTY = 3, BAR_V_FULL = 5, BAR_V_EMPTY = 7, BAR_S_FULL = 9,
       BAR_S_EMPTY = 11, BAR_P_FULL = 13, BAR_PV_DONE = 14, BAR_COUNT = 15 };

}  // namespace

template <int D>
__global__ void __launch_bounds__(kThreads, 1) prefill_attn_kernel(
    const __nv_bfloat16* __restrict__ q_roped, __nv_bfloat16* __restrict__ out,
    const __nv_bfloat16* __restrict__ k_pool, const __nv_bfloat16* __restrict__ v_pool,
    const int32_t* __restrict__ cu, const int32_t* __restrict__ ncached, const int32_t* __restrict__ tables,
    int max_blocks, const int4* __restrict__ work, int Hq, int Hkv, float scale_log2) {
    using L = Smem<D>;
    extern __shared__ __align__(1024) uint8_t smem[];
    const uint32_t sbase = ptx::smem_u32(smem);
    const uint32_t bars = sbase + L::kBar;
    auto bar = [&](int i) { return bars + 8u * (uint32_t)i; };
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + L::kBar + 8 * BAR_COUNT);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int4 w = __ldg(work + blockIdx.x);
    const int r = w.x, kvh = w.y, row0 = w.z, num_kv = w.w;
    const int g = Hq / Hkv;
    const int q_begin = __ldg(cu + r);
    const int s_len = __ldg(cu + r + 1) - q_begin;
    const int c = __ldg(ncached + r);
    const int rows_total = s_len * g;
    const int n_tiles = (num_kv + kTileN - 1) / kTileN;

    if (threadIdx.x == 0) {
        ptx::mbar_init(bar(BAR_Q_FULL), 128);
        for (int i = 0; i < kStages; ++i) {
            ptx::mbar_init(bar(BAR_K_FULL + i), 1);
            ptx::mbar_init(bar(BAR_K_EMPTY + i), 1);
            ptx::mbar_init(bar(BAR_V_FULL + i), 1);
            ptx::mbar_init(bar(BAR_V_EMPTY + i), 1);
        }
        for (int i = 0; i < 2; ++i) {
            ptx::mbar_init(bar(BAR_S_FULL + i), 1);
            ptx::mbar_init(bar(BAR_S_EMPTY + i), 128);
        }
        ptx::mbar_init(bar(BAR_P_FULL), 128);
        ptx::mbar_init(bar(BAR_PV_DONE), 1);
        ptx::fence_mbar_init();
    }
    if (warp == 5) ptx::tmem_alloc(ptx::smem_u32(tmem_slot), 512);
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const uint32_t tmem_S0 = tmem, tmem_O = tmem + 256;

    if (warp == 4) {
        // ================================ loader ================================
        constexpr uint32_t kBlockBytes = 16 * D * 2;
        const int32_t* table = tables + (size_t)r * max_blocks;
        for (int j = 0; j < n_tiles; ++j) {
            const int st = j % kStages;
            const uint32_t ph = (uint32_t)(j / kStages) & 1u;
            const int kv_left = num_kv - j * kTileN;
            const int nblk = kv_left >= kTileN ? 8 : (kv_left + 15) >> 4;
            int blk = 0;
            if (lane < nblk) blk = __ldg(table + j * 8 + lane);
            const size_t src_off = ((size_t)blk * Hkv + kvh) * (16 * D);
            // K tile
            ptx::mbar_wait(bar(BAR_K_EMPTY + st), ph ^ 1u);
            if (lane == 0) ptx::mbar_arrive_expect_tx(bar(BAR_K_FULL + st), kBlockBytes * (uint32_t)nblk);
            __syncwarp();
            if (lane < nblk)
                ptx::bulk_g2s(sbase + L::kK + st * L::kKVBytes + lane * kBlockBytes, k_pool + src_off, kBlockBytes,
                              bar(BAR_K_FULL + st));
            // V tile
            ptx::mbar_wait(bar(BAR_V_EMPTY + st), ph ^ 1u);
            if (lane == 0) ptx::mbar_arrive_expect_tx(bar(BAR_V_FULL + st), kBlockBytes * (uint32_t)nblk);
            __syncwarp();
            if (lane < nblk)
                ptx::bulk_g2s(sbase + L::kV + st * L::kKVBytes + lane * kBlockBytes, v_pool + src_off, kBlockBytes,
                              bar(BAR_V_FULL + st));
        }
    } else if (warp == 5) {
        // ================================ MMA issuer ================================
        constexpr uint32_t kIdescQK = ptx::umma_idesc_bf16(kTileM, kTileN, 0, 0);
        constexpr uint32_t kIdescPV = ptx::umma_idesc_bf16(kTileM, D, 0, 1);
        constexpr uint32_t kGroupStride = (D / 64) * 1024;        // bytes between 8-key groups of a K/V tile
        auto issue_qk = [&](int j) {
            const int st = j % kStages;
            ptx::mbar_wait(bar(BAR_K_FULL + st), (uint32_t)(j / kStages) & 1u);
            ptx::mbar_wait(bar(BAR_S_EMPTY + (j & 1)), ((uint32_t)(j >> 1) & 1u) ^ 1u);
            ptx::tc_fence_after();
            if (ptx::elect_one()) {
                const uint32_t kb = sbase + L::kK + st * L::kKVBytes;
#pragma unroll
                for (int ks = 0; ks < D / 16; ++ks) {
                    const uint64_t a = ptx::umma_desc_sw128(sbase + L::kQ + (ks >> 2) * (kTileM * 128) + (ks & 3) * 32, 16, 1024);
                    const uint64_t b = ptx::umma_desc_sw128(kb + (ks >> 2) * 1024 + (ks & 3) * 32, 16, kGroupStride);
                    ptx::umma_ss(tmem_S0 + (uint32_t)(j & 1) * 128u, a, b, kIdescQK, ks > 0);
                }
                ptx::umma_commit(bar(BAR_K_EMPTY + st));
                ptx::umma_commit(bar(BAR_S_FULL + (j & 1)));
            }
            __syncwarp();
        };
        ptx::mbar_wait(bar(BAR_Q_FULL), 0);
        issue_qk(0);
        for (int j = 0; j < n_tiles; ++j) {
            if (j + 1 < n_tiles) issue_qk(j + 1);
            const int st = j % kStages;
            const int kv_left = num_kv - j * kTileN;
            const int ksteps = kv_left >= kTileN ? 8 : (kv_left + 15) >> 4;   // skip 16-key steps with no valid key
            ptx::mbar_wait(bar(BAR_V_FULL + st), (uint32_t)(j / kStages) & 1u);
            ptx::mbar_wait(bar(BAR_P_FULL), (uint32_t)j & 1u);
            ptx::tc_fence_after();
            if (ptx::elect_one()) {
                const uint32_t vb = sbase + L::kV + st * L::kKVBytes;
                for (int ks = 0; ks < ksteps; ++ks) {
                    const uint64_t a = ptx::umma_desc_sw128(sbase + L::kP + (ks >> 2) * (kTileM * 128) + (ks & 3) * 32, 16, 1024);
                    const uint64_t b = ptx::umma_desc_sw128(vb + ks * 2 * kGroupStride, 1024, kGroupStride);
                    ptx::umma_ss(tmem_O, a, b, kIdescPV, (j > 0 || ks > 0) ? 1u : 0u);
                }
                ptx::umma_commit(bar(BAR_V_EMPTY + st));
                ptx::umma_commit(bar(BAR_PV_DONE));
            }
            __syncwarp();
        }
    } else {
        // ================================ softmax / correction / epilogue ================================
        const int row = threadIdx.x;                       // TMEM lane == packed row within the tile
        const int prow = row0 + row;
        const bool row_valid = prow < rows_total;
        const int tok = (row_valid ? prow : rows_total - 1) / g;
        const int hh = (row_valid ? prow : rows_total - 1) % g;
        const int limit = c + tok;                         // last visible key (inclusive)
        const uint32_t lane_base = ((uint32_t)(warp * 32)) << 16;

        // ---- Q tile -> smem (K-major, 128B swizzle), zero-filled past the end of the request ----
        {
            constexpr int CH = D / 8;                      // 16-byte chunks per row
            const int ch = threadIdx.x % CH;
            const __nv_bfloat16* qbase = q_roped + ((size_t)q_begin * Hq + (size_t)kvh * g) * D;
            for (int rr = threadIdx.x / CH; rr < kTileM; rr += 128 / CH) {
                const int pr = row0 + rr;
                uint4 val = make_uint4(0, 0, 0, 0);
                if (pr < rows_total)
                    val = *reinterpret_cast<const uint4*>(qbase + ((size_t)(pr / g) * Hq + (pr % g)) * D + ch * 8);
                const uint32_t dst = sbase + L::kQ + (ch >> 3) * (kTileM * 128) + rr * 128 + (((ch & 7) ^ (rr & 7)) << 4);
                ptx::st_shared_v4(dst, val.x, val.y, val.z, val.w);
            }
            ptx::fence_proxy_async_smem();
            ptx::mbar_arrive(bar(BAR_Q_FULL));
        }

        float m_ref = -INFINITY, l_sum = 0.f;
        for (int j = 0; j < n_tiles; ++j) {
            const uint32_t tS = tmem_S0 + (uint32_t)(j & 1) * 128u + lane_base;
            ptx::mbar_wait(bar(BAR_S_FULL + (j & 1)), (uint32_t)(j >> 1) & 1u);
            ptx::tc_fence_after();
            uint32_t sv[4][32];
#pragma unroll
            for (int i = 0; i < 4; ++i) ptx::tmem_ld32(tS + i * 32, sv[i]);
            ptx::tmem_ld_wait();
            ptx::tc_fence_before();
            ptx::mbar_arrive(bar(BAR_S_EMPTY + (j & 1)));

            const int kbase = j * kTileN;
            if (kbase + kTileN - 1 > limit) {
#pragma unroll
                for (int i = 0; i < 4; ++i)
#pragma unroll
                    for (int e = 0; e < 32; ++e)
                        if (kbase + i * 32 + e > limit) sv[i][e] = 0xFF800000u;   // -inf
            }
            float tmax = -INFINITY;
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int e = 0; e < 32; ++e) tmax = fmaxf(tmax, __uint_as_float(sv[i][e]));
            // lazy rescale decision (per row), then made warp-uniform for the TMEM round trip
            float alpha = 1.f;
            bool grow = (tmax - m_ref) * scale_log2 > kRescaleThreshold;   // true on the first tile (m_ref = -inf)
            if (grow) {
                alpha = ptx::ex2((m_ref - tmax) * scale_log2);             // 0 on the first tile
                m_ref = tmax;
            }
            const float mneg = -m_ref * scale_log2;
            float psum = 0.f;
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int e = 0; e < 32; e += 2) {
                    float p0 = ptx::ex2(fmaf(__uint_as_float(sv[i][e]), scale_log2, mneg));
                    float p1 = ptx::ex2(fmaf(__uint_as_float(sv[i][e + 1]), scale_log2, mneg));
                    psum += p0 + p1;
                    sv[i][e >> 1] = ptx::pack_bf16x2(p0, p1);              // packed P overwrites the front half
                }
            l_sum = l_sum * alpha + psum;

            // P smem and O are free once PV(j-1) has completed
            if (j > 0) {
                ptx::mbar_wait(bar(BAR_PV_DONE), (uint32_t)(j - 1) & 1u);
                ptx::tc_fence_after();
                if (__any_sync(0xffffffffu, grow)) {
#pragma unroll
                    for (int i = 0; i < D / 32; ++i) {
                        uint32_t o[32];
                        ptx::tmem_ld32(tmem_O + lane_base + i * 32, o);
                        ptx::tmem_ld_wait();
#pragma unroll
                        for (int e = 0; e < 32; ++e) o[e] = __float_as_uint(__uint_as_float(o[e]) * alpha);
                        ptx::tmem_st32(tmem_O + lane_base + i * 32, o);
                    }
                    ptx::tmem_st_wait();
                }
            }
            // P (bf16) -> smem, K-major 128B swizzle: [key half][row][64 keys]
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int q4 = 0; q4 < 4; ++q4) {
                    const int chunk = i * 4 + q4;                           // 8 keys per 16-byte chunk
                    const uint32_t dst = sbase + L::kP + (chunk >> 3) * (kTileM * 128) + row * 128 +
                                         (((chunk & 7) ^ (row & 7)) << 4);
                    ptx::st_shared_v4(dst, sv[i][q4 * 4], sv[i][q4 * 4 + 1], sv[i][q4 * 4 + 2], sv[i][q4 * 4 + 3]);
                }
            ptx::fence_proxy_async_smem();
            ptx::tc_fence_before();
            ptx::mbar_arrive(bar(BAR_P_FULL));
        }

        // ---- epilogue: O / l -> bf16 -> global ----
        ptx::mbar_wait(bar(BAR_PV_DONE), (uint32_t)(n_tiles - 1) & 1u);
        ptx::tc_fence_after();
        const float inv_l = 1.f / l_sum;
        __nv_bfloat16* orow = out + ((size_t)(q_begin + tok) * Hq + (size_t)kvh * g + hh) * D;
#pragma unroll
        for (int i = 0; i < D / 32; ++i) {
            uint32_t o[32];
            ptx::tmem_ld32(tmem_O + lane_base + i * 32, o);
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
    }

    __syncthreads();
    if (warp == 5) {
        ptx::tc_fence_after();
        ptx::tmem_dealloc(tmem, 512);
    }
}

// ---- host side: tile schedule and launch -------------------------------------------------------------------
int64_t attn_count_tiles(const cw_config& cfg, const int32_t* h_cu, int32_t B) {
    const int g = cfg.num_q_heads / cfg.num_kv_heads;
    int64_t n = 0;
    for (int r = 0; r < B; ++r) {
        int64_t rows = (int64_t)(h_cu[r + 1] - h_cu[r]) * g;
        n += (rows + kTileM - 1) / kTileM * cfg.num_kv_heads;
    }
    return n;
}

// Longest-first order: CTAs are dispatched in blockIdx order, so sorting tiles by descending KV length gives an
// LPT schedule over the 148 SMs without a persistent loop.
int64_t attn_build_schedule(const cw_config& cfg, const int32_t* h_cu, const int32_t* h_nc, int32_t B,
                            std::vector<int32_t>& work) {
    const int g = cfg.num_q_heads / cfg.num_kv_heads;
    struct T { int32_t r, kvh, row0, nkv; };
    std::vector<T> tiles;
    for (int r = 0; r < B; ++r) {
        const int s = h_cu[r + 1] - h_cu[r];
        const int64_t rows = (int64_t)s * g;
        for (int64_t row0 = 0; row0 < rows; row0 += kTileM) {
            const int64_t last = std::min<int64_t>(row0 + kTileM - 1, rows - 1);
            const int32_t nkv = h_nc[r] + (int32_t)(last / g) + 1;
            for (int kvh = 0; kvh < cfg.num_kv_heads; ++kvh) tiles.push_back(T{r, kvh, (int32_t)row0, nkv});
        }
    }
    std::stable_sort(tiles.begin(), tiles.end(), [](const T& a, const T& b) { return a.nkv > b.nkv; });
    work.resize(tiles.size() * 4);
    for (size_t i = 0; i < tiles.size(); ++i) {
        work[4 * i] = tiles[i].r; work[4 * i + 1] = tiles[i].kvh; work[4 * i + 2] = tiles[i].row0; work[4 * i + 3] = tiles[i].nkv;
    }
    return (int64_t)tiles.size();
}

int launch_prefill_attn(const cw_config& cfg, const void* q_roped, void* out, const int32_t* cu,
                        const int32_t* ncached, const int32_t* tables, int32_t max_blocks, const int32_t* d_work,
                        int64_t num_tiles, int /*num_sms*/, void* stream) {
    if (num_tiles == 0) return 0;
    auto s = static_cast<cudaStream_t>(stream);
    const float scale_log2 = 1.4426950408889634f / sqrtf((float)cfg.head_dim);
    // both head dims request the same dynamic smem so that exactly one CTA (512 TMEM columns) is resident per SM
    const int smem_bytes = Smem<128>::kTotal;
    cudaError_t e;
#define CW_LAUNCH_ATTN(DD)                                                                                          \
    do {                                                                                                            \
        e = cudaFuncSetAttribute(prefill_attn_kernel<DD>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes); \
        if (e != cudaSuccess) return (int)e;                                                                        \
        prefill_attn_kernel<DD><<<(unsigned)num_tiles, kThreads, smem_bytes, s>>>(                                  \
            (const __nv_bfloat16*)q_roped, (__nv_bfloat16*)out, (const __nv_bfloat16*)cfg.k_pool,                   \
            (const __nv_bfloat16*)cfg.v_pool, cu, ncached, tables, max_blocks, (const int4*)d_work,                 \
            cfg.num_q_heads, cfg.num_kv_heads, scale_log2);                                                         \
    } while (0)
    if (cfg.head_dim == 128) CW_LAUNCH_ATTN(128); else CW_LAUNCH_ATTN(64);
#undef CW_LAUNCH_ATTN
    return (int)cudaGetLastError();
}

}  // namespace cw
