// Kernel 1: fused RoPE + KV scatter (cw_append_kv) and the pool export kernel (cw_gather_kv).  sm_100a.
//
// For each suffix token at absolute position p (readings c4, §4):
//     q_roped = RoPE(q, p);  pool_K[slot(p)] = RoPE(k, p);  pool_V[slot(p)] = v;  slot(p) = (table[p/16], p%16)
// HBM-bound: every byte is read once and written once.  One CTA (128 threads) walks tokens grid-stride; inside a
// token a thread owns "units" = one 16-byte chunk of the low half of a head plus its RoPE partner chunk in the
// high half, so all global accesses are 16-byte vectors and 8 consecutive threads cover one full 128-byte line.
// The pool block layout is the tcgen05 canonical 128B-swizzled tile (cacheweaver.h: cw_pool_offset).
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include <algorithm>

#include "cw_internal.h"

namespace cw {

__device__ __forceinline__ uint4 ld_stream(const void* p) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ void st_stream(void* p, const uint4& v) {
    asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};"
                 :: "l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

__device__ __forceinline__ float2 bf2_to_f2(uint32_t u) {
    return make_float2(__uint_as_float(u << 16), __uint_as_float(u & 0xFFFF0000u));
}
__device__ __forceinline__ uint32_t f2_to_bf2(float a, float b) {
    __nv_bfloat162 h = __floats2bfloat162_rn(a, b);
    return *reinterpret_cast<uint32_t*>(&h);
}

// rotate one (lo, hi) chunk pair: cs = 8 x {cos, sin} fp32 for the 8 frequencies of this chunk (in registers)
__device__ __forceinline__ void rope_pair(uint4& lo, uint4& hi, const float4 (&cs)[4]) {
    uint32_t* l = reinterpret_cast<uint32_t*>(&lo);
    uint32_t* h = reinterpret_cast<uint32_t*>(&hi);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const float4 t = cs[j];                         // {cos0, sin0, cos1, sin1}
        float2 a = bf2_to_f2(l[j]), b = bf2_to_f2(h[j]);
        float x0 = a.x * t.x - b.x * t.y, y0 = b.x * t.x + a.x * t.y;
        float x1 = a.y * t.z - b.y * t.w, y1 = b.y * t.z + a.y * t.w;
        l[j] = f2_to_bf2(x0, x1);
        h[j] = f2_to_bf2(y0, y1);
    }
}

// element offset of dim d (multiple of 8) of token-in-block t inside one (block, kv head) run of 16*D elements
template <int D>
__device__ __forceinline__ int pool_chunk_offset(int t, int d) {
    return (t >> 3) * (8 * D) + (d >> 6) * 512 + (t & 7) * 64 + ((((d & 63) >> 3) ^ (t & 7)) << 3);
}

template <int D, int THREADS>
__global__ void __launch_bounds__(THREADS) append_kv_kernel(
    const __nv_bfloat16* __restrict__ q, const __nv_bfloat16* __restrict__ k, const __nv_bfloat16* __restrict__ v,
    __nv_bfloat16* __restrict__ q_roped, __nv_bfloat16* __restrict__ k_pool, __nv_bfloat16* __restrict__ v_pool,
    const float* __restrict__ rope_table, const int32_t* __restrict__ cu, const int32_t* __restrict__ ncached,
    const int32_t* __restrict__ tables, int max_blocks, int B, int T, int Hq, int Hkv, int max_position, int num_blocks) {
    constexpr int CPH = D / 16;                       // chunk pairs (units) per head
    const int g = Hq / Hkv, tpt = 128 / g;
    const int uq = Hq * CPH, uk = Hkv * CPH;
    const int units = uq + 2 * uk;
    // A CTA's tokens ascend, so most of them belong to the request of the token before: its descriptor is kept in registers
    // and the binary search (a chain of dependent loads in front of every token's payload loads) only runs when a token
    // leaves [q_begin, q_end).
    int r = -1, q_begin = 0, q_end = 0, nc_r = 0;
    for (int tok = blockIdx.x; tok < T; tok += gridDim.x) {
        if (r < 0 || tok < q_begin || tok >= q_end) {
            // request of this token: largest r with cu[r] <= tok
            int lo = 0, hi = B;
            while (hi - lo > 1) {
                int mid = (lo + hi) >> 1;
                if (__ldg(cu + mid) <= tok) lo = mid; else hi = mid;
            }
            r = lo;
            q_begin = __ldg(cu + r);
            q_end = __ldg(cu + r + 1);
            nc_r = __ldg(ncached + r);
        }
        const int s_len = q_end - q_begin, tl = tok - q_begin;
        int p = nc_r + tl;
        // q_roped tile: tpt tokens x g heads per (kv head, tile); rows of a tile are stored [64-dim half][row][64], 128B-swizzled
        const int qt = tl / tpt, tloc = tl - qt * tpt;
        const int rows_valid = min(tpt, s_len - qt * tpt) * g;
        const size_t q_tile_base = (size_t)q_begin * Hq * D + (size_t)qt * (tpt * g) * D;
        // A token whose position has no RoPE row or no table slot, or whose table entry is not a pool block, is skipped: nothing
        // of it is written (no clamping to a wrong rotation, no store outside the pool).  cw_prefill_attn reports a request
        // that is too long through its error flag.
        // cu is unchecked device data as well: a row outside its request's slice (non-monotone cu) or a slice that leaves
        // [0, T) is skipped too, so every q_roped store below stays inside the request's own part of the T*Hq*D buffer.
        const bool pos_ok = p >= 0 && p < max_position && (p >> 4) < max_blocks && q_begin >= 0 && tl < s_len &&
                            s_len <= T - q_begin;
        const int blk = pos_ok ? __ldg(tables + (size_t)r * max_blocks + (p >> 4)) : -1;
        if (blk < 0 || blk >= num_blocks) continue;
        const int tib = p & 15;
        const int prow = p;
        // A thread's units are THREADS apart and THREADS % CPH == 0, so all of them rotate the same 8 frequencies: the
        // {cos, sin} pairs are loaded once per token and thread (they would otherwise double the L1 load traffic).
        static_assert(THREADS % CPH == 0, "chunk index must be the same for every unit of a thread");
        float4 cs[4];
        {
            const float4* cs_row = reinterpret_cast<const float4*>(rope_table + (size_t)prow * D) + (threadIdx.x % CPH) * 4;
#pragma unroll
            for (int j = 0; j < 4; ++j) cs[j] = __ldg(cs_row + j);
        }
        // Units are processed in groups of kUnroll per thread: all loads of a group are issued before the first store, so a
        // thread keeps 2 * kUnroll 16-byte loads in flight (the kernel is bound by bytes in flight, not by arithmetic).
        constexpr int kUnroll = 3;
        for (int u0 = threadIdx.x; u0 < units; u0 += kUnroll * THREADS) {
            uint4 lo[kUnroll], hi[kUnroll];
#pragma unroll
            for (int i = 0; i < kUnroll; ++i) {
                const int u = u0 + i * THREADS;
                if (u < units) {
                    const __nv_bfloat16* src;
                    if (u < uq) src = q + ((size_t)tok * Hq + u / CPH) * D + (u % CPH) * 8;
                    else if (u < uq + uk) src = k + ((size_t)tok * Hkv + (u - uq) / CPH) * D + ((u - uq) % CPH) * 8;
                    else src = v + ((size_t)tok * Hkv + (u - uq - uk) / CPH) * D + ((u - uq - uk) % CPH) * 8;
                    lo[i] = ld_stream(src);
                    hi[i] = ld_stream(src + D / 2);
                }
            }
#pragma unroll
            for (int i = 0; i < kUnroll; ++i) {
                const int u = u0 + i * THREADS;
                if (u >= units) break;
                if (u < uq) {
                    const int h = u / CPH, c = u % CPH;
                    rope_pair(lo[i], hi[i], cs);
                    const int kvh = h / g, row = tloc * g + (h - kvh * g);
                    __nv_bfloat16* qb = q_roped + q_tile_base + (size_t)kvh * s_len * g * D + row * 64;
                    const int d0 = c * 8, d1 = c * 8 + D / 2;
                    st_stream(qb + (d0 >> 6) * rows_valid * 64 + ((((d0 & 63) >> 3) ^ (row & 7)) << 3), lo[i]);
                    st_stream(qb + (d1 >> 6) * rows_valid * 64 + ((((d1 & 63) >> 3) ^ (row & 7)) << 3), hi[i]);
                } else {
                    const bool is_k = u < uq + uk;
                    const int uu = is_k ? u - uq : u - uq - uk, h = uu / CPH, c = uu % CPH;
                    if (is_k) rope_pair(lo[i], hi[i], cs);
                    __nv_bfloat16* base = (is_k ? k_pool : v_pool) + ((size_t)blk * Hkv + h) * (16 * D);
                    st_stream(base + pool_chunk_offset<D>(tib, c * 8), lo[i]);
                    st_stream(base + pool_chunk_offset<D>(tib, c * 8 + D / 2), hi[i]);
                }
            }
        }
    }
}

int launch_append_kv(const cw_config& cfg, const void* q, const void* k, const void* v, void* q_roped,
                     const int32_t* cu, const int32_t* ncached, const int32_t* tables, int32_t max_blocks,
                     int32_t B, int32_t T, int num_sms, void* stream) {
    if (T == 0) return 0;
    auto s = static_cast<cudaStream_t>(stream);
    // threads per CTA: the multiple of 32 (<= 128) that leaves the fewest idle lanes in the last round over the token's
    // units (8B: 384 units = 3 x 128; 70B: 640 = 5 x 128; Qwen2.5-7B: 288 = 3 x 96) — idle lanes are bytes not in flight
    const int units = (cfg.num_q_heads + 2 * cfg.num_kv_heads) * (cfg.head_dim / 16);
    int64_t grid = 0;
    int threads = 128, best_waste = 1 << 30;
    for (int t = 128; t >= 64; t -= 32) {
        const int waste = (units + t - 1) / t * t - units;
        if (waste < best_waste) { best_waste = waste; threads = t; }
    }
    // grid = one full wave of resident CTAs (occupancy is set by registers, asked from the runtime once per variant):
    // a larger grid-stride grid would run a partial second wave
#define CW_LAUNCH_APPEND(DD, TT)                                                                                \
    static int occ_##DD##_##TT = 0;                                                                             \
    if (occ_##DD##_##TT == 0 &&                                                                                 \
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_##DD##_##TT, append_kv_kernel<DD, TT>, TT, 0) != cudaSuccess) \
        occ_##DD##_##TT = 2048 / TT;                                                                            \
    grid = std::min<int64_t>(T, (int64_t)num_sms * std::max(1, occ_##DD##_##TT));                               \
    append_kv_kernel<DD, TT><<<(unsigned)grid, TT, 0, s>>>(                                                               \
        (const __nv_bfloat16*)q, (const __nv_bfloat16*)k, (const __nv_bfloat16*)v, (__nv_bfloat16*)q_roped,     \
        (__nv_bfloat16*)cfg.k_pool, (__nv_bfloat16*)cfg.v_pool, (const float*)cfg.rope_table, cu, ncached,      \
        tables, max_blocks, B, T, cfg.num_q_heads, cfg.num_kv_heads, cfg.max_position, cfg.num_blocks)
#define CW_LAUNCH_APPEND_D(DD)                                                                                  \
    do {                                                                                                        \
        if (threads == 128) { CW_LAUNCH_APPEND(DD, 128); }                                                      \
        else if (threads == 96) { CW_LAUNCH_APPEND(DD, 96); }                                                   \
        else { CW_LAUNCH_APPEND(DD, 64); }                                                                      \
    } while (0)
    if (cfg.head_dim == 128) CW_LAUNCH_APPEND_D(128); else CW_LAUNCH_APPEND_D(64);
#undef CW_LAUNCH_APPEND_D
#undef CW_LAUNCH_APPEND
    return (int)cudaGetLastError();
}

// ---- export: pool -> plain [n, Hkv, D] ---------------------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(128) gather_kv_kernel(
    const __nv_bfloat16* __restrict__ k_pool, const __nv_bfloat16* __restrict__ v_pool,
    const int32_t* __restrict__ table, int n, int Hkv, __nv_bfloat16* __restrict__ k_out,
    __nv_bfloat16* __restrict__ v_out) {
    constexpr int CH = D / 8;
    const int per_tok = Hkv * CH;
    for (int tok = blockIdx.x; tok < n; tok += gridDim.x) {
        const int blk = __ldg(table + (tok >> 4)), tib = tok & 15;
        for (int u = threadIdx.x; u < per_tok; u += 128) {
            const int h = u / CH, c = u % CH;
            const size_t src = ((size_t)blk * Hkv + h) * (16 * D) + pool_chunk_offset<D>(tib, c * 8);
            const size_t dst = ((size_t)tok * Hkv + h) * D + c * 8;
            *reinterpret_cast<uint4*>(k_out + dst) = *reinterpret_cast<const uint4*>(k_pool + src);
            *reinterpret_cast<uint4*>(v_out + dst) = *reinterpret_cast<const uint4*>(v_pool + src);
        }
    }
}

int launch_gather_kv(const cw_config& cfg, const int32_t* table, int32_t n, void* k_out, void* v_out, int num_sms, void* stream) {
    if (n == 0) return 0;
    const int grid = n < num_sms * 8 ? n : num_sms * 8;
    auto s = static_cast<cudaStream_t>(stream);
    if (cfg.head_dim == 128)
        gather_kv_kernel<128><<<grid, 128, 0, s>>>((const __nv_bfloat16*)cfg.k_pool, (const __nv_bfloat16*)cfg.v_pool,
                                                   table, n, cfg.num_kv_heads, (__nv_bfloat16*)k_out, (__nv_bfloat16*)v_out);
    else
        gather_kv_kernel<64><<<grid, 128, 0, s>>>((const __nv_bfloat16*)cfg.k_pool, (const __nv_bfloat16*)cfg.v_pool,
                                                  table, n, cfg.num_kv_heads, (__nv_bfloat16*)k_out, (__nv_bfloat16*)v_out);
    return (int)cudaGetLastError();
}

}  // namespace cw
