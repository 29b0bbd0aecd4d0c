// cp_kernels_tc.cuh -- the tensor-core attention kernel of libcp (sm_100a only).
//
// One persistent, warp-specialised kernel serves both kinds of work item of the mixed batch
// (H3 prefill-chunk tiles and H4 decode splits of SURVEY.md 8(a)), pulling items from the
// LPT-sorted work list through an atomic counter:
//
//   warp 0      producer: walks the block table, one TMA (cp.async.bulk.tensor, 128B swizzle)
//               per (page, 64-wide half of D) into a ring of K/V tile slots (128 keys each)
//   warp 1      issues tcgen05.mma (one thread), accumulators in TMEM
//   warps 2-5   softmax: tcgen05.ld S from TMEM, online softmax in fp32 (log2 domain, lazy
//               rescale), P -> bf16 -> swizzled smem, O rescale / epilogue from TMEM
//
//   kKindTile   S[128 rows x 128 keys] = Q K^T, O[128 x D] += P V.  Rows = (token, q head of
//               the KV group): 128/G tokens x G heads share one K/V stream (GQA packing).
//   kKindSwap   <= 16 rows (decode, tiny chunks), D = 128: the operands are swapped so the 128
//               keys of a tile are the MMA M dimension: S^T[128 keys x 16] = K Q^T,
//               O^T[128 d x 16] += V^T P^T.  The step is HBM-bound; the MMAs are ~6 % of it.
//
// Operation: include/cp.h / DESIGN.md section 2.  Masking is by select (never by adding
// -inf to garbage), P of masked keys is exactly 0, so stale finite data never leaks.
#pragma once
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include "cp_internal.h"
#include "cp_ptx.cuh"

namespace cp {

constexpr int kTcThreads = 192;
constexpr int kStages = 5;
constexpr int kTmemCols = 512;
constexpr uint32_t kColS0 = 0, kColS1 = 128, kColO = 256;
constexpr float kRescaleThreshold = 8.0f;      // log2 units: rescale O only when the max grew > 2^8

template <int D>
struct TcLayout {
    static constexpr int kHalves = D / 64;                 // 64-element (128-byte) halves of D
    static constexpr uint32_t kHalfBytes = 128 * 128;      // 128 rows x 128 B
    static constexpr uint32_t kQBytes = kHalves * kHalfBytes;
    static constexpr uint32_t kPBytes = 2 * kHalfBytes;    // 128 rows x 128 keys bf16
    static constexpr uint32_t kSlotBytes = kHalves * kHalfBytes;
    static constexpr uint32_t kOffQ = 0;
    static constexpr uint32_t kOffP = kQBytes;
    static constexpr uint32_t kOffKV = kOffP + kPBytes;
    static constexpr uint32_t kOffMisc = kOffKV + kStages * kSlotBytes;
    static constexpr uint32_t kMiscBytes = 1024;
    static constexpr uint32_t kTotal = kOffMisc + kMiscBytes + 1024;   // + slack to align the base to 1024
};

struct TcMisc {                 // lives in the misc region
    uint64_t kv_full[kStages];
    uint64_t kv_empty[kStages];
    uint64_t q_full;
    uint64_t s_full[2];
    uint64_t p_full;
    uint64_t pv_done;
    uint32_t tmem_base;
    int32_t item;
    float cmax[2][4][16];       // swap path: per-warp column maxima, double buffered
    float lsum[4][16];          // swap path: per-warp column sums at the end of an item
};
static_assert(sizeof(TcMisc) <= 1024, "misc region too small");

struct TcParams {
    BatchMeta meta;
    Shape sh;
    const __nv_bfloat16* q;
    __nv_bfloat16* out;
    float* part_o;
    float2* part_ml;
    int32_t* counters;          // [0] next item, [1] finished CTAs
};

__device__ __forceinline__ uint32_t pack_bf16(float a, float b) {
    __nv_bfloat162 v = __floats2bfloat162_rn(a, b);
    return *reinterpret_cast<uint32_t*>(&v);
}

// ------------------------------------------------------------------------------------------
// producer: stream the K and V tiles of one item into the slot ring, in consumption order
//   K0, K1, V0, K2, V1, ..., K(n-1), V(n-2), V(n-1)
// ------------------------------------------------------------------------------------------
template <int D>
__device__ __forceinline__ void tc_produce_item(const WorkItem& it, const BatchMeta& meta, const Shape& sh,
                                                const CUtensorMap* tmap, uint8_t* kv_base, TcMisc* misc,
                                                uint32_t& ld_cnt, int lane) {
    using L = TcLayout<D>;
    const int n_tiles = (it.kv_end - it.kv_begin + kKeyTile - 1) / kKeyTile;
    const int32_t* bt = meta.block_table + meta.bt_off[it.req];
    for (int i = 0; i < 2 * n_tiles; ++i) {
        int is_v, tile;
        if (i == 0) { is_v = 0; tile = 0; }
        else if (i == 2 * n_tiles - 1) { is_v = 1; tile = n_tiles - 1; }
        else if (i & 1) { is_v = 0; tile = (i + 1) >> 1; }
        else { is_v = 1; tile = (i >> 1) - 1; }
        const int ts = it.kv_begin + tile * kKeyTile;
        const int n_pages = (min(it.kv_end, ts + kKeyTile) - ts + 15) >> 4;     // 1..8
        const uint32_t slot = ld_cnt % kStages;
        const uint32_t parity = ((ld_cnt / kStages) & 1) ^ 1;
        ptx::mbar_wait(&misc->kv_empty[slot], parity);
        if (lane == 0) ptx::mbar_arrive_expect_tx(&misc->kv_full[slot], (uint32_t)n_pages * 16u * D * 2u);
        __syncwarp();
        if (lane < n_pages) {
            const int page = bt[(ts >> 4) + lane];
            const int slab = (page * 2 + is_v) * sh.Hkv + it.kv_head;
            uint8_t* dst = kv_base + slot * L::kSlotBytes + lane * 2048;
#pragma unroll
            for (int h = 0; h < L::kHalves; ++h)
                ptx::tma_load_3d(dst + h * L::kHalfBytes, tmap, &misc->kv_full[slot], h * 64, 0, slab);
        }
        __syncwarp();
        ++ld_cnt;
    }
}

// ------------------------------------------------------------------------------------------
// MMA issuer (one thread)
// ------------------------------------------------------------------------------------------
template <int D>
__device__ __forceinline__ void tc_mma_item(const WorkItem& it, uint32_t smem_base, TcMisc* misc, uint32_t tmem,
                                            uint32_t& cons_cnt, uint32_t& gt, uint32_t item_cnt) {
    using L = TcLayout<D>;
    const int n_tiles = (it.kv_end - it.kv_begin + kKeyTile - 1) / kKeyTile;
    const bool swap = it.kind == kKindSwap;
    const uint32_t q_base = smem_base + L::kOffQ, p_base = smem_base + L::kOffP, kv_base = smem_base + L::kOffKV;
    // tile kind: S = Q K^T (M 128 rows, N 128 keys); O += P V (M 128, N D, V is MN-major B)
    // swap kind: S^T = K Q^T (M 128 keys, N 16);     O^T += V^T P^T (M 128 = D, N 16, V^T is MN-major A)
    const uint32_t idesc_qk = swap ? ptx::umma_idesc_bf16(128, 16, false, false) : ptx::umma_idesc_bf16(128, 128, false, false);
    const uint32_t idesc_pv = swap ? ptx::umma_idesc_bf16(128, 16, true, false) : ptx::umma_idesc_bf16(128, D, false, true);
    const uint32_t small_half = 2048;          // 16 rows x 128 B (Q^T / P^T halves in the swap kind)

    ptx::mbar_wait(&misc->q_full, item_cnt & 1);
    ptx::tc_fence_after();

    auto issue_qk = [&](uint32_t buf) {
        const uint32_t slot = cons_cnt % kStages;
        ptx::mbar_wait(&misc->kv_full[slot], (cons_cnt / kStages) & 1);
        ptx::tc_fence_after();
        const uint32_t k_tile = kv_base + slot * L::kSlotBytes;
        const uint32_t d_tmem = tmem + (buf ? kColS1 : kColS0);
#pragma unroll
        for (int ks = 0; ks < D / 16; ++ks) {
            const uint32_t koff = (ks >> 2) * L::kHalfBytes + (ks & 3) * 32;
            if (!swap) {
                ptx::umma_ss(d_tmem, ptx::umma_desc_sw128(q_base + koff, 16, 1024),
                             ptx::umma_desc_sw128(k_tile + koff, 16, 1024), idesc_qk, ks > 0);
            } else {
                const uint32_t qoff = (ks >> 2) * small_half + (ks & 3) * 32;
                ptx::umma_ss(d_tmem, ptx::umma_desc_sw128(k_tile + koff, 16, 1024),
                             ptx::umma_desc_sw128(q_base + qoff, 16, 1024), idesc_qk, ks > 0);
            }
        }
        ptx::umma_commit(&misc->kv_empty[slot]);
        ptx::umma_commit(&misc->s_full[buf]);
        ++cons_cnt;
    };
    auto issue_pv = [&](bool first) {
        ptx::mbar_wait(&misc->p_full, gt & 1);
        const uint32_t slot = cons_cnt % kStages;
        ptx::mbar_wait(&misc->kv_full[slot], (cons_cnt / kStages) & 1);
        ptx::tc_fence_after();
        const uint32_t v_tile = kv_base + slot * L::kSlotBytes;
        const uint32_t d_tmem = tmem + kColO;
#pragma unroll
        for (int ks = 0; ks < kKeyTile / 16; ++ks) {
            // V: 16 key rows (= MMA K) of 128 B per 64-wide half of D; halves are kHalfBytes apart (LBO)
            const uint64_t v_desc = ptx::umma_desc_sw128(v_tile + ks * 2048, L::kHalfBytes, 1024);
            if (!swap) {
                const uint32_t poff = (ks >> 2) * L::kHalfBytes + (ks & 3) * 32;
                ptx::umma_ss(d_tmem, ptx::umma_desc_sw128(p_base + poff, 16, 1024), v_desc, idesc_pv, !first || ks > 0);
            } else {
                const uint32_t poff = (ks >> 2) * small_half + (ks & 3) * 32;
                ptx::umma_ss(d_tmem, v_desc, ptx::umma_desc_sw128(p_base + poff, 16, 1024), idesc_pv, !first || ks > 0);
            }
        }
        ptx::umma_commit(&misc->kv_empty[slot]);
        ptx::umma_commit(&misc->pv_done);
        ++cons_cnt;
        ++gt;
    };

    issue_qk(gt & 1);
    for (int k = 0; k < n_tiles; ++k) {
        if (k + 1 < n_tiles) issue_qk((gt + 1) & 1);
        issue_pv(k == 0);
    }
}

// ------------------------------------------------------------------------------------------
// softmax warps, tile kind: thread <-> row of the 128-row Q tile
// ------------------------------------------------------------------------------------------
template <int D>
__device__ __forceinline__ void tc_softmax_tile(const WorkItem& it, const TcParams& p, uint8_t* smem, TcMisc* misc,
                                                uint32_t tmem, uint32_t& gt, int row, uint32_t lane_base) {
    using L = TcLayout<D>;
    const Shape& sh = p.sh;
    const int G = sh.G;
    const int R = it.q_tokens * G;
    const int n_tiles = (it.kv_end - it.kv_begin + kKeyTile - 1) / kKeyTile;
    const int tok0 = p.meta.cu_q[it.req] + it.q_start;
    const int ctx = p.meta.ctx_off[it.req];
    const bool valid_row = row < R;
    const int tok = tok0 + row / G;
    const int head = it.kv_head * G + row % G;
    const float scale = sh.sm_scale * 1.4426950408889634f;

    // ---- Q tile -> smem (K-major, 128B swizzle): row r, 16-byte chunk c -> r*128 + ((c ^ (r&7)) << 4)
    {
        uint8_t* qs = smem + L::kOffQ + row * 128;
        const uint4* src = reinterpret_cast<const uint4*>(p.q + ((int64_t)tok * sh.Hq + head) * D);
#pragma unroll
        for (int c = 0; c < D / 8; ++c) {
            uint4 v = valid_row ? src[c] : make_uint4(0, 0, 0, 0);
            *reinterpret_cast<uint4*>(qs + (c >> 3) * L::kHalfBytes + (((c & 7) ^ (row & 7)) << 4)) = v;
        }
    }
    ptx::fence_proxy_async_smem();
    ptx::mbar_arrive(&misc->q_full);

    const int limit = valid_row ? min(it.kv_end, ctx + it.q_start + row / G + 1) : 0;   // causal, diagonal inclusive
    float m_ref = -INFINITY, l = 0.f;
    uint8_t* ps = smem + L::kOffP + row * 128;
    const uint32_t t_row = tmem + (lane_base << 16);

    for (int k = 0; k < n_tiles; ++k) {
        const int ts = it.kv_begin + k * kKeyTile;
        const uint32_t buf = gt & 1;
        ptx::mbar_wait(&misc->s_full[buf], (gt >> 1) & 1);
        ptx::tc_fence_after();
        uint32_t sr[128];
#pragma unroll
        for (int c = 0; c < 4; ++c) ptx::tmem_ld32(t_row + (buf ? kColS1 : kColS0) + c * 32, sr + c * 32);
        ptx::tmem_wait_ld();
        const int nvalid = max(0, min(kKeyTile, limit - ts));
        float m_t = -INFINITY;
        if (nvalid == kKeyTile) {
#pragma unroll
            for (int j = 0; j < 128; ++j) m_t = fmaxf(m_t, __uint_as_float(sr[j]));
        } else {
#pragma unroll
            for (int j = 0; j < 128; ++j) m_t = fmaxf(m_t, j < nvalid ? __uint_as_float(sr[j]) : -INFINITY);
        }
        m_t *= scale;                                   // scale > 0
        float alpha = 1.f;
        bool rescale = false;
        if (m_t > m_ref + kRescaleThreshold) {          // also the first finite max (m_ref = -inf)
            alpha = (m_ref == -INFINITY) ? 0.f : ptx::ex2(m_ref - m_t);
            m_ref = m_t;
            rescale = true;
        }
        const float neg_m = (m_ref == -INFINITY) ? 0.f : -m_ref;
        float sum = 0.f;
        uint32_t pk[64];
        if (nvalid == kKeyTile) {
#pragma unroll
            for (int j = 0; j < 128; j += 2) {
                float a = ptx::ex2(fmaf(__uint_as_float(sr[j]), scale, neg_m));
                float b = ptx::ex2(fmaf(__uint_as_float(sr[j + 1]), scale, neg_m));
                sum += a + b;
                pk[j >> 1] = pack_bf16(a, b);
            }
        } else {
#pragma unroll
            for (int j = 0; j < 128; j += 2) {
                float a = j < nvalid ? ptx::ex2(fmaf(__uint_as_float(sr[j]), scale, neg_m)) : 0.f;
                float b = j + 1 < nvalid ? ptx::ex2(fmaf(__uint_as_float(sr[j + 1]), scale, neg_m)) : 0.f;
                sum += a + b;
                pk[j >> 1] = pack_bf16(a, b);
            }
        }
        l = l * alpha + sum;
        if (k > 0) {                                    // PV(k-1) done: P smem free, O readable
            ptx::mbar_wait(&misc->pv_done, (gt - 1) & 1);
            ptx::tc_fence_after();
        }
#pragma unroll
        for (int c = 0; c < 16; ++c)
            *reinterpret_cast<uint4*>(ps + (c >> 3) * L::kHalfBytes + (((c & 7) ^ (row & 7)) << 4)) =
                make_uint4(pk[4 * c], pk[4 * c + 1], pk[4 * c + 2], pk[4 * c + 3]);
        if (k > 0 && __any_sync(0xffffffffu, rescale)) {
#pragma unroll
            for (int c = 0; c < D / 32; ++c) {
                uint32_t o[32];
                ptx::tmem_ld32(t_row + kColO + c * 32, o);
                ptx::tmem_wait_ld();
#pragma unroll
                for (int j = 0; j < 32; ++j) o[j] = __float_as_uint(__uint_as_float(o[j]) * alpha);
                ptx::tmem_st32(t_row + kColO + c * 32, o);
            }
            ptx::tmem_wait_st();
        }
        ptx::fence_proxy_async_smem();
        ptx::tc_fence_before();
        ptx::mbar_arrive(&misc->p_full);
        ++gt;
    }

    // ---- epilogue: O row from TMEM -> out (bf16, normalised) or split workspace (fp32, unnormalised)
    ptx::mbar_wait(&misc->pv_done, (gt - 1) & 1);
    ptx::tc_fence_after();
    const float inv = 1.f / l;
#pragma unroll
    for (int c = 0; c < D / 32; ++c) {
        uint32_t o[32];
        ptx::tmem_ld32(t_row + kColO + c * 32, o);
        ptx::tmem_wait_ld();
        if (valid_row) {
            if (it.partial_row < 0) {
                uint4* dst = reinterpret_cast<uint4*>(p.out + ((int64_t)tok * sh.Hq + head) * D + c * 32);
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    dst[j] = make_uint4(pack_bf16(__uint_as_float(o[8 * j]) * inv, __uint_as_float(o[8 * j + 1]) * inv),
                                        pack_bf16(__uint_as_float(o[8 * j + 2]) * inv, __uint_as_float(o[8 * j + 3]) * inv),
                                        pack_bf16(__uint_as_float(o[8 * j + 4]) * inv, __uint_as_float(o[8 * j + 5]) * inv),
                                        pack_bf16(__uint_as_float(o[8 * j + 6]) * inv, __uint_as_float(o[8 * j + 7]) * inv));
            } else {
                uint4* dst = reinterpret_cast<uint4*>(p.part_o + ((int64_t)it.partial_row + row) * D + c * 32);
#pragma unroll
                for (int j = 0; j < 8; ++j) dst[j] = make_uint4(o[4 * j], o[4 * j + 1], o[4 * j + 2], o[4 * j + 3]);
            }
        }
    }
    if (valid_row && it.partial_row >= 0) p.part_ml[(int64_t)it.partial_row + row] = make_float2(m_ref, l);
    ptx::tc_fence_before();
}

// ------------------------------------------------------------------------------------------
// softmax warps, swap kind (D = 128, <= 16 rows): thread <-> key of the tile (S^T lane) during
// the key loop, thread <-> d (O^T lane) for rescale / epilogue.  Column c = (token, head) row.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void tc_softmax_swap(const WorkItem& it, const TcParams& p, uint8_t* smem, TcMisc* misc,
                                                uint32_t tmem, uint32_t& gt, int row, uint32_t lane_base, int swarp) {
    constexpr int D = 128;
    using L = TcLayout<D>;
    const Shape& sh = p.sh;
    const int G = sh.G;
    const int R = it.q_tokens * G;                       // <= 16
    const int n_tiles = (it.kv_end - it.kv_begin + kKeyTile - 1) / kKeyTile;
    const int tok0 = p.meta.cu_q[it.req] + it.q_start;
    const int ctx = p.meta.ctx_off[it.req];
    const float scale = sh.sm_scale * 1.4426950408889634f;
    const int lane = row & 31;

    // ---- Q^T -> smem: B operand [16 rows][D], K-major, 128B swizzle, halves 2 KB apart
    for (int id = row; id < 16 * (D / 8); id += 128) {
        const int r = id >> 4, c = id & 15;
        uint4 v = make_uint4(0, 0, 0, 0);
        if (r < R) {
            const int tok = tok0 + r / G, head = it.kv_head * G + r % G;
            v = *reinterpret_cast<const uint4*>(p.q + ((int64_t)tok * sh.Hq + head) * D + c * 8);
        }
        *reinterpret_cast<uint4*>(smem + L::kOffQ + (c >> 3) * 2048 + r * 128 + (((c & 7) ^ (r & 7)) << 4)) = v;
    }
    ptx::fence_proxy_async_smem();
    ptx::mbar_arrive(&misc->q_full);

    float m_ref[16], l_part[16];
    int limit[16];
#pragma unroll
    for (int c = 0; c < 16; ++c) {
        m_ref[c] = -INFINITY;
        l_part[c] = 0.f;
        limit[c] = c < R ? min(it.kv_end, ctx + it.q_start + c / G + 1) : 0;
    }
    const uint32_t t_row = tmem + (lane_base << 16);
    // P^T element (col c, key `row`): B operand [16 rows][128 keys], K-major, halves (64 keys) 2 KB apart
    uint8_t* pt = smem + L::kOffP + (row >> 6) * 2048 + (row & 7) * 2;
    const int pchunk = (row & 63) >> 3;

    for (int k = 0; k < n_tiles; ++k) {
        const int key = it.kv_begin + k * kKeyTile + row;
        const uint32_t buf = gt & 1;
        ptx::mbar_wait(&misc->s_full[buf], (gt >> 1) & 1);
        ptx::tc_fence_after();
        uint32_t sr[16];
        ptx::tmem_ld16(t_row + (buf ? kColS1 : kColS0), sr);
        ptx::tmem_wait_ld();
        float sv[16];
#pragma unroll
        for (int c = 0; c < 16; ++c) {
            sv[c] = key < limit[c] ? __uint_as_float(sr[c]) * scale : -INFINITY;
            float w = sv[c];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) w = fmaxf(w, __shfl_xor_sync(0xffffffffu, w, o));
            if (lane == c) misc->cmax[k & 1][swarp][c] = w;       // lanes 0..15 publish one column each
        }
        ptx::named_bar_sync(1, 128);
        bool any_rescale = false;
        float alpha[16];
#pragma unroll
        for (int c = 0; c < 16; ++c) {
            const float m_t = fmaxf(fmaxf(misc->cmax[k & 1][0][c], misc->cmax[k & 1][1][c]),
                                    fmaxf(misc->cmax[k & 1][2][c], misc->cmax[k & 1][3][c]));
            alpha[c] = 1.f;
            if (m_t > m_ref[c] + kRescaleThreshold) {
                alpha[c] = (m_ref[c] == -INFINITY) ? 0.f : ptx::ex2(m_ref[c] - m_t);
                m_ref[c] = m_t;
                any_rescale = true;
            }
            const float pc = key < limit[c] ? ptx::ex2(sv[c] - m_ref[c]) : 0.f;
            l_part[c] = l_part[c] * alpha[c] + pc;
            sv[c] = pc;
        }
        if (k > 0) {
            ptx::mbar_wait(&misc->pv_done, (gt - 1) & 1);
            ptx::tc_fence_after();
        }
#pragma unroll
        for (int c = 0; c < 16; ++c)
            *reinterpret_cast<__nv_bfloat16*>(pt + c * 128 + ((pchunk ^ (c & 7)) << 4)) = __float2bfloat16_rn(sv[c]);
        if (k > 0 && any_rescale) {                      // uniform over the 128 threads
            uint32_t o[16];
            ptx::tmem_ld16(t_row + kColO, o);
            ptx::tmem_wait_ld();
#pragma unroll
            for (int c = 0; c < 16; ++c) o[c] = __float_as_uint(__uint_as_float(o[c]) * alpha[c]);
            ptx::tmem_st16(t_row + kColO, o);
            ptx::tmem_wait_st();
        }
        ptx::fence_proxy_async_smem();
        ptx::tc_fence_before();
        ptx::mbar_arrive(&misc->p_full);
        ++gt;
    }

    // ---- column sums over the 128 key lanes
#pragma unroll
    for (int c = 0; c < 16; ++c) {
        float w = l_part[c];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) w += __shfl_xor_sync(0xffffffffu, w, o);
        if (lane == c) misc->lsum[swarp][c] = w;
    }
    ptx::named_bar_sync(1, 128);
    // ---- epilogue: O^T[d = row][c] -> out / workspace
    ptx::mbar_wait(&misc->pv_done, (gt - 1) & 1);
    ptx::tc_fence_after();
    uint32_t o[16];
    ptx::tmem_ld16(t_row + kColO, o);
    ptx::tmem_wait_ld();
#pragma unroll
    for (int c = 0; c < 16; ++c) {
        if (c < R) {
            const float lc = misc->lsum[0][c] + misc->lsum[1][c] + misc->lsum[2][c] + misc->lsum[3][c];
            if (it.partial_row < 0) {
                const int tok = tok0 + c / G, head = it.kv_head * G + c % G;
                p.out[((int64_t)tok * sh.Hq + head) * D + row] = __float2bfloat16_rn(__uint_as_float(o[c]) / lc);
            } else {
                p.part_o[((int64_t)it.partial_row + c) * D + row] = __uint_as_float(o[c]);
                if (row == c) p.part_ml[(int64_t)it.partial_row + c] = make_float2(m_ref[c], lc);
            }
        }
    }
    ptx::tc_fence_before();
    ptx::named_bar_sync(1, 128);                         // lsum / cmax are reused by the next item
}

// ------------------------------------------------------------------------------------------
// the kernel
// ------------------------------------------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(kTcThreads, 1)
attn_tc_kernel(const TcParams p, const __grid_constant__ CUtensorMap tmap) {
    using L = TcLayout<D>;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    TcMisc* misc = reinterpret_cast<TcMisc*>(smem + L::kOffMisc);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        for (int i = 0; i < kStages; ++i) { ptx::mbar_init(&misc->kv_full[i], 1); ptx::mbar_init(&misc->kv_empty[i], 1); }
        ptx::mbar_init(&misc->q_full, 128);
        ptx::mbar_init(&misc->s_full[0], 1);
        ptx::mbar_init(&misc->s_full[1], 1);
        ptx::mbar_init(&misc->p_full, 128);
        ptx::mbar_init(&misc->pv_done, 1);
        ptx::fence_barrier_init();
        ptx::prefetch_tmap(&tmap);
    }
    if (warp == 1) ptx::tmem_alloc(&misc->tmem_base, kTmemCols);
    // stale shared memory may hold NaN bit patterns; tiles are only partly overwritten by short
    // requests, and 0 x NaN would poison the accumulators
    for (uint32_t i = threadIdx.x * 16; i < L::kOffMisc; i += kTcThreads * 16)
        *reinterpret_cast<uint4*>(smem + i) = make_uint4(0, 0, 0, 0);
    ptx::fence_proxy_async_smem();
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem = misc->tmem_base;

    uint32_t ld_cnt = 0, cons_cnt = 0, gt = 0, item_cnt = 0;
    while (true) {
        if (threadIdx.x == 0) misc->item = atomicAdd(&p.counters[0], 1);
        __syncthreads();
        const int item = misc->item;
        if (item >= p.meta.n_work) break;
        const WorkItem it = p.meta.work[item];
        if (warp == 0) {
            tc_produce_item<D>(it, p.meta, p.sh, &tmap, smem + L::kOffKV, misc, ld_cnt, lane);
        } else if (warp == 1) {
            if (lane == 0) tc_mma_item<D>(it, ptx::smem_u32(smem), misc, tmem, cons_cnt, gt, item_cnt);
            __syncwarp();
        } else {
            const uint32_t lane_base = (warp & 3) * 32;
            const int row = lane_base + lane;
            if (it.kind == kKindSwap) {
                if constexpr (D == 128) tc_softmax_swap(it, p, smem, misc, tmem, gt, row, lane_base, warp & 3);
            } else {
                tc_softmax_tile<D>(it, p, smem, misc, tmem, gt, row, lane_base);
            }
        }
        ++item_cnt;
        __syncthreads();
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 1) ptx::tmem_dealloc(tmem, kTmemCols);
    if (threadIdx.x == 0) {
        __threadfence();
        if (atomicAdd(&p.counters[1], 1) == (int)gridDim.x - 1) {      // last CTA re-arms the counters
            p.counters[0] = 0;
            p.counters[1] = 0;
            __threadfence();
        }
    }
}

}  // namespace cp
