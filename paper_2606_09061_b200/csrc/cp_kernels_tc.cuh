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

constexpr int kProducers = 2;                // TMA producer warps (issue rate scales with warps)
constexpr int kTcThreads = 32 * (kProducers + 5);   // producers, MMA issuer, 4 softmax warps
constexpr int kStages = 5;
constexpr int kTmemCols = 512;
constexpr int kItemRing = 2;
constexpr uint32_t kColS0 = 0, kColS1 = 128, kColO = 256;
constexpr float kRescaleThreshold = 8.0f;      // log2 units: rescale O only when the max grew > 2^8

template <int D>
struct TcLayout {
    static constexpr int kHalves = D / 64;                 // 64-element (128-byte) halves of D
    static constexpr uint32_t kHalfBytes = 128 * 128;      // 128 rows x 128 B
    static constexpr uint32_t kQBytes = kHalves * kHalfBytes;
    static constexpr uint32_t kPBytes = 2 * kHalfBytes;    // 128 rows x 128 keys bf16
    static constexpr uint32_t kSlotBytes = kHalves * kHalfBytes;
    // K/V slot: [16 row groups][kHalves][8 rows][128 B] (one TMA box per page = 2 row groups)
    static constexpr uint32_t kGroupBytes = kHalves * 1024;   // UMMA SBO of a K/V slot
    static constexpr uint32_t kPageBytes = 2 * kGroupBytes;
    static constexpr uint32_t kOffQ = 0;
    static constexpr uint32_t kOffP = kQBytes;
    static constexpr uint32_t kOffKV = kOffP + kPBytes;
    static constexpr uint32_t kOffMisc = kOffKV + kStages * kSlotBytes;
    static constexpr uint32_t kMiscBytes = 2048;
    static constexpr uint32_t kTotal = kOffMisc + kMiscBytes + 1024;   // + slack to align the base to 1024
};

// Optional role-level wait-time profile (build with -DCP_TC_PROF; debugging aid only).
#ifdef CP_TC_PROF2
#define CP_STAMP(id) do { if (threadIdx.x == 32 * (kProducers + 2)) { long long t__ = clock64(); misc->prof[id] += (unsigned long long)(t__ - tprev__); tprev__ = t__; } } while (0)
#define CP_STAMP_INIT long long tprev__ = clock64()
#else
#define CP_STAMP(id) do {} while (0)
#define CP_STAMP_INIT do {} while (0)
#endif
#ifdef CP_TC_PROF
#define CP_PWAIT(id, bar, par)                                                        \
    do {                                                                              \
        const long long t0__ = clock64();                                             \
        ptx::mbar_wait(bar, par);                                                     \
        if (threadIdx.x == 0 || threadIdx.x == 32 * kProducers || threadIdx.x == 32 * (kProducers + 2)) \
            misc->prof[id] += (unsigned long long)(clock64() - t0__);                 \
    } while (0)
#else
#define CP_PWAIT(id, bar, par) ptx::mbar_wait(bar, par)
#endif

struct TcMisc {                 // lives in the misc region
    uint64_t kv_full[kStages];
    uint64_t kv_empty[kStages];
    uint64_t q_full;
    uint64_t s_full[2];
    uint64_t p_full;
    uint64_t pv_done[2];        // PV of tile gt completes on pv_done[gt & 1]
    uint64_t item_full[kItemRing];
    uint64_t item_empty[kItemRing];
    WorkItem items[kItemRing];  // published by the producer warp; kind < 0 = no more work
    uint32_t tmem_base;
#if defined(CP_TC_PROF) || defined(CP_TC_PROF2)
    unsigned long long prof[16];
#endif
    float cmax[2][4][16];       // swap path: per-warp column maxima, double buffered
    float lsum[4][16];          // swap path: per-warp column sums at the end of an item
};
static_assert(sizeof(TcMisc) <= 2048, "misc region too small");

struct TcParams {
    BatchMeta meta;
    Shape sh;
    const __nv_bfloat16* q;
    __nv_bfloat16* out;
    float* part_o;
    float2* part_ml;
    int32_t* counters;          // [0] next item, [1] finished CTAs
    unsigned long long* prof;   // [grid][16] wait-time profile (CP_TC_PROF builds), else unused
};

__device__ __forceinline__ uint32_t pack_bf16(float a, float b) {
    __nv_bfloat162 v = __floats2bfloat162_rn(a, b);
    return *reinterpret_cast<uint32_t*>(&v);
}

// ------------------------------------------------------------------------------------------
// producer warp: fetches work items (atomic counter), publishes them to the other roles through
// a small smem ring, and streams the K and V tiles of each item into the slot ring in
// consumption order  K0, K1, V0, K2, V1, ..., K(n-1), V(n-2), V(n-1)  (tile kind) or
// K0, V0, K1, V1, ... (swap kind).  It runs ahead of the
// consumers by up to kStages tile loads, across item boundaries.  Page ids are prefetched 32 at
// a time (one per lane) so no dependent global load sits between two TMA issues.
// ------------------------------------------------------------------------------------------
template <int D>
__device__ __forceinline__ void tc_producer(const TcParams& p, const CUtensorMap* tmap, uint8_t* kv_base,
                                            TcMisc* misc, int lane, int pw) {
    using L = TcLayout<D>;
    uint32_t ld_base = 0, item_cnt = 0;          // ld_base: tile loads of all previous items
    for (;;) {
        const uint32_t islot = item_cnt % kItemRing;
        int w;
        if (pw == 0) {                           // producer 0 fetches the next item and publishes it
            int idx = 0;
            if (lane == 0) idx = atomicAdd(&p.counters[0], 1);
            idx = __shfl_sync(0xffffffffu, idx, 0);
            const bool done = idx >= p.meta.n_work;
            w = 0;                               // one int32 of the 32-byte WorkItem per lane 0..7
            if (!done && lane < 8) w = reinterpret_cast<const int32_t*>(p.meta.work + idx)[lane];
            if (done && lane == 7) w = -1;       // kind = -1: sentinel
            CP_PWAIT(0, &misc->item_empty[islot], ((item_cnt / kItemRing) & 1) ^ 1);
            if (lane < 8) reinterpret_cast<int32_t*>(&misc->items[islot])[lane] = w;
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(&misc->item_full[islot]);
        } else {
            CP_PWAIT(0, &misc->item_full[islot], (item_cnt / kItemRing) & 1);
            w = lane < 8 ? reinterpret_cast<const int32_t*>(&misc->items[islot])[lane] : 0;
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(&misc->item_empty[islot]);
        }
        ++item_cnt;
        if (__shfl_sync(0xffffffffu, w, 7) < 0) break;
        const int req = __shfl_sync(0xffffffffu, w, 0), kv_head = __shfl_sync(0xffffffffu, w, 1);
        const int kv_begin = __shfl_sync(0xffffffffu, w, 4), kv_end = __shfl_sync(0xffffffffu, w, 5);
        const int n_tiles = (kv_end - kv_begin + kKeyTile - 1) / kKeyTile;
        const int32_t* bt = p.meta.block_table + p.meta.bt_off[req] + (kv_begin >> 4);
        const int n_pages_item = (kv_end - kv_begin + 15) >> 4;
        // page-id windows of 32 pages (4 tiles), one id per lane: cur = window cur_w, nxt = the next.
        // This warp's tile sequence is monotone, so windows only ever advance.
        int cur_w = 0;
        int cur = lane < n_pages_item ? bt[lane] : 0;
        int nxt = 32 + lane < n_pages_item ? bt[32 + lane] : 0;
        const bool swap = __shfl_sync(0xffffffffu, w, 7) == kKindSwap;
        for (int i = pw; i < 2 * n_tiles; i += kProducers) {
            int is_v, tile;
            if (swap) { is_v = i & 1; tile = i >> 1; }                   // K0, V0, K1, V1, ...
            else if (i == 0) { is_v = 0; tile = 0; }
            else if (i == 2 * n_tiles - 1) { is_v = 1; tile = n_tiles - 1; }
            else if (i & 1) { is_v = 0; tile = (i + 1) >> 1; }
            else { is_v = 1; tile = (i >> 1) - 1; }
            while ((tile >> 2) > cur_w) {
                cur = nxt;
                ++cur_w;
                const int pi = (cur_w + 1) * 32 + lane;
                nxt = pi < n_pages_item ? bt[pi] : 0;
            }
            const int n_pages = min(8, n_pages_item - tile * 8);          // 1..8
            const uint32_t ld = ld_base + i;
            const uint32_t slot = ld % kStages;
            CP_PWAIT(1, &misc->kv_empty[slot], ((ld / kStages) & 1) ^ 1);
            const bool leader = ptx::elect_one();
            if (leader) ptx::mbar_arrive_expect_tx(&misc->kv_full[slot], (uint32_t)n_pages * 16u * D * 2u);
            uint8_t* dst = kv_base + slot * L::kSlotBytes;
            // every operand below is warp-uniform (shuffle from a uniform lane), so the TMA issue
            // needs no per-lane serialisation
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const int pg = __shfl_sync(0xffffffffu, cur, (tile & 3) * 8 + j);
                if (j < n_pages) {
                    const int slab = (pg * 2 + is_v) * p.sh.Hkv + kv_head;
                    if (leader) ptx::tma_load_5d(dst + j * L::kPageBytes, tmap, &misc->kv_full[slot], 0, 0, 0, 0, slab);
                }
            }
            __syncwarp();
        }
        ld_base += 2 * n_tiles;
    }
}

// ------------------------------------------------------------------------------------------
// MMA issuer (one thread)
// ------------------------------------------------------------------------------------------
template <int D>
__device__ __forceinline__ void tc_mma_item(const WorkItem& it, uint32_t smem_base, TcMisc* misc, uint32_t tmem,
                                            uint32_t& cons_cnt, uint32_t& gt, uint32_t item_cnt) {
    using L = TcLayout<D>;
    // the whole warp runs this convergently with warp-uniform values; only the tcgen05 issue is
    // elected, so descriptors stay in uniform registers
    const int n_tiles = (__shfl_sync(0xffffffffu, it.kv_end - it.kv_begin, 0) + kKeyTile - 1) / kKeyTile;
    const bool swap = __shfl_sync(0xffffffffu, it.kind, 0) == kKindSwap;
    const uint32_t q_base = smem_base + L::kOffQ, p_base = smem_base + L::kOffP, kv_base = smem_base + L::kOffKV;
    // tile kind: S = Q K^T (M 128 rows, N 128 keys); O += P V (M 128, N D, V is MN-major B)
    // swap kind: S^T = K Q^T (M 128 keys, N 16);     O^T += V^T P^T (M 128 = D, N 16, V^T is MN-major A)
    const uint32_t idesc_qk = swap ? ptx::umma_idesc_bf16(128, 16, false, false) : ptx::umma_idesc_bf16(128, 128, false, false);
    const uint32_t idesc_pv = swap ? ptx::umma_idesc_bf16(128, 16, true, false) : ptx::umma_idesc_bf16(128, D, false, true);
    const uint32_t small_half = 2048;          // 16 rows x 128 B (Q^T / P^T halves in the swap kind)

    CP_PWAIT(2, &misc->q_full, item_cnt & 1);
    ptx::tc_fence_after();

    auto issue_qk = [&](uint32_t buf) {
        const uint32_t slot = cons_cnt % kStages;
        CP_PWAIT(3, &misc->kv_full[slot], (cons_cnt / kStages) & 1);
        ptx::tc_fence_after();
        const uint32_t k_tile = kv_base + slot * L::kSlotBytes;
        const uint32_t d_tmem = tmem + (buf ? kColS1 : kColS0);
        if (ptx::elect_one()) {
#pragma unroll
        for (int ks = 0; ks < D / 16; ++ks) {
            const uint32_t qoff_t = (ks >> 2) * L::kHalfBytes + (ks & 3) * 32;     // Q tile: halves 16 KB apart
            const uint32_t koff = (ks >> 2) * 1024 + (ks & 3) * 32;                // K slot: halves 1 KB apart
            const uint64_t k_desc = ptx::umma_desc_sw128(k_tile + koff, 16, L::kGroupBytes);
            if (!swap) {
                ptx::umma_ss(d_tmem, ptx::umma_desc_sw128(q_base + qoff_t, 16, 1024), k_desc, idesc_qk, ks > 0);
            } else {
                const uint32_t qoff = (ks >> 2) * small_half + (ks & 3) * 32;
                ptx::umma_ss(d_tmem, k_desc, ptx::umma_desc_sw128(q_base + qoff, 16, 1024), idesc_qk, ks > 0);
            }
        }
        ptx::umma_commit(&misc->kv_empty[slot]);
        ptx::umma_commit(&misc->s_full[buf]);
        }
        __syncwarp();
        ++cons_cnt;
    };
    auto issue_pv = [&](bool first) {
        CP_PWAIT(4, &misc->p_full, gt & 1);
        const uint32_t slot = cons_cnt % kStages;
        CP_PWAIT(5, &misc->kv_full[slot], (cons_cnt / kStages) & 1);
        ptx::tc_fence_after();
        const uint32_t v_tile = kv_base + slot * L::kSlotBytes;
        const uint32_t d_tmem = tmem + kColO;
        if (ptx::elect_one()) {
#pragma unroll
        for (int ks = 0; ks < kKeyTile / 16; ++ks) {
            // V (MN-major): 16 key rows = 2 row groups (SBO apart); the next 64 d are 1 KB further (LBO)
            const uint64_t v_desc = ptx::umma_desc_sw128(v_tile + ks * L::kPageBytes, 1024, L::kGroupBytes);
            if (!swap) {
                const uint32_t poff = (ks >> 2) * L::kHalfBytes + (ks & 3) * 32;
                ptx::umma_ss(d_tmem, ptx::umma_desc_sw128(p_base + poff, 16, 1024), v_desc, idesc_pv, !first || ks > 0);
            } else {
                const uint32_t poff = (gt & 1) * 4096 + (ks >> 2) * small_half + (ks & 3) * 32;   // P^T is double buffered
                ptx::umma_ss(d_tmem, v_desc, ptx::umma_desc_sw128(p_base + poff, 16, 1024), idesc_pv, !first || ks > 0);
            }
        }
        ptx::umma_commit(&misc->kv_empty[slot]);
        ptx::umma_commit(&misc->pv_done[gt & 1]);
        }
        __syncwarp();
        ++cons_cnt;
        ++gt;
    };

    if (swap) {
        // QK(k+1) is issued only after p_full(k) was observed: the swap-kind softmax has no other
        // back-pressure (P^T is double buffered), and without it a fast softmax could complete
        // p_full phase k+1 before this thread looked at phase k (parity aliasing -> deadlock).
        // The step is HBM-bound; the lost QK/softmax overlap is not on the critical path.
        for (int k = 0; k < n_tiles; ++k) {
            issue_qk(gt & 1);
            issue_pv(k == 0);
        }
    } else {
        issue_qk(gt & 1);
        for (int k = 0; k < n_tiles; ++k) {
            if (k + 1 < n_tiles) issue_qk((gt + 1) & 1);
            issue_pv(k == 0);
        }
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
        CP_PWAIT(6, &misc->s_full[buf], (gt >> 1) & 1);
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
            CP_PWAIT(7, &misc->pv_done[(gt - 1) & 1], ((gt - 1) >> 1) & 1);
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
    CP_PWAIT(8, &misc->pv_done[(gt - 1) & 1], ((gt - 1) >> 1) & 1);
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
// softmax warps, swap kind (D = 128, R <= RC <= 16 rows): thread <-> key of the tile (S^T lane)
// during the key loop, thread <-> d (O^T lane) for rescale / epilogue.  Column c = (token, head)
// row; columns in [R, RC) are computed as fully masked.  Straight-line code per column so the
// independent chains interleave; the column max is one REDUX per column and warp.
// ------------------------------------------------------------------------------------------
template <int RC>
__device__ __forceinline__ void tc_softmax_swap(const WorkItem& it, const TcParams& p, uint8_t* smem, TcMisc* misc,
                                                uint32_t tmem, uint32_t& gt, int row, uint32_t lane_base, int swarp) {
    constexpr int D = 128;
    using L = TcLayout<D>;
    const Shape& sh = p.sh;
    const int G = sh.G;
    const int R = it.q_tokens * G;                       // <= RC
    const int n_tiles = (it.kv_end - it.kv_begin + kKeyTile - 1) / kKeyTile;
    const int tok0 = p.meta.cu_q[it.req] + it.q_start;
    const int ctx = p.meta.ctx_off[it.req];
    const float scale = sh.sm_scale * 1.4426950408889634f;
    const int lane = row & 31;
    CP_STAMP_INIT;

    // ---- Q^T -> smem: B operand [16 rows][D], K-major, 128B swizzle, halves 2 KB apart
    for (int id = row; id < RC * (D / 8); id += 128) {
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
    CP_STAMP(10);

    float m_ref[RC], l_part[RC];
    int limit[RC];
#pragma unroll
    for (int c = 0; c < RC; ++c) {
        m_ref[c] = -INFINITY;
        l_part[c] = 0.f;
        limit[c] = c < R ? min(it.kv_end, ctx + it.q_start + c / G + 1) : 0;
    }
    const uint32_t t_row = tmem + (lane_base << 16);
    // P^T element (col c, key `row`): B operand [16 rows][128 keys], K-major, halves (64 keys) 2 KB apart
    uint8_t* pt = smem + L::kOffP + (row >> 6) * 2048 + (row & 7) * 2;
    const int pchunk = (row & 63) >> 3;

    for (int k = 0; k < n_tiles; ++k) {
        CP_STAMP(12);
        const int key = it.kv_begin + k * kKeyTile + row;
        const uint32_t buf = gt & 1;
        CP_PWAIT(6, &misc->s_full[buf], (gt >> 1) & 1);
        ptx::tc_fence_after();
        CP_STAMP(0);
        uint32_t sr[RC];
        ptx::tmem_ld<RC>(t_row + (buf ? kColS1 : kColS0), sr);
        ptx::tmem_wait_ld();
        CP_STAMP(1);
        float sv[RC];
        int* cm = reinterpret_cast<int*>(&misc->cmax[k & 1][swarp][0]);
#pragma unroll
        for (int c = 0; c < RC; ++c) {
            sv[c] = key < limit[c] ? __uint_as_float(sr[c]) * scale : -INFINITY;
            const int w = __reduce_max_sync(0xffffffffu, ptx::f2ord(sv[c]));
            if (lane == 0) cm[c] = w;
        }
        CP_STAMP(2);
        ptx::named_bar_sync(1, 128);
        CP_STAMP(3);
        bool any_rescale = false;
        float alpha[RC];
        const int* cm0 = reinterpret_cast<const int*>(&misc->cmax[k & 1][0][0]);
#pragma unroll
        for (int c = 0; c < RC; ++c) {
            const float m_t = ptx::ord2f(max(max(cm0[c], cm0[16 + c]), max(cm0[32 + c], cm0[48 + c])));
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
        CP_STAMP(4);
        if (k >= 2) {                                    // PV(gt-2) done: this P^T buffer is free again
            CP_PWAIT(7, &misc->pv_done[gt & 1], ((gt - 2) >> 1) & 1);
        }
        {
            uint8_t* ptb = pt + (gt & 1) * 4096;
#pragma unroll
            for (int c = 0; c < RC; ++c)
                *reinterpret_cast<__nv_bfloat16*>(ptb + c * 128 + ((pchunk ^ (c & 7)) << 4)) = __float2bfloat16_rn(sv[c]);
        }
        CP_STAMP(5);
        if (k > 0 && any_rescale) {                      // uniform over the 128 threads
            CP_PWAIT(9, &misc->pv_done[(gt - 1) & 1], ((gt - 1) >> 1) & 1);
            ptx::tc_fence_after();
            uint32_t o[RC];
            ptx::tmem_ld<RC>(t_row + kColO, o);
            ptx::tmem_wait_ld();
#pragma unroll
            for (int c = 0; c < RC; ++c) o[c] = __float_as_uint(__uint_as_float(o[c]) * alpha[c]);
            ptx::tmem_st<RC>(t_row + kColO, o);
            ptx::tmem_wait_st();
        }
        CP_STAMP(6);
        ptx::fence_proxy_async_smem();
        CP_STAMP(7);
        ptx::tc_fence_before();
        ptx::mbar_arrive(&misc->p_full);
        CP_STAMP(8);
        ++gt;
    }
    CP_STAMP(12);

    // ---- column sums over the 128 key lanes
#pragma unroll
    for (int c = 0; c < RC; ++c) {
        float w = l_part[c];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) w += __shfl_xor_sync(0xffffffffu, w, o);
        if (lane == 0) misc->lsum[swarp][c] = w;
    }
    ptx::named_bar_sync(1, 128);
    // ---- epilogue: O^T[d = row][c] -> out / workspace
    CP_PWAIT(8, &misc->pv_done[(gt - 1) & 1], ((gt - 1) >> 1) & 1);
    ptx::tc_fence_after();
    uint32_t o[RC];
    ptx::tmem_ld<RC>(t_row + kColO, o);
    ptx::tmem_wait_ld();
#pragma unroll
    for (int c = 0; c < RC; ++c) {
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
    CP_STAMP(9);
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
        ptx::mbar_init(&misc->pv_done[0], 1);
        ptx::mbar_init(&misc->pv_done[1], 1);
        for (int i = 0; i < kItemRing; ++i) { ptx::mbar_init(&misc->item_full[i], 1); ptx::mbar_init(&misc->item_empty[i], 128 + kProducers); }
        ptx::fence_barrier_init();
        ptx::prefetch_tmap(&tmap);
    }
#if defined(CP_TC_PROF) || defined(CP_TC_PROF2)
    if (threadIdx.x < 16) misc->prof[threadIdx.x] = 0;
    const long long t_start__ = clock64();
#endif
    if (warp == kProducers) ptx::tmem_alloc(&misc->tmem_base, kTmemCols);
    // stale shared memory may hold NaN bit patterns; tiles are only partly overwritten by short
    // requests, and 0 x NaN would poison the accumulators
    for (uint32_t i = threadIdx.x * 16; i < L::kOffMisc; i += kTcThreads * 16)
        *reinterpret_cast<uint4*>(smem + i) = make_uint4(0, 0, 0, 0);
    ptx::fence_proxy_async_smem();
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    const uint32_t tmem = misc->tmem_base;

    // Roles run decoupled: the producer publishes items through misc->items[]; each consumer copies
    // the item, frees the ring slot at once, and works from its private copy.
    if (warp < kProducers) {
        tc_producer<D>(p, &tmap, smem + L::kOffKV, misc, lane, warp);
    } else if (warp == kProducers) {
        uint32_t cons_cnt = 0, gt = 0, item_cnt = 0;
        for (;;) {
            const uint32_t islot = item_cnt % kItemRing;
            CP_PWAIT(10, &misc->item_full[islot], (item_cnt / kItemRing) & 1);
            const WorkItem it = misc->items[islot];
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(&misc->item_empty[islot]);
            if (it.kind < 0) break;
            tc_mma_item<D>(it, ptx::smem_u32(smem), misc, tmem, cons_cnt, gt, item_cnt);
            ++item_cnt;
        }
    } else {
        const uint32_t lane_base = (warp & 3) * 32;
        const int row = lane_base + lane;
        uint32_t gt = 0, item_cnt = 0;
        for (;;) {
            const uint32_t islot = item_cnt % kItemRing;
            CP_PWAIT(11, &misc->item_full[islot], (item_cnt / kItemRing) & 1);
            const WorkItem it = misc->items[islot];
            ptx::mbar_arrive(&misc->item_empty[islot]);
            if (it.kind < 0) break;
            if (it.kind == kKindSwap) {
                if constexpr (D == 128) {
                    const int R = it.q_tokens * p.sh.G;
                    if (R <= 4) tc_softmax_swap<4>(it, p, smem, misc, tmem, gt, row, lane_base, warp & 3);
                    else if (R <= 8) tc_softmax_swap<8>(it, p, smem, misc, tmem, gt, row, lane_base, warp & 3);
                    else tc_softmax_swap<16>(it, p, smem, misc, tmem, gt, row, lane_base, warp & 3);
                }
            } else {
                tc_softmax_tile<D>(it, p, smem, misc, tmem, gt, row, lane_base);
            }
            ++item_cnt;
        }
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (warp == kProducers) ptx::tmem_dealloc(tmem, kTmemCols);
#if defined(CP_TC_PROF) || defined(CP_TC_PROF2)
    if (threadIdx.x == 0) misc->prof[15] = (unsigned long long)(clock64() - t_start__);
    __syncthreads();
    if (threadIdx.x < 16 && p.prof) p.prof[blockIdx.x * 16 + threadIdx.x] = misc->prof[threadIdx.x];
#endif
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
