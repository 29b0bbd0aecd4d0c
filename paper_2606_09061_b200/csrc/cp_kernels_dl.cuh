// cp_kernels_dl.cuh -- the dual-lane tensor-core attention kernel of libcp (sm_100a only).
//
// One persistent CTA per SM runs TWO independent pipelines ("lanes") side by side, so that the
// tensor-bound prefill-chunk tiles (H3) and the HBM-bound decode streams (H4) of a mixed batch
// overlap on every SM instead of taking turns ("H3+H4+H5 are one logical launch
// driven by a persistent work list"):
//
//   lane T  chunk tiles (kKindTile); when the tile list is exhausted it also pulls decode items
//   lane S  decode / <=16-row items (kKindSwap) only
//
// Each lane owns a TMA producer warp, an MMA issuer warp, four softmax warps, a K/V tile ring in
// shared memory, its TMEM columns and its mbarriers; the lanes share nothing but the SM.
//
//   warpgroup 0: warp 0 producer T, warp 1 producer S, warp 2 MMA T, warp 3 MMA S  (64 regs)
//   warpgroup 1: softmax T (thread <-> Q-tile row)                                 (224 regs)
//   warpgroup 2: softmax S (thread <-> key of the tile)                            (128 regs)
//
//   kKindTile   S[128 rows x 128 keys] = Q K^T with Q held in TMEM (A operand from TMEM, written
//               once per item with tcgen05.st), P written back over S in TMEM as bf16 and consumed
//               as the A operand of O[128 x D] += P V.  Neither Q nor P touches shared memory, so
//               the smem crossbar carries only the K/V tiles (TMA writes + one MMA read each).
//   kKindSwap   <= 16 rows, D = 128: S^T[128 keys x 16] = K Q^T, O^T[128 d x 16] += V^T P^T.
//
// Operation: include/cp.h / DESIGN.md section 2.  Masking is by select, masked P is exactly 0.
#pragma once
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include "cp_internal.h"
#include "cp_ptx.cuh"

namespace cp {
namespace dl {

constexpr int kThreads = 384;
constexpr int kStagesT = 3, kStagesS = 3, kMaxStages = 4;
constexpr int kItemRing = 2;
constexpr int kTmemCols = 512;
// TMEM columns.  Lane T: S0, S1 (fp32 scores, P aliased over their first 64 columns), O, Q.
// Lane S: 16-column S^T0, S^T1, O^T.
constexpr uint32_t kColS[2][2] = {{0, 128}, {448, 464}};
constexpr uint32_t kColO[2] = {256, 480};
constexpr uint32_t kColQ = 384;
constexpr float kRescaleThreshold = 8.0f;      // log2 units: rescale O only when the max grew > 2^8
constexpr uint32_t kSmallBytes = 12288;        // per lane: Q^T (4 KiB) + double-buffered P^T (8 KiB)

template <int D>
struct Layout {
    static constexpr int kHalves = D / 64;                    // 64-element (128-byte) halves of D
    static constexpr uint32_t kSlotBytes = kHalves * 16384;   // one K or V tile: 128 keys x D bf16
    // slot: [16 row groups][kHalves][8 rows][128 B] (one TMA box per page = 2 row groups)
    static constexpr uint32_t kGroupBytes = kHalves * 1024;   // UMMA SBO of a K/V slot
    static constexpr uint32_t kPageBytes = 2 * kGroupBytes;
    static constexpr uint32_t kOffKv[2] = {0, kStagesT * kSlotBytes};
    static constexpr uint32_t kOffSmall[2] = {(kStagesT + kStagesS) * kSlotBytes,
                                              (kStagesT + kStagesS) * kSlotBytes + kSmallBytes};
    static constexpr uint32_t kOffMisc = kOffSmall[1] + kSmallBytes;
    static constexpr uint32_t kMiscBytes = 4096;
    static constexpr uint32_t kTotal = kOffMisc + kMiscBytes + 1024;   // + slack to align the base to 1024
};

struct LaneState {              // one per lane, in the misc region
    uint64_t kv_full[kMaxStages];
    uint64_t kv_empty[kMaxStages];
    uint64_t q_full;
    uint64_t s_full[2];
    uint64_t p_full[2];         // indexed by tile parity: a waiter can never be two phases behind
    uint64_t pv_done[2];        // PV of tile gt completes on pv_done[gt & 1]
    uint64_t item_full[kItemRing];
    uint64_t item_empty[kItemRing];
    WorkItem items[kItemRing];  // published by the lane's producer; kind < 0 = no more work
    float cmax[2][4][16];       // swap kind: per-warp column maxima, double buffered
    float lsum[4][16];          // swap kind: per-warp column sums at the end of an item
};

struct Misc {
    LaneState lane[2];
    uint32_t tmem_base;
};
static_assert(sizeof(Misc) <= 4096, "misc region too small");

struct Params {
    BatchMeta meta;
    Shape sh;
    const __nv_bfloat16* q;
    __nv_bfloat16* out;
    float* part_o;
    float2* part_ml;
    int32_t* counters;          // [0] next tile item, [1] next swap item, [2] finished CTAs
};

__device__ __forceinline__ uint32_t pack_bf16(float a, float b) {
    __nv_bfloat162 v = __floats2bfloat162_rn(a, b);
    return *reinterpret_cast<uint32_t*>(&v);
}

template <int N> __device__ __forceinline__ void reg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N> __device__ __forceinline__ void reg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }

// D[tmem] (+)= A[tmem] * B[smem]; issued by ONE thread.  A: lane = row, one 32-bit column holds
// two consecutive bf16 along K (16 K-elements = 8 columns per instruction).
__device__ __forceinline__ void umma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, bool accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
        ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"((uint32_t)accumulate)
        : "memory");
}

// ------------------------------------------------------------------------------------------
// producer warp of a lane: fetches work items, publishes them to the lane's MMA and softmax
// warps through a small smem ring, and streams the K and V tiles of each item into the lane's
// slot ring in consumption order K0, K1, V0, K2, V1, ..., K(n-1), V(n-2), V(n-1).  It runs ahead
// of the consumers by up to kStages tile loads, across item boundaries.  Page ids are prefetched
// 32 at a time (one per lane, three windows) so no dependent global load sits between TMA issues.
// ------------------------------------------------------------------------------------------
template <int D, int LANE>
__device__ __forceinline__ void producer(const Params& p, const CUtensorMap* tmap, uint8_t* smem, LaneState* ls, int lane) {
    using L = Layout<D>;
    constexpr int kStages = LANE == 0 ? kStagesT : kStagesS;
    uint8_t* kv_base = smem + L::kOffKv[LANE];
    uint32_t ld_base = 0, item_cnt = 0;          // ld_base: tile loads of all previous items
    bool tiles_left = LANE == 0;
    for (;;) {
        const uint32_t islot = item_cnt % kItemRing;
        int idx = -1;
        if (tiles_left) {
            if (lane == 0) idx = atomicAdd(&p.counters[0], 1);
            idx = __shfl_sync(0xffffffffu, idx, 0);
            if (idx >= p.meta.n_tile) { tiles_left = false; idx = -1; }
        }
        if (idx < 0) {
            if (lane == 0) idx = atomicAdd(&p.counters[1], 1);
            idx = __shfl_sync(0xffffffffu, idx, 0);
            idx = idx < p.meta.n_work - p.meta.n_tile ? idx + p.meta.n_tile : -1;
        }
        int w = 0;                               // one int32 of the 32-byte WorkItem per lane 0..7
        if (idx >= 0 && lane < 8) w = reinterpret_cast<const int32_t*>(p.meta.work + idx)[lane];
        if (idx < 0 && lane == 7) w = -1;        // kind = -1: sentinel
        ptx::mbar_wait(&ls->item_empty[islot], ((item_cnt / kItemRing) & 1) ^ 1);
        if (lane < 8) reinterpret_cast<int32_t*>(&ls->items[islot])[lane] = w;
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(&ls->item_full[islot]);
        ++item_cnt;
        if (idx < 0) break;
        const int req = __shfl_sync(0xffffffffu, w, 0), kv_head = __shfl_sync(0xffffffffu, w, 1);
        const int kv_begin = __shfl_sync(0xffffffffu, w, 4), kv_end = __shfl_sync(0xffffffffu, w, 5);
        const int n_tiles = (kv_end - kv_begin + kKeyTile - 1) / kKeyTile;
        const int32_t* bt = p.meta.block_table + p.meta.bt_off[req] + (kv_begin >> 4);
        const int n_pages_item = (kv_end - kv_begin + 15) >> 4;
        // page-id windows of 32 pages (4 tiles), one id per lane.  V tiles advance the window; the
        // K stream is at most one tile ahead of the V stream, so it reads window cur_w or cur_w + 1.
        int cur_w = 0;
        int win0 = lane < n_pages_item ? bt[lane] : 0;
        int win1 = 32 + lane < n_pages_item ? bt[32 + lane] : 0;
        int win2 = 64 + lane < n_pages_item ? bt[64 + lane] : 0;
        for (int i = 0; i < 2 * n_tiles; ++i) {
            int is_v, tile;
            if (i == 0) { is_v = 0; tile = 0; }
            else if (i == 2 * n_tiles - 1) { is_v = 1; tile = n_tiles - 1; }
            else if (i & 1) { is_v = 0; tile = (i + 1) >> 1; }
            else { is_v = 1; tile = (i >> 1) - 1; }
            if (is_v && (tile >> 2) > cur_w) {
                win0 = win1;
                win1 = win2;
                ++cur_w;
                const int pi = (cur_w + 2) * 32 + lane;
                win2 = pi < n_pages_item ? bt[pi] : 0;
            }
            const int win = (tile >> 2) == cur_w ? win0 : win1;
            const int n_pages = min(8, n_pages_item - tile * 8);          // 1..8
            const uint32_t ld = ld_base + i;
            const uint32_t slot = ld % kStages;
            ptx::mbar_wait(&ls->kv_empty[slot], ((ld / kStages) & 1) ^ 1);
            const bool leader = ptx::elect_one();
            if (leader) ptx::mbar_arrive_expect_tx(&ls->kv_full[slot], (uint32_t)n_pages * 16u * D * 2u);
            uint8_t* dst = kv_base + slot * L::kSlotBytes;
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const int pg = __shfl_sync(0xffffffffu, win, (tile & 3) * 8 + j);
                if (j < n_pages) {
                    const int slab = (pg * 2 + is_v) * p.sh.Hkv + kv_head;
                    if (leader) ptx::tma_load_5d(dst + j * L::kPageBytes, tmap, &ls->kv_full[slot], 0, 0, 0, 0, slab);
                }
            }
            __syncwarp();
        }
        ld_base += 2 * n_tiles;
    }
}

// ------------------------------------------------------------------------------------------
// MMA issuer warp of a lane (tcgen05.mma is issued by one elected thread; the warp stays
// convergent so descriptors live in uniform registers)
// ------------------------------------------------------------------------------------------
template <int D, int LANE>
__device__ __forceinline__ void mma_item(const WorkItem& it, uint32_t smem_base, LaneState* ls, uint32_t tmem,
                                         uint32_t& cons_cnt, uint32_t& gt, uint32_t item_cnt) {
    using L = Layout<D>;
    constexpr int kStages = LANE == 0 ? kStagesT : kStagesS;
    const int n_tiles = (__shfl_sync(0xffffffffu, it.kv_end - it.kv_begin, 0) + kKeyTile - 1) / kKeyTile;
    const bool swap = LANE == 1 || __shfl_sync(0xffffffffu, it.kind, 0) == kKindSwap;
    const uint32_t small = smem_base + L::kOffSmall[LANE], kv_base = smem_base + L::kOffKv[LANE];
    // tile kind: S = Q K^T (A = Q in TMEM, M 128 rows, N 128 keys); O += P V (A = P in TMEM, V MN-major B)
    // swap kind: S^T = K Q^T (M 128 keys, N 16);   O^T += V^T P^T (M 128 = D, N 16, V^T is MN-major A)
    const uint32_t idesc_qk = swap ? ptx::umma_idesc_bf16(128, 16, false, false) : ptx::umma_idesc_bf16(128, 128, false, false);
    const uint32_t idesc_pv = swap ? ptx::umma_idesc_bf16(128, 16, true, false) : ptx::umma_idesc_bf16(128, D, false, true);
    const uint32_t small_half = 2048;          // 16 rows x 128 B (Q^T / P^T halves in the swap kind)

    ptx::mbar_wait(&ls->q_full, item_cnt & 1);
    ptx::tc_fence_after();

    auto issue_qk = [&](uint32_t g) {          // g: global tile counter of the tile being scored
        const uint32_t slot = cons_cnt % kStages, buf = g & 1;
        ptx::mbar_wait(&ls->kv_full[slot], (cons_cnt / kStages) & 1);
        ptx::tc_fence_after();
        const uint32_t k_tile = kv_base + slot * L::kSlotBytes;
        const uint32_t d_tmem = tmem + kColS[LANE][buf];
        if (ptx::elect_one()) {
#pragma unroll
            for (int ks = 0; ks < D / 16; ++ks) {
                const uint32_t koff = (ks >> 2) * 1024 + (ks & 3) * 32;                // K slot: halves 1 KB apart
                const uint64_t k_desc = ptx::umma_desc_sw128(k_tile + koff, 16, L::kGroupBytes);
                if (LANE == 0 && !swap) {
                    umma_ts(d_tmem, tmem + kColQ + ks * 8, k_desc, idesc_qk, ks > 0);
                } else {
                    const uint32_t qoff = (ks >> 2) * small_half + (ks & 3) * 32;
                    ptx::umma_ss(d_tmem, k_desc, ptx::umma_desc_sw128(small + qoff, 16, 1024), idesc_qk, ks > 0);
                }
            }
            ptx::umma_commit(&ls->kv_empty[slot]);
            ptx::umma_commit(&ls->s_full[buf]);
        }
        __syncwarp();
        ++cons_cnt;
    };
    auto issue_pv = [&](bool first) {
        const uint32_t buf = gt & 1;
        ptx::mbar_wait(&ls->p_full[buf], (gt >> 1) & 1);
        const uint32_t slot = cons_cnt % kStages;
        ptx::mbar_wait(&ls->kv_full[slot], (cons_cnt / kStages) & 1);
        ptx::tc_fence_after();
        const uint32_t v_tile = kv_base + slot * L::kSlotBytes;
        const uint32_t d_tmem = tmem + kColO[LANE];
        if (ptx::elect_one()) {
#pragma unroll
            for (int ks = 0; ks < kKeyTile / 16; ++ks) {
                // V (MN-major): 16 key rows = 2 row groups (SBO apart); the next 64 d are 1 KB further (LBO)
                const uint64_t v_desc = ptx::umma_desc_sw128(v_tile + ks * L::kPageBytes, 1024, L::kGroupBytes);
                if (LANE == 0 && !swap) {
                    umma_ts(d_tmem, tmem + kColS[0][buf] + ks * 8, v_desc, idesc_pv, !first || ks > 0);
                } else {
                    const uint32_t poff = 4096 + buf * 4096 + (ks >> 2) * small_half + (ks & 3) * 32;   // P^T is double buffered
                    ptx::umma_ss(d_tmem, v_desc, ptx::umma_desc_sw128(small + poff, 16, 1024), idesc_pv, !first || ks > 0);
                }
            }
            ptx::umma_commit(&ls->kv_empty[slot]);
            ptx::umma_commit(&ls->pv_done[buf]);
        }
        __syncwarp();
        ++cons_cnt;
        ++gt;
    };

    // QK(k+1) is issued before PV(k) so the softmax of tile k overlaps the next score MMA.  p_full is
    // indexed by tile parity: the softmax of tile k+2 needs QK(k+2), which is issued only after
    // p_full[k & 1] of tile k was observed here, so a wait can never alias onto a later phase.
    issue_qk(gt);
    for (int k = 0; k < n_tiles; ++k) {
        if (k + 1 < n_tiles) issue_qk(gt + 1);
        issue_pv(k == 0);
    }
}

template <int D, int LANE>
__device__ __forceinline__ void mma_warp(uint32_t smem_base, Misc* misc, int lane) {
    LaneState* ls = &misc->lane[LANE];
    const uint32_t tmem = misc->tmem_base;
    uint32_t cons_cnt = 0, gt = 0, item_cnt = 0;
    for (;;) {
        const uint32_t islot = item_cnt % kItemRing;
        ptx::mbar_wait(&ls->item_full[islot], (item_cnt / kItemRing) & 1);
        const WorkItem it = ls->items[islot];
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(&ls->item_empty[islot]);
        if (it.kind < 0) break;
        mma_item<D, LANE>(it, smem_base, ls, tmem, cons_cnt, gt, item_cnt);
        ++item_cnt;
    }
}
