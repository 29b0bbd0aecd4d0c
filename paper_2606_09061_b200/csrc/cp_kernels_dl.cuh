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
// Each lane owns its TMA producer warps, MMA issuer warp(s), four softmax warps, a K/V tile ring in
// shared memory, its TMEM columns and its mbarriers; the lanes share nothing but the SM.
//
//   warpgroups 0-1: warps 0-2 TMA producers T, warps 3-4 TMA producers S, warps 5-6 MMA T (score
//                   blocks / PV blocks), warp 7 MMA S                               (56 regs)
//   warpgroup 2:    softmax T (thread <-> Q-tile row; also the decode items lane T runs once the
//                   tile list is exhausted: thread <-> key)                         (232 regs)
//   warpgroup 3:    softmax S (thread <-> key of the tile)                         (160 regs)
// (Measured alternatives, round 1 -- two softmax warpgroups per score tile or taking half-tiles in
// turn, chunked score reads, software-pipelined score loads, L2 prefetch, other ring splits -- are
// in DESIGN.md section 7 with their timelines.)
//
//   kKindTile   S[128 rows x 64 keys] = Q K^T per half-tile (four S buffers in flight), with Q held
//               in TMEM (A operand from TMEM, written once per item with tcgen05.st), P written back
//               over S in TMEM as bf16 and consumed as the A operand of O[128 x D] += P V.  Neither Q
//               nor P touches shared memory, so the smem crossbar carries only the K/V tiles (TMA
//               writes + one MMA read each).
//   kKindSwap   <= 16 rows, D = 128: S^T[128 keys x 16] = K Q^T, O^T[128 d x 16] += V^T P^T.
//
//
// SPLIT mode (template parameter; the instantiation the host launches for TENSOR-BOUND batches): there are no
// decode streams worth a lane of their own, and a chunk tile is bound by its softmax (16 K exponentials, the
// row maxima and sums of a 128 x 128 score tile on ONE warpgroup take ~2200 cycles against 1024 cycles of MMA).
// So lane S's warpgroup joins lane T: the two softmax warpgroups split every score tile by COLUMNS -- warpgroup w
// takes keys [64 w, 64 w + 64) of each 128-key tile for all 128 rows -- and exchange their row maxima through
// shared memory (one named barrier per tile and pair of warps that hold the same rows), so both keep the same running reference maximum
// without ever talking again; each keeps the partial row sum of its own columns and owns half of the O columns
// for the (rare) rescale and for the epilogue.  Scores come as ONE N = 128 block per tile into one of two
// 128-column S buffers (a tcgen05.mma has a ~50-cycle minimum: N = 64 blocks run at 51 cycles per instruction
// against a 32-cycle floor, N = 128 blocks at their 64-cycle floor), PV as one K = 128 block; a
// single issuer warp; all five producer warps feed one 6-slot ring.  Decode items of such a batch run after its
// tile items on warpgroup 2 (swap kind).
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

constexpr int kThreads = 512;
// SPLIT mode: kSplitWG softmax warpgroups share every chunk tile (each thread <-> a row and 128 / kSplitWG of its
// keys).  Two (512 threads) is the measured optimum on B200: four (768 threads, 96 registers per softmax thread,
// 32 keys per thread) runs the chunk-only batch in 361 us against 331 us and the 70B-shaped batch in 37.8 ms
// against 34.7 ms -- the per-tile fixed cost of a warp (barrier waits, TMEM round trips, the maximum exchange)
// is paid by twice as many warps in lockstep.
#ifndef DL_SPLIT_WG
#define DL_SPLIT_WG 2
#endif
constexpr int kSplitWG = DL_SPLIT_WG;
static_assert(kSplitWG == 2 || kSplitWG == 4, "SPLIT: two or four softmax warpgroups");
constexpr int kSplitCols = 128 / kSplitWG;           // keys of a tile per softmax thread
constexpr int kThreadsSplit = 256 + 128 * kSplitWG;
template <bool SPLIT> __host__ __device__ constexpr int threads_of() { return SPLIT ? kThreadsSplit : kThreads; }
constexpr int kStagesT = 3, kStagesS = 3, kMaxStages = 6;
constexpr int kStagesSplit = 6, kProdSplit = 5;  // SPLIT mode: one ring, all five producer warps
constexpr int kStagesS8 = 6;                     // fp8 pools: lane S's ring is six 16 KiB slots (same bytes in flight)
constexpr uint32_t kSlot8Bytes = 16384, kPage8Bytes = 2048;   // a 128-key fp8 tile (D = 128); a 16-token page slab
constexpr int kProdT = 3, kProdS = 2;         // TMA producer warps per lane (kProdT + kProdS + 3 MMA warps = 8 warps)
// a producer waiting for slot reuse may be at most one phase behind only if kProd <= kStages
static_assert(kProdT <= kStagesT && kProdS <= kStagesS && kProdT + kProdS == 5, "producer / stage configuration");
constexpr int kItemRing = 2;
constexpr int kTmemCols = 512;
// TMEM columns.  Lane T: four 64-column S buffers at 0 / 64 / 128 / 192 (fp32 scores of a 64-key
// half-tile, P aliased over their first 32 columns; the swap kind uses columns 0 and 128), O, Q.
// Lane S: 16-column S^T0, S^T1, O^T.
__host__ __device__ constexpr uint32_t col_s(int lane, uint32_t buf) { return lane == 0 ? buf * 128u : 448u + buf * 16u; }
__host__ __device__ constexpr uint32_t col_o(int lane) { return lane == 0 ? 256u : 480u; }
constexpr uint32_t kColQ = 384;
#ifndef DL_POLY_EVERY
#define DL_POLY_EVERY 4
#endif
// tile kind: in the POLY instantiation of the kernel every kPolyEvery-th exponential runs on the FMA pipe.
// Measured on B200 (final kernel): 4 -> -3.5 % on chunk-only batches, -2 % on the 70B-shaped chunk, +1 % on the
// mixed batch of configs[2] (HBM-bound: the exponentials are not its limit and the extra FMA-pipe instructions
// are).  The host therefore picks the instantiation per batch: POLY for tensor-bound batches only (cp_api.cu).
constexpr int kPolyEvery = DL_POLY_EVERY;
constexpr float kRescaleThreshold = 8.0f;      // log2 units: rescale O only when the max grew > 2^8
constexpr uint32_t kSmallBytes = 12288;        // per lane: Q^T (4 KiB) + double-buffered P^T (8 KiB)

template <int D, bool SPLIT = false>
struct Layout {
    static constexpr int kHalves = D / 64;                    // 64-element (128-byte) halves of D
    static constexpr uint32_t kSlotBytes = kHalves * 16384;   // one K or V tile: 128 keys x D bf16
    // slot: [16 row groups][kHalves][8 rows][128 B] (one TMA box per page = 2 row groups)
    static constexpr uint32_t kGroupBytes = kHalves * 1024;   // UMMA SBO of a K/V slot
    static constexpr uint32_t kPageBytes = 2 * kGroupBytes;
    static constexpr int kStages = SPLIT ? kStagesSplit : kStagesT;     // of lane 0's ring
    // SPLIT: the same 6 slots form ONE ring (lane 0); small[0] also holds the warpgroups' exchange arrays
    static constexpr uint32_t kOffKv[2] = {0, SPLIT ? 0 : kStagesT * kSlotBytes};
    static constexpr uint32_t kOffSmall[2] = {(kStagesT + kStagesS) * kSlotBytes,
                                              (kStagesT + kStagesS) * kSlotBytes + kSmallBytes};
    static constexpr uint32_t kOffMisc = kOffSmall[1] + kSmallBytes;
    static constexpr uint32_t kMiscBytes = 4096;
    static constexpr uint32_t kTotal = kOffMisc + kMiscBytes + 1024;   // + slack to align the base to 1024
};


struct LaneState {              // one per lane, in the misc region
    uint64_t kv_full[kMaxStages];
    uint64_t kv_empty[kMaxStages];
    // q_full / p_full exist per item kind ("set" 0 = tile kind, set 1 = swap kind), each with its
    // own phase counters; lane S uses set 1 only
    uint64_t q_full[2];
    uint64_t s_full[2];
    uint64_t p_full[2][2];      // [set][tile parity]: a waiter can never be two phases behind
    uint64_t pv_done[2];        // PV of tile gt completes on pv_done[gt & 1]
    // lane T, tile kind: a 128-key tile is scored as two 64-key half-tiles; FOUR 64-column S buffers
    // (index = half-tile counter & 3) keep four softmax <-> MMA round trips in flight
    uint64_t ts_full[4];        // scores of half-tile j are in S buffer j & 3
    uint64_t tp_full[4];        // P of half-tile j is in place
    uint64_t tpv_done[4];       // PV of half-tile j has completed
    uint64_t pv_issued[4];      // the PV issuer has put PV(j) into the pipe
    uint64_t item_full[kItemRing];
    uint64_t item_empty[kItemRing];
    WorkItem items[kItemRing];  // published by the lane's producer; kind < 0 = no more work
    int32_t aux[kItemRing];     // BatchMeta::work_aux of the item
    int32_t cur_aux;            // aux word of the item the lane's softmax warpgroup is working on (kept out of registers)
    int32_t last_split;         // swap kind: this item's split was the last of its group to arrive
    float cmax[2][4][16];       // swap kind: per-warp column maxima, double buffered
    float lsum[4][16];          // swap kind: per-warp column sums at the end of an item
    float qs[8];                // fp8 swap kind: per-row scale of the quantised Q^T
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
    const float* kv_scale;      // fp8 pools: [block][K|V][kv head][slot] power-of-two row scales, else unused
    int32_t* group_cnt;         // [fused groups] arrivals of the splits of a group merged in this kernel (all 0 between launches)
    // APPEND instantiation (decode-only batches over bf16 pages: H2 inside this kernel, no append launch)
    const uint4* k_new;         // [T, Hkv, D] rows of the step, or nullptr (the caller wrote the pages: only the page tails are cleared)
    const uint4* v_new;
    __nv_bfloat16* cache;       // the pool the descriptors point into
};

// element e of a half-tile row: MUFU or FMA-pipe exponential (e is a constant after unrolling)
template <bool POLY>
__device__ __forceinline__ float ex2_sel(float x, int e) {
    return (POLY && kPolyEvery > 0 && e % (kPolyEvery > 0 ? kPolyEvery : 1) == (kPolyEvery > 0 ? kPolyEvery : 1) - 1) ? ptx::ex2_poly(x) : ptx::ex2(x);
}

__device__ __forceinline__ uint32_t pack_bf16(float a, float b) {
    __nv_bfloat162 v = __floats2bfloat162_rn(a, b);
    return *reinterpret_cast<uint32_t*>(&v);
}

// One arrival per warp (after all its lanes are done) instead of 32: 128 single-word smem atomics
// per barrier phase were a measurable part of every tile's critical path.
__device__ __forceinline__ void warp_arrive(uint64_t* bar) {
    __syncwarp();
    if ((threadIdx.x & 31) == 0) ptx::mbar_arrive(bar);
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
// producer warps of a lane.  Producer 0 fetches work items (atomic counters) and publishes them to
// the lane's other warps through a small smem ring; all kProd producers stream the K and V tiles of
// each item into the lane's slot ring in consumption order K0, K1, V0, K2, V1, ..., K(n-1), V(n-2),
// V(n-1), load number ld (counted over the whole kernel) going to producer ld mod kProd.  The eight boxes (4 KiB page
// slabs) of a tile are issued by eight lanes of the warp in ONE instruction: a single thread sustains one box per
// ~230 cycles, so a leader issuing them one after the other held a ring slot ~1800 cycles before its last byte was
// even requested -- with three slots per lane that capped the decode lane of a mixed batch at ~39 GB/s (148 lanes:
// 5.8 TB/s, below the HBM rate) while lane T was busy with chunk tiles (configs[2] 629 -> 608 us).
// Together the producers run ahead of the consumers by up to kStages tile loads, across item
// boundaries.  Page ids are prefetched 32 at a time (one per lane of the warp, two windows; each
// producer's tile sequence is monotone) so no dependent global load sits between two TMA issues.
// ------------------------------------------------------------------------------------------
// ONE copy of this code serves both lanes (LANE is a warp-uniform runtime value): the kernel's hot
// instruction footprint has to stay inside the 32 KB L1.5 instruction cache of the SM -- with one copy
// per lane (and the other per-lane duplicates) it was 39 KB in a mixed batch and the tile softmax spent
// 40-50 % of its issue slots waiting for instruction fetch (ncu: stall_no_inst; 4 % in a chunk-only batch).
// fp8 pools (KV8): swap-kind items stream the e4m3 pages themselves (tmap8: one 2 KiB box per page, 16 KiB per
// 128-key tile; lane S's ring is six such slots, lane T's slots keep their 32 KiB stride); tile-kind items read
// the request's dequantised pages from the library's bf16 scratch pool (tmap), where they are contiguous from
// scratch_base[req] -- no block table.
// APPEND (decode-only batches): the producer that is about to load the K (V) tile holding positions of the step's new
// tokens first copies their k_new (v_new) rows into the page slots -- and clears the slots of the request's last page
// past its last key, as kv_append_kernel does -- then orders those generic-proxy stores before its TMA reads.  Tiles
// are page-aligned and the splits of a request partition its keys, so every new row is written by exactly one warp
// of one CTA, and only that warp reads the page in this launch.
template <int D, bool SPLIT, bool KV8, bool APPEND>
__device__ __forceinline__ void producer(const Params& p, const CUtensorMap* tmap, const CUtensorMap* tmap8, uint8_t* smem, Misc* misc, int lane, int warp) {
    using L = Layout<D, SPLIT>;
    static_assert(kStagesT == kStagesS, "the shared producer code assumes one ring depth");
    const int kStages = (KV8 && warp >= kProdT) ? kStagesS8 : L::kStages;
    const uint32_t slot_bytes = (KV8 && warp >= kProdT) ? kSlot8Bytes : L::kSlotBytes;
    const int LANE = SPLIT ? 0 : (warp < kProdT ? 0 : 1);
    const int pw = LANE == 0 ? warp : warp - kProdT;
    const int kProd = SPLIT ? kProdSplit : (LANE == 0 ? kProdT : kProdS);
    LaneState* ls = &misc->lane[LANE];
    constexpr uint32_t kOff0 = L::kOffKv[0], kOff1 = L::kOffKv[1];
    uint8_t* kv_base = smem + (LANE == 0 ? kOff0 : kOff1);
    uint32_t ld_base = 0, item_cnt = 0;          // ld_base: tile loads of all previous items
    bool tiles_left = LANE == 0;
    for (;;) {
        const uint32_t islot = item_cnt % kItemRing;
        int w;
        if (pw == 0) {                           // producer 0 fetches the next item and publishes it
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
            w = 0;                               // one int32 of the 32-byte WorkItem per lane 0..7, its aux word in lane 8
            if (idx >= 0 && lane < 8) w = reinterpret_cast<const int32_t*>(p.meta.work + idx)[lane];
            if (idx >= 0 && lane == 8) w = p.meta.work_aux[idx];
            if (idx < 0 && lane == 7) w = -1;    // kind = -1: sentinel
            ptx::mbar_wait(&ls->item_empty[islot], ((item_cnt / kItemRing) & 1) ^ 1);
            if (lane < 8) reinterpret_cast<int32_t*>(&ls->items[islot])[lane] = w;
            if (lane == 8) ls->aux[islot] = w;
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(&ls->item_full[islot]);
        } else {
            ptx::mbar_wait(&ls->item_full[islot], (item_cnt / kItemRing) & 1);
            w = lane < 8 ? reinterpret_cast<const int32_t*>(&ls->items[islot])[lane] : 0;
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(&ls->item_empty[islot]);
        }
        ++item_cnt;
        if (__shfl_sync(0xffffffffu, w, 7) < 0) break;
        const int req = __shfl_sync(0xffffffffu, w, 0), kv_head = __shfl_sync(0xffffffffu, w, 1);
        const int kv_begin = __shfl_sync(0xffffffffu, w, 4), kv_end = __shfl_sync(0xffffffffu, w, 5);
        const int n_tiles = (kv_end - kv_begin + kKeyTile - 1) / kKeyTile;
        const int32_t* bt = p.meta.block_table + p.meta.bt_off[req] + (kv_begin >> 4);
        const int n_pages_item = (kv_end - kv_begin + 15) >> 4;
        int np0 = 0, np1 = 0;                            // APPEND: positions [np0, np1) of the request's new tokens
        if constexpr (APPEND) {
            np0 = p.meta.ctx_off[req];
            np1 = np0 + p.meta.q_len[req];
            if (np1 > kv_begin && np0 < kv_end) {        // the item's key range holds new rows (its last tiles)
                // H2 for the tiles THIS warp will load, now: the stores are on their way while the item's earlier tiles stream
                const int tok_base = p.meta.cu_q[req];
                const int32_t* bt_req = p.meta.block_table + p.meta.bt_off[req];
                constexpr int kChunks = D / 8;           // 16-byte chunks per row
                const int tA = (max(np0, kv_begin) - kv_begin) / kKeyTile, tB = (min(np1, kv_end) - 1 - kv_begin) / kKeyTile;
                for (int tt = tA; tt <= tB; ++tt)
                    for (int is_v = 0; is_v < 2; ++is_v) {
                        const int i = is_v ? (tt == n_tiles - 1 ? 2 * n_tiles - 1 : 2 * tt + 2) : (tt == 0 ? 0 : 2 * tt - 1);
                        if ((int)((ld_base + i) % kProd) != pw) continue;      // another producer of the lane loads that tile
                        const int t_lo = kv_begin + tt * kKeyTile, t_hi = min(kv_end, t_lo + kKeyTile);
                        const int a = max(np0, t_lo), b = min(np1, t_hi);
                        const uint4* src = is_v ? p.v_new : p.k_new;
                        if (src)
                            for (int u = lane; u < (b - a) * kChunks; u += 32) {
                                const int pos = a + u / kChunks, c = u % kChunks;
                                const int64_t page = bt_req[pos >> 4];
                                __nv_bfloat16* dst = p.cache + (((page * 2 + is_v) * p.sh.Hkv + kv_head) * 16 + (pos & 15)) * (int64_t)D + c * 8;
                                *reinterpret_cast<uint4*>(dst) = src[((int64_t)(tok_base + pos - np0) * p.sh.Hkv + kv_head) * kChunks + c];
                            }
                        if (np1 - 1 >= t_lo && np1 - 1 < t_hi) {      // the request's last key is in this tile: the tail of its page
                            const int first_free = ((np1 - 1) & 15) + 1;
                            const int64_t page = bt_req[(np1 - 1) >> 4];
                            uint4* dst = reinterpret_cast<uint4*>(p.cache + (((page * 2 + is_v) * p.sh.Hkv + kv_head) * 16 + first_free) * (int64_t)D);
                            for (int u = lane; u < (16 - first_free) * kChunks; u += 32) dst[u] = make_uint4(0, 0, 0, 0);
                        }
                    }
            }
        }
        const bool fp8_item = KV8 && __shfl_sync(0xffffffffu, w, 7) == kKindSwap;
        const bool scratch = KV8 && !fp8_item;
        const int sbase = scratch ? p.meta.scratch_base[req] + (kv_begin >> 4) : 0;
        auto page_id = [&](int i) { return scratch ? sbase + i : bt[i]; };
        // page-id windows of 32 pages (4 tiles), one id per lane: cur = window cur_w, nxt = the next
        int cur_w = 0;
        int cur = lane < n_pages_item ? page_id(lane) : 0;
        int nxt = 32 + lane < n_pages_item ? page_id(32 + lane) : 0;
        // load number ld = ld_base + i (global over the whole kernel) belongs to producer ld % kProd, so a
        // producer's previous load is always ld - kProd: with kProd <= kStages the slot it waits for is at
        // most one phase behind and the parity wait cannot alias
        for (int i = (pw + kProd - (int)(ld_base % kProd)) % kProd; i < 2 * n_tiles; i += kProd) {
            int is_v, tile;
            if (i == 0) { is_v = 0; tile = 0; }
            else if (i == 2 * n_tiles - 1) { is_v = 1; tile = n_tiles - 1; }
            else if (i & 1) { is_v = 0; tile = (i + 1) >> 1; }
            else { is_v = 1; tile = (i >> 1) - 1; }
            while ((tile >> 2) > cur_w) {
                cur = nxt;
                ++cur_w;
                const int pi = (cur_w + 1) * 32 + lane;
                nxt = pi < n_pages_item ? page_id(pi) : 0;
            }
            const int n_pages = min(8, n_pages_item - tile * 8);          // 1..8
            const uint32_t ld = ld_base + i;
            const uint32_t slot = ld % kStages;
            ptx::mbar_wait(&ls->kv_empty[slot], ((ld / kStages) & 1) ^ 1);
            if constexpr (APPEND) {
                // this tile holds new rows (written by this warp when the item began): order those generic-proxy stores
                // before the TMA reads of the same bytes -- cheap by now, the stores landed long ago
                const int t_lo = kv_begin + tile * kKeyTile;
                if (np1 > t_lo && np0 < min(kv_end, t_lo + kKeyTile)) {      // warp-uniform
                    __threadfence();
                    asm volatile("fence.proxy.async;" ::: "memory");
                    __syncwarp();
                }
            }
            const bool leader = ptx::elect_one();
            if (leader) ptx::mbar_arrive_expect_tx(&ls->kv_full[slot], (uint32_t)n_pages * (fp8_item ? kPage8Bytes : 16u * D * 2u));
            __syncwarp();
            uint8_t* dst = kv_base + slot * slot_bytes;
            // lanes 0 .. n_pages-1 issue one box (page slab) each, in ONE warp instruction: a leader issuing the eight boxes
            // of a tile one after the other held the slot ~1800 cycles before its last byte was even requested
            {
                const int j = lane & 7;
                const int pg = __shfl_sync(0xffffffffu, cur, (tile & 3) * 8 + j);
                if (lane < n_pages) {
                    const int slab = (pg * 2 + is_v) * p.sh.Hkv + kv_head;
                    if (KV8 && fp8_item) ptx::tma_load_3d(dst + j * kPage8Bytes, tmap8, &ls->kv_full[slot], 0, 0, slab);
                    else ptx::tma_load_5d(dst + j * L::kPageBytes, tmap, &ls->kv_full[slot], 0, 0, 0, 0, slab);
                }
            }
            __syncwarp();
        }
        ld_base += 2 * n_tiles;
    }
}

// ------------------------------------------------------------------------------------------
// MMA issuer warps (tcgen05.mma is issued by one elected thread; the warp stays convergent so
// descriptors live in uniform registers).
//
// The tensor pipe queues only a few instructions, and the serial work of an issuing thread between
// two 8-instruction blocks (two or three mbarrier waits at ~90 cycles each, fences, descriptor
// setup) left the pipe idle for about as long as a block runs.  Lane T therefore has TWO issuers
// for chunk tiles: ROLE 1 issues the score blocks QK(t), ROLE 2 the PV(t) blocks; each does its
// waiting while the other's block executes.  The only ordering the pipe needs between them is
// "PV(t-2) before QK(t)" (QK(t) overwrites the S/P buffer PV(t-2) reads): ROLE 2 arrives on
// pv_issued after issuing PV(t), ROLE 1 waits for it before QK(t+2).  Swap-kind items (lane S, and
// lane T after its tile list is exhausted) are HBM-bound and keep a single issuer (ROLE 0 / ROLE 1).
// ------------------------------------------------------------------------------------------
// Lane T, tile kind.  The item's key range is scored in 64-key half-tiles j = 0 .. nh-1 (tile j >> 1,
// half j & 1); half-tile j uses S buffer (gh0 + j) & 3.  ROLE 1 issues QK(j) (N = 64), ROLE 2 issues
// PV(j) (4 K-steps of 16 keys).  A K/V ring slot still holds a whole 128-key tile: it is waited for at
// its first half and released (tcgen05.commit -> kv_empty) after its last.
template <int D, int ROLE>
__device__ __forceinline__ void mma_tile_item(const WorkItem& it, uint32_t smem_base, LaneState* ls, uint32_t tmem,
                                              uint32_t& ld_base, uint32_t& gh, uint32_t (&ic)[2]) {
    using L = Layout<D>;
    constexpr int kStages = kStagesT;
    const int n_keys = __shfl_sync(0xffffffffu, it.kv_end - it.kv_begin, 0);
    const int n_tiles = (n_keys + kKeyTile - 1) / kKeyTile, nh = (n_keys + 63) / 64;
    const uint32_t kv_base = smem_base + L::kOffKv[0];
    const uint32_t idesc_qk = ptx::umma_idesc_bf16(128, 64, false, false);
    const uint32_t idesc_pv = ptx::umma_idesc_bf16(128, D, false, true);
    const uint32_t gh0 = gh;
    if (ROLE == 1) {
        ptx::mbar_wait(&ls->q_full[0], ic[0] & 1);
        ptx::tc_fence_after();
    }
    ++ic[0];
    for (int j = 0; j < nh; ++j) {
        const int t = j >> 1, h = j & 1;
        const uint32_t g = gh0 + j, buf = g & 3;
        const bool last_of_slot = h == 1 || j == nh - 1;
        if (ROLE == 1) {
            // load order of the producers: K0, K1, V0, K2, V1, ..., K(n-1), V(n-2), V(n-1)
            const uint32_t ld = ld_base + (t == 0 ? 0 : 2 * t - 1);
            const uint32_t slot = ld % kStages;
            if (j >= 4) ptx::mbar_wait(&ls->pv_issued[buf], ((g - 4) >> 2) & 1);      // PV(j-4) (same S buffer) is in the pipe
            if (h == 0) ptx::mbar_wait(&ls->kv_full[slot], (ld / kStages) & 1);
            ptx::tc_fence_after();
            const uint32_t k_half = kv_base + slot * L::kSlotBytes + h * 8 * L::kGroupBytes;   // rows 64 h .. 64 h + 63
            const uint32_t d_tmem = tmem + buf * 64;
            if (ptx::elect_one()) {
                const uint64_t k_desc0 = ptx::umma_desc_sw128(k_half, 16, L::kGroupBytes);
#pragma unroll
                for (int ks = 0; ks < D / 16; ++ks) {
                    const uint32_t koff = (ks >> 2) * 1024 + (ks & 3) * 32;            // K slot: halves of D 1 KB apart
                    umma_ts(d_tmem, tmem + kColQ + ks * 8, ptx::umma_desc_advance(k_desc0, koff), idesc_qk, ks > 0);
                }
                if (last_of_slot) ptx::umma_commit(&ls->kv_empty[slot]);
                ptx::umma_commit(&ls->ts_full[buf]);
            }
            __syncwarp();
        } else {
            const uint32_t ld = ld_base + (t == n_tiles - 1 ? 2 * n_tiles - 1 : 2 * t + 2);
            const uint32_t slot = ld % kStages;
            ptx::mbar_wait(&ls->tp_full[buf], (g >> 2) & 1);
            if (h == 0) ptx::mbar_wait(&ls->kv_full[slot], (ld / kStages) & 1);
            ptx::tc_fence_after();
            const uint32_t v_half = kv_base + slot * L::kSlotBytes + h * 4 * L::kPageBytes;     // keys 64 h .. 64 h + 63
            const uint32_t d_tmem = tmem + col_o(0);
            if (ptx::elect_one()) {
                const uint64_t v_desc0 = ptx::umma_desc_sw128(v_half, 1024, L::kGroupBytes);
#pragma unroll
                for (int ks = 0; ks < 4; ++ks) {
                    // V (MN-major): 16 key rows = 2 row groups (SBO apart); the next 64 d are 1 KB further (LBO)
                    umma_ts(d_tmem, tmem + buf * 64 + ks * 8, ptx::umma_desc_advance(v_desc0, ks * L::kPageBytes),
                            idesc_pv, j > 0 || ks > 0);
                }
                if (last_of_slot) ptx::umma_commit(&ls->kv_empty[slot]);
                ptx::umma_commit(&ls->tpv_done[buf]);
                ptx::mbar_arrive(&ls->pv_issued[buf]);
            }
            __syncwarp();
        }
    }
    gh += nh;
    ld_base += 2 * n_tiles;
}

// SPLIT mode, tile kind (one issuer warp): per 128-key tile t one score block QK(t) -- TS form, Q in TMEM, N = 128
// keys, into S buffer (tile counter & 1) -- and one PV block over the whole tile once ALL softmax warpgroups have
// delivered their part of P(t) (tp_full counts their warps).  QK(t+1) is issued ahead of PV(t), so the next
// scores wait for the warpgroups while the pipe runs PV(t); it overwrites the buffer PV(t-1) read: same thread,
// program order, in-order pipe -- no barrier.  K-steps (pages) past the item's last key are not multiplied.
template <int D>
__device__ __forceinline__ void mma_split_item(const WorkItem& it, uint32_t smem_base, LaneState* ls, uint32_t tmem,
                                               uint32_t& ld_base, uint32_t& gt, uint32_t& ic) {
    using L = Layout<D, true>;
    constexpr int kStages = L::kStages;
    const int n_keys = __shfl_sync(0xffffffffu, it.kv_end - it.kv_begin, 0);
    const int n_tiles = (n_keys + kKeyTile - 1) / kKeyTile;
    const uint32_t kv_base = smem_base + L::kOffKv[0];
    const uint32_t idesc_qk = ptx::umma_idesc_bf16(128, 128, false, false);
    const uint32_t idesc_pv = ptx::umma_idesc_bf16(128, D, false, true);
    const uint32_t g0 = gt;
    ptx::mbar_wait(&ls->q_full[0], ic & 1);
    ++ic;
    ptx::tc_fence_after();
    auto issue_qk = [&](int t) {
        // load order of the producers: K0, K1, V0, K2, V1, ..., K(n-1), V(n-2), V(n-1)
        const uint32_t ld = ld_base + (t == 0 ? 0 : 2 * t - 1);
        const uint32_t slot = ld % kStages, buf = (g0 + t) & 1;
        ptx::mbar_wait(&ls->kv_full[slot], (ld / kStages) & 1);
        ptx::tc_fence_after();
        if (ptx::elect_one()) {
            const uint64_t k_desc0 = ptx::umma_desc_sw128(kv_base + slot * L::kSlotBytes, 16, L::kGroupBytes);
#pragma unroll
            for (int ks = 0; ks < D / 16; ++ks) {
                const uint32_t koff = (ks >> 2) * 1024 + (ks & 3) * 32;            // K slot: halves of D 1 KB apart
                umma_ts(tmem + buf * 128, tmem + kColQ + ks * 8, ptx::umma_desc_advance(k_desc0, koff), idesc_qk, ks > 0);
            }
            ptx::umma_commit(&ls->kv_empty[slot]);
            ptx::umma_commit(&ls->ts_full[buf]);
        }
        __syncwarp();
    };
    issue_qk(0);
    for (int t = 0; t < n_tiles; ++t) {
        if (t + 1 < n_tiles) issue_qk(t + 1);
        const uint32_t ld = ld_base + (t == n_tiles - 1 ? 2 * n_tiles - 1 : 2 * t + 2);
        const uint32_t slot = ld % kStages, g = g0 + t, buf = g & 1;
        ptx::mbar_wait(&ls->tp_full[buf], (g >> 1) & 1);
        ptx::mbar_wait(&ls->kv_full[slot], (ld / kStages) & 1);
        ptx::tc_fence_after();
        if (ptx::elect_one()) {
            const uint64_t v_desc0 = ptx::umma_desc_sw128(kv_base + slot * L::kSlotBytes, 1024, L::kGroupBytes);
#pragma unroll
            for (int ks = 0; ks < kKeyTile / 16; ++ks) {
                // V (MN-major): 16 key rows = 2 row groups (SBO apart); the next 64 d are 1 KB further (LBO).
                // P of keys kSplitCols w .. kSplitCols (w + 1) - 1 sits in the first kSplitCols / 2 columns of
                // part w of the S buffer.
                if (t * kKeyTile + ks * 16 < n_keys)
                    umma_ts(tmem + col_o(0), tmem + buf * 128 + (ks * 16 / kSplitCols) * kSplitCols + (ks * 16 % kSplitCols) / 2,
                            ptx::umma_desc_advance(v_desc0, ks * L::kPageBytes), idesc_pv, t > 0 || ks > 0);
            }
            ptx::umma_commit(&ls->kv_empty[slot]);
            ptx::umma_commit(&ls->tpv_done[buf]);
        }
        __syncwarp();
    }
    gt += n_tiles;
    ld_base += 2 * n_tiles;
}

// fp8 pools, swap kind (<= 8 rows, D = 128): the e4m3 pages feed kind::f8f6f4 MMAs directly (K = 32 per instruction).
// Both operands must be 8-bit, so Q^T and P^T come as e4m3 too, each value split x = hi + lo / 16 into two codes
// stacked along N (rows 0..7 = hi, 8..15 = lo of the 16-row B operand: N = 16 as in the bf16 kind) -- ~2^-8 relative,
// what bf16 gives; the softmax adds the two column groups after tcgen05.ld.
//   S^T[128 keys x 16] = K[128 x D] Q8^T      (A = K tile, K-major, 4 K-steps of 32 d)
//   O^T[128 d x 16]   += V^T[D x 128] P8^T    (A = V tile MN-major, 4 K-steps of 32 keys; B = P8^T, K-major along keys)
// Same barriers and tile order as the bf16 swap kind.  Lane S's ring: six 16 KiB slots; lane T's: 32 KiB stride.
template <int D, int LANE>
__device__ __forceinline__ void mma_swap8_item(const WorkItem& it, uint32_t smem_base, LaneState* ls, uint32_t tmem,
                                               uint32_t& ld_base, uint32_t& gt, uint32_t& gp, uint32_t& ic) {
    using L = Layout<D, false>;
    constexpr int kStages = LANE == 0 ? kStagesT : kStagesS8;
    constexpr uint32_t kStride = LANE == 0 ? L::kSlotBytes : kSlot8Bytes;
    const int n_tiles = (__shfl_sync(0xffffffffu, it.kv_end - it.kv_begin, 0) + kKeyTile - 1) / kKeyTile;
    const uint32_t small = smem_base + L::kOffSmall[LANE], kv_base = smem_base + L::kOffKv[LANE];
    const uint32_t idesc_qk = ptx::umma_idesc_e4m3(128, 16, false, false);
    const uint32_t idesc_pv = ptx::umma_idesc_e4m3(128, 16, true, false);
    const uint32_t g0 = gt;
    ptx::mbar_wait(&ls->q_full[1], ic & 1);
    ptx::tc_fence_after();
    ++ic;
    auto issue_qk = [&](int t) {
        const uint32_t ld = ld_base + (t == 0 ? 0 : 2 * t - 1);
        const uint32_t slot = ld % kStages, buf = (g0 + t) & 1;
        ptx::mbar_wait(&ls->kv_full[slot], (ld / kStages) & 1);
        ptx::tc_fence_after();
        if (ptx::elect_one()) {
            const uint64_t k_desc0 = ptx::umma_desc_sw128(kv_base + slot * kStride, 16, 1024);     // rows of 128 B, 8-row groups 1 KB apart
            const uint64_t q_desc0 = ptx::umma_desc_sw128(small, 16, 1024);
#pragma unroll
            for (int ks = 0; ks < 4; ++ks)
                ptx::umma_ss_f8(tmem + col_s(LANE, buf), ptx::umma_desc_advance(k_desc0, ks * 32), ptx::umma_desc_advance(q_desc0, ks * 32),
                                idesc_qk, ks > 0);
            ptx::umma_commit(&ls->kv_empty[slot]);
            ptx::umma_commit(&ls->s_full[buf]);
        }
        __syncwarp();
    };
    auto issue_pv = [&](int t) {
        const uint32_t ld = ld_base + (t == n_tiles - 1 ? 2 * n_tiles - 1 : 2 * t + 2);
        const uint32_t slot = ld % kStages, buf = (g0 + t) & 1;
        ptx::mbar_wait(&ls->p_full[1][gp & 1], (gp >> 1) & 1);
        ++gp;
        ptx::mbar_wait(&ls->kv_full[slot], (ld / kStages) & 1);
        ptx::tc_fence_after();
        if (ptx::elect_one()) {
            // V (MN-major, 8-bit): a key row is 128 B = all 128 d; 32 keys = 4 row groups, SBO = 1 KB apart
            const uint64_t v_desc0 = ptx::umma_desc_sw128(kv_base + slot * kStride, 1024, 1024);
            const uint64_t p_desc0 = ptx::umma_desc_sw128(small + 4096 + buf * 4096, 16, 1024);     // P8^T is double buffered
#pragma unroll
            for (int ks = 0; ks < 4; ++ks)
                ptx::umma_ss_f8(tmem + col_o(LANE), ptx::umma_desc_advance(v_desc0, ks * 4096), ptx::umma_desc_advance(p_desc0, ks * 32),
                                idesc_pv, t > 0 || ks > 0);
            ptx::umma_commit(&ls->kv_empty[slot]);
            ptx::umma_commit(&ls->pv_done[buf]);
        }
        __syncwarp();
    };
    issue_qk(0);
    for (int t = 0; t < n_tiles; ++t) {
        if (t + 1 < n_tiles) issue_qk(t + 1);
        issue_pv(t);
    }
    gt += n_tiles;
    ld_base += 2 * n_tiles;
}

template <int D, int LANE, int ROLE, bool SPLIT, bool KV8>
__device__ __forceinline__ void mma_item(const WorkItem& it, uint32_t smem_base, LaneState* ls, uint32_t tmem,
                                         uint32_t& ld_base, uint32_t& gt, uint32_t& gp, uint32_t (&ic)[2], uint32_t& gpt) {
    using L = Layout<D, SPLIT>;
    constexpr int kStages = SPLIT ? L::kStages : (LANE == 0 ? kStagesT : kStagesS);
    const int n_tiles = (__shfl_sync(0xffffffffu, it.kv_end - it.kv_begin, 0) + kKeyTile - 1) / kKeyTile;
    const bool swap = LANE == 1 || __shfl_sync(0xffffffffu, it.kind, 0) == kKindSwap;
    const bool all = ROLE == 0 || swap;        // this warp issues both kinds of block
    if (!swap) {
        if constexpr (SPLIT) mma_split_item<D>(it, smem_base, ls, tmem, ld_base, gpt, ic[0]);
        else if constexpr (LANE == 0 && ROLE != 0) mma_tile_item<D, ROLE>(it, smem_base, ls, tmem, ld_base, gpt, ic);
        return;
    }
    if (ROLE == 2) {                           // swap item on lane T: ROLE 1 issues it; stay in step
        gt += n_tiles;
        ld_base += 2 * n_tiles;
        return;
    }
    if constexpr (KV8 && D == 128) {
        mma_swap8_item<D, LANE>(it, smem_base, ls, tmem, ld_base, gt, gp, ic[1]);
        return;
    }
    const bool do_qk = all || ROLE == 1, do_pv = all || ROLE == 2;
    const uint32_t small = smem_base + L::kOffSmall[LANE], kv_base = smem_base + L::kOffKv[LANE];
    // tile kind: S = Q K^T (A = Q in TMEM, M 128 rows, N 128 keys); O += P V (A = P in TMEM, V MN-major B)
    // swap kind: S^T = K Q^T (M 128 keys, N 16);   O^T += V^T P^T (M 128 = D, N 16, V^T is MN-major A)
    const uint32_t idesc_qk = swap ? ptx::umma_idesc_bf16(128, 16, false, false) : ptx::umma_idesc_bf16(128, 128, false, false);
    const uint32_t idesc_pv = swap ? ptx::umma_idesc_bf16(128, 16, true, false) : ptx::umma_idesc_bf16(128, D, false, true);
    const uint32_t small_half = 2048;          // 16 rows x 128 B (Q^T / P^T halves in the swap kind)
    const int set = swap ? 1 : 0;              // barrier set and phase counters of this item kind
    const uint32_t g0 = gt, t0 = gpt;          // global tile counter / tile-kind tile counter at item start

    if (do_qk) {
        ptx::mbar_wait(&ls->q_full[set], ic[set] & 1);
        ptx::tc_fence_after();
    }
    ++ic[set];

    // load order of the producers = consumption order: K0, K1, V0, K2, V1, ..., K(n-1), V(n-2), V(n-1)
    auto issue_qk = [&](int t) {
        const uint32_t ld = ld_base + (t == 0 ? 0 : 2 * t - 1);
        const uint32_t slot = ld % kStages, buf = (g0 + t) & 1;
        if (!all && t >= 2) ptx::mbar_wait(&ls->pv_issued[(t0 + t) & 1], ((t0 + t - 2) >> 1) & 1);   // PV(t-2) is in the pipe
        ptx::mbar_wait(&ls->kv_full[slot], (ld / kStages) & 1);
        ptx::tc_fence_after();
        const uint32_t k_tile = kv_base + slot * L::kSlotBytes;
        const uint32_t d_tmem = tmem + col_s(LANE, buf);
        if (ptx::elect_one()) {
            const uint64_t k_desc0 = ptx::umma_desc_sw128(k_tile, 16, L::kGroupBytes);
            const uint64_t q_desc0 = ptx::umma_desc_sw128(small, 16, 1024);
#pragma unroll
            for (int ks = 0; ks < D / 16; ++ks) {
                const uint32_t koff = (ks >> 2) * 1024 + (ks & 3) * 32;                // K slot: halves 1 KB apart
                const uint64_t k_desc = ptx::umma_desc_advance(k_desc0, koff);
                if (LANE == 0 && !swap) {
                    umma_ts(d_tmem, tmem + kColQ + ks * 8, k_desc, idesc_qk, ks > 0);
                } else {
                    const uint32_t qoff = (ks >> 2) * small_half + (ks & 3) * 32;
                    ptx::umma_ss(d_tmem, k_desc, ptx::umma_desc_advance(q_desc0, qoff), idesc_qk, ks > 0);
                }
            }
            ptx::umma_commit(&ls->kv_empty[slot]);
            ptx::umma_commit(&ls->s_full[buf]);
        }
        __syncwarp();
    };
    auto issue_pv = [&](int t) {
        const uint32_t ld = ld_base + (t == n_tiles - 1 ? 2 * n_tiles - 1 : 2 * t + 2);
        const uint32_t slot = ld % kStages, buf = (g0 + t) & 1;
        ptx::mbar_wait(&ls->p_full[set][gp & 1], (gp >> 1) & 1);
        ++gp;
        ptx::mbar_wait(&ls->kv_full[slot], (ld / kStages) & 1);
        ptx::tc_fence_after();
        const uint32_t v_tile = kv_base + slot * L::kSlotBytes;
        const uint32_t d_tmem = tmem + col_o(LANE);
        if (ptx::elect_one()) {
            const uint64_t v_desc0 = ptx::umma_desc_sw128(v_tile, 1024, L::kGroupBytes);
            const uint64_t p_desc0 = ptx::umma_desc_sw128(small + 4096 + buf * 4096, 16, 1024);      // P^T is double buffered
#pragma unroll
            for (int ks = 0; ks < kKeyTile / 16; ++ks) {
                // V (MN-major): 16 key rows = 2 row groups (SBO apart); the next 64 d are 1 KB further (LBO)
                const uint64_t v_desc = ptx::umma_desc_advance(v_desc0, ks * L::kPageBytes);
                if (LANE == 0 && !swap) {
                    umma_ts(d_tmem, tmem + col_s(0, buf) + ks * 8, v_desc, idesc_pv, t > 0 || ks > 0);
                } else {
                    const uint32_t poff = (ks >> 2) * small_half + (ks & 3) * 32;
                    ptx::umma_ss(d_tmem, v_desc, ptx::umma_desc_advance(p_desc0, poff), idesc_pv, t > 0 || ks > 0);
                }
            }
            ptx::umma_commit(&ls->kv_empty[slot]);
            ptx::umma_commit(&ls->pv_done[buf]);
            if (!all) ptx::mbar_arrive(&ls->pv_issued[(t0 + t) & 1]);
        }
        __syncwarp();
    };

    // QK(t+1) is issued before PV(t) so the softmax of tile t overlaps the next score MMA.  p_full is
    // indexed by tile parity (per item kind): the softmax of tile t+2 needs QK(t+2), which is issued
    // only after PV(t) was issued, i.e. after p_full of tile t was observed, so no wait can alias onto
    // a later phase; the same argument covers pv_issued.
    if (do_qk) issue_qk(0);
    for (int t = 0; t < n_tiles; ++t) {
        if (do_qk && t + 1 < n_tiles) issue_qk(t + 1);
        if (do_pv) issue_pv(t);
    }
    gt += n_tiles;
    ld_base += 2 * n_tiles;
}

template <int D, int LANE, int ROLE, bool SPLIT, bool KV8>
__device__ __forceinline__ void mma_warp(uint32_t smem_base, Misc* misc, int lane) {
    LaneState* ls = &misc->lane[LANE];
    const uint32_t tmem = misc->tmem_base;
    uint32_t ld_base = 0, gt = 0, item_cnt = 0, gp = 0, gpt = 0, ic[2] = {0, 0};
    for (;;) {
        const uint32_t islot = item_cnt % kItemRing;
        ptx::mbar_wait(&ls->item_full[islot], (item_cnt / kItemRing) & 1);
        const WorkItem it = ls->items[islot];
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(&ls->item_empty[islot]);
        if (it.kind < 0) break;
        mma_item<D, LANE, ROLE, SPLIT, KV8>(it, smem_base, ls, tmem, ld_base, gt, gp, ic, gpt);
        ++item_cnt;
    }
}

// ------------------------------------------------------------------------------------------
// softmax warpgroup of lane T, tile kind: thread <-> row of the 128-row Q tile.  Q row -> TMEM once,
// then per key tile: the whole score row from TMEM in ONE load batch (a tcgen05.ld/wait round trip
// costs ~70 cycles per warp that has one in flight, whatever its size, so it is issued once per
// tile), online softmax (log2 domain, lazy rescale), P row -> TMEM over the first 64 columns of the
// same S buffer (bf16 pairs), O rescale / epilogue from TMEM.
// ------------------------------------------------------------------------------------------
template <int D, bool POLY, bool NARROW>      // NARROW: 200 registers per thread (fp8 pools: one code copy for both softmax warpgroups)
__device__ __forceinline__ void softmax_tile(const WorkItem& it, const Params& p, LaneState* ls, uint32_t tmem,
                                             uint32_t& gh, int row, uint32_t lane_base) {
    const Shape& sh = p.sh;
    const int G = sh.G;
    const int gs = 31 - __clz(G);                        // G is a power of two (cp_create): shifts, not divisions
    const int R = it.q_tokens * G;
    const int n_tiles = (it.kv_end - it.kv_begin + kKeyTile - 1) / kKeyTile;
    const int tok0 = p.meta.cu_q[it.req] + it.q_start;
    const int ctx = p.meta.ctx_off[it.req];
    const bool valid_row = row < R;
    const int tok = tok0 + (row >> gs);
    const int head = it.kv_head * G + (row & (G - 1));
    const float scale = sh.sm_scale * 1.4426950408889634f;
    const uint32_t t_row = tmem + (lane_base << 16);

    // ---- Q row -> TMEM (A operand of QK^T): column j holds elements (2j, 2j+1)
    {
        const uint4* src = reinterpret_cast<const uint4*>(p.q + ((int64_t)tok * sh.Hq + head) * D);
#pragma unroll
        for (int c = 0; c < D / 64; ++c) {
            uint32_t r[32];
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const uint4 v = valid_row ? src[c * 8 + j] : make_uint4(0, 0, 0, 0);
                r[4 * j] = v.x; r[4 * j + 1] = v.y; r[4 * j + 2] = v.z; r[4 * j + 3] = v.w;
            }
            ptx::tmem_st32(t_row + kColQ + c * 32, r);
        }
        ptx::tmem_wait_st();
        ptx::tc_fence_before();
        warp_arrive(&ls->q_full[0]);
    }

    const int limit = valid_row ? min(it.kv_end, ctx + it.q_start + (row >> gs) + 1) : 0;   // causal, diagonal inclusive
    float m_ref = -INFINITY, l = 0.f;
    const int nh = (it.kv_end - it.kv_begin + 63) / 64;          // 64-key half-tiles, S buffer = gh & 3

    for (int j = 0; j < nh; ++j) {
        const int ts = it.kv_begin + j * 64;
        const uint32_t buf = gh & 3;
        const uint32_t t_s = t_row + buf * 64;
        ptx::mbar_wait(&ls->ts_full[buf], (gh >> 2) & 1);
        ptx::tc_fence_after();
        uint32_t sr[64];
        ptx::tmem_ld32(t_s, sr);
        ptx::tmem_ld32(t_s + 32, sr + 32);
        ptx::tmem_wait_ld();
        const int nvalid = max(0, min(64, limit - ts));
        float mx[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};      // independent max chains
        if (nvalid == 64) {
#pragma unroll
            for (int i = 0; i < 64; ++i) mx[i & 3] = fmaxf(mx[i & 3], __uint_as_float(sr[i]));
        } else {
#pragma unroll
            for (int i = 0; i < 64; ++i) mx[i & 3] = fmaxf(mx[i & 3], i < nvalid ? __uint_as_float(sr[i]) : -INFINITY);
        }
        const float m_t = fmaxf(fmaxf(mx[0], mx[1]), fmaxf(mx[2], mx[3])) * scale;      // scale > 0
        float alpha = 1.f;
        bool rescale = false;
        if (m_t > m_ref + kRescaleThreshold) {          // also the first finite max (m_ref = -inf)
            alpha = (m_ref == -INFINITY) ? 0.f : ptx::ex2(m_ref - m_t);
            m_ref = m_t;
            rescale = true;
        }
        const float neg_m = (m_ref == -INFINITY) ? 0.f : -m_ref;
        float sm[4] = {0.f, 0.f, 0.f, 0.f};             // independent sum chains
        uint32_t pk[32];                                // 64 scores -> 32 packed P columns
        if (nvalid == 64) {
            // two columns per instruction (FFMA2 / FADD2), as in softmax_split
            const float2 sc2 = make_float2(scale, scale), nm2 = make_float2(neg_m, neg_m);
            float2 s2[4] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
#pragma unroll
            for (int i = 0; i < 32; ++i) {
                const float2 x = ptx::fma2(make_float2(__uint_as_float(sr[2 * i]), __uint_as_float(sr[2 * i + 1])), sc2, nm2);
                float2 e;
                if (POLY && kPolyEvery > 0 && i % (kPolyEvery > 0 ? kPolyEvery : 1) == (kPolyEvery > 0 ? kPolyEvery : 1) - 1) e = ptx::ex2_poly2(x);
                else e = make_float2(ptx::ex2(x.x), ptx::ex2(x.y));
                s2[i & 3] = ptx::add2(s2[i & 3], e);
                pk[i] = pack_bf16(e.x, e.y);
            }
            const float2 s01 = ptx::add2(ptx::add2(s2[0], s2[1]), ptx::add2(s2[2], s2[3]));
            sm[0] = s01.x + s01.y;
        } else {
#pragma unroll
            for (int i = 0; i < 64; i += 2) {
                const float a = i < nvalid ? ex2_sel<POLY>(fmaf(__uint_as_float(sr[i]), scale, neg_m), i) : 0.f;
                const float b = i + 1 < nvalid ? ex2_sel<POLY>(fmaf(__uint_as_float(sr[i + 1]), scale, neg_m), i + 1) : 0.f;
                sm[(i >> 1) & 3] += a + b;
                pk[i >> 1] = pack_bf16(a, b);
            }
        }
        ptx::tmem_st32(t_s, pk);
        l = l * alpha + ((sm[0] + sm[1]) + (sm[2] + sm[3]));
        if (j > 0 && __any_sync(0xffffffffu, rescale)) {
            ptx::mbar_wait(&ls->tpv_done[(gh - 1) & 3], ((gh - 1) >> 2) & 1);      // PV(j-1) (and all before) done: O readable
            ptx::tc_fence_after();
#pragma unroll 1
            for (int c = 0; c < D / 32; ++c) {
                uint32_t o[32];
                ptx::tmem_ld32(t_row + col_o(0) + c * 32, o);
                ptx::tmem_wait_ld();
#pragma unroll
                for (int i = 0; i < 32; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * alpha);
                ptx::tmem_st32(t_row + col_o(0) + c * 32, o);
            }
        }
        ptx::tmem_wait_st();
        ptx::tc_fence_before();
        warp_arrive(&ls->tp_full[buf]);
        ++gh;
    }

    // ---- epilogue: O row from TMEM (one load batch) -> out (bf16, normalised) or split workspace (fp32, unnormalised)
    ptx::mbar_wait(&ls->tpv_done[(gh - 1) & 3], ((gh - 1) >> 2) & 1);
    ptx::tc_fence_after();
    const float inv = 1.f / l;
    if constexpr (NARROW) {
#pragma unroll 1
        for (int c = 0; c < D / 64; ++c) {               // 64 columns at a time
            uint32_t o[64];
            ptx::tmem_ld32(t_row + col_o(0) + c * 64, o);
            ptx::tmem_ld32(t_row + col_o(0) + c * 64 + 32, o + 32);
            ptx::tmem_wait_ld();
            if (!valid_row) continue;
            if (it.partial_row < 0) {
                uint4* dst = reinterpret_cast<uint4*>(p.out + ((int64_t)tok * sh.Hq + head) * D + c * 64);
#pragma unroll
                for (int j = 0; j < 8; ++j)
                    dst[j] = make_uint4(pack_bf16(__uint_as_float(o[8 * j]) * inv, __uint_as_float(o[8 * j + 1]) * inv),
                                        pack_bf16(__uint_as_float(o[8 * j + 2]) * inv, __uint_as_float(o[8 * j + 3]) * inv),
                                        pack_bf16(__uint_as_float(o[8 * j + 4]) * inv, __uint_as_float(o[8 * j + 5]) * inv),
                                        pack_bf16(__uint_as_float(o[8 * j + 6]) * inv, __uint_as_float(o[8 * j + 7]) * inv));
            } else {
                uint4* dst = reinterpret_cast<uint4*>(p.part_o + ((int64_t)it.partial_row + row) * D + c * 64);
#pragma unroll
                for (int j = 0; j < 16; ++j) dst[j] = make_uint4(o[4 * j], o[4 * j + 1], o[4 * j + 2], o[4 * j + 3]);
            }
        }
        if (valid_row && it.partial_row >= 0) p.part_ml[(int64_t)it.partial_row + row] = make_float2(m_ref, l);
        ptx::tc_fence_before();
        return;
    }
    uint32_t o[D];
#pragma unroll
    for (int c = 0; c < D / 32; ++c) ptx::tmem_ld32(t_row + col_o(0) + c * 32, o + c * 32);
    ptx::tmem_wait_ld();
    if (valid_row) {
        if (it.partial_row < 0) {
            uint4* dst = reinterpret_cast<uint4*>(p.out + ((int64_t)tok * sh.Hq + head) * D);
#pragma unroll
            for (int j = 0; j < D / 8; ++j)
                dst[j] = make_uint4(pack_bf16(__uint_as_float(o[8 * j]) * inv, __uint_as_float(o[8 * j + 1]) * inv),
                                    pack_bf16(__uint_as_float(o[8 * j + 2]) * inv, __uint_as_float(o[8 * j + 3]) * inv),
                                    pack_bf16(__uint_as_float(o[8 * j + 4]) * inv, __uint_as_float(o[8 * j + 5]) * inv),
                                    pack_bf16(__uint_as_float(o[8 * j + 6]) * inv, __uint_as_float(o[8 * j + 7]) * inv));
        } else {
            uint4* dst = reinterpret_cast<uint4*>(p.part_o + ((int64_t)it.partial_row + row) * D);
#pragma unroll
            for (int j = 0; j < D / 4; ++j) dst[j] = make_uint4(o[4 * j], o[4 * j + 1], o[4 * j + 2], o[4 * j + 3]);
            p.part_ml[(int64_t)it.partial_row + row] = make_float2(m_ref, l);
        }
    }
    ptx::tc_fence_before();
}

// ------------------------------------------------------------------------------------------
// SPLIT mode: softmax of warpgroup w (0 .. kSplitWG - 1) for a chunk tile: thread <-> row of the 128-row Q tile,
// columns (keys) [kSplitCols w, kSplitCols (w + 1)) of every 128-key score tile.  Per tile: the part of the score
// row from TMEM, its maximum, the exchange of the part-row maxima through shared memory (one named barrier over
// the kSplitWG warps that hold the same 32 rows), then all threads of a row take the SAME decision about the
// reference maximum (lazy rescale: only when the row maximum grew by more than 2^8), exponentials, partial row sum
// of the own columns, P (bf16 pairs) back over the scores of the own part.  Warpgroup w owns O columns
// [w D / kSplitWG, (w + 1) D / kSplitWG) for the rescale and the epilogue; the partial row sums meet in shared
// memory at the end.  Warpgroup 0 puts the Q tile into TMEM.
// ------------------------------------------------------------------------------------------
template <int D, bool POLY>
__device__ __forceinline__ void softmax_split(const WorkItem& it, const Params& p, LaneState* ls, uint32_t tmem, uint8_t* xchg,
                                              uint32_t& gt, int row, uint32_t lane_base, int w) {
    constexpr int NW = kSplitWG, CW = kSplitCols;        // warpgroups; keys of a tile per thread
    constexpr int OC = D / NW;                           // O columns per warpgroup
    constexpr int CH = OC < 32 ? OC : 32;                // ... handled CH at a time
    const Shape& sh = p.sh;
    const int G = sh.G;
    const int gs = 31 - __clz(G);                        // G is a power of two (cp_create): shifts, not divisions
    const int R = it.q_tokens * G;
    const int n_tiles = (it.kv_end - it.kv_begin + kKeyTile - 1) / kKeyTile;
    const int tok0 = p.meta.cu_q[it.req] + it.q_start;
    const int ctx = p.meta.ctx_off[it.req];
    const bool valid_row = row < R;
    const int tok = tok0 + (row >> gs);
    const int head = it.kv_head * G + (row & (G - 1));
    const float scale = sh.sm_scale * 1.4426950408889634f;
    const uint32_t t_row = tmem + (lane_base << 16);
    const uint32_t c_o = col_o(0) + w * OC;              // this warpgroup's part of the O columns
    float* xmax = reinterpret_cast<float*>(xchg);        // [tile parity][warpgroup][row]: part-row maxima (raw scores)
    float* xl = xmax + 2 * NW * 128;                     // [warpgroup][row]: partial row sums
    const int bar_id = 3 + (int)(lane_base >> 5);        // the NW warps that hold the same 32 rows
    constexpr int bar_n = 32 * NW;

    if (w == 0) {
        // ---- Q row -> TMEM (A operand of QK^T): column j holds elements (2j, 2j+1)
        const uint4* src = reinterpret_cast<const uint4*>(p.q + ((int64_t)tok * sh.Hq + head) * D);
#pragma unroll
        for (int c = 0; c < D / 64; ++c) {
            uint32_t r[32];
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const uint4 v = valid_row ? src[c * 8 + j] : make_uint4(0, 0, 0, 0);
                r[4 * j] = v.x; r[4 * j + 1] = v.y; r[4 * j + 2] = v.z; r[4 * j + 3] = v.w;
            }
            ptx::tmem_st32(t_row + kColQ + c * 32, r);
        }
        ptx::tmem_wait_st();
        ptx::tc_fence_before();
        warp_arrive(&ls->q_full[0]);
    }

    const int limit = valid_row ? min(it.kv_end, ctx + it.q_start + (row >> gs) + 1) : 0;   // causal, diagonal inclusive
    float m_ref = -INFINITY, l = 0.f;

    for (int t = 0; t < n_tiles; ++t) {
        const int ts = it.kv_begin + t * kKeyTile + w * CW;
        const uint32_t buf = gt & 1;
        const uint32_t t_s = t_row + buf * 128 + w * CW;
        ptx::mbar_wait(&ls->ts_full[buf], (gt >> 1) & 1);
        ptx::tc_fence_after();
        uint32_t sr[CW];
#pragma unroll
        for (int c = 0; c < CW / 32; ++c) ptx::tmem_ld32(t_s + c * 32, sr + c * 32);
        ptx::tmem_wait_ld();
        const int nvalid = max(0, min(CW, limit - ts));
        float mx[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};      // independent max chains
        if (nvalid == CW) {
#pragma unroll
            for (int i = 0; i < CW; ++i) mx[i & 3] = fmaxf(mx[i & 3], __uint_as_float(sr[i]));
        } else {
#pragma unroll
            for (int i = 0; i < CW; ++i) mx[i & 3] = fmaxf(mx[i & 3], i < nvalid ? __uint_as_float(sr[i]) : -INFINITY);
        }
        const float m_loc = fmaxf(fmaxf(mx[0], mx[1]), fmaxf(mx[2], mx[3]));
        float* xm = xmax + (gt & 1) * NW * 128 + row;
        xm[w * 128] = m_loc;
        ptx::named_bar_sync(bar_id, bar_n);               // the warps of the other warpgroups with the same rows: their maxima are there
        float m_all = m_loc;
#pragma unroll
        for (int k = 1; k < NW; ++k) m_all = fmaxf(m_all, xm[((w + k) & (NW - 1)) * 128]);
        const float m_t = m_all * scale;                  // scale > 0
        float alpha = 1.f;
        bool rescale = false;
        if (m_t > m_ref + kRescaleThreshold) {          // also the first finite max (m_ref = -inf)
            alpha = (m_ref == -INFINITY) ? 0.f : ptx::ex2(m_ref - m_t);
            m_ref = m_t;
            rescale = true;
        }
        const float neg_m = (m_ref == -INFINITY) ? 0.f : -m_ref;
        float sm[4] = {0.f, 0.f, 0.f, 0.f};             // independent sum chains
        uint32_t pk[CW / 2];                            // CW scores -> CW / 2 packed P columns
        if (nvalid == CW) {
            // two columns per instruction (FFMA2 / FADD2); every kPolyEvery-th PAIR takes the FMA-pipe exponential
            const float2 sc2 = make_float2(scale, scale), nm2 = make_float2(neg_m, neg_m);
            float2 s2[4] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
#pragma unroll
            for (int j = 0; j < CW / 2; ++j) {
                const float2 x = ptx::fma2(make_float2(__uint_as_float(sr[2 * j]), __uint_as_float(sr[2 * j + 1])), sc2, nm2);
                float2 e;
                if (POLY && kPolyEvery > 0 && j % (kPolyEvery > 0 ? kPolyEvery : 1) == (kPolyEvery > 0 ? kPolyEvery : 1) - 1) e = ptx::ex2_poly2(x);
                else e = make_float2(ptx::ex2(x.x), ptx::ex2(x.y));
                s2[j & 3] = ptx::add2(s2[j & 3], e);
                pk[j] = pack_bf16(e.x, e.y);
            }
            const float2 s01 = ptx::add2(ptx::add2(s2[0], s2[1]), ptx::add2(s2[2], s2[3]));
            sm[0] = s01.x + s01.y;
        } else {
#pragma unroll
            for (int i = 0; i < CW; i += 2) {
                const float a = i < nvalid ? ex2_sel<POLY>(fmaf(__uint_as_float(sr[i]), scale, neg_m), i) : 0.f;
                const float b = i + 1 < nvalid ? ex2_sel<POLY>(fmaf(__uint_as_float(sr[i + 1]), scale, neg_m), i + 1) : 0.f;
                sm[(i >> 1) & 3] += a + b;
                pk[i >> 1] = pack_bf16(a, b);
            }
        }
        ptx::tmem_st<CW / 2>(t_s, pk);
        l = l * alpha + ((sm[0] + sm[1]) + (sm[2] + sm[3]));
        // same rows, same m_t, same m_ref in warp k of every warpgroup: the same decision on all sides
        if (t > 0 && __any_sync(0xffffffffu, rescale)) {
            ptx::mbar_wait(&ls->tpv_done[(gt - 1) & 1], ((gt - 1) >> 1) & 1);      // PV(t-1) (and all before) done: O readable
            ptx::tc_fence_after();
#pragma unroll 1
            for (int c = 0; c < OC / CH; ++c) {
                uint32_t o[CH];
                ptx::tmem_ld<CH>(t_row + c_o + c * CH, o);
                ptx::tmem_wait_ld();
#pragma unroll
                for (int i = 0; i < CH; ++i) o[i] = __float_as_uint(__uint_as_float(o[i]) * alpha);
                ptx::tmem_st<CH>(t_row + c_o + c * CH, o);
            }
        }
        ptx::tmem_wait_st();
        ptx::tc_fence_before();
        warp_arrive(&ls->tp_full[buf]);
        ++gt;
    }

    // ---- epilogue: this warpgroup's part of the O row -> out (bf16, normalised) or split workspace (fp32, unnormalised)
    ptx::mbar_wait(&ls->tpv_done[(gt - 1) & 1], ((gt - 1) >> 1) & 1);
    ptx::tc_fence_after();
    xl[w * 128 + row] = l;
    ptx::named_bar_sync(bar_id, bar_n);
    // every warpgroup adds the partial sums in the same order: the same l on all sides
    l = 0.f;
#pragma unroll
    for (int k = 0; k < NW; ++k) l += xl[k * 128 + row];
    const float inv = 1.f / l;
#pragma unroll 1
    for (int c = 0; c < OC / CH; ++c) {
        uint32_t o[CH];
        ptx::tmem_ld<CH>(t_row + c_o + c * CH, o);
        ptx::tmem_wait_ld();
        if (!valid_row) continue;
        const int d0 = w * OC + c * CH;
        if (it.partial_row < 0) {
            uint4* dst = reinterpret_cast<uint4*>(p.out + ((int64_t)tok * sh.Hq + head) * D + d0);
#pragma unroll
            for (int j = 0; j < CH / 8; ++j)
                dst[j] = make_uint4(pack_bf16(__uint_as_float(o[8 * j]) * inv, __uint_as_float(o[8 * j + 1]) * inv),
                                    pack_bf16(__uint_as_float(o[8 * j + 2]) * inv, __uint_as_float(o[8 * j + 3]) * inv),
                                    pack_bf16(__uint_as_float(o[8 * j + 4]) * inv, __uint_as_float(o[8 * j + 5]) * inv),
                                    pack_bf16(__uint_as_float(o[8 * j + 6]) * inv, __uint_as_float(o[8 * j + 7]) * inv));
        } else {
            uint4* dst = reinterpret_cast<uint4*>(p.part_o + ((int64_t)it.partial_row + row) * D + d0);
#pragma unroll
            for (int j = 0; j < CH / 4; ++j) dst[j] = make_uint4(o[4 * j], o[4 * j + 1], o[4 * j + 2], o[4 * j + 3]);
        }
    }
    if (w == 0 && valid_row && it.partial_row >= 0) p.part_ml[(int64_t)it.partial_row + row] = make_float2(m_ref, l);
    ptx::tc_fence_before();
    ptx::named_bar_sync(bar_id, bar_n);                  // the exchange arrays are reused by the next item
}

// ------------------------------------------------------------------------------------------
// softmax warps, swap kind (D = 128, R <= RC <= 16 rows): thread <-> key of the tile (S^T lane)
// during the key loop, thread <-> d (O^T lane) for rescale / epilogue.  Column c = (token, head)
// row; columns in [R, RC) are computed as fully masked.  Straight-line code per column so the
// independent chains interleave; the column max is one REDUX per column and warp.
// ------------------------------------------------------------------------------------------
// fp8 pools: softmax warps of the swap kind (R <= RC <= 8 rows, D = 128): thread <-> key, as in softmax_swap.
// What differs (mma_swap8_item): Q^T and P^T are e4m3 operands, every value split into two codes x = hi + lo / 16
// stacked along N, so a score is S^T[key][c] + S^T[key][8 + c] / 16; the row scales of the pages are per key,
// i.e. per THREAD here: the K scale multiplies the thread's scores; the V scale goes into the weight
// w = p * vs (as an exponent shift lv = log2 vs, so the running maximum normalises w, not p, and w stays in
// (0, 2^8] whatever the scale), and the row sum takes w / vs = p back.  Q rows are scaled to amax 448 per row
// (qs[c], folded into the score).  One lg2 per thread and tile; nothing per element beyond the bf16 kind.
// ------------------------------------------------------------------------------------------
// ------------------------------------------------------------------------------------------
// Split-KV groups of the swap kind are merged INSIDE this kernel (H5 without a launch: the combine kernel and its
// dependency hop cost a decode-only round 6-12 us per layer): every split writes its partial rows,
// fences, and arrives on the group's counter; the split that arrives last merges all of them.  The counter is back
// at 0 when the kernel ends.  Rolled loops, inlined (a call would put a stack frame into the kernel): it runs once per
// group, outside every hot loop.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ int arrive_split(const Params& p, int aux) {
    const int n = p.meta.combine[p.meta.n_combine + aux].n_splits;
    if (atomicAdd(&p.group_cnt[aux], 1) != n - 1) return 0;
    p.group_cnt[aux] = 0;                                // nobody else touches it in this launch
    return 1;
}
// The 4 warps of the warpgroup take the group's rows round-robin; per row the lanes first hold one split each
// ((m_s, l_s) -> m = max m_s, w_s = 2^(m_s - m), sum w_s l_s by shuffles), then four d each: O = sum w_s O_s with the
// weights broadcast by shuffle, so the loads of a row are independent and issue back to back (combine_kernel's scheme).
__device__ __forceinline__ void merge_swap_group(const CombineItem* group, const float2* part_ml, const float* part_o,
                                                 __nv_bfloat16* out, int G, int Hq, int warp, int lane) {
    const CombineItem ci = *group;
    const int R = ci.q_tokens * G, gs = 31 - __clz(G);     // G is a power of two (cp_create)
    __threadfence();                                     // the other splits' rows were fenced before their arrival
#pragma unroll 1
    for (int r = warp; r < R; r += 4) {
        // 32-bit offsets from the row's base pointers (n_splits * R * 128 stays far below 2^31)
        const float2* ml_r = part_ml + ((int64_t)ci.partial_row + r);
        const float* o_r = part_o + ((int64_t)ci.partial_row + r) * 128 + lane * 4;
        float M = -INFINITY;
#pragma unroll 1
        for (int s = lane; s < ci.n_splits; s += 32) M = fmaxf(M, __ldcg(ml_r + s * R).x);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, o));
        float L = 0.f, acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll 1
        for (int s0 = 0; s0 < ci.n_splits; s0 += 32) {
            float w = 0.f;
            if (s0 + lane < ci.n_splits) {
                const float2 ml = __ldcg(ml_r + (s0 + lane) * R);
                w = (ml.x == -INFINITY) ? 0.f : exp2f(ml.x - M);      // empty split: weight 0
                L = fmaf(w, ml.y, L);                                  // this lane's share; summed over the lanes below
            }
            const int ns = min(32, ci.n_splits - s0);
#pragma unroll 4
            for (int j = 0; j < ns; ++j) {
                const float wj = __shfl_sync(0xffffffffu, w, j);
                const float4 v = __ldcg(reinterpret_cast<const float4*>(o_r + (s0 + j) * R * 128));
                acc[0] = fmaf(wj, v.x, acc[0]); acc[1] = fmaf(wj, v.y, acc[1]);
                acc[2] = fmaf(wj, v.z, acc[2]); acc[3] = fmaf(wj, v.w, acc[3]);
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) L += __shfl_xor_sync(0xffffffffu, L, o);
        const int tok = ci.tok0 + (r >> gs), head = ci.kv_head * G + (r & (G - 1));
        const float inv = 1.f / L;
        uint2 o2;
        o2.x = pack_bf16(acc[0] * inv, acc[1] * inv);
        o2.y = pack_bf16(acc[2] * inv, acc[3] * inv);
        *reinterpret_cast<uint2*>(out + ((int64_t)tok * Hq + head) * 128 + lane * 4) = o2;
    }
}
__device__ __forceinline__ void finish_swap_item(const Params& p, LaneState* ls, int d, int bar_id) {
    const int aux = ls->cur_aux;
    if (aux >= 0) {                                      // uniform over the 128 threads
        __threadfence();                                 // this split's partial rows, before its arrival
        ptx::named_bar_sync(bar_id, 128);
        if (d == 0) ls->last_split = arrive_split(p, aux);
        ptx::named_bar_sync(bar_id, 128);
        if (ls->last_split) merge_swap_group(p.meta.combine + p.meta.n_combine + aux, p.part_ml, p.part_o, p.out, p.sh.G, p.sh.Hq, d >> 5, d & 31);
    }
}

__device__ __forceinline__ uint32_t e4m3_of(float x) {             // round to nearest even, saturating
    uint16_t r;
    asm("cvt.rn.satfinite.e4m3x2.f32 %0, %1, %2;" : "=h"(r) : "f"(0.f), "f"(x));
    return r & 0xffu;
}
__device__ __forceinline__ float e4m3_value(uint32_t code) {
    uint32_t h2;
    asm("cvt.rn.f16x2.e4m3x2 %0, %1;" : "=r"(h2) : "h"((uint16_t)code));
    return __half2float(__ushort_as_half((unsigned short)(h2 & 0xffffu)));
}

template <int RC>
__device__ __forceinline__ void softmax_swap8(const WorkItem& it, const Params& p, uint8_t* small, LaneState* ls,
                                              uint32_t tmem, uint32_t& gt, uint32_t& gp, int row, uint32_t lane_base, int swarp, int LANE) {
    constexpr int D = 128;
    const Shape& sh = p.sh;
    const int G = sh.G;
    const int gs = 31 - __clz(G);
    const int R = it.q_tokens * G;                       // <= RC
    const int n_tiles = (it.kv_end - it.kv_begin + kKeyTile - 1) / kKeyTile;
    const int tok0 = p.meta.cu_q[it.req] + it.q_start;
    const int ctx = p.meta.ctx_off[it.req];
    const float scale = sh.sm_scale * 1.4426950408889634f;
    const int lane = row & 31;
    const int32_t* bt = p.meta.block_table + p.meta.bt_off[it.req];

    // ---- Q8^T -> smem: B operand [16 rows][128 B], K-major, 128B swizzle: row c = hi codes of Q row c, row 8 + c = lo codes.
    // 16 threads per Q row, 8 elements each; the row maximum by shuffles inside the half-warp.
    for (int id = row; id < RC * 16; id += 128) {
        const int r = id >> 4, c = id & 15;
        float x[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) x[j] = 0.f;
        if (r < R) {
            const int tok = tok0 + (r >> gs), head = it.kv_head * G + (r & (G - 1));
            const uint4 v = *reinterpret_cast<const uint4*>(p.q + ((int64_t)tok * sh.Hq + head) * D + c * 8);
            const __nv_bfloat162* h2 = reinterpret_cast<const __nv_bfloat162*>(&v);
#pragma unroll
            for (int j = 0; j < 4; ++j) { const float2 f = __bfloat1622float2(h2[j]); x[2 * j] = f.x; x[2 * j + 1] = f.y; }
        }
        float amax = 0.f;
#pragma unroll
        for (int j = 0; j < 8; ++j) amax = fmaxf(amax, fabsf(x[j]));
#pragma unroll
        for (int o = 8; o > 0; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
        const float qs = amax > 0.f ? amax * (1.f / 448.f) : 1.f;
        const float inv = 1.f / qs;
        uint32_t hi[2] = {0, 0}, lo[2] = {0, 0};
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const float y = x[j] * inv;
            const uint32_t h = e4m3_of(y);
            const uint32_t l = e4m3_of((y - e4m3_value(h)) * 16.f);
            hi[j >> 2] |= h << ((j & 3) * 8);
            lo[j >> 2] |= l << ((j & 3) * 8);
        }
        const uint32_t off = (((uint32_t)(c >> 1) ^ (uint32_t)(r & 7)) << 4) + (c & 1) * 8;      // (8 + r) & 7 == r & 7
        *reinterpret_cast<uint2*>(small + r * 128 + off) = make_uint2(hi[0], hi[1]);
        *reinterpret_cast<uint2*>(small + (8 + r) * 128 + off) = make_uint2(lo[0], lo[1]);
        if (c == 0) ls->qs[r] = qs;
    }
    ptx::fence_proxy_async_smem();
    warp_arrive(&ls->q_full[1]);
    ptx::named_bar_sync(1 + LANE, 128);                  // the row scales of Q8^T are there
    float qsc[RC];
#pragma unroll
    for (int c = 0; c < RC; ++c) qsc[c] = ls->qs[c] * scale;

    float m_ref[RC], l_part[RC];
    int limit[RC];
#pragma unroll
    for (int c = 0; c < RC; ++c) {
        m_ref[c] = -INFINITY;
        l_part[c] = 0.f;
        limit[c] = c < R ? min(it.kv_end, ctx + it.q_start + (c >> gs) + 1) : 0;
    }
    const uint32_t t_row = tmem + (lane_base << 16);
    // P8^T code (col c, key `row`): B operand [16 rows][128 keys], K-major along keys, one byte per key
    const uint32_t pchunk = (uint32_t)row >> 4;          // 16-byte chunk of this thread's key byte; swizzled with the row (c & 7)
    // the row scales of this thread's key, one tile ahead (a dependent pair of global loads: page id, then scales)
    auto load_scales = [&](int k, float& ks, float& vs) {
        const int key = it.kv_begin + k * kKeyTile + row;
        ks = 1.f; vs = 1.f;
        if (k < n_tiles && key < it.kv_end) {
            const int64_t pg = bt[key >> 4];
            const int64_t base = (pg * 2 * sh.Hkv + it.kv_head) * 16 + (key & 15);
            ks = p.kv_scale[base];
            vs = p.kv_scale[base + (int64_t)sh.Hkv * 16];
        }
    };
    float ks_n, vs_n;
    load_scales(0, ks_n, vs_n);

    for (int k = 0; k < n_tiles; ++k) {
        const int key = it.kv_begin + k * kKeyTile + row;
        const float ksc = ks_n, vs = vs_n;
        load_scales(k + 1, ks_n, vs_n);
        const float lv = __log2f(vs), ivs = 1.f / vs;        // vs is a power of two: both exact
        const uint32_t buf = gt & 1;
        ptx::mbar_wait(&ls->s_full[buf], (gt >> 1) & 1);
        ptx::tc_fence_after();
        uint32_t sh_[RC], sl_[RC];
        ptx::tmem_ld<RC>(t_row + col_s(LANE, buf), sh_);
        ptx::tmem_ld<RC>(t_row + col_s(LANE, buf) + 8, sl_);
        ptx::tmem_wait_ld();
        float sv[RC];
        int* cm = reinterpret_cast<int*>(&ls->cmax[k & 1][swarp][0]);
#pragma unroll
        for (int c = 0; c < RC; ++c) {
            const float raw = fmaf(__uint_as_float(sl_[c]), 0.0625f, __uint_as_float(sh_[c]));
            sv[c] = key < limit[c] ? fmaf(raw, ksc * qsc[c], lv) : -INFINITY;
            const int w = __reduce_max_sync(0xffffffffu, ptx::f2ord(sv[c]));
            if (lane == 0) cm[c] = w;
        }
        ptx::named_bar_sync(1 + LANE, 128);
        bool any_rescale = false;
        float alpha[RC];
        const int* cm0 = reinterpret_cast<const int*>(&ls->cmax[k & 1][0][0]);
#pragma unroll
        for (int c = 0; c < RC; ++c) {
            const float m_t = ptx::ord2f(max(max(cm0[c], cm0[16 + c]), max(cm0[32 + c], cm0[48 + c])));
            alpha[c] = 1.f;
            if (m_t > m_ref[c] + kRescaleThreshold) {
                alpha[c] = (m_ref[c] == -INFINITY) ? 0.f : ptx::ex2(m_ref[c] - m_t);
                m_ref[c] = m_t;
                any_rescale = true;
            }
            const float w = key < limit[c] ? ptx::ex2(sv[c] - m_ref[c]) : 0.f;      // weight p * vs, in (0, 2^8]
            l_part[c] = l_part[c] * alpha[c] + w * ivs;
            sv[c] = w;
        }
        if (k >= 2) {                                    // PV(gt-2) done: this P8^T buffer is free again
            ptx::mbar_wait(&ls->pv_done[buf], ((gt - 2) >> 1) & 1);
        }
        {
            uint8_t* ptb = small + 4096 + buf * 4096 + (row & 15);
#pragma unroll
            for (int c = 0; c < RC; ++c) {
                const uint32_t h = e4m3_of(sv[c]);
                const uint32_t l = e4m3_of((sv[c] - e4m3_value(h)) * 16.f);
                const uint32_t off = (pchunk ^ (uint32_t)(c & 7)) << 4;
                ptb[c * 128 + off] = (uint8_t)h;
                ptb[(8 + c) * 128 + off] = (uint8_t)l;
            }
        }
        if (k > 0 && any_rescale) {                      // uniform over the 128 threads
            ptx::mbar_wait(&ls->pv_done[(gt - 1) & 1], ((gt - 1) >> 1) & 1);
            ptx::tc_fence_after();
            uint32_t o[RC];
#pragma unroll
            for (int half = 0; half < 2; ++half) {
                ptx::tmem_ld<RC>(t_row + col_o(LANE) + half * 8, o);
                ptx::tmem_wait_ld();
#pragma unroll
                for (int c = 0; c < RC; ++c) o[c] = __float_as_uint(__uint_as_float(o[c]) * alpha[c]);
                ptx::tmem_st<RC>(t_row + col_o(LANE) + half * 8, o);
            }
            ptx::tmem_wait_st();
        }
        ptx::fence_proxy_async_smem();
        ptx::tc_fence_before();
        warp_arrive(&ls->p_full[1][gp & 1]);
        ++gt;
        ++gp;
    }

    // ---- column sums over the 128 key lanes
#pragma unroll
    for (int c = 0; c < RC; ++c) {
        float w = l_part[c];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) w += __shfl_xor_sync(0xffffffffu, w, o);
        if (lane == 0) ls->lsum[swarp][c] = w;
    }
    ptx::named_bar_sync(1 + LANE, 128);
    // ---- epilogue: O^T[d = row][c] = hi part + lo part / 16 -> out / workspace
    ptx::mbar_wait(&ls->pv_done[(gt - 1) & 1], ((gt - 1) >> 1) & 1);
    ptx::tc_fence_after();
    uint32_t oh[RC], ol[RC];
    ptx::tmem_ld<RC>(t_row + col_o(LANE), oh);
    ptx::tmem_ld<RC>(t_row + col_o(LANE) + 8, ol);
    ptx::tmem_wait_ld();
#pragma unroll
    for (int c = 0; c < RC; ++c) {
        if (c < R) {
            const float lc = ls->lsum[0][c] + ls->lsum[1][c] + ls->lsum[2][c] + ls->lsum[3][c];
            const float o = fmaf(__uint_as_float(ol[c]), 0.0625f, __uint_as_float(oh[c]));
            if (it.partial_row < 0) {
                const int tok = tok0 + (c >> gs), head = it.kv_head * G + (c & (G - 1));
                p.out[((int64_t)tok * sh.Hq + head) * D + row] = __float2bfloat16_rn(__fdividef(o, lc));
            } else {
                p.part_o[((int64_t)it.partial_row + c) * D + row] = o;
                if (row == c) p.part_ml[(int64_t)it.partial_row + c] = make_float2(m_ref[c], lc);
            }
        }
    }
    ptx::tc_fence_before();
    ptx::named_bar_sync(1 + LANE, 128);                  // lsum / cmax / qs are reused by the next item
}
// ------------------------------------------------------------------------------------------
template <int RC>
__device__ __forceinline__ void softmax_swap(const WorkItem& it, const Params& p, uint8_t* small, LaneState* ls,
                                             uint32_t tmem, uint32_t& gt, uint32_t& gp, int row, uint32_t lane_base, int swarp, int LANE) {
    constexpr int D = 128;
    const Shape& sh = p.sh;
    const int G = sh.G;
    const int gs = 31 - __clz(G);                        // G is a power of two (cp_create): a runtime division per
                                                         // unrolled column made the per-item code tens of KB of SASS
    const int R = it.q_tokens * G;                       // <= RC
    const int n_tiles = (it.kv_end - it.kv_begin + kKeyTile - 1) / kKeyTile;
    const int tok0 = p.meta.cu_q[it.req] + it.q_start;
    const int ctx = p.meta.ctx_off[it.req];
    const float scale = sh.sm_scale * 1.4426950408889634f;
    const int lane = row & 31;

    // ---- Q^T -> smem: B operand [16 rows][D], K-major, 128B swizzle, halves 2 KB apart
    for (int id = row; id < RC * (D / 8); id += 128) {
        const int r = id >> 4, c = id & 15;
        uint4 v = make_uint4(0, 0, 0, 0);
        if (r < R) {
            const int tok = tok0 + (r >> gs), head = it.kv_head * G + (r & (G - 1));
            v = *reinterpret_cast<const uint4*>(p.q + ((int64_t)tok * sh.Hq + head) * D + c * 8);
        }
        *reinterpret_cast<uint4*>(small + (c >> 3) * 2048 + r * 128 + (((c & 7) ^ (r & 7)) << 4)) = v;
    }
    ptx::fence_proxy_async_smem();
    warp_arrive(&ls->q_full[1]);

    float m_ref[RC], l_part[RC];
    int limit[RC];
#pragma unroll
    for (int c = 0; c < RC; ++c) {
        m_ref[c] = -INFINITY;
        l_part[c] = 0.f;
        limit[c] = c < R ? min(it.kv_end, ctx + it.q_start + (c >> gs) + 1) : 0;
    }
    const uint32_t t_row = tmem + (lane_base << 16);
    // P^T element (col c, key `row`): B operand [16 rows][128 keys], K-major, halves (64 keys) 2 KB apart
    uint8_t* pt = small + 4096 + (row >> 6) * 2048 + (row & 7) * 2;
    const int pchunk = (row & 63) >> 3;

    for (int k = 0; k < n_tiles; ++k) {
        const int key = it.kv_begin + k * kKeyTile + row;
        const uint32_t buf = gt & 1;
        ptx::mbar_wait(&ls->s_full[buf], (gt >> 1) & 1);
        ptx::tc_fence_after();
        uint32_t sr[RC];
        ptx::tmem_ld<RC>(t_row + col_s(LANE, buf), sr);
        ptx::tmem_wait_ld();
        float sv[RC];
        int* cm = reinterpret_cast<int*>(&ls->cmax[k & 1][swarp][0]);
#pragma unroll
        for (int c = 0; c < RC; ++c) {
            sv[c] = key < limit[c] ? __uint_as_float(sr[c]) * scale : -INFINITY;
            const int w = __reduce_max_sync(0xffffffffu, ptx::f2ord(sv[c]));
            if (lane == 0) cm[c] = w;
        }
        ptx::named_bar_sync(1 + LANE, 128);
        bool any_rescale = false;
        float alpha[RC];
        const int* cm0 = reinterpret_cast<const int*>(&ls->cmax[k & 1][0][0]);
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
        if (k >= 2) {                                    // PV(gt-2) done: this P^T buffer is free again
            ptx::mbar_wait(&ls->pv_done[buf], ((gt - 2) >> 1) & 1);
        }
        {
            uint8_t* ptb = pt + buf * 4096;
#pragma unroll
            for (int c = 0; c < RC; ++c)
                *reinterpret_cast<__nv_bfloat16*>(ptb + c * 128 + ((pchunk ^ (c & 7)) << 4)) = __float2bfloat16_rn(sv[c]);
        }
        if (k > 0 && any_rescale) {                      // uniform over the 128 threads
            ptx::mbar_wait(&ls->pv_done[(gt - 1) & 1], ((gt - 1) >> 1) & 1);
            ptx::tc_fence_after();
            uint32_t o[RC];
            ptx::tmem_ld<RC>(t_row + col_o(LANE), o);
            ptx::tmem_wait_ld();
#pragma unroll
            for (int c = 0; c < RC; ++c) o[c] = __float_as_uint(__uint_as_float(o[c]) * alpha[c]);
            ptx::tmem_st<RC>(t_row + col_o(LANE), o);
            ptx::tmem_wait_st();
        }
        ptx::fence_proxy_async_smem();
        ptx::tc_fence_before();
        warp_arrive(&ls->p_full[1][gp & 1]);
        ++gt;
        ++gp;
    }

    // ---- column sums over the 128 key lanes
#pragma unroll
    for (int c = 0; c < RC; ++c) {
        float w = l_part[c];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) w += __shfl_xor_sync(0xffffffffu, w, o);
        if (lane == 0) ls->lsum[swarp][c] = w;
    }
    ptx::named_bar_sync(1 + LANE, 128);
    // ---- epilogue: O^T[d = row][c] -> out / workspace
    ptx::mbar_wait(&ls->pv_done[(gt - 1) & 1], ((gt - 1) >> 1) & 1);
    ptx::tc_fence_after();
    uint32_t o[RC];
    ptx::tmem_ld<RC>(t_row + col_o(LANE), o);
    ptx::tmem_wait_ld();
#pragma unroll
    for (int c = 0; c < RC; ++c) {
        if (c < R) {
            const float lc = ls->lsum[0][c] + ls->lsum[1][c] + ls->lsum[2][c] + ls->lsum[3][c];
            if (it.partial_row < 0) {
                const int tok = tok0 + (c >> gs), head = it.kv_head * G + (c & (G - 1));
                p.out[((int64_t)tok * sh.Hq + head) * D + row] = __float2bfloat16_rn(__fdividef(__uint_as_float(o[c]), lc));
            } else {
                p.part_o[((int64_t)it.partial_row + c) * D + row] = __uint_as_float(o[c]);
                if (row == c) p.part_ml[(int64_t)it.partial_row + c] = make_float2(m_ref[c], lc);
            }
        }
    }
    ptx::tc_fence_before();
    ptx::named_bar_sync(1 + LANE, 128);                  // lsum / cmax are reused by the next item
}

// softmax warpgroup loop.  ROLE 0: lane T (tile kind, and the swap-kind items lane T picks up);
// ROLE 2: lane S.
// SPLIT: all warpgroups follow lane 0's item ring; ROLE 0 = warpgroup 0 of the column split (and the swap-kind
// items), ROLE 2 = warpgroups wg >= 1 (swap-kind items are skipped).
template <int D, bool POLY, bool SPLIT, bool KV8>
__device__ __forceinline__ void softmax_warps(const Params& p, uint8_t* smem, Misc* misc, int warp, int lane, int ROLE, int wg) {
    using L = Layout<D, SPLIT>;
    // ROLE is a warp-uniform runtime value (as the lane is in producer()): where the kernel calls this from ONE site
    // (fp8 pages) one copy of the code serves both softmax warpgroups; where it calls it once per warpgroup with a
    // constant, each call is specialised as if ROLE were a template parameter (bf16 pages)
    const int LANE = (ROLE == 2 && !SPLIT) ? 1 : 0;
    LaneState* ls = &misc->lane[LANE];
    const uint32_t tmem = misc->tmem_base;
    const uint32_t lane_base = (warp & 3) * 32;
    const int row = lane_base + lane;
    constexpr uint32_t kOffSmall0 = L::kOffSmall[0], kOffSmall1 = L::kOffSmall[1];
    uint8_t* small = smem + (LANE == 0 ? kOffSmall0 : kOffSmall1);
    uint32_t gt = 0, item_cnt = 0, gh_tile = 0, gp_swap = 0;      // gt / gp_swap: swap-kind tiles; gh_tile: tile-kind half-tiles
    for (;;) {
        const uint32_t islot = item_cnt % kItemRing;
        ptx::mbar_wait(&ls->item_full[islot], (item_cnt / kItemRing) & 1);
        const WorkItem it = ls->items[islot];
        // (SPLIT: both warpgroups follow this ring, only the first works on swap-kind items)
        if ((threadIdx.x & 127) == 0 && (!SPLIT || ROLE == 0)) ls->cur_aux = ls->aux[islot];    // read back in finish_swap_item, barriers in between
        warp_arrive(&ls->item_empty[islot]);
        if (it.kind < 0) break;
        if constexpr (SPLIT) {
            if (it.kind == kKindTile) {
                softmax_split<D, POLY>(it, p, ls, tmem, small, gh_tile, row, lane_base, ROLE == 2 ? wg : 0);
                ++item_cnt;
                continue;
            }
            if (ROLE == 2) { ++item_cnt; continue; }
        }
        if (ROLE == 2 || it.kind == kKindSwap) {
            if constexpr (D == 128) {
                const int R = it.q_tokens * p.sh.G;
                if constexpr (KV8) {
                    if (R <= 4) softmax_swap8<4>(it, p, small, ls, tmem, gt, gp_swap, row, lane_base, warp & 3, LANE);
                    else softmax_swap8<8>(it, p, small, ls, tmem, gt, gp_swap, row, lane_base, warp & 3, LANE);
                } else
                if (R <= 4) softmax_swap<4>(it, p, small, ls, tmem, gt, gp_swap, row, lane_base, warp & 3, LANE);
                else if (R <= 8) softmax_swap<8>(it, p, small, ls, tmem, gt, gp_swap, row, lane_base, warp & 3, LANE);
                else softmax_swap<16>(it, p, small, ls, tmem, gt, gp_swap, row, lane_base, warp & 3, LANE);
                if (it.partial_row >= 0) finish_swap_item(p, ls, row, 1 + LANE);       // H5 for the item's group, if it is the last split
            }
        } else {
            if constexpr (!SPLIT) softmax_tile<D, POLY, KV8>(it, p, ls, tmem, gh_tile, row, lane_base);
        }
        ++item_cnt;
    }
}

// ------------------------------------------------------------------------------------------
// the kernel
// ------------------------------------------------------------------------------------------
// KV8 (fp8 pools, dual-lane only): tmap = the library's bf16 scratch pool (chunk tiles), tmap8 = the e4m3 pool (decode
// streams); otherwise tmap = the bf16 pool and tmap8 is a copy of it, unused.
template <int D, bool POLY, bool SPLIT, bool KV8, bool APPEND = false>
__global__ void __launch_bounds__(threads_of<SPLIT>(), 1)
attn_dl_kernel(const Params p, const __grid_constant__ CUtensorMap tmap, const __grid_constant__ CUtensorMap tmap8) {
    static_assert(!(KV8 && (SPLIT || D != 128)), "fp8 pools: dual-lane instantiation, D = 128");
    static_assert(!(APPEND && (SPLIT || KV8 || D != 128)), "fused append: decode-only batches over bf16 pages, D = 128");
    using L = Layout<D, SPLIT>;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    Misc* misc = reinterpret_cast<Misc*>(smem + L::kOffMisc);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        for (int ln = 0; ln < 2; ++ln) {
            LaneState* ls = &misc->lane[ln];
            for (int i = 0; i < kMaxStages; ++i) { ptx::mbar_init(&ls->kv_full[i], 1); ptx::mbar_init(&ls->kv_empty[i], 1); }
            ptx::mbar_init(&ls->q_full[0], 4);
            ptx::mbar_init(&ls->q_full[1], 4);
            for (int i = 0; i < 2; ++i) {
                ptx::mbar_init(&ls->s_full[i], 1);
                ptx::mbar_init(&ls->p_full[0][i], 4);
                ptx::mbar_init(&ls->p_full[1][i], 4);
                ptx::mbar_init(&ls->pv_done[i], 1);
            }
            for (int i = 0; i < 4; ++i) {
                ptx::mbar_init(&ls->ts_full[i], 1);
                ptx::mbar_init(&ls->tp_full[i], SPLIT ? 4 * kSplitWG : 4);      // SPLIT: every warpgroup delivers its part of P
                ptx::mbar_init(&ls->tpv_done[i], 1);
                ptx::mbar_init(&ls->pv_issued[i], 1);
            }
            // readers of the item ring (one arrival per warp): the lane's 4 softmax warps, its MMA warp(s), its other producers
            // (SPLIT: one ring for everybody -- the softmax warps, 1 issuer, the other producers)
            for (int i = 0; i < kItemRing; ++i) { ptx::mbar_init(&ls->item_full[i], 1); ptx::mbar_init(&ls->item_empty[i], SPLIT ? 4 * kSplitWG + 1 + kProdSplit - 1 : 4 + (ln == 0 ? 2 + kProdT - 1 : 1 + kProdS - 1)); }
        }
        ptx::fence_barrier_init();
        ptx::prefetch_tmap(&tmap);
        if (KV8) ptx::prefetch_tmap(&tmap8);
    }
    if (warp == 6) ptx::tmem_alloc(&misc->tmem_base, kTmemCols);
    // Stale shared memory may hold NaN bit patterns, tiles are only partly overwritten by short requests, and
    // masked P = 0 times a NaN V row would poison the accumulators.  After this clear everything that ever sits
    // in the ring is finite: K/V rows that are keys of their request, page tails that the append kernel zeroed
    // (cp_kernels_simt.cuh), or these zeros.
    for (uint32_t i = threadIdx.x * 16; i < L::kOffMisc; i += threads_of<SPLIT>() * 16)
        *reinterpret_cast<uint4*>(smem + i) = make_uint4(0, 0, 0, 0);
    ptx::fence_proxy_async_smem();
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    // up to here nothing written by the preceding kernels (KV append; the previous step) was read
    ptx::grid_dep_wait();
    ptx::grid_dep_launch();                              // the combine kernel may stage its launch

    // launch allocation: 128 registers per thread (SPLIT with four warpgroups: 768 threads at 80).  The two
    // producer / MMA warpgroups give most of their share to the tile softmax (a score row, or its part, in
    // registers) and the decode softmax.
    constexpr bool kWide = SPLIT && kSplitWG == 4;       // 8 warps x 48 + 16 warps x 96 = 24 warps x 80
    if (warp < 8) {
        reg_dec<kWide ? 48 : 56>();
        if (warp < kProdT + kProdS) producer<D, SPLIT, KV8, APPEND>(p, &tmap, &tmap8, smem, misc, lane, warp);
        else if (warp == 5) mma_warp<D, 0, 1, SPLIT, KV8>(ptx::smem_u32(smem), misc, lane);     // lane T: score blocks (and swap items); SPLIT: the one issuer
        else if (SPLIT) { }                                                                      // SPLIT: warps 6, 7 have no role
        else if (warp == 6) mma_warp<D, 0, 2, false, KV8>(ptx::smem_u32(smem), misc, lane);     // lane T: PV blocks
        else mma_warp<D, 1, 0, false, KV8>(ptx::smem_u32(smem), misc, lane);                    // lane S
    } else if (KV8) {
        // fp8 pages: ONE call site, so both softmax warpgroups run the same code copy and take the same register
        // budget (2 x 128 x 200 + 256 x 56 = 64 K registers).  A copy of the fp8 decode softmax per warpgroup did not
        // fit the instruction cache (stall_no_instruction 2.2 per issue): 512 decodes 334 -> 296 us.
        reg_inc<200>();
        softmax_warps<D, POLY, SPLIT, KV8>(p, smem, misc, warp, lane, warp < 12 ? 0 : 2, 0);
    } else if (warp < 12) {
        // bf16 pages: a copy per warpgroup, each with the register budget its role wants -- the shared copy measured
        // 0.6 % slower on configs[2] (626 against 622 us) and 0.4-0.8 % slower in SPLIT mode (A/B on one box)
        reg_inc<kWide ? 96 : SPLIT ? 200 : 232>();
        softmax_warps<D, POLY, SPLIT, KV8>(p, smem, misc, warp, lane, 0, 0);
    } else {
        reg_inc<kWide ? 96 : SPLIT ? 200 : 160>();
        softmax_warps<D, POLY, SPLIT, KV8>(p, smem, misc, warp, lane, 2, (warp - 8) >> 2);
    }
    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 6) ptx::tmem_dealloc(misc->tmem_base, kTmemCols);
    if (threadIdx.x == 0) {
        __threadfence();
        if (atomicAdd(&p.counters[2], 1) == (int)gridDim.x - 1) {      // last CTA re-arms the counters
            p.counters[0] = 0;
            p.counters[1] = 0;
            p.counters[2] = 0;
            __threadfence();
        }
    }
}

}  // namespace dl
}  // namespace cp
