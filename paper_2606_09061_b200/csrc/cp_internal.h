// cp_internal.h -- structures shared by libcp's host code and its kernels.
#pragma once
#include <cstdint>

#include "cp.h"

void cp_set_error(const char* fmt, ...);

namespace cp {

constexpr int kKeyTile = 128;        // keys per KV tile (8 pages of 16)

// kinds of work item
constexpr int kKindTile = 0;         // Q tile of up to 128 rows (tokens x G heads) vs a key range
constexpr int kKindSwap = 1;         // <= 16 rows (decode / tiny chunk): keys are the MMA M dim

// One unit of work for the attention kernels: the G q-heads of KV head `kv_head`, for
// tokens [q_start, q_start + q_tokens) of request `req`, against keys
// [kv_begin, kv_end) (absolute positions in the request; kv_begin is a multiple of
// kKeyTile, kv_end <= ctx_off + q_start + q_tokens = the causal limit of the last row).
struct WorkItem {
    int32_t req;
    int32_t kv_head;
    int32_t q_start;
    int32_t q_tokens;
    int32_t kv_begin;
    int32_t kv_end;
    int32_t partial_row;   // >= 0: rows [partial_row, +q_tokens*G) of the split workspace; -1: write `out`
    int32_t kind;
};
static_assert(sizeof(WorkItem) == 32, "WorkItem is 32 bytes");

// Merge the n_splits partials of one (request, q tile, KV head) group into `out`.
struct CombineItem {
    int32_t tok0;          // global token index of the tile's first token
    int32_t q_tokens;
    int32_t kv_head;
    int32_t n_splits;
    int32_t partial_row;   // split s occupies rows [partial_row + s*R, +R), R = q_tokens*G
    int32_t row_base;      // sum of R over the preceding combine items (warp <-> row mapping)
    int32_t pad[2];
};
static_assert(sizeof(CombineItem) == 32, "CombineItem is 32 bytes");

// Device views of the batch metadata blob (one H2D copy per cp_build_batch).
struct BatchMeta {
    const int32_t* cu_q;         // [n_reqs + 1] prefix sums of q_len
    const int32_t* q_len;        // [n_reqs]
    const int32_t* ctx_off;      // [n_reqs]
    const int32_t* bt_off;       // [n_reqs + 1]
    const int32_t* block_table;  // [total pages]
    const WorkItem* work;        // [n_work] sorted by descending cost
    const CombineItem* combine;  // [n_combine]
    const int32_t* tok_req;      // [T] request of each token (for the append kernel)
    const int32_t* work_aux;     // [n_work] split item of a group merged INSIDE the attention kernel: its index among
                                 // those groups (combine[n_combine + aux]); -1 otherwise
    const int32_t* scratch_base; // fp8 pools: [n_reqs] first page of the request in the bf16 scratch pool, -1 = none
    const int32_t* scratch_req;  // fp8 pools: [scratch pages in use] request of each scratch page
    int32_t n_reqs, n_tokens, n_work, n_combine;   // n_combine: groups merged by combine_kernel (combine[0, n_combine))
    int32_t n_tile;              // dual-lane kernel: work[0, n_tile) are tile-kind items, the rest swap-kind
};

struct Shape {
    int32_t Hq, Hkv, D, B, G;
    float sm_scale;
};

}  // namespace cp
