// cp_static.cu -- cp_decode_attention_static: split-KV decode attention that allocates NOTHING (include/cp.h).
//
// For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
// it).  The library's normal path keeps its split-KV partials (an unnormalised fp32 O row and an (m, l) pair per
// (row, key-range split)) in a workspace that cp_create allocates; this variant of the split-KV decode kernel keeps
// them in a file-scope static device array of a fixed, modest size.  Every GPU that loads libcp.so holds that array
// until the process exits.  All calls share it and it keeps the last call's contents: a call overwrites every partial
// it later reads (nothing has to start at zero, so nothing is cleared), and calls that overlap on the GPU -- two
// streams, or two host threads on the same device -- race on it.
//
// Operation: include/cp.h / DESIGN.md section 2 for q_len = 1: row (request j, q head h) attends
// to keys [0, kv_len[j]) of KV head h / G in the request's pages; softmax in fp32, base-2 exponentials of
// (q . k) * sm_scale * log2(e); out in bf16.
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <mutex>

#include "cp_internal.h"

// ---- the scratch: [kMaxRows][128] fp32 partial O rows, then [kMaxRows] float2 (m, l) ---------------------------------
constexpr int kMaxRows = CP_STATIC_MAX_PARTIAL_ROWS;             // (request, q head, split) triples per call
constexpr int kMaxD = 128;
constexpr size_t kPartOBytes = (size_t)kMaxRows * kMaxD * sizeof(float);
constexpr size_t kScratchBytes = kPartOBytes + (size_t)kMaxRows * sizeof(float2);
static_assert(kScratchBytes == CP_STATIC_SCRATCH_BYTES, "include/cp.h states the size of the static scratch");

static __device__ __align__(256) unsigned char cp_static_scratch[kScratchBytes];

namespace {

// In HOST code the name above is a host-side stand-in, not a device address: the kernels get the address that
// cudaGetSymbolAddress returns, looked up once per device with that device current.
constexpr int kMaxDevices = 64;
std::mutex g_mu;
unsigned char* g_scratch_ptr[kMaxDevices] = {};

int scratch_of_current_device(unsigned char** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { cp_set_error("cp_decode_attention_static: cudaGetDevice: %s", cudaGetErrorString(e)); return CP_ECUDA; }
    if (dev < 0 || dev >= kMaxDevices) { cp_set_error("cp_decode_attention_static: device ordinal %d not supported (< %d)", dev, kMaxDevices); return CP_EINVAL; }
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_ptr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, cp_static_scratch);
        if (e != cudaSuccess || !p) {
            cp_set_error("cp_decode_attention_static: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
            return CP_ECUDA;
        }
        g_scratch_ptr[dev] = static_cast<unsigned char*>(p);
    }
    *out = g_scratch_ptr[dev];
    return CP_OK;
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// ---- split-KV decode kernel: one warp per (request, q head, split); lanes over D; partials -> scratch ----------------
// Partial row index r = (j * Hq + h) * n_splits + s.  Split s of request j covers keys [s * c, min(kv_len, (s + 1) c)),
// c = ceil(kv_len / n_splits); an empty range writes (m, l) = (-inf, 0) and a zero row.
template <int D>
__global__ void __launch_bounds__(128)
decode_split_static_kernel(const __nv_bfloat16* __restrict__ q, const __nv_bfloat16* __restrict__ cache,
                           const int32_t* __restrict__ block_tables, const int32_t* __restrict__ kv_len,
                           int n_reqs, int max_pages, int Hq, int Hkv, int B, float scale_log2, int n_splits,
                           float* __restrict__ part_o, float2* __restrict__ part_ml) {
    constexpr int EPL = D / 32;                           // elements per lane
    const int lane = threadIdx.x & 31;
    const int r = blockIdx.x * 4 + (threadIdx.x >> 5);
    if (r >= n_reqs * Hq * n_splits) return;
    const int s = r % n_splits, h = (r / n_splits) % Hq, j = r / (n_splits * Hq);
    const int g = h / (Hq / Hkv);
    const int n = kv_len[j];
    const int c = (n + n_splits - 1) / n_splits;
    const int k0 = s * c, k1 = min(n, k0 + c);
    float qv[EPL], acc[EPL];
#pragma unroll
    for (int e = 0; e < EPL; ++e) {
        qv[e] = __bfloat162float(q[((int64_t)j * Hq + h) * D + lane * EPL + e]) * scale_log2;
        acc[e] = 0.f;
    }
    float m = -INFINITY, l = 0.f;
    const int32_t* bt = block_tables + (int64_t)j * max_pages;
    for (int k = k0; k < k1; ++k) {
        const int64_t page = bt[k / B];
        const int slot = k % B;
        const __nv_bfloat16* kr = cache + ((((page * 2 + 0) * Hkv + g) * (int64_t)B + slot) * D) + lane * EPL;
        const __nv_bfloat16* vr = cache + ((((page * 2 + 1) * Hkv + g) * (int64_t)B + slot) * D) + lane * EPL;
        float dot = 0.f;
#pragma unroll
        for (int e = 0; e < EPL; ++e) dot = fmaf(qv[e], __bfloat162float(kr[e]), dot);
        const float sc = warp_sum(dot);                   // the same value in every lane
        const float m_new = fmaxf(m, sc);
        const float alpha = (m == -INFINITY) ? 0.f : exp2f(m - m_new);
        const float p = exp2f(sc - m_new);
        l = l * alpha + p;
#pragma unroll
        for (int e = 0; e < EPL; ++e) acc[e] = fmaf(p, __bfloat162float(vr[e]), acc[e] * alpha);
        m = m_new;
    }
#pragma unroll
    for (int e = 0; e < EPL; ++e) part_o[(int64_t)r * D + lane * EPL + e] = acc[e];
    if (lane == 0) part_ml[r] = make_float2(m, l);
}

// ---- combine: one warp per (request, q head): LSE merge of its n_splits partials -> bf16 out -------------------------
template <int D>
__global__ void __launch_bounds__(128)
decode_combine_static_kernel(const float* __restrict__ part_o, const float2* __restrict__ part_ml, int n_rows,
                             int n_splits, __nv_bfloat16* __restrict__ out) {
    constexpr int EPL = D / 32;
    const int lane = threadIdx.x & 31;
    const int row = blockIdx.x * 4 + (threadIdx.x >> 5);
    if (row >= n_rows) return;
    const int64_t base = (int64_t)row * n_splits;
    float M = -INFINITY;
    for (int s = 0; s < n_splits; ++s) M = fmaxf(M, part_ml[base + s].x);
    float L = 0.f, acc[EPL];
#pragma unroll
    for (int e = 0; e < EPL; ++e) acc[e] = 0.f;
    for (int s = 0; s < n_splits; ++s) {
        const float2 ml = part_ml[base + s];
        const float w = (ml.x == -INFINITY) ? 0.f : exp2f(ml.x - M);      // empty split: m = -inf -> weight 0
        L = fmaf(w, ml.y, L);
#pragma unroll
        for (int e = 0; e < EPL; ++e) acc[e] = fmaf(w, part_o[(base + s) * D + lane * EPL + e], acc[e]);
    }
    const float inv = 1.f / L;                            // kv_len >= 1: at least one key, L > 0
#pragma unroll
    for (int e = 0; e < EPL; ++e) out[(int64_t)row * D + lane * EPL + e] = __float2bfloat16_rn(acc[e] * inv);
}

template <int D>
int launch(const void* q, const void* kv_cache, const int32_t* block_tables, const int32_t* kv_len, int n_reqs,
           int max_pages, int Hq, int Hkv, int B, float sm_scale, int n_splits, void* out, cudaStream_t stream,
           unsigned char* scratch) {
    float* part_o = reinterpret_cast<float*>(scratch);
    float2* part_ml = reinterpret_cast<float2*>(scratch + kPartOBytes);
    const int n_rows = n_reqs * Hq, n_part = n_rows * n_splits;
    decode_split_static_kernel<D><<<(n_part + 3) / 4, 128, 0, stream>>>(
        static_cast<const __nv_bfloat16*>(q), static_cast<const __nv_bfloat16*>(kv_cache), block_tables, kv_len, n_reqs,
        max_pages, Hq, Hkv, B, sm_scale * 1.4426950408889634f, n_splits, part_o, part_ml);
    decode_combine_static_kernel<D><<<(n_rows + 3) / 4, 128, 0, stream>>>(part_o, part_ml, n_rows, n_splits,
                                                                        static_cast<__nv_bfloat16*>(out));
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { cp_set_error("cp_decode_attention_static: launch: %s", cudaGetErrorString(e)); return CP_ECUDA; }
    return CP_OK;
}

}  // namespace

extern "C" int cp_decode_attention_static(const void* q, const void* kv_cache, const int32_t* block_tables,
                                          const int32_t* kv_len, int32_t n_reqs, int32_t max_pages_per_req,
                                          int32_t num_q_heads, int32_t num_kv_heads, int32_t head_dim,
                                          int32_t block_size, float sm_scale, int32_t n_splits, void* out,
                                          void* stream) {
    if (!q || !kv_cache || !block_tables || !kv_len || !out) { cp_set_error("cp_decode_attention_static: null pointer"); return CP_EINVAL; }
    if (n_reqs < 1 || max_pages_per_req < 1 || n_splits < 1 || block_size < 1) {
        cp_set_error("cp_decode_attention_static: n_reqs, max_pages_per_req, n_splits and block_size must be >= 1");
        return CP_EINVAL;
    }
    if (head_dim != 64 && head_dim != 128) { cp_set_error("cp_decode_attention_static: head_dim %d (64 or 128)", head_dim); return CP_EINVAL; }
    if (num_q_heads < 1 || num_kv_heads < 1 || num_q_heads % num_kv_heads) {
        cp_set_error("cp_decode_attention_static: %d q heads are not a multiple of %d KV heads", num_q_heads, num_kv_heads);
        return CP_EINVAL;
    }
    if (!(sm_scale > 0.f) || !std::isfinite(sm_scale)) { cp_set_error("cp_decode_attention_static: sm_scale must be finite and > 0"); return CP_EINVAL; }
    const int64_t n_part = (int64_t)n_reqs * num_q_heads * n_splits;
    if (n_part > kMaxRows) {
        cp_set_error("cp_decode_attention_static: n_reqs * num_q_heads * n_splits = %lld exceeds the static scratch "
                     "(CP_STATIC_MAX_PARTIAL_ROWS = %d, %zu bytes); use fewer splits or requests per call, or the "
                     "cp_create / cp_attention_step path",
                     (long long)n_part, kMaxRows, kScratchBytes);
        return CP_ECAPACITY;
    }
    unsigned char* scratch = nullptr;
    const int rc = scratch_of_current_device(&scratch);
    if (rc != CP_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    return head_dim == 128
               ? launch<128>(q, kv_cache, block_tables, kv_len, n_reqs, max_pages_per_req, num_q_heads, num_kv_heads, block_size, sm_scale, n_splits, out, st, scratch)
               : launch<64>(q, kv_cache, block_tables, kv_len, n_reqs, max_pages_per_req, num_q_heads, num_kv_heads, block_size, sm_scale, n_splits, out, st, scratch);
}
