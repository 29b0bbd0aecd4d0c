// cp_kernels_simt.cuh -- plain-ALU kernels of libcp for sm_100a:
//   kv_append_kernel   H2: scatter the iteration's new K/V rows into their pages
//   attn_simt_kernel   H3/H4 cross-check for bisecting (-DCP_DEBUG_VARIANTS builds only,
//                      kernel_variant = 1): one warp per (token, q head) row, no tensor cores
//   combine_kernel     H5: LSE merge of split-KV partials -> bf16 out
// Operation defined in include/cp.h / DESIGN.md section 2.
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include "cp_internal.h"

namespace cp {

__device__ __forceinline__ int64_t slab_elem_offset(int64_t page, int kv, int head, int Hkv, int B, int D) {
    return (((page * 2 + kv) * Hkv + head) * (int64_t)B) * D;
}

// ---------------------------------------------------------------------------------
// Stale page tails.  The attention kernel moves whole 16-token page slabs with TMA and masks the scores
// of slots that are not keys by select; but masked P = 0 still multiplies the V row of such a slot in the
// tensor-core PV product, and 0 x NaN is NaN.  So every step zeroes, for every request of the batch, the
// slots of its LAST page that lie past its last key (<= 15 slots x Hkv x K|V): they belong to the request,
// hold no key, and later appends overwrite them.  (K tails too: a K tile's stale rows can be left in a ring
// slot that a shorter V tile later only partly overwrites.)  With that and the kernel's prologue clear, a
// torch.empty pool or NaN-filled tails cannot reach a result (include/cp.h; reading R6).
// ---------------------------------------------------------------------------------
__device__ __forceinline__ void zero_page_tails(const BatchMeta& meta, const Shape& sh, __nv_bfloat16* __restrict__ cache) {
    // one warp per (request, K|V, kv head) slab of the request's last page: the 32 lanes sweep the 16-byte chunks of
    // the slots past the last key (contiguous memory: slots are adjacent rows of the slab)
    const int lane = threadIdx.x & 31;
    const int64_t n_warps = (int64_t)gridDim.x * (blockDim.x >> 5);
    const int64_t total = (int64_t)meta.n_reqs * 2 * sh.Hkv;
    for (int64_t w = blockIdx.x * (int64_t)(blockDim.x >> 5) + (threadIdx.x >> 5); w < total; w += n_warps) {
        const int g = (int)(w % sh.Hkv);
        const int kv = (int)((w / sh.Hkv) & 1);
        const int req = (int)(w / (2 * sh.Hkv));
        const int last = meta.ctx_off[req] + meta.q_len[req] - 1;       // position of the request's last key
        const int first_free = last % sh.B + 1;
        if (first_free >= sh.B) continue;
        const int64_t page = meta.block_table[meta.bt_off[req] + last / sh.B];
        uint4* dst = reinterpret_cast<uint4*>(cache + slab_elem_offset(page, kv, g, sh.Hkv, sh.B, sh.D) + (int64_t)first_free * sh.D);
        const int n16 = (sh.B - first_free) * sh.D / 8;
        for (int i = lane; i < n16; i += 32) dst[i] = make_uint4(0, 0, 0, 0);
    }
}

// ---------------------------------------------------------------------------------
// H2: one thread per 16-byte chunk of a (token, kv head, K|V) row; then the page tails (above).
// k_new == nullptr (the caller wrote the pages itself): only the page tails.
// ---------------------------------------------------------------------------------
__global__ void kv_append_kernel(BatchMeta meta, Shape sh, const uint4* __restrict__ k_new,
                                 const uint4* __restrict__ v_new, __nv_bfloat16* __restrict__ cache) {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");   // the attention kernel may start its prologue
    zero_page_tails(meta, sh, cache);
    const int chunks = sh.D / 8;                          // 16-byte chunks per row
    const int64_t total = k_new ? (int64_t)meta.n_tokens * sh.Hkv * chunks * 2 : 0;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < total;
         i += (int64_t)gridDim.x * blockDim.x) {
        int c = (int)(i % chunks);
        int64_t r = i / chunks;
        int kv = (int)(r & 1);
        r >>= 1;
        int g = (int)(r % sh.Hkv);
        int tok = (int)(r / sh.Hkv);
        int req = meta.tok_req[tok];
        int pos = meta.ctx_off[req] + (tok - meta.cu_q[req]);
        int64_t page = meta.block_table[meta.bt_off[req] + pos / sh.B];
        const uint4* src = (kv ? v_new : k_new) + ((int64_t)tok * sh.Hkv + g) * chunks + c;
        __nv_bfloat16* dst = cache + slab_elem_offset(page, kv, g, sh.Hkv, sh.B, sh.D) +
                             (int64_t)(pos % sh.B) * sh.D + c * 8;
        *reinterpret_cast<uint4*>(dst) = *src;
    }
}

// ---------------------------------------------------------------------------------
// N2: rotary position embedding fused into H2.
// rope_table_kernel runs once per cp_build_batch: cs[tok][i] = (cos, sin)(pos_tok * w_i), the angle
// and its cosine / sine in fp64 (an fp32 angle is off by 1e-2 rad at position 1e5), rounded to fp32.
// kv_append_rope_kernel then does, per layer, in one pass over the step's new rows: V rows copied to
// their page slots, K rows rotated on their way into the pages, Q rows rotated into `q_rot` (the Q the
// attention kernel reads).  Rotate-half pairing (include/cp.h); fp32 products and sums without fused
// multiply-add, round-to-nearest-even to bf16 -- the same decision oracle/rope.py takes.
// ---------------------------------------------------------------------------------
__global__ void rope_table_kernel(BatchMeta meta, int half, const double* __restrict__ inv_freq,
                                  float2* __restrict__ cs) {
    const int64_t total = (int64_t)meta.n_tokens * half;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < total;
         i += (int64_t)gridDim.x * blockDim.x) {
        const int tok = (int)(i / half), f = (int)(i % half);
        const int req = meta.tok_req[tok];
        const int pos = meta.ctx_off[req] + (tok - meta.cu_q[req]);
        double s, c;
        sincos((double)pos * inv_freq[f], &s, &c);
        cs[i] = make_float2((float)c, (float)s);
    }
}

__device__ __forceinline__ void rope_rotate8(const uint4& lo, const uint4& hi, const float2* __restrict__ cs,
                                             uint4& out_lo, uint4& out_hi) {
    const __nv_bfloat162* l2 = reinterpret_cast<const __nv_bfloat162*>(&lo);
    const __nv_bfloat162* h2 = reinterpret_cast<const __nv_bfloat162*>(&hi);
    __nv_bfloat162* ol = reinterpret_cast<__nv_bfloat162*>(&out_lo);
    __nv_bfloat162* oh = reinterpret_cast<__nv_bfloat162*>(&out_hi);
    const float4* cs4 = reinterpret_cast<const float4*>(cs);          // two (cos, sin) pairs per load
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const float4 t = cs4[j];
        const float2 a = __bfloat1622float2(l2[j]), b = __bfloat1622float2(h2[j]);
        const float lx = __fsub_rn(__fmul_rn(a.x, t.x), __fmul_rn(b.x, t.y));
        const float hx = __fadd_rn(__fmul_rn(b.x, t.x), __fmul_rn(a.x, t.y));
        const float ly = __fsub_rn(__fmul_rn(a.y, t.z), __fmul_rn(b.y, t.w));
        const float hy = __fadd_rn(__fmul_rn(b.y, t.z), __fmul_rn(a.y, t.w));
        ol[j] = __floats2bfloat162_rn(lx, ly);
        oh[j] = __floats2bfloat162_rn(hx, hy);
    }
}

// One thread per unit: a 16-byte chunk of a V row (copy), or the 16-byte chunk c of the lower half of a
// K / Q row together with chunk c of its upper half (rotate).
__global__ void kv_append_rope_kernel(BatchMeta meta, Shape sh, const uint4* __restrict__ q,
                                      const uint4* __restrict__ k_new, const uint4* __restrict__ v_new,
                                      const float2* __restrict__ cs, __nv_bfloat16* __restrict__ cache,
                                      uint4* __restrict__ q_rot) {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");   // the attention kernel may start its prologue
    zero_page_tails(meta, sh, cache);
    const int chunks = sh.D / 8, hc = sh.D / 16, half = sh.D / 2;
    const int v_units = sh.Hkv * chunks;
    const int per_tok = v_units + (sh.Hkv + sh.Hq) * hc;
    const int64_t total = (int64_t)meta.n_tokens * per_tok;
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < total;
         i += (int64_t)gridDim.x * blockDim.x) {
        const int tok = (int)(i / per_tok);
        int r = (int)(i % per_tok);
        const int req = meta.tok_req[tok];
        const int pos = meta.ctx_off[req] + (tok - meta.cu_q[req]);
        const int64_t page = meta.block_table[meta.bt_off[req] + pos / sh.B];
        if (r < v_units) {
            const int g = r / chunks, c = r % chunks;
            __nv_bfloat16* dst = cache + slab_elem_offset(page, 1, g, sh.Hkv, sh.B, sh.D) +
                                 (int64_t)(pos % sh.B) * sh.D + c * 8;
            *reinterpret_cast<uint4*>(dst) = v_new[((int64_t)tok * sh.Hkv + g) * chunks + c];
            continue;
        }
        r -= v_units;
        const int head = r / hc, c = r % hc;
        const float2* cs_row = cs + (int64_t)tok * half + c * 8;
        uint4 lo, hi, olo, ohi;
        if (head < sh.Hkv) {
            const uint4* src = k_new + ((int64_t)tok * sh.Hkv + head) * chunks;
            lo = src[c];
            hi = src[hc + c];
            rope_rotate8(lo, hi, cs_row, olo, ohi);
            uint4* dst = reinterpret_cast<uint4*>(cache + slab_elem_offset(page, 0, head, sh.Hkv, sh.B, sh.D) +
                                                  (int64_t)(pos % sh.B) * sh.D);
            dst[c] = olo;
            dst[hc + c] = ohi;
        } else {
            const int64_t row = ((int64_t)tok * sh.Hq + (head - sh.Hkv)) * chunks;
            lo = q[row + c];
            hi = q[row + hc + c];
            rope_rotate8(lo, hi, cs_row, olo, ohi);
            q_rot[row + c] = olo;
            q_rot[row + hc + c] = ohi;
        }
    }
}

// ---------------------------------------------------------------------------------
// N2, second half: FP8 (e4m3) KV pages.  Layout and quantisation rule: include/cp.h
// (cp_attention_step_fp8) / DESIGN.md R13-R15 / oracle/kv_fp8.py.
//
// kv_append_q8_kernel: 16 threads per (token, K|V, kv head) row of D = 128 elements, 8 elements each: row
// maximum by shuffles, e = the smallest integer with 448 * 2^e >= amax clamped to [-15, 7] -- integer
// arithmetic on the fp32 fields, the decision oracle/kv_fp8.py takes with frexp -- then x * 2^-e (exact) is
// rounded to nearest even onto the e4m3 grid, saturating (cvt.rn.satfinite.e4m3x2.f32).  Then the tails of the
// requests' last pages: codes 0, scales 1.
// ---------------------------------------------------------------------------------
__device__ __forceinline__ int64_t slab8_offset(int64_t page, int kv, int head, int Hkv, int B) {
    return ((page * 2 + kv) * Hkv + head) * (int64_t)B;           // in rows (tokens); x D for codes
}

__device__ __forceinline__ int e4m3_scale_exponent(float amax) {
    if (amax == 0.f) return -15;
    int k;                                                        // amax = f * 2^k, f in [0.5, 1)
    const float f = frexpf(amax, &k);
    const int e = (f <= 0.875f) ? k - 9 : k - 8;                  // 448 = 0.875 * 2^9
    return min(7, max(-15, e));
}

__device__ __forceinline__ uint32_t e4m3x4(float a, float b, float c, float d) {
    uint16_t lo, hi;
    asm("cvt.rn.satfinite.e4m3x2.f32 %0, %2, %1;" : "=h"(lo) : "f"(a), "f"(b));      // upper byte = first operand
    asm("cvt.rn.satfinite.e4m3x2.f32 %0, %2, %1;" : "=h"(hi) : "f"(c), "f"(d));
    return (uint32_t)lo | ((uint32_t)hi << 16);
}

__device__ __forceinline__ void zero_page_tails8(const BatchMeta& meta, const Shape& sh, uint8_t* __restrict__ cache8,
                                                 float* __restrict__ scales) {
    // one warp per (request, K|V, kv head) slab of the request's last page, as zero_page_tails
    const int lane = threadIdx.x & 31;
    const int64_t n_warps = (int64_t)gridDim.x * (blockDim.x >> 5);
    const int64_t total = (int64_t)meta.n_reqs * 2 * sh.Hkv;
    for (int64_t w = blockIdx.x * (int64_t)(blockDim.x >> 5) + (threadIdx.x >> 5); w < total; w += n_warps) {
        const int g = (int)(w % sh.Hkv);
        const int kv = (int)((w / sh.Hkv) & 1);
        const int req = (int)(w / (2 * sh.Hkv));
        const int last = meta.ctx_off[req] + meta.q_len[req] - 1;
        const int first_free = last % sh.B + 1;
        if (first_free >= sh.B) continue;
        const int64_t page = meta.block_table[meta.bt_off[req] + last / sh.B];
        const int64_t row0 = slab8_offset(page, kv, g, sh.Hkv, sh.B) + first_free;
        uint4* dst = reinterpret_cast<uint4*>(cache8 + row0 * sh.D);
        const int n16 = (sh.B - first_free) * sh.D / 16;
        for (int i = lane; i < n16; i += 32) dst[i] = make_uint4(0, 0, 0, 0);
        if (lane < sh.B - first_free) scales[row0 + lane] = 1.f;
    }
}

__global__ void kv_append_q8_kernel(BatchMeta meta, Shape sh, const uint4* __restrict__ k_new,
                                    const uint4* __restrict__ v_new, uint8_t* __restrict__ cache8,
                                    float* __restrict__ scales) {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    zero_page_tails8(meta, sh, cache8, scales);
    // D = 128: 16 threads x 8 elements per row; a warp holds two rows
    const int64_t total = k_new ? (int64_t)meta.n_tokens * sh.Hkv * 2 * 16 : 0;
    const int64_t total_pad = (total + 31) & ~(int64_t)31;       // whole warps take part in the shuffles
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < total_pad;
         i += (int64_t)gridDim.x * blockDim.x) {
        const bool live = i < total;
        const int c = (int)(i & 15);
        int64_t r = live ? i >> 4 : 0;
        const int kv = (int)(r & 1);
        r >>= 1;
        const int g = (int)(r % sh.Hkv);
        const int tok = (int)(r / sh.Hkv);
        const uint4 v = live ? (kv ? v_new : k_new)[((int64_t)tok * sh.Hkv + g) * 16 + c] : make_uint4(0, 0, 0, 0);
        const __nv_bfloat162* h2 = reinterpret_cast<const __nv_bfloat162*>(&v);
        float x[8];
#pragma unroll
        for (int j = 0; j < 4; ++j) { const float2 f = __bfloat1622float2(h2[j]); x[2 * j] = f.x; x[2 * j + 1] = f.y; }
        float amax = 0.f;
#pragma unroll
        for (int j = 0; j < 8; ++j) amax = fmaxf(amax, fabsf(x[j]));
#pragma unroll
        for (int o = 8; o > 0; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
        const int e = e4m3_scale_exponent(amax);
        const float inv = __int_as_float((127 - e) << 23);        // 2^-e, exact
        if (!live) continue;
        const int req = meta.tok_req[tok];
        const int pos = meta.ctx_off[req] + (tok - meta.cu_q[req]);
        const int64_t page = meta.block_table[meta.bt_off[req] + pos / sh.B];
        const int64_t row = slab8_offset(page, kv, g, sh.Hkv, sh.B) + pos % sh.B;
        uint2 out;
        out.x = e4m3x4(x[0] * inv, x[1] * inv, x[2] * inv, x[3] * inv);
        out.y = e4m3x4(x[4] * inv, x[5] * inv, x[6] * inv, x[7] * inv);
        *reinterpret_cast<uint2*>(cache8 + row * sh.D + c * 8) = out;
        if (c == 0) scales[row] = __int_as_float((127 + e) << 23);
    }
}

// kv8_dequant_kernel: the pages of every request that has a prefill chunk -> the bf16 scratch pool, page p of
// request j at scratch page scratch_base[j] + p, same slab layout as a bf16 pool.  code_value * 2^e is exact in
// bf16 (4 significant bits), so the chunk tiles then compute on exactly the values the fp8 pages hold.  One CTA
// per scratch page (grid-stride): the page's id is looked up ONCE per CTA (the first version did the four dependent
// index loads and two 64-bit divisions per 16-byte chunk: 72 us for the 324 MB of configs[2]; HBM time 50 us), then
// one thread per 16-byte chunk of codes, consecutive threads on consecutive chunks.  Unused slots of a last page
// were cleared by the append kernel (code 0).
__global__ void __launch_bounds__(256)
kv8_dequant_kernel(BatchMeta meta, Shape sh, const uint8_t* __restrict__ cache8,
                   const float* __restrict__ scales, __nv_bfloat16* __restrict__ scratch,
                   int32_t n_scratch_pages) {
    const int chunks = sh.D / 16;                                 // 16-byte chunks of codes per row
    const int per_page = 2 * sh.Hkv * sh.B * chunks;              // (kv, head, slot, chunk)
    __shared__ int64_t page_s;
    for (int sp = blockIdx.x; sp < n_scratch_pages; sp += gridDim.x) {
        __syncthreads();                                          // page_s of the previous page has been read
        if (threadIdx.x == 0) {
            const int req = meta.scratch_req[sp];
            page_s = meta.block_table[meta.bt_off[req] + (sp - meta.scratch_base[req])];
        }
        __syncthreads();
        const int64_t src_row0 = page_s * 2 * sh.Hkv * sh.B;
        const int64_t dst_row0 = (int64_t)sp * 2 * sh.Hkv * sh.B;
        for (int w = threadIdx.x; w < per_page; w += blockDim.x) {
            const int row_in_page = w / chunks, c = w % chunks;   // (kv * Hkv + head) * B + slot
            const uint4 codes = *reinterpret_cast<const uint4*>(cache8 + (src_row0 + row_in_page) * sh.D + c * 16);
            const float sc = scales[src_row0 + row_in_page];
            const uint16_t* c2 = reinterpret_cast<const uint16_t*>(&codes);
            uint4 o[2];
            __nv_bfloat162* ob = reinterpret_cast<__nv_bfloat162*>(o);
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                uint32_t h2;
                asm("cvt.rn.f16x2.e4m3x2 %0, %1;" : "=r"(h2) : "h"(c2[j]));
                const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&h2));
                ob[j] = __floats2bfloat162_rn(f.x * sc, f.y * sc);
            }
            uint4* dst = reinterpret_cast<uint4*>(scratch + (dst_row0 + row_in_page) * sh.D + c * 16);
            dst[0] = o[0];
            dst[1] = o[1];
        }
    }
}

#ifdef CP_DEBUG_VARIANTS
// ---------------------------------------------------------------------------------
// Cross-check attention (debug builds only, kernel_variant 1): CTA per work item, warp per row, lane owns D/32 dims.
// Scores are kept in log2 units (q pre-scaled by sm_scale * log2 e).
// ---------------------------------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(128)
attn_simt_kernel(BatchMeta meta, Shape sh, const __nv_bfloat16* __restrict__ q,
                 const __nv_bfloat16* __restrict__ cache, __nv_bfloat16* __restrict__ out,
                 float* __restrict__ part_o, float2* __restrict__ part_ml) {
    constexpr int EPL = D / 32;                           // elements per lane: 2 or 4
    const WorkItem it = meta.work[blockIdx.x];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const int G = sh.G;
    const int rows = it.q_tokens * G;
    const int tok0 = meta.cu_q[it.req] + it.q_start;
    const int ctx = meta.ctx_off[it.req];
    const int32_t* bt = meta.block_table + meta.bt_off[it.req];
    const float qscale = sh.sm_scale * 1.4426950408889634f;

    for (int r = warp; r < rows; r += nwarps) {
        const int tl = r / G, hg = r % G;
        const int tok = tok0 + tl;
        const int h = it.kv_head * G + hg;
        const int limit = min(it.kv_end, ctx + it.q_start + tl + 1);   // causal, diagonal inclusive
        float qv[EPL];
        {
            const __nv_bfloat16* qp = q + ((int64_t)tok * sh.Hq + h) * D + lane * EPL;
#pragma unroll
            for (int e = 0; e < EPL; e += 2) {
                float2 f = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(qp + e));
                qv[e] = f.x * qscale;
                qv[e + 1] = f.y * qscale;
            }
        }
        float m = -INFINITY, l = 0.f, acc[EPL];
#pragma unroll
        for (int e = 0; e < EPL; ++e) acc[e] = 0.f;

        for (int t = it.kv_begin; t < limit; ++t) {
            const int64_t page = bt[t / sh.B];
            const int slot = t % sh.B;
            const __nv_bfloat16* kp = cache + slab_elem_offset(page, 0, it.kv_head, sh.Hkv, sh.B, D) +
                                      (int64_t)slot * D + lane * EPL;
            const __nv_bfloat16* vp = kp + (int64_t)sh.Hkv * sh.B * D;     // V slab follows K slabs
            float s = 0.f, vv[EPL];
#pragma unroll
            for (int e = 0; e < EPL; e += 2) {
                float2 kf = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(kp + e));
                float2 vf = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(vp + e));
                s = fmaf(qv[e], kf.x, s);
                s = fmaf(qv[e + 1], kf.y, s);
                vv[e] = vf.x;
                vv[e + 1] = vf.y;
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
            const float m_new = fmaxf(m, s);
            const float alpha = exp2f(m - m_new);          // m = -inf -> 0
            const float p = exp2f(s - m_new);
            l = l * alpha + p;
#pragma unroll
            for (int e = 0; e < EPL; ++e) acc[e] = acc[e] * alpha + p * vv[e];
            m = m_new;
        }

        if (it.partial_row < 0) {
            const float inv = 1.f / l;
            __nv_bfloat16* op = out + ((int64_t)tok * sh.Hq + h) * D + lane * EPL;
#pragma unroll
            for (int e = 0; e < EPL; e += 2)
                *reinterpret_cast<__nv_bfloat162*>(op + e) =
                    __floats2bfloat162_rn(acc[e] * inv, acc[e + 1] * inv);
        } else {
            const int64_t pr = (int64_t)it.partial_row + r;
            float* po = part_o + pr * D + lane * EPL;
#pragma unroll
            for (int e = 0; e < EPL; ++e) po[e] = acc[e];
            if (lane == 0) part_ml[pr] = make_float2(m, l);
        }
    }
}

#endif  // CP_DEBUG_VARIANTS

// ---------------------------------------------------------------------------------
// H5: out = sum_s w_s O_s / sum_s w_s l_s, w_s = 2^(m_s - max m).  One warp per (token, head) row
// that has split partials: global warp gw finds its combine item by binary search over the items'
// row_base prefix sums (a grid of one block per item x 32 row slots was dominated by the launch of
// empty blocks).  The (m, l) pairs of up to 32 splits are read one per lane and the weights
// broadcast by shuffle, so the O_s loads of a row are independent and issue back to back.
// ---------------------------------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(128)
combine_kernel(BatchMeta meta, Shape sh, const float* __restrict__ part_o,
               const float2* __restrict__ part_ml, __nv_bfloat16* __restrict__ out) {
    constexpr int EPL = D / 32;
    asm volatile("griddepcontrol.wait;" ::: "memory");                  // the attention kernel's partials are visible
    const int lane = threadIdx.x & 31;
    const int gw = blockIdx.x * 4 + (threadIdx.x >> 5);
    int lo = 0, hi = meta.n_combine - 1;                  // last item with row_base <= w
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (meta.combine[mid].row_base <= gw) lo = mid; else hi = mid - 1;
    }
    const CombineItem it = meta.combine[lo];
    const int R = it.q_tokens * sh.G;
    const int r = gw - it.row_base;
    if (r >= R) return;                                   // past the last row
    const int64_t base = (int64_t)it.partial_row + r;
    float M = -INFINITY;
    for (int s0 = 0; s0 < it.n_splits; s0 += 32) {
        const int s = s0 + lane;
        float m = s < it.n_splits ? part_ml[base + (int64_t)s * R].x : -INFINITY;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
        M = fmaxf(M, m);
    }
    float L = 0.f, acc[EPL];
#pragma unroll
    for (int e = 0; e < EPL; ++e) acc[e] = 0.f;
    for (int s0 = 0; s0 < it.n_splits; s0 += 32) {
        const int s = s0 + lane;
        float w = 0.f, wl = 0.f;
        if (s < it.n_splits) {
            const float2 ml = part_ml[base + (int64_t)s * R];
            w = (ml.x == -INFINITY) ? 0.f : exp2f(ml.x - M);      // empty split: m = -inf -> w = 0
            wl = w * ml.y;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) wl += __shfl_xor_sync(0xffffffffu, wl, o);
        L += wl;
        const int ns = min(32, it.n_splits - s0);
#pragma unroll 4
        for (int j = 0; j < ns; ++j) {
            const float wj = __shfl_sync(0xffffffffu, w, j);
            const float* po = part_o + (base + (int64_t)(s0 + j) * R) * D + lane * EPL;
            if constexpr (EPL == 4) {
                const float4 v = *reinterpret_cast<const float4*>(po);
                acc[0] += wj * v.x; acc[1] += wj * v.y; acc[2] += wj * v.z; acc[3] += wj * v.w;
            } else {
                const float2 v = *reinterpret_cast<const float2*>(po);
                acc[0] += wj * v.x; acc[1] += wj * v.y;
            }
        }
    }
    const int tok = it.tok0 + r / sh.G;
    const int h = it.kv_head * sh.G + r % sh.G;
    const float inv = 1.f / L;
    __nv_bfloat16* op = out + ((int64_t)tok * sh.Hq + h) * D + lane * EPL;
#pragma unroll
    for (int e = 0; e < EPL; e += 2)
        *reinterpret_cast<__nv_bfloat162*>(op + e) =
            __floats2bfloat162_rn(acc[e] * inv, acc[e + 1] * inv);
}

}  // namespace cp
