// elementwise.cu -- embedding gather, RoPE + bf16 KV append, row gathers (steps a5, a6).
#include "common.cuh"
#include "kernels.cuh"

namespace sagc {

// x[row][:] = embed[tok[row]][:] widened to fp32.  One CTA per row, 8 elements per thread-iteration.
__global__ void __launch_bounds__(128) k_embed(const bf16_t* __restrict__ embed, const int* __restrict__ tok,
                                               const int* m_dev, int m_max, int d, float* __restrict__ x) {
    trace_mark(0); pdl_wait(); trace_mark(1);
    pdl_launch();
    const int M = m_dev ? min(*m_dev, m_max) : m_max;
    const int row = blockIdx.x;
    if (row >= M) return;
    const bf16_t* src = embed + (size_t)tok[row] * d;
    float* dst = x + (size_t)row * d;
    for (int k = threadIdx.x * 8; k < d; k += blockDim.x * 8) {
        uint4 w = *reinterpret_cast<const uint4*>(src + k);
        float4 a = make_float4(bf16lo_to_f32(w.x), bf16hi_to_f32(w.x), bf16lo_to_f32(w.y), bf16hi_to_f32(w.y));
        float4 b = make_float4(bf16lo_to_f32(w.z), bf16hi_to_f32(w.z), bf16lo_to_f32(w.w), bf16hi_to_f32(w.w));
        *reinterpret_cast<float4*>(dst + k) = a;
        *reinterpret_cast<float4*>(dst + k + 4) = b;
    }
}

int launch_embed(const bf16_t* embed, const int* tok, const int* m_dev, int m_max, int d, float* x,
                 cudaStream_t st) {
    if (m_max <= 0) return 0;
    launch_pdl(k_embed, dim3(m_max), dim3(128), 0, st, g_pdl_all, embed, tok, m_dev, m_max, d, x);
    return 1;
}

// RoPE (rotate-half: pairs (i, i+hd/2), table cos/sin from fp64 angles) on the q and k heads of
// one activation row; q is rotated in place (fp32); k (rotated) and v are rounded to bf16 (RNE)
// and written to slot pos%page of page page_table[sid][pos/page] -- the ONLY rounding point of
// the forward pass (reading C1).  grid = (rows, Hq+2*Hkv heads), block = hd/2 threads.
__global__ void k_rope_append(RopeArgs a) {
    trace_mark(8);
    // Positions, the live count, the page table and the RoPE table were written by EARLIER steps (or are
    // constants): fetch them before the dependency wait so that only the q/k/v loads remain after it.
    const int M = a.m_dev ? min(*a.m_dev, a.m_max) : a.m_max;
    const int row = blockIdx.x;
    const int head = blockIdx.y;
    const int half = a.hd >> 1;
    const int i = threadIdx.x;
    const bool live = row < M && i < half;
    int pos = 0, pg = -1;
    float2 cs = make_float2(1.f, 0.f);
    if (live) {
        pos = a.row_pos[row];
        if (head < a.Hq + a.Hkv) cs = *reinterpret_cast<const float2*>(a.rope_cs + ((size_t)pos * half + i) * 2);
        if (head >= a.Hq) pg = a.page_table[(size_t)a.row_sid[row] * a.max_blocks + pos / a.page];
    }
    pdl_wait();
    trace_mark(9);
    pdl_launch();
    if (!live) return;
    const int ld = (a.Hq + 2 * a.Hkv) * a.hd;
    float* hp = a.qkv + (size_t)row * ld + (size_t)head * a.hd;
    float x0 = hp[i], x1 = hp[i + half];
    if (head < a.Hq + a.Hkv) {
        float r0 = x0 * cs.x - x1 * cs.y;
        float r1 = x1 * cs.x + x0 * cs.y;
        x0 = r0; x1 = r1;
    }
    if (head < a.Hq) {
        hp[i] = x0; hp[i + half] = x1;
        return;
    }
    if (pg < 0) return;   // unmapped (only after a pool-exhaustion error)
    const int isv = head >= a.Hq + a.Hkv;
    const int kvh = head - a.Hq - (isv ? a.Hkv : 0);
    bf16_t* dst = a.kv_layer + (((size_t)pg * 2 + isv) * a.Hkv + kvh) * (size_t)a.page * a.hd +
                  (size_t)(pos % a.page) * a.hd;
    dst[i] = (bf16_t)f32_to_bf16_bits(x0);
    dst[i + half] = (bf16_t)f32_to_bf16_bits(x1);
}

int launch_rope_append(const RopeArgs& a, cudaStream_t st) {
    if (a.m_max <= 0) return 0;
    dim3 grid(a.m_max, a.Hq + 2 * a.Hkv);
    launch_pdl(k_rope_append, grid, dim3(a.hd / 2), 0, st, g_pdl_all, a);
    return 1;
}

// out[i][:] = x[row_idx[i]][:]
__global__ void k_gather_rows(const float* __restrict__ x, const int* __restrict__ row_idx, int d,
                              float* __restrict__ out) {
    const float* src = x + (size_t)row_idx[blockIdx.x] * d;
    float* dst = out + (size_t)blockIdx.x * d;
    for (int k = threadIdx.x; k < d; k += blockDim.x) dst[k] = src[k];
}
int launch_gather_rows(const float* x, const int* row_idx, int n, int d, float* out, cudaStream_t st) {
    if (n <= 0) return 0;
    k_gather_rows<<<n, 256, 0, st>>>(x, row_idx, d, out);
    return 1;
}

// Prefill row descriptors: row r of prompt p at offset j: sid = p*G (the group's first
// completion owns the prefill writes), pos = j, ctx = j + 1, tok = prompt token.
__global__ void k_prefill_rows(const int* __restrict__ prompt_tokens, const int* __restrict__ offs, int n_prompts,
                               int G, int total, int* row_sid, int* row_pos, int* row_ctx, int* row_tok) {
    int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= total) return;
    int lo = 0, hi = n_prompts;          // largest p with offs[p] <= r
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (offs[mid] <= r) lo = mid; else hi = mid;
    }
    int j = r - offs[lo];
    row_sid[r] = lo * G;
    row_pos[r] = j;
    row_ctx[r] = j + 1;
    row_tok[r] = prompt_tokens[r];
}
int launch_prefill_rows(const int* prompt_tokens, const int* prompt_offsets_dev, int n_prompts, int G,
                        int total_rows, int* row_sid, int* row_pos, int* row_ctx, int* row_tok,
                        cudaStream_t st) {
    if (total_rows <= 0) return 0;
    k_prefill_rows<<<(total_rows + 255) / 256, 256, 0, st>>>(prompt_tokens, prompt_offsets_dev, n_prompts, G,
                                                             total_rows, row_sid, row_pos, row_ctx, row_tok);
    return 1;
}

// tcgen05 variant of the embedding step: besides the fp32 residual row it writes the pre-split
// operand rows of the first RMSNorm (x * w_norm as hi / lo bf16) and the row's sum of squares
// (tile 0 of the partial-sum buffer; the other tiles are zeroed).
__global__ void __launch_bounds__(256) k_embed_split(const bf16_t* __restrict__ embed, const int* __restrict__ tok,
                                                     const int* m_dev, int m_max, int d, float* __restrict__ x,
                                                     const bf16_t* __restrict__ norm_w, bf16_t* __restrict__ xs,
                                                     float* __restrict__ ssq, int ssq_ld, int ssq_tiles) {
    __shared__ float red[8];
    trace_mark(4); pdl_wait(); trace_mark(5);
    pdl_launch();
    const int M = m_dev ? min(*m_dev, m_max) : m_max;
    const int row = blockIdx.x;
    if (row >= M) return;
    const bf16_t* src = embed + (size_t)tok[row] * d;
    float acc = 0.f;
    for (int k = threadIdx.x; k < d; k += blockDim.x) {
        const float v = bf16_to_f32(src[k]);
        x[(size_t)row * d + k] = v;
        acc += v * v;
        const float xw = v * bf16_to_f32(norm_w[k]);
        const uint32_t hi = f32_to_bf16_bits(xw);
        xs[(size_t)(2 * row) * d + k] = (bf16_t)hi;
        xs[(size_t)(2 * row + 1) * d + k] = (bf16_t)f32_to_bf16_bits(xw - __uint_as_float(hi << 16));
    }
    acc = warp_sum(acc);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        float t = 0.f;
        for (int i = 0; i < 8; ++i) t += red[i];
        ssq[row] = t;
        for (int i = 1; i < ssq_tiles; ++i) ssq[(size_t)i * ssq_ld + row] = 0.f;
    }
}
int launch_embed_split(const bf16_t* embed, const int* tok, const int* m_dev, int m_max, int d, float* x,
                       const bf16_t* norm_w, bf16_t* xs, float* ssq, int ssq_ld, int ssq_tiles, cudaStream_t st) {
    if (m_max <= 0) return 0;
    launch_pdl(k_embed_split, dim3(m_max), dim3(256), 0, st, g_pdl_all, embed, tok, m_dev, m_max, d, x, norm_w, xs, ssq, ssq_ld, ssq_tiles);
    return 1;
}

}  // namespace sagc
