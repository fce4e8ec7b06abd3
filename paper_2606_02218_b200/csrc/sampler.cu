// sampler.cu -- greedy / Philox-keyed Gumbel-max sampler (steps a3, a12).
//   Philox4x32-10, key = (seed lo, seed hi), counter = (v >> 2, t, sid, 0); word v & 3 is the
//   draw for vocab id v.  u = ((x >> 9) + 0.5) * 2^-23;  g = -log(-log u) (gumbel_from_u32, common.cuh);
//   token = argmax_v(logit_v * (1 / T) + g_v), lowest v on exact ties (reading C2).
#include "common.cuh"
#include "kernels.cuh"

namespace sagc {

__global__ void k_philox_debug(uint32_t k0, uint32_t k1, int sid, int t, int v0, int n, uint32_t* out) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int v = v0 + i;
    uint32_t w[4];
    philox4x32_10((uint32_t)v >> 2, (uint32_t)t, (uint32_t)sid, 0u, k0, k1, w);
    out[i] = w[v & 3];
}
int launch_philox_debug(uint64_t seed, int sid, int t, int v0, int n, uint32_t* out, cudaStream_t st) {
    if (n <= 0) return 0;
    k_philox_debug<<<(n + 255) / 256, 256, 0, st>>>((uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32), sid, t,
                                                    v0, n, out);
    return 1;
}

static constexpr int SMP_THREADS = 256;

__device__ __forceinline__ void better(float& bs, int& bi, float s, int i) {
    if (s > bs || (s == bs && i < bi)) { bs = s; bi = i; }
}

// grid = (rows, SMP_CHUNKS): each CTA scans one contiguous slice of the vocabulary and writes its
// best (score, index); the step-advance kernel takes the best of the SMP_CHUNKS partials in
// ascending chunk order (lowest index wins exact ties).
__global__ void __launch_bounds__(SMP_THREADS) k_sample(SampleArgs a) {
    __shared__ float ws[8];
    __shared__ int wi[8];
    trace_mark(24); pdl_wait(); trace_mark(25);
    pdl_launch();
    const int M = a.m_dev ? min(*a.m_dev, a.m_max) : a.m_max;
    const int row = blockIdx.x;
    if (row >= M) return;
    const float* lg = a.logits + (size_t)(row / a.row_div) * a.V;
    const int sid = a.row_sid[row];
    const int mode = (int)a.params[0];
    const float inv_t = 1.f / __uint_as_float(a.params[1]);
    const uint32_t k0 = a.params[2], k1 = a.params[3];
    const int t = *a.step_dev;
    float bs = -INFINITY;
    int bi = 0x7fffffff;
    const int nblk = (a.V + 3) >> 2;
    const int per = (nblk + SMP_CHUNKS - 1) / SMP_CHUNKS;
    const int b_lo = blockIdx.y * per, b_hi = min(nblk, b_lo + per);
    for (int b = b_lo + threadIdx.x; b < b_hi; b += SMP_THREADS) {
        const int v = b << 2;
        float s[4];
        if (v + 3 < a.V) {
            float4 x = __ldcs(reinterpret_cast<const float4*>(lg + v));
            s[0] = x.x; s[1] = x.y; s[2] = x.z; s[3] = x.w;
        } else {
#pragma unroll
            for (int e = 0; e < 4; ++e) s[e] = (v + e < a.V) ? lg[v + e] : -INFINITY;
        }
        if (mode == 1) {
            uint32_t w[4];
            philox4x32_10((uint32_t)b, (uint32_t)t, (uint32_t)sid, 0u, k0, k1, w);
#pragma unroll
            for (int e = 0; e < 4; ++e) s[e] = fmaf(s[e], inv_t, gumbel_from_u32(w[e]));
        }
#pragma unroll
        for (int e = 0; e < 4; ++e)
            if (v + e < a.V) better(bs, bi, s[e], v + e);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        float s2 = __shfl_xor_sync(0xffffffffu, bs, o);
        int i2 = __shfl_xor_sync(0xffffffffu, bi, o);
        better(bs, bi, s2, i2);
    }
    if ((threadIdx.x & 31) == 0) { ws[threadIdx.x >> 5] = bs; wi[threadIdx.x >> 5] = bi; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w2 = 1; w2 < SMP_THREADS / 32; ++w2) better(bs, bi, ws[w2], wi[w2]);
        a.part_score[row * SMP_CHUNKS + blockIdx.y] = bs;
        a.part_tok[row * SMP_CHUNKS + blockIdx.y] = bi;
    }
}

int launch_sample(const SampleArgs& a, cudaStream_t st) {
    if (a.m_max <= 0) return 0;
    launch_pdl(k_sample, dim3(a.m_max, SMP_CHUNKS), dim3(SMP_THREADS), 0, st, g_pdl_all, a);
    return 1;
}

// grid = n_dump; entry e = (sid, t): if t == *step, find the slot holding sid and copy its row.
__global__ void k_dump_logits(const int* __restrict__ dump_sid_t, const int* step_dev, const int* __restrict__ live,
                              const int* n_live, int row_div, const float* __restrict__ logits, int V,
                              float* __restrict__ out) {
    __shared__ int slot_s;
    const int e = blockIdx.x;
    const int sid = dump_sid_t[2 * e], t = dump_sid_t[2 * e + 1];
    if (t != *step_dev) return;
    if (threadIdx.x == 0) slot_s = -1;
    __syncthreads();
    const int n = *n_live;
    for (int i = threadIdx.x; i < n; i += blockDim.x)
        if (live[i] == sid) slot_s = i;
    __syncthreads();
    const int slot = slot_s;
    if (slot < 0) return;
    const float* src = logits + (size_t)(slot / row_div) * V;
    float* dst = out + (size_t)e * V;
    for (int v = threadIdx.x; v < V; v += blockDim.x) dst[v] = src[v];
}
int launch_dump_logits(const int* dump_sid_t, int n_dump, const int* step_dev, const int* live, const int* n_live,
                       int row_div, const float* logits, int V, float* out, cudaStream_t st) {
    if (n_dump <= 0) return 0;
    k_dump_logits<<<n_dump, 256, 0, st>>>(dump_sid_t, step_dev, live, n_live, row_div, logits, V, out);
    return 1;
}

// ---- teacher-forced log-prob pass (row f4) ------------------------------------------------------------------
// Row descriptors: sequence sid = prompt tokens of its group followed by its own generated tokens but the last;
// rows of all sequences are concatenated (seq_off).  row r of sid at offset j: pos = j, ctx = j + 1.
__global__ void k_score_rows(const int* __restrict__ prompt_tokens, const int* __restrict__ prompt_offs, const int* __restrict__ seq_off,
                             const int* __restrict__ gen_tokens, int nseq, int G, int max_new, int total, int* row_sid, int* row_pos,
                             int* row_ctx, int* row_tok) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= total) return;
    int lo = 0, hi = nseq;               // largest sid with seq_off[sid] <= r
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (seq_off[mid] <= r) lo = mid; else hi = mid;
    }
    const int sid = lo, j = r - seq_off[sid], p = sid / G;
    const int P = prompt_offs[p + 1] - prompt_offs[p];
    row_sid[r] = sid; row_pos[r] = j; row_ctx[r] = j + 1;
    row_tok[r] = j < P ? prompt_tokens[prompt_offs[p] + j] : gen_tokens[(size_t)sid * max_new + (j - P)];
}
int launch_score_rows(const int* prompt_tokens, const int* prompt_offs_dev, const int* seq_off_dev, const int* gen_tokens, int nseq,
                      int G, int max_new, int total, int* row_sid, int* row_pos, int* row_ctx, int* row_tok, cudaStream_t st) {
    if (total <= 0) return 0;
    k_score_rows<<<(total + 255) / 256, 256, 0, st>>>(prompt_tokens, prompt_offs_dev, seq_off_dev, gen_tokens, nseq, G, max_new, total,
                                                      row_sid, row_pos, row_ctx, row_tok);
    return 1;
}

// log pi(y_t | x, y_<t) = logit[y_t] - logsumexp(logits) for every row that predicts a generated token:
// row (sid, pos) with pos >= P - 1 predicts token t = pos - (P - 1) (0-based).  One CTA per row; fp32, max-subtracted.
__global__ void __launch_bounds__(256) k_token_logprob(const float* __restrict__ logits, int V, const int* __restrict__ row_sid,
                                                        const int* __restrict__ row_pos, const int* __restrict__ prompt_offs, int G,
                                                        const int* __restrict__ gen_tokens, int max_new, float* __restrict__ out) {
    __shared__ float red[8];
    const int r = blockIdx.x;
    const int sid = row_sid[r], pos = row_pos[r], p = sid / G;
    const int P = prompt_offs[p + 1] - prompt_offs[p];
    if (pos < P - 1) return;
    const int t = pos - (P - 1);
    const float* lg = logits + (size_t)r * V;
    float mx = -INFINITY;
    for (int v = threadIdx.x; v < V; v += 256) mx = fmaxf(mx, lg[v]);
    mx = warp_max(mx);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = mx;
    __syncthreads();
    mx = red[0];
    for (int i = 1; i < 8; ++i) mx = fmaxf(mx, red[i]);
    __syncthreads();
    float sum = 0.f;
    for (int v = threadIdx.x; v < V; v += 256) sum += __expf(lg[v] - mx);
    sum = warp_sum(sum);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = sum;
    __syncthreads();
    if (threadIdx.x == 0) {
        float tot = 0.f;
        for (int i = 0; i < 8; ++i) tot += red[i];
        const int tok = gen_tokens[(size_t)sid * max_new + t];
        out[(size_t)sid * max_new + t] = lg[tok] - mx - logf(tot);
    }
}
int launch_token_logprob(const float* logits, int V, int rows, const int* row_sid, const int* row_pos, const int* prompt_offs_dev, int G,
                         const int* gen_tokens, int max_new, float* out, cudaStream_t st) {
    if (rows <= 0) return 0;
    k_token_logprob<<<rows, 256, 0, st>>>(logits, V, row_sid, row_pos, prompt_offs_dev, G, gen_tokens, max_new, out);
    return 1;
}

}  // namespace sagc
