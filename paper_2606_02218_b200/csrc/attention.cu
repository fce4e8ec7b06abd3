// attention.cu -- paged GQA decode attention over ragged contexts (step a7).
//
// One CTA per (activation row, kv head, K-split).  The r = Hq/Hkv query heads that share a kv
// head are processed together so every K/V byte is read once per (row, kv head).  Contexts are
// walked through the page table in tiles of 128 tokens:
//   phase 1  thread = token: s[h] = q[h] . k  for the r heads (q pre-scaled, fp32, smem broadcast)
//   softmax  online (running max / sum per head), warp-shuffle reductions, probabilities in smem
//   phase 2  thread = (token group, 4 head-dim columns): o[h][:] += p[h][tok] * v[tok][:]
// Split-K: split s covers tokens [s*cps, (s+1)*cps); partial (o, max, sum) go to scratch and the
// last CTA to arrive for a (row, kv head) merges them with the log-sum-exp rule.
// The same kernel serves prefill: every prompt position is a row with ctx = position + 1.
#include "common.cuh"
#include "kernels.cuh"

namespace sagc {

static constexpr int ATT_THREADS = 128;
static constexpr int ATT_TILE = 128;
static constexpr int ATT_MAXR = 8;

template <int HD>
__global__ void __launch_bounds__(ATT_THREADS) k_attention(AttnArgs a) {
    constexpr int LPR = HD / 4;                 // lanes per V row in phase 2
    constexpr int NG = ATT_THREADS / LPR;       // token groups in phase 2
    __shared__ __align__(16) float q_s[ATT_MAXR][HD];
    __shared__ __align__(16) float s_s[ATT_MAXR][ATT_TILE];
    __shared__ float m_s[ATT_MAXR], l_s[ATT_MAXR], sc_s[ATT_MAXR];
    __shared__ __align__(16) float red_s[NG][ATT_MAXR][HD + 4];
    __shared__ int last_s;

    pdl_wait();
    pdl_launch();
    const int M = a.m_dev ? min(*a.m_dev, a.m_max) : a.m_max;
    const int row = blockIdx.x, kvh = blockIdx.y, split = blockIdx.z;
    if (row >= M) return;
    const int r = a.Hq / a.Hkv;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int ctx = a.row_ctx[row];
    const int sid = a.row_sid[row];
    const int* pt = a.page_table + (size_t)sid * a.max_blocks;
    const int nsp = a.n_splits;
    int cps = (ctx + nsp - 1) / nsp;
    cps = ((cps + ATT_TILE - 1) / ATT_TILE) * ATT_TILE;
    const int t_begin = split * cps;
    const int t_end = min(ctx, t_begin + cps);
    const float scale = rsqrtf((float)HD);

    for (int i = tid; i < r * HD; i += ATT_THREADS) {
        int h = i / HD, d = i % HD;
        q_s[h][d] = a.q[(size_t)row * a.ldq + (size_t)(kvh * r + h) * HD + d] * scale;
    }
    if (tid < ATT_MAXR) { m_s[tid] = -INFINITY; l_s[tid] = 0.f; }
    float acc[ATT_MAXR][4];
#pragma unroll
    for (int h = 0; h < ATT_MAXR; ++h)
#pragma unroll
        for (int e = 0; e < 4; ++e) acc[h][e] = 0.f;
    __syncthreads();

    const size_t head_stride = (size_t)a.page * HD;                 // one (page, K|V, kv head) slab
    const int tg = tid / LPR, dl = tid % LPR;

    for (int t0 = t_begin; t0 < t_end; t0 += ATT_TILE) {
        // ---- phase 1: scores --------------------------------------------------------
        {
            const int tok = t0 + tid;
            float s[ATT_MAXR];
#pragma unroll
            for (int h = 0; h < ATT_MAXR; ++h) s[h] = 0.f;
            if (tok < t_end) {
                const int pg = pt[tok / a.page];
                const bf16_t* kp = a.kv_layer + ((size_t)pg * 2 * a.Hkv + kvh) * head_stride +
                                   (size_t)(tok % a.page) * HD;
#pragma unroll 4
                for (int d = 0; d < HD; d += 8) {
                    uint4 w = *reinterpret_cast<const uint4*>(kp + d);
                    float k0 = bf16lo_to_f32(w.x), k1 = bf16hi_to_f32(w.x), k2 = bf16lo_to_f32(w.y),
                          k3 = bf16hi_to_f32(w.y), k4 = bf16lo_to_f32(w.z), k5 = bf16hi_to_f32(w.z),
                          k6 = bf16lo_to_f32(w.w), k7 = bf16hi_to_f32(w.w);
#pragma unroll
                    for (int h = 0; h < ATT_MAXR; ++h) {
                        if (h < r) {
                            float4 qa = *reinterpret_cast<const float4*>(&q_s[h][d]);
                            float4 qb = *reinterpret_cast<const float4*>(&q_s[h][d + 4]);
                            float t = s[h];
                            t = fmaf(qa.x, k0, t); t = fmaf(qa.y, k1, t); t = fmaf(qa.z, k2, t); t = fmaf(qa.w, k3, t);
                            t = fmaf(qb.x, k4, t); t = fmaf(qb.y, k5, t); t = fmaf(qb.z, k6, t); t = fmaf(qb.w, k7, t);
                            s[h] = t;
                        }
                    }
                }
            }
#pragma unroll
            for (int h = 0; h < ATT_MAXR; ++h)
                if (h < r) s_s[h][tid] = (tok < t_end) ? s[h] : -INFINITY;
        }
        __syncthreads();
        // ---- online softmax: warp w owns heads w, w+4 ----------------------------------
        for (int h = warp; h < r; h += 4) {
            float4 v = *reinterpret_cast<const float4*>(&s_s[h][lane * 4]);
            float tmax = warp_max(fmaxf(fmaxf(v.x, v.y), fmaxf(v.z, v.w)));
            const float m_old = m_s[h];
            const float m_new = fmaxf(m_old, tmax);
            v.x = __expf(v.x - m_new); v.y = __expf(v.y - m_new);
            v.z = __expf(v.z - m_new); v.w = __expf(v.w - m_new);
            *reinterpret_cast<float4*>(&s_s[h][lane * 4]) = v;
            const float lsum = warp_sum(v.x + v.y + v.z + v.w);
            if (lane == 0) {
                const float f = __expf(m_old - m_new);      // exp(-inf) = 0 on the first tile
                sc_s[h] = f;
                l_s[h] = l_s[h] * f + lsum;
                m_s[h] = m_new;
            }
        }
        __syncthreads();
        // ---- phase 2: o += p . V -----------------------------------------------------
#pragma unroll
        for (int h = 0; h < ATT_MAXR; ++h) {
            if (h < r) {
                const float f = sc_s[h];
#pragma unroll
                for (int e = 0; e < 4; ++e) acc[h][e] *= f;
            }
        }
        const int n_tok = min(ATT_TILE, t_end - t0);
#pragma unroll 2
        for (int j = tg; j < n_tok; j += NG) {
            const int tok = t0 + j;
            const int pg = pt[tok / a.page];
            const bf16_t* vp = a.kv_layer + (((size_t)pg * 2 + 1) * a.Hkv + kvh) * head_stride +
                               (size_t)(tok % a.page) * HD + dl * 4;
            uint2 w = *reinterpret_cast<const uint2*>(vp);
            const float v0 = bf16lo_to_f32(w.x), v1 = bf16hi_to_f32(w.x), v2 = bf16lo_to_f32(w.y),
                        v3 = bf16hi_to_f32(w.y);
#pragma unroll
            for (int h = 0; h < ATT_MAXR; ++h) {
                if (h < r) {
                    const float p = s_s[h][j];
                    acc[h][0] = fmaf(p, v0, acc[h][0]); acc[h][1] = fmaf(p, v1, acc[h][1]);
                    acc[h][2] = fmaf(p, v2, acc[h][2]); acc[h][3] = fmaf(p, v3, acc[h][3]);
                }
            }
        }
        __syncthreads();
    }

    // ---- reduce the NG token groups (fixed order) -----------------------------------------
#pragma unroll
    for (int h = 0; h < ATT_MAXR; ++h)
        if (h < r) *reinterpret_cast<float4*>(&red_s[tg][h][dl * 4]) = make_float4(acc[h][0], acc[h][1], acc[h][2], acc[h][3]);
    __syncthreads();
    for (int i = tid; i < r * HD; i += ATT_THREADS) {
        const int h = i / HD, d = i % HD;
        float o = 0.f;
#pragma unroll
        for (int g2 = 0; g2 < NG; ++g2) o += red_s[g2][h][d];
        const int hq = kvh * r + h;
        if (nsp == 1) {
            a.out[(size_t)row * a.Hq * HD + (size_t)hq * HD + d] = o / l_s[h];
        } else {
            a.part_o[(((size_t)row * a.Hq + hq) * nsp + split) * HD + d] = o;
        }
    }
    if (nsp == 1) return;
    if (tid < r) {
        const int hq = kvh * r + tid;
        float* ml = a.part_ml + (((size_t)row * a.Hq + hq) * nsp + split) * 2;
        ml[0] = m_s[tid];
        ml[1] = l_s[tid];
    }
    __threadfence();
    __syncthreads();
    if (tid == 0) {
        int prev = atomicAdd(&a.counters[row * a.Hkv + kvh], 1);
        last_s = (prev == nsp - 1);
    }
    __syncthreads();
    if (!last_s) return;
    __threadfence();
    // ---- merge: this CTA arrived last for (row, kvh) -----------------------------------------
    for (int i = tid; i < r * HD; i += ATT_THREADS) {
        const int h = i / HD, d = i % HD;
        const int hq = kvh * r + h;
        const float* ml = a.part_ml + ((size_t)row * a.Hq + hq) * nsp * 2;
        float mx = -INFINITY;
        for (int s2 = 0; s2 < nsp; ++s2) mx = fmaxf(mx, __ldcg(ml + 2 * s2));
        float num = 0.f, den = 0.f;
        for (int s2 = 0; s2 < nsp; ++s2) {
            const float l2 = __ldcg(ml + 2 * s2 + 1);
            if (l2 > 0.f) {
                const float f = __expf(__ldcg(ml + 2 * s2) - mx);
                num += f * __ldcg(a.part_o + (((size_t)row * a.Hq + hq) * nsp + s2) * HD + d);
                den += f * l2;
            }
        }
        a.out[(size_t)row * a.Hq * HD + (size_t)hq * HD + d] = num / den;
    }
    if (tid == 0) a.counters[row * a.Hkv + kvh] = 0;
}

int launch_attention(const AttnArgs& a, cudaStream_t st) {
    if (a.m_max <= 0) return 0;
    dim3 grid(a.m_max, a.Hkv, a.n_splits);
    if (a.hd == 128) k_attention<128><<<grid, ATT_THREADS, 0, st>>>(a);
    else if (a.hd == 64) k_attention<64><<<grid, ATT_THREADS, 0, st>>>(a);
    else if (a.hd == 32) k_attention<32><<<grid, ATT_THREADS, 0, st>>>(a);
    else return -1;
    return 1;
}

}  // namespace sagc
