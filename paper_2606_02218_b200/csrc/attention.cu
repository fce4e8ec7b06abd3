// attention.cu -- paged GQA decode attention over ragged contexts (step a7).
//
// One CTA per (activation row, kv head, K-split).  The r = Hq/Hkv query heads that share a kv
// head are processed together so every K/V byte is read once per (row, kv head).  Contexts are
// walked through the page table in tiles of 64 tokens, staged in shared memory by a 3-stage
// cp.async pipeline (K and V rows, padded so that per-token 16-byte reads are conflict-free):
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
static constexpr int ATT_TILE = 64;          // tokens per pipeline stage
static constexpr int ATT_STAGES = 3;
static constexpr int ATT_MAXR = 8;

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc, int src_bytes) {
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(d), "l"(gsrc), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

template <int HD>
struct AttSmem {
    static constexpr int ROWB = HD * 2 + 16;                  // padded row: conflict-free LDS.128 by token
    static constexpr int STAGE = 2 * ATT_TILE * ROWB;         // K rows then V rows
    static constexpr int BYTES = ATT_STAGES * STAGE;
};

template <int HD>
__global__ void __launch_bounds__(ATT_THREADS) k_attention(AttnArgs a) {
    constexpr int LPR = HD / 4;                 // lanes per V row in phase 2
    constexpr int NG = ATT_THREADS / LPR;       // token groups in phase 2
    constexpr int ROWB = AttSmem<HD>::ROWB;
    constexpr int CPR = HD * 2 / 16;            // 16-byte chunks per row
    extern __shared__ __align__(16) unsigned char kv_s[];
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
    const int n_tiles = t_end > t_begin ? (t_end - t_begin + ATT_TILE - 1) / ATT_TILE : 0;
    const float scale = rsqrtf((float)HD);
    const size_t head_stride = (size_t)a.page * HD;                 // one (page, K|V, kv head) slab

    // async copy of one tile (K and V rows of 64 tokens) into a stage; rows past t_end are zero-filled
    auto load_tile = [&](int tile, int stage) {
        unsigned char* base = kv_s + (size_t)stage * AttSmem<HD>::STAGE;
        const int t0 = t_begin + tile * ATT_TILE;
#pragma unroll
        for (int c = tid; c < ATT_TILE * CPR; c += ATT_THREADS) {
            const int j = c / CPR, part = c % CPR;
            const int tok = t0 + j;
            const bool ok = tok < t_end;
            const int pg = ok ? pt[tok / a.page] : 0;
            const bf16_t* kp = a.kv_layer + ((size_t)pg * 2 * a.Hkv + kvh) * head_stride +
                               (size_t)(ok ? tok % a.page : 0) * HD + part * 8;
            const bf16_t* vp = kp + (size_t)a.Hkv * head_stride;
            cp_async16(base + (size_t)j * ROWB + part * 16, kp, ok ? 16 : 0);
            cp_async16(base + (size_t)(ATT_TILE + j) * ROWB + part * 16, vp, ok ? 16 : 0);
        }
    };
    if (n_tiles > 0) load_tile(0, 0);
    cp_async_commit();
    if (n_tiles > 1) load_tile(1, 1);
    cp_async_commit();

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

    const int tg = tid / LPR, dl = tid % LPR;
    // phase-1 mapping: token = tid % 64, heads h = (tid / 64), +2, +4, ...
    const int p1_tok = tid & (ATT_TILE - 1), p1_h0 = tid / ATT_TILE;

    for (int tile = 0; tile < n_tiles; ++tile) {
        cp_async_wait<1>();
        __syncthreads();                         // tile landed; previous tile's stage is free
        if (tile + 2 < n_tiles) load_tile(tile + 2, (tile + 2) % ATT_STAGES);
        cp_async_commit();
        const unsigned char* base = kv_s + (size_t)(tile % ATT_STAGES) * AttSmem<HD>::STAGE;
        const int t0 = t_begin + tile * ATT_TILE;
        // ---- phase 1: scores --------------------------------------------------------
        {
            float s[ATT_MAXR / 2];
#pragma unroll
            for (int hh = 0; hh < ATT_MAXR / 2; ++hh) s[hh] = 0.f;
            const unsigned char* kp = base + (size_t)p1_tok * ROWB;
#pragma unroll 4
            for (int d = 0; d < HD; d += 8) {
                uint4 w = *reinterpret_cast<const uint4*>(kp + d * 2);
                float k0 = bf16lo_to_f32(w.x), k1 = bf16hi_to_f32(w.x), k2 = bf16lo_to_f32(w.y),
                      k3 = bf16hi_to_f32(w.y), k4 = bf16lo_to_f32(w.z), k5 = bf16hi_to_f32(w.z),
                      k6 = bf16lo_to_f32(w.w), k7 = bf16hi_to_f32(w.w);
#pragma unroll
                for (int hh = 0; hh < ATT_MAXR / 2; ++hh) {
                    const int h = p1_h0 + 2 * hh;
                    if (h < r) {
                        float4 qa = *reinterpret_cast<const float4*>(&q_s[h][d]);
                        float4 qb = *reinterpret_cast<const float4*>(&q_s[h][d + 4]);
                        float t = s[hh];
                        t = fmaf(qa.x, k0, t); t = fmaf(qa.y, k1, t); t = fmaf(qa.z, k2, t); t = fmaf(qa.w, k3, t);
                        t = fmaf(qb.x, k4, t); t = fmaf(qb.y, k5, t); t = fmaf(qb.z, k6, t); t = fmaf(qb.w, k7, t);
                        s[hh] = t;
                    }
                }
            }
#pragma unroll
            for (int hh = 0; hh < ATT_MAXR / 2; ++hh) {
                const int h = p1_h0 + 2 * hh;
                if (h < r) s_s[h][p1_tok] = (t0 + p1_tok < t_end) ? s[hh] : -INFINITY;
            }
        }
        __syncthreads();
        // ---- online softmax: warp w owns heads w, w+4 ----------------------------------
        for (int h = warp; h < r; h += 4) {
            float2 v = *reinterpret_cast<const float2*>(&s_s[h][lane * 2]);
            float tmax = warp_max(fmaxf(v.x, v.y));
            const float m_old = m_s[h];
            const float m_new = fmaxf(m_old, tmax);
            v.x = __expf(v.x - m_new); v.y = __expf(v.y - m_new);
            *reinterpret_cast<float2*>(&s_s[h][lane * 2]) = v;
            const float lsum = warp_sum(v.x + v.y);
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
        const unsigned char* vbase = base + (size_t)ATT_TILE * ROWB + dl * 8;
#pragma unroll 4
        for (int j = tg; j < ATT_TILE; j += NG) {
            uint2 w = *reinterpret_cast<const uint2*>(vbase + (size_t)j * ROWB);
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
    }
    cp_async_wait<0>();
    __syncthreads();

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

template <int HD>
static int launch_att(const AttnArgs& a, cudaStream_t st) {
    static bool attr_set = false;
    if (!attr_set) {
        if (cudaFuncSetAttribute(k_attention<HD>, cudaFuncAttributeMaxDynamicSharedMemorySize, AttSmem<HD>::BYTES) != cudaSuccess)
            return -1;
        attr_set = true;
    }
    dim3 grid(a.m_max, a.Hkv, a.n_splits);
    k_attention<HD><<<grid, ATT_THREADS, AttSmem<HD>::BYTES, st>>>(a);
    return 1;
}

int launch_attention(const AttnArgs& a, cudaStream_t st) {
    if (a.m_max <= 0) return 0;
    if (a.hd == 128) return launch_att<128>(a, st);
    if (a.hd == 64) return launch_att<64>(a, st);
    if (a.hd == 32) return launch_att<32>(a, st);
    return -1;
}

}  // namespace sagc
