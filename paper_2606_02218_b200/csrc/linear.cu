// linear.cu -- decode / prefill projections  Y = epi( rms?(X) . W^T )  (steps a6, a8-a11).
//
// Weight-streaming "skinny GEMM": the bf16 weight matrix is the MMA A operand (16 rows x 16 k
// per HMMA), read ONCE per launch straight from HBM into registers in fragment order (no shared
// memory round trip); the fp32 activations are split x = hi + lo into two bf16 halves (~16
// mantissa bits) and staged in shared memory in B-fragment
// order, so each weight fragment feeds 2*NT HMMAs (NT = live rows / 8).  fp32 accumulation.
// RMSNorm is fused: the staged operand is x*w_norm and the accumulator is scaled by
// rsqrt(mean(x^2)+eps) in the epilogue (the row sums are formed while staging).
//
//   mode A (wide N): one 16-row tile per warp over the full K, 8 tiles per CTA.
//   mode B (narrow N, e.g. O / down projections): one 16-row tile per CTA, the 8 warps
//          interleave the 32-wide k blocks and reduce through shared memory (fixed order).
// A separate fp32-activation GEMV kernel (LIN_GEMV) serves the straggler tail.
#include <cooperative_groups.h>

#include <cstdlib>

#include "common.cuh"
#include "kernels.cuh"

namespace cg = cooperative_groups;

namespace sagc {

static constexpr int LIN_THREADS = 256;
static constexpr int LIN_WARPS = 8;

struct LinDev {
    const bf16_t* W0; const bf16_t* W1; const bf16_t* W2;
    int r0, r1;                 // segment boundaries: rows [0,r0) -> W0, [r0,r1) -> W1, rest W2
    const float* X; const bf16_t* norm_w; float eps;
    float* Y; const float* R; int ldy;
    int K, N;
    const int* m_dev; int m_max;
};

__device__ __forceinline__ const bf16_t* seg_row(const LinDev& a, int n) {
    if (n < a.r0) return a.W0 + (size_t)n * a.K;
    if (n < a.r1) return a.W1 + (size_t)(n - a.r0) * a.K;
    return a.W2 + (size_t)(n - a.r1) * a.K;
}

// Stage a K-chunk of X (rows m0 .. m0+8*NT) into B-fragment order.
//   layout: [kb][nt][half(hi,lo)][lane = (m%8)*4 + (k8%4)][4 words]   (16 B per lane: conflict-free LDS.128)
// Each item = 8 consecutive k of one row.  Registers hold the raw floats between issue and store.
template <int NT, int KC>
struct Stager {
    static constexpr int ITEMS = NT * 8 * (KC / 8);
    static constexpr int PER_THREAD = (ITEMS + LIN_THREADS - 1) / LIN_THREADS;
    float4 v[PER_THREAD][2];
    float ssq[PER_THREAD];

    __device__ __forceinline__ void init() {
#pragma unroll
        for (int i = 0; i < PER_THREAD; ++i) ssq[i] = 0.f;
    }
    __device__ __forceinline__ void issue(const LinDev& a, int m0, int M, int k0) {
#pragma unroll
        for (int i = 0; i < PER_THREAD; ++i) {
            int item = i * LIN_THREADS + threadIdx.x;
            int m = item / (KC / 8), j = item % (KC / 8);
            int k = k0 + j * 8;
            v[i][0] = make_float4(0.f, 0.f, 0.f, 0.f);
            v[i][1] = v[i][0];
            if (item < ITEMS && (m0 + m) < M && k < a.K) {
                const float4* p = reinterpret_cast<const float4*>(a.X + (size_t)(m0 + m) * a.K + k);
                v[i][0] = __ldcg(p);
                v[i][1] = __ldcg(p + 1);
            }
        }
    }
    __device__ __forceinline__ void store(const LinDev& a, uint32_t* buf, int k0) {
#pragma unroll
        for (int i = 0; i < PER_THREAD; ++i) {
            int item = i * LIN_THREADS + threadIdx.x;
            if (item >= ITEMS) continue;
            int m = item / (KC / 8), j = item % (KC / 8);
            float4 x0 = v[i][0], x1 = v[i][1];
            ssq[i] += x0.x * x0.x + x0.y * x0.y + x0.z * x0.z + x0.w * x0.w + x1.x * x1.x + x1.y * x1.y +
                      x1.z * x1.z + x1.w * x1.w;
            int k = k0 + j * 8;
            if (a.norm_w != nullptr && k < a.K) {
                uint4 w = *reinterpret_cast<const uint4*>(a.norm_w + k);
                x0.x *= bf16lo_to_f32(w.x); x0.y *= bf16hi_to_f32(w.x);
                x0.z *= bf16lo_to_f32(w.y); x0.w *= bf16hi_to_f32(w.y);
                x1.x *= bf16lo_to_f32(w.z); x1.y *= bf16hi_to_f32(w.z);
                x1.z *= bf16lo_to_f32(w.w); x1.w *= bf16hi_to_f32(w.w);
            }
            uint4 hi, lo;
            split2(x0.x, x0.y, hi.x, lo.x);
            split2(x0.z, x0.w, hi.y, lo.y);
            split2(x1.x, x1.y, hi.z, lo.z);
            split2(x1.z, x1.w, hi.w, lo.w);
            int kb = j >> 2, nt = m >> 3, lane = ((m & 7) << 2) | (j & 3);
            uint32_t* dst = buf + ((size_t)(kb * NT + nt) * 2) * 128 + lane * 4;
            *reinterpret_cast<uint4*>(dst) = hi;
            *reinterpret_cast<uint4*>(dst + 128) = lo;
        }
    }
    // per-row sum of squares -> smem ssq_s[m].  The KC/8 threads of a row are consecutive lanes.
    __device__ __forceinline__ void finish(float* ssq_s) {
        constexpr int TPR = KC / 8;   // threads per row: 16 or 32
#pragma unroll
        for (int i = 0; i < PER_THREAD; ++i) {
            float s = ssq[i];
#pragma unroll
            for (int o = TPR / 2; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
            int item = i * LIN_THREADS + threadIdx.x;
            if (item < ITEMS && (item % TPR) == 0) ssq_s[item / TPR] = s;
        }
    }
};

// one k-block (32 k) of one 16-row weight tile against NT batch tiles
template <int NT>
__device__ __forceinline__ void mma_block(float (&acc)[NT][4], const uint4& wa, const uint4& wb,
                                          const uint32_t* bk, int lane) {
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) {
        const uint32_t* p = bk + (size_t)nt * 256 + lane * 4;
        uint4 hi = *reinterpret_cast<const uint4*>(p);
        uint4 lo = *reinterpret_cast<const uint4*>(p + 128);
        mma_bf16_16816(acc[nt], wa.x, wb.x, wa.y, wb.y, hi.x, hi.y);
        mma_bf16_16816(acc[nt], wa.z, wb.z, wa.w, wb.w, hi.z, hi.w);
        mma_bf16_16816(acc[nt], wa.x, wb.x, wa.y, wb.y, lo.x, lo.y);
        mma_bf16_16816(acc[nt], wa.z, wb.z, wa.w, wb.w, lo.z, lo.w);
    }
}

__device__ __forceinline__ float silu_f(float z) { return z / (1.f + __expf(-z)); }

// Epilogue for one row tile: acc[nt] = (rows g, g+8) x (batch cols 2q, 2q+1).
template <int NT, int EPI>
__device__ __forceinline__ void epilogue(const LinDev& a, float (&acc)[NT][4], float (&acc2)[NT][4],
                                         int row0, int m0, int M, const float* rstd_s, int lane) {
    int g = lane >> 2, q = lane & 3;
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) {
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            int ml = nt * 8 + 2 * q + (e & 1);
            int m = m0 + ml;
            int n = row0 + g + ((e & 2) ? 8 : 0);
            if (m >= M || n >= a.N) continue;
            float s = (a.norm_w != nullptr) ? rstd_s[ml] : 1.f;
            float v = acc[nt][e] * s;
            size_t o = (size_t)m * a.ldy + n;
            if (EPI == EPI_RESID) v += a.R[o];
            if (EPI == EPI_SWIGLU) v = silu_f(v) * (acc2[nt][e] * s);
            a.Y[o] = v;
        }
    }
}

// ---------------------------------------------------------------------------------------
// mode A: warp = one 16-row tile, full K.   KC = 128 (4 k-blocks per chunk).
// ---------------------------------------------------------------------------------------
template <int NT, int EPI>
__global__ void __launch_bounds__(LIN_THREADS) k_linear_wide(LinDev a) {
    constexpr int KC = 128, KB = KC / 32;
    constexpr int NS = (EPI == EPI_SWIGLU) ? 2 : 1;
    extern __shared__ __align__(16) uint32_t smem[];
    uint32_t* buf[2] = {smem, smem + KB * NT * 256};
    float* ssq_s = reinterpret_cast<float*>(smem + 2 * KB * NT * 256);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = lane >> 2, q = lane & 3;
    const int rt = blockIdx.x * LIN_WARPS + warp;
    const int row0 = rt * 16;
    const bool active = row0 < a.N;
    const int m0 = blockIdx.y * (NT * 8);

    // weight row pointers (A fragment rows g and g+8); k offset 8q inside each 32-wide block
    const bf16_t* pa[NS]; const bf16_t* pb[NS];
    if (active) {
        if (EPI == EPI_SWIGLU) {
            pa[0] = a.W0 + (size_t)(row0 + g) * a.K + 8 * q;
            pb[0] = a.W0 + (size_t)(row0 + g + 8) * a.K + 8 * q;
            pa[NS - 1] = a.W1 + (size_t)(row0 + g) * a.K + 8 * q;
            pb[NS - 1] = a.W1 + (size_t)(row0 + g + 8) * a.K + 8 * q;
        } else {
            pa[0] = seg_row(a, row0 + g) + 8 * q;
            pb[0] = seg_row(a, row0 + g + 8) + 8 * q;
        }
    }
    const int n_chunks = (a.K + KC - 1) / KC;
    uint4 wc[NS][KB][2], wn[NS][KB][2];
    auto load_w = [&](uint4 (&w)[NS][KB][2], int c) {
#pragma unroll
        for (int s = 0; s < NS; ++s)
#pragma unroll
            for (int kb = 0; kb < KB; ++kb) {
                int k = c * KC + kb * 32;
                if (active && k < a.K) {
                    w[s][kb][0] = ldg_stream(pa[s] + k);
                    w[s][kb][1] = ldg_stream(pb[s] + k);
                } else {
                    w[s][kb][0] = make_uint4(0, 0, 0, 0);
                    w[s][kb][1] = w[s][kb][0];
                }
            }
    };
    // weights do not depend on the upstream kernel: fetch the first chunk before the PDL wait
    load_w(wc, 0);
    pdl_wait();
    pdl_launch();
    const int M = a.m_dev ? min(*a.m_dev, a.m_max) : a.m_max;
    if (m0 >= M) return;

    Stager<NT, KC> stg;
    stg.init();
    stg.issue(a, m0, M, 0);
    stg.store(a, buf[0], 0);
    __syncthreads();

    float acc[NS][NT][4];
#pragma unroll
    for (int s = 0; s < NS; ++s)
#pragma unroll
        for (int nt = 0; nt < NT; ++nt)
#pragma unroll
            for (int e = 0; e < 4; ++e) acc[s][nt][e] = 0.f;

    for (int c = 0; c < n_chunks; ++c) {
        const bool more = (c + 1) < n_chunks;
        if (more) {
            load_w(wn, c + 1);
            stg.issue(a, m0, M, (c + 1) * KC);
        }
        if (active) {
            const uint32_t* b = buf[c & 1];
#pragma unroll
            for (int kb = 0; kb < KB; ++kb)
#pragma unroll
                for (int s = 0; s < NS; ++s)
                    mma_block<NT>(acc[s], wc[s][kb][0], wc[s][kb][1], b + (size_t)kb * NT * 256, lane);
        }
        if (more) {
            stg.store(a, buf[(c + 1) & 1], (c + 1) * KC);
#pragma unroll
            for (int s = 0; s < NS; ++s)
#pragma unroll
                for (int kb = 0; kb < KB; ++kb) { wc[s][kb][0] = wn[s][kb][0]; wc[s][kb][1] = wn[s][kb][1]; }
        }
        __syncthreads();
    }
    if (a.norm_w != nullptr) {
        stg.finish(ssq_s);
        __syncthreads();
        if (threadIdx.x < NT * 8) ssq_s[threadIdx.x] = rsqrtf(ssq_s[threadIdx.x] / (float)a.K + a.eps);
        __syncthreads();
    }
    if (active) epilogue<NT, EPI>(a, acc[0], acc[NS - 1], row0, m0, M, ssq_s, lane);
}

// ---------------------------------------------------------------------------------------
// mode B: CTA = one 16-row tile; warp w takes k-block w of every 256-wide chunk; 4-deep
// register ring of weight fragments; fixed-order reduction over the 8 warps.
// ---------------------------------------------------------------------------------------
template <int NT, int EPI>
__global__ void __launch_bounds__(LIN_THREADS) k_linear_narrow(LinDev a) {
    constexpr int KC = 256, KB = KC / 32, RING = 4;
    constexpr int NS = (EPI == EPI_SWIGLU) ? 2 : 1;
    extern __shared__ __align__(16) uint32_t smem[];
    uint32_t* buf[2] = {smem, smem + KB * NT * 256};
    float* ssq_s = reinterpret_cast<float*>(smem + 2 * KB * NT * 256);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = lane >> 2, q = lane & 3;
    const int row0 = blockIdx.x * 16;
    const int m0 = blockIdx.y * (NT * 8);
    const bf16_t* pa[NS]; const bf16_t* pb[NS];
    if (EPI == EPI_SWIGLU) {
        pa[0] = a.W0 + (size_t)(row0 + g) * a.K;
        pb[0] = a.W0 + (size_t)(row0 + g + 8) * a.K;
        pa[NS - 1] = a.W1 + (size_t)(row0 + g) * a.K;
        pb[NS - 1] = a.W1 + (size_t)(row0 + g + 8) * a.K;
    } else {
        pa[0] = seg_row(a, row0 + g);
        pb[0] = seg_row(a, row0 + g + 8);
    }
    const int koff = 8 * q + warp * 32;
    const int n_chunks = (a.K + KC - 1) / KC;

    uint4 ring[NS][RING][2];
    auto load_w = [&](int slot, int c) {
        int k = c * KC + warp * 32;
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            if (c < n_chunks && k < a.K) {
                ring[s][slot][0] = ldg_stream(pa[s] + (size_t)c * KC + koff);
                ring[s][slot][1] = ldg_stream(pb[s] + (size_t)c * KC + koff);
            } else {
                ring[s][slot][0] = make_uint4(0, 0, 0, 0);
                ring[s][slot][1] = ring[s][slot][0];
            }
        }
    };
#pragma unroll
    for (int u = 0; u < RING; ++u) load_w(u, u);
    pdl_wait();
    pdl_launch();
    const int M = a.m_dev ? min(*a.m_dev, a.m_max) : a.m_max;
    if (m0 >= M) return;

    Stager<NT, KC> stg;
    stg.init();
    stg.issue(a, m0, M, 0);
    stg.store(a, buf[0], 0);
    __syncthreads();

    float acc[NS][NT][4];
#pragma unroll
    for (int s = 0; s < NS; ++s)
#pragma unroll
        for (int nt = 0; nt < NT; ++nt)
#pragma unroll
            for (int e = 0; e < 4; ++e) acc[s][nt][e] = 0.f;

    for (int c0 = 0; c0 < n_chunks; c0 += RING) {
#pragma unroll
        for (int u = 0; u < RING; ++u) {
            const int c = c0 + u;
            if (c < n_chunks) {
                const bool more = (c + 1) < n_chunks;
                if (more) stg.issue(a, m0, M, (c + 1) * KC);
                if (c * KC + warp * 32 < a.K) {
#pragma unroll
                    for (int s = 0; s < NS; ++s)
                        mma_block<NT>(acc[s], ring[s][u][0], ring[s][u][1],
                                      buf[c & 1] + (size_t)warp * NT * 256, lane);
                }
                load_w(u, c + RING);
                if (more) stg.store(a, buf[(c + 1) & 1], (c + 1) * KC);
                __syncthreads();
            }
        }
    }
    if (a.norm_w != nullptr) stg.finish(ssq_s);
    // reduce the 8 partial accumulators in warp order (deterministic); red overlays the buffers
    float* red = reinterpret_cast<float*>(smem);
#pragma unroll
    for (int s = 0; s < NS; ++s)
#pragma unroll
        for (int nt = 0; nt < NT; ++nt)
#pragma unroll
            for (int e = 0; e < 4; ++e)
                red[(((s * LIN_WARPS + warp) * NT + nt) * 4 + e) * 32 + lane] = acc[s][nt][e];
    __syncthreads();
    if (a.norm_w != nullptr && threadIdx.x < NT * 8)
        ssq_s[threadIdx.x] = rsqrtf(ssq_s[threadIdx.x] / (float)a.K + a.eps);
    __syncthreads();
    // warps 0..NT-1: one batch tile each -- sum the partials and run the epilogue
    if (warp < NT) {
        float r[NS][1][4];
#pragma unroll
        for (int s = 0; s < NS; ++s)
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                float t = 0.f;
#pragma unroll
                for (int w = 0; w < LIN_WARPS; ++w)
                    t += red[(((s * LIN_WARPS + w) * NT + warp) * 4 + e) * 32 + lane];
                r[s][0][e] = t;
            }
        epilogue<1, EPI>(a, r[0], r[NS - 1], row0, m0 + warp * 8, M, ssq_s + warp * 8, lane);
    }
}

// ---------------------------------------------------------------------------------------
// tail kernel (M <= 8): no shared-memory staging at all.  Weight fragments AND the matching
// fp32 activation slices are fetched straight into registers (the activations are a few KB and
// L2-resident), split hi/lo on the fly and fed to HMMA.  SPLITK: the 8 warps of a CTA share one
// 16-row tile and interleave the 32-wide k blocks (narrow N); otherwise one tile per warp.
// ---------------------------------------------------------------------------------------
template <int EPI, bool SPLITK, int NW>
__global__ void __launch_bounds__(NW * 32) k_linear_tail(LinDev a) {
    constexpr int NS = (EPI == EPI_SWIGLU) ? 2 : 1;
    constexpr int U = 4;                                   // k blocks in flight per warp
    __shared__ float red[SPLITK ? NS * NW * 4 * 32 : 1];
    __shared__ float ssq_w[NW][8];
    __shared__ float rstd_s[8];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = lane >> 2, q = lane & 3;
    const int row0 = (SPLITK ? blockIdx.x : blockIdx.x * NW + warp) * 16;
    const bool active = row0 < a.N;
    // narrow N with long K: a cluster of KC CTAs splits K (rank = blockIdx.y), reduced through DSMEM
    cg::cluster_group cluster = cg::this_cluster();
    const int KC = SPLITK ? (int)cluster.num_blocks() : 1;
    const int crank = SPLITK ? (int)cluster.block_rank() : 0;
    const int kb_all = a.K >> 5;
    const int kb_per = (kb_all + KC - 1) / KC;
    const int kb0 = crank * kb_per + (SPLITK ? warp : 0), kbs = SPLITK ? NW : 1;
    const int n_kb = min(kb_all, (crank + 1) * kb_per);
    const bf16_t* pa[NS]; const bf16_t* pb[NS];
    if (active) {
        if (EPI == EPI_SWIGLU) {
            pa[0] = a.W0 + (size_t)(row0 + g) * a.K + 8 * q;
            pb[0] = a.W0 + (size_t)(row0 + g + 8) * a.K + 8 * q;
            pa[NS - 1] = a.W1 + (size_t)(row0 + g) * a.K + 8 * q;
            pb[NS - 1] = a.W1 + (size_t)(row0 + g + 8) * a.K + 8 * q;
        } else {
            pa[0] = seg_row(a, row0 + g) + 8 * q;
            pb[0] = seg_row(a, row0 + g + 8) + 8 * q;
        }
    }
    // Ask L2 for this CTA's whole weight slab right away (one bulk prefetch per row): the DRAM reads then
    // overlap the upstream kernel and the later register loads of the k loop hit L2.
    if (SPLITK && active && warp == 0 && lane < 16 * NS) {
        const int s = lane >> 4, rr = lane & 15;
        const bf16_t* rowp = (EPI == EPI_SWIGLU) ? ((s == 0 ? a.W0 : a.W1) + (size_t)(row0 + rr) * a.K)
                                                 : seg_row(a, row0 + rr);
        asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;\n" ::"l"(rowp), "r"(a.K * 2) : "memory");
    }
    uint4 w[NS][U][2];
    auto load_w = [&](int u, int kb) {
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            if (active && kb < n_kb) {
                w[s][u][0] = ldg_stream(pa[s] + (size_t)kb * 32);
                w[s][u][1] = ldg_stream(pb[s] + (size_t)kb * 32);
            } else {
                w[s][u][0] = make_uint4(0, 0, 0, 0);
                w[s][u][1] = w[s][u][0];
            }
        }
    };
#pragma unroll
    for (int u = 0; u < U; ++u) load_w(u, kb0 + u * kbs);
    trace_mark(16); pdl_wait(); trace_mark(17);
    pdl_launch();
    const int M = a.m_dev ? min(*a.m_dev, a.m_max) : a.m_max;
    if (M <= 0) return;
    const float* xrow = a.X + (size_t)g * a.K + 8 * q;
    const bool xok = g < M;
    float4 x[U][2];
    auto load_x = [&](int u, int kb) {
        if (xok && kb < n_kb) {
            const float4* p = reinterpret_cast<const float4*>(xrow + (size_t)kb * 32);
            x[u][0] = __ldcg(p); x[u][1] = __ldcg(p + 1);
        } else {
            x[u][0] = make_float4(0.f, 0.f, 0.f, 0.f); x[u][1] = x[u][0];
        }
    };
#pragma unroll
    for (int u = 0; u < U; ++u) load_x(u, kb0 + u * kbs);

    float acc[NS][4];
#pragma unroll
    for (int s = 0; s < NS; ++s)
#pragma unroll
        for (int e = 0; e < 4; ++e) acc[s][e] = 0.f;
    float ssq = 0.f;

    for (int kbase = kb0; kbase < n_kb; kbase += U * kbs) {
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int kb = kbase + u * kbs;
            float4 x0 = x[u][0], x1 = x[u][1];
            uint4 wa[NS], wb[NS];
#pragma unroll
            for (int s = 0; s < NS; ++s) { wa[s] = w[s][u][0]; wb[s] = w[s][u][1]; }
            // refill this ring slot before the math
            load_w(u, kb + U * kbs);
            load_x(u, kb + U * kbs);
            if (kb < n_kb) {
                ssq += x0.x * x0.x + x0.y * x0.y + x0.z * x0.z + x0.w * x0.w + x1.x * x1.x + x1.y * x1.y +
                       x1.z * x1.z + x1.w * x1.w;
                if (a.norm_w != nullptr) {
                    uint4 nw = *reinterpret_cast<const uint4*>(a.norm_w + (size_t)kb * 32 + 8 * q);
                    x0.x *= bf16lo_to_f32(nw.x); x0.y *= bf16hi_to_f32(nw.x);
                    x0.z *= bf16lo_to_f32(nw.y); x0.w *= bf16hi_to_f32(nw.y);
                    x1.x *= bf16lo_to_f32(nw.z); x1.y *= bf16hi_to_f32(nw.z);
                    x1.z *= bf16lo_to_f32(nw.w); x1.w *= bf16hi_to_f32(nw.w);
                }
                uint4 hi, lo;
                split2(x0.x, x0.y, hi.x, lo.x);
                split2(x0.z, x0.w, hi.y, lo.y);
                split2(x1.x, x1.y, hi.z, lo.z);
                split2(x1.z, x1.w, hi.w, lo.w);
#pragma unroll
                for (int s = 0; s < NS; ++s) {
                    mma_bf16_16816(acc[s], wa[s].x, wb[s].x, wa[s].y, wb[s].y, hi.x, hi.y);
                    mma_bf16_16816(acc[s], wa[s].z, wb[s].z, wa[s].w, wb[s].w, hi.z, hi.w);
                    mma_bf16_16816(acc[s], wa[s].x, wb[s].x, wa[s].y, wb[s].y, lo.x, lo.y);
                    mma_bf16_16816(acc[s], wa[s].z, wb[s].z, wa[s].w, wb[s].w, lo.z, lo.w);
                }
            }
        }
    }
    trace_mark_allblocks(4 * 4 + 2);
    // row sums of squares: lanes (g, q = 0..3) hold disjoint k slices of batch row g
    if (a.norm_w != nullptr) {
        ssq += __shfl_xor_sync(0xffffffffu, ssq, 1);
        ssq += __shfl_xor_sync(0xffffffffu, ssq, 2);
        if (q == 0) ssq_w[warp][g] = ssq;
    }
    if (SPLITK) {
#pragma unroll
        for (int s = 0; s < NS; ++s)
#pragma unroll
            for (int e = 0; e < 4; ++e) red[((s * NW + warp) * 4 + e) * 32 + lane] = acc[s][e];
    }
    __syncthreads();
    if (a.norm_w != nullptr && threadIdx.x < 8) {
        float t = 0.f;
        if (SPLITK) {
#pragma unroll
            for (int wi = 0; wi < NW; ++wi) t += ssq_w[wi][threadIdx.x];
        }
        rstd_s[threadIdx.x] = t;
    }
    if (!SPLITK && a.norm_w != nullptr) {
        // every warp saw the whole of X: its own sums are complete
        __syncwarp();
    }
    __syncthreads();
    if (SPLITK) {
        __shared__ float cred[NS * 4 * 32 + 8];
        float r[NS][1][4];
        if (warp == 0) {
#pragma unroll
            for (int s = 0; s < NS; ++s)
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    float t = 0.f;
#pragma unroll
                    for (int wi = 0; wi < NW; ++wi) t += red[((s * NW + wi) * 4 + e) * 32 + lane];
                    r[s][0][e] = t;
                }
            if (KC > 1 && crank != 0) {
#pragma unroll
                for (int s = 0; s < NS; ++s)
#pragma unroll
                    for (int e = 0; e < 4; ++e) cred[(s * 4 + e) * 32 + lane] = r[s][0][e];
                if (lane < 8) cred[NS * 4 * 32 + lane] = rstd_s[lane];
            }
        }
        if (KC > 1) cluster.sync();
        if (warp == 0 && crank == 0) {
            for (int p = 1; p < KC; ++p) {                         // rank order: deterministic
                const float* pc = cluster.map_shared_rank(cred, p);
#pragma unroll
                for (int s = 0; s < NS; ++s)
#pragma unroll
                    for (int e = 0; e < 4; ++e) r[s][0][e] += pc[(s * 4 + e) * 32 + lane];
                if (lane < 8) rstd_s[lane] += pc[NS * 4 * 32 + lane];
            }
            if (a.norm_w != nullptr) {
                if (lane < 8) rstd_s[lane] = rsqrtf(rstd_s[lane] / (float)a.K + a.eps);
                __syncwarp();
            }
            if (active) epilogue<1, EPI>(a, r[0], r[NS - 1], row0, 0, M, rstd_s, lane);
        }
        if (KC > 1) cluster.sync();                                // keep cred alive until rank 0 has read it
    } else {
        float* mine = ssq_w[warp];
        if (a.norm_w != nullptr) {
            if (lane < 8) mine[lane] = rsqrtf(mine[lane] / (float)a.K + a.eps);
            __syncwarp();
        }
        float r[NS][1][4];
#pragma unroll
        for (int s = 0; s < NS; ++s)
#pragma unroll
            for (int e = 0; e < 4; ++e) r[s][0][e] = acc[s][e];
        if (active) epilogue<1, EPI>(a, r[0], r[NS - 1], row0, 0, M, mine, lane);
    }
}

// ---------------------------------------------------------------------------------------
// LIN_GEMV: fp32-activation GEMV for the straggler tail (M <= 4 per pass, exact fp32 x).
// One warp = two output rows over the full K; 16-byte weight loads, activations through L1.
// ---------------------------------------------------------------------------------------
template <int MB, int EPI>
__global__ void __launch_bounds__(LIN_THREADS) k_linear_gemv(LinDev a) {
    constexpr int NS = (EPI == EPI_SWIGLU) ? 2 : 1;
    constexpr int R = (EPI == EPI_SWIGLU) ? 1 : 2;       // rows per warp per stream
    __shared__ float rstd_s[MB];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int row0 = (blockIdx.x * LIN_WARPS + warp) * R;
    const int m0 = blockIdx.y * MB;
    const bool active = row0 < a.N;
    const bf16_t* pw[NS][R];
    if (active) {
        if (EPI == EPI_SWIGLU) {
            pw[0][0] = a.W0 + (size_t)row0 * a.K;
            pw[NS - 1][0] = a.W1 + (size_t)row0 * a.K;
        } else {
#pragma unroll
            for (int r = 0; r < R; ++r) pw[0][r] = seg_row(a, min(row0 + r, a.N - 1));
        }
        // warm L2 with the head of the rows while the upstream kernel drains
#pragma unroll
        for (int s = 0; s < NS; ++s)
#pragma unroll
            for (int r = 0; r < R; ++r) prefetch_l2(pw[s][r] + lane * 64);
    }
    pdl_wait();
    pdl_launch();
    const int M = a.m_dev ? min(*a.m_dev, a.m_max) : a.m_max;
    if (m0 >= M) return;
    if (a.norm_w != nullptr) {
        // sum of squares of each of the MB rows: warp w handles row w (MB <= 8)
        if (warp < MB) {
            float s = 0.f;
            if (m0 + warp < M) {
                const float4* xr = reinterpret_cast<const float4*>(a.X + (size_t)(m0 + warp) * a.K);
                for (int k = lane; k < a.K / 4; k += 32) {
                    float4 v = __ldg(xr + k);
                    s += v.x * v.x + v.y * v.y + v.z * v.z + v.w * v.w;
                }
            }
            s = warp_sum(s);
            if (lane == 0) rstd_s[warp] = rsqrtf(s / (float)a.K + a.eps);
        }
        __syncthreads();
    }
    if (!active) return;
    float acc[NS][R][MB];
#pragma unroll
    for (int s = 0; s < NS; ++s)
#pragma unroll
        for (int r = 0; r < R; ++r)
#pragma unroll
            for (int m = 0; m < MB; ++m) acc[s][r][m] = 0.f;

#pragma unroll 2
    for (int k = lane * 8; k < a.K; k += 256) {
        uint4 w[NS][R];
#pragma unroll
        for (int s = 0; s < NS; ++s)
#pragma unroll
            for (int r = 0; r < R; ++r) w[s][r] = ldg_stream(pw[s][r] + k);
        float nw[8];
        if (a.norm_w != nullptr) {
            uint4 t = *reinterpret_cast<const uint4*>(a.norm_w + k);
            nw[0] = bf16lo_to_f32(t.x); nw[1] = bf16hi_to_f32(t.x); nw[2] = bf16lo_to_f32(t.y); nw[3] = bf16hi_to_f32(t.y);
            nw[4] = bf16lo_to_f32(t.z); nw[5] = bf16hi_to_f32(t.z); nw[6] = bf16lo_to_f32(t.w); nw[7] = bf16hi_to_f32(t.w);
        }
#pragma unroll
        for (int m = 0; m < MB; ++m) {
            float x[8];
            if (m0 + m < M) {
                const float4* xp = reinterpret_cast<const float4*>(a.X + (size_t)(m0 + m) * a.K + k);
                float4 x0 = __ldg(xp), x1 = __ldg(xp + 1);
                x[0] = x0.x; x[1] = x0.y; x[2] = x0.z; x[3] = x0.w; x[4] = x1.x; x[5] = x1.y; x[6] = x1.z; x[7] = x1.w;
            } else {
#pragma unroll
                for (int i = 0; i < 8; ++i) x[i] = 0.f;
            }
            if (a.norm_w != nullptr) {
#pragma unroll
                for (int i = 0; i < 8; ++i) x[i] *= nw[i];
            }
#pragma unroll
            for (int s = 0; s < NS; ++s)
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const uint4& ww = w[s][r];
                    float t = acc[s][r][m];
                    t = fmaf(bf16lo_to_f32(ww.x), x[0], t); t = fmaf(bf16hi_to_f32(ww.x), x[1], t);
                    t = fmaf(bf16lo_to_f32(ww.y), x[2], t); t = fmaf(bf16hi_to_f32(ww.y), x[3], t);
                    t = fmaf(bf16lo_to_f32(ww.z), x[4], t); t = fmaf(bf16hi_to_f32(ww.z), x[5], t);
                    t = fmaf(bf16lo_to_f32(ww.w), x[6], t); t = fmaf(bf16hi_to_f32(ww.w), x[7], t);
                    acc[s][r][m] = t;
                }
        }
    }
#pragma unroll
    for (int s = 0; s < NS; ++s)
#pragma unroll
        for (int r = 0; r < R; ++r)
#pragma unroll
            for (int m = 0; m < MB; ++m) acc[s][r][m] = warp_sum(acc[s][r][m]);
    if (lane == 0) {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            int n = row0 + r;
            if (n >= a.N) continue;
#pragma unroll
            for (int m = 0; m < MB; ++m) {
                if (m0 + m >= M) continue;
                float sc = (a.norm_w != nullptr) ? rstd_s[m] : 1.f;
                float v = acc[0][r][m] * sc;
                size_t o = (size_t)(m0 + m) * a.ldy + n;
                if (EPI == EPI_RESID) v += a.R[o];
                if (EPI == EPI_SWIGLU) v = silu_f(v) * (acc[NS - 1][r][m] * sc);
                a.Y[o] = v;
            }
        }
    }
}

// ---------------------------------------------------------------------------------------
// launcher
// ---------------------------------------------------------------------------------------
template <typename Kern>
static cudaError_t launch_cfg(Kern kern, dim3 grid, int smem, bool pdl, cudaStream_t st, LinDev d, int threads = LIN_THREADS,
                              int cluster_y = 1) {
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = dim3(threads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[2];
    int na = 0;
    if (pdl) {
        at[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[na].val.programmaticStreamSerializationAllowed = 1;
        ++na;
    }
    if (cluster_y > 1) {
        at[na].id = cudaLaunchAttributeClusterDimension;
        at[na].val.clusterDim.x = 1; at[na].val.clusterDim.y = cluster_y; at[na].val.clusterDim.z = 1;
        ++na;
    }
    cfg.attrs = at;
    cfg.numAttrs = na;
    return cudaLaunchKernelEx(&cfg, kern, d);
}

template <int EPI>
static cudaError_t launch_epi(const LinearArgs& a, const LinDev& d, cudaStream_t st) {
    const int tiles = (a.N + 15) / 16;
    if (a.kind == LIN_GEMV) {
        constexpr int R = (EPI == EPI_SWIGLU) ? 1 : 2;
        int mb = a.m_max <= 1 ? 1 : (a.m_max <= 2 ? 2 : 4);
        dim3 grid((a.N + LIN_WARPS * R - 1) / (LIN_WARPS * R), (a.m_max + mb - 1) / mb);
        if (mb == 1) return launch_cfg(k_linear_gemv<1, EPI>, grid, 0, a.pdl, st, d);
        if (mb == 2) return launch_cfg(k_linear_gemv<2, EPI>, grid, 0, a.pdl, st, d);
        return launch_cfg(k_linear_gemv<4, EPI>, grid, 0, a.pdl, st, d);
    }
    const bool wide = tiles >= 148 * LIN_WARPS;
    if (a.m_max <= 8) {
        if (wide) return launch_cfg(k_linear_tail<EPI, false, 8>, dim3((tiles + 7) / 8), 0, a.pdl, st, d, 256);
        // narrow N: one 16-row tile per CTA, the warps interleave the k blocks.  Pick the warp count so
        // that the grid is ONE wave (small CTAs co-reside) and long K gets more warps (fewer load rounds).
        const int n_kb = a.K / 32;
        if (tiles > 148 * 2) return launch_cfg(k_linear_tail<EPI, true, 4>, dim3(tiles), 0, a.pdl, st, d, 128);
        if (false && n_kb >= 96 && tiles <= 74) {   // optional: K split over a 2-CTA cluster (DSMEM reduce)
            return launch_cfg(k_linear_tail<EPI, true, 16>, dim3(tiles, 2), 0, a.pdl, st, d, 512, 2);
        }
        if (n_kb >= 96 && tiles <= 148) return launch_cfg(k_linear_tail<EPI, true, 16>, dim3(tiles), 0, a.pdl, st, d, 512);
        return launch_cfg(k_linear_tail<EPI, true, 8>, dim3(tiles), 0, a.pdl, st, d, 256);
    }
    int nt = a.m_max <= 16 ? 2 : (a.m_max <= 32 ? 4 : 8);
    const int my = (a.m_max + nt * 8 - 1) / (nt * 8);
    if (wide) {
        dim3 grid((tiles + LIN_WARPS - 1) / LIN_WARPS, my);
        int smem = 2 * 4 * nt * 1024 + 64 * 4;
        switch (nt) {
            case 1: return launch_cfg(k_linear_wide<1, EPI>, grid, smem, a.pdl, st, d);
            case 2: return launch_cfg(k_linear_wide<2, EPI>, grid, smem, a.pdl, st, d);
            case 4: return launch_cfg(k_linear_wide<4, EPI>, grid, smem, a.pdl, st, d);
            default: return launch_cfg(k_linear_wide<8, EPI>, grid, smem, a.pdl, st, d);
        }
    }
    dim3 grid(tiles, my);
    int smem = 2 * 8 * nt * 1024 + 64 * 4;
    switch (nt) {
        case 1: return launch_cfg(k_linear_narrow<1, EPI>, grid, smem, a.pdl, st, d);
        case 2: return launch_cfg(k_linear_narrow<2, EPI>, grid, smem, a.pdl, st, d);
        case 4: return launch_cfg(k_linear_narrow<4, EPI>, grid, smem, a.pdl, st, d);
        default: return launch_cfg(k_linear_narrow<8, EPI>, grid, smem, a.pdl, st, d);
    }
}

int launch_linear(const LinearArgs& a, cudaStream_t st) {
    LinDev d;
    d.W0 = a.W[0]; d.W1 = a.W[1]; d.W2 = a.W[2];
    d.r0 = a.rows[0]; d.r1 = a.rows[0] + a.rows[1];
    if (a.W[1] == nullptr) { d.r0 = a.N; d.r1 = a.N; }
    d.X = a.X; d.norm_w = a.norm_w; d.eps = a.eps; d.Y = a.Y; d.R = a.R; d.ldy = a.ldy;
    d.K = a.K; d.N = a.N; d.m_dev = a.m_dev; d.m_max = a.m_max;
    if (a.m_max <= 0) return 0;
    cudaError_t e;
    if (a.epi == EPI_SWIGLU) e = launch_epi<EPI_SWIGLU>(a, d, st);
    else if (a.epi == EPI_RESID) e = launch_epi<EPI_RESID>(a, d, st);
    else e = launch_epi<EPI_STORE>(a, d, st);
    return e == cudaSuccess ? 1 : -1;
}

}  // namespace sagc
