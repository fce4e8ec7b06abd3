// tc_linear.cu -- tcgen05 / TMEM / TMA projections for the large-batch regime (M > 8 rows) and
// prefill (steps a2, a6, a8-a11).
//
// Swapped-operand skinny GEMM: the bf16 weight tile (128 rows x 64 k, TMA, 128B swizzle) is the
// UMMA A operand (M = 128); the activations are the B operand.  Activations arrive pre-split in
// HBM as interleaved bf16 rows  Xs[2m] = hi(x[m]),  Xs[2m+1] = lo(x[m])  (x = hi + lo keeps ~16
// mantissa bits), so ONE weight tile read from HBM feeds both
// halves: UMMA N = 2 * (batch rows in the tile), and  y[m][n] = D[n][2m] + D[n][2m+1].
// fp32 accumulators live in TMEM.  Narrow outputs (N = d_model) are parallelised by splitting K
// across a thread-block cluster; the partial accumulators are reduced through distributed shared
// memory in rank order (deterministic), every CTA of the cluster finishing a slice of the batch
// columns.  Warp roles: 0 = TMA producer, 1 = MMA issuer (one elected lane), 2..5 = epilogue
// (TMEM lanes 32*(warp%4)); warp 2 also owns the TMEM allocation.
#include <cooperative_groups.h>
#include <cuda.h>

#include <cstdlib>

#include "common.cuh"
#include "kernels.cuh"
#include "tc_ptx.cuh"

namespace cg = cooperative_groups;

namespace sagc {

static constexpr int TC_THREADS = 192;
static constexpr int TC_BK = 64;             // k elements per stage (one 128-byte swizzle atom)

struct TcDev {
    int K, N;                       // weight shape [N][K]
    int kb_per_cta;                 // 64-wide k blocks per CTA (cluster rank r takes blocks [r*kb, (r+1)*kb))
    int n_kb;                       // total k blocks
    const int* m_dev; int m_max;
    float* Y; int ldy;              // EPI_STORE / EPI_RESID: fp32 [M][ldy]
    const float* R;
    bf16_t* xs_out; int ld_xs;      // EPI_SWIGLU / EPI_RESID: pre-split output rows [2m], [2m+1]
    const bf16_t* norm_next;        // EPI_RESID: gain of the NEXT RMSNorm, folded into xs_out
    float* ssq_out;                 // EPI_RESID: [N/128][ssq_ld] partial sums of squares of the new x
    const float* ssq_in; int ssq_in_tiles;   // fused RMSNorm of the INPUT: rstd[m] from these partials
    int ssq_ld; float eps; int k_norm;
    int stages;                     // smem ring depth chosen by the launcher
    int mtiles;                     // batch tiles of MB rows; blockIdx.x = weight tile * mtiles + batch tile
    float* scratch;                 // split-K partial tiles [cta][NA][MB][128] (L2-resident), KS > 1 only
    // EPI_QKV (fused RoPE + KV append)
    const float* rope_cs; const int* row_pos; const int* row_sid; const int* page_table; bf16_t* kv_layer;
    int max_blocks, page, Hkv, hd, q_rows, kv_rows;
};

template <int NB, int NA>
struct TcCfg {
    static constexpr int A_BYTES = 128 * 128;
    static constexpr int B_BYTES = NB * 128;
    static constexpr int STAGE = NA * A_BYTES + B_BYTES;
    // ~100 KB of stages per CTA so that two CTAs share an SM (one's epilogue overlaps the other's loads)
    // SwiGLU at UMMA N = 32 (36 KB stages): three stages and no receive buffer still fit two CTAs per SM (111 KB each)
    static constexpr bool GU32 = (NA == 2 && NB == 32);
    static constexpr int STAGES = GU32 ? 3 : ((100 * 1024 / STAGE) < 2 ? 2 : ((100 * 1024 / STAGE) > 6 ? 6 : (100 * 1024 / STAGE)));
    static constexpr int MB = NB / 2;
    static constexpr int TMEM_COLS = NA * NB <= 32 ? 32 : (NA * NB <= 64 ? 64 : (NA * NB <= 128 ? 128 : (NA * NB <= 256 ? 256 : 512)));
    static constexpr int TAIL = 1024;                                  // barriers, tmem slot, rstd, ssq scratch
    static constexpr int MAXSTAGES = (196 * 1024 / STAGE) > 8 ? 8 : (196 * 1024 / STAGE);
    static constexpr bool PUSH_OK = !GU32 && NA * (NB / 2) * 128 * 4 <= 16 * 1024;   // keep the SwiGLU kernel at two CTAs per SM
    static constexpr int RECV = PUSH_OK ? NA * (NB / 2) * 128 * 4 : 0;     // split-K partials pushed by the cluster peers
    static constexpr int EXCH = 32 * 128 * 4;                          // RoPE partner exchange (EPI_QKV)
    // the exchange buffer exists only in the EPI_QKV instantiation: 16 KB more would cost the SwiGLU kernel its
    // second CTA per SM (152 CTAs -> two waves)
    static constexpr int smem_bytes(int stages, bool qkv) { return stages * STAGE + TAIL + 5 * MB * 4 + (qkv ? EXCH : 0) + RECV + 1024; }
};

__device__ __forceinline__ float silu_tc(float z) { return z / (1.f + __expf(-z)); }

// TMEM -> (hi + lo) -> where the reduction will read it.  KS == 1: this CTA's shared memory.  KS > 1 and a
// small partial tile (<= 16 KB): PUSHED straight into the shared memory of the cluster rank that owns the
// column (remote stores are fire-and-forget, so the split-K exchange costs no load round trip; the tile is
// <= 32 KB, well within DSMEM's ~20 B/clk).  Otherwise: the L2 scratch.
template <int NB, int NA, int KS>
__device__ __forceinline__ void tc_drain(const TcDev& a, cg::cluster_group& cluster, float* red, float* recv, uint32_t tmem_base,
                                         int lg, int row, int rank, int cta_id, bool have_acc) {
    constexpr int MB = NB / 2;
    constexpr bool PUSH = (KS > 1) && TcCfg<NB, NA>::PUSH_OK;
    float* rp[KS];
    if (PUSH) {
#pragma unroll
        for (int d = 0; d < KS; ++d) rp[d] = cluster.map_shared_rank(recv, d);
    }
#pragma unroll
    for (int na = 0; na < NA; ++na) {
#pragma unroll
        for (int c = 0; c < NB / 32; ++c) {
            float v[32];
            if (have_acc) {
                tc_ld32(tmem_base + ((uint32_t)(lg * 32) << 16) + (uint32_t)(na * NB + c * 32), v);
            } else {
#pragma unroll
                for (int j = 0; j < 32; ++j) v[j] = 0.f;
            }
#pragma unroll
            for (int j = 0; j < 16; ++j) {
                const int m = c * 16 + j;
                const float val = v[2 * j] + v[2 * j + 1];
                if (KS == 1) {
                    red[((size_t)na * MB + m) * 128 + row] = val;
                } else if (PUSH) {
                    rp[m % KS][(((size_t)rank * NA + na) * (MB / KS) + m / KS) * 128 + row] = val;
                } else {
                    __stcg(a.scratch + (size_t)cta_id * (NA * MB * 128) + ((size_t)na * MB + m) * 128 + row, val);
                }
            }
        }
    }
}

// Final epilogue of one CTA: rank r of a KS-way split finishes batch columns r, r+KS, ...  KS is a
// compile-time constant so that EVERY load of a batch (all ranks' partial tiles from L2, or the local
// tile from shared memory, plus the residual) is issued before the first use: one memory round trip per
// batch of 64 / (NA*KS) columns, partials summed in rank order (deterministic).
template <int NB, int EPI, int KS>
__device__ __forceinline__ void tc_epilogue(const TcDev& a, const float* red, const float* rstd_s, float* ssq_s, float* exch,
                                            const float* recv, int warp, int lane, int row0, int m0, int tile, int rank, int cta_id,
                                            int M, float nw) {
    constexpr int NA = (EPI == EPI_SWIGLU) ? 2 : 1;
    constexpr int MB = NB / 2;
    constexpr int MBATCH = (KS == 1) ? 16 / NA : 64 / (NA * KS);
    const int lg = warp & 3;
    const int row = lg * 32 + lane;
    const int n = row0 + row;
    constexpr bool PUSH = (KS > 1) && TcCfg<NB, NA>::PUSH_OK;
    const float* base = (KS == 1) ? red : a.scratch + (size_t)(cta_id - rank) * (NA * MB * 128);
    for (int mb = rank; mb < MB; mb += KS * MBATCH) {
        if (m0 + mb >= M) break;
        int mc[MBATCH];
        float v[KS][MBATCH][NA], res[MBATCH];
#pragma unroll
        for (int j = 0; j < MBATCH; ++j) {
            mc[j] = min(mb + j * KS, MB - 1);
            res[j] = (EPI == EPI_RESID) ? a.R[(size_t)min(m0 + mc[j], M - 1) * a.ldy + n] : 0.f;
        }
#pragma unroll
        for (int p = 0; p < KS; ++p)
#pragma unroll
            for (int j = 0; j < MBATCH; ++j)
#pragma unroll
                for (int na = 0; na < NA; ++na) {
                    if (PUSH) {
                        v[p][j][na] = recv[(((size_t)p * NA + na) * (MB / KS) + mc[j] / KS) * 128 + row];
                    } else {
                        const float* src = base + (size_t)p * (NA * MB * 128) + ((size_t)na * MB + mc[j]) * 128 + row;
                        v[p][j][na] = (KS == 1) ? *src : __ldcg(src);
                    }
                }
        float outv[MBATCH], q2[MBATCH];
        uint32_t ohi[MBATCH], olo[MBATCH];
#pragma unroll
        for (int j = 0; j < MBATCH; ++j) {
            float acc[NA];
#pragma unroll
            for (int na = 0; na < NA; ++na) {
                float t = v[0][j][na];
#pragma unroll
                for (int p = 1; p < KS; ++p) t += v[p][j][na];
                acc[na] = t;
            }
            const float sc = (a.ssq_in != nullptr) ? rstd_s[mc[j]] : 1.f;
            float o;
            if (EPI == EPI_STORE || EPI == EPI_QKV) o = acc[0] * sc;
            else if (EPI == EPI_RESID) o = res[j] + acc[0] * sc;
            else o = silu_tc(acc[0] * sc) * (acc[NA - 1] * sc);
            outv[j] = o;
            const float xw = (EPI == EPI_RESID) ? o * nw : o;
            ohi[j] = f32_to_bf16_bits(xw);
            olo[j] = f32_to_bf16_bits(xw - __uint_as_float(ohi[j] << 16));
            q2[j] = o * o;
        }
        if (EPI == EPI_RESID && a.ssq_out != nullptr) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1)
#pragma unroll
                for (int j = 0; j < MBATCH; ++j) q2[j] += __shfl_xor_sync(0xffffffffu, q2[j], o);
        }
        if (EPI == EPI_QKV) {
            // RoPE (rotate-half): the partner feature n +- hd/2 lives in another lane / warp of this CTA
            const int half = a.hd >> 1;
            const bool is_v = row0 >= a.q_rows + a.kv_rows;
            const bool is_q = row0 < a.q_rows;
            const int d = n & (a.hd - 1);
            int posj[MBATCH];
            float2 cs[MBATCH];
#pragma unroll
            for (int j = 0; j < MBATCH; ++j) posj[j] = a.row_pos[max(min(m0 + mc[j], M - 1), 0)];
#pragma unroll
            for (int j = 0; j < MBATCH; ++j)
                cs[j] = is_v ? make_float2(1.f, 0.f)
                             : *reinterpret_cast<const float2*>(a.rope_cs + ((size_t)posj[j] * half + (d & (half - 1))) * 2);
#pragma unroll
            for (int j = 0; j < MBATCH; ++j) exch[j * 128 + row] = outv[j];
            asm volatile("bar.sync 1, 128;\n" ::: "memory");
#pragma unroll
            for (int j = 0; j < MBATCH; ++j) {
                const float partner = exch[j * 128 + (row ^ half)];
                const float rot = (d < half) ? outv[j] * cs[j].x - partner * cs[j].y : outv[j] * cs[j].x + partner * cs[j].y;
                outv[j] = is_v ? outv[j] : rot;
            }
            asm volatile("bar.sync 1, 128;\n" ::: "memory");
#pragma unroll
            for (int j = 0; j < MBATCH; ++j) {
                const int m = mb + j * KS;
                const int mg = m0 + m;
                if (m < MB && mg < M) {
                    if (is_q) {
                        a.Y[(size_t)mg * a.ldy + n] = outv[j];
                    } else {
                        const int sid = a.row_sid[mg];
                        const int pg = a.page_table[(size_t)sid * a.max_blocks + posj[j] / a.page];
                        if (pg >= 0) {
                            const int feat = n - a.q_rows - (is_v ? a.kv_rows : 0);
                            const int kvh = feat / a.hd;
                            bf16_t* dst = a.kv_layer + (((size_t)pg * 2 + (is_v ? 1 : 0)) * a.Hkv + kvh) * (size_t)a.page * a.hd +
                                          (size_t)(posj[j] % a.page) * a.hd + d;
                            *dst = (bf16_t)f32_to_bf16_bits(outv[j]);
                        }
                    }
                }
            }
            continue;
        }
#pragma unroll
        for (int j = 0; j < MBATCH; ++j) {
            const int m = mb + j * KS;
            const int mg = m0 + m;
            if (m < MB && mg < M) {
                if (EPI != EPI_SWIGLU) a.Y[(size_t)mg * a.ldy + n] = outv[j];
                if (EPI != EPI_STORE && a.xs_out != nullptr) {
                    a.xs_out[(size_t)(2 * mg) * a.ld_xs + n] = (bf16_t)ohi[j];
                    a.xs_out[(size_t)(2 * mg + 1) * a.ld_xs + n] = (bf16_t)olo[j];
                }
                if (EPI == EPI_RESID && a.ssq_out != nullptr && lane == 0) ssq_s[lg * MB + m] = q2[j];
            }
        }
    }
    trace_mark_thread(9 * 4 + 1, 64);
    if (EPI == EPI_RESID && a.ssq_out != nullptr) {
        asm volatile("bar.sync 1, 128;\n" ::: "memory");
        const int et = (warp - 2) * 32 + lane;
        for (int m = et; m < MB; m += 128) {
            if ((m % KS) == rank && m0 + m < M)
                a.ssq_out[(size_t)tile * a.ssq_ld + m0 + m] =
                    ssq_s[0 * MB + m] + ssq_s[1 * MB + m] + ssq_s[2 * MB + m] + ssq_s[3 * MB + m];
        }
    }
}

template <int NB, int EPI>
__global__ void __launch_bounds__(TC_THREADS, 1)
k_linear_tc(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmA2,
            const __grid_constant__ CUtensorMap tmA3, const __grid_constant__ CUtensorMap tmB, int seg0, int seg1,
            TcDev a) {
    constexpr int NA = (EPI == EPI_SWIGLU) ? 2 : 1;
    using C = TcCfg<NB, NA>;
    constexpr int MB = C::MB;
    const int S = a.stages;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem + S * C::STAGE);
    uint64_t* empty = full + S;
    uint64_t* accum = empty + S;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(accum + 1);
    float* rstd_s = reinterpret_cast<float*>(smem + S * C::STAGE + C::TAIL);
    float* ssq_s = rstd_s + MB;                                         // [4][MB]
    float* exch = ssq_s + 4 * MB;                                       // [32][128] (EPI_QKV)
    float* recv = reinterpret_cast<float*>(smem + S * C::STAGE + C::TAIL + 5 * MB * 4 + (EPI == EPI_QKV ? C::EXCH : 0));   // pushed partials
    float* red = reinterpret_cast<float*>(smem);                        // [NA][MB][128], overlays the stages

    cg::cluster_group cluster = cg::this_cluster();
    const int rank = (int)cluster.block_rank();
    const int KS = (int)cluster.num_blocks();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // the batch tiles of one weight tile are NEIGHBOURS in launch order: they run in the same wave, so the weight tile
    // comes from DRAM once and the other batch tiles hit L2 (with batch tiles in grid.z every wave re-read the matrix:
    // dram__bytes_read was 2x the weights at 256 rows, profiles/r02_ncu_top_kernels.md)
    // (decode steps with <= 128 rows have ONE batch tile: no division on their prologue path)
    const int tile = a.mtiles == 1 ? (int)blockIdx.x : (int)blockIdx.x / a.mtiles, row0 = tile * 128;
    const int m0 = a.mtiles == 1 ? 0 : ((int)blockIdx.x % a.mtiles) * MB;
    const int cta_id = (int)blockIdx.x * KS + rank;
    const int kb0 = rank * a.kb_per_cta;
    const int nk = max(0, min(a.n_kb, kb0 + a.kb_per_cta) - kb0);

    // which weight matrix holds this row tile (q | k | v segments, or gate + up)
    const CUtensorMap* mapA = &tmA;
    int arow = row0;
    if (EPI != EPI_SWIGLU) {
        if (row0 >= seg1) { mapA = &tmA3; arow = row0 - seg1; }
        else if (row0 >= seg0) { mapA = &tmA2; arow = row0 - seg0; }
    }

    if (warp == 1 && lane == 0) {
        for (int s = 0; s < S; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
        mbar_init(accum, 1);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    if (warp == 2) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" ::"r"(smem_u32(tmem_slot)),
                     "n"(C::TMEM_COLS));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    int M_pre = a.m_max;
    float nw_pre = 1.f;
    if (warp == 0) {
        // ===== TMA producer =====
        if (lane == 0) {
            tma_prefetch_desc(mapA);
            tma_prefetch_desc(&tmB);
            if (EPI == EPI_SWIGLU) tma_prefetch_desc(&tmA2);
            // weights never depend on the upstream kernel: fill the ring's A halves before the PDL wait
            const int pre = min(S, nk);
            for (int i = 0; i < pre; ++i) {
                uint8_t* st = smem + i * C::STAGE;
                mbar_expect_tx(&full[i], C::STAGE);
                tma_load_2d(st, mapA, &full[i], (kb0 + i) * TC_BK, arow);
                if (EPI == EPI_SWIGLU) tma_load_2d(st + C::A_BYTES, &tmA2, &full[i], (kb0 + i) * TC_BK, arow);
            }
            trace_mark(5 * 4); pdl_wait(); trace_mark(5 * 4 + 1);
            for (int i = 0; i < pre; ++i)
                tma_load_2d(smem + i * C::STAGE + NA * C::A_BYTES, &tmB, &full[i], (kb0 + i) * TC_BK, 2 * m0);
            for (int i = pre; i < nk; ++i) {
                const int s = i % S;
                mbar_wait(&empty[s], ((i / S) - 1) & 1);
                uint8_t* st = smem + s * C::STAGE;
                mbar_expect_tx(&full[s], C::STAGE);
                tma_load_2d(st, mapA, &full[s], (kb0 + i) * TC_BK, arow);
                if (EPI == EPI_SWIGLU) tma_load_2d(st + C::A_BYTES, &tmA2, &full[s], (kb0 + i) * TC_BK, arow);
                tma_load_2d(st + NA * C::A_BYTES, &tmB, &full[s], (kb0 + i) * TC_BK, 2 * m0);
            }
        }
        trace_mark(8 * 4 + 0);
        pdl_launch();
    } else if (warp == 1) {
        // ===== MMA issuer =====
        pdl_launch();
        const uint32_t idesc = umma_idesc(NB);
        for (int i = 0; i < nk; ++i) {
            const int s = i % S;
            mbar_wait(&full[s], (i / S) & 1);
            tc_fence_after();
            if (lane == 0) {
                const uint32_t sa = smem_u32(smem + s * C::STAGE);
                const uint64_t bdesc = umma_desc_sw128(sa + NA * C::A_BYTES);
#pragma unroll
                for (int na = 0; na < NA; ++na) {
                    const uint64_t adesc = umma_desc_sw128(sa + na * C::A_BYTES);
#pragma unroll
                    for (int k = 0; k < TC_BK / 16; ++k)
                        tc_mma(tmem_base + na * NB, adesc + 2 * k, bdesc + 2 * k, idesc, (i > 0 || k > 0) ? 1u : 0u);
                }
                tc_commit(&empty[s]);                 // frees the stage once these MMAs have read it
                if (i == nk - 1) tc_commit(accum);    // accumulator complete
            }
            __syncwarp();
        }
    } else {
        // ===== epilogue warps: TMEM -> (hi + lo) -> shared reduce buffer =====
        const int lg = warp & 3;                      // TMEM lane group of this warp
        const int row = lg * 32 + lane;
        // everything the final epilogue needs that does not depend on the accumulator is fetched now,
        // off the critical path: the next norm's gain (a weight: even before the dependency wait) and the live count
        if (EPI == EPI_RESID && a.norm_next != nullptr) nw_pre = bf16_to_f32(a.norm_next[row0 + row]);
        pdl_wait();
        pdl_launch();
        M_pre = a.m_dev ? min(*a.m_dev, a.m_max) : a.m_max;
        const int et = (warp - 2) * 32 + lane;        // 0..127
        if (a.ssq_in != nullptr) {
            for (int m = et; m < MB; m += 128) {
                float t = 0.f;
                for (int i = 0; i < a.ssq_in_tiles; ++i) t += a.ssq_in[(size_t)i * a.ssq_ld + m0 + m];
                rstd_s[m] = rsqrtf(t / (float)a.k_norm + a.eps);
            }
        }
        if (nk > 0) {
            mbar_wait(accum, 0);
            tc_fence_after();
        }
        trace_mark_thread(8 * 4 + 1, 64);
        if (C::PUSH_OK && KS > 1) {
            switch (KS) {
                case 2: tc_drain<NB, NA, 2>(a, cluster, red, recv, tmem_base, lg, row, rank, cta_id, nk > 0); break;
                case 4: tc_drain<NB, NA, 4>(a, cluster, red, recv, tmem_base, lg, row, rank, cta_id, nk > 0); break;
                default: tc_drain<NB, NA, 8>(a, cluster, red, recv, tmem_base, lg, row, rank, cta_id, nk > 0); break;
            }
        } else {
#pragma unroll
            for (int na = 0; na < NA; ++na) {
#pragma unroll
                for (int c = 0; c < NB / 32; ++c) {
                    float v[32];
                    if (nk > 0) {
                        tc_ld32(tmem_base + ((uint32_t)(lg * 32) << 16) + (uint32_t)(na * NB + c * 32), v);
                    } else {
#pragma unroll
                        for (int j = 0; j < 32; ++j) v[j] = 0.f;
                    }
                    if (KS == 1) {
#pragma unroll
                        for (int j = 0; j < 16; ++j) red[((size_t)na * MB + c * 16 + j) * 128 + row] = v[2 * j] + v[2 * j + 1];
                    } else {      // large partial tiles go through the L2 scratch
                        float* mine = a.scratch + (size_t)cta_id * (NA * MB * 128);
#pragma unroll
                        for (int j = 0; j < 16; ++j) __stcg(mine + ((size_t)na * MB + c * 16 + j) * 128 + row, v[2 * j] + v[2 * j + 1]);
                    }
                }
            }
        }
        tc_fence_before();
        trace_mark_thread(8 * 4 + 2, 64);
    }
    // every rank's partial tile is now in the L2 scratch (KS > 1) or in this CTA's shared memory (KS == 1);
    // all tcgen05.ld of this CTA have completed, so the TMEM columns can go back right away
    if (KS > 1) cluster.sync(); else __syncthreads();
    trace_mark_thread(8 * 4 + 3, 64);
    if (warp == 2) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(tmem_base), "n"(C::TMEM_COLS));
    }
    if (warp >= 2) {
        switch (KS) {
            case 1: tc_epilogue<NB, EPI, 1>(a, red, rstd_s, ssq_s, exch, recv, warp, lane, row0, m0, tile, rank, cta_id, M_pre, nw_pre); break;
            case 2: tc_epilogue<NB, EPI, 2>(a, red, rstd_s, ssq_s, exch, recv, warp, lane, row0, m0, tile, rank, cta_id, M_pre, nw_pre); break;
            case 4: tc_epilogue<NB, EPI, 4>(a, red, rstd_s, ssq_s, exch, recv, warp, lane, row0, m0, tile, rank, cta_id, M_pre, nw_pre); break;
            default: tc_epilogue<NB, EPI, 8>(a, red, rstd_s, ssq_s, exch, recv, warp, lane, row0, m0, tile, rank, cta_id, M_pre, nw_pre); break;
        }
    }
    // no second cluster barrier: peers read this CTA's partials from the L2 scratch, never from its
    // shared memory, so the CTA may retire as soon as its own columns are written
    trace_mark_thread(9 * 4 + 2, 64);
}

// ---- x fp32 [M][K] -> pre-split rows (test / debug entry and embedding path) ---------------
__global__ void k_split_rows(const float* __restrict__ x, int K, const int* m_dev, int m_max, bf16_t* __restrict__ xs) {
    const int M = m_dev ? min(*m_dev, m_max) : m_max;
    const int m = blockIdx.x;
    if (m >= M) return;
    for (int k = threadIdx.x; k < K; k += blockDim.x) {
        const float v = x[(size_t)m * K + k];
        const uint32_t hi = f32_to_bf16_bits(v);
        xs[(size_t)(2 * m) * K + k] = (bf16_t)hi;
        xs[(size_t)(2 * m + 1) * K + k] = (bf16_t)f32_to_bf16_bits(v - __uint_as_float(hi << 16));
    }
}
int launch_split_rows(const float* x, int K, const int* m_dev, int m_max, bf16_t* xs, cudaStream_t st) {
    if (m_max <= 0) return 0;
    k_split_rows<<<m_max, 256, 0, st>>>(x, K, m_dev, m_max, xs);
    return 1;
}

// ---- host: tensor maps ---------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn get_encode_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}
// bf16 matrix [rows][K] row-major; box = 64 (k) x box_rows, 128-byte swizzle
int tc_make_map(TcMap* out, const void* base, long long rows, int K, int box_rows) {
    EncodeTiledFn fn = get_encode_fn();
    if (!fn) return -1;
    static_assert(sizeof(TcMap) == sizeof(CUtensorMap), "TcMap must mirror CUtensorMap");
    cuuint64_t dims[2] = {(cuuint64_t)K, (cuuint64_t)rows};
    cuuint64_t strides[1] = {(cuuint64_t)K * 2};
    cuuint32_t box[2] = {(cuuint32_t)TC_BK, (cuuint32_t)box_rows};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = fn(reinterpret_cast<CUtensorMap*>(out), CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims,
                    strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                    CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? 0 : -1;
}

template <int NB, int EPI>
static cudaError_t launch_tc_inst(const TcLinearArgs& t, const TcDev& d, dim3 grid, int KS, cudaStream_t st) {
    constexpr int NA = (EPI == EPI_SWIGLU) ? 2 : 1;
    using C = TcCfg<NB, NA>;
    // grids that fit the chip in one wave get the deepest ring; multi-wave grids (LM head, prefill) keep
    // ~100 KB so two CTAs share an SM and one's epilogue overlaps the other's loads
    const bool one_wave = (long long)grid.x * grid.y * grid.z <= g_num_sms;
    // wide batch tiles (UMMA N = 256) are throughput-bound per CTA: give them the deepest ring as well
    const int stages = (one_wave || NB == 256) ? C::MAXSTAGES : C::STAGES;
    // (asking for MORE shared memory than the ring needs, so that PDL successors cannot become co-resident, helps the attention
    // kernel -- attention.cu -- and changes nothing here: 18 758 / 18 779 / 18 776 tokens/s for +0 / 116 / 160 KB.)
    const int smem = C::smem_bytes(stages, EPI == EPI_QKV);
    TcDev d2 = d; d2.stages = stages;
    {   // per launch: a per-process flag would miss a second device
        cudaError_t e = cudaFuncSetAttribute(k_linear_tc<NB, EPI>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             C::smem_bytes(C::MAXSTAGES, EPI == EPI_QKV));
        if (e != cudaSuccess) return e;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = dim3(TC_THREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[2];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = 1; at[0].val.clusterDim.y = KS; at[0].val.clusterDim.z = 1;
    at[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[1].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = t.pdl ? 2 : 1;
    const CUtensorMap* a0 = reinterpret_cast<const CUtensorMap*>(t.a[0]);
    const CUtensorMap* a1 = reinterpret_cast<const CUtensorMap*>(t.a[1] ? t.a[1] : t.a[0]);
    const CUtensorMap* a2 = reinterpret_cast<const CUtensorMap*>(t.a[2] ? t.a[2] : t.a[0]);
    const CUtensorMap* b = reinterpret_cast<const CUtensorMap*>(t.b);
    const int seg0 = t.a[1] ? t.seg_rows[0] : t.N + 128;
    const int seg1 = t.a[2] ? t.seg_rows[0] + t.seg_rows[1] : t.N + 128;
    return cudaLaunchKernelEx(&cfg, k_linear_tc<NB, EPI>, *a0, *a1, *a2, *b, seg0, seg1, d2);
}

int tc_nb_index(int m_max) { return m_max <= 16 ? 0 : (m_max <= 32 ? 1 : (m_max <= 64 ? 2 : 3)); }

int tc_plan(int N, int K, int m_max, bool swiglu, bool has_scratch, int* kb_per_cta) {
    const int nbi = tc_nb_index(m_max);
    const int MB = (32 << nbi) / 2;
    const int tiles = N / 128, mtiles = (m_max + MB - 1) / MB, n_kb = K / TC_BK;
    // K-split policy (measured with the in-kernel timeline): a CTA streams its weight slab through a deep
    // TMA ring at well over 150 GB/s, while every extra cluster rank adds DSMEM round trips to the
    // epilogue -- so K is split down to ~30 KB slabs per CTA (swept on cfg2), in powers of two up to 8, and never beyond two CTAs per SM.
    const double slab = (swiglu ? 2.0 : 1.0) * 128.0 * K * 2.0;
    const double slab_max = 30.0e3;
    int KS = (int)((slab + slab_max - 1) / slab_max);
    const int room = (2 * g_num_sms) / (tiles * mtiles);
    if (KS > room) KS = room;
    if (KS < 1) KS = 1;
    if (KS > 8) KS = 8;     // cap re-swept in round 2 (decode step, cap 8 / 4 / 2): 1.5B 1.42 / - / 1.80 ms, 7B 3.35 / 3.60 / 5.06 ms
    if (KS > n_kb) KS = n_kb;
    if (!has_scratch) KS = 1;
    { int p2 = 1; while (p2 * 2 <= KS) p2 *= 2; KS = p2; }      // the epilogue is specialised for 1, 2, 4, 8
    if (kb_per_cta) *kb_per_cta = (n_kb + KS - 1) / KS;            // trailing ranks may get fewer (or zero) k blocks
    return KS;
}

int launch_linear_tc(const TcLinearArgs& t, cudaStream_t st) {
    if (t.m_max <= 0) return 0;
    TcDev d;
    d.K = t.K; d.N = t.N; d.n_kb = t.K / TC_BK; d.m_dev = t.m_dev; d.m_max = t.m_max; d.Y = t.Y; d.ldy = t.ldy; d.R = t.R;
    d.xs_out = t.xs_out; d.ld_xs = t.ld_xs; d.norm_next = t.norm_next; d.ssq_out = t.ssq_out; d.ssq_in = t.ssq_in;
    d.ssq_in_tiles = t.ssq_in_tiles; d.ssq_ld = t.ssq_ld; d.eps = t.eps; d.k_norm = t.k_norm; d.scratch = t.scratch;
    d.rope_cs = t.rope_cs; d.row_pos = t.row_pos; d.row_sid = t.row_sid; d.page_table = t.page_table; d.kv_layer = t.kv_layer;
    d.max_blocks = t.max_blocks; d.page = t.page; d.Hkv = t.Hkv; d.hd = t.hd; d.q_rows = t.q_rows; d.kv_rows = t.kv_rows;
    const int nbi = tc_nb_index(t.m_max);
    const int NB = 32 << nbi, MB = NB / 2;
    const int tiles = t.N / 128, mtiles = (t.m_max + MB - 1) / MB;
    if ((size_t)2 * g_num_sms * 2 * 128 * 128 > TC_SCRATCH_FLOATS) return -1;      // split-K scratch is sized for 296 CTAs
    const int KS = tc_plan(t.N, t.K, t.m_max, t.epi == EPI_SWIGLU, t.scratch != nullptr, &d.kb_per_cta);
    d.mtiles = mtiles;
    dim3 grid(tiles * mtiles, KS, 1);
    cudaError_t e;
#define TC_CASE(NBV)                                                                         \
    case NBV:                                                                                \
        if (t.epi == EPI_SWIGLU) e = launch_tc_inst<NBV, EPI_SWIGLU>(t, d, grid, KS, st);    \
        else if (t.epi == EPI_RESID) e = launch_tc_inst<NBV, EPI_RESID>(t, d, grid, KS, st); \
        else if (t.epi == EPI_QKV) e = launch_tc_inst<NBV, EPI_QKV>(t, d, grid, KS, st);     \
        else e = launch_tc_inst<NBV, EPI_STORE>(t, d, grid, KS, st);                         \
        break;
    switch (NB) {
        TC_CASE(32)
        TC_CASE(64)
        TC_CASE(128)
        default:
        TC_CASE(256)
    }
#undef TC_CASE
    return e == cudaSuccess ? 1 : -1;
}


// =============================================================================================
// k_lmhead_sample -- final norm + LM head + sampler in ONE persistent kernel (steps a11 + a12; SURVEY
// 8(a): "fuse with a12 so logits [M][V] fp32 never hit HBM").  One CTA per SM walks the vocabulary
// tiles  blockIdx.x, blockIdx.x + gridDim.x, ...: the TMA ring runs ahead across tile boundaries and the
// accumulator is double-buffered in TMEM, so the epilogue of tile j (TMEM -> logit -> Philox Gumbel
// perturbation -> running arg-max in registers) overlaps the weight stream of tile j+1.  Each CTA
// writes ONE (score, token) candidate per batch row; k_advance takes the best of the gridDim.x
// candidates (ties: lowest token id, the comparator is order-independent).
// Philox block (v >> 2, t, sid) is shared by the four lanes that hold vocab ids 4b..4b+3: lane q of the
// quad computes the block of batch row m0 + q and the words are exchanged by shuffles, so no block is
// computed twice.  Accumulator slot x of a quad therefore holds batch row m0 + (x ^ q) (undone at the end).
// =============================================================================================
struct LmDev {
    int n_kb, tiles, V;
    const int* m_dev; int m_max;
    const float* ssq_in; int ssq_in_tiles, ssq_ld; float eps; int k_norm;
    int stages;
    int bres;                                           // activations (all k blocks) stay resident in shared memory
    const int* row_sid; const int* step_dev; const uint32_t* params;
    float* part_score; int* part_tok; int part_ld;      // [gridDim.x][part_ld]
    float* Y; int ldy;                                  // optional logits dump (parity / debugging), may be null
};

template <typename T>
__device__ __forceinline__ T sel4(T a0, T a1, T a2, T a3, int i) {
    const T lo = (i & 1) ? a1 : a0, hi = (i & 1) ? a3 : a2;
    return (i & 2) ? hi : lo;
}

static constexpr int LM_EPI_THREADS = 256;                    // 8 epilogue warps
static constexpr int LM_THREADS = 64 + LM_EPI_THREADS;       // + TMA producer warp + MMA issuer warp

template <int NB>
__global__ void __launch_bounds__(LM_THREADS, 1)
k_lmhead_sample(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, LmDev a) {
    constexpr int MB = NB / 2;
    constexpr int A_BYTES = 128 * 128, STAGE = A_BYTES + NB * 128;
    constexpr int B_BYTES = NB * 128;
    const int S = a.stages;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    // bres: [n_kb activation tiles, loaded once][ring of weight-only stages]; else: ring of (weight + activation) stages.
    // The activation tile of a k block is the same for every vocabulary tile: keeping it resident removes it from the
    // per-stage L2 -> SM traffic (a quarter of it at UMMA N = 32, a third at N = 64).
    const int stage_sz = a.bres ? A_BYTES : STAGE;
    uint8_t* ring = smem + (a.bres ? a.n_kb * B_BYTES : 0);
    uint64_t* full = reinterpret_cast<uint64_t*>(ring + S * stage_sz);
    uint64_t* empty = full + S;
    uint64_t* tfull = empty + S;           // [2] accumulator slot complete
    uint64_t* tempty = tfull + 2;          // [2] accumulator slot drained by the eight epilogue warps
    uint64_t* bfull = tempty + 2;          // resident activations landed (bres)
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bfull + 1);
    float* rstd_s = reinterpret_cast<float*>(ring + S * stage_sz + 512);
    int* sid_s = reinterpret_cast<int*>(rstd_s + MB);
    float* red_sc = reinterpret_cast<float*>(smem);            // [MB][128] final reduction, overlays the ring
    int* red_ix = reinterpret_cast<int*>(red_sc + MB * 128);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_my = (a.tiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;    // tiles of this CTA
    const int total = n_my * a.n_kb;

    if (warp == 1 && lane == 0) {
        for (int s = 0; s < S; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
        for (int s = 0; s < 2; ++s) { mbar_init(&tfull[s], 1); mbar_init(&tempty[s], LM_EPI_THREADS / 32); }
        mbar_init(bfull, 1);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    if (warp == 2) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" ::"r"(smem_u32(tmem_slot)), "n"(2 * NB));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    if (warp == 0) {
        // ===== TMA producer: one flat iteration space over (tile, k block) =====
        if (lane == 0) {
            tma_prefetch_desc(&tmA);
            tma_prefetch_desc(&tmB);
            const int pre = min(S, total);
            for (int i = 0; i < pre; ++i) {       // weights never depend on the upstream kernel
                const int tile = (int)blockIdx.x + (i / a.n_kb) * (int)gridDim.x, kb = i % a.n_kb;
                mbar_expect_tx(&full[i], stage_sz);
                tma_load_2d(ring + i * stage_sz, &tmA, &full[i], kb * TC_BK, tile * 128);
            }
            pdl_wait();
            if (a.bres) {
                mbar_expect_tx(bfull, a.n_kb * B_BYTES);
                for (int kb = 0; kb < a.n_kb; ++kb) tma_load_2d(smem + kb * B_BYTES, &tmB, bfull, kb * TC_BK, 0);
            } else {
                for (int i = 0; i < pre; ++i) tma_load_2d(ring + i * STAGE + A_BYTES, &tmB, &full[i], (i % a.n_kb) * TC_BK, 0);
            }
            for (int i = pre; i < total; ++i) {
                const int s = i % S;
                const int tile = (int)blockIdx.x + (i / a.n_kb) * (int)gridDim.x, kb = i % a.n_kb;
                mbar_wait(&empty[s], ((i / S) - 1) & 1);
                mbar_expect_tx(&full[s], stage_sz);
                tma_load_2d(ring + s * stage_sz, &tmA, &full[s], kb * TC_BK, tile * 128);
                if (!a.bres) tma_load_2d(ring + s * STAGE + A_BYTES, &tmB, &full[s], kb * TC_BK, 0);
            }
        }
        pdl_launch();
    } else if (warp == 1) {
        // ===== MMA issuer =====
        pdl_launch();
        const uint32_t idesc = umma_idesc(NB);
        int i = 0;
        if (a.bres) { mbar_wait(bfull, 0); tc_fence_after(); }
        for (int j = 0; j < n_my; ++j) {
            const int slot = j & 1, use = j >> 1;
            if (use > 0) { mbar_wait(&tempty[slot], (use - 1) & 1); tc_fence_after(); }
            for (int kb = 0; kb < a.n_kb; ++kb, ++i) {
                const int s = i % S;
                mbar_wait(&full[s], (i / S) & 1);
                tc_fence_after();
                if (lane == 0) {
                    const uint32_t sa = smem_u32(ring + s * stage_sz);
                    const uint64_t adesc = umma_desc_sw128(sa);
                    const uint64_t bdesc = umma_desc_sw128(a.bres ? smem_u32(smem + kb * B_BYTES) : sa + A_BYTES);
#pragma unroll
                    for (int k = 0; k < TC_BK / 16; ++k)
                        tc_mma(tmem_base + slot * NB, adesc + 2 * k, bdesc + 2 * k, idesc, (kb > 0 || k > 0) ? 1u : 0u);
                    tc_commit(&empty[s]);
                    if (kb == a.n_kb - 1) tc_commit(&tfull[slot]);
                }
                __syncwarp();
            }
        }
    } else {
        // ===== epilogue warps: logits -> perturbed scores -> running arg-max =====
        // Eight warps: TMEM lane group lg = warp % 4 is served by two warps (h = 0, 1) that split the batch
        // columns, so every SM sub-partition holds two independent instruction streams (the Philox / logf
        // chains are latency-bound in a single warp).
        constexpr int NCH = NB / 32;                  // 32-column TMEM chunks = 16 batch rows each
        constexpr int SLOTS = MB / 2;                 // batch rows per warp
        const int lg = warp & 3, row = lg * 32 + lane, q = lane & 3, h = (warp - 2) >> 2;
        pdl_wait();
        pdl_launch();
        const int M = a.m_dev ? min(*a.m_dev, a.m_max) : a.m_max;
        const int et = (warp - 2) * 32 + lane;        // 0..255
        for (int m = et; m < MB; m += LM_EPI_THREADS) {
            float t = 0.f;
            if (a.ssq_in != nullptr)
                for (int i = 0; i < a.ssq_in_tiles; ++i) t += a.ssq_in[(size_t)i * a.ssq_ld + m];
            rstd_s[m] = (a.ssq_in != nullptr) ? rsqrtf(t / (float)a.k_norm + a.eps) : 1.f;
            sid_s[m] = (m < M) ? a.row_sid[m] : 0;
        }
        const int mode = (int)a.params[0];
        const float inv_t = 1.f / __uint_as_float(a.params[1]);
        const uint32_t k0 = a.params[2], k1 = a.params[3];
        const uint32_t tstep = (uint32_t)*a.step_dev;
        asm volatile("bar.sync 1, 256;\n" ::: "memory");
        float bs[SLOTS];
        int bi[SLOTS];
#pragma unroll
        for (int m = 0; m < SLOTS; ++m) { bs[m] = -INFINITY; bi[m] = 0x7fffffff; }
        for (int j = 0; j < n_my; ++j) {
            const int slot = j & 1;
            const int v = ((int)blockIdx.x + j * (int)gridDim.x) * 128 + row;      // this thread's vocab id in tile j
            mbar_wait(&tfull[slot], (j >> 1) & 1);
            tc_fence_after();
#pragma unroll
            for (int ci = 0; ci < (NCH == 1 ? 1 : NCH / 2); ++ci) {
                const int c = (NCH == 1) ? 0 : 2 * ci + h;                 // this warp's chunk
                const int g_lo = (NCH == 1) ? 2 * h : 0;                   // and its quads of 4 batch rows
                constexpr int NG = (NCH == 1) ? 2 : 4;
                const bool live = (c * 16 + 4 * g_lo) < M;                 // warp-uniform
                float acc[32];
                if (live) tc_ld32(tmem_base + ((uint32_t)(lg * 32) << 16) + (uint32_t)(slot * NB + c * 32), acc);
                if (ci == (NCH == 1 ? 1 : NCH / 2) - 1) {                  // slot drained by this warp
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&tempty[slot]);
                }
                if (!live) continue;
                float L[4 * NG];
#pragma unroll
                for (int i = 0; i < 4 * NG; ++i) {
                    float sum = acc[2 * i] + acc[2 * i + 1];
                    if constexpr (NCH == 1) {         // the warp's columns start at 8 * h (h is runtime: select, static indices)
                        const float hi = acc[2 * (i + 8)] + acc[2 * (i + 8) + 1];
                        sum = h ? hi : sum;
                    }
                    L[i] = sum * rstd_s[c * 16 + 4 * g_lo + i];
                }
                if (a.Y != nullptr) {
#pragma unroll
                    for (int i = 0; i < 4 * NG; ++i) {
                        const int mrow = c * 16 + 4 * g_lo + i;
                        if (mrow < M) a.Y[(size_t)mrow * a.ldy + v] = L[i];
                    }
                }
                uint32_t W[NG][4];
                if (mode == 1) {
#pragma unroll
                    for (int g = 0; g < NG; ++g)      // independent Philox chains: no early exit between them
                        philox4x32_10((uint32_t)v >> 2, tstep, (uint32_t)sid_s[c * 16 + 4 * (g_lo + g) + q], 0u, k0, k1, W[g]);
                }
#pragma unroll
                for (int g = 0; g < NG; ++g) {
#pragma unroll
                    for (int x = 0; x < 4; ++x) {
                        const int mm = q ^ x;                                  // batch row (quad base) + mm sits in slot x
                        float sc = sel4(L[4 * g], L[4 * g + 1], L[4 * g + 2], L[4 * g + 3], mm);
                        if (mode == 1) {
                            // lane q' = q ^ x computed the block of row base + q'; this lane needs its word q
                            const uint32_t send = sel4(W[g][0], W[g][1], W[g][2], W[g][3], mm);
                            const uint32_t w = (x == 0) ? send : __shfl_xor_sync(0xffffffffu, send, x);
                            sc = fmaf(sc, inv_t, gumbel_from_u32(w));
                        }
                        const int sl = ci * 16 + 4 * g + x;
                        if (sc > bs[sl]) { bs[sl] = sc; bi[sl] = v; }          // tiles ascend: strict > keeps the lowest id
                    }
                }
            }
        }
        // ---- best over the 128 vocabulary lanes of this CTA, one candidate per batch row ----
        // (the last tfull wait implies every MMA has finished reading the ring: safe to overlay)
        asm volatile("bar.sync 1, 256;\n" ::: "memory");
#pragma unroll
        for (int sl = 0; sl < SLOTS; ++sl) {
            const int ci = sl >> 4, r4 = sl & 15;
            const int base = (NCH == 1) ? 8 * h + (r4 & ~3) : (2 * ci + h) * 16 + (r4 & ~3);
            const int mt = base + ((r4 & 3) ^ q);
            red_sc[mt * 128 + row] = bs[sl];
            red_ix[mt * 128 + row] = bi[sl];
        }
        asm volatile("bar.sync 1, 256;\n" ::: "memory");
        if (et < MB && et < M) {
            float b = -INFINITY;
            int ix = 0x7fffffff;
#pragma unroll 8
            for (int i = 0; i < 128; ++i) {
                const int r = (i + et) & 127;
                const float s2 = red_sc[et * 128 + r];
                const int i2 = red_ix[et * 128 + r];
                if (s2 > b || (s2 == b && i2 < ix)) { b = s2; ix = i2; }
            }
            a.part_score[(size_t)blockIdx.x * a.part_ld + et] = b;
            a.part_tok[(size_t)blockIdx.x * a.part_ld + et] = ix;
        }
        tc_fence_before();
    }
    __syncthreads();
    if (warp == 2) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(tmem_base), "n"(2 * NB));
    }
}

template <int NB>
static cudaError_t launch_lm_inst(const LmSampleArgs& t, LmDev d, int grid, cudaStream_t st) {
    constexpr int A_BYTES = 128 * 128, B_BYTES = NB * 128, STAGE = A_BYTES + B_BYTES;
    // SAGC_LM_BRES: 0 = activation tile re-fetched with every stage, 1 = resident at UMMA N = 32, 2 = also at N = 64
    // (only when at least four weight stages still fit beside it)
    constexpr int bres_knob = 0;        // resident activation tiles: measured no gain, kept for reference
    const int b_all = d.n_kb * B_BYTES;
    const bool want = (bres_knob >= 1 && NB == 32) || (bres_knob >= 2 && NB == 64);
    d.bres = (want && b_all + 4 * A_BYTES <= 196 * 1024) ? 1 : 0;
    int stages = d.bres ? (196 * 1024 - b_all) / A_BYTES : (196 * 1024) / STAGE;
    if (stages > 10) stages = 10;
    d.stages = stages;
    const int smem = (d.bres ? b_all + stages * A_BYTES : stages * STAGE) + 512 + (NB / 2) * 8 + 1024;
    {
        cudaError_t e = cudaFuncSetAttribute(k_lmhead_sample<NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        if (e != cudaSuccess) return e;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(LM_THREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = t.pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, k_lmhead_sample<NB>, *reinterpret_cast<const CUtensorMap*>(t.a),
                              *reinterpret_cast<const CUtensorMap*>(t.b), d);
}

// best of the per-CTA candidates (debug entry; in a rollout k_advance does this)
__global__ void k_pick_candidates(const float* part_score, const int* part_tok, int n_parts, int ld, int M, int* out_tok) {
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= M) return;
    float b = part_score[m];
    int ix = part_tok[m];
    for (int c = 1; c < n_parts; ++c) {
        const float s2 = part_score[(size_t)c * ld + m];
        const int i2 = part_tok[(size_t)c * ld + m];
        if (s2 > b || (s2 == b && i2 < ix)) { b = s2; ix = i2; }
    }
    out_tok[m] = ix;
}
int launch_pick_candidates(const float* part_score, const int* part_tok, int n_parts, int ld, int M, int* out_tok, cudaStream_t st) {
    k_pick_candidates<<<1, 64, 0, st>>>(part_score, part_tok, n_parts, ld, M, out_tok);
    return 1;
}

int lm_sample_grid(int V) {
    const char* e = getenv("SAGC_LM_CTAS");          // read per call (graph build time): tests force several tiles per CTA
    const int g = (e && atoi(e) > 0) ? atoi(e) : g_num_sms;
    const int tiles = V / 128;
    return tiles < g ? tiles : (g > LM_MAX_PARTS ? LM_MAX_PARTS : g);
}

int launch_lmhead_sample(const LmSampleArgs& t, cudaStream_t st) {
    if (t.m_max <= 0) return 0;
    if (t.m_max > 64 || (t.V % 128) != 0 || (t.K % TC_BK) != 0) return -1;
    LmDev d;
    d.n_kb = t.K / TC_BK; d.tiles = t.V / 128; d.V = t.V; d.m_dev = t.m_dev; d.m_max = t.m_max; d.ssq_in = t.ssq_in;
    d.ssq_in_tiles = t.ssq_in_tiles; d.ssq_ld = t.ssq_ld; d.eps = t.eps; d.k_norm = t.k_norm; d.stages = 0;
    d.row_sid = t.row_sid; d.step_dev = t.step_dev; d.params = t.params; d.part_score = t.part_score; d.part_tok = t.part_tok;
    d.part_ld = t.part_ld; d.Y = t.Y; d.ldy = t.ldy;
    const int grid = lm_sample_grid(t.V);
    cudaError_t e;
    switch (tc_nb_index(t.m_max)) {
        case 0: e = launch_lm_inst<32>(t, d, grid, st); break;
        case 1: e = launch_lm_inst<64>(t, d, grid, st); break;
        default: e = launch_lm_inst<128>(t, d, grid, st); break;
    }
    return e == cudaSuccess ? 1 : -1;
}

}  // namespace sagc
