// decode_step.cu -- ONE persistent kernel for the whole layer stack of a decode step (steps a5-a10 of
// DESIGN.md; <= 64 live rows): embedding + per layer { QKV | RoPE + KV append + paged attention | O + residual |
// gate/up + SwiGLU | down + residual } + the operand of the LM head.  One CTA per SM; kernel boundaries are
// replaced by grid-wide arrive/poll counters in L2, and -- the point of the exercise -- the weight stream never
// stops at them:
//
//   warp 0   A producer : walks this CTA's static work list (every layer, every GEMM phase) and TMA-loads the
//                         128 x 64 bf16 weight tiles into a ring of 16 KB slots.  Weights depend on nothing,
//                         so it runs as far ahead as the ring allows, across phase and layer boundaries.
//   warp 1   MMA issuer : tcgen05.mma (weights = A, M = 128; activations = B, N = 2 x batch), fp32 in TMEM.
//   warp 2   owns the TMEM allocation; warp 3 idle.
//   warps 4-11 workers  : build the activation operand of their unit in shared memory (hi/lo bf16 split, 128-byte
//                         swizzle, RMSNorm gain / SwiGLU fused), drain the accumulators, run the attention units
//                         (attention_body.cuh), the per-row bookkeeping (residual stream, 1/rms) and the embedding.
//
// Data flow between phases (what makes a phase boundary ONE L2 round trip): a GEMM phase never stores finished
// activations.  Every unit (128-row weight tile x k range; K is split so that every SM streams a share of every
// matrix) adds its partial products to a 64-bit FIXED-POINT accumulator in L2 (value * 2^32, red.add.u64: integer
// addition is associative, so the sum is bit-reproducible whatever the arrival order).  The consumer of the next
// phase reads the finished sums of exactly the k columns its own unit needs, applies what sits between the two GEMMs
// (residual + norm gain, or SwiGLU) and writes the hi/lo bf16 operand tile straight into its shared memory.
// 1/rms is a per-row scalar: it is computed on the side by the CTA that owns the row (which also carries the fp32
// residual stream forward) and applied one phase later (attention scales q, k, v; the down projection scales gate
// and up), so it is never on the critical path.
#include <cuda.h>

#include <algorithm>
#include <cstdlib>
#include <vector>

#include "attention_body.cuh"
#include "common.cuh"
#include "kernels.cuh"
#include "tc_ptx.cuh"

namespace sagc {

static constexpr int STEP_THREADS = 384;
static constexpr int STEP_SLOT = 16384;                  // ring slot: one 128 x 64 bf16 weight tile
static constexpr int STEP_ATT_BYTES = 65536;             // K/V staging of the attention units; GEMM phases: 2 x 32 KB B buffers
static constexpr int STEP_BBUF = 32768;
static constexpr int STEP_MISC = 3072;                   // barriers, plan copy, small scratch
static constexpr unsigned long long STEP_WATCHDOG_NS = 4000000000ull;
static constexpr float FX_SCALE = 4294967296.f;          // 2^32
static constexpr float FX_INV = 2.3283064365386963e-10f; // 2^-32

// attention geometry inside the step kernel: 64 KB of K/V staging either way
template <int HD> struct StepAtt { static constexpr int WARPS = 4; static constexpr int NSTAGE = HD >= 128 ? 2 : 4; };   // 64-token tiles

struct StepDev {
    int n_layers, n_cta, NB, n_slots, chunk;             // chunk = k blocks per B buffer = STEP_BBUF / (NB * 128)
    int prefetch;                        // k blocks the L2 prefetch runs ahead of the ring loads inside a unit (0 = off)
    StepGemm g[4];
    const CUtensorMap* wmaps;            // device [n_layers][7]: q k v o g u d (box 64 x 128)
    const StepPhasePlan* plan;           // device [4][n_cta]
    float* xa; float* xb;                // fp32 residual stream, ping-pong [64][d_model]
    long long* accQ; long long* accO; long long* accG; long long* accD;     // fixed-point sums [64][Nqkv | d | 2 d_ff | d]
    float* rstd1; float* rstd2;          // [64] 1/rms of the rows entering QKV / gate-up
    float* x; bf16_t* xs; float* ssq;    // LM-head operand (final residual rows, pre-split x * w_final, sums of squares)
    bf16_t* att_s;
    int ssq_ld, d_tiles, d_model, Nqkv, qd, d_ff;
    const bf16_t* const* norm1; const bf16_t* const* norm2; const bf16_t* final_norm; const bf16_t* embed;
    float eps;
    unsigned* sync_base; int gbar_n;     // [2][gbar_n] phase counters, double-buffered by step parity
    const int* live; const int* pos; const int* ctx; const int* tok; const int* n_live; const int* step; int m_max;
    AttnArgs att; bf16_t* kv_pool; size_t layer_stride;
    int* err;
    int flags;                           // experiment knobs (SAGC_STEP_FLAGS), see launch_decode_step
    unsigned long long* trace;           // optional timeline: [0] = step to record, [1] = event count, then (tag, ns) pairs
};

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];\n" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void red_release_add(unsigned* p, unsigned v) {
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;\n" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void red_add_fx(long long* p, float v) {
    const long long q = __float2ll_rn(v * FX_SCALE);
    asm volatile("red.relaxed.gpu.global.add.u64 [%0], %1;\n" ::"l"(p), "l"(q) : "memory");
}
__device__ __forceinline__ float fx_to_f32(long long v) { return __ll2float_rn(v) * FX_INV; }
__device__ __forceinline__ unsigned long long globaltimer_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;\n" : "=l"(t));
    return t;
}
// a wait that can never end (lost arrival, bad tensor map) must not hang the GPU: record and trap
__device__ __noinline__ void step_die(int* err, int code) {
    atomicExch(err, code);
    __threadfence_system();
    __trap();
}
__device__ __forceinline__ void step_wait_mbar(uint64_t* bar, uint32_t parity, int* err, int code) {
    if (mbar_try(bar, parity)) return;
    const unsigned long long t0 = globaltimer_ns();
    unsigned n = 0;
    while (!mbar_try(bar, parity))
        if (((++n) & 255u) == 0 && globaltimer_ns() - t0 > STEP_WATCHDOG_NS) step_die(err, code);
}
__device__ __forceinline__ void step_wait_count(const unsigned* ctr, unsigned target, int* err, int code) {
    if (ld_acquire_u32(ctr) >= target) return;
    const unsigned long long t0 = globaltimer_ns();
    unsigned n = 0;
    while (ld_acquire_u32(ctr) < target)
        if (((++n) & 1023u) == 0 && globaltimer_ns() - t0 > STEP_WATCHDOG_NS) step_die(err, code);
}
// optional timeline (SAGC_STEP_TRACE=1): CTA 0 and the last CTA record (role, event, phase) stamps of one chosen step
__device__ __forceinline__ void step_trace(const StepDev& a, bool on, int role, int ev, int p) {
    if (!on) return;
    const unsigned long long i = atomicAdd(a.trace + 1, 1ull);
    if (i < 16000) {
        a.trace[2 + 2 * i] = ((unsigned long long)blockIdx.x << 40) | ((unsigned long long)role << 32) | ((unsigned long long)ev << 16) | (unsigned long long)p;
        a.trace[3 + 2 * i] = globaltimer_ns();
    }
}
__device__ __forceinline__ void worker_sync() { asm volatile("bar.sync 1, 256;\n" ::: "memory"); }
__device__ __forceinline__ float silu_f(float z) { return z / (1.f + __expf(-z)); }

struct StepShared {                      // lives in the STEP_MISC region
    uint64_t full[12], empty[12], acc_full[2], bfull[2], bempty[2];
    uint32_t tmem_slot; int M, par, ns; unsigned ld_n;
    StepPhasePlan pl[4];
    float red[8];
    int ctx_max[8];
    float rstd[64];
};
static_assert(sizeof(StepShared) <= STEP_MISC, "StepShared outgrew its region");

// weight tensor map + row coordinate of a tile (QKV: three matrices back to back; gate/up: na selects)
__device__ __forceinline__ const CUtensorMap* step_wmap(const StepDev& a, const CUtensorMap* w7, int ph, int tile, int na, int& arow) {
    arow = tile * 128;
    if (ph == 0) {
        const int tq = a.g[0].seg0_tiles, tk = a.g[0].seg1_tiles;
        if (tile < tq) return &w7[0];
        if (tile < tq + tk) { arow = (tile - tq) * 128; return &w7[1]; }
        arow = (tile - tq - tk) * 128;
        return &w7[2];
    }
    if (ph == 1) return &w7[3];
    if (ph == 2) return &w7[4 + na];
    return &w7[6];
}

// 8 consecutive k of batch row m -> rows 2m (hi) and 2m+1 (lo) of a K-major, 128-byte-swizzled B tile of one k block
// (tile = NB rows x 128 B; 16-byte chunk c of row r sits at chunk c ^ (r & 7))
__device__ __forceinline__ void store_b_chunk(uint8_t* tile, int m, int c, const float (&v)[8]) {
    uint32_t hi[4], lo[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) split2(v[2 * i], v[2 * i + 1], hi[i], lo[i]);
    const int r0 = 2 * m, r1 = 2 * m + 1;
    *reinterpret_cast<uint4*>(tile + (size_t)r0 * 128 + ((c ^ (r0 & 7)) << 4)) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
    *reinterpret_cast<uint4*>(tile + (size_t)r1 * 128 + ((c ^ (r1 & 7)) << 4)) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
}
__device__ __forceinline__ void load_fx8(const long long* p, float (&o)[8]) {
    const longlong2* q = reinterpret_cast<const longlong2*>(p);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const longlong2 v = __ldcg(q + i);
        o[2 * i] = fx_to_f32(v.x);
        o[2 * i + 1] = fx_to_f32(v.y);
    }
}
__device__ __forceinline__ void load_f8(const float* p, float (&o)[8]) {
    const float4 a = __ldcg(reinterpret_cast<const float4*>(p)), b = __ldcg(reinterpret_cast<const float4*>(p + 4));
    o[0] = a.x; o[1] = a.y; o[2] = a.z; o[3] = a.w; o[4] = b.x; o[5] = b.y; o[6] = b.z; o[7] = b.w;
}
__device__ __forceinline__ void load_bf8(const bf16_t* p, float (&o)[8]) {
    const uint4 w = *reinterpret_cast<const uint4*>(p);
    o[0] = bf16lo_to_f32(w.x); o[1] = bf16hi_to_f32(w.x); o[2] = bf16lo_to_f32(w.y); o[3] = bf16hi_to_f32(w.y);
    o[4] = bf16lo_to_f32(w.z); o[5] = bf16hi_to_f32(w.z); o[6] = bf16lo_to_f32(w.w); o[7] = bf16hi_to_f32(w.w);
}

template <int HD>
__global__ void __launch_bounds__(STEP_THREADS, 1)
k_decode_step(const StepDev a) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    uint8_t* ring = smem;
    uint8_t* att_kv = smem + (size_t)a.n_slots * STEP_SLOT;          // attention K/V ring | the two B buffers of the GEMM phases
    AttSmall* att_sm = reinterpret_cast<AttSmall*>(att_kv + STEP_ATT_BYTES);
    StepShared* sh = reinterpret_cast<StepShared*>(reinterpret_cast<uint8_t*>(att_sm) + ((sizeof(AttSmall) + 15) & ~(size_t)15));
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int cta = blockIdx.x, nCTA = a.n_cta, NS = a.n_slots, NB = a.NB, L = a.n_layers, CH = a.chunk;

    if (tid < 4) sh->pl[tid] = a.plan[(size_t)tid * nCTA + cta];
    if (tid == 4) sh->ld_n = 0u;
    if (warp == 1 && lane == 0) {
        for (int s = 0; s < NS; ++s) { mbar_init(&sh->full[s], 1); mbar_init(&sh->empty[s], 1); }
        for (int s = 0; s < 2; ++s) { mbar_init(&sh->acc_full[s], 1); mbar_init(&sh->bfull[s], 1); mbar_init(&sh->bempty[s], 1); }
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    if (warp == 2) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" ::"r"(smem_u32(&sh->tmem_slot)), "n"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = sh->tmem_slot;
    pdl_launch();
    const bool tr_cta = a.trace != nullptr && (cta == 0 || cta == nCTA - 1);

    if (warp == 0) {
        // =========================== A producer: weights, as far ahead as the ring allows ===========================
        // (Warp 3 walks the same list a.prefetch tiles further ahead and only asks the TMA unit to pull the tile into L2.)
        if (lane == 0) {
            unsigned n = 0;
            for (int i = 0; i < 7 && L > 0; ++i) tma_prefetch_desc(&a.wmaps[i]);
            for (int l = 0; l < L; ++l) {
                const CUtensorMap* w7 = a.wmaps + (size_t)l * 7;
                if (l + 1 < L) for (int i = 0; i < 7; ++i) tma_prefetch_desc(&w7[7 + i]);
                for (int ph = 0; ph < 4; ++ph) {
                    const int NA = a.g[ph].na;
                    for (int s = 0; s < sh->pl[ph].nseg; ++s) {
                        const StepSeg sg = sh->pl[ph].seg[s];
                        int arow;
                        const CUtensorMap* m0 = step_wmap(a, w7, ph, sg.tile, 0, arow);
                        const CUtensorMap* m1 = step_wmap(a, w7, ph, sg.tile, 1, arow);
                        for (int kb = sg.kb0; kb < sg.kb1; ++kb)
                            for (int na = 0; na < NA; ++na, ++n) {
                                const unsigned slot = n % NS, use = n / NS;
                                if (use > 0) step_wait_mbar(&sh->empty[slot], (use - 1) & 1, a.err, 1);
                                if (a.prefetch > 0 && (n & 3u) == 0) *reinterpret_cast<volatile unsigned*>(&sh->ld_n) = n;
                                mbar_expect_tx(&sh->full[slot], STEP_SLOT);
                                tma_load_2d(ring + (size_t)slot * STEP_SLOT, na ? m1 : m0, &sh->full[slot], kb * 64, arow);
                            }
                    }
                }
            }
        }
        __syncwarp();
    } else if (warp == 3) {
        // =========================== L2 prefetcher (optional): same walk as the A producer, a.prefetch tiles ahead ===========
        // While the consumers sit in a phase boundary the ring is full and the A producer stalls; this warp keeps HBM
        // streaming into L2, from where the ring refills at L2 speed.
        if (lane == 0 && a.prefetch > 0) {
            unsigned n = 0;
            for (int l = 0; l < L; ++l) {
                const CUtensorMap* w7 = a.wmaps + (size_t)l * 7;
                for (int ph = 0; ph < 4; ++ph) {
                    const int NA = a.g[ph].na;
                    for (int s = 0; s < sh->pl[ph].nseg; ++s) {
                        const StepSeg sg = sh->pl[ph].seg[s];
                        int arow;
                        const CUtensorMap* m0 = step_wmap(a, w7, ph, sg.tile, 0, arow);
                        const CUtensorMap* m1 = step_wmap(a, w7, ph, sg.tile, 1, arow);
                        for (int kb = sg.kb0; kb < sg.kb1; ++kb)
                            for (int na = 0; na < NA; ++na, ++n) {
                                if (n < (unsigned)NS) continue;            // the first ring-full is loaded directly
                                while (n > *reinterpret_cast<volatile unsigned*>(&sh->ld_n) + (unsigned)a.prefetch) __nanosleep(64);
                                asm volatile("cp.async.bulk.prefetch.tensor.2d.L2.global.tile [%0, {%1, %2}];\n" ::"l"(na ? m1 : m0),
                                             "r"(kb * 64), "r"(arow) : "memory");
                            }
                    }
                }
            }
        }
        __syncwarp();
    } else if (warp == 1) {
        // =========================== MMA issuer ===========================
        if (lane == 0) {
            const uint32_t idesc = umma_idesc(NB);
            unsigned n = 0, cn = 0;                       // ring item / B chunk sequence numbers
            for (int l = 0; l < L; ++l) {
                for (int ph = 0; ph < 4; ++ph) {
                    const int NA = a.g[ph].na;
                    for (int s = 0; s < sh->pl[ph].nseg; ++s) {
                        const StepSeg sg = sh->pl[ph].seg[s];
                        for (int kc = sg.kb0; kc < sg.kb1; kc += CH, ++cn) {
                            const int nk = min(CH, sg.kb1 - kc);
                            const unsigned buf = cn & 1u, buse = cn >> 1;
                            step_wait_mbar(&sh->bfull[buf], buse & 1, a.err, 4);
                            for (int j = 0; j < nk; ++j)
                                for (int na = 0; na < NA; ++na, ++n) {
                                    const unsigned slot = n % NS, use = n / NS;
                                    step_wait_mbar(&sh->full[slot], use & 1, a.err, 5);
                                    tc_fence_after();
                                    const uint64_t adesc = umma_desc_sw128(smem_u32(ring + (size_t)slot * STEP_SLOT));
                                    const uint64_t bdesc = umma_desc_sw128(smem_u32(att_kv + (size_t)buf * STEP_BBUF + (size_t)j * NB * 128));
                                    const uint32_t dcol = tmem_base + (uint32_t)((s * 2 + na) * NB);
#pragma unroll
                                    for (int k = 0; k < 4; ++k)
                                        tc_mma(dcol, adesc + 2 * k, bdesc + 2 * k, idesc, (kc + j > sg.kb0 || k > 0) ? 1u : 0u);
                                    tc_commit(&sh->empty[slot]);
                                }
                            tc_commit(&sh->bempty[buf]);
                        }
                        tc_commit(&sh->acc_full[s]);
                    }
                }
            }
        }
        __syncwarp();
    } else if (warp >= 4) {
        // =========================== workers ===========================
        const int wt = tid - 128, wi = warp - 4, lg = wi & 3, h = wi >> 2;
        const int row = lg * 32 + lane;                       // output feature inside a 128-row tile = TMEM lane
        const int d = a.d_model, F = a.d_ff;
        pdl_wait();
        if (wt == 0) {
            sh->M = min(*a.n_live, a.m_max);
            sh->par = *a.step & 1;
        }
        worker_sync();
        const int M = sh->M, par = sh->par;
        const bool tron = tr_cta && wt == 0 && (unsigned long long)*a.step == a.trace[0];
        step_trace(a, tron, 3, 9, 0);
        unsigned* gbar = a.sync_base + (size_t)par * a.gbar_n;
        {   // clear the other parity set for the next step (nobody touches it during this one)
            unsigned* other = a.sync_base + (size_t)(par ^ 1) * a.gbar_n;
            for (int i = cta * 256 + wt; i < a.gbar_n; i += nCTA * 256) other[i] = 0u;
        }
        // largest context of the step -> number of attention K-splits (same value on every CTA)
        {
            int cm = 0;
            for (int i = wt; i < M; i += 256) cm = max(cm, a.ctx[i]);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) cm = max(cm, __shfl_xor_sync(0xffffffffu, cm, o));
            if (lane == 0) sh->ctx_max[wi] = cm;
            worker_sync();
            if (wt == 0) {
                int c2 = 0;
                for (int i = 0; i < 8; ++i) c2 = max(c2, sh->ctx_max[i]);
                constexpr int TILE = StepAtt<HD>::WARPS * 16;
                const int units0 = max(1, M * a.att.Hkv);
                int ns = nCTA / units0;
                const int cap = (c2 + TILE - 1) / TILE;          // at least one tile per split
                if (ns > cap) ns = cap;
                if (ns > 32) ns = 32;
                if (ns < 1) ns = 1;
                sh->ns = ns;
            }
            worker_sync();
        }
        const int ns_att = sh->ns;
        auto arrive = [&](int p) {
            worker_sync();                                    // every worker's stores / reds of this phase are issued ...
            if (wt == 0) red_release_add(gbar + p, 1u);       // ... and ordered before this release (cumulative over the barrier)
            step_trace(a, tron, 3, 8, p);
        };
        auto wait_phase = [&](int p) {
            if (wt == 0) step_wait_count(gbar + p, (unsigned)nCTA, a.err, 6);
            worker_sync();
            step_trace(a, tron, 3, 0, p + 1);
        };
        // zero rows [0, M) of a fixed-point accumulator (all CTAs share the work)
        auto zero_acc = [&](long long* acc, int ncol) {
            const int n2 = M * (ncol / 2);
            longlong2* p2 = reinterpret_cast<longlong2*>(acc);
            for (int i = cta * 256 + wt; i < n2; i += nCTA * 256) p2[i] = make_longlong2(0ll, 0ll);
        };
        // the CTA that owns row m (cta == m) carries the fp32 residual stream forward: xout[m] = xin[m] + acc[m],
        // and publishes 1/rms of the new row
        auto own_row = [&](const float* xin, const long long* acc, float* xout, float* rstd_out) {
            if (cta >= M) return;
            const int m = cta;
            float ss = 0.f;
            for (int k = wt * 4; k < d; k += 1024) {
                const float4 xv = __ldcg(reinterpret_cast<const float4*>(xin + (size_t)m * d + k));
                const longlong2 a0 = __ldcg(reinterpret_cast<const longlong2*>(acc + (size_t)m * d + k));
                const longlong2 a1 = __ldcg(reinterpret_cast<const longlong2*>(acc + (size_t)m * d + k + 2));
                float4 o;
                o.x = xv.x + fx_to_f32(a0.x); o.y = xv.y + fx_to_f32(a0.y); o.z = xv.z + fx_to_f32(a1.x); o.w = xv.w + fx_to_f32(a1.y);
                *reinterpret_cast<float4*>(xout + (size_t)m * d + k) = o;
                ss += o.x * o.x + o.y * o.y + o.z * o.z + o.w * o.w;
            }
            ss = warp_sum(ss);
            if (lane == 0) sh->red[wi] = ss;
            worker_sync();
            if (wt == 0) {
                float t = 0.f;
                for (int i = 0; i < 8; ++i) t += sh->red[i];
                rstd_out[m] = rsqrtf(t / (float)d + a.eps);
            }
            worker_sync();
        };

        // ---- phase 0: embedding rows -> xa; every accumulator starts the step at zero ----
        if (cta < M) {
            const bf16_t* src = a.embed + (size_t)a.tok[cta] * d;
            for (int k = wt * 8; k < d; k += 2048) {
                float v[8];
                load_bf8(src + k, v);
                *reinterpret_cast<float4*>(a.xa + (size_t)cta * d + k) = make_float4(v[0], v[1], v[2], v[3]);
                *reinterpret_cast<float4*>(a.xa + (size_t)cta * d + k + 4) = make_float4(v[4], v[5], v[6], v[7]);
            }
        }
        zero_acc(a.accQ, a.Nqkv); zero_acc(a.accO, d); zero_acc(a.accG, 2 * F); zero_acc(a.accD, d);
        arrive(0);

        unsigned acc_use[2] = {0u, 0u};
        unsigned cn = 0;                                      // B chunk sequence number (same walk as the MMA issuer)
        for (int l = 0; l < L; ++l) {
            for (int phx = 0; phx < 5; ++phx) {
                const int p = 1 + l * 5 + phx;
                wait_phase(p - 1);
                if (phx == 1) {
                    // ---------------- attention (fused RoPE + KV append); accD is free again ----------------
                    zero_acc(a.accD, d);
                    const int units = M * a.att.Hkv * ns_att;
                    if (cta < units) {
                        AttnArgs aa = a.att;
                        aa.kv_layer = a.kv_pool + (size_t)l * a.layer_stride;
                        aa.kv_layer_w = a.kv_pool + (size_t)l * a.layer_stride;
                        for (int u = cta; u < units; u += nCTA) {
                            const int r0 = u / (a.att.Hkv * ns_att), rem = u - r0 * (a.att.Hkv * ns_att);
                            attention_unit<HD, StepAtt<HD>::WARPS, StepAtt<HD>::NSTAGE, true>(aa, r0, rem / ns_att, rem % ns_att, ns_att,
                                                                                               att_kv, att_sm, nullptr, wt);
                        }
                    }
                    arrive(p);
                    continue;
                }
                const int ph = phx == 0 ? 0 : phx - 1;               // 0 QKV, 1 O, 2 gate/up, 3 down
                const int nseg = sh->pl[ph].nseg;
                const int NA = a.g[ph].na;
                const float* xin = (ph == 0) ? a.xa : a.xb;          // QKV reads xa (+ accD), gate/up reads xb (+ accO)
                const long long* accin = (ph == 0) ? a.accD : a.accO;
                const bf16_t* gain = (ph == 0) ? a.norm1[l] : a.norm2[l];
                if (ph == 3) {
                    if (wt < M) sh->rstd[wt] = __ldcg(a.rstd2 + wt);
                    worker_sync();
                }
                // ---- build the B operand of every unit, one <= 32 KB chunk of k blocks at a time ----
                for (int s = 0; s < nseg; ++s) {
                    const StepSeg sg = sh->pl[ph].seg[s];
                    for (int kc = sg.kb0; kc < sg.kb1; kc += CH, ++cn) {
                        const int nk = min(CH, sg.kb1 - kc);
                        const unsigned buf = cn & 1u, buse = cn >> 1;
                        if (buse > 0) step_wait_mbar(&sh->bempty[buf], (buse - 1) & 1, a.err, 3);
                        uint8_t* bb = att_kv + (size_t)buf * STEP_BBUF;
                        const int tasks = M * nk * 8;                // (batch row, k block, 16-byte chunk)
                        // two tasks per thread and iteration, every load of both issued before the first use
                        for (int i0 = wt; i0 < tasks; i0 += 512) {
                            int tc[2], tj[2], tm[2], tk[2];
                            bool on[2];
#pragma unroll
                            for (int u = 0; u < 2; ++u) {
                                const int i = i0 + 256 * u;
                                on[u] = i < tasks;
                                const int ii = on[u] ? i : i0;
                                tc[u] = ii & 7; tj[u] = (ii >> 3) % nk; tm[u] = ii / (8 * nk);
                                tk[u] = (kc + tj[u]) * 64 + tc[u] * 8;
                            }
                            if (ph == 1) {                            // attention output, already split: plain copy
                                uint4 hi[2], lo[2];
#pragma unroll
                                for (int u = 0; u < 2; ++u) {
                                    hi[u] = __ldcg(reinterpret_cast<const uint4*>(a.att_s + (size_t)(2 * tm[u]) * a.qd + tk[u]));
                                    lo[u] = __ldcg(reinterpret_cast<const uint4*>(a.att_s + (size_t)(2 * tm[u] + 1) * a.qd + tk[u]));
                                }
#pragma unroll
                                for (int u = 0; u < 2; ++u) {
                                    if (!on[u]) continue;
                                    uint8_t* tile = bb + (size_t)tj[u] * NB * 128;
                                    const int r0 = 2 * tm[u], r1 = 2 * tm[u] + 1;
                                    *reinterpret_cast<uint4*>(tile + (size_t)r0 * 128 + ((tc[u] ^ (r0 & 7)) << 4)) = hi[u];
                                    *reinterpret_cast<uint4*>(tile + (size_t)r1 * 128 + ((tc[u] ^ (r1 & 7)) << 4)) = lo[u];
                                }
                            } else if (ph == 3) {                     // SwiGLU of the gate / up sums (1/rms applied here)
                                float gt[2][8], up[2][8];
#pragma unroll
                                for (int u = 0; u < 2; ++u) {
                                    load_fx8(a.accG + (size_t)tm[u] * 2 * F + tk[u], gt[u]);
                                    load_fx8(a.accG + (size_t)tm[u] * 2 * F + F + tk[u], up[u]);
                                }
#pragma unroll
                                for (int u = 0; u < 2; ++u) {
                                    if (!on[u]) continue;
                                    const float rs = sh->rstd[tm[u]];
                                    float v[8];
#pragma unroll
                                    for (int e = 0; e < 8; ++e) v[e] = silu_f(gt[u][e] * rs) * (up[u][e] * rs);
                                    store_b_chunk(bb + (size_t)tj[u] * NB * 128, tm[u], tc[u], v);
                                }
                            } else {                                  // (x + acc) * norm gain
                                float xv[2][8], av[2][8], gv[2][8];
#pragma unroll
                                for (int u = 0; u < 2; ++u) {
                                    load_f8(xin + (size_t)tm[u] * d + tk[u], xv[u]);
                                    load_fx8(accin + (size_t)tm[u] * d + tk[u], av[u]);
                                    load_bf8(gain + tk[u], gv[u]);
                                }
#pragma unroll
                                for (int u = 0; u < 2; ++u) {
                                    if (!on[u]) continue;
                                    float v[8];
#pragma unroll
                                    for (int e = 0; e < 8; ++e) v[e] = (xv[u][e] + av[u][e]) * gv[u][e];
                                    store_b_chunk(bb + (size_t)tj[u] * NB * 128, tm[u], tc[u], v);
                                }
                            }
                        }
                        asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");   // generic-proxy smem writes -> tcgen05.mma reads
                        worker_sync();
                        if (wt == 0) mbar_arrive(&sh->bfull[buf]);
                    }
                }
                step_trace(a, tron, 3, 1, p);
                // ---- off the critical path: residual stream / 1/rms of the rows this CTA owns, accumulator recycling ----
                if (ph == 0) { own_row(a.xa, a.accD, a.xb, a.rstd1); zero_acc(a.accG, 2 * F); }
                if (ph == 1) zero_acc(a.accQ, a.Nqkv);
                if (ph == 2) own_row(a.xb, a.accO, a.xa, a.rstd2);
                if (ph == 3) zero_acc(a.accO, d);
                // ---- drain: TMEM -> (hi + lo) -> fixed-point add into the phase's accumulator in L2 ----
                long long* accout = (ph == 0) ? a.accQ : (ph == 1 ? a.accO : (ph == 2 ? a.accG : a.accD));
                const int ldo = (ph == 0) ? a.Nqkv : (ph == 2 ? 2 * F : d);
                for (int s = 0; s < nseg; ++s) {
                    const StepSeg sg = sh->pl[ph].seg[s];
                    step_wait_mbar(&sh->acc_full[s], acc_use[s] & 1, a.err, 7);
                    ++acc_use[s];
                    tc_fence_after();
                    if (s == 0) step_trace(a, tron, 3, 2, p);
                    for (int na = 0; na < NA; ++na) {
                        const int n = sg.tile * 128 + row + na * F;          // gate rows, then up rows
                        for (int c = h; c * 16 < M && c < NB / 32; c += 2) {
                            float v[32];
                            tc_ld32(tmem_base + ((uint32_t)(lg * 32) << 16) + (uint32_t)((s * 2 + na) * NB + c * 32), v);
#pragma unroll
                            for (int j = 0; j < 16; ++j) {
                                const int m = c * 16 + j;
                                if (m < M) red_add_fx(accout + (size_t)m * ldo + n, v[2 * j] + v[2 * j + 1]);
                            }
                        }
                    }
                }
                tc_fence_before();
                step_trace(a, tron, 3, 4, p);
                arrive(p);
            }
        }
        // ---- last phase: the LM-head operand of the rows this CTA owns (final residual, x * w_final split, sum of squares) ----
        wait_phase(5 * L);
        if (cta < M) {
            const int m = cta;
            float ss = 0.f;
            for (int k = wt * 8; k < d; k += 2048) {
                float xv[8], av[8], gv[8], v[8];
                load_f8(a.xa + (size_t)m * d + k, xv);
                load_fx8(a.accD + (size_t)m * d + k, av);
                load_bf8(a.final_norm + k, gv);
#pragma unroll
                for (int e = 0; e < 8; ++e) { xv[e] += av[e]; ss += xv[e] * xv[e]; v[e] = xv[e] * gv[e]; }
                *reinterpret_cast<float4*>(a.x + (size_t)m * d + k) = make_float4(xv[0], xv[1], xv[2], xv[3]);
                *reinterpret_cast<float4*>(a.x + (size_t)m * d + k + 4) = make_float4(xv[4], xv[5], xv[6], xv[7]);
                uint32_t hi[4], lo[4];
#pragma unroll
                for (int i = 0; i < 4; ++i) split2(v[2 * i], v[2 * i + 1], hi[i], lo[i]);
                *reinterpret_cast<uint4*>(a.xs + (size_t)(2 * m) * d + k) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
                *reinterpret_cast<uint4*>(a.xs + (size_t)(2 * m + 1) * d + k) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
            }
            ss = warp_sum(ss);
            if (lane == 0) sh->red[wi] = ss;
            worker_sync();
            if (wt == 0) {
                float t = 0.f;
                for (int i = 0; i < 8; ++i) t += sh->red[i];
                a.ssq[m] = t;
                for (int i = 1; i < a.d_tiles; ++i) a.ssq[(size_t)i * a.ssq_ld + m] = 0.f;
            }
        }
    }
    __syncthreads();
    if (warp == 2) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(tmem_base), "n"(512));
    }
}

// ---------------------------------------------------------------------------------------------------------------
// host: work decomposition
// ---------------------------------------------------------------------------------------------------------------
// K-split of one GEMM phase: minimise the k blocks of the busiest CTA (at most two units per CTA), then the split count.
static bool choose_split(int tiles, int n_kb, int n_cta, int* ks_out) {
    int best = 0, best_load = 1 << 30;
    for (int ks = 1; ks <= STEP_KS_MAX && ks <= n_kb; ++ks) {
        const int units = tiles * ks, rounds = (units + n_cta - 1) / n_cta;
        if (rounds > 2) continue;
        const int load = rounds * ((n_kb + ks - 1) / ks);
        if (load < best_load) { best_load = load; best = ks; }
    }
    *ks_out = best;
    return best > 0;
}

bool build_step_plan(int n_cta, int d_model, int qd, int kvd, int d_ff, StepGemm g[4], std::vector<StepPhasePlan>& plan,
                     int* tiles_per_layer) {
    if (d_model % 128 || qd % 128 || kvd % 128 || d_ff % 128) return false;
    const int Nqkv = qd + 2 * kvd;
    const int K[4] = {d_model, qd, d_model, d_ff};
    const int N[4] = {Nqkv, d_model, d_ff, d_model};
    plan.assign((size_t)4 * n_cta, StepPhasePlan{});
    int toff = 0, rot = 0;
    for (int ph = 0; ph < 4; ++ph) {
        StepGemm& gm = g[ph];
        gm = StepGemm{};
        gm.K = K[ph]; gm.n_kb = K[ph] / 64; gm.tiles = N[ph] / 128; gm.na = ph == 2 ? 2 : 1;
        gm.seg0_tiles = ph == 0 ? qd / 128 : gm.tiles; gm.seg1_tiles = ph == 0 ? kvd / 128 : 0;
        gm.tile_ctr_off = toff;
        toff += gm.tiles;
        int ks;
        if (!choose_split(gm.tiles, gm.n_kb, n_cta, &ks)) return false;
        gm.ks = ks;
        const int q = gm.n_kb / ks, rem = gm.n_kb % ks;
        for (int u = 0; u < gm.tiles * ks; ++u) {
            const int tile = u / ks, rank = u % ks;
            const int cta = (u + rot) % n_cta;
            StepPhasePlan& pp = plan[(size_t)ph * n_cta + cta];
            if (pp.nseg >= 2) return false;
            StepSeg& sg = pp.seg[pp.nseg++];
            sg.tile = tile; sg.rank = rank; sg.ks = ks; sg.slot0 = tile * ks;
            sg.kb0 = rank * q + std::min(rank, rem);
            sg.kb1 = sg.kb0 + q + (rank < rem ? 1 : 0);
        }
        rot = (rot + gm.tiles * ks) % n_cta;          // the next phase starts on the CTAs this one left idle
    }
    *tiles_per_layer = toff;
    return true;
}

int step_smem_bytes(int n_slots) {
    return 1024 + n_slots * STEP_SLOT + STEP_ATT_BYTES + (int)((sizeof(AttSmall) + 15) & ~(size_t)15) + STEP_MISC;
}
int step_ring_slots(int smem_limit) {
    int n = (smem_limit - step_smem_bytes(0)) / STEP_SLOT;
    return n > 12 ? 12 : n;
}

int launch_decode_step(const StepLaunch& s, cudaStream_t st) {
    if (s.m_max <= 0 || s.m_max > 64 || (s.att.hd != 64 && s.att.hd != 128)) return -1;
    StepDev d = {};
    d.n_layers = s.n_layers; d.n_cta = s.n_cta; d.NB = 32 << tc_nb_index(s.m_max); d.n_slots = s.n_slots;
    d.chunk = STEP_BBUF / (d.NB * 128);
    for (int i = 0; i < 4; ++i) d.g[i] = s.g[i];
    d.wmaps = reinterpret_cast<const CUtensorMap*>(s.wmaps_dev); d.plan = s.plan_dev;
    d.xa = s.xa; d.xb = s.xb; d.accQ = s.accQ; d.accO = s.accO; d.accG = s.accG; d.accD = s.accD; d.rstd1 = s.rstd1; d.rstd2 = s.rstd2;
    d.x = s.x; d.xs = s.xs; d.att_s = s.att_s; d.ssq = s.ssq;
    d.ssq_ld = s.ssq_ld; d.d_tiles = s.d_tiles; d.d_model = s.d_model; d.Nqkv = s.Nqkv; d.qd = s.qd; d.d_ff = s.d_ff;
    d.norm1 = s.norm1_dev; d.norm2 = s.norm2_dev; d.final_norm = s.final_norm; d.embed = s.embed; d.eps = s.eps;
    d.sync_base = s.sync_base; d.gbar_n = s.gbar_n;
    d.live = s.live; d.pos = s.pos; d.ctx = s.ctx; d.tok = s.tok; d.n_live = s.n_live; d.step = s.step; d.m_max = s.m_max;
    d.att = s.att; d.kv_pool = s.kv_pool; d.layer_stride = s.layer_stride; d.err = s.err; d.trace = s.trace;
    { const char* e = getenv("SAGC_STEP_FLAGS"); d.flags = e ? atoi(e) : 0; }
    { const char* e = getenv("SAGC_STEP_PREFETCH"); d.prefetch = e ? atoi(e) : 0; if (d.prefetch > 0 && d.prefetch < 8) d.prefetch = 8; }   // < 8 could strand the prefetch warp behind the published count
    const int smem = step_smem_bytes(s.n_slots);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(s.n_cta);
    cfg.blockDim = dim3(STEP_THREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[2];
    int na = 0;
    if (s.cooperative) { at[na].id = cudaLaunchAttributeCooperative; at[na].val.cooperative = 1; ++na; }
    if (s.pdl) { at[na].id = cudaLaunchAttributeProgrammaticStreamSerialization; at[na].val.programmaticStreamSerializationAllowed = 1; ++na; }
    cfg.attrs = at; cfg.numAttrs = na;
    cudaError_t e;
    if (s.att.hd == 128) {
        e = cudaFuncSetAttribute(k_decode_step<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e == cudaSuccess) e = cudaLaunchKernelEx(&cfg, k_decode_step<128>, d);
    } else {
        e = cudaFuncSetAttribute(k_decode_step<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e == cudaSuccess) e = cudaLaunchKernelEx(&cfg, k_decode_step<64>, d);
    }
    return e == cudaSuccess ? 1 : -1;
}

// ---------------------------------------------------------------------------------------------------------------
// parity entry (sagc_debug_attention, variant 1): the attention units exactly as the step kernel runs them --
// 256 threads, StepAtt geometry, unit loop over a fixed number of CTAs, last-arriver merge through the L2 scratch
// ---------------------------------------------------------------------------------------------------------------
template <int HD>
__global__ void __launch_bounds__(256, 1) k_attention_units(AttnArgs a) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 127) & ~(uintptr_t)127);
    AttSmall* att_sm = reinterpret_cast<AttSmall*>(smem + STEP_ATT_BYTES);
    const int M = a.m_dev ? min(*a.m_dev, a.m_max) : a.m_max;
    const int ns = a.n_splits, units = M * a.Hkv * ns;
    for (int u = blockIdx.x; u < units; u += gridDim.x) {
        const int r0 = u / (a.Hkv * ns), rem = u - r0 * (a.Hkv * ns);
        attention_unit<HD, StepAtt<HD>::WARPS, StepAtt<HD>::NSTAGE, true>(a, r0, rem / ns, rem % ns, ns, smem, att_sm, nullptr, (int)threadIdx.x);
    }
}
int launch_attention_units(const AttnArgs& a, int n_cta, cudaStream_t st) {
    const int smem = 128 + STEP_ATT_BYTES + (int)sizeof(AttSmall);
    cudaError_t e;
    if (a.hd == 128) {
        e = cudaFuncSetAttribute(k_attention_units<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e == cudaSuccess) k_attention_units<128><<<n_cta, 256, smem, st>>>(a);
    } else if (a.hd == 64) {
        e = cudaFuncSetAttribute(k_attention_units<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e == cudaSuccess) k_attention_units<64><<<n_cta, 256, smem, st>>>(a);
    } else {
        return -1;
    }
    return e == cudaSuccess ? 1 : -1;
}

}  // namespace sagc
