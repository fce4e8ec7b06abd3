// decode_step.cu -- ONE persistent kernel for the whole layer stack of a decode step (steps a5-a10 of
// DESIGN.md; <= 64 live rows): embedding + per layer { QKV | RoPE + KV append + paged attention | O + residual |
// gate/up + SwiGLU | down + residual }.  One CTA per SM; kernel boundaries are replaced by grid-wide
// arrive/poll counters in L2, and -- the point of the exercise -- the weight stream never stops at them:
//
//   warp 0   A producer : walks this CTA's static work list (every layer, every GEMM phase) and TMA-loads the
//                         128 x 64 bf16 weight tiles into a ring of 16 KB slots.  Weights depend on nothing,
//                         so it runs as far ahead as the ring allows, across phase and layer boundaries.
//   warp 1   B producer : loads the activation operand (pre-split hi/lo bf16 rows) of the
//                         same work list into its own ring slots as soon as the phase that produces it has
//                         completed on every CTA.
//   warp 2   MMA issuer : tcgen05.mma (weights = A, M = 128; activations = B, N = 2 x batch), fp32 in TMEM.
//   warp 3   owns the TMEM allocation.
//   warps 4-11 workers  : epilogues (TMEM -> registers -> fused residual / SwiGLU / next-norm -> L2), the
//                         split-K reduction, the attention units (attention_body.cuh) and the embedding rows.
//
// Work decomposition (host, build_step_plan): a GEMM phase is cut into units (128-row weight tile, k range);
// unit -> CTA is static.  K is split so that every SM streams a share of every matrix.  The KS partial tiles
// of an output tile go through an L2 scratch; a per-tile counter tells the KS contributors when all partials
// have landed, and contributor `rank` then finishes batch rows rank, rank + KS, ... (sum in rank order:
// deterministic).  All counters are double-buffered by step parity: step t uses set t & 1 and clears the other.
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
static constexpr int STEP_ATT_BYTES = 65536;             // K/V staging of the attention units
static constexpr int STEP_MISC = 3072;                   // barriers, plan copy, rstd / ssq scratch
static constexpr int STEP_SCR_SLOT = 2 * 64 * 128;       // floats per split-K scratch slot: [na][m][row]
static constexpr unsigned long long STEP_WATCHDOG_NS = 4000000000ull;

// attention geometry inside the step kernel: 64 KB of K/V staging either way
template <int HD> struct StepAtt { static constexpr int WARPS = HD >= 128 ? 4 : 8; static constexpr int NSTAGE = 2; };

struct StepDev {
    int n_layers, n_cta, NB, n_slots, bper;
    StepGemm g[4];
    const CUtensorMap* wmaps;            // device [n_layers][7]: q k v o g u d (box 64 x 128)
    const StepPhasePlan* plan;           // device [4][n_cta]
    float* x; float* qkv; bf16_t* xs; bf16_t* att_s; bf16_t* act_s; float* ssq;
    int ssq_ld, d_tiles, d_model, Nqkv, qd, d_ff;
    const bf16_t* const* norm1; const bf16_t* const* norm2; const bf16_t* final_norm; const bf16_t* embed;
    float eps;
    float* scratch;
    unsigned* sync_base; int gbar_n, tcnt_n, tiles_per_layer;        // [2][gbar_n + tcnt_n]
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
__device__ __forceinline__ unsigned ld_relaxed_u32(const unsigned* p) {
    unsigned v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];\n" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void step_wait_count(const unsigned* ctr, unsigned target, int* err, int code, bool relaxed = false) {
    if (relaxed) {      // poll with relaxed loads, one acquire fence at the end
        if (ld_relaxed_u32(ctr) < target) {
            const unsigned long long t0 = globaltimer_ns();
            unsigned n = 0;
            while (ld_relaxed_u32(ctr) < target)
                if (((++n) & 1023u) == 0 && globaltimer_ns() - t0 > STEP_WATCHDOG_NS) step_die(err, code);
        }
        asm volatile("fence.acq_rel.gpu;\n" ::: "memory");
        return;
    }
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
    uint64_t full[12], empty[12], acc_full[2];
    uint32_t tmem_slot; int M, par, ns, pad;
    StepPhasePlan pl[4];
    float rstd[64];
    float ssq_s[4][64];
    float red[8];
    int ctx_max[8];
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

template <int HD>
__global__ void __launch_bounds__(STEP_THREADS, 1)
k_decode_step(const __grid_constant__ CUtensorMap tmXs, const __grid_constant__ CUtensorMap tmAtt,
              const __grid_constant__ CUtensorMap tmAct, const StepDev a) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    uint8_t* ring = smem;
    uint8_t* att_kv = smem + (size_t)a.n_slots * STEP_SLOT;
    AttSmall* att_sm = reinterpret_cast<AttSmall*>(att_kv + STEP_ATT_BYTES);
    StepShared* sh = reinterpret_cast<StepShared*>(reinterpret_cast<uint8_t*>(att_sm) + ((sizeof(AttSmall) + 15) & ~(size_t)15));
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int cta = blockIdx.x, nCTA = a.n_cta, NS = a.n_slots, NB = a.NB, L = a.n_layers;

    if (tid < 4) sh->pl[tid] = a.plan[(size_t)tid * nCTA + cta];
    if (warp == 2 && lane == 0) {
        for (int s = 0; s < NS; ++s) { mbar_init(&sh->full[s], 1); mbar_init(&sh->empty[s], 1); }
        mbar_init(&sh->acc_full[0], 1); mbar_init(&sh->acc_full[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    if (warp == 3) {
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
        if (lane == 0) {
            unsigned n = 0;
            for (int l = 0; l < L; ++l) {
                const CUtensorMap* w7 = a.wmaps + (size_t)l * 7;
                for (int i = 0; i < 7; ++i) tma_prefetch_desc(&w7[i]);
                for (int ph = 0; ph < 4; ++ph) {
                    const int NA = a.g[ph].na;
                    for (int s = 0; s < sh->pl[ph].nseg; ++s) {
                        const StepSeg sg = sh->pl[ph].seg[s];
                        int arow;
                        const CUtensorMap* m0 = step_wmap(a, w7, ph, sg.tile, 0, arow);
                        const CUtensorMap* m1 = step_wmap(a, w7, ph, sg.tile, 1, arow);
                        for (int kbg = sg.kb0; kbg < sg.kb1; kbg += a.bper) {
                            const int nbk = min(a.bper, sg.kb1 - kbg);
                            ++n;                                             // the group's B slot (filled by warp 1)
                            for (int j = 0; j < nbk; ++j)
                                for (int na = 0; na < NA; ++na, ++n) {
                                    const unsigned slot = n % NS, use = n / NS;
                                    if (use > 0) step_wait_mbar(&sh->empty[slot], (use - 1) & 1, a.err, 1);
                                    mbar_expect_tx(&sh->full[slot], STEP_SLOT);
                                    tma_load_2d(ring + (size_t)slot * STEP_SLOT, na ? m1 : m0, &sh->full[slot], (kbg + j) * 64, arow);
                                }
                        }
                    }
                }
            }
        }
        __syncwarp();
    } else if (warp == 1) {
        // =========================== B producer: activations, gated by the producing phase ===========================
        if (lane == 0) {
            pdl_wait();
            const int par = *a.step & 1;
            const bool tron = tr_cta && (unsigned long long)*a.step == a.trace[0];
            const unsigned* gbar = a.sync_base + (size_t)par * (a.gbar_n + a.tcnt_n);
            tma_prefetch_desc(&tmXs); tma_prefetch_desc(&tmAtt); tma_prefetch_desc(&tmAct);
            unsigned n = 0;
            for (int l = 0; l < L; ++l) {
                for (int ph = 0; ph < 4; ++ph) {
                    const int NA = a.g[ph].na;
                    const int p = 1 + l * 5 + (ph == 0 ? 0 : ph + 1);            // phase index of this GEMM
                    const CUtensorMap* bm = (ph == 1) ? &tmAtt : (ph == 3 ? &tmAct : &tmXs);
                    bool opened = false;
                    for (int s = 0; s < sh->pl[ph].nseg; ++s) {
                        const StepSeg sg = sh->pl[ph].seg[s];
                        for (int kbg = sg.kb0; kbg < sg.kb1; kbg += a.bper) {
                            const int nbk = min(a.bper, sg.kb1 - kbg);
                            const unsigned slot = n % NS, use = n / NS;
                            if (!opened) {
                                step_wait_count(gbar + (p - 1), (unsigned)nCTA, a.err, 2, (a.flags & 4) != 0);
                                asm volatile("fence.proxy.async;\n" ::: "memory");   // generic-proxy writes of other SMs -> TMA reads
                                opened = true;
                                step_trace(a, tron, 1, 0, p);
                            }
                            if (use > 0) step_wait_mbar(&sh->empty[slot], (use - 1) & 1, a.err, 3);
                            mbar_expect_tx(&sh->full[slot], (uint32_t)(nbk * NB * 128));
                            for (int j = 0; j < nbk; ++j)
                                tma_load_2d(ring + (size_t)slot * STEP_SLOT + (size_t)j * NB * 128, bm, &sh->full[slot], (kbg + j) * 64, 0);
                            n += 1 + nbk * NA;
                        }
                    }
                }
            }
        }
        __syncwarp();
    } else if (warp == 2) {
        // =========================== MMA issuer ===========================
        if (lane == 0) {
            const uint32_t idesc = umma_idesc(NB);
            unsigned n = 0;
            for (int l = 0; l < L; ++l) {
                for (int ph = 0; ph < 4; ++ph) {
                    const int NA = a.g[ph].na;
                    for (int s = 0; s < sh->pl[ph].nseg; ++s) {
                        const StepSeg sg = sh->pl[ph].seg[s];
                        for (int kbg = sg.kb0; kbg < sg.kb1; kbg += a.bper) {
                            const int nbk = min(a.bper, sg.kb1 - kbg);
                            const unsigned bslot = n % NS, buse = n / NS;
                            ++n;
                            step_wait_mbar(&sh->full[bslot], buse & 1, a.err, 4);
                            if (kbg == sg.kb0) step_trace(a, tr_cta, 2, 0, 1 + l * 5 + (ph == 0 ? 0 : ph + 1));
                            for (int j = 0; j < nbk; ++j)
                                for (int na = 0; na < NA; ++na, ++n) {
                                    const unsigned slot = n % NS, use = n / NS;
                                    step_wait_mbar(&sh->full[slot], use & 1, a.err, 5);
                                    tc_fence_after();
                                    const uint64_t adesc = umma_desc_sw128(smem_u32(ring + (size_t)slot * STEP_SLOT));
                                    const uint64_t bdesc = umma_desc_sw128(smem_u32(ring + (size_t)bslot * STEP_SLOT + (size_t)j * NB * 128));
                                    const uint32_t dcol = tmem_base + (uint32_t)((s * 2 + na) * NB);
#pragma unroll
                                    for (int k = 0; k < 4; ++k)
                                        tc_mma(dcol, adesc + 2 * k, bdesc + 2 * k, idesc, (kbg + j > sg.kb0 || k > 0) ? 1u : 0u);
                                    tc_commit(&sh->empty[slot]);
                                }
                            tc_commit(&sh->empty[bslot]);
                        }
                        tc_commit(&sh->acc_full[s]);
                        step_trace(a, tr_cta, 2, 1, 1 + l * 5 + (ph == 0 ? 0 : ph + 1));
                    }
                }
            }
        }
        __syncwarp();
    } else if (warp >= 4) {
        // =========================== workers ===========================
        const int wt = tid - 128, wi = warp - 4, lg = wi & 3, h = wi >> 2;
        const int row = lg * 32 + lane;                       // output feature inside a 128-row tile = TMEM lane
        pdl_wait();
        if (wt == 0) {
            sh->M = min(*a.n_live, a.m_max);
            sh->par = *a.step & 1;
        }
        worker_sync();
        const int M = sh->M, par = sh->par;
        const bool tron = tr_cta && wt == 0 && (unsigned long long)*a.step == a.trace[0];
        step_trace(a, tron, 3, 9, 0);
        unsigned* gbar = a.sync_base + (size_t)par * (a.gbar_n + a.tcnt_n);
        unsigned* tcnt = gbar + a.gbar_n;
        {   // clear the other parity set for the next step (nobody touches it during this one)
            unsigned* other = a.sync_base + (size_t)(par ^ 1) * (a.gbar_n + a.tcnt_n);
            for (int i = cta * 256 + wt; i < a.gbar_n + a.tcnt_n; i += nCTA * 256) other[i] = 0u;
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
                const int cap = c2 / (2 * TILE);
                if (ns > cap) ns = cap;
                if (ns > 32) ns = 32;
                if (ns < 1) ns = 1;
                sh->ns = ns;
            }
            worker_sync();
        }
        const int ns_att = sh->ns;
        auto arrive = [&](int p) {
            if (!(a.flags & 2)) asm volatile("fence.proxy.async;\n" ::: "memory");     // this thread's global writes -> later TMA reads elsewhere
            if (!(a.flags & 1)) __threadfence();
            worker_sync();
            if (wt == 0) red_release_add(gbar + p, 1u);
            step_trace(a, tron, 3, 8, p);
        };
        auto wait_phase = [&](int p) {
            if (wt == 0) step_wait_count(gbar + p, (unsigned)nCTA, a.err, 6, (a.flags & 4) != 0);
            worker_sync();
            step_trace(a, tron, 3, 0, p + 1);
        };

        // ---- phase 0: embedding rows (x, pre-split x * w_norm1[0], sum of squares) ----
        for (int r0 = cta; r0 < M; r0 += nCTA) {
            const int d = a.d_model;
            const bf16_t* src = a.embed + (size_t)a.tok[r0] * d;
            const bf16_t* nw = a.norm1[0];
            float acc = 0.f;
            for (int k = wt; k < d; k += 256) {
                const float v = bf16_to_f32(src[k]);
                a.x[(size_t)r0 * d + k] = v;
                acc += v * v;
                const float xw = v * bf16_to_f32(nw[k]);
                const uint32_t hi = f32_to_bf16_bits(xw);
                a.xs[(size_t)(2 * r0) * d + k] = (bf16_t)hi;
                a.xs[(size_t)(2 * r0 + 1) * d + k] = (bf16_t)f32_to_bf16_bits(xw - __uint_as_float(hi << 16));
            }
            acc = warp_sum(acc);
            if (lane == 0) sh->red[wi] = acc;
            worker_sync();
            if (wt == 0) {
                float t = 0.f;
                for (int i = 0; i < 8; ++i) t += sh->red[i];
                a.ssq[r0] = t;
                for (int i = 1; i < a.d_tiles; ++i) a.ssq[(size_t)i * a.ssq_ld + r0] = 0.f;
            }
            worker_sync();
        }
        arrive(0);

        unsigned acc_use[2] = {0u, 0u};
        // final epilogue of one output element group: thread = feature n of `tile`, batch row m
        auto finish = [&](int ph, int l, int tile, int m, float acc0, float acc1, float res, float nw) {
            const int n = tile * 128 + row;
            if (ph == 0) {
                a.qkv[(size_t)m * a.Nqkv + n] = acc0 * sh->rstd[m];
            } else if (ph == 2) {
                const float sc = sh->rstd[m];
                const float o = silu_f(acc0 * sc) * (acc1 * sc);
                const uint32_t hi = f32_to_bf16_bits(o);
                a.act_s[(size_t)(2 * m) * a.d_ff + n] = (bf16_t)hi;
                a.act_s[(size_t)(2 * m + 1) * a.d_ff + n] = (bf16_t)f32_to_bf16_bits(o - __uint_as_float(hi << 16));
            } else {
                const float o = res + acc0;
                a.x[(size_t)m * a.d_model + n] = o;
                const float xw = o * nw;
                const uint32_t hi = f32_to_bf16_bits(xw);
                a.xs[(size_t)(2 * m) * a.d_model + n] = (bf16_t)hi;
                a.xs[(size_t)(2 * m + 1) * a.d_model + n] = (bf16_t)f32_to_bf16_bits(xw - __uint_as_float(hi << 16));
                const float q2 = warp_sum(o * o);
                if (lane == 0) sh->ssq_s[lg][m] = q2;
            }
        };

        for (int l = 0; l < L; ++l) {
            for (int phx = 0; phx < 5; ++phx) {
                const int p = 1 + l * 5 + phx;
                if (phx == 1) {
                    // ---------------- attention (fused RoPE + KV append) ----------------
                    const int units = M * a.att.Hkv * ns_att;
                    if (cta < units) {
                        wait_phase(p - 1);
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
                if (nseg > 0) {
                    const int NA = a.g[ph].na;
                    const bool resid = (ph == 1 || ph == 3);
                    wait_phase(p - 1);
                    if (ph == 0 || ph == 2) {                         // fused RMSNorm of the input: 1/rms from the partial sums of squares
                        if (wt < M) {
                            float t = 0.f;
                            for (int i = 0; i < a.d_tiles; ++i) t += __ldcg(a.ssq + (size_t)i * a.ssq_ld + wt);
                            sh->rstd[wt] = rsqrtf(t / (float)a.d_model + a.eps);
                        }
                        worker_sync();
                    }
                    const bf16_t* nwp = nullptr;
                    if (ph == 1) nwp = a.norm2[l];
                    if (ph == 3) nwp = (l + 1 < L) ? a.norm1[l + 1] : a.final_norm;
                    bool any_split = false;
                    for (int s = 0; s < nseg; ++s) {
                        const StepSeg sg = sh->pl[ph].seg[s];
                        const int n = sg.tile * 128 + row;
                        const float nw = resid ? bf16_to_f32(nwp[n]) : 1.f;
                        step_wait_mbar(&sh->acc_full[s], acc_use[s] & 1, a.err, 7);
                        ++acc_use[s];
                        tc_fence_after();
                        step_trace(a, tron, 3, 1, p);
                        if (sg.ks == 1) {
                            for (int c = h; c * 16 < M && c < NB / 32; c += 2) {
                                float res[16];
#pragma unroll
                                for (int j = 0; j < 16; ++j)
                                    res[j] = (resid && c * 16 + j < M) ? __ldcg(a.x + (size_t)(c * 16 + j) * a.d_model + n) : 0.f;
                                float v0[32], v1[32];
                                tc_ld32(tmem_base + ((uint32_t)(lg * 32) << 16) + (uint32_t)((s * 2) * NB + c * 32), v0);
                                if (NA == 2) tc_ld32(tmem_base + ((uint32_t)(lg * 32) << 16) + (uint32_t)((s * 2 + 1) * NB + c * 32), v1);
#pragma unroll
                                for (int j = 0; j < 16; ++j) {
                                    const int m = c * 16 + j;
                                    if (m < M) finish(ph, l, sg.tile, m, v0[2 * j] + v0[2 * j + 1], NA == 2 ? v1[2 * j] + v1[2 * j + 1] : 0.f, res[j], nw);
                                }
                            }
                        } else {
                            any_split = true;
                            float* mine = a.scratch + (size_t)(sg.slot0 + sg.rank) * STEP_SCR_SLOT;
                            for (int na = 0; na < NA; ++na)
                                for (int c = h; c * 16 < M && c < NB / 32; c += 2) {
                                    float v[32];
                                    tc_ld32(tmem_base + ((uint32_t)(lg * 32) << 16) + (uint32_t)((s * 2 + na) * NB + c * 32), v);
#pragma unroll
                                    for (int j = 0; j < 16; ++j)
                                        if (c * 16 + j < M) __stcg(mine + ((size_t)na * 64 + c * 16 + j) * 128 + row, v[2 * j] + v[2 * j + 1]);
                                }
                        }
                        if (sg.ks == 1 && resid) {                    // partial sums of squares of the new residual rows of this tile
                            worker_sync();
                            if (wt < M)
                                a.ssq[(size_t)sg.tile * a.ssq_ld + wt] = sh->ssq_s[0][wt] + sh->ssq_s[1][wt] + sh->ssq_s[2][wt] + sh->ssq_s[3][wt];
                            worker_sync();
                        }
                    }
                    step_trace(a, tron, 3, 2, p);
                    if (any_split) {
                        unsigned* tc = tcnt + (size_t)l * a.tiles_per_layer + a.g[ph].tile_ctr_off;
                        if (!(a.flags & 8)) __threadfence();
                        worker_sync();
                        if (wt == 0)
                            for (int s = 0; s < nseg; ++s)
                                if (sh->pl[ph].seg[s].ks > 1) red_release_add(tc + sh->pl[ph].seg[s].tile, 1u);
                        for (int s = 0; s < nseg; ++s) {
                            const StepSeg sg = sh->pl[ph].seg[s];
                            if (sg.ks == 1) continue;
                            if (wt == 0) step_wait_count(tc + sg.tile, (unsigned)sg.ks, a.err, 8, (a.flags & 4) != 0);
                            worker_sync();
                            step_trace(a, tron, 3, 3, p);
                            const int n = sg.tile * 128 + row;
                            const float nw = resid ? bf16_to_f32(nwp[n]) : 1.f;
                            const float* base = a.scratch + (size_t)sg.slot0 * STEP_SCR_SLOT + row;
                            // rank finishes batch rows rank, rank + KS, ...; the two warps of a lane group alternate over them
                            for (int m = sg.rank + sg.ks * h; m < M; m += 2 * sg.ks) {
                                float pv[2][STEP_KS_MAX];
                                const float res = resid ? __ldcg(a.x + (size_t)m * a.d_model + n) : 0.f;
#pragma unroll
                                for (int na = 0; na < 2; ++na)
#pragma unroll
                                    for (int q = 0; q < STEP_KS_MAX; ++q)
                                        pv[na][q] = (q < sg.ks && na < NA) ? __ldcg(base + (size_t)q * STEP_SCR_SLOT + ((size_t)na * 64 + m) * 128) : 0.f;
                                float acc0 = pv[0][0], acc1 = pv[1][0];
#pragma unroll
                                for (int q = 1; q < STEP_KS_MAX; ++q) { acc0 += pv[0][q]; acc1 += pv[1][q]; }   // rank order: deterministic
                                finish(ph, l, sg.tile, m, acc0, acc1, res, nw);
                            }
                            if (resid) {
                                worker_sync();
                                if (wt < M && (wt % sg.ks) == sg.rank)
                                    a.ssq[(size_t)sg.tile * a.ssq_ld + wt] = sh->ssq_s[0][wt] + sh->ssq_s[1][wt] + sh->ssq_s[2][wt] + sh->ssq_s[3][wt];
                                worker_sync();
                            }
                        }
                    }
                    tc_fence_before();
                    step_trace(a, tron, 3, 4, p);
                }
                arrive(p);
            }
        }
    }
    __syncthreads();
    if (warp == 3) {
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
    d.bper = STEP_SLOT / (d.NB * 128);
    for (int i = 0; i < 4; ++i) d.g[i] = s.g[i];
    d.wmaps = reinterpret_cast<const CUtensorMap*>(s.wmaps_dev); d.plan = s.plan_dev;
    d.x = s.x; d.qkv = s.qkv; d.xs = s.xs; d.att_s = s.att_s; d.act_s = s.act_s; d.ssq = s.ssq;
    d.ssq_ld = s.ssq_ld; d.d_tiles = s.d_tiles; d.d_model = s.d_model; d.Nqkv = s.Nqkv; d.qd = s.qd; d.d_ff = s.d_ff;
    d.norm1 = s.norm1_dev; d.norm2 = s.norm2_dev; d.final_norm = s.final_norm; d.embed = s.embed; d.eps = s.eps;
    d.scratch = s.scratch; d.sync_base = s.sync_base; d.gbar_n = s.gbar_n; d.tcnt_n = s.tcnt_n; d.tiles_per_layer = s.tiles_per_layer;
    d.live = s.live; d.pos = s.pos; d.ctx = s.ctx; d.tok = s.tok; d.n_live = s.n_live; d.step = s.step; d.m_max = s.m_max;
    d.att = s.att; d.kv_pool = s.kv_pool; d.layer_stride = s.layer_stride; d.err = s.err; d.trace = s.trace;
    { const char* e = getenv("SAGC_STEP_FLAGS"); d.flags = e ? atoi(e) : 0; }
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
    const int nbi = tc_nb_index(s.m_max);
    const CUtensorMap* bx = reinterpret_cast<const CUtensorMap*>(&s.bmaps[0][nbi]);
    const CUtensorMap* ba = reinterpret_cast<const CUtensorMap*>(&s.bmaps[1][nbi]);
    const CUtensorMap* bc = reinterpret_cast<const CUtensorMap*>(&s.bmaps[2][nbi]);
    cudaError_t e;
    if (s.att.hd == 128) {
        e = cudaFuncSetAttribute(k_decode_step<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e == cudaSuccess) e = cudaLaunchKernelEx(&cfg, k_decode_step<128>, *bx, *ba, *bc, d);
    } else {
        e = cudaFuncSetAttribute(k_decode_step<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e == cudaSuccess) e = cudaLaunchKernelEx(&cfg, k_decode_step<64>, *bx, *ba, *bc, d);
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
