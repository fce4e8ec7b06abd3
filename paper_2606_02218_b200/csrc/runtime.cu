// runtime.cu -- host side of the C ABI (include/sagc.h): model handle, KV pool, step loop,
// CUDA graphs, phase accounting.  No CPU fallback: every compute entry point needs a device.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <string>
#include <vector>

#include "../../include/sagc.h"
#include "common.cuh"
#include "kernels.cuh"

using namespace sagc;

namespace sagc { bool g_pdl_all = false; int g_num_sms = 148; }

#ifdef SAGC_TRACE
namespace sagc { __device__ unsigned long long* g_trace = nullptr; }
static unsigned long long* g_trace_host = nullptr;
extern "C" int sagc_debug_trace(unsigned long long* out, long long cap, long long* n) {
    if (!g_trace_host) { *n = 0; return 0; }
    cudaDeviceSynchronize();
    unsigned long long cnt = 0;
    cudaMemcpy(&cnt, g_trace_host, 8, cudaMemcpyDeviceToHost);
    if ((long long)cnt > cap) cnt = cap;
    if (cnt > (1ull << 20) - 2) cnt = (1ull << 20) - 2;
    cudaMemcpy(out, g_trace_host + 1, cnt * 8, cudaMemcpyDeviceToHost);
    cudaMemset(g_trace_host, 0, 8);
    *n = (long long)cnt;
    return 0;
}
#endif

static thread_local char g_err[512] = "";
static int set_err(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}
extern "C" const char* sagc_last_error(void) { return g_err; }
namespace sagc { int api_set_error(int code, const char* msg) { return set_err(code, "%s", msg); } }   // for entry points in other files
extern "C" const char* sagc_version(void) { return "sagc-rollout 0.1 (sm_100a)"; }

#define CU(x)                                                                                   \
    do {                                                                                        \
        cudaError_t e_ = (x);                                                                   \
        if (e_ != cudaSuccess)                                                                  \
            return set_err(e_ == cudaErrorMemoryAllocation ? SAGC_ENOMEM : SAGC_ECUDA, "%s: %s (%s:%d)", #x, \
                           cudaGetErrorString(e_), __FILE__, __LINE__);                         \
    } while (0)

static int env_int(const char* name, int dflt) {
    const char* s = getenv(name);
    return s ? atoi(s) : dflt;
}

struct GraphKey {
    int m_max, n_splits, kind, dump;
    bool operator<(const GraphKey& o) const {
        if (m_max != o.m_max) return m_max < o.m_max;
        if (n_splits != o.n_splits) return n_splits < o.n_splits;
        if (kind != o.kind) return kind < o.kind;
        return dump < o.dump;
    }
};
struct GraphVal { cudaGraphExec_t exec; int n_kernels; };

struct sagc_model {
    sagc_model_config cfg;
    std::vector<const bf16_t*> wq, wk, wv, wo, wg, wu, wd, norm1, norm2;
    const bf16_t *embed, *lm_head, *final_norm;
    int Nqkv, max_blocks, max_rows, max_splits;
    size_t page_elems, layer_stride;          // bf16 elements per (layer, page) and per layer
    std::vector<void*> allocs;                 // everything cudaMalloc'ed by the handle
    bf16_t* kv_pool;
    float* rope_cs;
    PageState ps;
    // scratch activations
    float *x, *qkv, *att, *act, *logits, *xlast, *part_o, *part_ml;
    float* part_score;
    float* lm_score; int* lm_tok;              // fused LM head + sampler: [lm_sample_grid][64] candidates
    int lm_fused;                              // SAGC_LM_FUSED (default 1): decode steps with <= 64 live rows and no logits dump
    int *counters, *sampled, *row_sid, *row_pos, *row_ctx, *row_tok, *last_idx, *prompt_len_d, *offs_d;
    int row_cap;
    // per-call device buffers (grown on demand)
    int *tok_buf, *len_buf, *forced_len_d, *dump_list_d, *prompt_tok_d;
    size_t tok_cap, forced_cap, dump_cap, prompt_cap;
    uint32_t* sample_params_d;                 // [mode, temperature bits, key lo, key hi]
    // graph cache, valid for one rollout signature
    std::map<GraphKey, GraphVal> graphs;
    std::string signature;
    int last_nseq, last_max_blocks;
    bool use_pdl;
    int gemv_max;
    int tc_min;                                // smallest live-row bucket routed to the tcgen05 path
    int skip_mask;                             // SAGC_SKIP debug ablation: 1 attention, 2 sampler, 4 linears, 8 rope, 16 lm head
    // tcgen05 path: pre-split activation buffers, partial sums of squares, tensor maps
    bool tc_ok;
    bf16_t *xs, *att_s, *act_s;
    float* ssq;
    float* tc_scratch;
    int ssq_ld, d_tiles;
    std::vector<TcMap> wmaps;                  // per layer: q k v o g u d ; last = lm_head
    std::vector<TcMap> kvmaps;                 // per layer: the KV pool as a 2-D tensor (tcgen05 decode attention)
    int att_tc, att_tc_stages;                 // SAGC_ATT_TC (default 1 at head_dim 128; 2 = on every decode step, 0 = never): decode attention on tcgen05; ring depth (0 = deepest)
    TcMap amaps[3][4];                         // {xs, att_s, act_s} x UMMA N {32, 64, 128, 256}
    // persistent decode-step kernel (decode_step.cu): static work plan, device copies of the per-layer tables, counters
    bool step_ok; int n_sm, step_slots, gbar_n, tcnt_n, tiles_per_layer;
    StepGemm step_g[4];
    void* wmaps_d; StepPhasePlan* plan_d; const bf16_t** norm1_d; const bf16_t** norm2_d; unsigned* step_sync; int* step_err;
    float *step_xa, *step_xb, *step_rstd; long long *step_accQ, *step_accO, *step_accG, *step_accD;
    bool step_coop; int step_max_rows;
    unsigned long long* step_trace;            // SAGC_STEP_TRACE=1: in-kernel timeline of one decode step (sagc_debug_step_trace)
    // host-buffer entry point: device staging buffers, grown on demand and kept by the handle
    int *h_prompt, *h_tok, *h_len, *h_stats; float* h_ratio; size_t h_prompt_cap, h_tok_cap, h_len_cap, h_grp_cap;
    float* score_logits; size_t score_cap; int* seq_off_d; size_t seq_off_cap;    // teacher-forced log-prob pass
    cudaStream_t own_stream;                   // used when the caller passes the legacy default stream
    cudaEvent_t own_event;
};

template <typename T>
static int dev_alloc(sagc_model* m, T** p, size_t n) {
    void* q = nullptr;
    cudaError_t e = cudaMalloc(&q, n * sizeof(T) + 256);
    if (e != cudaSuccess) return set_err(SAGC_ENOMEM, "cudaMalloc(%zu bytes): %s", n * sizeof(T), cudaGetErrorString(e));
    m->allocs.push_back(q);
    *p = reinterpret_cast<T*>(q);
    return SAGC_OK;
}
#define DA(ptr, n)                                         \
    do {                                                   \
        int rc_ = dev_alloc(m, &(ptr), (size_t)(n));       \
        if (rc_ != SAGC_OK) { sagc_model_destroy(m); return rc_; } \
    } while (0)

static void clear_graphs(sagc_model* m) {
    for (auto& kv : m->graphs) cudaGraphExecDestroy(kv.second.exec);
    m->graphs.clear();
}

extern "C" void sagc_model_destroy(sagc_model* m) {
    if (!m) return;
    clear_graphs(m);
    if (m->own_stream) cudaStreamDestroy(m->own_stream);
    if (m->own_event) cudaEventDestroy(m->own_event);
    for (void* p : m->allocs) cudaFree(p);
    delete m;
}

static const int PREFILL_ROWS = 2048;

extern "C" int sagc_model_create(const sagc_model_config* cfg, const sagc_weights* w, sagc_model** out) {
    if (!cfg || !w || !out) return set_err(SAGC_EINVAL, "null argument");
    const sagc_model_config& c = *cfg;
    if (c.head_dim != 32 && c.head_dim != 64 && c.head_dim != 128) return set_err(SAGC_EINVAL, "head_dim must be 32, 64 or 128");
    if (c.n_kv_heads <= 0 || c.n_q_heads % c.n_kv_heads != 0 || c.n_q_heads / c.n_kv_heads > 8)
        return set_err(SAGC_EINVAL, "n_q_heads / n_kv_heads must be an integer <= 8");
    if (c.d_model % 32 || c.d_ff % 32 || c.vocab % 16 || (c.n_q_heads * c.head_dim) % 32 || c.n_layers < 0)
        return set_err(SAGC_EINVAL, "d_model, d_ff, q_dim must be multiples of 32 and vocab of 16");
    if (c.page_tokens != 16 && c.page_tokens != 32 && c.page_tokens != 64) return set_err(SAGC_EINVAL, "page_tokens must be 16, 32 or 64");
    if (c.max_seqs < 1 || c.max_seqs > 1024 || c.n_pages < 1 || c.max_ctx < 2) return set_err(SAGC_EINVAL, "bad max_seqs / n_pages / max_ctx");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return set_err(SAGC_ECUDA, "no CUDA device (there is no CPU fallback)");

#ifdef SAGC_TRACE
    if (!g_trace_host && env_int("SAGC_TRACE", 0)) {
        cudaMalloc(&g_trace_host, (1ull << 20) * 8);
        cudaMemset(g_trace_host, 0, 8);
        cudaMemcpyToSymbol(sagc::g_trace, &g_trace_host, sizeof(g_trace_host));
    }
#endif
    sagc_model* m = new sagc_model();
    m->cfg = c;
    m->own_stream = nullptr; m->own_event = nullptr;
    const int L = c.n_layers;
    auto cp = [&](std::vector<const bf16_t*>& v, const void* const* src) {
        v.resize(L);
        for (int l = 0; l < L; ++l) v[l] = reinterpret_cast<const bf16_t*>(src[l]);
    };
    if (L > 0) { cp(m->wq, w->wq); cp(m->wk, w->wk); cp(m->wv, w->wv); cp(m->wo, w->wo); cp(m->wg, w->wg);
                 cp(m->wu, w->wu); cp(m->wd, w->wd); cp(m->norm1, w->norm1); cp(m->norm2, w->norm2); }
    m->embed = reinterpret_cast<const bf16_t*>(w->embed);
    m->lm_head = reinterpret_cast<const bf16_t*>(w->lm_head);
    m->final_norm = reinterpret_cast<const bf16_t*>(w->final_norm);
    m->Nqkv = (c.n_q_heads + 2 * c.n_kv_heads) * c.head_dim;
    m->max_blocks = (c.max_ctx + c.page_tokens - 1) / c.page_tokens;
    m->max_rows = c.max_seqs > PREFILL_ROWS ? c.max_seqs : PREFILL_ROWS;
    m->max_splits = 64;
    m->page_elems = (size_t)2 * c.n_kv_heads * c.page_tokens * c.head_dim;
    m->layer_stride = m->page_elems * (size_t)c.n_pages;
    m->use_pdl = env_int("SAGC_PDL", 1) != 0;
    sagc::g_pdl_all = m->use_pdl;
    { int dev = 0, n = 0; cudaGetDevice(&dev); if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && n > 0) sagc::g_num_sms = n; }
    m->gemv_max = 0;                          // the GEMV kernels serve SAGC_PATH_GEMV only: slower than the tensor-core paths even at 1 row
    m->skip_mask = env_int("SAGC_SKIP", 0);
    m->lm_fused = env_int("SAGC_LM_FUSED", 1);
    m->tc_min = 1;                            // measured: the tcgen05 path beats the register-HMMA tail kernels at every batch size
    m->tok_buf = m->len_buf = m->forced_len_d = m->dump_list_d = m->prompt_tok_d = nullptr;
    m->tok_cap = m->forced_cap = m->dump_cap = m->prompt_cap = 0;
    m->row_cap = 0;
    m->row_sid = m->row_pos = m->row_ctx = m->row_tok = nullptr;
    m->h_prompt = m->h_tok = m->h_len = m->h_stats = nullptr; m->h_ratio = nullptr;
    m->h_prompt_cap = m->h_tok_cap = m->h_len_cap = m->h_grp_cap = 0;
    m->score_logits = nullptr; m->score_cap = 0; m->seq_off_d = nullptr; m->seq_off_cap = 0;
    m->step_ok = false; m->n_sm = 0; m->step_trace = nullptr;

    DA(m->kv_pool, m->layer_stride * (size_t)(L > 0 ? L : 1));
    // finite everywhere: a masked position of a partially filled page meets p = 0 in the tcgen05 attention (0 * NaN would not be 0)
    if (cudaMemset(m->kv_pool, 0, m->layer_stride * (size_t)(L > 0 ? L : 1) * sizeof(bf16_t)) != cudaSuccess) {
        sagc_model_destroy(m);
        return set_err(SAGC_ECUDA, "cudaMemset of the KV pool failed");
    }
    // measured (profiles/r02_attention.md): the tcgen05 kernel wins at head_dim 128 (7B shape: 1.3 - 1.6x in the tail, 1.35x at 256
    // rows); at head_dim 64 its per-tile gain does not pay for its longer prologue / epilogue at the short contexts of those models
    m->att_tc = attention_tc_supports(c.head_dim, c.page_tokens, c.n_q_heads / c.n_kv_heads) ? env_int("SAGC_ATT_TC", c.head_dim == 128 ? 1 : 0) : 0;
    m->att_tc_stages = env_int("SAGC_ATT_TC_STAGES", 0);
    if (m->att_tc) {
        m->kvmaps.resize(L > 0 ? L : 1);
        for (int l = 0; l < L; ++l)
            if (attention_tc_make_map(&m->kvmaps[l], m->kv_pool + (size_t)l * m->layer_stride, c.n_pages, c.n_kv_heads, c.page_tokens, c.head_dim) != 0) {
                m->att_tc = 0;      // no driver entry point for tensor maps: the register-HMMA unit serves decode too
                break;
            }
    }
    // RoPE table: angle = pos * theta^(-2i/hd) and cos/sin in fp64 on the host, stored as fp32
    {
        const int half = c.head_dim / 2;
        std::vector<float> cs((size_t)c.max_ctx * half * 2);
        std::vector<double> inv(half);
        for (int i = 0; i < half; ++i) inv[i] = pow((double)c.rope_theta, -(2.0 * i) / (double)c.head_dim);
        for (int p = 0; p < c.max_ctx; ++p)
            for (int i = 0; i < half; ++i) {
                const double ang = (double)p * inv[i];
                cs[((size_t)p * half + i) * 2] = (float)cos(ang);
                cs[((size_t)p * half + i) * 2 + 1] = (float)sin(ang);
            }
        DA(m->rope_cs, cs.size());
        cudaError_t e = cudaMemcpy(m->rope_cs, cs.data(), cs.size() * sizeof(float), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) { sagc_model_destroy(m); return set_err(SAGC_ECUDA, "rope upload: %s", cudaGetErrorString(e)); }
    }
    PageState& ps = m->ps;
    ps.n_pages = c.n_pages; ps.max_blocks = m->max_blocks; ps.page = c.page_tokens; ps.max_seqs = c.max_seqs;
    ps.log_cap_alloc = c.n_pages * 16 + 65536; ps.log_cap_retire = c.max_seqs;
    DA(ps.free_stack, c.n_pages); DA(ps.refcnt, c.n_pages);
    DA(ps.page_table, (size_t)c.max_seqs * m->max_blocks);
    DA(ps.n_blocks, c.max_seqs); DA(ps.n_shared, c.max_seqs); DA(ps.live, c.max_seqs);
    DA(ps.pos, c.max_seqs); DA(ps.ctx, c.max_seqs); DA(ps.tok, c.max_seqs);
    int* scal = nullptr;
    DA(scal, 16);
    ps.n_free = scal; ps.n_live = scal + 1; ps.step = scal + 2; ps.err = scal + 3; ps.peak_used = scal + 4;
    ps.n_alloc = scal + 5; ps.n_retire = scal + 6;
    DA(ps.alloc_log, (size_t)ps.log_cap_alloc * 3); DA(ps.retire_log, (size_t)ps.log_cap_retire * 2);
    cudaMemset(scal, 0, 16 * sizeof(int));

    const size_t R = m->max_rows;
    DA(m->x, R * c.d_model); DA(m->qkv, R * m->Nqkv); DA(m->att, R * c.n_q_heads * c.head_dim);
    DA(m->act, R * c.d_ff);
    DA(m->logits, (size_t)c.max_seqs * c.vocab);
    DA(m->xlast, (size_t)c.max_seqs * c.d_model);
    DA(m->part_o, (size_t)c.max_seqs * c.n_q_heads * m->max_splits * c.head_dim);
    DA(m->part_ml, (size_t)c.max_seqs * c.n_q_heads * m->max_splits * 2);
    DA(m->counters, R * c.n_kv_heads);
    cudaMemset(m->counters, 0, R * c.n_kv_heads * sizeof(int));
    DA(m->sampled, (size_t)c.max_seqs * SMP_CHUNKS); DA(m->part_score, (size_t)c.max_seqs * SMP_CHUNKS); DA(m->last_idx, c.max_seqs); DA(m->prompt_len_d, c.max_seqs);
    DA(m->offs_d, c.max_seqs + 1);
    DA(m->lm_score, (size_t)LM_MAX_PARTS * 64); DA(m->lm_tok, (size_t)LM_MAX_PARTS * 64);
    DA(m->sample_params_d, 4);
    m->last_nseq = 0; m->last_max_blocks = m->max_blocks;
    {
        const int qd = c.n_q_heads * c.head_dim, kvd = c.n_kv_heads * c.head_dim;
        m->tc_ok = env_int("SAGC_TC", 1) != 0 && L > 0 && c.d_model % 128 == 0 && qd % 128 == 0 && kvd % 128 == 0 &&
                   c.d_ff % 128 == 0 && c.vocab % 128 == 0;
        m->xs = m->att_s = m->act_s = nullptr; m->ssq = nullptr;
        if (m->tc_ok) {
            const size_t Rp = ((R + 127) / 128) * 128;
            m->ssq_ld = (int)Rp; m->d_tiles = c.d_model / 128;
            DA(m->xs, 2 * Rp * c.d_model); DA(m->att_s, 2 * Rp * qd); DA(m->act_s, 2 * Rp * c.d_ff);
            DA(m->ssq, (size_t)m->d_tiles * Rp);
            DA(m->tc_scratch, TC_SCRATCH_FLOATS);
            cudaMemset(m->xs, 0, 2 * Rp * c.d_model * 2); cudaMemset(m->att_s, 0, 2 * Rp * qd * 2);
            cudaMemset(m->act_s, 0, 2 * Rp * c.d_ff * 2); cudaMemset(m->ssq, 0, (size_t)m->d_tiles * Rp * 4);
            m->wmaps.resize((size_t)L * 7 + 1);
            int bad = 0;
            for (int l = 0; l < L; ++l) {
                TcMap* w7 = &m->wmaps[(size_t)l * 7];
                bad |= tc_make_map(&w7[0], m->wq[l], qd, c.d_model, 128);
                bad |= tc_make_map(&w7[1], m->wk[l], kvd, c.d_model, 128);
                bad |= tc_make_map(&w7[2], m->wv[l], kvd, c.d_model, 128);
                bad |= tc_make_map(&w7[3], m->wo[l], c.d_model, qd, 128);
                bad |= tc_make_map(&w7[4], m->wg[l], c.d_ff, c.d_model, 128);
                bad |= tc_make_map(&w7[5], m->wu[l], c.d_ff, c.d_model, 128);
                bad |= tc_make_map(&w7[6], m->wd[l], c.d_model, c.d_ff, 128);
            }
            bad |= tc_make_map(&m->wmaps[(size_t)L * 7], m->lm_head, c.vocab, c.d_model, 128);
            for (int i = 0; i < 4; ++i) {
                bad |= tc_make_map(&m->amaps[0][i], m->xs, 2 * (long long)Rp, c.d_model, 32 << i);
                bad |= tc_make_map(&m->amaps[1][i], m->att_s, 2 * (long long)Rp, qd, 32 << i);
                bad |= tc_make_map(&m->amaps[2][i], m->act_s, 2 * (long long)Rp, c.d_ff, 32 << i);
            }
            if (bad) { sagc_model_destroy(m); return set_err(SAGC_ECUDA, "cuTensorMapEncodeTiled failed"); }
        }
        // persistent decode-step kernel: one CTA per SM, static unit -> CTA plan, tensor maps / norm gains in device tables
        m->step_ok = false; m->wmaps_d = nullptr; m->plan_d = nullptr; m->norm1_d = m->norm2_d = nullptr; m->step_sync = nullptr; m->step_err = nullptr;
        {
            int dev = 0, smem_optin = 0;
            cudaGetDevice(&dev);
            cudaDeviceGetAttribute(&m->n_sm, cudaDevAttrMultiProcessorCount, dev);
            cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
            m->step_slots = step_ring_slots(smem_optin);
            m->step_coop = env_int("SAGC_STEP_COOP", 1) != 0;
            m->step_max_rows = env_int("SAGC_STEP_MAXROWS", 64);
            std::vector<StepPhasePlan> plan;
            // SAGC_STEP=1 routes decode steps with <= 64 live rows through the persistent decode-step kernel.  Off by default:
            // measured slower than the per-layer kernels on every shape (~1 us per L2 hop, 5 hops per phase)
            if (m->tc_ok && env_int("SAGC_STEP", 0) != 0 && c.head_dim >= 64 && m->n_sm > 0 && m->step_slots >= 4 &&
                build_step_plan(m->n_sm, c.d_model, qd, kvd, c.d_ff, m->step_g, plan, &m->tiles_per_layer)) {
                m->gbar_n = 2 + 5 * L; m->tcnt_n = 0;
                unsigned char* wm = nullptr;
                DA(wm, (size_t)L * 7 * sizeof(TcMap)); m->wmaps_d = wm;
                DA(m->plan_d, plan.size()); DA(m->norm1_d, L); DA(m->norm2_d, L);
                DA(m->step_sync, (size_t)2 * (m->gbar_n + m->tcnt_n)); DA(m->step_err, 1);
                DA(m->step_xa, (size_t)64 * c.d_model); DA(m->step_xb, (size_t)64 * c.d_model); DA(m->step_rstd, 128);
                DA(m->step_accQ, (size_t)64 * m->Nqkv); DA(m->step_accO, (size_t)64 * c.d_model);
                DA(m->step_accG, (size_t)64 * 2 * c.d_ff); DA(m->step_accD, (size_t)64 * c.d_model);
                cudaMemcpy(m->wmaps_d, m->wmaps.data(), (size_t)L * 7 * sizeof(TcMap), cudaMemcpyHostToDevice);
                cudaMemcpy(m->plan_d, plan.data(), plan.size() * sizeof(StepPhasePlan), cudaMemcpyHostToDevice);
                cudaMemcpy(m->norm1_d, m->norm1.data(), L * sizeof(void*), cudaMemcpyHostToDevice);
                cudaMemcpy(m->norm2_d, m->norm2.data(), L * sizeof(void*), cudaMemcpyHostToDevice);
                cudaMemset(m->step_sync, 0, (size_t)2 * (m->gbar_n + m->tcnt_n) * sizeof(unsigned));
                cudaMemset(m->step_err, 0, sizeof(int));
                m->step_ok = true;
                if (env_int("SAGC_STEP_TRACE", 0)) {
                    DA(m->step_trace, 2 + 2 * 16000);
                    cudaMemset(m->step_trace, 0, (2 + 2 * 16000) * sizeof(unsigned long long));
                }
            }
        }
    }
    cudaError_t e = cudaDeviceSynchronize();
    if (e != cudaSuccess) { sagc_model_destroy(m); return set_err(SAGC_ECUDA, "create: %s", cudaGetErrorString(e)); }
    *out = m;
    return SAGC_OK;
}

// ---------------------------------------------------------------------------------------
// forward pass over `m_max` activation rows (decode: live slots; prefill: prompt positions)
// ---------------------------------------------------------------------------------------
struct RowSet {
    const int* sid; const int* pos; const int* ctx; const int* tok; const int* m_dev; int m_max;
};

static int pick_kind(const sagc_model* m, int path, int m_max) {
    if (path == SAGC_PATH_GEMV) return LIN_GEMV;
    if (path == SAGC_PATH_GEMM) return m->tc_ok ? LIN_TC : LIN_MMA;
    if (m_max <= m->gemv_max) return LIN_GEMV;
    if (m_max < m->tc_min || !m->tc_ok) return LIN_MMA;   // tail: register-resident HMMA kernel
    return LIN_TC;                                    // large batch / prefill: tcgen05 + TMEM
}

static int enqueue_layers_tc(sagc_model* m, const RowSet& rs, int n_splits, cudaStream_t st);

// layers only (x ends up holding the final residual stream).  Returns kernels launched or <0.
static int enqueue_layers(sagc_model* m, const RowSet& rs, int n_splits_enc, int kind, cudaStream_t st) {
    const int n_splits = n_splits_enc & 0xfff;
    const sagc_model_config& c = m->cfg;
    if (kind == LIN_TC) return enqueue_layers_tc(m, rs, n_splits_enc, st);
    int n = 0, r;
#define LAUNCH(expr) do { r = (expr); if (r < 0) return -1; n += r; } while (0)
    const int skip = m->skip_mask;
    LAUNCH(launch_embed(m->embed, rs.tok, rs.m_dev, rs.m_max, c.d_model, m->x, st));
    const int qd = c.n_q_heads * c.head_dim, kvd = c.n_kv_heads * c.head_dim;
    for (int l = 0; l < c.n_layers; ++l) {
        LinearArgs a = {};
        a.W[0] = m->wq[l]; a.W[1] = m->wk[l]; a.W[2] = m->wv[l];
        a.rows[0] = qd; a.rows[1] = kvd; a.rows[2] = kvd;
        a.X = m->x; a.norm_w = m->norm1[l]; a.eps = c.rms_eps; a.Y = m->qkv; a.R = nullptr; a.ldy = m->Nqkv;
        a.K = c.d_model; a.N = m->Nqkv; a.m_dev = rs.m_dev; a.m_max = rs.m_max; a.epi = EPI_STORE; a.kind = kind;
        a.pdl = m->use_pdl;
        if (!(skip & 4)) LAUNCH(launch_linear(a, st));

        RopeArgs ra = {};
        ra.qkv = m->qkv; ra.row_sid = rs.sid; ra.row_pos = rs.pos; ra.m_dev = rs.m_dev; ra.m_max = rs.m_max;
        ra.rope_cs = m->rope_cs; ra.kv_layer = m->kv_pool + (size_t)l * m->layer_stride;
        ra.page_table = m->ps.page_table; ra.max_blocks = m->max_blocks; ra.page = c.page_tokens;
        ra.Hq = c.n_q_heads; ra.Hkv = c.n_kv_heads; ra.hd = c.head_dim;
        if (!(skip & 8)) LAUNCH(launch_rope_append(ra, st));

        AttnArgs aa = {};
        aa.q = m->qkv; aa.ldq = m->Nqkv; aa.kv_layer = ra.kv_layer; aa.page_table = m->ps.page_table;
        aa.max_blocks = m->max_blocks; aa.row_sid = rs.sid; aa.row_ctx = rs.ctx; aa.m_dev = rs.m_dev; aa.m_max = rs.m_max;
        aa.Hq = c.n_q_heads; aa.Hkv = c.n_kv_heads; aa.hd = c.head_dim; aa.page = c.page_tokens;
        aa.n_splits = n_splits; aa.part_o = m->part_o; aa.part_ml = m->part_ml; aa.counters = m->counters;
        aa.out = m->att; aa.prefetch = (rs.m_dev != nullptr) ? 1 : 0;
        if (!(skip & 1)) LAUNCH(launch_attention(aa, st));

        LinearArgs o = {};
        o.W[0] = m->wo[l]; o.rows[0] = c.d_model; o.X = m->att; o.Y = m->x; o.R = m->x; o.ldy = c.d_model;
        o.K = qd; o.N = c.d_model; o.m_dev = rs.m_dev; o.m_max = rs.m_max; o.epi = EPI_RESID; o.kind = kind;
        o.pdl = m->use_pdl; o.eps = c.rms_eps;
        if (!(skip & 4)) LAUNCH(launch_linear(o, st));

        LinearArgs gu = {};
        gu.W[0] = m->wg[l]; gu.W[1] = m->wu[l]; gu.rows[0] = c.d_ff; gu.rows[1] = c.d_ff;
        gu.X = m->x; gu.norm_w = m->norm2[l]; gu.eps = c.rms_eps; gu.Y = m->act; gu.ldy = c.d_ff;
        gu.K = c.d_model; gu.N = c.d_ff; gu.m_dev = rs.m_dev; gu.m_max = rs.m_max; gu.epi = EPI_SWIGLU; gu.kind = kind;
        gu.pdl = m->use_pdl;
        if (!(skip & 4)) LAUNCH(launch_linear(gu, st));

        LinearArgs dn = {};
        dn.W[0] = m->wd[l]; dn.rows[0] = c.d_model; dn.X = m->act; dn.Y = m->x; dn.R = m->x; dn.ldy = c.d_model;
        dn.K = c.d_ff; dn.N = c.d_model; dn.m_dev = rs.m_dev; dn.m_max = rs.m_max; dn.epi = EPI_RESID; dn.kind = kind;
        dn.pdl = m->use_pdl; dn.eps = c.rms_eps;
        if (!(skip & 4)) LAUNCH(launch_linear(dn, st));
    }
    return n;
}

// tcgen05 variant of the layer stack: activations travel between kernels as pre-split bf16 rows
// (xs / att_s / act_s), the RMSNorm gain is folded in by the producer and 1/rms by the consumer.
static int enqueue_layers_tc(sagc_model* m, const RowSet& rs, int n_splits_enc, cudaStream_t st) {
    const bool att_tc_step = (n_splits_enc & 0x1000) != 0;
    const int n_splits = n_splits_enc & 0xfff;
    const sagc_model_config& c = m->cfg;
    int n = 0, r;
    const int skip = m->skip_mask;
    const int qd = c.n_q_heads * c.head_dim, kvd = c.n_kv_heads * c.head_dim;
    const int nbi = tc_nb_index(rs.m_max);
    LAUNCH(launch_embed_split(m->embed, rs.tok, rs.m_dev, rs.m_max, c.d_model, m->x, m->norm1[0], m->xs, m->ssq,
                              m->ssq_ld, m->d_tiles, st));
    for (int l = 0; l < c.n_layers; ++l) {
        const TcMap* w7 = &m->wmaps[(size_t)l * 7];
        TcLinearArgs t = {};
        t.a[0] = &w7[0]; t.a[1] = &w7[1]; t.a[2] = &w7[2]; t.seg_rows[0] = qd; t.seg_rows[1] = kvd; t.seg_rows[2] = kvd;
        t.b = &m->amaps[0][nbi]; t.K = c.d_model; t.N = m->Nqkv; t.m_dev = rs.m_dev; t.m_max = rs.m_max; t.epi = EPI_QKV;
        t.Y = m->qkv; t.ldy = m->Nqkv; t.ssq_in = m->ssq; t.ssq_in_tiles = m->d_tiles; t.ssq_ld = m->ssq_ld;
        t.eps = c.rms_eps; t.k_norm = c.d_model; t.pdl = m->use_pdl; t.scratch = m->tc_scratch;
        // RoPE + bf16 KV append run in this GEMM's epilogue (no separate kernel on the tcgen05 path)
        bf16_t* kv_layer = m->kv_pool + (size_t)l * m->layer_stride;
        t.rope_cs = m->rope_cs; t.row_pos = rs.pos; t.row_sid = rs.sid; t.page_table = m->ps.page_table; t.kv_layer = kv_layer;
        t.max_blocks = m->max_blocks; t.page = c.page_tokens; t.Hkv = c.n_kv_heads; t.hd = c.head_dim; t.q_rows = qd; t.kv_rows = kvd;
        const bool fuse_rope = false;          // RoPE + append in the QKV epilogue (EPI_QKV): measured -4% in FULL, kept off
        if (!fuse_rope) t.epi = EPI_STORE;
        if (!(skip & 4)) LAUNCH(launch_linear_tc(t, st));
        // decode: RoPE + KV append are done inside the attention kernel (one launch less per layer)
        const bool fuse_att = !fuse_rope && rs.m_dev != nullptr && c.head_dim >= 64;
        if (!fuse_rope && !fuse_att) {
            RopeArgs ra = {};
            ra.qkv = m->qkv; ra.row_sid = rs.sid; ra.row_pos = rs.pos; ra.m_dev = rs.m_dev; ra.m_max = rs.m_max;
            ra.rope_cs = m->rope_cs; ra.kv_layer = kv_layer; ra.page_table = m->ps.page_table; ra.max_blocks = m->max_blocks;
            ra.page = c.page_tokens; ra.Hq = c.n_q_heads; ra.Hkv = c.n_kv_heads; ra.hd = c.head_dim;
            LAUNCH(launch_rope_append(ra, st));
        }

        AttnArgs aa = {};
        aa.q = m->qkv; aa.ldq = m->Nqkv; aa.kv_layer = kv_layer; aa.page_table = m->ps.page_table;
        aa.max_blocks = m->max_blocks; aa.row_sid = rs.sid; aa.row_ctx = rs.ctx; aa.m_dev = rs.m_dev; aa.m_max = rs.m_max;
        aa.Hq = c.n_q_heads; aa.Hkv = c.n_kv_heads; aa.hd = c.head_dim; aa.page = c.page_tokens;
        aa.n_splits = n_splits; aa.part_o = m->part_o; aa.part_ml = m->part_ml; aa.counters = m->counters;
        aa.out = m->att; aa.prefetch = (rs.m_dev != nullptr) ? 1 : 0; aa.out_split = m->att_s; aa.ld_split = qd;
        aa.fuse_rope = fuse_att ? 1 : 0; aa.rope_cs = m->rope_cs; aa.row_pos = rs.pos; aa.kv_layer_w = kv_layer;
        if (!(skip & 1)) {
            if (fuse_att && m->att_tc && att_tc_step) LAUNCH(launch_attention_tc(aa, &m->kvmaps[l], m->att_tc_stages, st));
            else LAUNCH(launch_attention(aa, st));
        }

        TcLinearArgs o = {};
        o.a[0] = &w7[3]; o.seg_rows[0] = c.d_model; o.b = &m->amaps[1][nbi]; o.K = qd; o.N = c.d_model;
        o.m_dev = rs.m_dev; o.m_max = rs.m_max; o.epi = EPI_RESID; o.Y = m->x; o.R = m->x; o.ldy = c.d_model;
        o.xs_out = m->xs; o.ld_xs = c.d_model; o.norm_next = m->norm2[l]; o.ssq_out = m->ssq; o.ssq_ld = m->ssq_ld;
        o.eps = c.rms_eps; o.pdl = m->use_pdl; o.scratch = m->tc_scratch;
        if (!(skip & 4)) LAUNCH(launch_linear_tc(o, st));

        TcLinearArgs gu = {};
        gu.a[0] = &w7[4]; gu.a[1] = &w7[5]; gu.seg_rows[0] = c.d_ff; gu.seg_rows[1] = c.d_ff;
        gu.b = &m->amaps[0][nbi]; gu.K = c.d_model; gu.N = c.d_ff; gu.m_dev = rs.m_dev; gu.m_max = rs.m_max;
        gu.epi = EPI_SWIGLU; gu.xs_out = m->act_s; gu.ld_xs = c.d_ff; gu.ssq_in = m->ssq; gu.ssq_in_tiles = m->d_tiles;
        gu.ssq_ld = m->ssq_ld; gu.eps = c.rms_eps; gu.k_norm = c.d_model; gu.pdl = m->use_pdl; gu.scratch = m->tc_scratch;
        if (!(skip & 4)) LAUNCH(launch_linear_tc(gu, st));

        TcLinearArgs dn = {};
        dn.a[0] = &w7[6]; dn.seg_rows[0] = c.d_model; dn.b = &m->amaps[2][nbi]; dn.K = c.d_ff; dn.N = c.d_model;
        dn.m_dev = rs.m_dev; dn.m_max = rs.m_max; dn.epi = EPI_RESID; dn.Y = m->x; dn.R = m->x; dn.ldy = c.d_model;
        dn.xs_out = m->xs; dn.ld_xs = c.d_model; dn.norm_next = (l + 1 < c.n_layers) ? m->norm1[l + 1] : m->final_norm;
        dn.ssq_out = m->ssq; dn.ssq_ld = m->ssq_ld; dn.eps = c.rms_eps; dn.pdl = m->use_pdl; dn.scratch = m->tc_scratch;
        if (!(skip & 4)) LAUNCH(launch_linear_tc(dn, st));
    }
    return n;
}
#undef LAUNCH

// final norm + LM head over rows of `xsrc` -> m->logits
static int enqueue_lm_head(sagc_model* m, const float* xsrc, const int* m_dev, int m_max, int kind, cudaStream_t st,
                           float* Y = nullptr) {
    const sagc_model_config& c = m->cfg;
    if (m->skip_mask & 16) return 0;
    if (!Y) Y = m->logits;
    if (kind == LIN_TC && xsrc == m->x) {
        // decode: the last down-projection left x * w_final pre-split in xs and its row sums in ssq
        TcLinearArgs t = {};
        t.a[0] = &m->wmaps[(size_t)c.n_layers * 7]; t.seg_rows[0] = c.vocab; t.b = &m->amaps[0][tc_nb_index(m_max)];
        t.K = c.d_model; t.N = c.vocab; t.m_dev = m_dev; t.m_max = m_max; t.epi = EPI_STORE; t.Y = Y; t.ldy = c.vocab;
        t.ssq_in = m->ssq; t.ssq_in_tiles = m->d_tiles; t.ssq_ld = m->ssq_ld; t.eps = c.rms_eps; t.k_norm = c.d_model;
        t.pdl = m->use_pdl; t.scratch = m->tc_scratch;
        return launch_linear_tc(t, st);
    }
    if (kind == LIN_TC) kind = LIN_MMA;          // gathered fp32 rows (first token): register HMMA path
    LinearArgs a = {};
    a.W[0] = m->lm_head; a.rows[0] = c.vocab; a.X = xsrc; a.norm_w = m->final_norm; a.eps = c.rms_eps;
    a.Y = Y; a.ldy = c.vocab; a.K = c.d_model; a.N = c.vocab; a.m_dev = m_dev; a.m_max = m_max;
    a.epi = EPI_STORE; a.kind = kind; a.pdl = m->use_pdl;
    return launch_linear(a, st);
}

template <typename T>
static int grow(sagc_model* m, T** p, size_t* cap, size_t need, bool* changed) {
    if (need <= *cap && *p) return SAGC_OK;
    T* q = nullptr;
    size_t n = need + need / 4 + 64;
    int rc = dev_alloc(m, &q, n);
    if (rc != SAGC_OK) return rc;
    *p = q; *cap = n;      // the old block stays owned by the handle until destroy
    if (changed) *changed = true;
    return SAGC_OK;
}

static int round_bucket(int live) {
    if (live <= 8) return 8;
    if (live <= 16) return 16;
    if (live <= 32) return 32;
    return ((live + 63) / 64) * 64;
}

static constexpr int ATT_TC_FLAG = 0x1000;      // pick_splits: this step's attention runs on the tcgen05 kernel
static int pick_splits(const sagc_model* m, int m_bucket, int ctx_bound, int live) {
    const int ctas = m_bucket * m->cfg.n_kv_heads;
    const int target = (3 * sagc::g_num_sms) / 2;
    int want = target / ctas;                  // ~1.5 CTAs per SM; no split once the grid fills the chip
    if (want < 1) want = 1;
    int cap = ctx_bound / 128;
    if (cap < 1) cap = 1;
    if (want > cap) want = cap;
    if (want > m->max_splits) want = m->max_splits;
    int s = 1;
    while (s * 2 <= want) s *= 2;
    const int smax = 8;                       // <= 8 splits merge inside a cluster (attention.cu)
    if (s > smax) s = smax;
    // The tcgen05 kernel pays ~4 us more prologue / epilogue / L2 merge than the register-HMMA unit and streams a tile in half
    // the time: it wins from ~2 000 cached tokens per row, or at any context once the grid is large (256 rows x 1 100 tokens:
    // 104 vs 159 us); with few rows at ~1 000 tokens it loses (19.5 vs 17.1 us).  The choice travels in bit 12 of the split count.
    if (m->att_tc && m->cfg.head_dim >= 64 && (m_bucket >= 32 || ctx_bound >= 2048 || m->att_tc > 1)) {
        // tcgen05 decode attention: one CTA per SM (the K/V ring fills shared memory), >= 2 tiles of 128 tokens per split,
        // partials merged through L2 by the last arriver, so ANY split count works: it is sized by the rows that are really
        // live (exact with forced lengths, a polled upper bound otherwise), not by the batch bucket -- in the 7B tail the
        // bucket of 8 holds 4.2 rows on average and attention is 25 % of the step (SAGC_SKIP ablation).  More than 16 splits
        // cost more in the merge than they save in the scan (1 row x 16 000 tokens: 26 us with 16 splits, 30 us with 32).
        const int rows = live > 0 && live < m_bucket ? live : m_bucket;
        int w2 = sagc::g_num_sms / (rows * m->cfg.n_kv_heads);
        const int cap2 = ctx_bound / 256;
        if (w2 > cap2) w2 = cap2;
        if (w2 > 16) w2 = 16;
        if (w2 > m->max_splits) w2 = m->max_splits;
        s = w2 < 1 ? 1 : w2;
        s |= ATT_TC_FLAG;
    }
    return s;
}

// ---------------------------------------------------------------------------------------
// sagc_rollout_group
// ---------------------------------------------------------------------------------------
// the persistent decode-step kernel covers the tcgen05 path at <= 64 live rows (head_dim 64 / 128)
static bool step_kernel_applies(const sagc_model* m, int kind, int m_bucket) {
    return m->step_ok && kind == LIN_TC && m_bucket <= m->step_max_rows && m->skip_mask == 0;
}

static int enqueue_decode_step(sagc_model* m, const RolloutDev& rd, int m_bucket, int n_splits, int kind,
                               int n_dump, float* dump_out, cudaStream_t st, std::vector<cudaEvent_t>* evs = nullptr) {
    // SAGC_FLAG_TIME_KERNELS: four events per step bracket the layer stack, the LM head + sampler and the advance kernel
    auto stamp = [&]() { if (evs) { cudaEvent_t e; cudaEventCreate(&e); cudaEventRecord(e, st); evs->push_back(e); } };
    stamp();
    RowSet rs = {m->ps.live, m->ps.pos, m->ps.ctx, m->ps.tok, m->ps.n_live, m_bucket};
    const sagc_model_config& c = m->cfg;
    int n;
    if (step_kernel_applies(m, kind, m_bucket)) {
        // a5 - a10 of every layer in ONE persistent kernel (decode_step.cu)
        StepLaunch s = {};
        s.n_layers = c.n_layers; s.n_cta = m->n_sm; s.n_slots = m->step_slots; s.m_max = m_bucket;
        for (int i = 0; i < 4; ++i) s.g[i] = m->step_g[i];
        s.wmaps_dev = m->wmaps_d; s.plan_dev = m->plan_d;
        s.xa = m->step_xa; s.xb = m->step_xb; s.accQ = m->step_accQ; s.accO = m->step_accO; s.accG = m->step_accG; s.accD = m->step_accD;
        s.rstd1 = m->step_rstd; s.rstd2 = m->step_rstd + 64;
        s.x = m->x; s.xs = m->xs; s.att_s = m->att_s; s.ssq = m->ssq;
        s.ssq_ld = m->ssq_ld; s.d_tiles = m->d_tiles; s.d_model = c.d_model; s.Nqkv = m->Nqkv; s.qd = c.n_q_heads * c.head_dim; s.d_ff = c.d_ff;
        s.norm1_dev = m->norm1_d; s.norm2_dev = m->norm2_d; s.final_norm = m->final_norm; s.embed = m->embed; s.eps = c.rms_eps;
        s.sync_base = m->step_sync; s.gbar_n = m->gbar_n;
        s.live = m->ps.live; s.pos = m->ps.pos; s.ctx = m->ps.ctx; s.tok = m->ps.tok; s.n_live = m->ps.n_live; s.step = m->ps.step;
        AttnArgs& aa = s.att;
        aa.q = nullptr; aa.q_fx = m->step_accQ; aa.q_rstd = m->step_rstd; aa.ldq = m->Nqkv; aa.page_table = m->ps.page_table;
        aa.max_blocks = m->max_blocks; aa.row_sid = m->ps.live;
        aa.row_ctx = m->ps.ctx; aa.m_dev = m->ps.n_live; aa.m_max = m_bucket; aa.Hq = c.n_q_heads; aa.Hkv = c.n_kv_heads; aa.hd = c.head_dim;
        aa.page = c.page_tokens; aa.n_splits = 1; aa.part_o = m->part_o; aa.part_ml = m->part_ml; aa.counters = m->counters; aa.out = m->att;
        aa.out_split = m->att_s; aa.ld_split = c.n_q_heads * c.head_dim; aa.fuse_rope = 1; aa.rope_cs = m->rope_cs; aa.row_pos = m->ps.pos;
        aa.prefetch = 0; aa.cluster_merge = 0;
        s.kv_pool = m->kv_pool; s.layer_stride = m->layer_stride; s.err = m->step_err; s.trace = m->step_trace;
        s.cooperative = m->step_coop; s.pdl = m->use_pdl && !m->step_coop;
        n = launch_decode_step(s, st);
    } else {
        n = enqueue_layers(m, rs, n_splits, kind, st);
    }
    if (n < 0) return -1;
    stamp();
    if (m->lm_fused && kind == LIN_TC && m_bucket <= 64 && n_dump == 0 && (c.vocab % 128) == 0 && !(m->skip_mask & (2 | 16))) {
        // a11 + a12 in one persistent kernel: the logits never reach HBM
        LmSampleArgs f = {};
        f.a = &m->wmaps[(size_t)c.n_layers * 7]; f.b = &m->amaps[0][tc_nb_index(m_bucket)]; f.K = c.d_model; f.V = c.vocab;
        f.m_dev = m->ps.n_live; f.m_max = m_bucket; f.ssq_in = m->ssq; f.ssq_in_tiles = m->d_tiles; f.ssq_ld = m->ssq_ld;
        f.eps = c.rms_eps; f.k_norm = c.d_model; f.row_sid = m->ps.live; f.step_dev = m->ps.step; f.params = m->sample_params_d;
        f.part_score = m->lm_score; f.part_tok = m->lm_tok; f.part_ld = 64; f.Y = nullptr; f.ldy = c.vocab; f.pdl = m->use_pdl;
        int r = launch_lmhead_sample(f, st);
        if (r < 0) return -1;
        n += r;
        stamp();
        n += launch_advance(m->ps, rd, m->lm_score, m->lm_tok, 0, st, lm_sample_grid(c.vocab), 64, 1);
        stamp();
        return n;
    }
    int r = enqueue_lm_head(m, m->x, m->ps.n_live, m_bucket, kind, st);
    if (r < 0) return -1;
    n += r;
    SampleArgs sa = {};
    sa.logits = m->logits; sa.V = m->cfg.vocab; sa.row_sid = m->ps.live; sa.step_dev = m->ps.step;
    sa.m_dev = m->ps.n_live; sa.m_max = m_bucket; sa.params = m->sample_params_d; sa.row_div = 1;
    sa.part_score = m->part_score; sa.part_tok = m->sampled;
    if (!(m->skip_mask & 2)) n += launch_sample(sa, st);
    if (n_dump > 0)
        n += launch_dump_logits(m->dump_list_d, n_dump, m->ps.step, m->ps.live, m->ps.n_live, 1, m->logits,
                                m->cfg.vocab, dump_out, st);
    stamp();
    n += launch_advance(m->ps, rd, m->part_score, m->sampled, 0, st);
    stamp();
    return n;
}

static int phase_of(int live, int nseq) {
    if (live <= 8 && 2 * live < nseq) return 2;    // TAIL
    if (2 * live >= nseq) return 0;                // FULL
    return 1;                                      // MID
}

extern "C" int sagc_rollout_group(sagc_model* m, const int32_t* prompt_tokens, const int32_t* prompt_offsets,
                                  int32_t n_prompts, int32_t G, const sagc_rollout_params* prm,
                                  int32_t* out_tokens, int32_t* out_lengths, float* out_ratio,
                                  int32_t* out_len_stats, sagc_rollout_timing* timing, void* stream) {
    if (!m || !prompt_offsets || !prm || !out_tokens || !out_lengths) return set_err(SAGC_EINVAL, "null argument");
    const sagc_model_config& c = m->cfg;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    if (st == nullptr || st == cudaStreamLegacy) {
        // the legacy default stream cannot be captured into a graph: run on an internal stream
        // ordered after it (the call synchronises before returning, so later work is ordered too)
        if (!m->own_stream) {
            CU(cudaStreamCreateWithFlags(&m->own_stream, cudaStreamNonBlocking));
            CU(cudaEventCreateWithFlags(&m->own_event, cudaEventDisableTiming));
        }
        CU(cudaEventRecord(m->own_event, st));
        CU(cudaStreamWaitEvent(m->own_stream, m->own_event, 0));
        st = m->own_stream;
    }
    const int nseq = n_prompts * G;
    const int max_new = prm->max_new_tokens;
    const bool structure_only = (prm->flags & SAGC_FLAG_STRUCTURE_ONLY) != 0;
    const bool time_kernels = (prm->flags & SAGC_FLAG_TIME_KERNELS) != 0 && timing != nullptr;
    const bool use_graph = !(prm->flags & SAGC_FLAG_NO_GRAPH) && !time_kernels;
    std::vector<cudaEvent_t> kev;
    if (n_prompts < 1 || G < 1 || nseq > c.max_seqs) return set_err(SAGC_EINVAL, "n_prompts*G = %d exceeds max_seqs = %d", nseq, c.max_seqs);
    if (max_new < 1) return set_err(SAGC_EINVAL, "max_new_tokens must be >= 1");
    if (structure_only && !prm->forced_lengths) return set_err(SAGC_EINVAL, "STRUCTURE_ONLY needs forced_lengths");
    if (!structure_only && !prompt_tokens) return set_err(SAGC_EINVAL, "prompt_tokens is null");
    if (prm->mode != SAGC_MODE_GREEDY && prm->mode != SAGC_MODE_GUMBEL) return set_err(SAGC_EINVAL, "bad sampling mode");
    if (prm->mode == SAGC_MODE_GUMBEL && !(prm->temperature > 0.f)) return set_err(SAGC_EINVAL, "temperature must be > 0");
    if (prompt_offsets[0] != 0) return set_err(SAGC_EINVAL, "prompt_offsets[0] must be 0");
    std::vector<int> plen(n_prompts);
    int total_rows = 0, pmax = 0;
    for (int p = 0; p < n_prompts; ++p) {
        plen[p] = prompt_offsets[p + 1] - prompt_offsets[p];
        if (plen[p] < 1) return set_err(SAGC_EINVAL, "prompt %d is empty", p);
        if (plen[p] + max_new > c.max_ctx) return set_err(SAGC_EINVAL, "prompt %d: length + max_new_tokens exceeds max_ctx", p);
        total_rows += plen[p];
        if (plen[p] > pmax) pmax = plen[p];
    }
    if (prm->n_dump > 0 && (!prm->dump_sid_t || !prm->dump_logits)) return set_err(SAGC_EINVAL, "dump arrays are null");

    // ---- per-call device buffers ------------------------------------------------------
    bool changed = false;
    int rc;
    if ((rc = grow(m, &m->tok_buf, &m->tok_cap, (size_t)nseq * max_new, &changed)) != SAGC_OK) return rc;
    if (!m->len_buf) { size_t cap = 0; if ((rc = grow(m, &m->len_buf, &cap, (size_t)c.max_seqs, &changed)) != SAGC_OK) return rc; }
    if (prm->forced_lengths && (rc = grow(m, &m->forced_len_d, &m->forced_cap, (size_t)nseq, &changed)) != SAGC_OK) return rc;
    if (prm->n_dump > 0 && (rc = grow(m, &m->dump_list_d, &m->dump_cap, (size_t)prm->n_dump * 2, &changed)) != SAGC_OK) return rc;
    if (!structure_only) {
        size_t cap = (size_t)m->row_cap;
        if ((size_t)total_rows > cap) {
            size_t c1 = 0, c2 = 0, c3 = 0, c4 = 0;
            m->row_sid = m->row_pos = m->row_ctx = m->row_tok = nullptr;
            if ((rc = grow(m, &m->row_sid, &c1, (size_t)total_rows, &changed)) != SAGC_OK) return rc;
            if ((rc = grow(m, &m->row_pos, &c2, (size_t)total_rows, &changed)) != SAGC_OK) return rc;
            if ((rc = grow(m, &m->row_ctx, &c3, (size_t)total_rows, &changed)) != SAGC_OK) return rc;
            if ((rc = grow(m, &m->row_tok, &c4, (size_t)total_rows, &changed)) != SAGC_OK) return rc;
            m->row_cap = (int)c1;
        }
    }
    CU(cudaMemcpyAsync(m->prompt_len_d, plen.data(), n_prompts * sizeof(int), cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(m->offs_d, prompt_offsets, (n_prompts + 1) * sizeof(int), cudaMemcpyHostToDevice, st));
    if (prm->forced_lengths)
        CU(cudaMemcpyAsync(m->forced_len_d, prm->forced_lengths, nseq * sizeof(int), cudaMemcpyHostToDevice, st));
    if (prm->n_dump > 0)
        CU(cudaMemcpyAsync(m->dump_list_d, prm->dump_sid_t, (size_t)prm->n_dump * 2 * sizeof(int), cudaMemcpyHostToDevice, st));
    uint32_t sp[4];
    sp[0] = (uint32_t)prm->mode;
    float temp = prm->mode == SAGC_MODE_GUMBEL ? prm->temperature : 1.f;
    memcpy(&sp[1], &temp, 4);
    sp[2] = (uint32_t)(prm->seed & 0xffffffffull); sp[3] = (uint32_t)(prm->seed >> 32);
    CU(cudaMemcpyAsync(m->sample_params_d, sp, sizeof(sp), cudaMemcpyHostToDevice, st));

    RolloutDev rd = {};
    rd.prompt_len = m->prompt_len_d;
    rd.forced_len = prm->forced_lengths ? m->forced_len_d : nullptr;
    rd.forced_tok = prm->forced_tokens;
    rd.out_tokens = m->tok_buf; rd.out_lengths = m->len_buf;
    rd.n_prompts = n_prompts; rd.G = G; rd.nseq = nseq; rd.max_new = max_new; rd.stop_token = prm->stop_token;
    rd.log = (prm->flags & SAGC_FLAG_LOG) ? 1 : 0;

    // graphs bake every kernel argument: they are valid for one signature only
    char sig[256];
    snprintf(sig, sizeof(sig), "%d/%d/%d/%d/%d/%p/%p/%p/%d/%p/%d", n_prompts, G, max_new, prm->stop_token, rd.log,
             (const void*)rd.forced_len, (const void*)rd.forced_tok, (const void*)m->tok_buf, prm->n_dump,
             (const void*)prm->dump_logits, (int)m->use_pdl);
    if (changed || m->signature != sig) { clear_graphs(m); m->signature = sig; }
    m->last_nseq = nseq;

    // ---- host-side schedule -------------------------------------------------------------
    // With forced lengths the live count of every step is known in advance.
    std::vector<int> eff(nseq, max_new);
    if (prm->forced_lengths)
        for (int i = 0; i < nseq; ++i) { int f = prm->forced_lengths[i]; eff[i] = (f >= 1 && f < max_new) ? f : max_new; }
    int t_last = 0;
    for (int i = 0; i < nseq; ++i) if (eff[i] > t_last) t_last = eff[i];
    std::vector<int> live_at(t_last + 2, 0), glive_at;     // live_at[t] = #{eff >= t}
    std::vector<double> gplen_at;                          // sum of the prompt lengths of the groups still live at step t
    {
        std::vector<int> cnt(t_last + 2, 0);
        for (int i = 0; i < nseq; ++i) cnt[eff[i]]++;
        int run = 0;
        for (int t = t_last; t >= 1; --t) { run += cnt[t]; live_at[t] = run; }
        glive_at.assign(t_last + 2, 0);
        gplen_at.assign(t_last + 2, 0.0);
        std::vector<int> gcnt(t_last + 2, 0);
        std::vector<double> gpl(t_last + 2, 0.0);
        for (int p = 0; p < n_prompts; ++p) {
            int mx = 0;
            for (int g = 0; g < G; ++g) mx = eff[p * G + g] > mx ? eff[p * G + g] : mx;
            gcnt[mx]++; gpl[mx] += plen[p];
        }
        run = 0;
        double prun = 0.0;
        for (int t = t_last; t >= 1; --t) { run += gcnt[t]; glive_at[t] = run; prun += gpl[t]; gplen_at[t] = prun; }
    }
    const bool known = prm->forced_lengths != nullptr && prm->stop_token < 0;

    const bool want_t = timing != nullptr;
    if (want_t) memset(timing, 0, sizeof(*timing));
    cudaEvent_t ev[8];
    int n_ev = 0;
    auto mark = [&]() -> cudaEvent_t { cudaEvent_t e; cudaEventCreate(&e); cudaEventRecord(e, st); ev[n_ev++] = e; return e; };
    long long launches = 0;
    int r;

    // ---- a1: pool reset + prefix pages ----------------------------------------------------
    launches += launch_pool_reset(m->ps, rd, st);
    launches += launch_prefill_alloc(m->ps, rd, st);
    cudaEvent_t e_start = nullptr, e_pf = nullptr;
    if (want_t) e_start = mark();

    if (!structure_only) {
        // a pool too small for the prefixes leaves the page tables unmapped: stop before any kernel walks them
        int perr = 0;
        CU(cudaMemcpyAsync(&perr, m->ps.err, sizeof(int), cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
        if (perr) {
            for (int i = 0; i < n_ev; ++i) cudaEventDestroy(ev[i]);
            return set_err(SAGC_EPAGES, "KV page pool exhausted by the prompt prefixes (n_pages = %d)", c.n_pages);
        }
        // ---- a2: prefill, once per prompt, in row chunks ----------------------------------
        const int* ptok = prompt_tokens;      // device pointer supplied by the caller
        launches += launch_prefill_rows(ptok, m->offs_d, n_prompts, G, total_rows, m->row_sid, m->row_pos, m->row_ctx,
                                        m->row_tok, st);
        const int kind_pf = pick_kind(m, prm->path, PREFILL_ROWS);
        std::vector<int> idx;
        for (int r0 = 0; r0 < total_rows; r0 += PREFILL_ROWS) {
            const int rows = (total_rows - r0) < PREFILL_ROWS ? (total_rows - r0) : PREFILL_ROWS;
            RowSet rs = {m->row_sid + r0, m->row_pos + r0, m->row_ctx + r0, m->row_tok + r0, nullptr, rows};
            r = enqueue_layers(m, rs, 1, kind_pf, st);
            if (r < 0) return set_err(SAGC_ECUDA, "prefill launch failed: %s", cudaGetErrorString(cudaGetLastError()));
            launches += r;
            // last row of every prompt that ends inside this chunk -> xlast[p]
            idx.clear();
            int p_first = -1;
            for (int p = 0; p < n_prompts; ++p) {
                const int last = prompt_offsets[p + 1] - 1 - prompt_offsets[0];
                if (last >= r0 && last < r0 + rows) { if (p_first < 0) p_first = p; idx.push_back(last - r0); }
            }
            if (!idx.empty()) {
                CU(cudaMemcpyAsync(m->last_idx + p_first, idx.data(), idx.size() * sizeof(int), cudaMemcpyHostToDevice, st));
                CU(cudaStreamSynchronize(st));       // idx is reused by the next chunk
                launches += launch_gather_rows(m->x, m->last_idx + p_first, (int)idx.size(), c.d_model,
                                               m->xlast + (size_t)p_first * c.d_model, st);
            }
        }
        launches += launch_copy_partial_block(m->ps, rd, m->kv_pool, m->layer_stride, c.n_layers > 0 ? c.n_layers : 0,
                                              (int)m->page_elems, st);
        // ---- a3: first token of each completion from its prompt's last-row logits -----------
        r = enqueue_lm_head(m, m->xlast, nullptr, n_prompts, pick_kind(m, prm->path, n_prompts), st);
        if (r < 0) return set_err(SAGC_ECUDA, "lm head launch failed");
        launches += r;
        SampleArgs sa = {};
        sa.logits = m->logits; sa.V = c.vocab; sa.row_sid = m->ps.live; sa.step_dev = m->ps.step;
        sa.m_dev = m->ps.n_live; sa.m_max = nseq; sa.params = m->sample_params_d; sa.row_div = G; sa.part_score = m->part_score; sa.part_tok = m->sampled;
        launches += launch_sample(sa, st);
        if (prm->n_dump > 0)
            launches += launch_dump_logits(m->dump_list_d, prm->n_dump, m->ps.step, m->ps.live, m->ps.n_live, G,
                                           m->logits, c.vocab, prm->dump_logits, st);
    }
    launches += launch_advance(m->ps, rd, m->part_score, m->sampled, structure_only ? 1 : 0, st);     // end of step 1
    if (want_t) e_pf = mark();

    // ---- decode loop: steps t = 2 .. ---------------------------------------------------
    const double Wb = 2.0 * ((double)c.n_layers * ((double)c.d_model * c.n_q_heads * c.head_dim * 2 +
                                                   2.0 * c.d_model * c.n_kv_heads * c.head_dim + 3.0 * c.d_model * c.d_ff) +
                             (double)c.vocab * c.d_model);
    const double KVB = 2.0 * c.n_layers * c.n_kv_heads * c.head_dim * 2.0;
    int cur_phase = -1;
    cudaEvent_t ph_start[3] = {nullptr, nullptr, nullptr}, ph_end[3] = {nullptr, nullptr, nullptr};
    int live_bound = nseq;
    bool prev_mega = false;
    int t = 2;
    while (true) {
        int live;
        if (known) {
            if (t > t_last) break;
            live = live_at[t];
            if (!structure_only && (t & 255) == 0) {      // a pool exhausted mid-rollout ends it early (k_advance publishes 0 live rows)
                int herr2 = 0;
                CU(cudaMemcpyAsync(&herr2, m->ps.err, sizeof(int), cudaMemcpyDeviceToHost, st));
                CU(cudaStreamSynchronize(st));
                if (herr2) break;
            }
        } else {
            if (t > max_new) break;
            if ((t - 2) % 16 == 0) {          // poll the device's live count
                int h[2];
                CU(cudaMemcpyAsync(h, m->ps.n_live, sizeof(int), cudaMemcpyDeviceToHost, st));
                CU(cudaMemcpyAsync(h + 1, m->ps.err, sizeof(int), cudaMemcpyDeviceToHost, st));
                CU(cudaStreamSynchronize(st));
                live_bound = h[0];
                if (h[1] || live_bound == 0) break;
            }
            live = live_bound;
        }
        if (live == 0) break;
        const int ph = phase_of(live, nseq);
        if (want_t && ph != cur_phase) {
            cudaEvent_t e = mark();
            if (cur_phase >= 0) ph_end[cur_phase] = e;
            if (!ph_start[ph]) ph_start[ph] = e;
            cur_phase = ph;
        }
        if (want_t) {
            timing->phase_steps[ph] += 1;
            timing->phase_tokens[ph] += live;
            const double prefix = known ? gplen_at[t] : (double)total_rows;      // stop-token mode: every group counted until the end
            timing->phase_bytes[ph] += Wb + KVB * (prefix + (double)live * (t - 1)) + KVB * live;
        }
        if (structure_only) {
            launches += launch_advance(m->ps, rd, m->part_score, m->sampled, 1, st);
        } else {
            const int mb = round_bucket(live);
            const int kind = pick_kind(m, prm->path, mb);
            const bool mega = step_kernel_applies(m, kind, mb);
            const int ns = mega ? 0 : pick_splits(m, mb, pmax + t - 1, live);      // the step kernel picks its K-splits on the device
            if (mega && !prev_mega)       // both counter sets must be clear when the step kernel takes over
                CU(cudaMemsetAsync(m->step_sync, 0, (size_t)2 * (m->gbar_n + m->tcnt_n) * sizeof(unsigned), st));
            prev_mega = mega;
            if (use_graph) {
                GraphKey key = {mb, ns, kind, prm->n_dump};
                auto it = m->graphs.find(key);
                if (it == m->graphs.end()) {
                    cudaGraph_t g;
                    CU(cudaStreamBeginCapture(st, cudaStreamCaptureModeRelaxed));
                    int nk = enqueue_decode_step(m, rd, mb, ns, kind, prm->n_dump, prm->dump_logits, st);
                    cudaError_t ce = cudaStreamEndCapture(st, &g);
                    if (nk < 0 || ce != cudaSuccess) return set_err(SAGC_ECUDA, "graph capture failed: %s", cudaGetErrorString(ce));
                    GraphVal gv;
                    gv.n_kernels = nk;
                    CU(cudaGraphInstantiate(&gv.exec, g, 0));
                    cudaGraphDestroy(g);
                    it = m->graphs.emplace(key, gv).first;
                }
                CU(cudaGraphLaunch(it->second.exec, st));
                launches += it->second.n_kernels;
            } else {
                r = enqueue_decode_step(m, rd, mb, ns, kind, prm->n_dump, prm->dump_logits, st, time_kernels ? &kev : nullptr);
                if (r < 0) return set_err(SAGC_ECUDA, "decode launch failed: %s", cudaGetErrorString(cudaGetLastError()));
                launches += r;
            }
        }
        ++t;
    }
    cudaEvent_t e_end = nullptr;
    if (want_t) { e_end = mark(); if (cur_phase >= 0) ph_end[cur_phase] = e_end; }

    // ---- a14: length statistics, outputs ---------------------------------------------------
    // group offsets = p*G: reuse offs_d (prompt offsets are no longer needed on the device)
    {
        std::vector<int> goffs(n_prompts + 1);
        for (int p = 0; p <= n_prompts; ++p) goffs[p] = p * G;
        CU(cudaMemcpyAsync(m->offs_d, goffs.data(), (n_prompts + 1) * sizeof(int), cudaMemcpyHostToDevice, st));
        CU(cudaStreamSynchronize(st));
    }
    if (out_ratio || out_len_stats)
        launches += launch_length_stats(m->len_buf, m->offs_d, n_prompts, out_len_stats, out_ratio, st);
    CU(cudaMemcpyAsync(out_tokens, m->tok_buf, (size_t)nseq * max_new * sizeof(int), cudaMemcpyDeviceToDevice, st));
    CU(cudaMemcpyAsync(out_lengths, m->len_buf, (size_t)nseq * sizeof(int), cudaMemcpyDeviceToDevice, st));
    int herr = 0;
    CU(cudaMemcpyAsync(&herr, m->ps.err, sizeof(int), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    CU(cudaGetLastError());
    if (want_t) {
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e_start, e_pf); timing->prefill_ms = ms;
        cudaEventElapsedTime(&ms, e_pf, e_end); timing->decode_ms = ms;
        for (int p = 0; p < 3; ++p)
            if (ph_start[p] && ph_end[p]) { cudaEventElapsedTime(&ms, ph_start[p], ph_end[p]); timing->phase_ms[p] = ms; }
        timing->prefill_tokens = structure_only ? 0 : total_rows;
        timing->prefill_flops = structure_only ? 0.0 : (double)total_rows * Wb;   // 2 flop per bf16 weight per row (+attention, not counted)
        long long tot = 0;
        if (known) {
            for (int i = 0; i < nseq; ++i) tot += eff[i];
        } else {                                  // stop-token mode: the lengths are only known on the device
            std::vector<int> hl(nseq);
            CU(cudaMemcpy(hl.data(), m->len_buf, (size_t)nseq * sizeof(int), cudaMemcpyDeviceToHost));
            for (int i = 0; i < nseq; ++i) tot += hl[i];
        }
        timing->total_tokens = tot;
        timing->kernel_launches = launches;
        for (size_t i = 0; i + 3 < kev.size(); i += 4) {
            for (int k = 0; k < 3; ++k) { cudaEventElapsedTime(&ms, kev[i + k], kev[i + k + 1]); timing->kernel_ms[k] += ms; }
            timing->kernel_steps += 1;
        }
    }
    for (int i = 0; i < n_ev; ++i) cudaEventDestroy(ev[i]);
    for (cudaEvent_t e : kev) cudaEventDestroy(e);
    if (herr) return set_err(SAGC_EPAGES, "KV page pool exhausted (n_pages = %d)", c.n_pages);
    return SAGC_OK;
}

extern "C" int sagc_rollout_group_host(sagc_model* m, const int32_t* prompt_tokens, const int32_t* prompt_offsets,
                                       int32_t n_prompts, int32_t G, const sagc_rollout_params* prm,
                                       int32_t* out_tokens, int32_t* out_lengths, float* out_ratio,
                                       int32_t* out_len_stats, sagc_rollout_timing* timing, void* stream) {
    if (!m || !prompt_offsets || !prm || !out_tokens || !out_lengths) return set_err(SAGC_EINVAL, "null argument");
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    const int nseq = n_prompts * G;
    if (n_prompts < 1 || G < 1 || prm->max_new_tokens < 1) return set_err(SAGC_EINVAL, "bad sizes");
    const size_t ntok = (size_t)nseq * prm->max_new_tokens;
    const int total = prompt_offsets[n_prompts];
    int rc;
    // device staging buffers live in the handle (grown on demand): no cudaMalloc / cudaFree in the timed call
    if ((rc = grow(m, &m->h_prompt, &m->h_prompt_cap, (size_t)(total > 0 ? total : 1), nullptr)) != SAGC_OK) return rc;
    if ((rc = grow(m, &m->h_tok, &m->h_tok_cap, ntok, nullptr)) != SAGC_OK) return rc;
    if ((rc = grow(m, &m->h_len, &m->h_len_cap, (size_t)nseq, nullptr)) != SAGC_OK) return rc;
    if ((size_t)n_prompts > m->h_grp_cap || !m->h_stats) {
        size_t c1 = 0, c2 = 0;
        m->h_stats = nullptr; m->h_ratio = nullptr;
        if ((rc = grow(m, &m->h_stats, &c1, (size_t)n_prompts * 3, nullptr)) != SAGC_OK) return rc;
        if ((rc = grow(m, &m->h_ratio, &c2, (size_t)n_prompts, nullptr)) != SAGC_OK) return rc;
        m->h_grp_cap = (size_t)n_prompts;
    }
    if (prompt_tokens && total > 0)
        CU(cudaMemcpyAsync(m->h_prompt, prompt_tokens, (size_t)total * sizeof(int), cudaMemcpyHostToDevice, st));
    rc = sagc_rollout_group(m, prompt_tokens ? m->h_prompt : nullptr, prompt_offsets, n_prompts, G, prm, m->h_tok, m->h_len,
                            m->h_ratio, m->h_stats, timing, stream);
    if (rc != SAGC_OK) return rc;
    CU(cudaMemcpyAsync(out_tokens, m->h_tok, ntok * sizeof(int), cudaMemcpyDeviceToHost, st));
    CU(cudaMemcpyAsync(out_lengths, m->h_len, (size_t)nseq * sizeof(int), cudaMemcpyDeviceToHost, st));
    if (out_ratio) CU(cudaMemcpyAsync(out_ratio, m->h_ratio, (size_t)n_prompts * sizeof(float), cudaMemcpyDeviceToHost, st));
    if (out_len_stats) CU(cudaMemcpyAsync(out_len_stats, m->h_stats, (size_t)n_prompts * 3 * sizeof(int), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    return SAGC_OK;
}


// ---------------------------------------------------------------------------------------
// sagc_score_tokens: teacher-forced log-prob pass
// ---------------------------------------------------------------------------------------
extern "C" int sagc_score_tokens(sagc_model* m, const int32_t* prompt_tokens, const int32_t* prompt_offsets, int32_t n_prompts, int32_t G,
                                 const int32_t* tokens, const int32_t* lengths, int32_t max_new, float* out_logprobs, void* stream) {
    if (!m || !prompt_tokens || !prompt_offsets || !tokens || !lengths || !out_logprobs) return set_err(SAGC_EINVAL, "null argument");
    const sagc_model_config& c = m->cfg;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    const int nseq = n_prompts * G;
    if (n_prompts < 1 || G < 1 || nseq > c.max_seqs || max_new < 1) return set_err(SAGC_EINVAL, "bad sizes (n_prompts*G <= max_seqs)");
    if (c.n_layers < 1) return set_err(SAGC_EINVAL, "model has no layers");
    std::vector<int> seq_off(nseq + 1, 0), seq_len(nseq);
    long long pages = 0;
    for (int sid = 0; sid < nseq; ++sid) {
        const int P = prompt_offsets[sid / G + 1] - prompt_offsets[sid / G];
        const int ell = lengths[sid];
        if (P < 1 || ell < 1 || ell > max_new || P + ell > c.max_ctx) return set_err(SAGC_EINVAL, "sequence %d: bad prompt / completion length", sid);
        seq_len[sid] = P + ell - 1;                    // the last generated token is only a target
        seq_off[sid + 1] = seq_off[sid] + seq_len[sid];
        pages += (seq_len[sid] + c.page_tokens - 1) / c.page_tokens;
    }
    if (pages > c.n_pages) return set_err(SAGC_EPAGES, "scoring needs %lld KV pages, the pool has %d", pages, c.n_pages);
    const int total_rows = seq_off[nseq];
    int rc;
    bool changed = false;
    if ((rc = grow(m, &m->tok_buf, &m->tok_cap, (size_t)nseq * max_new, &changed)) != SAGC_OK) return rc;
    if (!m->len_buf) { size_t cap = 0; if ((rc = grow(m, &m->len_buf, &cap, (size_t)c.max_seqs, &changed)) != SAGC_OK) return rc; }
    if ((size_t)total_rows > (size_t)m->row_cap) {
        size_t c1 = 0, c2 = 0, c3 = 0, c4 = 0;
        m->row_sid = m->row_pos = m->row_ctx = m->row_tok = nullptr;
        if ((rc = grow(m, &m->row_sid, &c1, (size_t)total_rows, &changed)) != SAGC_OK) return rc;
        if ((rc = grow(m, &m->row_pos, &c2, (size_t)total_rows, &changed)) != SAGC_OK) return rc;
        if ((rc = grow(m, &m->row_ctx, &c3, (size_t)total_rows, &changed)) != SAGC_OK) return rc;
        if ((rc = grow(m, &m->row_tok, &c4, (size_t)total_rows, &changed)) != SAGC_OK) return rc;
        m->row_cap = (int)c1;
    }
    if ((rc = grow(m, &m->score_logits, &m->score_cap, (size_t)PREFILL_ROWS * c.vocab, &changed)) != SAGC_OK) return rc;
    if ((rc = grow(m, &m->seq_off_d, &m->seq_off_cap, (size_t)nseq + 1, &changed)) != SAGC_OK) return rc;
    if (changed) { clear_graphs(m); m->signature.clear(); }          // the rollout graphs bake tok_buf / row buffers
    CU(cudaMemcpyAsync(m->seq_off_d, seq_off.data(), (nseq + 1) * sizeof(int), cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(m->prompt_len_d, seq_len.data(), nseq * sizeof(int), cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(m->offs_d, prompt_offsets, (n_prompts + 1) * sizeof(int), cudaMemcpyHostToDevice, st));
    CU(cudaMemsetAsync(out_logprobs, 0, (size_t)nseq * max_new * sizeof(float), st));
    // every sequence is its own "prompt" of length P + l - 1 (G = 1): the paging kernels lay its KV out in fresh pages
    RolloutDev rd = {};
    rd.prompt_len = m->prompt_len_d; rd.out_tokens = m->tok_buf; rd.out_lengths = m->len_buf;
    rd.n_prompts = nseq; rd.G = 1; rd.nseq = nseq; rd.max_new = max_new; rd.stop_token = -1;
    launch_pool_reset(m->ps, rd, st);
    launch_prefill_alloc(m->ps, rd, st);
    launch_score_rows(prompt_tokens, m->offs_d, m->seq_off_d, tokens, nseq, G, max_new, total_rows, m->row_sid, m->row_pos, m->row_ctx,
                      m->row_tok, st);
    const int kind = pick_kind(m, SAGC_PATH_AUTO, PREFILL_ROWS);
    for (int r0 = 0; r0 < total_rows; r0 += PREFILL_ROWS) {
        const int rows = (total_rows - r0) < PREFILL_ROWS ? (total_rows - r0) : PREFILL_ROWS;
        RowSet rs = {m->row_sid + r0, m->row_pos + r0, m->row_ctx + r0, m->row_tok + r0, nullptr, rows};
        if (enqueue_layers(m, rs, 1, kind, st) < 0) return set_err(SAGC_ECUDA, "scoring: layer launch failed");
        if (enqueue_lm_head(m, m->x, nullptr, rows, kind, st, m->score_logits) < 0) return set_err(SAGC_ECUDA, "scoring: LM head launch failed");
        launch_token_logprob(m->score_logits, c.vocab, rows, m->row_sid + r0, m->row_pos + r0, m->offs_d, G, tokens, max_new, out_logprobs, st);
    }
    int herr = 0;
    CU(cudaMemcpyAsync(&herr, m->ps.err, sizeof(int), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    CU(cudaGetLastError());
    m->last_nseq = nseq;
    if (herr) return set_err(SAGC_EPAGES, "KV page pool exhausted (n_pages = %d)", c.n_pages);
    return SAGC_OK;
}

// ---------------------------------------------------------------------------------------
// group statistics
// ---------------------------------------------------------------------------------------
extern "C" int sagc_group_advantage(const float* rewards, const int32_t* group_offsets, int32_t n_groups, int32_t mode,
                                    int32_t ddof, float eps, float* out_adv, uint8_t* out_keep, void* stream) {
    if (n_groups < 0 || (n_groups > 0 && (!rewards || !group_offsets || !out_adv || !out_keep)))
        return set_err(SAGC_EINVAL, "null argument");
    if (mode != SAGC_ADV_GRPO && mode != SAGC_ADV_DAPO) return set_err(SAGC_EINVAL, "mode must be GRPO or DAPO");
    if (ddof != 0 && ddof != 1) return set_err(SAGC_EINVAL, "ddof must be 0 or 1");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return set_err(SAGC_ECUDA, "no CUDA device (there is no CPU fallback)");
    launch_group_advantage(rewards, group_offsets, n_groups, mode, ddof, eps, out_adv, out_keep,
                           reinterpret_cast<cudaStream_t>(stream));
    CU(cudaGetLastError());
    return SAGC_OK;
}

extern "C" int sagc_length_stats(const int32_t* lengths, const int32_t* group_offsets, int32_t n_groups,
                                 int32_t* out_stats, float* out_ratio, void* stream) {
    if (n_groups < 0 || (n_groups > 0 && (!lengths || !group_offsets))) return set_err(SAGC_EINVAL, "null argument");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return set_err(SAGC_ECUDA, "no CUDA device (there is no CPU fallback)");
    launch_length_stats(lengths, group_offsets, n_groups, out_stats, out_ratio, reinterpret_cast<cudaStream_t>(stream));
    CU(cudaGetLastError());
    return SAGC_OK;
}

// ---------------------------------------------------------------------------------------
// debug / parity exports
// ---------------------------------------------------------------------------------------
extern "C" int sagc_debug_page_table(sagc_model* m, int32_t* out, int32_t capacity, int32_t* nseq, int32_t* max_blocks) {
    if (!m || !out) return set_err(SAGC_EINVAL, "null argument");
    const int n = m->last_nseq, mb = m->max_blocks;
    if (nseq) *nseq = n;
    if (max_blocks) *max_blocks = mb;
    if ((long long)n * mb > capacity) return set_err(SAGC_EINVAL, "capacity %d < %lld", capacity, (long long)n * mb);
    CU(cudaDeviceSynchronize());
    CU(cudaMemcpy(out, m->ps.page_table, (size_t)n * mb * sizeof(int), cudaMemcpyDeviceToHost));
    return SAGC_OK;
}
extern "C" int sagc_debug_free_stack(sagc_model* m, int32_t* out, int32_t capacity, int32_t* n_free) {
    if (!m || !out || !n_free) return set_err(SAGC_EINVAL, "null argument");
    CU(cudaDeviceSynchronize());
    CU(cudaMemcpy(n_free, m->ps.n_free, sizeof(int), cudaMemcpyDeviceToHost));
    if (*n_free > capacity) return set_err(SAGC_EINVAL, "capacity too small");
    CU(cudaMemcpy(out, m->ps.free_stack, (size_t)(*n_free) * sizeof(int), cudaMemcpyDeviceToHost));
    return SAGC_OK;
}
static int copy_log(const int* dev_log, const int* dev_n, int width, int cap_entries, int32_t* out, int32_t capacity, int32_t* n) {
    if (!out || !n) return set_err(SAGC_EINVAL, "null argument");
    CU(cudaDeviceSynchronize());
    CU(cudaMemcpy(n, dev_n, sizeof(int), cudaMemcpyDeviceToHost));
    int k = *n < cap_entries ? *n : cap_entries;
    if (k > capacity) return set_err(SAGC_EINVAL, "capacity %d < %d entries", capacity, k);
    CU(cudaMemcpy(out, dev_log, (size_t)k * width * sizeof(int), cudaMemcpyDeviceToHost));
    return SAGC_OK;
}
extern "C" int sagc_debug_alloc_log(sagc_model* m, int32_t* out, int32_t capacity, int32_t* n) {
    if (!m) return set_err(SAGC_EINVAL, "null argument");
    return copy_log(m->ps.alloc_log, m->ps.n_alloc, 3, m->ps.log_cap_alloc, out, capacity, n);
}
extern "C" int sagc_debug_retire_log(sagc_model* m, int32_t* out, int32_t capacity, int32_t* n) {
    if (!m) return set_err(SAGC_EINVAL, "null argument");
    return copy_log(m->ps.retire_log, m->ps.n_retire, 2, m->ps.log_cap_retire, out, capacity, n);
}
extern "C" int sagc_debug_peak_pages(sagc_model* m, int32_t* peak) {
    if (!m || !peak) return set_err(SAGC_EINVAL, "null argument");
    CU(cudaDeviceSynchronize());
    CU(cudaMemcpy(peak, m->ps.peak_used, sizeof(int), cudaMemcpyDeviceToHost));
    return SAGC_OK;
}
extern "C" int sagc_debug_step_trace(sagc_model* m, int64_t record_step, uint64_t* out, int32_t capacity, int32_t* n) {
    if (!m || !n) return set_err(SAGC_EINVAL, "null argument");
    *n = 0;
    if (!m->step_trace) return SAGC_OK;                      // tracing is off (SAGC_STEP_TRACE unset at model create)
    CU(cudaDeviceSynchronize());
    unsigned long long hdr[2];
    CU(cudaMemcpy(hdr, m->step_trace, sizeof(hdr), cudaMemcpyDeviceToHost));
    int k = (int)(hdr[1] < 16000ull ? hdr[1] : 16000ull);
    if (out) {
        if (k > capacity) k = capacity;
        CU(cudaMemcpy(out, m->step_trace + 2, (size_t)k * 2 * sizeof(unsigned long long), cudaMemcpyDeviceToHost));
        *n = k;
    }
    hdr[0] = (unsigned long long)record_step; hdr[1] = 0;    // arm the next recording
    CU(cudaMemcpy(m->step_trace, hdr, sizeof(hdr), cudaMemcpyHostToDevice));
    return SAGC_OK;
}
extern "C" int sagc_debug_philox(uint64_t seed, int32_t sid, int32_t t, int32_t v0, int32_t n, uint32_t* out, void* stream) {
    if (n < 0 || (n > 0 && !out)) return set_err(SAGC_EINVAL, "null argument");
    launch_philox_debug(seed, sid, t, v0, n, out, reinterpret_cast<cudaStream_t>(stream));
    CU(cudaGetLastError());
    return SAGC_OK;
}
extern "C" int sagc_debug_linear(const void* W, const float* x, float* y, int32_t M, int32_t N, int32_t K, int32_t path,
                                 void* stream) {
    if (!W || !x || !y || M < 1 || N % 16 || K % 32) return set_err(SAGC_EINVAL, "need N %% 16 == 0 and K %% 32 == 0");
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    if (path == SAGC_PATH_GEMM && N % 128 == 0 && K % 64 == 0) {
        // tcgen05 path: pre-split the activations, build the two tensor maps, one launch
        const int nbi = tc_nb_index(M), NB = 32 << nbi;
        static bf16_t* xs = nullptr;            // debug entry: grow-only buffers, kept for the process lifetime
        static size_t xs_cap = 0;
        const size_t rows = 2 * (size_t)(((M + NB / 2 - 1) / (NB / 2)) * (NB / 2));
        if (rows * K > xs_cap) {
            CU(cudaDeviceSynchronize());
            if (xs) cudaFree(xs);
            xs_cap = rows * K;
            CU(cudaMalloc(&xs, xs_cap * sizeof(bf16_t)));
            CU(cudaMemset(xs, 0, xs_cap * sizeof(bf16_t)));
        }
        launch_split_rows(x, K, nullptr, M, xs, st);
        TcMap ma, mb;
        if (tc_make_map(&ma, W, N, K, 128) != 0 || tc_make_map(&mb, xs, (long long)rows, K, NB) != 0) {
            return set_err(SAGC_ECUDA, "cuTensorMapEncodeTiled failed");
        }
        TcLinearArgs t = {};
        t.a[0] = &ma; t.seg_rows[0] = N; t.b = &mb; t.K = K; t.N = N; t.m_dev = nullptr; t.m_max = M; t.epi = EPI_STORE;
        static float* scr = nullptr;            // debug entry: allocated once per process
        if (!scr) CU(cudaMalloc(&scr, TC_SCRATCH_FLOATS * sizeof(float)));
        t.Y = y; t.ldy = N; t.pdl = false; t.scratch = scr;
        int r = launch_linear_tc(t, st);
        if (r < 0) return set_err(SAGC_ECUDA, "tcgen05 linear: %s", cudaGetErrorString(cudaGetLastError()));
        CU(cudaGetLastError());
        return SAGC_OK;
    }
    // rows beyond 64 are processed by the kernels' own m-chunk grid dimension
    LinearArgs a = {};
    a.W[0] = reinterpret_cast<const bf16_t*>(W); a.rows[0] = N; a.X = x; a.Y = y; a.ldy = N; a.K = K; a.N = N;
    a.m_dev = nullptr; a.m_max = M; a.epi = EPI_STORE; a.kind = (path == SAGC_PATH_GEMV) ? LIN_GEMV : LIN_MMA; a.pdl = false;
    if (launch_linear(a, st) < 0) return set_err(SAGC_ECUDA, "launch failed: %s", cudaGetErrorString(cudaGetLastError()));
    CU(cudaGetLastError());
    return SAGC_OK;
}
extern "C" int sagc_debug_lm_sample(const void* W, const float* x, int32_t M, int32_t V, int32_t K, int32_t mode, float temperature,
                                    uint64_t seed, int32_t t, const int32_t* sids, int32_t* out_tokens, float* out_logits,
                                    void* stream) {
    if (!W || !x || !sids || !out_tokens || M < 1 || M > 64 || V % 128 || K % 64 || temperature <= 0.f)
        return set_err(SAGC_EINVAL, "need 1 <= M <= 64, V %% 128 == 0, K %% 64 == 0, temperature > 0");
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    const int nbi = tc_nb_index(M), NB = 32 << nbi;
    static bf16_t* xs = nullptr;                // debug entry: grow-only buffers, kept for the process lifetime
    static size_t xs_cap = 0;
    static float* ps = nullptr; static int* pt = nullptr; static uint32_t* prm = nullptr; static int* step = nullptr;
    const size_t rows = (size_t)NB;
    if (rows * K > xs_cap) {
        CU(cudaDeviceSynchronize());
        if (xs) cudaFree(xs);
        xs_cap = rows * K;
        CU(cudaMalloc(&xs, xs_cap * sizeof(bf16_t)));
        CU(cudaMemset(xs, 0, xs_cap * sizeof(bf16_t)));
    }
    if (!ps) {
        CU(cudaMalloc(&ps, (size_t)LM_MAX_PARTS * 64 * sizeof(float)));
        CU(cudaMalloc(&pt, (size_t)LM_MAX_PARTS * 64 * sizeof(int)));
        CU(cudaMalloc(&prm, 4 * sizeof(uint32_t)));
        CU(cudaMalloc(&step, sizeof(int)));
    }
    uint32_t hp[4];
    hp[0] = (uint32_t)mode; memcpy(&hp[1], &temperature, 4); hp[2] = (uint32_t)(seed & 0xffffffffu); hp[3] = (uint32_t)(seed >> 32);
    static uint32_t last_hp[4] = {~0u, 0u, 0u, 0u};
    static int last_t = -1;
    if (memcmp(hp, last_hp, sizeof(hp)) != 0 || t != last_t) {      // repeated calls (timing loops) skip the upload
        CU(cudaMemcpyAsync(prm, hp, sizeof(hp), cudaMemcpyHostToDevice, st));
        CU(cudaMemcpyAsync(step, &t, sizeof(int), cudaMemcpyHostToDevice, st));
        CU(cudaStreamSynchronize(st));          // hp / t live on this frame
        memcpy(last_hp, hp, sizeof(hp)); last_t = t;
    }
    launch_split_rows(x, K, nullptr, M, xs, st);
    TcMap ma, mb;
    if (tc_make_map(&ma, W, V, K, 128) != 0 || tc_make_map(&mb, xs, (long long)rows, K, NB) != 0)
        return set_err(SAGC_ECUDA, "cuTensorMapEncodeTiled failed");
    LmSampleArgs f = {};
    f.a = &ma; f.b = &mb; f.K = K; f.V = V; f.m_dev = nullptr; f.m_max = M; f.ssq_in = nullptr; f.k_norm = K;
    f.row_sid = sids; f.step_dev = step; f.params = prm; f.part_score = ps; f.part_tok = pt; f.part_ld = 64;
    f.Y = out_logits; f.ldy = V; f.pdl = false;
    if (launch_lmhead_sample(f, st) < 0) return set_err(SAGC_ECUDA, "fused LM head: %s", cudaGetErrorString(cudaGetLastError()));
    launch_pick_candidates(ps, pt, lm_sample_grid(V), 64, M, out_tokens, st);
    CU(cudaGetLastError());
    return SAGC_OK;
}
extern "C" int sagc_debug_attention(const float* q, const void* kv, const int32_t* page_table, const int32_t* ctx, int32_t M,
                                    int32_t Hq, int32_t Hkv, int32_t hd, int32_t page_tokens, int32_t max_blocks, int32_t n_splits,
                                    int32_t variant, float* out, void* stream) {
    if (!q || !kv || !page_table || !ctx || !out || M < 1) return set_err(SAGC_EINVAL, "null argument");
    if (Hq % Hkv || Hq / Hkv > 8) return set_err(SAGC_EINVAL, "bad head counts");
    if (n_splits < 1 || n_splits > 64) return set_err(SAGC_EINVAL, "n_splits must be in 1..64");
    if (variant < 0 || variant > 2) return set_err(SAGC_EINVAL, "variant must be 0 (standalone kernel), 1 (decode-step units) or 2 (tcgen05 kernel)");
    if (variant == 2 && !attention_tc_supports(hd, page_tokens, Hq / Hkv)) return set_err(SAGC_EINVAL, "the tcgen05 kernel needs head_dim 64 / 128 and pages of 8 .. 128 tokens");
    if (variant == 1 && hd != 64 && hd != 128) return set_err(SAGC_EINVAL, "the decode-step units need head_dim 64 or 128");
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    int *sid = nullptr, *cnt = nullptr;
    float *po = nullptr, *pml = nullptr;
    CU(cudaMalloc(&sid, M * sizeof(int)));
    CU(cudaMalloc(&cnt, (size_t)M * Hkv * sizeof(int)));
    CU(cudaMalloc(&po, (size_t)M * Hq * n_splits * hd * sizeof(float)));
    CU(cudaMalloc(&pml, (size_t)M * Hq * n_splits * 2 * sizeof(float)));
    std::vector<int> ident(M);
    for (int i = 0; i < M; ++i) ident[i] = i;
    CU(cudaMemcpyAsync(sid, ident.data(), M * sizeof(int), cudaMemcpyHostToDevice, st));
    CU(cudaMemsetAsync(cnt, 0, (size_t)M * Hkv * sizeof(int), st));
    AttnArgs a = {};
    a.q = q; a.ldq = Hq * hd; a.kv_layer = reinterpret_cast<const bf16_t*>(kv); a.page_table = page_table;
    a.max_blocks = max_blocks; a.row_sid = sid; a.row_ctx = ctx; a.m_dev = nullptr; a.m_max = M; a.Hq = Hq; a.Hkv = Hkv;
    a.hd = hd; a.page = page_tokens; a.n_splits = n_splits; a.part_o = po; a.part_ml = pml; a.counters = cnt; a.out = out;
    int n_sm = 148;
    { int dev = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev); }
    int r;
    if (variant == 2) {
        // the pool's extent is not an argument: take it from the largest page id in the caller's table
        std::vector<int> pt_h((size_t)M * max_blocks);
        CU(cudaMemcpyAsync(pt_h.data(), page_table, pt_h.size() * sizeof(int), cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
        long long n_pages = 1;
        for (int v : pt_h) if ((long long)v + 1 > n_pages) n_pages = (long long)v + 1;
        TcMap kvmap;
        if (attention_tc_make_map(&kvmap, kv, n_pages, Hkv, page_tokens, hd) != 0) {
            cudaFree(sid); cudaFree(cnt); cudaFree(po); cudaFree(pml);
            return set_err(SAGC_ECUDA, "cuTensorMapEncodeTiled failed");
        }
        unsigned long long* dbg = nullptr;
        if (env_int("SAGC_ATT_DBG", 0)) {        // timeline of CTA (0,0,0): needs a library built with SAGC_ATT_TIMELINE=1
            CU(cudaMalloc(&dbg, 4 * 64 * 8 * sizeof(unsigned long long)));
            CU(cudaMemsetAsync(dbg, 0, 4 * 64 * 8 * sizeof(unsigned long long), st));
            a.dbg = dbg;
        }
        r = launch_attention_tc(a, &kvmap, env_int("SAGC_ATT_TC_STAGES", 0), st);
        if (dbg) {
            std::vector<unsigned long long> h(4 * 64 * 8);
            cudaStreamSynchronize(st);
            cudaMemcpy(h.data(), dbg, h.size() * 8, cudaMemcpyDeviceToHost);
            cudaFree(dbg);
            unsigned long long t0 = ~0ull;
            for (auto v : h) if (v && v < t0) t0 = v;
            for (int role = 0; role < 4; ++role)
                for (int tile = 0; tile < 64; ++tile) {
                    bool any = false;
                    for (int e = 0; e < 8; ++e) any |= h[(role * 64 + tile) * 8 + e] != 0;
                    if (!any) continue;
                    fprintf(stderr, "ATC role %d tile %2d:", role, tile);
                    for (int e = 0; e < 8; ++e) { auto v = h[(role * 64 + tile) * 8 + e]; fprintf(stderr, " %7lld", v ? (long long)(v - t0) : -1LL); }
                    fprintf(stderr, "\n");
                }
        }
    } else {
        r = variant == 1 ? launch_attention_units(a, n_sm, st) : launch_attention(a, st);
    }
    cudaError_t e = cudaStreamSynchronize(st);
    cudaFree(sid); cudaFree(cnt); cudaFree(po); cudaFree(pml);
    if (r < 0) return set_err(SAGC_EINVAL, "unsupported head_dim %d", hd);
    if (e != cudaSuccess) return set_err(SAGC_ECUDA, "attention: %s", cudaGetErrorString(e));
    return SAGC_OK;
}
