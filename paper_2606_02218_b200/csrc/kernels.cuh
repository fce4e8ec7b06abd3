// kernels.cuh -- launcher prototypes of the sm_100a kernels (internal; the public boundary is
// include/sagc.h).  Every launcher enqueues on `st` and returns the number of kernels it launched.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

namespace sagc {

typedef uint16_t bf16_t;   // raw bf16 bit pattern

extern bool g_pdl_all;     // launch the small kernels (embed, rope, attention, sampler, advance) with the PDL attribute too
extern int g_num_sms;      // multiprocessor count of the current device (set by sagc_model_create; 148 on B200)

enum { EPI_STORE = 0, EPI_RESID = 1, EPI_SWIGLU = 2, EPI_QKV = 3 };   // EPI_QKV: tcgen05 path only (fused RoPE + KV append)
enum { LIN_MMA = 0, LIN_GEMV = 1, LIN_TC = 2 };

// Y[M][N] = epi( rms?(X)[M][K] . W[N][K]^T ).  Steps a6, a8-a11 of DESIGN.md.
struct LinearArgs {
    const bf16_t* W[3];     // up to three row segments (q,k,v) -- or {gate, up} for EPI_SWIGLU
    int rows[3];            // rows per segment (EPI_SWIGLU: rows[0] == rows[1] == N)
    const float* X;         // [M][K] fp32 activations
    const bf16_t* norm_w;   // if non-null: fused RMSNorm, X <- X * norm_w * rsqrt(mean(X^2)+eps)
    float eps;
    float* Y;               // [M][ldy]
    const float* R;         // EPI_RESID: Y = R + acc (R may alias Y)
    int ldy;
    int K, N;
    const int* m_dev;       // device pointer to the live row count, or null
    int m_max;              // grid is sized for this many rows (>= *m_dev)
    int epi;
    int kind;               // LIN_MMA | LIN_GEMV
    bool pdl;               // launch with programmatic stream serialization
};
int launch_linear(const LinearArgs& a, cudaStream_t st);

// x[row][d] = embed[tok[row]][d]  (fp32 residual stream).  Step a5.
int launch_embed(const bf16_t* embed, const int* tok, const int* m_dev, int m_max, int d, float* x,
                 cudaStream_t st);

// RoPE on q and k heads, K/V rounded to bf16 (RNE) and appended to the sequence's page.  Step a6.
struct RopeArgs {
    float* qkv;             // [M][(Hq+2Hkv)*hd] fp32, q part rotated in place
    const int* row_sid;     // [M] page-table row of each activation row
    const int* row_pos;     // [M] position of each row
    const int* m_dev; int m_max;
    const float* rope_cs;   // [max_ctx][hd/2][2] (cos, sin) fp32, angles evaluated in fp64
    bf16_t* kv_layer;       // this layer's pool: [n_pages][2][Hkv][page][hd]
    const int* page_table;  // [max_seqs][max_blocks]
    int max_blocks, page, Hq, Hkv, hd;
};
int launch_rope_append(const RopeArgs& a, cudaStream_t st);

// Paged GQA attention over ragged contexts with split-K + in-kernel LSE merge.  Step a7.
struct AttnArgs {
    const float* q;         // [M][ldq] (first Hq*hd columns are the rotated queries)
    int ldq;
    const bf16_t* kv_layer; // [n_pages][2][Hkv][page][hd]
    const int* page_table; int max_blocks;
    const int* row_sid;     // [M]
    const int* row_ctx;     // [M] number of cached positions attended (incl. the current one)
    const int* m_dev; int m_max;
    int Hq, Hkv, hd, page;
    int n_splits;           // grid.z; every split covers ceil(ctx/n_splits) rounded up to a page
    float* part_o;          // [M][Hq][n_splits][hd] scratch
    float* part_ml;         // [M][Hq][n_splits][2]  (max, sum)
    int* counters;          // [M*Hkv] arrival counters (zero on entry, reset on exit)
    float* out;             // [M][Hq*hd] fp32 (used when out_split is null)
    bf16_t* out_split;      // pre-split rows [2m] = hi, [2m+1] = lo, row stride ld_split (tcgen05 path)
    int ld_split;
    // decode only (fuse_rope): q is the RAW qkv row; RoPE of q / k and the bf16 K,V append of the newest
    // position happen inside this kernel (no separate RoPE kernel).  head_dim >= 64.
    int fuse_rope; const float* rope_cs; const int* row_pos; bf16_t* kv_layer_w;
    // decode-step kernel: the q | k | v row is a 64-bit fixed-point sum (value * 2^32, see decode_step.cu) that still
    // lacks the 1/rms factor of its row; when q_fx is set it replaces q (same [row][ldq] indexing)
    const long long* q_fx; const float* q_rstd;
    int prefetch;           // 1 in decode: cached positions older than the newest one predate the upstream kernel
    int cluster_merge;      // set by the launcher: the n_splits CTAs of a (row, kv head) form a cluster and merge through DSMEM
    unsigned long long* dbg; // attention_tc.cu built with -DSAGC_ATT_TIMELINE: clock64 stamps of CTA (0,0,0), [role 4][tile 64][event 8]; else unused
};
int launch_attention(const AttnArgs& a, cudaStream_t st);

// tcgen05 decode attention (attention_tc.cu): head_dim 64 / 128, pages of 8 .. 128 tokens; split merge through the L2 scratch
struct TcMap;
bool attention_tc_supports(int hd, int page, int r);
int attention_tc_make_map(TcMap* out, const void* kv_layer, long long n_pages, int Hkv, int page, int hd);
int launch_attention_tc(const AttnArgs& a, const TcMap* kvmap, int stages, cudaStream_t st);

// Sampler over fp32 logits.  Step a3 / a12.
static constexpr int SMP_CHUNKS = 32;
struct SampleArgs {
    const float* logits;    // [M][V]
    int V;
    const int* row_sid;     // [M] completion id keyed into Philox (never the batch slot)
    const int* step_dev;    // [1] 1-based generated-token index t
    const int* m_dev; int m_max;
    const uint32_t* params; // device [4] = mode, temperature (float bits), Philox key lo, key hi
    int row_div;            // logits row of activation row i is i / row_div (first token: G)
    float* part_score;      // [M][SMP_CHUNKS] best perturbed score of each vocabulary slice
    int* part_tok;          // [M][SMP_CHUNKS] and its token id (0x7fffffff if the slice is empty)
};
int launch_sample(const SampleArgs& a, cudaStream_t st);
int launch_philox_debug(uint64_t seed, int sid, int t, int v0, int n, uint32_t* out, cudaStream_t st);

// Teacher-forced log-prob pass (row f4): row descriptors of prompt + generated tokens, and log-softmax at the target token.
int launch_score_rows(const int* prompt_tokens, const int* prompt_offs_dev, const int* seq_off_dev, const int* gen_tokens, int nseq,
                      int G, int max_new, int total, int* row_sid, int* row_pos, int* row_ctx, int* row_tok, cudaStream_t st);
int launch_token_logprob(const float* logits, int V, int rows, const int* row_sid, const int* row_pos, const int* prompt_offs_dev, int G,
                         const int* gen_tokens, int max_new, float* out, cudaStream_t st);

// Segmented per-group statistics.  Step a14.
int launch_group_advantage(const float* rewards, const int* offs, int n_groups, int mode, int ddof,
                           float eps, float* adv, uint8_t* keep, cudaStream_t st);
int launch_length_stats(const int* lengths, const int* offs, int n_groups, int* stats, float* ratio,
                        cudaStream_t st);

// Paging / retirement state machine (steps a1, a4, a13).  All arrays live on the device.
struct PageState {
    int* free_stack; int* n_free; int* refcnt; int* page_table; int* n_blocks; int* n_shared;
    int* live; int* n_live; int* pos; int* ctx; int* tok; int* step; int* err; int* peak_used;
    int* alloc_log; int* n_alloc; int* retire_log; int* n_retire; int log_cap_alloc, log_cap_retire;
    int n_pages, max_blocks, page, max_seqs;
};
struct RolloutDev {
    const int* prompt_len;      // [n_prompts]
    const int* forced_len;      // [nseq] or null
    const int* forced_tok;      // [nseq][max_new] or null
    int* out_tokens;            // [nseq][max_new]
    int* out_lengths;           // [nseq]
    int n_prompts, G, nseq, max_new, stop_token, log;
};
int launch_pool_reset(const PageState& ps, const RolloutDev& rd, cudaStream_t st);
int launch_prefill_alloc(const PageState& ps, const RolloutDev& rd, cudaStream_t st);
// End of step t (retire / free / compact) + start of step t+1 (page alloc, pos/ctx/tok).
// `sampled` holds the sampler's token for each live slot; first_step: slots are sids (t = 1).
int launch_advance(const PageState& ps, const RolloutDev& rd, const float* part_score, const int* part_tok,
                   int structure_only, cudaStream_t st, int n_parts = 32 /* SMP_CHUNKS */, int part_sc = 1,
                   int part_si = 32);      // candidate c of slot i at [c * part_sc + i * part_si]
// Prefill helpers: row_sid/row_pos/row_ctx/tok for every prompt token, and the copy of a partial
// last prompt block into the first private page of completions g >= 1.
int launch_prefill_rows(const int* prompt_tokens, const int* prompt_offsets_dev, int n_prompts, int G,
                        int total_rows, int* row_sid, int* row_pos, int* row_ctx, int* row_tok,
                        cudaStream_t st);
int launch_copy_partial_block(const PageState& ps, const RolloutDev& rd, bf16_t* kv_pool,
                              size_t layer_stride, int n_layers, int page_elems, cudaStream_t st);
// Gather the last prompt row of each prompt's logits source: xlast[p] = x[offsets[p+1]-1].
int launch_gather_rows(const float* x, const int* row_idx, int n, int d, float* out, cudaStream_t st);
// Copy the logits row of every (sid, t) dump request whose t equals the current step.
int launch_dump_logits(const int* dump_sid_t, int n_dump, const int* step_dev, const int* live, const int* n_live,
                       int row_div, const float* logits, int V, float* out, cudaStream_t st);


// ---- tcgen05 path (tc_linear.cu) --------------------------------------------------------------
struct alignas(64) TcMap { unsigned char opaque[128]; };     // mirrors CUtensorMap
int tc_make_map(TcMap* out, const void* base, long long rows, int K, int box_rows);
int tc_nb_index(int m_max);                                  // 0..3 -> UMMA N = 32, 64, 128, 256
// K-split ranks and k blocks per rank that launch_linear_tc will use for a GEMM of this shape (so that the PREVIOUS kernel can prefetch its streams)
int tc_plan(int N, int K, int m_max, bool swiglu, bool has_scratch, int* kb_per_cta);
static constexpr size_t TC_SCRATCH_FLOATS = (size_t)296 * 2 * 128 * 128;   // 296 CTAs x NA 2 x 128 cols x 128 rows
struct TcLinearArgs {
    const TcMap* a[3];          // weight maps (box 64 x 128): {w} | {q, k, v} | {gate, up}
    int seg_rows[3];
    const TcMap* b;             // activation map for the chosen N (box 64 x N): pre-split rows
    int K, N;                   // N = output rows (EPI_SWIGLU: d_ff)
    const int* m_dev; int m_max;
    int epi;
    float* Y; int ldy; const float* R;
    bf16_t* xs_out; int ld_xs; const bf16_t* norm_next; float* ssq_out;
    const float* ssq_in; int ssq_in_tiles; int ssq_ld; float eps; int k_norm;
    // EPI_QKV: rotate q and k (RoPE), store q as fp32 into Y, round k / v to bf16 into the sequence's KV page
    const float* rope_cs; const int* row_pos; const int* row_sid; const int* page_table; bf16_t* kv_layer;
    int max_blocks, page, Hkv, hd, q_rows, kv_rows;
    float* scratch;             // >= TC_SCRATCH_FLOATS floats for the split-K partial tiles (null: no K split)
    bool pdl;
};
int launch_linear_tc(const TcLinearArgs& t, cudaStream_t st);
// Fused final norm + LM head + sampler (persistent tcgen05 kernel, <= 64 live rows).  Steps a11 + a12.
static constexpr int LM_MAX_PARTS = 160;                     // candidates per row = CTAs of the fused kernel
struct LmSampleArgs {
    const TcMap* a;             // lm_head map (box 64 x 128)
    const TcMap* b;             // pre-split activation map for the chosen N
    int K, V;
    const int* m_dev; int m_max;
    const float* ssq_in; int ssq_in_tiles; int ssq_ld; float eps; int k_norm;
    const int* row_sid; const int* step_dev; const uint32_t* params;
    float* part_score; int* part_tok; int part_ld;           // [lm_sample_grid(V)][part_ld]
    float* Y; int ldy;          // optional logits dump (null in the product path)
    bool pdl;
};
int lm_sample_grid(int V);
int launch_lmhead_sample(const LmSampleArgs& t, cudaStream_t st);
int launch_pick_candidates(const float* part_score, const int* part_tok, int n_parts, int ld, int M, int* out_tok, cudaStream_t st);
int launch_embed_split(const bf16_t* embed, const int* tok, const int* m_dev, int m_max, int d, float* x,
                       const bf16_t* norm_w, bf16_t* xs, float* ssq, int ssq_ld, int ssq_tiles, cudaStream_t st);
int launch_split_rows(const float* x, int K, const int* m_dev, int m_max, bf16_t* xs, cudaStream_t st);

// ---- persistent decode-step kernel (decode_step.cu) ----------------------------------------------
static constexpr int STEP_KS_MAX = 16;                        // widest K split of one output tile
struct StepSeg { int tile, kb0, kb1, rank, ks, slot0, pad0, pad1; };   // one unit: weight tile x k blocks [kb0, kb1)
struct StepPhasePlan { int nseg, pad[3]; StepSeg seg[2]; };   // the units of one CTA in one GEMM phase
struct StepGemm { int K, n_kb, tiles, na, seg0_tiles, seg1_tiles, tile_ctr_off, ks; };   // phases: 0 QKV, 1 O, 2 gate/up, 3 down
struct StepLaunch {
    int n_layers, n_cta, n_slots, m_max;
    StepGemm g[4];
    const void* wmaps_dev;                  // device CUtensorMap [n_layers][7]
    const StepPhasePlan* plan_dev;          // device [4][n_cta]
    float* xa; float* xb;                   // fp32 residual stream ping-pong [64][d_model]
    long long* accQ; long long* accO; long long* accG; long long* accD;   // fixed-point sums [64][Nqkv | d | 2 d_ff | d]
    float* rstd1; float* rstd2;             // [64]
    float* x; bf16_t* xs; bf16_t* att_s; float* ssq;
    int ssq_ld, d_tiles, d_model, Nqkv, qd, d_ff;
    const bf16_t* const* norm1_dev; const bf16_t* const* norm2_dev; const bf16_t* final_norm; const bf16_t* embed;
    float eps;
    unsigned* sync_base; int gbar_n;        // [2][gbar_n] phase counters
    const int* live; const int* pos; const int* ctx; const int* tok; const int* n_live; const int* step;
    AttnArgs att;                           // everything but kv_layer / kv_layer_w (set per layer in the kernel)
    bf16_t* kv_pool; size_t layer_stride;
    int* err;
    unsigned long long* trace;              // optional in-kernel timeline (SAGC_STEP_TRACE=1), else null
    bool cooperative, pdl;
};
int launch_decode_step(const StepLaunch& s, cudaStream_t st);
// static unit -> CTA schedule of the four GEMM phases of a layer; false if the shape does not fit (<= 2 units per CTA and phase)
bool build_step_plan(int n_cta, int d_model, int qd, int kvd, int d_ff, StepGemm g[4], std::vector<StepPhasePlan>& plan,
                     int* tiles_per_layer);
int step_smem_bytes(int n_slots);
int launch_attention_units(const AttnArgs& a, int n_cta, cudaStream_t st);   // parity entry: head_dim 64 / 128
int step_ring_slots(int smem_limit);

}  // namespace sagc
