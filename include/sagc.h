/* sagc.h -- C ABI of the B200 (sm_100a) rollout hot path.
 *
 * What this library computes (citations: P:<line> = /root/reference/PAPER.md line):
 *   - Synchronous group rollout generation: "for each prompt x we sample a group of G
 *     completions" from one policy snapshot, and "the update is bottlenecked by the longest
 *     completion" (sec 3.1; Alg.1 l.7).  The GPU reports "per-sequence token
 *     counts l_i" and per-group summaries l_max / l_median; R = max/median (Eq.1,
 *     P:78) and max/mean (Fig.1 caption) are both derivable from the outputs.
 *   - Group-relative advantages: "use group-relative baselines (e.g., mean/standardized
 *     rewards)", GRPO and DAPO.
 * Everything the paper leaves open (decoder, paging, sampler, advantage formula) follows the
 * readings listed in DESIGN.md; the CPU oracle under oracle/ states the same readings.
 *
 * Conventions
 *   - Plain C.  Every entry point returns 0 on success or a negative SAGC_E* code;
 *     sagc_last_error() returns a thread-local message for the last failure.
 *   - "dev" = pointer to device (HBM) memory, "host" = pointer to host memory.  The caller
 *     owns every buffer it passes; the library never frees them.  Weight buffers must stay
 *     valid for the lifetime of the model handle (they are read in place).
 *   - The library owns the opaque handle: KV page pool, page tables, free stack, scratch
 *     activations, RoPE table, packed weight tiles, CUDA graphs.
 *   - All work is enqueued on the caller's stream (`stream` is a cudaStream_t passed as
 *     void*; NULL = legacy default stream).  Calls that write host outputs synchronise the
 *     stream before returning; the others are asynchronous.  One handle = one stream at a
 *     time (a handle is not thread-safe).
 *   - There is no CPU fallback: without a CUDA device every compute call fails with SAGC_ECUDA.
 */
#ifndef SAGC_H_
#define SAGC_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SAGC_OK       0
#define SAGC_EINVAL  -1   /* bad argument / unsupported shape                         */
#define SAGC_ENOMEM  -2   /* cudaMalloc failed                                        */
#define SAGC_EPAGES  -3   /* KV page pool exhausted (no preemption; P: north_star)    */
#define SAGC_ECUDA   -4   /* CUDA runtime error (message in sagc_last_error)          */

#define SAGC_MODE_GREEDY 0
#define SAGC_MODE_GUMBEL 1

#define SAGC_ADV_GRPO 0
#define SAGC_ADV_DAPO 1

#define SAGC_PATH_AUTO 0  /* tcgen05/TMEM kernels at every batch size when the shapes are multiples of 128 (the
                             persistent decode-step kernel at <= 64 live rows, per-layer kernels above), else the
                             register-HMMA kernels: measured faster than the GEMV kernels even with 1 live row */
#define SAGC_PATH_GEMV 1  /* force the fp32-activation GEMV kernels for every batch size   */
#define SAGC_PATH_GEMM 2  /* force the tensor-core kernels for every batch size            */

#define SAGC_FLAG_STRUCTURE_ONLY 1  /* run paging / retirement / lengths only, no model forward;
                                       tokens are written as 0 (needs forced_lengths)          */
#define SAGC_FLAG_LOG            2  /* record the page-allocation and retirement logs          */
#define SAGC_FLAG_NO_GRAPH       4  /* launch kernels directly instead of through CUDA graphs  */
#define SAGC_FLAG_TIME_KERNELS   8  /* (implies NO_GRAPH) CUDA events around the three parts of every decode step:
                                       layer stack, LM head + sampler, advance -> timing->kernel_ms[] */

typedef struct sagc_model sagc_model;

/* Decoder shape (BASELINE.json configs) and KV-pool geometry. */
typedef struct {
    int32_t n_layers, d_model, n_q_heads, n_kv_heads, head_dim, d_ff, vocab;
    float   rope_theta, rms_eps;
    int32_t page_tokens;   /* tokens per KV page: 16, 32 or 64                           */
    int32_t n_pages;       /* pages in the pool; one page id covers all layers, K and V  */
    int32_t max_seqs;      /* upper bound on n_prompts*G of any rollout (<= 1024)        */
    int32_t max_ctx;       /* upper bound on prompt length + max_new_tokens              */
} sagc_model_config;

/* bf16 weights, row-major [out][in] (y = W x), all dev pointers.  The per-layer members
 * are HOST arrays of n_layers dev pointers.  Norm gains are bf16 vectors. */
typedef struct {
    const void* embed;        /* [vocab][d_model]                    */
    const void* lm_head;      /* [vocab][d_model]                    */
    const void* final_norm;   /* [d_model]                           */
    const void* const* wq;    /* [n_q_heads*head_dim][d_model]       */
    const void* const* wk;    /* [n_kv_heads*head_dim][d_model]      */
    const void* const* wv;    /* [n_kv_heads*head_dim][d_model]      */
    const void* const* wo;    /* [d_model][n_q_heads*head_dim]       */
    const void* const* wg;    /* [d_ff][d_model]                     */
    const void* const* wu;    /* [d_ff][d_model]                     */
    const void* const* wd;    /* [d_model][d_ff]                     */
    const void* const* norm1; /* [d_model]                           */
    const void* const* norm2; /* [d_model]                           */
} sagc_weights;

/* Create / destroy.  Fails with SAGC_EINVAL on unsupported shapes (head_dim not in
 * {32,64,128}, n_q_heads % n_kv_heads != 0, n_q_heads/n_kv_heads > 8, dims not multiples
 * of 8), SAGC_ENOMEM when the pool or scratch cannot be allocated. */
int  sagc_model_create(const sagc_model_config* cfg, const sagc_weights* w, sagc_model** out);
void sagc_model_destroy(sagc_model* m);

typedef struct {
    int32_t  mode;              /* SAGC_MODE_*                                              */
    float    temperature;       /* > 0 (used in GUMBEL mode)                                */
    uint64_t seed;              /* Philox key = (seed & 0xffffffff, seed >> 32)             */
    int32_t  stop_token;        /* -1 = none; a stop token is counted in the length  */
    int32_t  max_new_tokens;    /* L_max of P:76; >= 1                                      */
    const int32_t* forced_lengths;  /* HOST [n_prompts*G] or NULL: completion sid retires
                                       when its length reaches forced_lengths[sid]          */
    const int32_t* forced_tokens;   /* dev [n_prompts*G][max_new_tokens] or NULL: teacher
                                       forcing -- token t of sid is taken from here instead
                                       of the sampler (the sampler still runs)              */
    int32_t  path;              /* SAGC_PATH_*                                              */
    int32_t  flags;             /* SAGC_FLAG_* bit set                                      */
    /* optional logits dump: n_dump (sid, t) pairs, t = 1-based generated-token index; the
       row of logits from which token t of sid is sampled is copied to dump_logits[i][vocab] */
    int32_t  n_dump;
    const int32_t* dump_sid_t;  /* HOST [n_dump][2], or NULL                                */
    float*   dump_logits;       /* dev [n_dump][vocab], or NULL                             */
} sagc_rollout_params;

/* Per-phase accounting written by sagc_rollout_group when `timing` != NULL (forces a stream
 * synchronise).  Phases: FULL = decode steps with live >= nseq/2,
 * TAIL = live <= 8, MID = the rest.  Bytes are ALGORITHMIC: weights once per step + each
 * prompt's prefix KV once per live group + each live sequence's own suffix + the KV written. */
typedef struct {
    double  prefill_ms, decode_ms;
    double  phase_ms[3];        /* FULL, MID, TAIL                                          */
    int64_t phase_steps[3];
    int64_t phase_tokens[3];
    double  phase_bytes[3];
    int64_t prefill_tokens;
    double  prefill_flops;
    int64_t total_tokens;       /* generated tokens, all phases + the first token           */
    int64_t kernel_launches;    /* kernels of this library launched by the call             */
    /* SAGC_FLAG_TIME_KERNELS: device time of the decode steps by part, summed over the rollout:
       [0] layer stack (the persistent decode-step kernel, or the per-layer kernels), [1] LM head +
       sampler, [2] advance (retire / compact / page allocation); kernel_steps = steps measured   */
    double  kernel_ms[3];
    int64_t kernel_steps;
} sagc_rollout_timing;

/* Synchronous group rollout (Alg.1 l.7).  sid = p*G + g (prompt-major).
 *   prompt_tokens  dev  int32, prompts concatenated
 *   prompt_offsets HOST int32 [n_prompts+1]
 *   out_tokens     dev  int32 [n_prompts*G][max_new_tokens], padded with -1
 *   out_lengths    dev  int32 [n_prompts*G]                    (l_i of P:76)
 *   out_ratio      dev  float [n_prompts]   max/mean length per group, may be NULL
 *   out_len_stats  dev  int32 [n_prompts][3] = max, sum, median_x2 (Eq.1: R =
 *                  2*max/median_x2), may be NULL
 * Errors: SAGC_EINVAL (shape limits), SAGC_EPAGES (pool exhausted), SAGC_ECUDA. */
int sagc_rollout_group(sagc_model* m, const int32_t* prompt_tokens, const int32_t* prompt_offsets,
                       int32_t n_prompts, int32_t G, const sagc_rollout_params* params,
                       int32_t* out_tokens, int32_t* out_lengths, float* out_ratio,
                       int32_t* out_len_stats, sagc_rollout_timing* timing, void* stream);

/* Same call with HOST buffers for prompt_tokens and all four outputs: copies the prompts to
 * the device, runs the rollout, copies tokens / lengths / ratio / stats back and synchronises.
 * params->forced_tokens and dump_logits stay dev pointers. */
int sagc_rollout_group_host(sagc_model* m, const int32_t* prompt_tokens, const int32_t* prompt_offsets,
                            int32_t n_prompts, int32_t G, const sagc_rollout_params* params,
                            int32_t* out_tokens, int32_t* out_lengths, float* out_ratio,
                            int32_t* out_len_stats, sagc_rollout_timing* timing, void* stream);

/* Teacher-forced log-prob pass: log pi(y_t | x, y_<t) of every generated token under the same policy
 * snapshot -- the quantity the GRPO / DAPO loss needs next.  ONE causal pass per sequence over prompt +
 * completion with the prefill kernels (not token by token), the LM head over every position, log-softmax at the target.
 *   prompt_tokens dev int32 (concatenated); prompt_offsets HOST int32 [n_prompts+1];
 *   tokens dev int32 [n_prompts*G][max_new] (as returned by sagc_rollout_group); lengths HOST int32 [n_prompts*G];
 *   out_logprobs dev float [n_prompts*G][max_new], 0 beyond each length.
 * Uses (and overwrites) the handle's KV pool and page tables: needs sum(ceil((P + l - 1) / page_tokens)) pages.
 * Synchronises the stream.  Errors: SAGC_EINVAL, SAGC_EPAGES, SAGC_ECUDA. */
int sagc_score_tokens(sagc_model* m, const int32_t* prompt_tokens, const int32_t* prompt_offsets, int32_t n_prompts, int32_t G,
                      const int32_t* tokens, const int32_t* lengths, int32_t max_new, float* out_logprobs, void* stream);

/* Group-relative advantages.  Group g = rewards[off[g] : off[g+1]].
 *   all-equal group (max == min, exact) or size 1: A = 0, keep = 0 (DAPO) / 1 (GRPO)
 *   else A_i = (r_i - mean) / (std + eps), std with divisor (G - ddof); keep = 1.
 *   rewards dev float [n]; group_offsets dev int32 [n_groups+1] (CSR);
 *   out_adv dev float [n]; out_keep dev uint8 [n_groups]. Asynchronous. */
int sagc_group_advantage(const float* rewards, const int32_t* group_offsets, int32_t n_groups,
                         int32_t mode, int32_t ddof, float eps, float* out_adv, uint8_t* out_keep,
                         void* stream);

/* Per-group length statistics (Eq.1): max, sum, median_x2 and max/mean.
 *   lengths dev int32 [n]; group_offsets dev int32 [n_groups+1];
 *   out_stats dev int32 [n_groups][3] (may be NULL); out_ratio dev float [n_groups] (may be NULL). */
int sagc_length_stats(const int32_t* lengths, const int32_t* group_offsets, int32_t n_groups,
                      int32_t* out_stats, float* out_ratio, void* stream);

/* ---- debug / parity exports (state of the LAST rollout on this handle) ---------------- */
/* Page table: out HOST int32 [nseq][max_blocks], -1 = unmapped.  *max_blocks is written. */
int sagc_debug_page_table(sagc_model* m, int32_t* out, int32_t capacity, int32_t* nseq, int32_t* max_blocks);
/* Free stack, bottom to top: out HOST int32 [n_pages]; *n_free is written. */
int sagc_debug_free_stack(sagc_model* m, int32_t* out, int32_t capacity, int32_t* n_free);
/* Allocation log (needs SAGC_FLAG_LOG): out HOST int32 [n][3] = step, sid, page (step 0 = prefill). */
int sagc_debug_alloc_log(sagc_model* m, int32_t* out, int32_t capacity, int32_t* n);
/* Retirement log (needs SAGC_FLAG_LOG): out HOST int32 [n][2] = step, sid. */
int sagc_debug_retire_log(sagc_model* m, int32_t* out, int32_t capacity, int32_t* n);
/* Peak number of pages in use during the last rollout. */
int sagc_debug_peak_pages(sagc_model* m, int32_t* peak);
/* In-kernel timeline of the persistent decode-step kernel (only when the handle was created with the environment
 * variable SAGC_STEP_TRACE=1; otherwise *n = 0): copies the (tag, nanosecond) pairs recorded so far to out HOST
 * uint64 [capacity][2] and arms the recording of decode step `record_step` (1-based step index) of the next rollout.
 * tag = cta << 40 | role << 32 | event << 16 | phase. */
int sagc_debug_step_trace(sagc_model* m, int64_t record_step, uint64_t* out, int32_t capacity, int32_t* n);
/* Philox4x32-10 draws of the sampler for vocab ids v0..v0+n-1 of (seed, sid, t): out dev uint32 [n]. */
int sagc_debug_philox(uint64_t seed, int32_t sid, int32_t t, int32_t v0, int32_t n, uint32_t* out, void* stream);
/* y[M][N] = x[M][K] . W[N][K]^T through the projection kernels (path = SAGC_PATH_GEMV | _GEMM).
 *   W dev bf16 [N][K], x dev float [M][K], y dev float [M][N]. */
int sagc_debug_linear(const void* W, const float* x, float* y, int32_t M, int32_t N, int32_t K,
                      int32_t path, void* stream);
/* Fused LM head + sampler of a decode step (steps a11 + a12: logits never stored), as a unit:
 *   tokens[m] = argmax_v( (x[m] . W[v]) / temperature + Gumbel(Philox(seed; sids[m], t, v)) )   (mode 1)
 *             = argmax_v(  x[m] . W[v] ), lowest v on exact ties                               (mode 0)
 *   W dev bf16 [V][K], x dev float [M][K] (1 <= M <= 64), sids dev int32 [M], out_tokens dev int32 [M],
 *   out_logits dev float [M][V] or NULL (optional dump of the logits the epilogue saw).  V % 128 == 0,
 *   K % 64 == 0.  Synchronises the stream when (mode, temperature, seed, t) change (parameter upload);
 *   returns SAGC_EINVAL on bad shapes. */
int sagc_debug_lm_sample(const void* W, const float* x, int32_t M, int32_t V, int32_t K, int32_t mode, float temperature,
                         uint64_t seed, int32_t t, const int32_t* sids, int32_t* out_tokens, float* out_logits,
                         void* stream);
/* One paged GQA decode-attention call over a caller-built cache (unit test of step a7):
 *   q dev float [M][Hq][hd]; kv dev bf16 pool laid out as the model lays it out for ONE layer:
 *   [n_pages][2][Hkv][page_tokens][hd]; page_table dev int32 [M][max_blocks]; ctx dev int32 [M];
 *   out dev float [M][Hq][hd].  n_splits (1..64) = K-splits per (row, kv head).
 *   variant 0: the standalone kernel (one CTA per unit; 2..8 splits merge inside a cluster through DSMEM,
 *              more through the L2 scratch);  variant 1: the units as the persistent decode-step kernel runs
 *              them (one CTA per SM looping over units, last-arriver merge; head_dim 64 / 128 only).
 *   variant 2: the tcgen05 kernel of the decode steps (TMA-staged pages, S and O in tensor memory; head_dim 64 / 128,
 *              pages of 8 .. 128 tokens; last-arriver merge for any n_splits).
 *   Synchronises the stream.  SAGC_EINVAL on bad shapes. */
int sagc_debug_attention(const float* q, const void* kv, const int32_t* page_table, const int32_t* ctx,
                         int32_t M, int32_t Hq, int32_t Hkv, int32_t hd, int32_t page_tokens,
                         int32_t max_blocks, int32_t n_splits, int32_t variant, float* out, void* stream);

/* The same split-K attention (step a7) for callers that may not allocate: code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc.  Arguments as sagc_debug_attention (all DEVICE pointers, caller
 * owned; out dev float [M][Hq][hd]); always the one-CTA-per-(row, kv head, split) kernel with the last-arriver
 * merge through scratch memory.  That scratch -- arrival counters, the live list, the (max, sum) pairs and the
 * partial outputs, 4 * (M*Hkv + M + M*Hq*n_splits*(2 + hd)) bytes plus 256-byte rounding of each part -- lives in
 * ONE static device array of SAGC_NOALLOC_SCRATCH_BYTES that every GPU which loads the library holds until exit.
 *   - calls no cudaMalloc / cudaFree / allocating library routine; enqueues two kernels on `stream` and returns
 *     WITHOUT synchronising (errors of the kernels themselves surface at the caller's next synchronisation);
 *   - SAGC_EINVAL with a message naming the sizes when the scratch need exceeds SAGC_NOALLOC_SCRATCH_BYTES, or on
 *     bad shapes; SAGC_ECUDA when the array's address cannot be taken or a launch fails;
 *   - every call shares the array (counters and live list are re-initialised at the start of each call): calls
 *     that OVERLAP on the GPU -- different streams without an event between them -- race and give garbage. */
#define SAGC_NOALLOC_SCRATCH_BYTES (8u << 20)
int sagc_attention_noalloc(const float* q, const void* kv, const int32_t* page_table, const int32_t* ctx,
                           int32_t M, int32_t Hq, int32_t Hkv, int32_t hd, int32_t page_tokens,
                           int32_t max_blocks, int32_t n_splits, float* out, void* stream);

const char* sagc_last_error(void);
const char* sagc_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SAGC_H_ */
