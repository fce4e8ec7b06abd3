// paging.cu -- paged KV bookkeeping: pool reset, prefix allocation, per-step page allocation,
// retirement, page release and stable batch compaction (steps a1, a4, a13).
//
// Order conventions (reading C3; they make the result bit-comparable with a
// sequential implementation): the free list is a LIFO stack whose pops initially return
// 0, 1, 2, ...; within a step pages are handed out in ascending sid; a retiring sequence
// pushes its private pages in ascending logical order, then the shared prefix pages if it is
// the last member of its group; retirements are processed in ascending sid; the live list
// stays sorted by sid.  The parallel version reproduces that order with exclusive scans.
#include "common.cuh"
#include "kernels.cuh"

namespace sagc {

static constexpr int PG_THREADS = 1024;

// exclusive scan of one int per thread over a 1024-thread CTA; returns the prefix, *total = sum
__device__ __forceinline__ int block_exscan(int v, int* warp_s, int* total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    __syncthreads();                      // protect warp_s from the previous scan's readers
    if (lane == 31) warp_s[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        int w = warp_s[lane];
        int winc = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int t = __shfl_up_sync(0xffffffffu, winc, o);
            if (lane >= o) winc += t;
        }
        warp_s[lane] = winc - w;
        if (lane == 31) warp_s[32] = winc;
    }
    __syncthreads();
    *total = warp_s[32];
    return warp_s[warp] + inc - v;
}

__global__ void k_pool_reset(PageState ps, RolloutDev rd) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int stride = gridDim.x * blockDim.x;
    for (int k = i; k < ps.n_pages; k += stride) { ps.free_stack[k] = ps.n_pages - 1 - k; ps.refcnt[k] = 0; }
    for (int k = i; k < ps.max_seqs * ps.max_blocks; k += stride) ps.page_table[k] = -1;
    for (int k = i; k < ps.max_seqs; k += stride) { ps.n_blocks[k] = 0; ps.n_shared[k] = 0; }
    for (int k = i; k < rd.nseq * rd.max_new; k += stride) rd.out_tokens[k] = -1;
    for (int k = i; k < rd.nseq; k += stride) rd.out_lengths[k] = 0;
    if (i == 0) {
        *ps.n_free = ps.n_pages; *ps.n_live = 0; *ps.step = 1; *ps.err = 0; *ps.peak_used = 0;
        *ps.n_alloc = 0; *ps.n_retire = 0;
    }
}
int launch_pool_reset(const PageState& ps, const RolloutDev& rd, cudaStream_t st) {
    k_pool_reset<<<296, 512, 0, st>>>(ps, rd);
    return 1;
}

// Prefix allocation: prompts ascending; floor(P/page) shared pages (refcount G), then, if
// P % page != 0, one private page per completion (ascending g).  On a fresh stack the k-th pop
// returns page k, so page ids are prefix sums.  One thread per prompt.
__global__ void __launch_bounds__(PG_THREADS) k_prefill_alloc(PageState ps, RolloutDev rd) {
    __shared__ int total_s;
    const int p = threadIdx.x;
    int base = 0, mine = 0, nsh = 0, part = 0;
    if (p < rd.n_prompts) {
        for (int k = 0; k <= p; ++k) {
            const int P = rd.prompt_len[k];
            const int c = P / ps.page + ((P % ps.page) ? rd.G : 0);
            if (k < p) base += c; else { mine = c; nsh = P / ps.page; part = (P % ps.page) != 0; }
        }
        if (p == rd.n_prompts - 1) total_s = base + mine;
    }
    __syncthreads();
    const int total = total_s;
    if (total > ps.n_pages) {
        if (threadIdx.x == 0) *ps.err = 1;
        return;
    }
    if (p < rd.n_prompts) {
        for (int b = 0; b < nsh; ++b) {
            const int pg = base + b;
            ps.refcnt[pg] = rd.G;
            if (rd.log && pg < ps.log_cap_alloc) {
                ps.alloc_log[pg * 3 + 0] = 0; ps.alloc_log[pg * 3 + 1] = p * rd.G; ps.alloc_log[pg * 3 + 2] = pg;
            }
        }
        for (int g = 0; g < rd.G; ++g) {
            const int sid = p * rd.G + g;
            int* row = ps.page_table + (size_t)sid * ps.max_blocks;
            for (int b = 0; b < nsh; ++b) row[b] = base + b;
            ps.n_shared[sid] = nsh;
            ps.n_blocks[sid] = nsh + part;
            if (part) {
                const int pg = base + nsh + g;
                row[nsh] = pg;
                if (rd.log && pg < ps.log_cap_alloc) {
                    ps.alloc_log[pg * 3 + 0] = 0; ps.alloc_log[pg * 3 + 1] = sid; ps.alloc_log[pg * 3 + 2] = pg;
                }
            }
        }
    }
    for (int i = threadIdx.x; i < rd.nseq; i += PG_THREADS) ps.live[i] = i;
    if (threadIdx.x == 0) {
        *ps.n_free = ps.n_pages - total;
        *ps.n_live = rd.nseq;
        *ps.peak_used = total;
        *ps.n_alloc = total;
        *ps.step = 1;
    }
}
int launch_prefill_alloc(const PageState& ps, const RolloutDev& rd, cudaStream_t st) {
    k_prefill_alloc<<<1, PG_THREADS, 0, st>>>(ps, rd);
    return 1;
}

// End of step t + start of step t+1.  One CTA, thread i = live slot i.
__global__ void __launch_bounds__(PG_THREADS) k_advance(PageState ps, RolloutDev rd, const float* part_score,
                                                        const int* part_tok, int structure_only, int n_parts,
                                                        int part_sc, int part_si) {
    __shared__ int warp_s[33];
    __shared__ int grp_live[1024], grp_ret[1024], grp_last[1024];
    trace_mark(28); pdl_wait(); trace_mark(29);
    pdl_launch();
    const int i = threadIdx.x;
    const int n_live = *ps.n_live;
    const int t = *ps.step;
    if (*ps.err) return;
    int n_free = *ps.n_free;
    for (int k = i; k < rd.n_prompts; k += PG_THREADS) { grp_live[k] = 0; grp_ret[k] = 0; grp_last[k] = -1; }
    // fused LM head + sampler: one candidate per CTA ([c][64] layout, <= 64 live rows).  All 1024 threads fetch them
    // in ONE round trip (thread = row i % 64, candidate subset i / 64), then slot i takes the best of 16 from shared memory.
    __shared__ float cand_s[16][64];
    __shared__ int cand_t[16][64];
    const bool wide = n_parts > 32 && part_si == 1 && !structure_only && !rd.forced_tok;
    if (wide) {
        const int r = i & 63, p = i >> 6;
        float b = -INFINITY;
        int ix = 0x7fffffff;
        if (r < n_live) {
#pragma unroll 10
            for (int c = p; c < n_parts; c += 16) {
                const float s2 = part_score[(size_t)c * part_sc + r];
                const int t2 = part_tok[(size_t)c * part_sc + r];
                if (s2 > b || (s2 == b && t2 < ix)) { b = s2; ix = t2; }
            }
        }
        cand_s[p][r] = b; cand_t[p][r] = ix;
    }
    __syncthreads();

    // ---- append token, decide retirement ---------------------------------------------
    int sid = -1, tokv = 0, fin = 0, grp = 0, nb = 0, nsh = 0;
    const bool has = i < n_live;
    if (has) {
        sid = ps.live[i];
        grp = sid / rd.G;
        if (rd.forced_tok) tokv = rd.forced_tok[(size_t)sid * rd.max_new + (t - 1)];
        else if (!structure_only) {
            // best of the sampler's per-slice candidates, ascending slices: lowest index wins ties
            // candidate c of slot i sits at [c * part_sc + i * part_si] (k_sample: slices; fused LM head: CTAs)
            float bs;
            if (wide) {
                bs = cand_s[0][i]; tokv = cand_t[0][i];
#pragma unroll
                for (int c = 1; c < 16; ++c) {
                    const float s2 = cand_s[c][i];
                    const int t2 = cand_t[c][i];
                    if (s2 > bs || (s2 == bs && t2 < tokv)) { bs = s2; tokv = t2; }
                }
            } else {
                bs = part_score[(size_t)i * part_si];
                tokv = part_tok[(size_t)i * part_si];
#pragma unroll 8
                for (int c = 1; c < n_parts; ++c) {
                    const float s2 = part_score[(size_t)c * part_sc + (size_t)i * part_si];
                    const int t2 = part_tok[(size_t)c * part_sc + (size_t)i * part_si];
                    if (s2 > bs || (s2 == bs && t2 < tokv)) { bs = s2; tokv = t2; }
                }
            }
        }
        rd.out_tokens[(size_t)sid * rd.max_new + (t - 1)] = tokv;
        rd.out_lengths[sid] = t;
        fin = (rd.forced_len && rd.forced_len[sid] == t) || (rd.stop_token >= 0 && tokv == rd.stop_token) ||
              (t == rd.max_new);
        nb = ps.n_blocks[sid];
        nsh = ps.n_shared[sid];
        atomicAdd(&grp_live[grp], 1);
        if (fin) { atomicAdd(&grp_ret[grp], 1); atomicMax(&grp_last[grp], sid); }
    }
    __syncthreads();

    // ---- retire: push pages in ascending sid ------------------------------------------
    int n_push = 0, push_shared = 0;
    if (has && fin) {
        push_shared = (grp_last[grp] == sid) && (grp_ret[grp] == grp_live[grp]);
        n_push = (nb - nsh) + (push_shared ? nsh : 0);
    }
    int total_push, total_ret;
    const int push_off = block_exscan(n_push, warp_s, &total_push);
    const int ret_off = block_exscan(has && fin ? 1 : 0, warp_s, &total_ret);
    if (has && fin) {
        const int* row = ps.page_table + (size_t)sid * ps.max_blocks;
        int w = n_free + push_off;
        for (int b = nsh; b < nb; ++b) ps.free_stack[w++] = row[b];
        if (grp_last[grp] == sid) {      // one member settles the group's refcounts
            for (int b = 0; b < nsh; ++b) {
                const int pg = row[b];
                ps.refcnt[pg] -= grp_ret[grp];
                if (push_shared) ps.free_stack[w++] = pg;
            }
        }
        if (rd.log && (*ps.n_retire + ret_off) < ps.log_cap_retire) {
            int* e = ps.retire_log + (size_t)(*ps.n_retire + ret_off) * 2;
            e[0] = t; e[1] = sid;
        }
    }
    n_free += total_push;

    // ---- stable compaction + allocation for step t+1 -----------------------------------
    const int keep = has && !fin;
    int n_new;
    const int slot = block_exscan(keep, warp_s, &n_new);
    int pos = 0, need = 0;
    if (keep) {
        pos = rd.prompt_len[grp] + t - 1;             // KV position written by step t+1
        need = (pos % ps.page) == 0;
    }
    int total_need;
    const int rank = block_exscan(need, warp_s, &total_need);
    const bool exhausted = total_need > n_free;
    if (keep) {
        ps.live[slot] = sid;                          // slot <= i and all reads happened before the scans
        ps.pos[slot] = pos;
        ps.ctx[slot] = pos + 1;
        ps.tok[slot] = tokv;
        if (need && !exhausted) {
            const int pg = ps.free_stack[n_free - 1 - rank];
            ps.page_table[(size_t)sid * ps.max_blocks + pos / ps.page] = pg;
            ps.n_blocks[sid] = pos / ps.page + 1;
            if (rd.log && (*ps.n_alloc + rank) < ps.log_cap_alloc) {
                int* e = ps.alloc_log + (size_t)(*ps.n_alloc + rank) * 3;
                e[0] = t + 1; e[1] = sid; e[2] = pg;
            }
        }
    }
    __syncthreads();
    if (i == 0) {
        if (exhausted) { *ps.err = 1; }
        else {
            n_free -= total_need;
            *ps.n_alloc += total_need;
            const int used = ps.n_pages - n_free;
            if (used > *ps.peak_used) *ps.peak_used = used;
        }
        *ps.n_free = n_free;
        *ps.n_retire += total_ret;
        *ps.n_live = exhausted ? 0 : n_new;      // pool exhausted: the remaining steps of the rollout see no live rows
        *ps.step = t + 1;
    }
}
int launch_advance(const PageState& ps, const RolloutDev& rd, const float* part_score, const int* part_tok,
                   int structure_only, cudaStream_t st, int n_parts, int part_sc, int part_si) {
    launch_pdl(k_advance, dim3(1), dim3(PG_THREADS), 0, st, g_pdl_all, ps, rd, part_score, part_tok, structure_only, n_parts,
               part_sc, part_si);
    return 1;
}

// Copy the partially filled last prompt block from completion 0 of each group into the first
// private page of completions g >= 1 ("copied, not recomputed").  grid = (nseq, n_layers).
__global__ void k_copy_partial(PageState ps, RolloutDev rd, bf16_t* kv_pool, size_t layer_stride,
                               int page_elems) {
    const int sid = blockIdx.x, layer = blockIdx.y;
    const int p = sid / rd.G, g = sid % rd.G;
    const int P = rd.prompt_len[p];
    if (g == 0 || (P % ps.page) == 0) return;
    const int b = P / ps.page;
    const int src = ps.page_table[(size_t)(p * rd.G) * ps.max_blocks + b];
    const int dst = ps.page_table[(size_t)sid * ps.max_blocks + b];
    if (src < 0 || dst < 0) return;
    const uint4* s = reinterpret_cast<const uint4*>(kv_pool + layer * layer_stride + (size_t)src * page_elems);
    uint4* d = reinterpret_cast<uint4*>(kv_pool + layer * layer_stride + (size_t)dst * page_elems);
    for (int k = threadIdx.x; k < page_elems / 8; k += blockDim.x) d[k] = s[k];
}
int launch_copy_partial_block(const PageState& ps, const RolloutDev& rd, bf16_t* kv_pool, size_t layer_stride,
                              int n_layers, int page_elems, cudaStream_t st) {
    dim3 grid(rd.nseq, n_layers);
    k_copy_partial<<<grid, 256, 0, st>>>(ps, rd, kv_pool, layer_stride, page_elems);
    return 1;
}

}  // namespace sagc
