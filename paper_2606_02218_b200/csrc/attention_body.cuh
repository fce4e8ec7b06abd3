// attention_body.cuh -- paged GQA decode attention over ragged contexts (step a7) as a device function, so that
// the standalone kernel (attention.cu: prefill, head_dim 32, > 64 live rows) and the persistent decode-step
// kernel (decode_step.cu) run the SAME code.
//
// One unit = (activation row, kv head, K-split), processed by 256 threads (8 warps).  The r = Hq/Hkv query
// heads that share a kv head are processed together so every K/V byte is read once per (row, kv head).
// Contexts are walked through the page table in tiles of WARPS*16 tokens staged in shared memory by an
// NSTAGE-deep cp.async pipeline (16-byte chunks XOR-swizzled so that fragment reads are conflict-free).
// Tensor-core formulation (HMMA m16n8k16, fp32 accumulate) with full-precision operands:
//   A rows g (0..7) carry the bf16 "hi" half of head g's operand and rows g+8 its "lo" half, so
//     S = q_hi.K + q_lo.K  and  O = p_hi.V + p_lo.V  are each the sum of two accumulator rows that
//     live in the SAME lane (c0/c1 and c2/c3) -- q and p keep ~16 mantissa bits, K and V are exact.
//   K^T is the B operand of S; lanes read 16-byte chunks of a token's row (the k order inside each
//     32-wide block is permuted identically for Q, which costs nothing).
//   V is the B operand of O through ldmatrix.trans.
// Each compute warp owns 16 tokens of a tile and keeps its own running (max, sum, O); the warps are merged
// once at the end.  Split-K: split s covers tokens [s*cps, (s+1)*cps); partials are merged with the
// log-sum-exp rule either inside a cluster through DSMEM (standalone kernel, 2..8 splits) or by the last
// unit to arrive for a (row, kv head) through an L2 scratch.
// Decode (fuse_rope): RoPE of q / k and the bf16 K,V append of the newest position happen here too.
#pragma once
#include <cooperative_groups.h>
#include "common.cuh"
#include "kernels.cuh"

namespace sagc {

static constexpr int ATT_THREADS = 256;      // all 8 warps stage K/V; the first WARPS of them compute
static constexpr int ATT_MAXR = 8;
static constexpr int ATT_MAXPG = 1104;       // page ids cached per split (17408 / 16 + slack)

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc, int src_bytes) {
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(d), "l"(gsrc), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

// attention output element (row, col): fp32, or pre-split hi / lo bf16 rows for the tcgen05 O-projection
__device__ __forceinline__ void store_out(const AttnArgs& a, int row, int col, float v) {
    if (a.out_split != nullptr) {
        const uint32_t hi = f32_to_bf16_bits(v);
        a.out_split[(size_t)(2 * row) * a.ld_split + col] = (bf16_t)hi;
        a.out_split[(size_t)(2 * row + 1) * a.ld_split + col] = (bf16_t)f32_to_bf16_bits(v - __uint_as_float(hi << 16));
    } else {
        a.out[(size_t)row * a.Hq * a.hd + col] = v;
    }
}

// element(s) of the activation row that holds q | k | v: fp32, or 64-bit fixed point * 2^-32 * (1/rms of the row)
static constexpr float ATT_FX_SCALE = 2.3283064365386963e-10f;      // 2^-32
template <bool FX = true>
__device__ __forceinline__ void att_load8(const AttnArgs& a, int row, size_t col, float rs, float (&o)[8]) {
    if (FX && a.q_fx != nullptr) {
        const longlong2* p = reinterpret_cast<const longlong2*>(a.q_fx + (size_t)row * a.ldq + col);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const longlong2 v = __ldcg(p + i);
            o[2 * i] = __ll2float_rn(v.x) * ATT_FX_SCALE * rs;
            o[2 * i + 1] = __ll2float_rn(v.y) * ATT_FX_SCALE * rs;
        }
    } else {
        const float4 x0 = __ldcg(reinterpret_cast<const float4*>(a.q + (size_t)row * a.ldq + col));
        const float4 x1 = __ldcg(reinterpret_cast<const float4*>(a.q + (size_t)row * a.ldq + col + 4));
        o[0] = x0.x; o[1] = x0.y; o[2] = x0.z; o[3] = x0.w; o[4] = x1.x; o[5] = x1.y; o[6] = x1.z; o[7] = x1.w;
    }
}
template <bool FX = true>
__device__ __forceinline__ float att_load1(const AttnArgs& a, int row, size_t col, float rs) {
    if (FX && a.q_fx != nullptr) return __ll2float_rn(__ldcg(a.q_fx + (size_t)row * a.ldq + col)) * ATT_FX_SCALE * rs;
    return __ldcg(a.q + (size_t)row * a.ldq + col);
}

__device__ __forceinline__ void ldmatrix_x4_trans(uint32_t (&r)[4], const void* smem_row) {
    const uint32_t a = (uint32_t)__cvta_generic_to_shared(smem_row);
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];\n"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3])
                 : "r"(a));
}

// K/V staging geometry: WARPS compute warps x 16 tokens per tile, NSTAGE tiles in the ring
template <int HD, int WARPS, int NSTAGE>
struct AttGeom {
    static constexpr int TILE = WARPS * 16;
    static constexpr int ROWB = HD * 2;                       // unpadded rows, 16-byte chunks XOR-swizzled
    static constexpr int STAGE = 2 * TILE * ROWB;             // K rows then V rows
    static constexpr int BYTES = NSTAGE * STAGE;
    static constexpr int OW_BYTES = WARPS * ATT_MAXR * (HD + 4) * 4;   // per-warp partial outputs, overlaid on the ring
    static_assert(OW_BYTES <= BYTES, "the warp-merge buffer overlays the K/V ring");
};

// small shared state of one unit (static __shared__ in the standalone kernel, carved from dynamic smem otherwise)
struct AttSmall {
    float m_w[8][ATT_MAXR], l_w[8][ATT_MAXR];
    float m_s[ATT_MAXR], l_s[ATT_MAXR];
    int last_s;
    int pg_s[ATT_MAXPG];                         // page ids of this split's blocks
};
// split merge inside a cluster (standalone kernel only): every split pushes slice k of its un-normalised output
// and its (max, sum) pairs into the shared memory of cluster rank k, which combines and stores that slice
template <int HD>
struct AttCluster {
    float rv_o[ATT_MAXR * HD + 8];               // [split][slice]
    float rv_ml[8][ATT_MAXR][2];
};

// MEGA = false: the unit is a whole CTA of 256 threads (__syncthreads, PDL, cluster merge allowed).
// MEGA = true : the unit is run by the 256 worker threads of the persistent decode-step kernel (named barrier 1).
template <bool MEGA>
__device__ __forceinline__ void att_sync() {
    if (MEGA) asm volatile("bar.sync 1, 256;\n" ::: "memory");
    else __syncthreads();
}

template <int HD, int WARPS, int NSTAGE, bool MEGA>
__device__ __forceinline__ void attention_unit(const AttnArgs& a, const int row, const int kvh, const int split, const int nsp,
                                               unsigned char* kv_s, AttSmall* sm, AttCluster<HD>* cl, const int tid) {
    using G = AttGeom<HD, WARPS, NSTAGE>;
    constexpr int ROWB = G::ROWB;
    constexpr int ATT_TILE = G::TILE;
    constexpr int ATT_STAGES = NSTAGE;
    constexpr int CPR = HD * 2 / 16;            // 16-byte chunks per row
    constexpr int KB = HD / 32;                 // 32-wide d blocks
    constexpr int NT = HD / 8;                  // output n-tiles
    float (*o_w)[ATT_MAXR][HD + 4] = reinterpret_cast<float (*)[ATT_MAXR][HD + 4]>(kv_s);   // valid after the tile loop only
    const bool cmerge = !MEGA && a.cluster_merge != 0;
    if (cmerge) asm volatile("barrier.cluster.arrive.relaxed.aligned;\n" ::: "memory");   // "this CTA has started"; waited on before the pushes
    const int r = a.Hq / a.Hkv;
    const int warp = tid >> 5, lane = tid & 31;
    const int g = lane >> 2, q = lane & 3;
    const int ctx = a.row_ctx[row];
    const int sid = a.row_sid[row];
    const int* pt = a.page_table + (size_t)sid * a.max_blocks;
    int cps = (ctx + nsp - 1) / nsp;
    cps = ((cps + ATT_TILE - 1) / ATT_TILE) * ATT_TILE;
    const int t_begin = split * cps;
    const int t_end = min(ctx, t_begin + cps);
    const int n_tiles = t_end > t_begin ? (t_end - t_begin + ATT_TILE - 1) / ATT_TILE : 0;
    const size_t head_stride = (size_t)a.page * HD;                 // one (page, K|V, kv head) slab
    const int pshift = 31 - __clz(a.page), pmask = a.page - 1;      // page_tokens is a power of two
    const int b_begin = t_begin >> pshift;
    const int n_blk = t_end > t_begin ? ((t_end - 1) >> pshift) - b_begin + 1 : 0;
    const bool pg_cached = n_blk <= ATT_MAXPG;
    if (MEGA) att_sync<MEGA>();                 // the previous unit of this CTA is done with pg_s and the ring
    if (pg_cached) {
        for (int b = tid; b < n_blk; b += ATT_THREADS) sm->pg_s[b] = pt[b_begin + b];
        att_sync<MEGA>();
    }

    // K chunk c of token j -> chunk c ^ ksw(j); V chunk c -> c ^ vsw(j)   (bank-conflict free)
    auto ksw = [](int j) { return CPR >= 8 ? ((j & 1) << 2) : 0; };
    auto vsw = [](int j) { return CPR >= 8 ? (j & 7) : ((j >> 1) & 3); };
    // Tile loader: 16-byte chunk c of the tile -> (token j = c / CPR, part = c % CPR).  (A variant with per-thread-constant
    // chunk / swizzle / base pointer -- 45 % fewer loader instructions -- measured 0.5 us SLOWER per launch at 64 rows x 2 kv heads.)
    auto load_tile = [&](int tile, int stage) {
        unsigned char* base = kv_s + (size_t)stage * G::STAGE;
        const int t0 = t_begin + tile * ATT_TILE;
#pragma unroll
        for (int c = tid; c < ATT_TILE * CPR; c += ATT_THREADS) {
            const int j = c / CPR, part = c % CPR;
            const int tok = t0 + j;
            const int blk = tok >> pshift;
            const int pg = (tok < t_end) ? (pg_cached ? sm->pg_s[blk - b_begin] : pt[blk]) : -1;
            const bool ok = pg >= 0;             // masked tail, or an unmapped block after a pool-exhaustion error: zero fill
            const bf16_t* kp = a.kv_layer + ((size_t)(ok ? pg : 0) * 2 * a.Hkv + kvh) * head_stride +
                               (size_t)(ok ? (tok & pmask) : 0) * HD + part * 8;
            const bf16_t* vp = kp + (size_t)a.Hkv * head_stride;
            cp_async16(base + (size_t)j * ROWB + ((part ^ ksw(j)) << 4), kp, ok ? 16 : 0);
            cp_async16(base + (size_t)(ATT_TILE + j) * ROWB + ((part ^ vsw(j)) << 4), vp, ok ? 16 : 0);
        }
    };
    // fused RoPE (decode): cos/sin of this row's position for the q fragments, fetched before the wait
    const bool fuse = a.fuse_rope != 0;
    float2 qcs[(KB / 2 > 0 ? KB / 2 : 1)][8];
    int pos_new = 0;
    if (fuse) {
        pos_new = a.row_pos[row];
#pragma unroll
        for (int kb = 0; kb < KB / 2; ++kb)
#pragma unroll
            for (int e = 0; e < 8; ++e)
                qcs[kb][e] = *reinterpret_cast<const float2*>(a.rope_cs + ((size_t)pos_new * (HD / 2) + kb * 32 + 8 * q + e) * 2);
    }
    // the split that holds the newest position appends its K,V (rotated, rounded to bf16)
    const bool designated = fuse && n_tiles > 0 && t_end == ctx;
    float2 kcs = make_float2(1.f, 0.f);
    if (designated && tid < HD / 2) kcs = *reinterpret_cast<const float2*>(a.rope_cs + ((size_t)pos_new * (HD / 2) + tid) * 2);
    // leading tiles that hold only positions older than ctx - 1 (at most ATT_STAGES - 1 of them) can be fetched
    // before the dependency wait: they were written by earlier steps
    int n_early = 0;
    if (a.prefetch) {
        while (n_early < ATT_STAGES - 1 && n_early < n_tiles && t_begin + (n_early + 1) * ATT_TILE <= ctx - 1) ++n_early;
    }
    for (int s2 = 0; s2 < n_early; ++s2) { load_tile(s2, s2); cp_async_commit(); }
    if (!MEGA) {
        if (a.prefetch) pdl_wait();
        trace_mark(13);
        pdl_launch();
    }
    for (int s2 = n_early; s2 < ATT_STAGES - 1; ++s2) { if (s2 < n_tiles) load_tile(s2, s2); cp_async_commit(); }

    // Q fragments (hi in rows g, lo in rows g+8), pre-scaled by 1/sqrt(hd); head g of this kv head
    uint32_t qf[KB][8];
    uint32_t knew = 0, vnew = 0;                    // designated unit: bf16 bits of the new k pair / v element
    {
        const float scale = rsqrtf((float)HD);
        const float rs = (MEGA && a.q_fx != nullptr) ? __ldcg(a.q_rstd + row) : 1.f;      // the fixed-point q source exists in the decode-step kernel only
        const size_t qcol = (size_t)(kvh * r + g) * HD + 8 * q;
        float xq[KB][8];
#pragma unroll
        for (int kb = 0; kb < KB; ++kb) {
            if (g < r) {
                att_load8<MEGA>(a, row, qcol + kb * 32, rs, xq[kb]);
            } else {
#pragma unroll
                for (int e = 0; e < 8; ++e) xq[kb][e] = 0.f;
            }
        }
        if (designated) {
            // raw k (pair i, i + hd/2) and v of the newest position from the same qkv row
            const size_t kcol = (size_t)a.Hq * HD + (size_t)kvh * HD;
            const size_t vcol = kcol + (size_t)a.Hkv * HD;
            if (tid < HD / 2) {
                const float k0 = att_load1<MEGA>(a, row, kcol + tid, rs), k1 = att_load1<MEGA>(a, row, kcol + tid + HD / 2, rs);
                knew = f32_to_bf16_bits(k0 * kcs.x - k1 * kcs.y) | (f32_to_bf16_bits(k1 * kcs.x + k0 * kcs.y) << 16);
            }
            if (tid < HD) vnew = f32_to_bf16_bits(att_load1<MEGA>(a, row, vcol + tid, rs));
        }
        if (fuse) {
#pragma unroll
            for (int kb = 0; kb < KB / 2; ++kb)
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const float lo = xq[kb][e], hi = xq[kb + KB / 2][e];
                    xq[kb][e] = lo * qcs[kb][e].x - hi * qcs[kb][e].y;
                    xq[kb + KB / 2][e] = hi * qcs[kb][e].x + lo * qcs[kb][e].y;
                }
        }
#pragma unroll
        for (int kb = 0; kb < KB; ++kb) {
            split2(xq[kb][0] * scale, xq[kb][1] * scale, qf[kb][0], qf[kb][4]);
            split2(xq[kb][2] * scale, xq[kb][3] * scale, qf[kb][1], qf[kb][5]);
            split2(xq[kb][4] * scale, xq[kb][5] * scale, qf[kb][2], qf[kb][6]);
            split2(xq[kb][6] * scale, xq[kb][7] * scale, qf[kb][3], qf[kb][7]);
        }
        if (designated) {
            // append to the page (for the later steps); this step's copy is patched into shared memory below
            const int tnew = ctx - 1;
            const int blk = tnew >> pshift;
            const int pg = pg_cached ? sm->pg_s[blk - b_begin] : pt[blk];
            if (pg >= 0) {
                bf16_t* kd = a.kv_layer_w + ((size_t)pg * 2 * a.Hkv + kvh) * head_stride + (size_t)(tnew & pmask) * HD;
                bf16_t* vd = kd + (size_t)a.Hkv * head_stride;
                if (tid < HD / 2) { kd[tid] = (bf16_t)(knew & 0xffffu); kd[tid + HD / 2] = (bf16_t)(knew >> 16); }
                if (tid < HD) vd[tid] = (bf16_t)vnew;
            }
        }
    }
    float o[NT][4];
#pragma unroll
    for (int n = 0; n < NT; ++n)
#pragma unroll
        for (int e = 0; e < 4; ++e) o[n][e] = 0.f;
    float m_run = -INFINITY, l_run = 0.f;       // head g (replicated over the quad)

    if (!MEGA) trace_mark(10 * 4 + 0);
    for (int tile = 0; tile < n_tiles; ++tile) {
        cp_async_wait<ATT_STAGES - 2>();
        att_sync<MEGA>();
        if (tile + ATT_STAGES - 1 < n_tiles) load_tile(tile + ATT_STAGES - 1, (tile + ATT_STAGES - 1) % ATT_STAGES);
        cp_async_commit();
        if (designated && tile == n_tiles - 1) {
            // the row of the newest position was copied stale from the page: overwrite it with the new K,V
            unsigned char* sb = kv_s + (size_t)(tile % ATT_STAGES) * G::STAGE;
            const int j = (ctx - 1) - (t_begin + tile * ATT_TILE);
            if (tid < HD / 2) {
                const int d0 = tid, d1 = tid + HD / 2;
                *reinterpret_cast<bf16_t*>(sb + (size_t)j * ROWB + (((d0 >> 3) ^ ksw(j)) << 4) + (d0 & 7) * 2) = (bf16_t)(knew & 0xffffu);
                *reinterpret_cast<bf16_t*>(sb + (size_t)j * ROWB + (((d1 >> 3) ^ ksw(j)) << 4) + (d1 & 7) * 2) = (bf16_t)(knew >> 16);
            }
            if (tid < HD)
                *reinterpret_cast<bf16_t*>(sb + (size_t)(ATT_TILE + j) * ROWB + (((tid >> 3) ^ vsw(j)) << 4) + (tid & 7) * 2) = (bf16_t)vnew;
            att_sync<MEGA>();
        }
        if (warp >= WARPS) continue;             // staging-only warps
        const unsigned char* kbase = kv_s + (size_t)(tile % ATT_STAGES) * G::STAGE;
        const unsigned char* vbase = kbase + (size_t)ATT_TILE * ROWB;
        const int tw = warp * 16;                // this warp's 16 tokens inside the tile
        const int t0 = t_begin + tile * ATT_TILE + tw;
        if (t0 >= t_end) continue;               // warp-uniform: nothing but masked tokens
        // ---- S = Q K^T for two 8-token n-tiles -------------------------------------------
        float s[2][4];
#pragma unroll
        for (int n = 0; n < 2; ++n) {
            s[n][0] = s[n][1] = s[n][2] = s[n][3] = 0.f;
            const int j = tw + n * 8 + g;        // B column = token
            const unsigned char* kr = kbase + (size_t)j * ROWB;
#pragma unroll
            for (int kb = 0; kb < KB; ++kb) {
                const uint4 w = *reinterpret_cast<const uint4*>(kr + (((kb * 4 + q) ^ ksw(j)) << 4));
                mma_bf16_16816(s[n], qf[kb][0], qf[kb][4], qf[kb][1], qf[kb][5], w.x, w.y);
                mma_bf16_16816(s[n], qf[kb][2], qf[kb][6], qf[kb][3], qf[kb][7], w.z, w.w);
            }
        }
        // full-precision score of head g for tokens (n*8 + 2q, +1): hi row + lo row
        float sc[4];
        sc[0] = s[0][0] + s[0][2]; sc[1] = s[0][1] + s[0][3];
        sc[2] = s[1][0] + s[1][2]; sc[3] = s[1][1] + s[1][3];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const int tok = t0 + (e >> 1) * 8 + 2 * q + (e & 1);
            if (tok >= t_end) sc[e] = -INFINITY;
        }
        float tmax = fmaxf(fmaxf(sc[0], sc[1]), fmaxf(sc[2], sc[3]));
        tmax = fmaxf(tmax, __shfl_xor_sync(0xffffffffu, tmax, 1));
        tmax = fmaxf(tmax, __shfl_xor_sync(0xffffffffu, tmax, 2));
        const float m_new = fmaxf(m_run, tmax);          // finite: token t0 is valid for every head
        const float f = __expf(m_run - m_new);           // exp(-inf) = 0 on the first tile
        float p[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) p[e] = __expf(sc[e] - m_new);
        float ls = p[0] + p[1] + p[2] + p[3];
        ls += __shfl_xor_sync(0xffffffffu, ls, 1);
        ls += __shfl_xor_sync(0xffffffffu, ls, 2);
        l_run = l_run * f + ls;
        m_run = m_new;
#pragma unroll
        for (int n = 0; n < NT; ++n) { o[n][0] *= f; o[n][1] *= f; o[n][2] *= f; o[n][3] *= f; }
        // P as the A operand: rows g = hi, rows g+8 = lo; k = 16 tokens
        uint32_t pa[4];
        split2(p[0], p[1], pa[0], pa[1]);
        split2(p[2], p[3], pa[2], pa[3]);
        // ---- O += P V : V^T fragments through ldmatrix.trans ------------------------------
        // lane -> (matrix = lane/8, row = lane%8): matrices 0,1 = tokens 0-7 / 8-15 of d block 2c,
        // matrices 2,3 = the same tokens of d block 2c+1
        const int lm = lane >> 3, lr = lane & 7;
        const int vtok = tw + (lm & 1) * 8 + lr;
        const unsigned char* vr = vbase + (size_t)vtok * ROWB;
#pragma unroll
        for (int c = 0; c < NT / 2; ++c) {
            uint32_t b[4];
            const int chunk = 2 * c + (lm >> 1);
            ldmatrix_x4_trans(b, vr + ((chunk ^ vsw(vtok)) << 4));
            mma_bf16_16816(o[2 * c], pa[0], pa[1], pa[2], pa[3], b[0], b[1]);
            mma_bf16_16816(o[2 * c + 1], pa[0], pa[1], pa[2], pa[3], b[2], b[3]);
        }
    }
    cp_async_wait<0>();
    att_sync<MEGA>();                            // every warp is done with the ring: o_w overlays it
    if (!MEGA) trace_mark(10 * 4 + 2);
    // ---- merge the compute warps (fixed order) ------------------------------------------------
    // lane (g, q) holds head g: o[n][0..1] + o[n][2..3] are columns n*8 + 2q, +1
    if (warp < WARPS && g < r) {
#pragma unroll
        for (int n = 0; n < NT; ++n) {
            o_w[warp][g][n * 8 + 2 * q] = o[n][0] + o[n][2];
            o_w[warp][g][n * 8 + 2 * q + 1] = o[n][1] + o[n][3];
        }
        if (q == 0) { sm->m_w[warp][g] = m_run; sm->l_w[warp][g] = l_run; }
    }
    att_sync<MEGA>();
    if (tid < r) {
        float mx = sm->m_w[0][tid];
#pragma unroll
        for (int w2 = 1; w2 < WARPS; ++w2) mx = fmaxf(mx, sm->m_w[w2][tid]);
        float l = 0.f;
#pragma unroll
        for (int w2 = 0; w2 < WARPS; ++w2) l += (sm->m_w[w2][tid] == -INFINITY) ? 0.f : __expf(sm->m_w[w2][tid] - mx) * sm->l_w[w2][tid];
        sm->m_s[tid] = mx; sm->l_s[tid] = l;
    }
    att_sync<MEGA>();
    const int slice = (r * HD + nsp - 1) / nsp;
    namespace cgn = cooperative_groups;
    if (cmerge) asm volatile("barrier.cluster.wait.aligned;\n" ::: "memory");             // every peer is running
    for (int i = tid; i < r * HD; i += ATT_THREADS) {
        const int h = i / HD, d = i % HD;
        const float mx = sm->m_s[h];
        float ov = 0.f;
#pragma unroll
        for (int w2 = 0; w2 < WARPS; ++w2)
            ov += (sm->m_w[w2][h] == -INFINITY) ? 0.f : __expf(sm->m_w[w2][h] - mx) * o_w[w2][h][d];
        const int hq = kvh * r + h;
        if (nsp == 1) {
            store_out(a, row, hq * HD + d, ov / sm->l_s[h]);
        } else if (cmerge) {
            if (!MEGA) {
                cgn::cluster_group cluster = cgn::this_cluster();
                const int owner = i / slice;
                cluster.map_shared_rank(cl->rv_o, owner)[split * slice + (i - owner * slice)] = ov;
            }
        } else {
            a.part_o[(((size_t)row * a.Hq + hq) * nsp + split) * HD + d] = ov;
        }
    }
    if (nsp == 1) { if (!MEGA) trace_mark(3 * 4 + 2); return; }
    if (cmerge) {
        if (!MEGA) {
            cgn::cluster_group cluster = cgn::this_cluster();
            if (tid < r * nsp) {
                const int h = tid / nsp, dst = tid % nsp;
                float* ml = &cluster.map_shared_rank(cl->rv_ml, dst)[split][h][0];
                ml[0] = sm->m_s[h];
                ml[1] = sm->l_s[h];
            }
            cluster.sync();                           // release the pushes / acquire the peers'
            const int total = r * HD;
            for (int e = tid; e < slice; e += ATT_THREADS) {
                const int i = split * slice + e;
                if (i >= total) break;
                const int h = i / HD, d = i % HD;
                float mx = -INFINITY;
                for (int s2 = 0; s2 < nsp; ++s2) mx = fmaxf(mx, cl->rv_ml[s2][h][0]);
                float num = 0.f, den = 0.f;
                for (int s2 = 0; s2 < nsp; ++s2) {
                    const float l2 = cl->rv_ml[s2][h][1];
                    const float f = (l2 > 0.f) ? __expf(cl->rv_ml[s2][h][0] - mx) : 0.f;
                    den += f * l2;
                    num += f * cl->rv_o[s2 * slice + e];
                }
                store_out(a, row, (kvh * r + h) * HD + d, num / den);
            }
            trace_mark(3 * 4 + 2);
        }
        return;
    }
    if (tid < r) {
        const int hq = kvh * r + tid;
        float* ml = a.part_ml + (((size_t)row * a.Hq + hq) * nsp + split) * 2;
        ml[0] = sm->m_s[tid];
        ml[1] = sm->l_s[tid];
    }
    __threadfence();
    att_sync<MEGA>();
    if (tid == 0) {
        int prev = atomicAdd(&a.counters[row * a.Hkv + kvh], 1);
        sm->last_s = (prev == nsp - 1);
    }
    att_sync<MEGA>();
    if (!sm->last_s) return;
    __threadfence();
    // ---- merge: this unit arrived last for (row, kvh) -----------------------------------------
    // warp w computes the normalised weight of every split for heads w, w+8 (lanes = splits) ...
    float* wgt = &o_w[0][0][0];                       // [r][nsp] (o_w is free again: everyone passed the barrier above)
    for (int h = warp; h < r; h += ATT_THREADS / 32) {
        const int hq = kvh * r + h;
        const float* ml = a.part_ml + ((size_t)row * a.Hq + hq) * nsp * 2;
        float mv[2], lv[2];
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            const int s2 = lane + 32 * u;
            mv[u] = (s2 < nsp) ? __ldcg(ml + 2 * s2) : -INFINITY;
            lv[u] = (s2 < nsp) ? __ldcg(ml + 2 * s2 + 1) : 0.f;
        }
        const float mx = warp_max(fmaxf(mv[0], mv[1]));
        float f[2];
#pragma unroll
        for (int u = 0; u < 2; ++u) f[u] = (lv[u] > 0.f) ? __expf(mv[u] - mx) : 0.f;
        const float den = warp_sum(f[0] * lv[0] + f[1] * lv[1]);
#pragma unroll
        for (int u = 0; u < 2; ++u)
            if (lane + 32 * u < nsp) wgt[h * nsp + lane + 32 * u] = f[u] / den;
    }
    att_sync<MEGA>();
    // ... then every thread combines its output columns (independent loads)
    for (int i = tid; i < r * HD; i += ATT_THREADS) {
        const int h = i / HD, d = i % HD;
        const int hq = kvh * r + h;
        const float* po = a.part_o + ((size_t)row * a.Hq + hq) * nsp * HD + d;
        float num = 0.f;
#pragma unroll 4
        for (int s2 = 0; s2 < nsp; ++s2) num += wgt[h * nsp + s2] * __ldcg(po + (size_t)s2 * HD);
        store_out(a, row, hq * HD + d, num);
    }
    if (tid == 0) a.counters[row * a.Hkv + kvh] = 0;
    if (!MEGA) trace_mark(3 * 4 + 2);
}

}  // namespace sagc
