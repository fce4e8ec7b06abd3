// attention_tc.cu -- paged GQA decode attention (step a7) on the 5th-generation tensor cores: the decode-step
// attention of head_dim 64 / 128 models.  One CTA per (activation row, kv head, K-split), 320 threads:
//
//   warp 0     TMA producer: per 128-token tile, one cp.async.bulk.tensor box per (page, K|V, 64-wide half of the
//              head) of the paged pool -- the pool of a layer is a 2-D tensor [n_pages * 2 * Hkv * page][hd], so a
//              (page, K|V, kv head) slab is `page` consecutive rows -- into an NSTAGE ring, 128-byte swizzled.
//   warp 1     tcgen05.mma issuer (one lane).  Per tile, with fp32 accumulators in tensor memory:
//                S^T[token][n] = K[token][:] . Q[n][:]         A = K tile (K-major), B = Q (16 rows: heads hi | lo)
//                O^T[d][n]    += V[token][d] . P[n][token]     A = V tile (MN-major: the tile IS V^T for the MMA),
//                                                              B = P (16 rows: heads hi | lo, K-major over tokens)
//              S of tile i+1 is issued before P.V of tile i, so the softmax of a tile overlaps both neighbours.
//   warps 2-9  two softmax warpgroups on alternate tiles (own S / P buffers and O accumulator, joined at the end by the
//              log-sum-exp rule): thread = token (TMEM lane).  It reads its 16 S columns (tcgen05.ld), adds the hi and lo
//              column of each head, takes the tile maximum per head over the 128 tokens (redux.sync on order-preserving
//              integers + one 128-thread named barrier), exponentiates, accumulates its share of the row sums and
//              writes p as bf16 hi + lo into the swizzled P operand.  The running maximum is LAZY: it moves (and O in
//              tensor memory is rescaled, one tcgen05.ld/st round trip) only when a tile exceeds it by more than 8,
//              so p <= e^8 and the exact softmax is recovered by the final division (m and l stay consistent).
//
// Precision is the register-HMMA unit's (attention_body.cuh): K, V exact bf16; q and p as hi + lo bf16 pairs
// (~16 mantissa bits); fp32 accumulation.  Split-K partials (o, m, l) merge through the L2 scratch by the last unit
// to arrive (all 320 threads of that CTA), with the arithmetic of attention_body.cuh.  Decode (fuse_rope): RoPE of q / k and the bf16 K,V append
// of the newest position happen here; the split that owns that position appends BEFORE its producer fetches the
// last tile (generic -> async proxy fence + mbarrier), so no shared-memory patching is needed.
// Masked positions: p = 0 exactly, and the pool is finite everywhere (zeroed at creation), so stale V rows of a
// partially filled last page contribute 0 * finite = 0.
#include "attention_body.cuh"
#include "tc_ptx.cuh"

namespace sagc {

static constexpr int ATC_THREADS = 320;       // TMA warp, MMA warp, two softmax warpgroups
static constexpr int ATC_TILE = 128;
static constexpr float ATC_LAZY = 8.0f;

template <int HD>
struct AttTc {
    static constexpr int HALVES = HD / 64;
    static constexpr int HALF_BYTES = ATC_TILE * 128;               // [128 tokens][64 bf16]
    static constexpr int KV_BYTES = 2 * HALVES * HALF_BYTES;        // V halves, then K halves
    static constexpr int MAXSTAGE = HD == 128 ? 3 : 6;              // 192 KB of K/V in flight
    static constexpr int Q_BYTES = HALVES * 16 * 128;               // [half][16 rows][64 bf16]
    static constexpr int P_BYTES = 2 * 16 * 128;                    // [token half][16 rows][64 tokens]
    static constexpr int tail_bytes() { return Q_BYTES + 4 * P_BYTES; }      // Q and the 2 x 2 P buffers follow the ring
};

struct AtcSmall {
    uint64_t kv_full[8], kv_empty[8], s_full[4], p_full[4], p_free[4], q_ready, app_done, o_done;      // [4] = [warpgroup][buffer]
    uint32_t tmem_slot;
    int last_s;
    float mt_s[4][4][8];            // [2 * warpgroup + buffer][warp][head]: per-warp tile maxima
    float l_s[2][4][8];
    float xm[8], xl[8];             // warpgroup 1 -> 0: its running maximum and row sum per head
    float wgt[ATT_MAXR * 64];       // split merge weights [r][nst]
    int pg_s[ATT_MAXPG];
};

__device__ __forceinline__ void tc_ld16(uint32_t taddr, float (&v)[16]) {
    uint32_t r[16];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];\n"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr));
    asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory");
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ void tc_st16(uint32_t taddr, const float (&v)[16]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};\n" ::
            "r"(taddr), "r"(__float_as_uint(v[0])), "r"(__float_as_uint(v[1])), "r"(__float_as_uint(v[2])), "r"(__float_as_uint(v[3])),
        "r"(__float_as_uint(v[4])), "r"(__float_as_uint(v[5])), "r"(__float_as_uint(v[6])), "r"(__float_as_uint(v[7])),
        "r"(__float_as_uint(v[8])), "r"(__float_as_uint(v[9])), "r"(__float_as_uint(v[10])), "r"(__float_as_uint(v[11])),
        "r"(__float_as_uint(v[12])), "r"(__float_as_uint(v[13])), "r"(__float_as_uint(v[14])), "r"(__float_as_uint(v[15]))
        : "memory");
    asm volatile("tcgen05.wait::st.sync.aligned;\n" ::: "memory");
}
// MN-major, 128-byte-swizzled operand (the V tile read as V^T): 64 contiguous M elements per 128-byte row, the next
// 64 at LBO; 8 K rows (tokens) per 1024-byte atom, the next 8 at SBO = 1024
__device__ __forceinline__ uint64_t umma_desc_mn_sw128(uint32_t smem_addr, uint32_t lbo_bytes) {
    uint64_t d = 0;
    d |= (uint64_t)((smem_addr & 0x3ffff) >> 4);
    d |= (uint64_t)((lbo_bytes >> 4) & 0x3fff) << 16;
    d |= (uint64_t)(1024 >> 4) << 32;
    d |= (uint64_t)1 << 46;
    d |= (uint64_t)2 << 61;
    return d;
}
// max over the warp of a float through redux.sync on an order-preserving integer image
__device__ __forceinline__ float warp_max_redux(float x) {
    int b = __float_as_int(x);
    b = b >= 0 ? b : b ^ 0x7fffffff;
    b = __reduce_max_sync(0xffffffffu, b);
    b = b >= 0 ? b : b ^ 0x7fffffff;
    return __int_as_float(b);
}
// Warp-converged issue: the TMA and MMA warps run their loops with all 32 lanes (uniform control flow, operands in
// uniform registers) and one elected lane executes the instruction.  Issuing from inside an `if (lane == 0)` region
// makes the compiler wrap every UTCHMMA / UTMALDG in an ELECT / R2UR / BRA.U.ANY loop: ~85 cycles per MMA measured.
__device__ __forceinline__ void tc_mma_e(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accum) {
    asm volatile(
        "{\n"
        ".reg .pred p, pe;\n"
        "elect.sync _|pe, 0xffffffff;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "@pe tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n"
        "}\n" ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accum)
        : "memory");
}
__device__ __forceinline__ void tc_commit_e(uint64_t* bar) {
    asm volatile(
        "{\n"
        ".reg .pred pe;\n"
        "elect.sync _|pe, 0xffffffff;\n"
        "@pe tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n"
        "}\n" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx_e(uint64_t* bar, uint32_t bytes) {
    asm volatile(
        "{\n"
        ".reg .pred pe;\n"
        "elect.sync _|pe, 0xffffffff;\n"
        "@pe mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_load_2d_e(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1) {
    asm volatile(
        "{\n"
        ".reg .pred pe;\n"
        "elect.sync _|pe, 0xffffffff;\n"
        "@pe cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];\n"
        "}\n" ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1)
        : "memory");
}

// non-blocking probe of a phase parity (mbarrier.try_wait may suspend the thread up to a time limit: not for polling two queues)
__device__ __forceinline__ bool mbar_test(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n" : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return ok != 0;
}

#ifdef SAGC_ATT_TIMELINE
#define ATC_MARK(role, tile, ev)                                                                                   \
    do {                                                                                                           \
        if (a.dbg != nullptr && blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0 && (tile) < 64)              \
            a.dbg[((role) * 64 + (tile)) * 8 + (ev)] = clock64();                                                  \
    } while (0)
#else
#define ATC_MARK(role, tile, ev) ((void)0)
#endif
__device__ __forceinline__ void bar_softmax(int wg) { asm volatile("bar.sync %0, 128;\n" ::"r"(1 + wg) : "memory"); }

template <int HD>
__global__ void __launch_bounds__(ATC_THREADS, 1) k_attention_tc(const __grid_constant__ CUtensorMap kvmap, AttnArgs a, int NS) {
    using C = AttTc<HD>;
    extern __shared__ unsigned char smem_raw[];
    unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    unsigned char* q_s = smem + (size_t)NS * C::KV_BYTES;
    unsigned char* p_s = q_s + C::Q_BYTES;
    AtcSmall* sm = reinterpret_cast<AtcSmall*>(p_s + 4 * C::P_BYTES);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    // decode (a.prefetch): the live list, contexts, page table and every cached position but the newest predate the
    // upstream kernel (this step's QKV projection); only q and the new k, v must wait for it
    if (!a.prefetch) pdl_wait();
    const int M = a.m_dev ? min(*a.m_dev, a.m_max) : a.m_max;
    const int row = blockIdx.x, kvh = blockIdx.y, split = blockIdx.z, nsp = a.n_splits;
    if (row >= M) { if (a.prefetch) pdl_wait(); pdl_launch(); return; }
    const int r = a.Hq / a.Hkv;
    const int ctx = a.row_ctx[row];
    const int sid = a.row_sid[row];
    const int* pt = a.page_table + (size_t)sid * a.max_blocks;
    int cps = (ctx + nsp - 1) / nsp;
    cps = ((cps + ATC_TILE - 1) / ATC_TILE) * ATC_TILE;
    const int t_begin = split * cps;
    const int t_end = min(ctx, t_begin + cps);
    const int n_tiles = t_end > t_begin ? (t_end - t_begin + ATC_TILE - 1) / ATC_TILE : 0;
    const int pshift = 31 - __clz(a.page), pmask = a.page - 1;
    const int b_begin = t_begin >> pshift;
    const int last_blk = n_tiles > 0 ? ((t_end - 1) >> pshift) : b_begin;
    const int n_blk = n_tiles > 0 ? last_blk - b_begin + 1 : 0;
    const bool pg_cached = n_blk <= ATT_MAXPG;
    const bool fuse = a.fuse_rope != 0;
    const bool designated = fuse && n_tiles > 0 && t_end == ctx;      // this split holds the newest position

    if (tid == 0) {
        for (int s = 0; s < NS; ++s) { mbar_init(&sm->kv_full[s], 1); mbar_init(&sm->kv_empty[s], 1); }
        for (int b = 0; b < 4; ++b) { mbar_init(&sm->s_full[b], 1); mbar_init(&sm->p_full[b], 4); mbar_init(&sm->p_free[b], 1); }
        mbar_init(&sm->q_ready, 4); mbar_init(&sm->app_done, 4); mbar_init(&sm->o_done, 1);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
        sm->last_s = 0;
        tma_prefetch_desc(&kvmap);
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" ::"r"(smem_u32(&sm->tmem_slot)), "n"(128));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n");
    }
    if (pg_cached)
        for (int b = tid; b < n_blk; b += ATC_THREADS) sm->pg_s[b] = pt[b_begin + b];
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = sm->tmem_slot;
    if (tid == 0) ATC_MARK(0, 63, 0);
    // tensor memory columns: S^T of (warpgroup g, buffer b) at 16 * (2g + b); O^T of warpgroup g at 64 + 16 g
    // tile i belongs to warpgroup i & 1; it is that warpgroup's tile j = i >> 1 and uses its buffer j & 1

    if (warp == 0) {
        // ===== TMA producer =====================================================================
        if (n_tiles > 0) {                                       // all 32 lanes, converged
            const int ppt = ATC_TILE >> pshift;                  // pages per tile
            const uint32_t box_bytes = (uint32_t)a.page * 128u;
            for (int i = 0; i < n_tiles; ++i) {
                const int s = i % NS, k = i / NS;
                mbar_wait(&sm->kv_empty[s], (uint32_t)((k & 1) ^ 1));
                if (designated && i == n_tiles - 1) mbar_wait(&sm->app_done, 0);      // the new K,V row is in the pool
                if (lane == 0) ATC_MARK(0, i, 0);
                mbar_expect_tx_e(&sm->kv_full[s], (uint32_t)C::KV_BYTES);
                unsigned char* st = smem + (size_t)s * C::KV_BYTES;
                const int blk0 = (t_begin + i * ATC_TILE) >> pshift;
                for (int p0 = 0; p0 < ppt; p0 += 2) {            // two pages at a time: their page ids and rows first, then the copies
                    int row_v[2];
#pragma unroll
                    for (int u = 0; u < 2; ++u) {
                        const int blk = min(blk0 + p0 + u, last_blk);      // past the context: any finite page (masked, p = 0)
                        int pg = pg_cached ? sm->pg_s[blk - b_begin] : pt[blk];
                        if (pg < 0) pg = 0;                                // unmapped block after a pool-exhaustion error
                        row_v[u] = ((pg * 2 + 1) * a.Hkv + kvh) * a.page;
                    }
                    const int k_off = a.Hkv * a.page;                      // the K slab sits Hkv slabs before the V slab
#pragma unroll
                    for (int u = 0; u < 2; ++u) {
                        if (p0 + u >= ppt) break;
                        unsigned char* dst = st + (size_t)(p0 + u) * box_bytes;
#pragma unroll
                        for (int h = 0; h < C::HALVES; ++h) {
                            tma_load_2d_e(dst + (size_t)h * C::HALF_BYTES, &kvmap, &sm->kv_full[s], h * 64, row_v[u]);
                            tma_load_2d_e(dst + (size_t)(C::HALVES + h) * C::HALF_BYTES, &kvmap, &sm->kv_full[s], h * 64, row_v[u] - k_off);
                        }
                    }
                }
                if (lane == 0) ATC_MARK(0, i, 1);
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer =======================================================================
        if (n_tiles > 0) {                                       // all 32 lanes, converged
            const uint32_t idesc_s = umma_idesc(16);                        // S^T: M = 128 tokens, N = 16, A and B K-major
            const uint32_t idesc_o = umma_idesc(16) | (1u << 15);           // O^T: M = 128 (d), N = 16, A MN-major
            const uint32_t q_a = smem_u32(q_s), p_a = smem_u32(p_s);
            mbar_wait(&sm->q_ready, 0);
            tc_fence_after();
            const uint64_t dq0 = umma_desc_sw128(q_a);
            // Two independent queues served by whichever is ready (a blocking wait on one would hold the other up and,
            // through the K/V ring, starve itself): S of tile is (needs its K/V tile and a free S buffer: S of tile
            // is - 4 has been consumed once p_full of that tile was seen), P.V of tile ip (needs that tile's P).
            int is = 0, ip = 0;
            while (ip < n_tiles) {
                bool idle = true;
                if (is < n_tiles && is < ip + 4) {
                    const int s = is % NS;
                    if (__any_sync(0xffffffffu, mbar_test(&sm->kv_full[s], (uint32_t)((is / NS) & 1)))) {
                        if (lane == 0) ATC_MARK(1, is, 1);
                        tc_fence_after();
                        // one descriptor per operand tile; a k step only advances the start-address field (bytes >> 4), which
                        // cannot carry out of its 14 bits here (every tile lies inside the 227 KB window, 16-byte aligned)
                        const uint64_t da0 = umma_desc_sw128(smem_u32(smem + (size_t)s * C::KV_BYTES + (size_t)C::HALVES * C::HALF_BYTES));
                        const int sb = 2 * (is & 1) + ((is >> 1) & 1);
                        const uint32_t d_s = tmem_base + 16 * sb;
#pragma unroll
                        for (int ks = 0; ks < HD / 16; ++ks)
                            tc_mma_e(d_s, da0 + (uint64_t)(((ks >> 2) * C::HALF_BYTES + (ks & 3) * 32) >> 4),
                                     dq0 + (uint64_t)(((ks >> 2) * 2048 + (ks & 3) * 32) >> 4), idesc_s, ks > 0 ? 1u : 0u);
                        tc_commit_e(&sm->s_full[sb]);
                        if (lane == 0) ATC_MARK(1, is, 2);
                        ++is;
                        idle = false;
                    }
                }
                if (ip < is) {
                    const int g = ip & 1, j = ip >> 1, pb = 2 * g + (j & 1), s = ip % NS;
                    if (__any_sync(0xffffffffu, mbar_test(&sm->p_full[pb], (uint32_t)((j >> 1) & 1)))) {
                        if (lane == 0) ATC_MARK(1, ip, 3);
                        tc_fence_after();
                        const uint64_t dv0 = umma_desc_mn_sw128(smem_u32(smem + (size_t)s * C::KV_BYTES), C::HALF_BYTES);
                        const uint64_t dp0 = umma_desc_sw128(p_a + pb * C::P_BYTES);
                        const uint32_t d_o = tmem_base + 64 + 16 * g;
#pragma unroll
                        for (int ks = 0; ks < ATC_TILE / 16; ++ks)
                            tc_mma_e(d_o, dv0 + (uint64_t)((ks * 2048) >> 4), dp0 + (uint64_t)(((ks >> 2) * 2048 + (ks & 3) * 32) >> 4), idesc_o,
                                     (j > 0 || ks > 0) ? 1u : 0u);
                        tc_commit_e(&sm->kv_empty[s]);
                        tc_commit_e(&sm->p_free[pb]);
                        if (lane == 0) ATC_MARK(1, ip, 4);
                        ++ip;
                        idle = false;
                    }
                }
                if (idle) __nanosleep(32);         // leave the issue slots of this scheduler to the softmax warps
            }
            tc_commit_e(&sm->o_done);
        }
    } else {
        // ===== softmax warps: thread = token lane of S^T, = output column d of O^T ================
        const int wg = (warp - 2) >> 2;                   // warpgroup 0 takes the even tiles, 1 the odd ones
        const int st = (tid - 64) & 127;                  // 0..127 inside the warpgroup
        const int sw = (warp - 2) & 3;                    // slot in the per-warp scratch
        const int quad = warp & 3;                        // TMEM lane quadrant this warp may access
        const int tl = quad * 32 + lane;                  // token inside the tile / d inside the head
        const uint32_t lane_off = (uint32_t)(quad * 32) << 16;
        // ---- q: RoPE, 1/sqrt(hd), hi / lo split into the swizzled B operand; append of the new k, v ----
        if (a.prefetch) pdl_wait();
        pdl_launch();
        if (wg == 0) {
            constexpr int CH = HD / 8;                    // 16-byte chunks per head row
            const int h = st / CH, c = st % CH;
            if (h < 8) {
                float x[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) x[e] = 0.f;
                if (h < r && n_tiles > 0) {
                    const float rs = a.q_fx != nullptr ? __ldcg(a.q_rstd + row) : 1.f;
                    const size_t qcol = (size_t)(kvh * r + h) * HD;
                    att_load8(a, row, qcol + 8 * c, rs, x);
                    if (fuse) {
                        float xp[8];
                        att_load8(a, row, qcol + 8 * (c ^ (CH / 2)), rs, xp);
                        const int pos = a.row_pos[row];
                        const float2* cs = reinterpret_cast<const float2*>(a.rope_cs) + (size_t)pos * (HD / 2) + (c % (CH / 2)) * 8;
                        const float sgn = c < CH / 2 ? -1.f : 1.f;
#pragma unroll
                        for (int e = 0; e < 8; ++e) { const float2 w = cs[e]; x[e] = x[e] * w.x + sgn * xp[e] * w.y; }
                    }
                }
                const float scale = rsqrtf((float)HD);
                uint32_t hi[4], lo[4];
#pragma unroll
                for (int e = 0; e < 4; ++e) split2(x[2 * e] * scale, x[2 * e + 1] * scale, hi[e], lo[e]);
                const int half = c >> 3, cc = c & 7;
                unsigned char* qh = q_s + half * 2048;
                *reinterpret_cast<uint4*>(qh + h * 128 + ((cc ^ (h & 7)) << 4)) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
                *reinterpret_cast<uint4*>(qh + (8 + h) * 128 + ((cc ^ (h & 7)) << 4)) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
            }
            asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
            __syncwarp();
            if (lane == 0) mbar_arrive(&sm->q_ready);
            if (designated) {
                const int tnew = ctx - 1, pos = a.row_pos[row];
                const int blk = tnew >> pshift;
                const int pg = pg_cached ? sm->pg_s[blk - b_begin] : pt[blk];
                if (pg >= 0) {
                    const float rs = a.q_fx != nullptr ? __ldcg(a.q_rstd + row) : 1.f;
                    const size_t head_stride = (size_t)a.page * HD;
                    const size_t kcol = (size_t)a.Hq * HD + (size_t)kvh * HD;
                    const size_t vcol = kcol + (size_t)a.Hkv * HD;
                    bf16_t* kd = a.kv_layer_w + ((size_t)pg * 2 * a.Hkv + kvh) * head_stride + (size_t)(tnew & pmask) * HD;
                    bf16_t* vd = kd + (size_t)a.Hkv * head_stride;
                    if (st < HD / 2) {
                        const float2 w = *reinterpret_cast<const float2*>(a.rope_cs + ((size_t)pos * (HD / 2) + st) * 2);
                        const float k0 = att_load1(a, row, kcol + st, rs), k1 = att_load1(a, row, kcol + st + HD / 2, rs);
                        kd[st] = (bf16_t)f32_to_bf16_bits(k0 * w.x - k1 * w.y);
                        kd[st + HD / 2] = (bf16_t)f32_to_bf16_bits(k1 * w.x + k0 * w.y);
                    }
                    if (st < HD) vd[st] = (bf16_t)f32_to_bf16_bits(att_load1(a, row, vcol + st, rs));
                }
                __threadfence();
                asm volatile("fence.proxy.async;\n" ::: "memory");      // generic-proxy global writes -> the TMA read of the last tile
                __syncwarp();
                if (lane == 0) mbar_arrive(&sm->app_done);
            }
        }
        // ---- tiles --------------------------------------------------------------------------------
        float m_used[8], l_part[8];
#pragma unroll
        for (int h = 0; h < 8; ++h) { m_used[h] = -INFINITY; l_part[h] = 0.f; }
        const uint32_t tm_o = tmem_base + 64 + 16 * wg;
        for (int i = wg; i < n_tiles; i += 2) {
            const int j = i >> 1, b = 2 * wg + (j & 1), k = j >> 1;
            if (st == 0) ATC_MARK(2 + wg, i, 0);
            mbar_wait(&sm->s_full[b], (uint32_t)(k & 1));
            if (st == 0) ATC_MARK(2 + wg, i, 1);
            tc_fence_after();
            float sv[16];
            tc_ld16(tmem_base + 16 * b + lane_off, sv);
            float s[8];
            const bool valid = t_begin + i * ATC_TILE + tl < t_end;
#pragma unroll
            for (int h = 0; h < 8; ++h) s[h] = valid ? sv[h] + sv[8 + h] : -INFINITY;
            {   // tile maximum per head over the 128 tokens
                float wm[8];
#pragma unroll
                for (int h = 0; h < 8; ++h) wm[h] = warp_max_redux(s[h]);
                if (lane == 0) {
                    *reinterpret_cast<float4*>(&sm->mt_s[b][sw][0]) = make_float4(wm[0], wm[1], wm[2], wm[3]);
                    *reinterpret_cast<float4*>(&sm->mt_s[b][sw][4]) = make_float4(wm[4], wm[5], wm[6], wm[7]);
                }
            }
            if (st == 0) ATC_MARK(2 + wg, i, 2);
            bar_softmax(wg);
            if (st == 0) ATC_MARK(2 + wg, i, 3);
            float mt[8];
            bool need = false;
#pragma unroll
            for (int h = 0; h < 8; ++h) {
                mt[h] = fmaxf(fmaxf(sm->mt_s[b][0][h], sm->mt_s[b][1][h]), fmaxf(sm->mt_s[b][2][h], sm->mt_s[b][3][h]));
                need |= mt[h] > m_used[h] + ATC_LAZY;         // also true on the first tile (m_used = -inf)
            }
            if (need) {                                       // uniform over the 128 threads
                float f[8];
#pragma unroll
                for (int h = 0; h < 8; ++h) {
                    const float mn = fmaxf(m_used[h], mt[h]);
                    f[h] = (m_used[h] == -INFINITY) ? 0.f : __expf(m_used[h] - mn);
                    m_used[h] = mn;
                    l_part[h] *= f[h];
                }
                if (j > 0) {                                  // O holds this warpgroup's earlier tiles once P.V of its tile j-1 has completed
                    mbar_wait(&sm->p_free[2 * wg + ((j - 1) & 1)], (uint32_t)(((j - 1) >> 1) & 1));
                    tc_fence_after();
                    float ov[16];
                    tc_ld16(tm_o + lane_off, ov);
#pragma unroll
                    for (int c = 0; c < 16; ++c) ov[c] *= f[c & 7];
                    tc_st16(tm_o + lane_off, ov);
                }
            }
            uint32_t ph[8], pl[8];
#pragma unroll
            for (int h = 0; h < 8; ++h) {
                const float p = __expf(s[h] - m_used[h]);     // masked tokens / padded heads of an all-masked column: exp(-inf) = 0
                l_part[h] += p;
                ph[h] = f32_to_bf16_bits(p);
                pl[h] = f32_to_bf16_bits(p - __uint_as_float(ph[h] << 16));
            }
            if (st == 0) ATC_MARK(2 + wg, i, 4);
            mbar_wait(&sm->p_free[b], (uint32_t)((k & 1) ^ 1));      // P.V of this warpgroup's tile j-2 has read this buffer
            if (st == 0) ATC_MARK(2 + wg, i, 5);
            {
                unsigned char* pb = p_s + b * C::P_BYTES + (tl >> 6) * 2048 + (tl & 7) * 2;
                const int ch = (tl & 63) >> 3;
#pragma unroll
                for (int h = 0; h < 8; ++h) {
                    *reinterpret_cast<bf16_t*>(pb + h * 128 + ((ch ^ h) << 4)) = (bf16_t)ph[h];
                    *reinterpret_cast<bf16_t*>(pb + (8 + h) * 128 + ((ch ^ h) << 4)) = (bf16_t)pl[h];
                }
            }
            asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(&sm->p_full[b]);
            if (st == 0) ATC_MARK(2 + wg, i, 6);
        }
        // ---- epilogue: O^T columns h (hi) + 8+h (lo) of this thread's d; row sums over the 128 token lanes ----
        float ov[8], l[8];
        if (st == 0) ATC_MARK(2 + wg, 62, 0);
        if (n_tiles > 0) {
            mbar_wait(&sm->o_done, 0);            // every P.V has completed: both O accumulators are final, the P buffers free
            tc_fence_after();
        }
        if (n_tiles > wg) {
            float o16[16];
            tc_ld16(tm_o + lane_off, o16);
#pragma unroll
            for (int h = 0; h < 8; ++h) ov[h] = o16[h] + o16[8 + h];
        } else {
#pragma unroll
            for (int h = 0; h < 8; ++h) ov[h] = 0.f;
        }
#pragma unroll
        for (int h = 0; h < 8; ++h) l[h] = warp_sum(l_part[h]);
        if (lane == 0) {
            *reinterpret_cast<float4*>(&sm->l_s[wg][sw][0]) = make_float4(l[0], l[1], l[2], l[3]);
            *reinterpret_cast<float4*>(&sm->l_s[wg][sw][4]) = make_float4(l[4], l[5], l[6], l[7]);
        }
        bar_softmax(wg);
#pragma unroll
        for (int h = 0; h < 8; ++h) l[h] = (sm->l_s[wg][0][h] + sm->l_s[wg][1][h]) + (sm->l_s[wg][2][h] + sm->l_s[wg][3][h]);
        // ---- the odd tiles' (o, m, l) join the even tiles' (same log-sum-exp rule as the split merge) ----
        float* xo = reinterpret_cast<float*>(p_s);          // [8][128 d] (conflict-free for thread = d), overlays the P buffers
        if (wg == 1) {
#pragma unroll
            for (int h = 0; h < 8; ++h) xo[h * 128 + tl] = ov[h];
            if (st == 0) {
#pragma unroll
                for (int h = 0; h < 8; ++h) { sm->xm[h] = m_used[h]; sm->xl[h] = l[h]; }
            }
        }
        if (st == 0) ATC_MARK(2 + wg, 62, 1);
        asm volatile("bar.sync 3, 256;\n" ::: "memory");
        if (st == 0) ATC_MARK(2 + wg, 62, 2);
        if (wg == 0) {
#pragma unroll
        for (int h = 0; h < 8; ++h) {
            const float mb = sm->xm[h], mn = fmaxf(m_used[h], mb);
            const float fa = (m_used[h] == -INFINITY) ? 0.f : __expf(m_used[h] - mn);
            const float fb = (mb == -INFINITY) ? 0.f : __expf(mb - mn);
            ov[h] = ov[h] * fa + xo[h * 128 + tl] * fb;
            l[h] = l[h] * fa + sm->xl[h] * fb;
            m_used[h] = mn;
        }
        if (nsp == 1) {
            if (tl < HD) {
#pragma unroll
                for (int h = 0; h < 8; ++h)
                    if (h < r) store_out(a, row, (kvh * r + h) * HD + tl, ov[h] / l[h]);
            }
        } else {
            if (tl < HD) {
#pragma unroll
                for (int h = 0; h < 8; ++h)
                    if (h < r) a.part_o[(((size_t)row * a.Hq + kvh * r + h) * nsp + split) * HD + tl] = ov[h];
            }
#pragma unroll
            for (int h = 0; h < 8; ++h)
                if (st == h && h < r) {
                    float* ml = a.part_ml + (((size_t)row * a.Hq + kvh * r + h) * nsp + split) * 2;
                    ml[0] = m_used[h];
                    ml[1] = l[h];
                }
            if (st == 0) ATC_MARK(2, 62, 3);
            __threadfence();
            bar_softmax(0);
            if (st == 0) ATC_MARK(2, 62, 4);
            if (st == 0) {
                const int prev = atomicAdd(&a.counters[row * a.Hkv + kvh], 1);
                sm->last_s = (prev == nsp - 1);
            }
            bar_softmax(0);
            if (st == 0) ATC_MARK(2, 62, 5);
        }
        }   // warpgroup 0
    }
    // ---- merge by the unit that arrived last for (row, kv head): ALL 320 threads (the partials sit in L2, so the merge is a
    // chain of round trips: the more loads in flight the shorter); arithmetic of attention_body.cuh ----
    if (nsp > 1) __syncthreads();            // (nsp is uniform over the CTA; the unsplit path has nothing to merge)
    if (nsp > 1 && sm->last_s) {
        __threadfence();
        for (int h = warp; h < r; h += ATC_THREADS / 32) {
            const float* ml = a.part_ml + ((size_t)row * a.Hq + kvh * r + h) * nsp * 2;
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
                if (lane + 32 * u < nsp) sm->wgt[h * nsp + lane + 32 * u] = f[u] / den;
        }
        __syncthreads();
        const int n_out = r * HD;
        for (int i0 = tid; i0 < n_out; i0 += 2 * ATC_THREADS) {      // two outputs x 8 splits in flight per thread
            const int i1 = i0 + ATC_THREADS;
            const bool two = i1 < n_out;
            const int h0 = i0 / HD, d0 = i0 % HD, h1 = two ? i1 / HD : h0, d1 = two ? i1 % HD : d0;
            const float* po0 = a.part_o + ((size_t)row * a.Hq + kvh * r + h0) * nsp * HD + d0;
            const float* po1 = a.part_o + ((size_t)row * a.Hq + kvh * r + h1) * nsp * HD + d1;
            const float* w0 = sm->wgt + h0 * nsp;
            const float* w1 = sm->wgt + h1 * nsp;
            float n0 = 0.f, n1 = 0.f;
            for (int s0 = 0; s0 < nsp; s0 += 8) {
                float v0[8], v1[8];
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const int s2 = min(s0 + u, nsp - 1);
                    v0[u] = __ldcg(po0 + (size_t)s2 * HD);
                    v1[u] = __ldcg(po1 + (size_t)s2 * HD);
                }
#pragma unroll
                for (int u = 0; u < 8; ++u)
                    if (s0 + u < nsp) { n0 += w0[s0 + u] * v0[u]; n1 += w1[s0 + u] * v1[u]; }
            }
            store_out(a, row, (kvh * r + h0) * HD + d0, n0);
            if (two) store_out(a, row, (kvh * r + h1) * HD + d1, n1);
        }
        if (tid == 0) { ATC_MARK(2, 62, 6); a.counters[row * a.Hkv + kvh] = 0; }
    }
    tc_fence_before();
    __syncthreads();
    if (tid == 0) ATC_MARK(0, 63, 1);
    if (warp == 1) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(tmem_base), "n"(128));
}

template <int HD>
static int launch_att_tc(const AttnArgs& a, const TcMap* kvmap, int stages, cudaStream_t st) {
    using C = AttTc<HD>;
    auto smem_bytes = [](int ns) { return ns * C::KV_BYTES + C::tail_bytes() + (int)sizeof(AtcSmall) + 1024; };   // + slack for the 1024-byte alignment
    if (stages < 2) stages = 2;
    if (stages > C::MAXSTAGE) stages = C::MAXSTAGE;
    if (cudaFuncSetAttribute(k_attention_tc<HD>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes(C::MAXSTAGE)) != cudaSuccess) return -1;
    dim3 grid(a.m_max, a.Hkv, a.n_splits);
    return launch_pdl(k_attention_tc<HD>, grid, dim3(ATC_THREADS), (size_t)smem_bytes(stages), st, g_pdl_all,
                      *reinterpret_cast<const CUtensorMap*>(kvmap), a, stages) == cudaSuccess ? 1 : -1;
}

// the tcgen05 kernel serves head_dim 64 / 128 with 8 <= page <= 128 tokens (TMA box = one page x 64 elements)
bool attention_tc_supports(int hd, int page, int r) {
    return (hd == 64 || hd == 128) && page >= 8 && page <= 128 && (page & (page - 1)) == 0 && r >= 1 && r <= 8;
}
// tensor map of one layer's pool [n_pages][2][Hkv][page][hd] as the 2-D bf16 tensor [n_pages * 2 * Hkv * page][hd]
int attention_tc_make_map(TcMap* out, const void* kv_layer, long long n_pages, int Hkv, int page, int hd) {
    (void)hd;
    return tc_make_map(out, kv_layer, n_pages * 2 * Hkv * page, hd, page);
}
// stages = K/V tiles in the ring (2 .. 3 at head_dim 128, 2 .. 6 at 64; 0 = deepest): fewer stages let several CTAs share an SM
int launch_attention_tc(const AttnArgs& a, const TcMap* kvmap, int stages, cudaStream_t st) {
    if (a.m_max <= 0) return 0;
    if (!attention_tc_supports(a.hd, a.page, a.Hq / a.Hkv) || a.n_splits < 1 || a.n_splits > 64) return -1;
    if (stages <= 0) stages = 8;
    return a.hd == 128 ? launch_att_tc<128>(a, kvmap, stages, st) : launch_att_tc<64>(a, kvmap, stages, st);
}

}  // namespace sagc
