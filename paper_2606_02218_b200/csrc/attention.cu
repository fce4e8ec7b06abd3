// attention.cu -- standalone launch of the paged GQA attention unit (attention_body.cuh): one CTA per
// (activation row, kv head, K-split).  Serves prefill (every prompt position is a row with ctx = position + 1),
// head_dim 32, decode steps with more than 64 live rows and the sagc_debug_attention parity entry; decode steps
// with <= 64 live rows run the same unit inside the persistent decode-step kernel (decode_step.cu).
#include <cstdlib>
#include "attention_body.cuh"

namespace sagc {

template <int HD>
struct AttStandalone {       // 8 compute warps x 16 tokens per tile; K/V tiles in flight: NSTAGE - 1 (<= ~100 KB per CTA)
    static constexpr int WARPS = 8;
    static constexpr int NSTAGE = HD >= 128 ? 2 : (HD >= 64 ? 3 : 6);
    using G = AttGeom<HD, WARPS, NSTAGE>;
};

template <int HD, int WARPS, int NSTAGE>
__global__ void __launch_bounds__(ATT_THREADS) k_attention(AttnArgs a) {
    extern __shared__ __align__(128) unsigned char kv_s[];
    __shared__ AttSmall sm;
    __shared__ AttCluster<HD> cl;
    trace_mark(12);
    // Decode (a.prefetch): the live list, contexts, page table and every cached position but the
    // newest were written by EARLIER steps, so they may be read before the upstream kernel (this
    // step's RoPE / KV append) has finished.  Prefill rows attend to positions appended by that very
    // kernel and must wait first.
    if (!a.prefetch) pdl_wait();
    const int M = a.m_dev ? min(*a.m_dev, a.m_max) : a.m_max;
    const int row = blockIdx.x, kvh = blockIdx.y, split = blockIdx.z;
    if (row >= M) { if (a.prefetch) pdl_wait(); pdl_launch(); return; }      // uniform over the cluster (same row)
    attention_unit<HD, WARPS, NSTAGE, false>(a, row, kvh, split, a.n_splits, kv_s, &sm, &cl, (int)threadIdx.x);
}

template <int HD, int WARPS, int NSTAGE>
static int launch_att_geom(const AttnArgs& a, cudaStream_t st) {
    constexpr int RING = AttGeom<HD, WARPS, NSTAGE>::BYTES;
    // Decode: ask for at least 114 KB, so that the CTAs of the NEXT kernel (the O projection, 113 KB each, launched early by
    // PDL) cannot become resident beside an attention CTA.  Co-resident successors fill their weight ring early, but they take
    // issue slots and shared-memory bandwidth from the kernel on the critical path: measured on one box, 0.5B shape, FULL / MID /
    // TAIL ms per step 1.098 / 0.945 / 0.876 with the bare 96 KB ring, 1.057 / 0.927 / 0.871 with 114 KB (120 KB: the same).
    // (Round 1's kernel had 25 KB of static shared memory on top of the ring and was never co-resident; the refactoring of round 2
    // that overlaid those buffers on the ring cost 3.7 % of FULL until this was found.)
    static const int pad_kb = [] { const char* e = getenv("SAGC_ATT_PAD_KB"); return e ? atoi(e) : 114; }();
    const int BYTES = (a.prefetch && RING < pad_kb * 1024) ? pad_kb * 1024 : RING;
    if (cudaFuncSetAttribute(k_attention<HD, WARPS, NSTAGE>, cudaFuncAttributeMaxDynamicSharedMemorySize, BYTES > RING ? BYTES : RING) != cudaSuccess) return -1;
    dim3 grid(a.m_max, a.Hkv, a.n_splits);
    if (a.n_splits > 1 && a.n_splits <= 8) {      // 2..8 splits merge inside a cluster through DSMEM
        AttnArgs ac = a;
        ac.cluster_merge = 1;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = grid; cfg.blockDim = dim3(ATT_THREADS); cfg.dynamicSmemBytes = BYTES; cfg.stream = st;
        cudaLaunchAttribute at[2];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = 1; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = a.n_splits;
        at[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[1].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = at; cfg.numAttrs = g_pdl_all ? 2 : 1;
        return cudaLaunchKernelEx(&cfg, k_attention<HD, WARPS, NSTAGE>, ac) == cudaSuccess ? 1 : -1;
    }
    return launch_pdl(k_attention<HD, WARPS, NSTAGE>, grid, dim3(ATT_THREADS), BYTES, st, g_pdl_all, a) == cudaSuccess ? 1 : -1;
}

template <int HD>
static int launch_att(const AttnArgs& a, cudaStream_t st) {
    // other staging geometries (64-token tiles x 3 / 4 stages, 128-token tiles x 3 / 6 stages = 192 KB) were measured
    // with this launcher and changed nothing: the kernel is bound by issue latency at 2 warps per scheduler, not by
    // bytes in flight (profiles/r02_attention.md)
    return launch_att_geom<HD, AttStandalone<HD>::WARPS, AttStandalone<HD>::NSTAGE>(a, st);
}

int launch_attention(const AttnArgs& a, cudaStream_t st) {
    if (a.m_max <= 0) return 0;
    if (a.hd == 128) return launch_att<128>(a, st);
    if (a.hd == 64) return launch_att<64>(a, st);
    if (a.hd == 32) return launch_att<32>(a, st);
    return -1;
}

}  // namespace sagc
