// common.cuh -- device helpers shared by the sm_100a kernels of the rollout hot path.
// (CUDA path only; the CPU oracle under oracle/ shares nothing with this tree.)
#pragma once
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stdint.h>

namespace sagc {

// ---- bf16 <-> fp32 (bit exact, RNE) -------------------------------------------------
__device__ __forceinline__ float bf16lo_to_f32(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf16hi_to_f32(uint32_t w) { return __uint_as_float(w & 0xffff0000u); }
__device__ __forceinline__ float bf16_to_f32(uint16_t b) { return __uint_as_float(((uint32_t)b) << 16); }

// round-to-nearest-even fp32 -> bf16 bits (finite inputs)
__device__ __forceinline__ uint32_t f32_to_bf16_bits(float x) {
    uint32_t u = __float_as_uint(x);
    return (u + 0x7fffu + ((u >> 16) & 1u)) >> 16;
}

// x = hi + lo with hi = bf16(x), lo = bf16(x - hi): ~16 mantissa bits carried into the MMA.
// pack2 puts element 0 in the low half (the MMA fragment convention).
__device__ __forceinline__ void split2(float x0, float x1, uint32_t& hi, uint32_t& lo) {
    uint32_t h0 = f32_to_bf16_bits(x0), h1 = f32_to_bf16_bits(x1);
    float r0 = x0 - __uint_as_float(h0 << 16), r1 = x1 - __uint_as_float(h1 << 16);
    hi = h0 | (h1 << 16);
    lo = f32_to_bf16_bits(r0) | (f32_to_bf16_bits(r1) << 16);
}

// ---- mma.sync m16n8k16 bf16 x bf16 -> fp32 (HMMA on sm_100a) --------------------------
__device__ __forceinline__ void mma_bf16_16816(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2,
                                               uint32_t a3, uint32_t b0, uint32_t b1) {
    asm volatile(
        "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, "
        "{%0,%1,%2,%3};\n"
        : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
        : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

// ---- streaming 16-byte global load (weights are read once per step: do not pollute L1) ----
__device__ __forceinline__ uint4 ldg_stream(const void* p) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];\n"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(p));
    return r;
}
__device__ __forceinline__ uint2 ldg_stream8(const void* p) {
    uint2 r;
    asm volatile("ld.global.nc.L1::no_allocate.v2.u32 {%0,%1}, [%2];\n" : "=r"(r.x), "=r"(r.y) : "l"(p));
    return r;
}
__device__ __forceinline__ void prefetch_l2(const void* p) {
    asm volatile("prefetch.global.L2 [%0];\n" ::"l"(p));
}

// ---- Philox4x32-10 (published round function; reading C2) -- the ONE device copy, used by the
// standalone sampler (sampler.cu) and by the fused LM-head epilogue (tc_linear.cu) ------------------------
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                              uint32_t k1, uint32_t (&out)[4]) {
#pragma unroll
    for (int i = 0; i < 10; ++i) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Gumbel draw of the sampler from one Philox word (step a12):  u = ((x >> 9) + 0.5) * 2^-23,  g = -log(-log u).
// Two MUFU.LG2 instead of two full-range logf: the inner log is taken as the series of -log(1 - e) with
// e = 1 - u formed EXACTLY when u is within 2^-6 of 1 (that is where the largest draws -- the likely winners
// of the arg-max -- live and where lg2 alone loses all relative accuracy); elsewhere |log u| > 0.0157 and the
// 2^-22 absolute error of lg2 is < 2e-5 relative.  |g - exact| < ~3e-5 over the whole range, far below the
// 1e-2 top-2 margin of the token rule.  Used by BOTH sampler paths (k_sample and the
// fused LM head) so that they pick identical tokens.
__device__ __forceinline__ float gumbel_from_u32(uint32_t x) {
    const float k = (float)(x >> 9);                               // 0 .. 2^23 - 1, exact
    const float u = (k + 0.5f) * 1.1920928955078125e-07f;          // exact in fp32
    const float e = (8388607.5f - k) * 1.1920928955078125e-07f;    // 1 - u, exact
    const float y_near1 = fmaf(e * e, fmaf(e, 0.33333334f, 0.5f), e);
    const float y_far = -__logf(u);
    const float y = (e < 0.015625f) ? y_near1 : y_far;
    return -__logf(y);
}

// ---- programmatic dependent launch (griddepcontrol) ---------------------------------
// pdl_wait(): block until the upstream grid's memory is visible (no-op without the PDL attr).
// pdl_launch(): allow the downstream grid to start its prologue.
// SAGC_PDL_EARLY: release the downstream grid BEFORE waiting on the upstream one, so that the launch
// chain runs ahead of execution and several kernels' weight prefetches are in flight at once
// (a kernel's wait still implies, transitively, that every earlier kernel of the stream is complete).
#ifdef SAGC_PDL_EARLY
__device__ __forceinline__ void pdl_wait() {
    asm volatile("griddepcontrol.launch_dependents;\n" ::: "memory");
    asm volatile("griddepcontrol.wait;\n" ::: "memory");
}
#else
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;\n" ::: "memory"); }
#endif
__device__ __forceinline__ void pdl_launch() { asm volatile("griddepcontrol.launch_dependents;\n" ::: "memory"); }

// ---- warp reductions -------------------------------------------------------------
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

// ---- optional in-kernel timeline (build with SAGC_TRACE_BUILD=1: -DSAGC_TRACE -rdc=true) -----
// thread 0 of block (0,0,0) appends (tag, %globaltimer) records; tag = kernel id * 4 + phase
// (0 = entered, 1 = upstream dependency satisfied, 2 = block 0 done).  Compiled out by default.
#ifdef SAGC_TRACE
extern __device__ unsigned long long* g_trace;
__device__ __forceinline__ void trace_mark(int tag) {
    if (g_trace != nullptr && threadIdx.x == 0 && blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0) {
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        const unsigned long long i = atomicAdd(g_trace, 1ull);
        if (i < (1ull << 20) - 2) g_trace[1 + i] = ((unsigned long long)tag << 56) | (t & 0x00ffffffffffffffull);
    }
}
__device__ __forceinline__ void trace_mark_thread(int tag, int thread) {
    if (g_trace != nullptr && (int)threadIdx.x == thread && blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0) {
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        const unsigned long long i = atomicAdd(g_trace, 1ull);
        if (i < (1ull << 20) - 2) g_trace[1 + i] = ((unsigned long long)tag << 56) | (t & 0x00ffffffffffffffull);
    }
}
__device__ __forceinline__ void trace_mark_allblocks(int tag) {
    if (g_trace != nullptr && threadIdx.x == 0) {
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        const unsigned long long i = atomicAdd(g_trace, 1ull);
        if (i < (1ull << 20) - 2) g_trace[1 + i] = ((unsigned long long)tag << 56) | (t & 0x00ffffffffffffffull);
    }
}
#else
#define trace_mark_allblocks(tag) ((void)0)
#define trace_mark(tag) ((void)0)
#define trace_mark_thread(tag, thread) ((void)0)
#endif

// Launch with the programmatic-stream-serialization attribute (PDL): the kernel may start while its
// predecessor is still running and must call pdl_wait() before touching anything the predecessor wrote.
template <typename... KArgs, typename... Args>
static inline cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, bool pdl,
                                     Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}

}  // namespace sagc
