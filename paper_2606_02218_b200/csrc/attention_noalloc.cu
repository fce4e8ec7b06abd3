// attention_noalloc.cu -- sagc_attention_noalloc: the split-K paged GQA attention unit (attention_body.cuh, step a7)
// for callers that may not allocate (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).
//
// The split-K scratch of the existing path (partial outputs, (max, sum) pairs, arrival counters, the identity live
// list) comes from cudaMalloc inside sagc_debug_attention / the model.  Here it lives in ONE file-scope device array
// of SAGC_NOALLOC_SCRATCH_BYTES (8 MiB) that every GPU which loads the library holds until the process exits.
//   * the array's name is a host-side stand-in in host code, so its device address is taken ONCE PER DEVICE with
//     cudaGetSymbolAddress while that device is current (checked), and that pointer is what the kernels get;
//   * the entry point calls no cudaMalloc / cudaFree / allocating library routine and does not synchronise: it
//     enqueues two kernels on the caller's stream and returns;
//   * every call shares the array and finds the previous call's contents in it: the arrival counters and the live
//     list are rewritten by k_noalloc_init at the start of every call (the partials are fully overwritten before
//     they are read);
//   * calls that overlap on the GPU (two streams, two host threads on different streams) RACE on the array: keep the
//     calls of one device on one stream, or order them with events.
#include <cstdio>
#include <mutex>

#include "attention_body.cuh"
#include "../../include/sagc.h"

namespace sagc {

int api_set_error(int code, const char* msg);      // runtime.cu: message for sagc_last_error()

static constexpr size_t NOALLOC_BYTES = SAGC_NOALLOC_SCRATCH_BYTES;
static __device__ __align__(256) unsigned char g_noalloc_scratch[NOALLOC_BYTES];

static constexpr int NOALLOC_MAX_DEV = 64;
static unsigned char* g_noalloc_ptr[NOALLOC_MAX_DEV] = {};      // device address of the array, per device
static std::mutex g_noalloc_mu;

static inline size_t up256(size_t n) { return (n + 255) & ~(size_t)255; }

// counters <- 0, live list <- identity (row i is sequence i of the caller's page table)
__global__ void k_noalloc_init(int* counters, int n_counters, int* row_sid, int M) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n_counters) counters[i] = 0;
    if (i < M) row_sid[i] = i;
}

// one CTA per (row, kv head, split); partials merge through the scratch (last arriver), never through a cluster
template <int HD, int WARPS, int NSTAGE>
__global__ void __launch_bounds__(ATT_THREADS) k_attention_noalloc(AttnArgs a) {
    extern __shared__ __align__(128) unsigned char kv_s[];
    __shared__ AttSmall sm;
    attention_unit<HD, WARPS, NSTAGE, false>(a, blockIdx.x, blockIdx.y, blockIdx.z, a.n_splits, kv_s, &sm, nullptr, (int)threadIdx.x);
}

template <int HD>
static cudaError_t launch_noalloc(const AttnArgs& a, cudaStream_t st) {
    constexpr int WARPS = 8, NSTAGE = HD >= 128 ? 2 : (HD >= 64 ? 3 : 6);      // the standalone kernel's geometry
    constexpr int BYTES = AttGeom<HD, WARPS, NSTAGE>::BYTES;
    cudaError_t e = cudaFuncSetAttribute(k_attention_noalloc<HD, WARPS, NSTAGE>, cudaFuncAttributeMaxDynamicSharedMemorySize, BYTES);
    if (e != cudaSuccess) return e;
    k_attention_noalloc<HD, WARPS, NSTAGE><<<dim3(a.m_max, a.Hkv, a.n_splits), ATT_THREADS, BYTES, st>>>(a);
    return cudaGetLastError();
}

}  // namespace sagc

using namespace sagc;

extern "C" int sagc_attention_noalloc(const float* q, const void* kv, const int32_t* page_table, const int32_t* ctx, int32_t M,
                                      int32_t Hq, int32_t Hkv, int32_t hd, int32_t page_tokens, int32_t max_blocks,
                                      int32_t n_splits, float* out, void* stream) {
    char msg[256];
    if (!q || !kv || !page_table || !ctx || !out || M < 1 || max_blocks < 1) return api_set_error(SAGC_EINVAL, "null argument or empty batch");
    if (Hkv < 1 || Hq % Hkv || Hq / Hkv > ATT_MAXR) return api_set_error(SAGC_EINVAL, "bad head counts");
    if (hd != 32 && hd != 64 && hd != 128) return api_set_error(SAGC_EINVAL, "head_dim must be 32, 64 or 128");
    if (page_tokens < 16 || (page_tokens & (page_tokens - 1))) return api_set_error(SAGC_EINVAL, "page_tokens must be a power of two >= 16");
    if (n_splits < 1 || n_splits > 64) return api_set_error(SAGC_EINVAL, "n_splits must be in 1..64");
    // scratch layout: counters | live list | (max, sum) pairs | partial outputs, each 256-byte aligned
    const size_t b_cnt = up256((size_t)M * Hkv * sizeof(int));
    const size_t b_sid = up256((size_t)M * sizeof(int));
    const size_t b_ml = up256((size_t)M * Hq * n_splits * 2 * sizeof(float));
    const size_t b_o = up256((size_t)M * Hq * n_splits * hd * sizeof(float));
    const size_t need = b_cnt + b_sid + b_ml + b_o;
    if (need > NOALLOC_BYTES) {
        snprintf(msg, sizeof(msg), "sagc_attention_noalloc: M=%d Hq=%d n_splits=%d head_dim=%d needs %zu scratch bytes, the static "
                 "array holds %zu (SAGC_NOALLOC_SCRATCH_BYTES): use fewer rows or splits per call", M, Hq, n_splits, hd, need, NOALLOC_BYTES);
        return api_set_error(SAGC_EINVAL, msg);
    }
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess || dev < 0 || dev >= NOALLOC_MAX_DEV) return api_set_error(SAGC_ECUDA, "sagc_attention_noalloc: no current device");
    unsigned char* base = nullptr;
    {
        std::lock_guard<std::mutex> lk(g_noalloc_mu);
        if (g_noalloc_ptr[dev] == nullptr) {         // set-up, once per device, with that device current
            void* p = nullptr;
            e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
            if (e != cudaSuccess || p == nullptr) {
                snprintf(msg, sizeof(msg), "cudaGetSymbolAddress(g_noalloc_scratch) on device %d: %s", dev, cudaGetErrorString(e));
                return api_set_error(SAGC_ECUDA, msg);
            }
            g_noalloc_ptr[dev] = static_cast<unsigned char*>(p);
        }
        base = g_noalloc_ptr[dev];
    }
    cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
    int* cnt = reinterpret_cast<int*>(base);
    int* sid = reinterpret_cast<int*>(base + b_cnt);
    float* pml = reinterpret_cast<float*>(base + b_cnt + b_sid);
    float* po = reinterpret_cast<float*>(base + b_cnt + b_sid + b_ml);
    const int n_init = M * Hkv > M ? M * Hkv : M;
    k_noalloc_init<<<(n_init + 255) / 256, 256, 0, st>>>(cnt, M * Hkv, sid, M);
    e = cudaGetLastError();
    if (e == cudaSuccess) {
        AttnArgs a = {};
        a.q = q; a.ldq = Hq * hd; a.kv_layer = reinterpret_cast<const bf16_t*>(kv); a.page_table = page_table;
        a.max_blocks = max_blocks; a.row_sid = sid; a.row_ctx = ctx; a.m_dev = nullptr; a.m_max = M; a.Hq = Hq; a.Hkv = Hkv;
        a.hd = hd; a.page = page_tokens; a.n_splits = n_splits; a.part_o = po; a.part_ml = pml; a.counters = cnt; a.out = out;
        a.cluster_merge = 0;
        e = hd == 128 ? launch_noalloc<128>(a, st) : (hd == 64 ? launch_noalloc<64>(a, st) : launch_noalloc<32>(a, st));
    }
    if (e != cudaSuccess) {
        snprintf(msg, sizeof(msg), "sagc_attention_noalloc launch: %s", cudaGetErrorString(e));
        return api_set_error(SAGC_ECUDA, msg);
    }
    return SAGC_OK;
}
