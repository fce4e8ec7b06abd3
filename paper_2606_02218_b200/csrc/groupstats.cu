// groupstats.cu -- segmented per-group kernels (step a14): group-relative advantages
// (GRPO mean/std, DAPO all-equal filter) and length statistics (max, sum, median_x2, max/mean).
// One warp per group over a CSR offsets array; reductions by warp shuffle in a fixed order.
#include "common.cuh"
#include "kernels.cuh"

namespace sagc {

__device__ __forceinline__ double warp_sum_d(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// all_equal := (max == min) exactly, or G == 1  ->  A = 0, keep = (mode == GRPO)
// else A_i = (r_i - mean) / (std + eps), std with divisor (G - ddof), two-pass in fp64.
__global__ void __launch_bounds__(256) k_group_advantage(const float* __restrict__ rewards,
                                                         const int* __restrict__ offs, int n_groups, int mode,
                                                         int ddof, float eps, float* __restrict__ adv,
                                                         uint8_t* __restrict__ keep) {
    const int g = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (g >= n_groups) return;
    const int lo = offs[g], hi = offs[g + 1];
    const int G = hi - lo;
    float mx = -INFINITY, mn = INFINITY;
    double sum = 0.0;
    for (int i = lo + lane; i < hi; i += 32) {
        const float r = rewards[i];
        mx = fmaxf(mx, r); mn = fminf(mn, r);
        sum += (double)r;
    }
    mx = warp_max(mx);
    mn = -warp_max(-mn);
    sum = warp_sum_d(sum);
    const bool degenerate = (G <= 1) || (mx == mn) || (G - ddof <= 0);
    if (degenerate) {
        for (int i = lo + lane; i < hi; i += 32) adv[i] = 0.f;
        if (lane == 0) keep[g] = (mode == 1) ? 0 : 1;
        return;
    }
    const double mean = sum / (double)G;
    double ss = 0.0;
    for (int i = lo + lane; i < hi; i += 32) {
        const double d = (double)rewards[i] - mean;
        ss += d * d;
    }
    ss = warp_sum_d(ss);
    const double denom = sqrt(ss / (double)(G - ddof)) + (double)eps;
    for (int i = lo + lane; i < hi; i += 32) adv[i] = (float)(((double)rewards[i] - mean) / denom);
    if (lane == 0) keep[g] = 1;
}

int launch_group_advantage(const float* rewards, const int* offs, int n_groups, int mode, int ddof, float eps,
                           float* adv, uint8_t* keep, cudaStream_t st) {
    if (n_groups <= 0) return 0;
    k_group_advantage<<<(n_groups + 7) / 8, 256, 0, st>>>(rewards, offs, n_groups, mode, ddof, eps, adv, keep);
    return 1;
}

// stats[g] = (max, sum, median_x2); median_x2 = sum of the two middle order statistics, found
// by rank counting (stable: ties broken by index).  ratio[g] = float(max*G) / float(sum).
__global__ void __launch_bounds__(256) k_length_stats(const int* __restrict__ lengths, const int* __restrict__ offs,
                                                      int n_groups, int* __restrict__ stats,
                                                      float* __restrict__ ratio) {
    const int g = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (g >= n_groups) return;
    const int lo = offs[g], hi = offs[g + 1];
    const int G = hi - lo;
    if (G <= 0) {
        if (lane == 0) {
            if (stats) { stats[g * 3] = 0; stats[g * 3 + 1] = 0; stats[g * 3 + 2] = 0; }
            if (ratio) ratio[g] = 0.f;
        }
        return;
    }
    int mx = 0;
    long long tot = 0;
    int med2 = 0;
    const int ra = (G - 1) / 2, rb = G / 2;
    for (int i = lo + lane; i < hi; i += 32) {
        const int v = lengths[i];
        mx = max(mx, v);
        tot += v;
        int rank = 0;
        for (int j = lo; j < hi; ++j) {
            const int u = lengths[j];
            rank += (u < v) || (u == v && j < i);
        }
        if (rank == ra) med2 += v;
        if (rank == rb) med2 += v;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
        tot += __shfl_xor_sync(0xffffffffu, tot, o);
        med2 += __shfl_xor_sync(0xffffffffu, med2, o);
    }
    if (lane == 0) {
        if (stats) { stats[g * 3] = mx; stats[g * 3 + 1] = (int)tot; stats[g * 3 + 2] = med2; }
        if (ratio) ratio[g] = __fdiv_rn(__ll2float_rn((long long)mx * G), __ll2float_rn(tot));
    }
}

int launch_length_stats(const int* lengths, const int* offs, int n_groups, int* stats, float* ratio,
                        cudaStream_t st) {
    if (n_groups <= 0) return 0;
    k_length_stats<<<(n_groups + 7) / 8, 256, 0, st>>>(lengths, offs, n_groups, stats, ratio);
    return 1;
}

}  // namespace sagc
