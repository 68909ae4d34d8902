// Stage 2b — prefix-aware scheduling (cw_schedule).  DESIGN.md R3.
//
// One CTA: the queue (R <= 8192) lives in shared memory as 192-bit keys
//   policy 0  (a | ~n_gpu , arrival_seq , req_id | idx)      PAPER.md 5.1 L207 "fewest additional blocks"
//   policy 1  (~n_gpu | a , arrival_seq , req_id | idx)      L45 / Fig. 11B "degree of overlap"
//   policy 2  (0         , arrival_seq , req_id | idx)       L281 FCFS
// sorted by a bitonic network (keys are unique => the permutation is unique), followed by a block-wide
// prefix sum of a over the sorted order for the admission rule (L177: admit while it fits).
#include <stdio.h>

#include "cw_internal.cuh"

namespace {

#define CWS_THREADS 1024

struct Key3 {
    u64 k0, k1, k2;
};
__device__ __forceinline__ bool key_less(const Key3& x, const Key3& y) {
    if (x.k0 != y.k0) return x.k0 < y.k0;
    if (x.k1 != y.k1) return x.k1 < y.k1;
    return x.k2 < y.k2;
}

__global__ void __launch_bounds__(CWS_THREADS, 1)
    schedule_kernel(u32 R, u32 N, const u32* __restrict__ need, const u32* __restrict__ n_gpu,
                    const u64* __restrict__ arrival, const u32* __restrict__ req_id, u32 policy, u32 free_blocks,
                    u32 evictable, u32 max_admit, u32* order, u32* num_admit, u32* deficit) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    u64* k0 = reinterpret_cast<u64*>(smem_raw);
    u64* k1 = k0 + N;
    u64* k2 = k1 + N;
    __shared__ u64 warp_sums[32];
    __shared__ u32 s_count;
    __shared__ unsigned long long s_need;
    const u32 tid = threadIdx.x;

    for (u32 i = tid; i < N; i += CWS_THREADS) {
        if (i < R) {
            const u32 d = need[i], g = n_gpu[i];
            const u64 a = d > g ? d - g : 0;
            const u64 inv = 0xFFFFFFFFull - g;
            k0[i] = policy == 0 ? (a << 32) | inv : policy == 1 ? (inv << 32) | a : 0ull;
            k1[i] = arrival[i];
            k2[i] = ((u64)req_id[i] << 32) | i;
        } else {
            k0[i] = k1[i] = k2[i] = ~0ull;
        }
    }
    if (tid == 0) {
        s_count = 0;
        s_need = 0;
    }
    __syncthreads();

    for (u32 k = 2; k <= N; k <<= 1) {
        for (u32 j = k >> 1; j > 0; j >>= 1) {
            for (u32 t = tid; t < (N >> 1); t += CWS_THREADS) {
                // t-th compare-exchange pair of this stage
                const u32 i = ((t & ~(j - 1)) << 1) | (t & (j - 1));
                const u32 p = i | j;
                const bool up = (i & k) == 0;
                Key3 x{k0[i], k1[i], k2[i]}, y{k0[p], k1[p], k2[p]};
                if (key_less(y, x) == up) {
                    k0[i] = y.k0; k1[i] = y.k1; k2[i] = y.k2;
                    k0[p] = x.k0; k1[p] = x.k1; k2[p] = x.k2;
                }
            }
            __syncthreads();
        }
    }

    // admission: each thread owns a contiguous run of the sorted queue
    const u32 per = (R + CWS_THREADS - 1) / CWS_THREADS;
    const u32 lo = min(R, tid * per), hi = min(R, lo + per);
    u64 local = 0;
    for (u32 p = lo; p < hi; ++p) {
        const u32 i = (u32)k2[p];
        order[p] = i;
        const u32 d = need[i], g = n_gpu[i];
        local += d > g ? d - g : 0;
    }
    // block exclusive scan of `local`
    const u32 lane = tid & 31, warp = tid >> 5;
    u64 inc = local;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        u64 y = shfl64_up(inc, d);
        if (lane >= d) inc += y;
    }
    if (lane == 31) warp_sums[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        u64 w = warp_sums[lane];
        u64 wi = w;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            u64 y = shfl64_up(wi, d);
            if (lane >= d) wi += y;
        }
        warp_sums[lane] = wi - w;  // exclusive
    }
    __syncthreads();
    u64 run = warp_sums[warp] + inc - local;
    const u64 budget = (u64)free_blocks + (u64)evictable;
    u32 cnt = 0;
    u64 last_need = 0;
    for (u32 p = lo; p < hi; ++p) {
        const u32 i = (u32)k2[p];
        const u32 d = need[i], g = n_gpu[i];
        run += d > g ? d - g : 0;
        if (p < max_admit && run <= budget) {  // monotone in p: the admitted set is a prefix
            ++cnt;
            last_need = run;
        }
    }
    if (cnt) {
        atomicAdd(&s_count, cnt);
        atomicMax(&s_need, (unsigned long long)last_need);
    }
    __syncthreads();
    if (tid == 0) {
        *num_admit = s_count;
        const u64 nd = s_need;
        *deficit = nd > free_blocks ? (u32)min(nd - free_blocks, (u64)0xFFFFFFFFull) : 0u;
    }
}

}  // namespace

int32_t cwi_schedule(cw_ctx* ctx, u32 R, const u32* d_need, const u32* d_n_gpu, const u64* d_arrival_seq,
                     const u32* d_req_id, u32 policy, u32 free_blocks, u32 evictable, u32 max_admit, u32* d_order,
                     u32* d_num_admit, u32* d_deficit) {
    u32 N = 2;
    while (N < R) N <<= 1;
    const size_t smem = (size_t)N * 24;
    static bool attr_set = false;
    if (!attr_set) {
        CW_CUDA(ctx, cudaFuncSetAttribute(schedule_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 8192 * 24));
        attr_set = true;
    }
    schedule_kernel<<<1, CWS_THREADS, smem, ctx->s_main>>>(R, N, d_need, d_n_gpu, d_arrival_seq, d_req_id, policy,
                                                           free_blocks, evictable, max_admit, d_order, d_num_admit,
                                                           d_deficit);
    CW_LAUNCH_CHECK(ctx);
    return CW_OK;
}
