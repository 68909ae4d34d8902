// Stage 2b — prefix-aware scheduling (cw_schedule).  DESIGN.md R3.
//
// The queue is ordered by a 192-bit key that is a TOTAL order (the input index is its last component):
//   policy 0  (a | ~n_gpu , arrival_seq , req_id | idx)      PAPER.md 5.1 L207 "fewest additional blocks"
//   policy 1  (~n_gpu | a , arrival_seq , req_id | idx)      L45 / Fig. 11B "degree of overlap"
//   policy 2  (arrival_seq , 0         , req_id | idx)       L281 FCFS
// A few thousand keys are too few to feed a radix sort and too many for one CTA's sorting network, so the
// sort is a RANK SORT spread over the whole GPU: rank(i) = #{j : key_j < key_i}, R^2 comparisons (16.7 M at
// R = 4096, one warp per element).  Only the LEADING word of every key is staged in shared memory (it decides
// almost every pair: a branch-free smaller/equal count); the other words are fetched from global memory for the
// few keys that tie on it.  order[rank(i)] = i.
// The last CTA to finish (atomic ticket, no spinning) runs the admission rule of L177 over the sorted
// order: exclusive prefix sum of a, admit while it fits, stop at the first misfit.
#include <stdio.h>

#include "cw_internal.cuh"

namespace {

#define CWS_THREADS 256
#define CWS_I_PER_CTA 8                       // elements ranked by one CTA
#define CWS_J_LANES (CWS_THREADS / CWS_I_PER_CTA)  // threads sharing one element (split the j range)
#define CWS_TILE 8192                         // leading key words staged per shared-memory tile (64 KiB)

struct Key3 {
    u64 k0, k1, k2;
};
__device__ __forceinline__ Key3 make_key(u32 i, const u32* need, const u32* n_gpu, const u64* arrival,
                                         const u32* req_id, u32 policy) {
    const u32 d = need[i], g = n_gpu[i];
    const u64 a = d > g ? d - g : 0;
    const u64 inv = 0xFFFFFFFFull - g;
    Key3 k;
    // FCFS puts arrival_seq in the leading word so that the first comparison decides almost every pair
    k.k0 = policy == 0 ? (a << 32) | inv : policy == 1 ? (inv << 32) | a : arrival[i];
    k.k1 = policy == 2 ? 0ull : arrival[i];
    k.k2 = ((u64)req_id[i] << 32) | i;
    return k;
}

__device__ __forceinline__ u64 make_k0(u32 i, const u32* need, const u32* n_gpu, const u64* arrival, u32 policy) {
    if (policy == 2) return arrival[i];
    const u32 d = need[i], g = n_gpu[i];
    const u64 a = d > g ? d - g : 0;
    const u64 inv = 0xFFFFFFFFull - g;
    return policy == 0 ? (a << 32) | inv : (inv << 32) | a;
}

__global__ void __launch_bounds__(CWS_THREADS)
    schedule_kernel(u32 R, const u32* __restrict__ need, const u32* __restrict__ n_gpu,
                    const u64* __restrict__ arrival, const u32* __restrict__ req_id, u32 policy, u32 free_blocks,
                    u32 evictable, u32 max_admit, u32* order, u32* a_sorted, u32* ticket, u32* num_admit,
                    u32* deficit) {
    extern __shared__ __align__(16) u64 s_k0[];  // leading words of up to CWS_TILE keys
    __shared__ u64 s_warp[CWS_THREADS / 32];
    __shared__ u32 s_last;
    __shared__ u32 s_count;
    __shared__ unsigned long long s_need;
    const u32 tid = threadIdx.x;
    const u32 il = tid / CWS_J_LANES, jl = tid % CWS_J_LANES;  // one warp per element
    const u32 i = blockIdx.x * CWS_I_PER_CTA + il;
    const bool live = i < R;
    Key3 mine{~0ull, ~0ull, ~0ull};
    if (live) mine = make_key(i, need, n_gpu, arrival, req_id, policy);

    // Per tile of keys: pass 1 (branch-free) counts the leading words that are smaller / equal — the leading word
    // decides almost every pair; pass 2 runs only if another key of the tile shares this element's leading word and
    // lets the remaining words (read from global memory: rare) decide among those.
    u32 rank = 0;
    for (u32 base = 0; base < R; base += CWS_TILE) {
        const u32 n = min((u32)CWS_TILE, R - base);
        __syncthreads();
        for (u32 t0 = tid; t0 < n; t0 += CWS_THREADS * 8) {  // 8 keys per thread in flight: one load latency, not 8
            u64 v[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const u32 t = t0 + k * CWS_THREADS;
                v[k] = t < n ? make_k0(base + t, need, n_gpu, arrival, policy) : 0ull;
            }
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const u32 t = t0 + k * CWS_THREADS;
                if (t < n) s_k0[t] = v[k];
            }
        }
        __syncthreads();
        u32 ties = 0;
        if (live) {
#pragma unroll 8
            for (u32 t = jl; t < n; t += CWS_J_LANES) {
                const u64 o0 = s_k0[t];
                rank += o0 < mine.k0 ? 1u : 0u;
                ties += o0 == mine.k0 ? 1u : 0u;
            }
        }
        ties = __reduce_add_sync(0xffffffffu, ties);  // the lanes of a warp share one element
        const u32 self = (live && i >= base && i < base + n) ? 1u : 0u;
        if (ties > self) {
            for (u32 t = jl; t < n; t += CWS_J_LANES) {
                const u32 jdx = base + t;
                if (s_k0[t] != mine.k0 || jdx == i) continue;
                const u64 o1 = policy == 2 ? 0ull : arrival[jdx];
                const u64 o2 = ((u64)req_id[jdx] << 32) | jdx;
                rank += (o1 < mine.k1 || (o1 == mine.k1 && o2 < mine.k2)) ? 1u : 0u;
            }
        }
    }
    rank = __reduce_add_sync(0xffffffffu, rank);
    if (live && jl == 0) {
        order[rank] = i;
        const u32 d = need[i], g = n_gpu[i];
        a_sorted[rank] = d > g ? d - g : 0;
    }

    // ---- the last CTA to arrive runs the admission rule over the sorted order
    __threadfence();
    __syncthreads();
    if (tid == 0) s_last = atomicAdd(ticket, 1u) == gridDim.x - 1 ? 1u : 0u;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    if (tid == 0) {
        *ticket = 0;  // self-cleaning: ready for the next call
        s_count = 0;
        s_need = 0;
    }
    __syncthreads();
    const u32 per = (R + CWS_THREADS - 1) / CWS_THREADS;
    const u32 lo = min(R, tid * per), hi = min(R, lo + per);
    // a_sorted was written by other CTAs: read it through L2 (__ldcg), loads independent of one another
    u64 local = 0;
#pragma unroll 8
    for (u32 p = lo; p < hi; ++p) local += __ldcg(a_sorted + p);
    const u32 lane = tid & 31, warp = tid >> 5;
    u64 inc = local;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        u64 y = shfl64_up(inc, d);
        if (lane >= d) inc += y;
    }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        u64 w = lane < CWS_THREADS / 32 ? s_warp[lane] : 0, wi = w;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            u64 y = shfl64_up(wi, d);
            if (lane >= d) wi += y;
        }
        if (lane < CWS_THREADS / 32) s_warp[lane] = wi - w;  // exclusive
    }
    __syncthreads();
    u64 run = s_warp[warp] + inc - local;
    const u64 budget = (u64)free_blocks + (u64)evictable;
    u32 cnt = 0;
    u64 last_need = 0;
#pragma unroll 8
    for (u32 p = lo; p < hi; ++p) {
        run += __ldcg(a_sorted + p);
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

__global__ void schedule_empty_kernel(u32* num_admit, u32* deficit) {
    *num_admit = 0;
    *deficit = 0;
}

}  // namespace

int32_t cwi_schedule(cw_ctx* ctx, u32 R, const u32* d_need, const u32* d_n_gpu, const u64* d_arrival_seq,
                     const u32* d_req_id, u32 policy, u32 free_blocks, u32 evictable, u32 max_admit, u32* d_order,
                     u32* d_num_admit, u32* d_deficit) {
    if (R == 0) {
        schedule_empty_kernel<<<1, 1, 0, ctx->s_main>>>(d_num_admit, d_deficit);
        CW_LAUNCH_CHECK(ctx);
        return CW_OK;
    }
    const u32 grid = (R + CWS_I_PER_CTA - 1) / CWS_I_PER_CTA;
    static bool attr_set = false;
    if (!attr_set) {
        CW_CUDA(ctx, cudaFuncSetAttribute(schedule_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, CWS_TILE * 8));
        attr_set = true;
    }
    const size_t smem = (size_t)(R < CWS_TILE ? R : CWS_TILE) * 8;
    schedule_kernel<<<grid, CWS_THREADS, smem, ctx->s_main>>>(R, d_need, d_n_gpu, d_arrival_seq, d_req_id, policy,
                                                           free_blocks, evictable, max_admit, d_order, ctx->sched_a,
                                                           ctx->sched_ticket, d_num_admit, d_deficit);
    CW_LAUNCH_CHECK(ctx);
    return CW_OK;
}
