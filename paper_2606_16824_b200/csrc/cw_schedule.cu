// Stage 2b — prefix-aware scheduling (cw_schedule).  DESIGN.md R3.
//
// The queue is ordered by a 192-bit key that is a TOTAL order (the input index is its last component):
//   policy 0  (a | ~n_gpu , arrival_seq , req_id | idx)      PAPER.md 5.1 L207 "fewest additional blocks"
//   policy 1  (~n_gpu | a , arrival_seq , req_id | idx)      L45 / Fig. 11B "degree of overlap"
//   policy 2  (arrival_seq , 0         , req_id | idx)       L281 FCFS
// A few thousand keys are too few to feed a radix sort and too many for one CTA's sorting network, so the
// sort is a RANK SORT spread over the whole GPU: rank(i) = #{j : key_j < key_i}, R^2 comparisons (16.7 M at
// R = 4096), one warp per element, ceil(R / #SM) elements per CTA so that every SM stages the keys exactly once.
// Only the LEADING word of every key is staged in shared memory (it decides almost every pair).  Fast path
// (R <= 16 x threads): the leading words are compressed to <= 30 bits, (hi - hi_min) << bits(lo range) | (lo - lo_min),
// so that a compare is the sign bit of a 32-bit difference (IMAD.IADD + LEA.HI: one instruction on each of the two
// integer pipes) and one LDS.128 feeds four compares; #{<} and #{<=} are counted, their difference is the tie count.
// Warps whose element ties on the leading word collect the tied indices (warp scan of the per-lane tie counts ->
// private list slices) and fetch the remaining words of exactly those keys from global memory, all loads in flight
// together.  Ranges that do not fit 30 bits, or R beyond the fast path, take the 64-bit tile loop.
// order[rank(i)] = i.
// A second one-CTA kernel runs the admission rule of L177 over the sorted order: exclusive prefix sum of a,
// admit while it fits, stop at the first misfit (a kernel boundary is a cheaper grid-wide hand-over than a fence +
// ticket in every rank CTA).
#include <stdio.h>

#include "cw_internal.cuh"

namespace {

#define CWS_MAX_THREADS 1024
#define CWS_MAX_I (CWS_MAX_THREADS / 32)      // elements ranked by one CTA (one warp each); the launch picks
                                              // ceil(R / #SM) so that every SM stages the keys exactly once
#define CWS_FAST_KEYS 16                      // keys held in registers per thread on the compressed-key fast path
#define CWS_TIE_CAP 128                       // tied keys resolved through the per-warp list
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

__global__ void __launch_bounds__(CWS_MAX_THREADS)
    schedule_kernel(u32 R, const u32* __restrict__ need, const u32* __restrict__ n_gpu,
                    const u64* __restrict__ arrival, const u32* __restrict__ req_id, u32 policy, u32 free_blocks,
                    u32 evictable, u32 max_admit, u32* order, u32* a_sorted) {
    extern __shared__ __align__(16) u64 s_k0[];  // leading words of up to CWS_TILE keys
    {   // the tie-break words are gathered at random by the few warps that tie: pull them into L2 up front
        const u32 line = blockIdx.x * blockDim.x + threadIdx.x;  // one 128-byte line per thread
        if (line * 16 < R) asm volatile("prefetch.global.L2 [%0];" ::"l"(arrival + line * 16));
        if (line * 32 < R) asm volatile("prefetch.global.L2 [%0];" ::"l"(req_id + line * 32));
    }
    const u32 tid = threadIdx.x;
    const u32 n_thr = blockDim.x;
    const u32 il = tid >> 5, jl = tid & 31;  // one warp per element
    const u32 i = blockIdx.x * (n_thr >> 5) + il;
    const bool live = i < R;
    Key3 mine{~0ull, ~0ull, ~0ull};
    if (live) mine = make_key(i, need, n_gpu, arrival, req_id, policy);

    u32 rank = 0;
    // ---- fast path (R <= CWS_FAST_KEYS per thread x threads): the leading words are COMPRESSED to <= 30 bits,
    // (hi - hi_min) << bits(lo range) | (lo - lo_min) — order-preserving and injective on the leading word — so that
    // a compare is two 32-bit ALU operations on the sign of a difference instead of a 64-bit set-predicate pair, and
    // one LDS.128 feeds four compares.  Falls through to the 64-bit tile loop when the ranges do not fit.
    bool done = false;
    if (R <= CWS_FAST_KEYS * n_thr) {
        u32* s_c = reinterpret_cast<u32*>(s_k0);
        __shared__ u32 s_mm[4][CWS_MAX_I];  // per-warp partial min / max (no shared-memory atomics: they serialise)
        __shared__ u32 s_tie[CWS_MAX_I][CWS_TIE_CAP];
        u32 hi[CWS_FAST_KEYS], lo[CWS_FAST_KEYS];
        u32 hmin = 0xFFFFFFFFu, hmax = 0, lmin = 0xFFFFFFFFu, lmax = 0;
        // unconditional loads at clamped indices (policy hoisted): all of a thread's loads are in flight together
        if (policy == 2) {
#pragma unroll
            for (int k = 0; k < CWS_FAST_KEYS; ++k) {
                if (k * n_thr >= R) break;  // CTA-uniform
                const u64 v = arrival[min(tid + k * n_thr, R - 1)];
                hi[k] = (u32)(v >> 32);
                lo[k] = (u32)v;
            }
        } else {
#pragma unroll
            for (int k = 0; k < CWS_FAST_KEYS; ++k) {
                if (k * n_thr >= R) break;  // CTA-uniform
                const u32 t = min(tid + k * n_thr, R - 1);
                hi[k] = need[t];
                lo[k] = n_gpu[t];
            }
#pragma unroll
            for (int k = 0; k < CWS_FAST_KEYS; ++k) {
                if (k * n_thr >= R) break;
                const u32 a = hi[k] > lo[k] ? hi[k] - lo[k] : 0u, inv = 0xFFFFFFFFu - lo[k];
                hi[k] = policy == 0 ? a : inv;
                lo[k] = policy == 0 ? inv : a;
            }
        }
#pragma unroll
        for (int k = 0; k < CWS_FAST_KEYS; ++k) {
            const u32 t = tid + k * n_thr;
            if (t < R) {
                hmin = min(hmin, hi[k]);
                hmax = max(hmax, hi[k]);
                lmin = min(lmin, lo[k]);
                lmax = max(lmax, lo[k]);
            }
        }
        hmin = __reduce_min_sync(0xffffffffu, hmin);
        hmax = __reduce_max_sync(0xffffffffu, hmax);
        lmin = __reduce_min_sync(0xffffffffu, lmin);
        lmax = __reduce_max_sync(0xffffffffu, lmax);
        if (jl == 0) {
            s_mm[0][il] = hmin;
            s_mm[1][il] = hmax;
            s_mm[2][il] = lmin;
            s_mm[3][il] = lmax;
        }
        __syncthreads();
        {   // every warp folds the per-warp partials on its own (32 lanes, 4 redux): no second barrier
            const u32 nw = n_thr >> 5;
            hmin = __reduce_min_sync(0xffffffffu, jl < nw ? s_mm[0][jl] : 0xFFFFFFFFu);
            hmax = __reduce_max_sync(0xffffffffu, jl < nw ? s_mm[1][jl] : 0u);
            lmin = __reduce_min_sync(0xffffffffu, jl < nw ? s_mm[2][jl] : 0xFFFFFFFFu);
            lmax = __reduce_max_sync(0xffffffffu, jl < nw ? s_mm[3][jl] : 0u);
        }
        const u32 hb = 32 - __clz(hmax - hmin), lb = 32 - __clz(lmax - lmin);
        if (hb + lb <= 30) {  // CTA-uniform
            done = true;
            const u32 n_pad = (R + 127) & ~127u;  // one warp-wide LDS.128 covers 128 keys; pad never compares below
#pragma unroll
            for (int k = 0; k < CWS_FAST_KEYS; ++k) {
                const u32 t = tid + k * n_thr;
                if (t < n_pad) s_c[t] = t < R ? ((hi[k] - hmin) << lb) | (lo[k] - lmin) : 0x7FFFFFFFu;
            }
            __syncthreads();
            const u32 m = live ? (((u32)(mine.k0 >> 32) - hmin) << lb) | ((u32)mine.k0 - lmin) : 0u;
            const u32 m1 = m + 1;
            u32 lt = 0, le = 0;  // #{c_j < m}, #{c_j <= m}: sign bits of c_j - m and c_j - (m + 1), all values < 2^31
            const uint4* s_c4 = reinterpret_cast<const uint4*>(s_c);
#pragma unroll 4
            for (u32 q = jl; q < n_pad / 4; q += 32) {
                const uint4 v = s_c4[q];
                lt += ((v.x - m) >> 31) + ((v.y - m) >> 31) + ((v.z - m) >> 31) + ((v.w - m) >> 31);
                le += ((v.x - m1) >> 31) + ((v.y - m1) >> 31) + ((v.z - m1) >> 31) + ((v.w - m1) >> 31);
            }
            const u32 ties = __reduce_add_sync(0xffffffffu, le - lt);
            rank = lt;
            if (live && ties > 1) {  // warp-uniform: other keys share the leading word; the remaining words decide.
                // The lanes that saw an equal key rescan their own quarter-words and append the tied indices to a
                // per-warp list; the list is then resolved with one lane per tied key, so that the global loads of
                // a large tie group overlap instead of forming one dependent chain per key.
                const u32 n_tied = ties - 1;
                u32* list = s_tie[il];
                if (n_tied <= CWS_TIE_CAP) {
                    // each lane knows how many tied keys its own quarter-words hold: an exclusive warp scan gives
                    // it a private slice of the list (no atomics, no ballots, predicated stores only)
                    const u32 mine_tied = le - lt - ((((i >> 2) & 31) == jl) ? 1u : 0u);
                    u32 off = mine_tied;
#pragma unroll
                    for (int d = 1; d < 32; d <<= 1) {
                        const u32 y = __shfl_up_sync(0xffffffffu, off, d);
                        if (jl >= (u32)d) off += y;
                    }
                    off -= mine_tied;
                    if (mine_tied) {
#pragma unroll 4
                        for (u32 q = jl; q < n_pad / 4; q += 32) {
                            const uint4 v = s_c4[q];
                            const u32 t = q * 4;
                            if (v.x == m && t != i) list[off++] = t;
                            if (v.y == m && t + 1 != i) list[off++] = t + 1;
                            if (v.z == m && t + 2 != i) list[off++] = t + 2;
                            if (v.w == m && t + 3 != i) list[off++] = t + 3;
                        }
                    }
                    __syncwarp();
                    for (u32 e0 = jl; e0 < n_tied; e0 += 128) {  // 4 tied keys per lane in flight
                        u32 j[4];
                        u64 o1[4];
                        u32 rq[4];
#pragma unroll
                        for (int k = 0; k < 4; ++k) j[k] = list[min(e0 + 32 * k, n_tied - 1)];
#pragma unroll
                        for (int k = 0; k < 4; ++k) {
                            o1[k] = policy == 2 ? 0ull : arrival[j[k]];
                            rq[k] = req_id[j[k]];
                        }
#pragma unroll
                        for (int k = 0; k < 4; ++k) {
                            const u64 o2 = ((u64)rq[k] << 32) | j[k];
                            const bool less = o1[k] < mine.k1 || (o1[k] == mine.k1 && o2 < mine.k2);
                            rank += (e0 + 32 * k < n_tied && less) ? 1u : 0u;
                        }
                    }
                } else {  // a tie group larger than the list: plain scan
                    for (u32 t = jl; t < R; t += 32) {
                        if (s_c[t] != m || t == i) continue;
                        const u64 o1 = policy == 2 ? 0ull : arrival[t];
                        const u64 o2 = ((u64)req_id[t] << 32) | t;
                        rank += (o1 < mine.k1 || (o1 == mine.k1 && o2 < mine.k2)) ? 1u : 0u;
                    }
                }
            }
        }
    }
    // ---- general path.  Per tile of keys: pass 1 (branch-free) counts the leading words that are smaller / equal;
    // pass 2 runs only if another key of the tile shares this element's leading word and lets the remaining words
    // (read from global memory: rare) decide among those.
    for (u32 base = 0; base < (done ? 0u : R); base += CWS_TILE) {
        const u32 n = min((u32)CWS_TILE, R - base);
        __syncthreads();
        for (u32 t0 = tid; t0 < n; t0 += n_thr * 8) {  // 8 keys per thread in flight: one load latency, not 8
            u64 v[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const u32 t = t0 + k * n_thr;
                v[k] = t < n ? make_k0(base + t, need, n_gpu, arrival, policy) : 0ull;
            }
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const u32 t = t0 + k * n_thr;
                if (t < n) s_k0[t] = v[k];
            }
        }
        __syncthreads();
        u32 ties = 0;
        if (live) {
#pragma unroll 8
            for (u32 t = jl; t < n; t += 32) {
                const u64 o0 = s_k0[t];
                rank += o0 < mine.k0 ? 1u : 0u;
                ties += o0 == mine.k0 ? 1u : 0u;
            }
        }
        ties = __reduce_add_sync(0xffffffffu, ties);  // the lanes of a warp share one element
        const u32 self = (live && i >= base && i < base + n) ? 1u : 0u;
        if (ties > self) {
            for (u32 t = jl; t < n; t += 32) {
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
}

// Admission rule of L177 over the sorted order (one CTA; a kernel boundary is a cheaper grid-wide hand-over than a
// fence + ticket in every rank CTA): exclusive prefix sum of a, admit while it fits, stop at the first misfit.
#define CWA_THREADS 1024
#define CWA_REG 8
__global__ void __launch_bounds__(CWA_THREADS)
    admit_kernel(u32 R, const u32* __restrict__ a_sorted, u32 free_blocks, u32 evictable, u32 max_admit,
                 u32* num_admit, u32* deficit) {
    __shared__ u64 s_warp[CWA_THREADS / 32];
    __shared__ u32 s_count;
    __shared__ unsigned long long s_need;
    const u32 tid = threadIdx.x;
    if (tid == 0) {
        s_count = 0;
        s_need = 0;
    }
    const u32 per = (R + CWA_THREADS - 1) / CWA_THREADS;
    const u32 lo = min(R, tid * per), hi = min(R, lo + per);
    // up to CWA_REG values per thread stay in registers between the two passes (R <= 8192)
    u32 av[CWA_REG];
    const bool in_regs = per <= CWA_REG;
    u64 local = 0;
    if (in_regs) {
#pragma unroll
        for (int k = 0; k < CWA_REG; ++k) {
            av[k] = lo + k < hi ? a_sorted[lo + k] : 0u;
            local += av[k];
        }
    } else {
#pragma unroll 4
        for (u32 p = lo; p < hi; ++p) local += a_sorted[p];
    }
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
        u64 w = s_warp[lane], wi = w;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            u64 y = shfl64_up(wi, d);
            if (lane >= d) wi += y;
        }
        s_warp[lane] = wi - w;  // exclusive
    }
    __syncthreads();
    u64 run = s_warp[warp] + inc - local;
    const u64 budget = (u64)free_blocks + (u64)evictable;
    u32 cnt = 0;
    u64 last_need = 0;
    if (in_regs) {
#pragma unroll
        for (int k = 0; k < CWA_REG; ++k) {
            const u32 p = lo + k;
            run += av[k];
            if (p < hi && p < max_admit && run <= budget) {  // monotone in p: the admitted set is a prefix
                ++cnt;
                last_need = run;
            }
        }
    } else {
#pragma unroll 4
        for (u32 p = lo; p < hi; ++p) {
            run += a_sorted[p];
            if (p < max_admit && run <= budget) {
                ++cnt;
                last_need = run;
            }
        }
    }
    {   // one shared-memory atomic per warp, not per thread
        const u32 wc = __reduce_add_sync(0xffffffffu, cnt);
        const u32 nh = __reduce_max_sync(0xffffffffu, (u32)(last_need >> 32));
        const u32 nl = __reduce_max_sync(0xffffffffu, (u32)(last_need >> 32) == nh ? (u32)last_need : 0u);
        if (lane == 0 && wc) {
            atomicAdd(&s_count, wc);
            atomicMax(&s_need, ((unsigned long long)nh << 32) | nl);
        }
    }
    __syncthreads();
    if (tid == 0) {
        *num_admit = s_count;
        const u64 nd = s_need;
        *deficit = nd > free_blocks ? (u32)min(nd - free_blocks, (u64)0xFFFFFFFFull) : 0u;
    }
}

// NEXT-3: admission under a chunked-prefill token budget (PAPER.md 6.1 L271, R8).  Both
// running sums (blocks, tokens) only grow along the dispatch order, so "admitted" is a prefix of it and every test of
// the sequential walk becomes a test on exclusive / inclusive prefix sums: one CTA, two 64-bit block scans.
__global__ void __launch_bounds__(CWA_THREADS)
    admit_chunked_kernel(u32 R, const u32* __restrict__ order, const u32* __restrict__ need, const u32* __restrict__ n_gpu,
                         const u32* __restrict__ new_tokens, u32 free_blocks, u32 evictable, u32 max_admit,
                         u64 token_budget, u32* chunk_tokens, u32* num_admit, u32* deficit, u32* status) {
    __shared__ u64 s_a[CWA_THREADS / 32], s_t[CWA_THREADS / 32];
    __shared__ u32 s_count;
    __shared__ unsigned long long s_need;
    const u32 tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) {
        s_count = 0;
        s_need = 0;
    }
    const u32 per = (R + CWA_THREADS - 1) / CWA_THREADS;
    const u32 lo = min(R, tid * per), hi = min(R, lo + per);
    u64 sum_a = 0, sum_t = 0;
    bool bad = false;
    for (u32 p = lo; p < hi; ++p) {
        const u32 i = order[p];
        if (i >= R) {
            bad = true;
            continue;
        }
        const u32 d = need[i], g = n_gpu[i];
        sum_a += d > g ? d - g : 0;
        sum_t += new_tokens[i];
    }
    if (bad) atomicOr(status, CWS_INVAL);
    u64 inc_a = sum_a, inc_t = sum_t;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const u64 ya = shfl64_up(inc_a, d), yt = shfl64_up(inc_t, d);
        if (lane >= (u32)d) {
            inc_a += ya;
            inc_t += yt;
        }
    }
    if (lane == 31) {
        s_a[warp] = inc_a;
        s_t[warp] = inc_t;
    }
    __syncthreads();
    if (warp == 0) {
        const u64 wa = s_a[lane], wt = s_t[lane];
        u64 ia = wa, it = wt;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const u64 ya = shfl64_up(ia, d), yt = shfl64_up(it, d);
            if (lane >= (u32)d) {
                ia += ya;
                it += yt;
            }
        }
        s_a[lane] = ia - wa;  // exclusive
        s_t[lane] = it - wt;
    }
    __syncthreads();
    u64 run_a = s_a[warp] + inc_a - sum_a, run_t = s_t[warp] + inc_t - sum_t;  // sums over everything before `lo`
    const u64 budget = (u64)free_blocks + (u64)evictable;
    u32 cnt = 0;
    u64 last_need = 0;
    for (u32 p = lo; p < hi; ++p) {
        const u32 i = order[p];
        if (i >= R) continue;
        const u32 d = need[i], g = n_gpu[i];
        const u64 a = d > g ? d - g : 0, t = new_tokens[i];
        const bool in = p < max_admit && run_a + a <= budget && run_t < token_budget;  // monotone in p
        u32 chunk = 0;
        if (in) {
            chunk = (u32)min(t, token_budget - run_t);
            ++cnt;
            last_need = run_a + a;
        }
        chunk_tokens[i] = chunk;
        run_a += a;
        run_t += t;
    }
    const u32 wc = __reduce_add_sync(0xffffffffu, cnt);
    const u32 nh = __reduce_max_sync(0xffffffffu, (u32)(last_need >> 32));
    const u32 nl = __reduce_max_sync(0xffffffffu, (u32)(last_need >> 32) == nh ? (u32)last_need : 0u);
    if (lane == 0 && wc) {
        atomicAdd(&s_count, wc);
        atomicMax(&s_need, ((unsigned long long)nh << 32) | nl);
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

int32_t cwi_schedule_init(cw_ctx* ctx) {
    CW_CUDA(ctx, cudaFuncSetAttribute(schedule_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, CWS_TILE * 8));
    return CW_OK;
}

int32_t cwi_schedule(cw_ctx* ctx, u32 R, const u32* d_need, const u32* d_n_gpu, const u64* d_arrival_seq,
                     const u32* d_req_id, u32 policy, u32 free_blocks, u32 evictable, u32 max_admit, u32* d_order,
                     u32* d_num_admit, u32* d_deficit) {
    if (R == 0) {
        schedule_empty_kernel<<<1, 1, 0, ctx->s_main>>>(d_num_admit, d_deficit);
        CW_LAUNCH_CHECK(ctx);
        return CW_OK;
    }
    u32 ipc = (R + ctx->n_sm - 1) / ctx->n_sm;  // elements (warps) per CTA
    ipc = ipc < 8 ? 8 : ipc > CWS_MAX_I ? CWS_MAX_I : ipc;
    const u32 grid = (R + ipc - 1) / ipc;
    size_t smem = (size_t)(R < CWS_TILE ? R : CWS_TILE) * 8;
    if (smem < 512) smem = 512;  // the fast path pads to 128 compressed keys
    schedule_kernel<<<grid, ipc * 32, smem, ctx->s_main>>>(R, d_need, d_n_gpu, d_arrival_seq, d_req_id, policy,
                                                           free_blocks, evictable, max_admit, d_order, ctx->sched_a);
    CW_LAUNCH_CHECK(ctx);
    admit_kernel<<<1, CWA_THREADS, 0, ctx->s_main>>>(R, ctx->sched_a, free_blocks, evictable, max_admit, d_num_admit,
                                                     d_deficit);
    CW_LAUNCH_CHECK(ctx);
    return CW_OK;
}

int32_t cwi_admit_chunked(cw_ctx* ctx, u32 R, const u32* d_order, const u32* d_need, const u32* d_n_gpu,
                          const u32* d_new_tokens, u32 free_blocks, u32 evictable, u32 max_admit, u64 token_budget,
                          u32* d_chunk_tokens, u32* d_num_admit, u32* d_deficit) {
    if (R == 0) {
        schedule_empty_kernel<<<1, 1, 0, ctx->s_main>>>(d_num_admit, d_deficit);
        CW_LAUNCH_CHECK(ctx);
        return CW_OK;
    }
    admit_chunked_kernel<<<1, CWA_THREADS, 0, ctx->s_main>>>(R, d_order, d_need, d_n_gpu, d_new_tokens, free_blocks,
                                                             evictable, max_admit, token_budget, d_chunk_tokens,
                                                             d_num_admit, d_deficit, ctx->d_status);
    CW_LAUNCH_CHECK(ctx);
    return CW_OK;
}
