// Stage 3 — reuse-aware eviction (cw_score_evict).  DESIGN.md R4 / "Kernels: evict".
//
// ONE cooperative persistent kernel (one CTA per SM, hand-rolled grid barrier), phases:
//   A  tau_q[s] per session: int32 dot product of uint8 features and int16 weights (PAPER.md 5.2 L217-219:
//      one predicted time-to-next-reuse per session, L252), state overrides (L181, L277).  Every CTA
//      computes all sessions into shared memory (S <= 4096), else one grid-wide pass through global memory.
//   B  per block: evictable? -> 64-bit fixed-point score -> compacted candidate list + level-0 histogram
//   C  exact k-smallest of the 96-bit key (score : block id) by MSD radix select, 11 bits per level.  The
//      digit of a level is gathered from the top 11 bits that actually VARY inside the current candidate set
//      (OR / AND masks accumulated while the set is written), so every level splits the set — no wasted
//      levels when thousands of blocks share tau and age.  Bins below the threshold bin are victims, the
//      threshold bin becomes the next candidate set; a set of <= 4096 is finished by one CTA in shared memory
//      (the same levels without grid barriers, then rank counting once <= 256 candidates are left).
//      Histograms use warp-aggregated shared-memory atomics (blocks of one session share a digit).
//   D  victims are ordered by (score, id): one more split on the top 16 bits that vary among the victims
//      (65536 buckets: global histogram, distributed scan, scatter), then every non-empty bucket is finished on its
//      own — up to 128 keys by one warp (bitonic network in its shared-memory chunk, __syncwarp only), up to 4096
//      by one CTA (warp-chunk bitonic + merge-path rounds in shared memory), anything larger by a grid-wide
//      bitonic network (fallback, adversarial keys only).
//      An answer of <= 4096 victims is sorted by one CTA directly.
//   E  scratch is re-zeroed for the next call (the kernel is self-cleaning => graph-capturable)
// This replaces the paper's eviction heap + rebuild every N_rebuild=3 iterations (L252-254): a full
// re-score and exact selection per call equals popping a heap rebuilt at this instant.
#include <stddef.h>
#include <stdio.h>

#include "cw_internal.cuh"

namespace {

#define CWE_THREADS 1024
#define CWE_WARPS (CWE_THREADS / 32)
#define CWE_ITEMS 2  // measured: 2 -> 80 us, 3 -> 82, 4 -> 83, 6 -> 86 (configs[2], whole kernel)
#define CWE_TILE (CWE_THREADS * CWE_ITEMS)
#define CWE_MI 4     // blocks per thread and tile in the passes over the metadata: four CONSECUTIVE blocks, one 128-bit
                     // load per array (64 bytes in flight per thread: a reduced grid is bound by bytes in flight per SM)
#define CWE_MTILE (CWE_THREADS * CWE_MI)
#define CWE_SMEM_SESS 4096                       // sessions whose tau fits the per-CTA shared-memory table
#define CWE_RANK_SESS 512                        // up to here level 0 resolves tau COMPLETELY (digit = rank of the session's tau)
#define CWE_SMEM_SORT (CWE_SORT_RUN * 24)        // two (score,id) buffers of the CTA sort (alias the histogram)
#define CWE_SMEM_BYTES (CWE_SMEM_SORT + CWE_SMEM_SESS * 4)

struct EvictArgs {
    // inputs
    const uint8_t* features;
    const int16_t* weights;
    const uint8_t* session_state;
    const u32* tau_override;
    const u32* deficit;
    const u32* m_session;
    const u32* m_last;
    const u32* m_depth;
    const u32* m_ref;
    u32 tick_now, S, F, M, cap;
    i32 bias;
    // scratch
    u32* tau_q;
    u64* cand_score[2];
    u32* cand_id[2];
    u64* out_score;
    u32* out_id;
    u32* bhist;      // phase D: victims per bucket, exclusive scan, scatter cursors, bucket work lists
    u64* brec;       // phase D: one record per non-empty bucket: first position << 32 | min(size, 0xFFFF) << 16 | bucket
    u32* boff;
    u32* bcur;
    u32* blist;
    u32* hist;       // [CWE_PASSES][CWE_BINS]
    cw_evict_state* st;
    u32* status;
    // outputs
    u32* victims;
    u64* victim_scores;
    u32* num_victims;
};

// Grid barrier of the cooperative launch.  The arrival counter only ever grows: a CTA arrives with ONE
// fire-and-forget release reduction (no returning atomic: 148 returning atomics on one word serialise) and then
// acquire-polls the counter until it reaches `target` = (value at kernel start) + G x (barriers so far).  CTA 0
// records the reached value in bar_gen, where the next launch finds its starting point.  Wrap-safe (signed
// difference of 32-bit counters).
__device__ __forceinline__ void grid_barrier(cw_evict_state* st, u32 nblocks, u32& target) {
    __syncthreads();
    if (threadIdx.x == 0) {
        target += nblocks;
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(&st->bar_count) : "memory");
        while ((i32)(ld_acquire_u32(&st->bar_count) - target) < 0) {
        }
        if (blockIdx.x == 0) st->bar_gen = target;
    }
    __syncthreads();
}

// phase timestamps of the last call (CTA 0 only; read back by cw_debug_evict_times)
__device__ __forceinline__ void stamp(cw_evict_state* st, u32& n) {
#ifdef CW_DEBUG
    if (blockIdx.x == 0 && threadIdx.x == 0 && n < CWE_STAMPS) {
        u64 t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        st->stamps[n] = t;
    }
#endif
    ++n;
}

__device__ __forceinline__ bool key_lt(u64 s1, u32 i1, u64 s2, u32 i2) { return s1 < s2 || (s1 == s2 && i1 < i2); }

// ---- digit plan: up to 11 bit positions of the 96-bit key (95 = MSB of the score, 0 = LSB of the id), descending
#define CWE_BUCKET_BITS 16                       // digit of the victim bucketing (phase D)
#define CWE_BUCKETS (1u << CWE_BUCKET_BITS)
// The chosen positions are stored as RUNS of adjacent bits inside one 32-bit word of the key (word 2 = score
// high, 1 = score low, 0 = id), so that extracting a digit costs one shift-and-mask per run (typically 2-4 runs)
// instead of one per bit.
struct DigitPlan {
    u32 nbits;
    u32 nruns;
    u32 word[CWE_BUCKET_BITS];   // which 32-bit word of the key
    u32 shift[CWE_BUCKET_BITS];  // lowest bit of the run inside that word
    u32 mask[CWE_BUCKET_BITS];   // (1 << run length) - 1
    u32 dst[CWE_BUCKET_BITS];    // position of the run's lowest bit inside the digit
};
template <int MAXBITS = CWE_DIGIT_BITS>
__device__ __forceinline__ u32 plan_digit(const DigitPlan& pl, u64 score, u32 id) {
    const u32 w2 = (u32)(score >> 32), w1 = (u32)score;
    u32 d = 0;
    for (u32 r = 0; r < pl.nruns; ++r) {  // warp-uniform trip count
        const u32 w = pl.word[r] == 2 ? w2 : (pl.word[r] == 1 ? w1 : id);
        d |= ((w >> pl.shift[r]) & pl.mask[r]) << pl.dst[r];
    }
    return d;
}
// the top `maxbits` set bits of (vary_hi : vary_lo); then, if `fill_from` < 96, contiguous bits from there downwards.
// WARP-COOPERATIVE (all 32 lanes of one warp call it with the same arguments): lane i looks at bit i of each of the
// three key words, ballots give the kept bits, every lane that holds the lowest bit of a run writes that run.
__device__ __forceinline__ void make_plan(DigitPlan* pl, u64 vary_hi, u32 vary_lo, u32 fill_from,
                                          u32 maxbits = CWE_DIGIT_BITS) {
    const u32 lane = threadIdx.x & 31;
    const u32 w[3] = {vary_lo, (u32)vary_hi, (u32)(vary_hi >> 32)};
    u32 k[3];
    u32 budget = maxbits;
#pragma unroll
    for (int x = 2; x >= 0; --x) {
        const u32 above = lane == 31 ? 0u : (u32)__popc(w[x] >> (lane + 1));
        k[x] = __ballot_sync(0xffffffffu, ((w[x] >> lane) & 1u) && above < budget);
        budget -= (u32)__popc(k[x]);
    }
    u32 n = maxbits - budget;
    if (fill_from < 96 && n < maxbits) {  // plain bits below every chosen one keep the digit monotone in the key
        const u32 lowest = k[0] ? (u32)__ffs(k[0]) - 1 : k[1] ? 31 + (u32)__ffs(k[1]) : k[2] ? 63 + (u32)__ffs(k[2]) : 96u;
        if (lowest != 0) {
            const u32 p = lowest == 96 ? fill_from : min(fill_from, lowest - 1);
            const u32 cnt = min(maxbits - n, p + 1);
            const u32 lo_p = p + 1 - cnt;
#pragma unroll
            for (int x = 0; x < 3; ++x) {
                const u32 pos = 32 * x + lane;
                k[x] |= __ballot_sync(0xffffffffu, pos >= lo_p && pos <= p);
            }
            n += cnt;
        }
    }
    const u32 below[3] = {0u, (u32)__popc(k[0]), (u32)(__popc(k[0]) + __popc(k[1]))};
    u32 runs = 0;
#pragma unroll
    for (int x = 2; x >= 0; --x) {  // runs of adjacent kept bits inside one 32-bit word
        const u32 kw = k[x];
        const u32 low = kw & ~(kw << 1);
        if ((low >> lane) & 1u) {
            const u32 idx = runs + (lane == 31 ? 0u : (u32)__popc(low >> (lane + 1)));
            const u32 inv = ~(kw >> lane);
            const u32 len = inv ? (u32)__ffs(inv) - 1 : 32 - lane;
            pl->word[idx] = (u32)x;
            pl->shift[idx] = lane;
            pl->mask[idx] = len >= 32 ? 0xFFFFFFFFu : (1u << len) - 1;
            pl->dst[idx] = below[x] + (u32)__popc(kw & ((1u << lane) - 1));
        }
        runs += (u32)__popc(low);
    }
    if (lane == 0) {
        pl->nbits = n;
        pl->nruns = runs;
    }
}

// the key bits a plan reads, as masks over (score : id)
__device__ __forceinline__ void plan_bits(const DigitPlan& pl, u64& hi, u32& lo) {
    hi = 0;
    lo = 0;
    for (u32 r = 0; r < pl.nruns; ++r) {
        const u64 m = (u64)pl.mask[r] << pl.shift[r];
        if (pl.word[r] == 2) hi |= m << 32;
        else if (pl.word[r] == 1) hi |= m;
        else lo |= (u32)m;
    }
}

// CTA sort of N keys (score,id), N a power of two, 128 <= N <= CWE_SORT_RUN, ascending.
//   1. every warp sorts 128-key chunks with a bitonic network in shared memory (__syncwarp only)
//   2. log2(N/128) merge-path rounds between the two buffers: each thread finds its diagonal split by binary
//      search and merges 4 consecutive outputs
// On return (rs, ri) point at the buffer that holds the result.
__device__ void cta_sort(u64* ss, u32* si, u64* ts, u32* ti, u32 N, u64*& rs, u32*& ri) {
    const u32 lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (u32 chunk = warp; chunk < (N >> 7); chunk += CWE_WARPS) {
        u64* cs = ss + (chunk << 7);
        u32* ci = si + (chunk << 7);
        for (u32 k = 2; k <= 128; k <<= 1) {
            for (u32 j = k >> 1; j > 0; j >>= 1) {
#pragma unroll
                for (u32 q = 0; q < 2; ++q) {
                    const u32 t = lane + 32 * q;
                    const u32 i = ((t & ~(j - 1)) << 1) | (t & (j - 1));
                    const u32 p = i | j;
                    const bool up = (i & k) == 0;
                    const u64 xs = cs[i], ys = cs[p];
                    const u32 xi = ci[i], yi = ci[p];
                    if (key_lt(ys, yi, xs, xi) == up) {
                        cs[i] = ys; ci[i] = yi;
                        cs[p] = xs; ci[p] = xi;
                    }
                }
                __syncwarp();
            }
        }
    }
    for (u32 L = 128; L < N; L <<= 1) {
        __syncthreads();
        for (u32 o0 = threadIdx.x * 4; o0 < N; o0 += CWE_THREADS * 4) {
            const u32 pair = o0 / (2 * L), d = o0 - pair * 2 * L;
            const u64* As = ss + pair * 2 * L;
            const u32* Ai = si + pair * 2 * L;
            const u64* Bs = As + L;
            const u32* Bi = Ai + L;
            u32 lo = d > L ? d - L : 0, hi = min(d, L);
            while (lo < hi) {  // how many of the first d outputs come from A
                const u32 mid = (lo + hi) >> 1;
                if (key_lt(As[mid], Ai[mid], Bs[d - 1 - mid], Bi[d - 1 - mid])) lo = mid + 1;
                else hi = mid;
            }
            u32 x = lo, y = d - lo;
#pragma unroll
            for (u32 o = 0; o < 4; ++o) {
                const bool take_a = y >= L || (x < L && key_lt(As[x], Ai[x], Bs[y], Bi[y]));
                ts[o0 + o] = take_a ? As[x] : Bs[y];
                ti[o0 + o] = take_a ? Ai[x] : Bi[y];
                if (take_a) ++x;
                else ++y;
            }
        }
        u64* s_ = ss; ss = ts; ts = s_;
        u32* i_ = si; si = ti; ti = i_;
    }
    __syncthreads();
    rs = ss;
    ri = si;
}
__device__ __forceinline__ u32 sort_size(u32 n) {  // power of two, at least one 128-key chunk
    u32 N = 128;
    while (N < n) N <<= 1;
    return N;
}
// warp-aggregated shared-memory histogram increment (lanes of a warp mostly share a digit)
__device__ __forceinline__ void hist_add(u32* s_hist, bool valid, u32 digit) {
    const u32 act = __ballot_sync(0xffffffffu, valid);
    if (valid) {
        const u32 peers = __match_any_sync(act, digit);
        if ((threadIdx.x & 31) == (u32)__ffs(peers) - 1) atomicAdd(&s_hist[digit], (u32)__popc(peers));
    }
}

// Block-cooperative compaction of one tile: flags f0 (-> list 0) and f1 (-> list 1) per item.
template <int NI>
__device__ __forceinline__ void tile_append(const bool (&f0)[NI], const bool (&f1)[NI],
                                            u32 (&pos0)[NI], u32 (&pos1)[NI], u32* ctr0, u32* ctr1,
                                            u32* s_w0, u32* s_w1, u32* s_base) {
    const u32 lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    u32 c0 = 0, c1 = 0;
    u32 r0[NI], r1[NI];
#pragma unroll
    for (int k = 0; k < NI; ++k) {
        const u32 b0 = __ballot_sync(0xffffffffu, f0[k]);
        const u32 b1 = __ballot_sync(0xffffffffu, f1[k]);
        r0[k] = c0 + __popc(b0 & ((1u << lane) - 1));
        r1[k] = c1 + __popc(b1 & ((1u << lane) - 1));
        c0 += __popc(b0);
        c1 += __popc(b1);
    }
    if (lane == 0) {
        s_w0[warp] = c0;
        s_w1[warp] = c1;
    }
    __syncthreads();
    if (warp == 0) {
        u32 v0 = s_w0[lane], v1 = s_w1[lane];
        u32 i0 = v0, i1 = v1;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            u32 y0 = __shfl_up_sync(0xffffffffu, i0, d), y1 = __shfl_up_sync(0xffffffffu, i1, d);
            if (lane >= d) {
                i0 += y0;
                i1 += y1;
            }
        }
        s_w0[lane] = i0 - v0;
        s_w1[lane] = i1 - v1;
        if (lane == 31) {
            s_base[0] = i0 ? atomicAdd(ctr0, i0) : 0;
            s_base[1] = i1 ? atomicAdd(ctr1, i1) : 0;
        }
    }
    __syncthreads();
    const u32 o0 = s_base[0] + s_w0[warp], o1 = s_base[1] + s_w1[warp];
#pragma unroll
    for (int k = 0; k < NI; ++k) {
        pos0[k] = o0 + r0[k];
        pos1[k] = o1 + r1[k];
    }
    __syncthreads();  // s_w*/s_base are reused by the next tile
}

// block-wide OR of N (u64,u32) pairs of masks into accumulators in global (or shared) memory: hardware warp
// reductions (redux.sync), per-warp partials in shared memory folded by one warp per word, one atomic per CTA and
// word at the target
template <int N>
__device__ __forceinline__ void block_or_n(const u64 (&hi)[N], const u32 (&lo)[N], u64* const (&g_hi)[N],
                                           u32* const (&g_lo)[N], u64* s_hi, u32* s_lo) {
    // s_hi / s_lo hold N x CWE_WARPS per-warp partials (no shared-memory atomics: 32 warps on one word serialise)
    const u32 tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
#pragma unroll
    for (int n = 0; n < N; ++n) {
        const u32 a = __reduce_or_sync(0xffffffffu, (u32)hi[n]);
        const u32 b = __reduce_or_sync(0xffffffffu, (u32)(hi[n] >> 32));
        const u32 c = __reduce_or_sync(0xffffffffu, lo[n]);
        if (lane == 0) {
            s_hi[n * CWE_WARPS + warp] = ((u64)b << 32) | a;
            s_lo[n * CWE_WARPS + warp] = c;
        }
    }
    __syncthreads();
#pragma unroll
    for (int n = 0; n < N; ++n) {
        if (warp == (u32)n) {  // warp n folds word n and issues the one atomic per CTA and word
            const u64 h = s_hi[n * CWE_WARPS + lane];
            const u32 a = __reduce_or_sync(0xffffffffu, (u32)h);
            const u32 b = __reduce_or_sync(0xffffffffu, (u32)(h >> 32));
            const u32 c = __reduce_or_sync(0xffffffffu, s_lo[n * CWE_WARPS + lane]);
            if (lane == 0) {
                if (a | b) atomicOr(reinterpret_cast<unsigned long long*>(g_hi[n]), ((unsigned long long)b << 32) | a);
                if (c) atomicOr(g_lo[n], c);
            }
        }
    }
    __syncthreads();
}
__device__ __forceinline__ void block_or_to_global(u64 hi, u32 lo, u64* g_hi, u32* g_lo, u64* s_hi, u32* s_lo) {
    const u64 h[1] = {hi};
    const u32 l[1] = {lo};
    u64* const gh[1] = {g_hi};
    u32* const gl[1] = {g_lo};
    block_or_n<1>(h, l, gh, gl, s_hi, s_lo);
}

// threshold bin of a level: the bin in which the `remaining`-th smallest candidate falls
template <bool GLOBAL>
__device__ __forceinline__ void find_threshold(const u32* h, u32 remaining, u32* s_scan, u32* s_thr) {
    constexpr int PER = CWE_BINS / CWE_THREADS;
    const u32 tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    u32 v[PER], sum = 0;
#pragma unroll
    for (int k = 0; k < PER; ++k) {
        v[k] = GLOBAL ? __ldcg(h + tid * PER + k) : h[tid * PER + k];
        sum += v[k];
    }
    u32 inc = sum;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        u32 y = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += y;
    }
    if (lane == 31) s_scan[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        u32 w = s_scan[lane], wi = w;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            u32 y = __shfl_up_sync(0xffffffffu, wi, d);
            if (lane >= d) wi += y;
        }
        s_scan[lane] = wi - w;
    }
    __syncthreads();
    u32 run = s_scan[warp] + inc - sum;  // exclusive prefix of this thread's first bin
#pragma unroll
    for (int k = 0; k < PER; ++k) {
        if (run < remaining && remaining <= run + v[k]) {
            s_thr[0] = tid * PER + k;
            s_thr[1] = run;
            s_thr[2] = v[k];
        }
        run += v[k];
    }
    __syncthreads();
}

__device__ __forceinline__ void flush_hist(const u32* s_hist, u32* g_hist) {
    __syncthreads();
    for (u32 i = threadIdx.x; i < CWE_BINS; i += CWE_THREADS)
        if (s_hist[i]) atomicAdd(&g_hist[i], s_hist[i]);
}

__global__ void __launch_bounds__(CWE_THREADS, 1) evict_kernel(const EvictArgs a) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    u32* s_hist = reinterpret_cast<u32*>(smem_raw);                       // phases B/C
    u64* s_score = reinterpret_cast<u64*>(smem_raw);                      // sorts
    u32* s_id = reinterpret_cast<u32*>(smem_raw + CWE_SORT_RUN * 8);
    u64* t_score = reinterpret_cast<u64*>(smem_raw + CWE_SORT_RUN * 12);
    u32* t_id = reinterpret_cast<u32*>(smem_raw + CWE_SORT_RUN * 20);
    u32* s_tau = reinterpret_cast<u32*>(smem_raw + CWE_SMEM_SORT);
    __shared__ u32 s_w0[CWE_WARPS], s_w1[CWE_WARPS], s_base[2];
    __shared__ u32 s_scan[CWE_WARPS];
    __shared__ u32 s_thr[3];  // threshold bin, count before it, count inside it
    __shared__ u64 s_mhi[4 * CWE_WARPS];
    __shared__ u32 s_mlo[4 * CWE_WARPS];
    __shared__ u64 s_acc_hi, s_acc2_hi;
    __shared__ u32 s_acc_lo, s_acc2_lo, s_cnt[2];
    __shared__ DigitPlan s_plan, s_plan2;
    __shared__ unsigned short s_rank[CWE_RANK_SESS];  // level-0 digit of a session in rank mode (<= S)
    const u32 tid = threadIdx.x, G = gridDim.x;
    cw_evict_state* st = a.st;
    const bool tau_smem = a.S <= CWE_SMEM_SESS;
    u32 bar_gen = ld_acquire_u32(&st->bar_gen);  // counter value when the previous launch ended (written by its CTA 0)
    u32 n_stamp = 0;
    stamp(st, n_stamp);

    // the metadata of this CTA's first tile is requested before phase A: its DRAM latency hides behind the tau pass
    u32 rf[CWE_MI], se[CWE_MI], la[CWE_MI], dp[CWE_MI];
    auto load_tile = [&](u32 tile) {
        const u64 b0 = (u64)tile * CWE_MTILE + (u64)tid * CWE_MI;  // four consecutive blocks: 16-byte aligned in every array
        if (b0 + CWE_MI <= a.M) {
            const uint4 r4 = *reinterpret_cast<const uint4*>(a.m_ref + b0);
            const uint4 s4 = *reinterpret_cast<const uint4*>(a.m_session + b0);
            const uint4 l4 = *reinterpret_cast<const uint4*>(a.m_last + b0);
            const uint4 d4 = *reinterpret_cast<const uint4*>(a.m_depth + b0);
            rf[0] = r4.x; rf[1] = r4.y; rf[2] = r4.z; rf[3] = r4.w;
            se[0] = s4.x; se[1] = s4.y; se[2] = s4.z; se[3] = s4.w;
            la[0] = l4.x; la[1] = l4.y; la[2] = l4.z; la[3] = l4.w;
            dp[0] = d4.x; dp[1] = d4.y; dp[2] = d4.z; dp[3] = d4.w;
        } else {
#pragma unroll
            for (int k = 0; k < CWE_MI; ++k) {  // ragged end of the pool (or a tile past it: nothing is loaded)
                const u64 b = b0 + k;
                const bool in = b < a.M;
                rf[k] = in ? a.m_ref[b] : 0u;
                se[k] = in ? a.m_session[b] : 0u;
                la[k] = in ? a.m_last[b] : 0u;
                dp[k] = in ? a.m_depth[b] : 0u;
            }
        }
    };
    load_tile(blockIdx.x);

    // ---------------------------------------------------------------- A: per-session tau
    {
        if (tid == 0) {
            s_acc_hi = 0;
            s_acc_lo = 0;
        }
        __syncthreads();
        u32 t_or = 0, t_nand = 0xFFFFFFu;  // over v = TAU_MAX - tau; v = 0 (idle / unknown session) always counts
        const u32 s0 = tau_smem ? tid : blockIdx.x * CWE_THREADS + tid;
        const u32 sstep = tau_smem ? CWE_THREADS : G * CWE_THREADS;
        for (u32 s = s0; s < a.S; s += sstep) {
            // the predictor inputs are requested together with the session state (one memory latency, not two)
            const u32 stt = a.session_state[s];
            i32 raw = a.bias;
            u32 ov = 0;
            if (a.tau_override) {
                ov = a.tau_override[s];
            } else {
                const uint8_t* x = a.features + (u64)s * a.F;
#pragma unroll
                for (u32 f = 0; f < 16; ++f)  // F <= 16: predicated, independent loads
                    if (f < a.F) raw += (i32)a.weights[f] * (i32)x[f];
            }
            u32 tau;
            if (stt == CW_SESSION_QUEUED || stt == CW_SESSION_RUNNING) tau = 0;
            else if (stt >= CW_SESSION_IDLE) tau = CW_TAU_MAX;
            else if (a.tau_override) tau = min(ov, CW_TAU_MAX - 1);
            else tau = (u32)min(max(raw, 0), (i32)(CW_TAU_MAX - 1));
            if (tau_smem) s_tau[s] = tau;
            else a.tau_q[s] = tau;
            const u32 v = CW_TAU_MAX - tau;
            t_or |= v;
            t_nand |= ~v & 0xFFFFFFu;
        }
        const u64 packed = ((u64)t_or << 32) | t_nand;
        if (tau_smem) {
            block_or_to_global(packed, 0u, &s_acc_hi, &s_acc_lo, s_mhi, s_mlo);
        } else {
            block_or_to_global(packed, 0u, &st->tau_masks, &s_acc_lo, s_mhi, s_mlo);
            grid_barrier(st, G, bar_gen);
            stamp(st, n_stamp);
            if (tid == 0) s_acc_hi = __ldcg(reinterpret_cast<const unsigned long long*>(&st->tau_masks));
            __syncthreads();
        }
        if (tid < 32) {
            const u32 vary_tau = (u32)(s_acc_hi >> 32) & (u32)s_acc_hi & 0xFFFFFFu;
            make_plan(&s_plan, (u64)vary_tau << 40, 0u, 39 + 32);
        }
        __syncthreads();
    }

    // Rank mode (S <= 512): the level-0 digit of a block is the number of sessions whose tau is LARGER than its
    // session's (one prediction per session) — monotone in the score's tau field and injective on it, so
    // level 0 resolves all 24 tau bits at once, whatever their bit patterns, and the threshold set holds ONE tau value.
    const bool rank_mode = tau_smem && a.S <= CWE_RANK_SESS;
    if (rank_mode) {
        for (u32 sidx = tid >> 5; sidx < a.S; sidx += CWE_WARPS) {  // one warp per session, the lanes share the scan
            const u32 mine = s_tau[sidx];
            u32 larger = 0;
            for (u32 j = tid & 31; j < a.S; j += 32) larger += s_tau[j] > mine ? 1u : 0u;
            larger = __reduce_add_sync(0xffffffffu, larger);
            // blocks of an unknown session (id >= S) count as tau = TAU_MAX (digit 0): every real tau below TAU_MAX
            // ranks behind them whether or not a real session sits at TAU_MAX, so that equal taus share a digit and
            // different taus never do
            if ((tid & 31) == 0) s_rank[sidx] = (unsigned short)(larger + (mine < CW_TAU_MAX ? 1u : 0u));
        }
        __syncthreads();
    }
    stamp(st, n_stamp);  // end of phase A
    // ---------------------------------------------------------------- B: score + level-0 histogram
    // Nothing is written here: the candidates are NOT materialised (835 k of the 1 M blocks of configs[2] are evictable:
    // 10 MB out and back, and three block-wide barriers per tile for the compaction).  The level-0 filter re-reads the
    // metadata instead (16 MB, L2-resident by then) and recomputes the scores.  What the pass does collect: the level-0
    // histogram, the number of evictable blocks, and the bits that vary over ALL evictable keys (for the level-1 plan).
    for (u32 i = tid; i < CWE_BINS; i += CWE_THREADS) s_hist[i] = 0;
    __syncthreads();
    auto block_score = [&](u32 k) -> u64 {  // rf/se/la/dp[k] hold the metadata of one evictable block
        const u32 tau = se[k] < a.S ? (tau_smem ? s_tau[se[k]] : __ldcg(a.tau_q + se[k])) : CW_TAU_MAX;
        const u32 age = min(a.tick_now >= la[k] ? a.tick_now - la[k] : 0u, 0xFFFFFu);
        const u32 dpc = min(dp[k], 0xFFFFFu);
        return ((u64)(CW_TAU_MAX - tau) << 40) | ((u64)(0xFFFFFu - age) << 20) | (u64)(0xFFFFFu - dpc);
    };
    auto digit0 = [&](u32 k, u64 sc, u32 b) -> u32 {  // level-0 digit of the block whose metadata sits in slot k
        if (rank_mode) return se[k] < a.S ? (u32)s_rank[se[k]] : 0u;  // unknown session: tau = TAU_MAX, nobody is larger
        return plan_digit(s_plan, sc, b);
    };
    auto evictable = [&](u32 k) -> bool {
        return (rf[k] & CW_REF_VALID) && !(rf[k] & CW_REF_PINNED) && (rf[k] & 0x3FFFFFFFu) == 0;
    };
    {
        u64 a_or_hi = 0, a_nand_hi = 0;
        u32 a_or_lo = 0, a_nand_lo = 0, my_cnt = 0;
        for (u32 tile = blockIdx.x; (u64)tile * CWE_MTILE < a.M; tile += G) {
            if (tile != blockIdx.x) load_tile(tile);
#pragma unroll
            for (int k = 0; k < CWE_MI; ++k) {
                const u32 b = tile * CWE_MTILE + tid * CWE_MI + k;
                const bool ev = evictable(k);
                u64 sc = 0;
                if (ev) {
                    sc = block_score(k);
                    a_or_hi |= sc;
                    a_nand_hi |= ~sc;
                    a_or_lo |= b;
                    a_nand_lo |= ~b;
                    ++my_cnt;
                }
                hist_add(s_hist, ev, ev ? digit0(k, sc, b) : 0u);
            }
        }
        stamp(st, n_stamp);  // CTA 0 done with its tiles
        flush_hist(s_hist, a.hist);
        {
            const u64 h2[2] = {a_or_hi, a_nand_hi};
            const u32 l2[2] = {a_or_lo, a_nand_lo};
            u64* const gh[2] = {&st->all_or_hi, &st->all_nand_hi};
            u32* const gl[2] = {&st->all_or_lo, &st->all_nand_lo};
            block_or_n<2>(h2, l2, gh, gl, s_mhi, s_mlo);
        }
        my_cnt = __reduce_add_sync(0xffffffffu, my_cnt);
        if ((tid & 31) == 0) s_w0[tid >> 5] = my_cnt;
        __syncthreads();
        if (tid < 32) {
            const u32 c = __reduce_add_sync(0xffffffffu, s_w0[tid]);
            if (tid == 0 && c) atomicAdd(&st->n_cand[0], c);
        }
    }
    grid_barrier(st, G, bar_gen);
    stamp(st, n_stamp);

    // ---------------------------------------------------------------- C: radix select
    const u32 n_evictable = __ldcg(&st->n_cand[0]);
    // a.deficit == NULL: speculative selection of the whole eviction budget (cw_score_evict_begin); the deficit
    // is applied — and a shortfall reported — by the trim kernel of cw_score_evict_end
    const u32 asked = a.deficit ? min(*a.deficit, a.cap) : a.cap;
    const u32 want = min(asked, n_evictable);
    if (blockIdx.x == 0 && tid == 0) {
        if (a.deficit && n_evictable < asked) atomicOr(a.status, CWS_CAPACITY);
        *a.num_victims = want;
    }
    u32 remaining = want;
    u32 n_cur = n_evictable;
    int p_first = 0;
    if (want > 0 && n_evictable <= CWE_LOCAL) {
        // small candidate set: materialise it (one more pass over the metadata) and let one CTA finish it below
        for (u32 tile = blockIdx.x; (u64)tile * CWE_MTILE < a.M; tile += G) {
            bool f0[CWE_MI], f1[CWE_MI];
            u32 p0[CWE_MI], p1[CWE_MI];
            u64 sc[CWE_MI];
            load_tile(tile);
#pragma unroll
            for (int k = 0; k < CWE_MI; ++k) {
                f0[k] = evictable(k);
                f1[k] = false;
                sc[k] = f0[k] ? block_score(k) : 0ull;
            }
            tile_append(f0, f1, p0, p1, &st->cursor0, &st->cursor0, s_w0, s_w1, s_base);
#pragma unroll
            for (int k = 0; k < CWE_MI; ++k)
                if (f0[k]) {
                    a.cand_score[0][p0[k]] = sc[k];
                    a.cand_id[0][p0[k]] = tile * CWE_MTILE + tid * CWE_MI + k;
                }
        }
        grid_barrier(st, G, bar_gen);
        stamp(st, n_stamp);
    } else if (want > 0) {
        // ---- level 0, straight from the metadata, FUSED with the level-1 histogram.  The level-1 digit is taken from
        // the bits that vary over all evictable keys and that level 0 did not use (a static plan: it is known before
        // the threshold set exists, so the set's histogram can be built while the set is written: one grid barrier
        // and one pass less than "filter, reduce the masks, barrier, histogram, barrier").
        find_threshold<true>(a.hist, remaining, s_scan, s_thr);
        const u32 thr = s_thr[0], before = s_thr[1], inside = s_thr[2];
        const u32 need_here = remaining - before;
        const bool take_all = need_here == inside;
        const bool next = !take_all && inside > CWE_LOCAL;  // a level-1 pass over the grid will follow
        if (tid < 32) {
            u64 used_hi;
            u32 used_lo;
            plan_bits(s_plan, used_hi, used_lo);
            if (rank_mode) {  // level 0 consumed the whole tau field
                used_hi = 0xFFFFFF0000000000ull;
                used_lo = 0;
            }
            const u64 vh = __ldcg(reinterpret_cast<const unsigned long long*>(&st->all_or_hi)) &
                           __ldcg(reinterpret_cast<const unsigned long long*>(&st->all_nand_hi)) & ~used_hi;
            const u32 vl = __ldcg(&st->all_or_lo) & __ldcg(&st->all_nand_lo) & ~used_lo;
            make_plan(&s_plan2, vh, vl, 96);
        }
        for (u32 i = tid; i < CWE_BINS; i += CWE_THREADS) s_hist[i] = 0;
        __syncthreads();
        stamp(st, n_stamp);  // threshold found
        {
            const DigitPlan& pn = s_plan2;
            u64 m_or_hi = 0, m_nand_hi = 0, v_or_hi = 0, v_nand_hi = 0;  // next candidate set / victims
            u32 m_or_lo = 0, m_nand_lo = 0, v_or_lo = 0, v_nand_lo = 0;
            // The tiles of this pass cost very different amounts (a tile of an idle session appends 4096 entries, most
            // tiles nothing), and a pool that keeps a session's blocks together hands whole tiles of one kind to one
            // CTA: behind the first tile the CTAs therefore draw tickets.  The ticket of the NEXT tile is requested
            // before the current one is processed (its round trip hides behind the tile) and handed round at the end.
            __shared__ u32 s_next_tile;
            u32 tile = blockIdx.x;
            while ((u64)tile * CWE_MTILE < a.M) {
                bool f0[CWE_MI], f1[CWE_MI];
                u32 p0[CWE_MI], p1[CWE_MI];
                u64 sc[CWE_MI];
                u32 nxt = 0;
                if (tid == 0) nxt = G + atomicAdd(&st->tile_cursor, 1u);
                load_tile(tile);
#pragma unroll
                for (int k = 0; k < CWE_MI; ++k) {
                    const u32 b = tile * CWE_MTILE + tid * CWE_MI + k;
                    f0[k] = f1[k] = false;
                    sc[k] = 0;
                    if (evictable(k)) {
                        sc[k] = block_score(k);
                        const u32 dg = digit0(k, sc[k], b);
                        if (dg < thr || (take_all && dg == thr)) {
                            f0[k] = true;
                            v_or_hi |= sc[k];
                            v_nand_hi |= ~sc[k];
                            v_or_lo |= b;
                            v_nand_lo |= ~b;
                        } else if (dg == thr) {
                            f1[k] = true;
                            m_or_hi |= sc[k];
                            m_nand_hi |= ~sc[k];
                            m_or_lo |= b;
                            m_nand_lo |= ~b;
                        }
                    }
                    if (next) hist_add(s_hist, f1[k], f1[k] ? plan_digit(pn, sc[k], b) : 0u);
                }
                {   // most tiles hold neither victims nor candidates (sessions above the threshold): one barrier, not
                    // the three barriers and the scan of an append
                    bool any = false;
#pragma unroll
                    for (int k = 0; k < CWE_MI; ++k) any |= f0[k] | f1[k];
                    if (__syncthreads_or(any)) {
                        tile_append(f0, f1, p0, p1, &st->n_out, &st->n_cand[1], s_w0, s_w1, s_base);
#pragma unroll
                        for (int k = 0; k < CWE_MI; ++k) {
                            const u32 b = tile * CWE_MTILE + tid * CWE_MI + k;
                            if (f0[k]) {
                                a.out_score[p0[k]] = sc[k];
                                a.out_id[p0[k]] = b;
                            } else if (f1[k]) {
                                a.cand_score[1][p1[k]] = sc[k];
                                a.cand_id[1][p1[k]] = b;
                            }
                        }
                    }
                }
                if (tid == 0) s_next_tile = nxt;
                __syncthreads();
                tile = s_next_tile;
                __syncthreads();
            }
            stamp(st, n_stamp);  // CTA 0 done with its filter tiles
            if (next) flush_hist(s_hist, a.hist + CWE_BINS);
            const u64 h4[4] = {v_or_hi, v_nand_hi, next ? m_or_hi : 0ull, next ? m_nand_hi : 0ull};
            const u32 l4[4] = {v_or_lo, v_nand_lo, next ? m_or_lo : 0u, next ? m_nand_lo : 0u};
            u64* const gh[4] = {&st->vic_or_hi, &st->vic_nand_hi, &st->or_hi[1], &st->nand_hi[1]};
            u32* const gl[4] = {&st->vic_or_lo, &st->vic_nand_lo, &st->or_lo[1], &st->nand_lo[1]};
            block_or_n<4>(h4, l4, gh, gl, s_mhi, s_mlo);
        }
        grid_barrier(st, G, bar_gen);
        stamp(st, n_stamp);
        if (take_all) {
            remaining = 0;
        } else {
            remaining = need_here;
            n_cur = inside;
            p_first = 1;
            if (tid < 32) {  // level 1 reads its digits with the static plan
                DigitPlan* d = &s_plan;
                const DigitPlan* c = &s_plan2;
                const u32 lane = tid;
                if (lane < CWE_BUCKET_BITS) {
                    d->word[lane] = c->word[lane];
                    d->shift[lane] = c->shift[lane];
                    d->mask[lane] = c->mask[lane];
                    d->dst[lane] = c->dst[lane];
                }
                if (lane == 0) {
                    d->nbits = c->nbits;
                    d->nruns = c->nruns;
                }
            }
            __syncthreads();
        }
    }
    if (want > 0 && remaining > 0) {
        for (int p = p_first;; ++p) {
            const u64* cs = a.cand_score[p & 1];
            const u32* ci = a.cand_id[p & 1];
            if (n_cur <= CWE_LOCAL || p >= CWE_PASSES) {
                // finish in one CTA, entirely in shared memory: the same radix select without grid barriers,
                // down to <= 256 candidates, then the `remaining` smallest by rank counting
                if (blockIdx.x == 0) {
                    u64 *c_s = s_score, *n_s = t_score;
                    u32 *c_i = s_id, *n_i = t_id;
                    u32* l_hist = s_tau;  // the tau table is dead after phase B
                    const u32 base = __ldcg(&st->n_out);
                    u32 emitted = 0, n = n_cur;
                    u64 v_or_hi = 0, v_nand_hi = 0;
                    u32 v_or_lo = 0, v_nand_lo = 0;
                    __syncthreads();
                    {   // n <= CWE_LOCAL = 4 x CWE_THREADS: all of a thread's loads are issued before the first store
                        // (one memory round trip instead of four on the kernel's single-CTA critical path)
                        static_assert(CWE_LOCAL <= 4 * CWE_THREADS, "local finish loads");
                        u64 ts_[4];
                        u32 ti_[4];
                        const u32 n_ld = min(n, (u32)CWE_LOCAL);
#pragma unroll
                        for (int k = 0; k < 4; ++k) {
                            const u32 i = min(tid + k * CWE_THREADS, n_ld ? n_ld - 1 : 0u);
                            ts_[k] = __ldcg(cs + i);
                            ti_[k] = __ldcg(ci + i);
                        }
#pragma unroll
                        for (int k = 0; k < 4; ++k) {
                            const u32 i = tid + k * CWE_THREADS;
                            if (i < n_ld) {
                                c_s[i] = ts_[k];
                                c_i[i] = ti_[k];
                            }
                        }
                        for (u32 i = tid + 4 * CWE_THREADS; i < n; i += CWE_THREADS) {  // p >= CWE_PASSES fallback only
                            c_s[i] = __ldcg(cs + i);
                            c_i[i] = __ldcg(ci + i);
                        }
                    }
                    for (;;) {
                        __syncthreads();
                        if (n <= CWE_SMALL) {  // 4 threads per candidate
                            const u32 e = tid >> 2, part = tid & 3;
                            u32 rank = 0;
                            u64 ms = 0;
                            u32 mi = 0;
                            if (e < n) {
                                ms = c_s[e];
                                mi = c_i[e];
                                for (u32 o = part; o < n; o += 4) rank += key_lt(c_s[o], c_i[o], ms, mi) ? 1u : 0u;
                            }
                            rank += __shfl_xor_sync(0xffffffffu, rank, 1);
                            rank += __shfl_xor_sync(0xffffffffu, rank, 2);
                            if (e < n && part == 0 && rank < remaining) {
                                a.out_score[base + emitted + rank] = ms;
                                a.out_id[base + emitted + rank] = mi;
                                v_or_hi |= ms;
                                v_nand_hi |= ~ms;
                                v_or_lo |= mi;
                                v_nand_lo |= ~mi;
                            }
                            break;
                        }
                        // bits that vary inside the current set -> digit plan
                        u64 o_hi = 0, x_hi = 0;
                        u32 o_lo = 0, x_lo = 0;
                        for (u32 i = tid; i < n; i += CWE_THREADS) {
                            o_hi |= c_s[i];
                            x_hi |= ~c_s[i];
                            o_lo |= c_i[i];
                            x_lo |= ~c_i[i];
                        }
                        if (tid == 0) {
                            s_acc_hi = 0;
                            s_acc_lo = 0;
                            s_acc2_hi = 0;
                            s_acc2_lo = 0;
                            s_cnt[0] = 0;
                            s_cnt[1] = 0;
                        }
                        for (u32 i = tid; i < CWE_BINS; i += CWE_THREADS) l_hist[i] = 0;
                        __syncthreads();
                        {
                            const u64 h2[2] = {o_hi, x_hi};
                            const u32 l2[2] = {o_lo, x_lo};
                            u64* const gh[2] = {&s_acc_hi, &s_acc2_hi};
                            u32* const gl[2] = {&s_acc_lo, &s_acc2_lo};
                            block_or_n<2>(h2, l2, gh, gl, s_mhi, s_mlo);
                        }
                        if (tid < 32) make_plan(&s_plan, s_acc_hi & s_acc2_hi, s_acc_lo & s_acc2_lo, 96);
                        __syncthreads();
                        const DigitPlan& lp = s_plan;
                        for (u32 i = tid; i < n; i += CWE_THREADS) atomicAdd(&l_hist[plan_digit(lp, c_s[i], c_i[i])], 1u);
                        __syncthreads();
                        find_threshold<false>(l_hist, remaining, s_scan, s_thr);
                        const u32 thr = s_thr[0], before = s_thr[1], inside = s_thr[2];
                        const u32 need_here = remaining - before;
                        const bool take_all = need_here == inside;
                        for (u32 i0 = 0; i0 < n; i0 += CWE_THREADS) {  // warp-uniform trip count
                            const u32 i = i0 + tid;
                            const bool ok = i < n;
                            const u64 ms = ok ? c_s[i] : 0ull;
                            const u32 mi = ok ? c_i[i] : 0u;
                            const u32 dg = ok ? plan_digit(lp, ms, mi) : 0xFFFFFFFFu;
                            const bool out = ok && (dg < thr || (take_all && dg == thr));
                            const bool keep = ok && !out && dg == thr;
                            // one returning shared-memory atomic per warp and list (per-element returning atomics on
                            // one counter serialise: this loop was most of the CTA-local finish)
                            const u32 lane = tid & 31, lt = (1u << lane) - 1;
                            const u32 bo = __ballot_sync(0xffffffffu, out), bk = __ballot_sync(0xffffffffu, keep);
                            u32 po = 0, pk = 0;
                            if (lane == 0) {
                                if (bo) po = atomicAdd(&s_cnt[0], (u32)__popc(bo));
                                if (bk) pk = atomicAdd(&s_cnt[1], (u32)__popc(bk));
                            }
                            po = __shfl_sync(0xffffffffu, po, 0);
                            pk = __shfl_sync(0xffffffffu, pk, 0);
                            if (out) {
                                const u32 pos = base + emitted + po + __popc(bo & lt);
                                a.out_score[pos] = ms;
                                a.out_id[pos] = mi;
                                v_or_hi |= ms;
                                v_nand_hi |= ~ms;
                                v_or_lo |= mi;
                                v_nand_lo |= ~mi;
                            } else if (keep) {
                                const u32 pos = pk + __popc(bk & lt);
                                n_s[pos] = ms;
                                n_i[pos] = mi;
                            }
                        }
                        __syncthreads();
                        if (take_all) break;
                        emitted += before;
                        remaining = need_here;
                        n = inside;
                        u64* ts_ = c_s; c_s = n_s; n_s = ts_;
                        u32* ti_ = c_i; c_i = n_i; n_i = ti_;
                    }
                    __syncthreads();
                    {
                        const u64 h2[2] = {v_or_hi, v_nand_hi};
                        const u32 l2[2] = {v_or_lo, v_nand_lo};
                        u64* const gh[2] = {&st->vic_or_hi, &st->vic_nand_hi};
                        u32* const gl[2] = {&st->vic_or_lo, &st->vic_nand_lo};
                        block_or_n<2>(h2, l2, gh, gl, s_mhi, s_mlo);
                    }
                }
                break;
            }
            // threshold bin of this level (every CTA computes it redundantly from the global histogram)
            find_threshold<true>(a.hist + p * CWE_BINS, remaining, s_scan, s_thr);
            const u32 thr = s_thr[0], before = s_thr[1], inside = s_thr[2];
            const u32 need_here = remaining - before;
            const bool take_all = need_here == inside;
            const DigitPlan& pl = s_plan;
            __syncthreads();
            stamp(st, n_stamp);  // threshold found
            // filter: bins below the threshold are victims, the threshold bin is the next candidate set
            u64* ns = a.cand_score[(p + 1) & 1];
            u32* ni = a.cand_id[(p + 1) & 1];
            u64 m_or_hi = 0, m_nand_hi = 0, v_or_hi = 0, v_nand_hi = 0;  // next candidate set / victims
            u32 m_or_lo = 0, m_nand_lo = 0, v_or_lo = 0, v_nand_lo = 0;
            for (u32 tile = blockIdx.x; (u64)tile * CWE_TILE < n_cur; tile += G) {
                bool f0[CWE_ITEMS], f1[CWE_ITEMS];
                u32 p0[CWE_ITEMS], p1[CWE_ITEMS];
                u64 sc[CWE_ITEMS];
                u32 id[CWE_ITEMS];
#pragma unroll
                for (int k = 0; k < CWE_ITEMS; ++k) {
                    const u32 e = tile * CWE_TILE + k * CWE_THREADS + tid;
                    f0[k] = f1[k] = false;
                    sc[k] = 0;
                    id[k] = 0;
                    if (e < n_cur) {
                        sc[k] = __ldcg(cs + e);
                        id[k] = __ldcg(ci + e);
                        const u32 dg = plan_digit(pl, sc[k], id[k]);
                        if (dg < thr || (take_all && dg == thr)) {
                            f0[k] = true;
                            v_or_hi |= sc[k];
                            v_nand_hi |= ~sc[k];
                            v_or_lo |= id[k];
                            v_nand_lo |= ~id[k];
                        } else if (dg == thr) {
                            f1[k] = true;
                            m_or_hi |= sc[k];
                            m_nand_hi |= ~sc[k];
                            m_or_lo |= id[k];
                            m_nand_lo |= ~id[k];
                        }
                    }
                }
                tile_append(f0, f1, p0, p1, &st->n_out, &st->n_cand[p + 1], s_w0, s_w1, s_base);
#pragma unroll
                for (int k = 0; k < CWE_ITEMS; ++k) {
                    if (f0[k]) {
                        a.out_score[p0[k]] = sc[k];
                        a.out_id[p0[k]] = id[k];
                    } else if (f1[k]) {
                        ns[p1[k]] = sc[k];
                        ni[p1[k]] = id[k];
                    }
                }
            }
            stamp(st, n_stamp);  // CTA 0 done with its filter tiles
            {
                const bool next = !take_all && inside > CWE_LOCAL;  // the next level needs the masks of its set
                const u64 h4[4] = {v_or_hi, v_nand_hi, next ? m_or_hi : 0ull, next ? m_nand_hi : 0ull};
                const u32 l4[4] = {v_or_lo, v_nand_lo, next ? m_or_lo : 0u, next ? m_nand_lo : 0u};
                u64* const gh[4] = {&st->vic_or_hi, &st->vic_nand_hi, &st->or_hi[p + 1], &st->nand_hi[p + 1]};
                u32* const gl[4] = {&st->vic_or_lo, &st->vic_nand_lo, &st->or_lo[p + 1], &st->nand_lo[p + 1]};
                block_or_n<4>(h4, l4, gh, gl, s_mhi, s_mlo);
            }
            grid_barrier(st, G, bar_gen);
            stamp(st, n_stamp);
            if (take_all) {
                remaining = 0;
                break;
            }
            remaining = need_here;
            n_cur = inside;
            if (n_cur <= CWE_LOCAL || p + 1 >= CWE_PASSES) continue;  // finished by one CTA at the top of the loop
            // histogram of the next level over the bits that still vary inside the new candidate set
            if (tid < 32) {
                const u64 vh = __ldcg(reinterpret_cast<const unsigned long long*>(&st->or_hi[p + 1])) &
                               __ldcg(reinterpret_cast<const unsigned long long*>(&st->nand_hi[p + 1]));
                const u32 vl = __ldcg(&st->or_lo[p + 1]) & __ldcg(&st->nand_lo[p + 1]);
                make_plan(&s_plan, vh, vl, 96);
            }
            for (u32 i = tid; i < CWE_BINS; i += CWE_THREADS) s_hist[i] = 0;
            __syncthreads();
            {
                const DigitPlan& pn = s_plan;
                for (u32 base = blockIdx.x * CWE_THREADS; base < n_cur; base += G * CWE_THREADS) {
                    const u32 e = base + tid;
                    const bool ok = e < n_cur;
                    u32 dg = 0;
                    if (ok) dg = plan_digit(pn, __ldcg(ns + e), __ldcg(ni + e));
                    hist_add(s_hist, ok, dg);
                }
            }
            flush_hist(s_hist, a.hist + (p + 1) * CWE_BINS);
            grid_barrier(st, G, bar_gen);
            stamp(st, n_stamp);
        }
    }
    grid_barrier(st, G, bar_gen);
    stamp(st, n_stamp);

    // ---------------------------------------------------------------- E (early): re-zero scratch
    // (nothing reads hist / the selection state any more: every CTA carries `want` in registers)
    for (u32 i = blockIdx.x * CWE_THREADS + tid; i < CWE_PASSES * CWE_BINS; i += G * CWE_THREADS) a.hist[i] = 0;
    // bits that vary among the victims -> digit plan of the bucketing (read before CTA 0 clears the masks)
    if (tid < 32) {
        const u64 vh = __ldcg(reinterpret_cast<const unsigned long long*>(&st->vic_or_hi)) &
                       __ldcg(reinterpret_cast<const unsigned long long*>(&st->vic_nand_hi));
        const u32 vl = __ldcg(&st->vic_or_lo) & __ldcg(&st->vic_nand_lo);
        make_plan(&s_plan, vh, vl, 96, CWE_BUCKET_BITS);
    }
    __syncthreads();
    if (blockIdx.x == 0) {  // keeps bar_count/bar_gen and the ordering-phase words
        u32* w = reinterpret_cast<u32*>(st);
        for (u32 i = 2 + tid; i < offsetof(cw_evict_state, vic_or_hi) / 4; i += CWE_THREADS) w[i] = 0;
        if (tid == 0) {
            st->n_medium = 0;
            st->n_large = 0;
            st->n_nonempty = 0;
        }
    }
    if (want == 0) return;

    // ---------------------------------------------------------------- D: order the victims by (score, id)
    if (want <= CWE_SORT_RUN) {  // small answer: one CTA sorts it (no further grid barrier)
        if (blockIdx.x == 0) {
            const u32 N = sort_size(want);
            __syncthreads();
            for (u32 i = tid; i < N; i += CWE_THREADS) {
                s_score[i] = i < want ? __ldcg(a.out_score + i) : ~0ull;
                s_id[i] = i < want ? __ldcg(a.out_id + i) : 0xFFFFFFFFu;
            }
            __syncthreads();
            u64* rs;
            u32* ri;
            cta_sort(s_score, s_id, t_score, t_id, N, rs, ri);
            for (u32 i = tid; i < want; i += CWE_THREADS) {
                a.victims[i] = ri[i];
                if (a.victim_scores) a.victim_scores[i] = rs[i];
            }
            stamp(st, n_stamp);
            if (tid == 0) {  // the masks were only needed for the bucketed path
                st->stamps[CWE_STAMPS - 1] = n_stamp;
                st->vic_or_hi = 0;
                st->vic_nand_hi = 0;
                st->vic_or_lo = 0;
                st->vic_nand_lo = 0;
            }
        }
        return;
    }
    // D1: bucket = the top 16 bits that vary among the victims (a monotone function of the key), histogram
    const DigitPlan& bp = s_plan;
    //     plus a coarse histogram over the 128 slices of 512 buckets (warp-aggregated), which gives every CTA of D2
    //     the offset of its slice without re-reading the fine histogram
    u32* chist = a.bhist + CWE_BUCKETS;
    // (warp w of CTA c takes the 32 victims at (w * G + c) * 32: the ~1600 busy warps are spread over all SMs)
    for (u32 e = ((tid >> 5) * G + blockIdx.x) * 32 + (tid & 31); e < want; e += G * CWE_THREADS) {
        const u32 dg = plan_digit<CWE_BUCKET_BITS>(bp, __ldcg(a.out_score + e), __ldcg(a.out_id + e));
        // neighbouring victims mostly share a bucket: one atomic per warp and distinct bucket / slice
        const u32 act = __activemask();
        const u32 same = __match_any_sync(act, dg);
        if ((tid & 31) == (u32)__ffs(same) - 1) atomicAdd(&a.bhist[dg], (u32)__popc(same));
        const u32 cg = dg >> 9;
        const u32 peers = __match_any_sync(act, cg);
        if ((tid & 31) == (u32)__ffs(peers) - 1) atomicAdd(&chist[cg], (u32)__popc(peers));
    }
    grid_barrier(st, G, bar_gen);
    stamp(st, n_stamp);
    // D2: exclusive scan of the bucket sizes, every CTA on its own slice of 512 buckets: the offset of the slice
    //     is the sum of the coarse counts of all earlier slices, so no CTA waits for another
    {
        constexpr u32 SLICE = 512;
        const u32 lane = tid & 31, warp = tid >> 5;
        for (u32 sl = blockIdx.x; sl < CWE_BUCKETS / SLICE; sl += G) {
            const u32 first = sl * SLICE;
            const u32 before = tid < sl ? __ldcg(chist + tid) : 0u;  // SLICE == 512 == 1 << 9 (the coarse digit)
            const u32 mine = tid < SLICE ? __ldcg(a.bhist + first + tid) : 0u;
            // block scan of (before: plain sum, mine: inclusive prefix over tid)
            u32 inc = mine, tot = before;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                u32 y = __shfl_up_sync(0xffffffffu, inc, d);
                if (lane >= d) inc += y;
                tot += __shfl_xor_sync(0xffffffffu, tot, d);
            }
            __syncthreads();
            if (lane == 31) s_scan[warp] = inc;
            if (lane == 0) s_w0[warp] = tot;
            __syncthreads();
            if (warp == 0) {
                u32 w = s_scan[lane], wi = w, t2 = s_w0[lane];
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) {
                    u32 y = __shfl_up_sync(0xffffffffu, wi, d);
                    if (lane >= d) wi += y;
                    t2 += __shfl_xor_sync(0xffffffffu, t2, d);
                }
                s_scan[lane] = wi - w;
                if (lane == 0) s_base[0] = t2;
            }
            __syncthreads();
            if (tid < SLICE) {
                const u32 off = s_base[0] + s_scan[warp] + inc - mine;
                a.boff[first + tid] = off;
                a.bcur[first + tid] = off;
            }
            // compact list of the non-empty buckets (order irrelevant): one atomic per warp
            const u32 ne = __ballot_sync(0xffffffffu, mine != 0);
            u32 lbase = 0;
            if (lane == 0 && ne) lbase = atomicAdd(&st->n_nonempty, (u32)__popc(ne));
            lbase = __shfl_sync(0xffffffffu, lbase, 0);
            if (mine != 0)  // everything the bucket's sorter needs in one load
                a.brec[lbase + __popc(ne & ((1u << lane) - 1))] =
                    ((u64)(s_base[0] + s_scan[warp] + inc - mine) << 32) | ((u64)min(mine, 0xFFFFu) << 16) | (first + tid);
        }
        if (blockIdx.x == 0 && tid == 0) {
            a.boff[CWE_BUCKETS] = want;
            st->vic_or_hi = 0;
            st->vic_nand_hi = 0;
            st->vic_or_lo = 0;
            st->vic_nand_lo = 0;
        }
    }
    grid_barrier(st, G, bar_gen);
    stamp(st, n_stamp);
    // D3: scatter into bucket order (inside a bucket the order is arbitrary for now)
    if (blockIdx.x == 0 && tid < CWE_BUCKETS / 512) chist[tid] = 0;  // self-cleaning
    u64* tmp_score = a.cand_score[0];
    u32* tmp_id = a.cand_id[0];
    for (u32 e = ((tid >> 5) * G + blockIdx.x) * 32 + (tid & 31); e < want; e += G * CWE_THREADS) {
        const u64 sc = __ldcg(a.out_score + e);
        const u32 id = __ldcg(a.out_id + e);
        const u32 dg = plan_digit<CWE_BUCKET_BITS>(bp, sc, id);
        const u32 same = __match_any_sync(__activemask(), dg);  // one returning atomic per warp and distinct bucket
        const u32 leader = (u32)__ffs(same) - 1;
        u32 pos = 0;
        if ((tid & 31) == leader) pos = atomicAdd(&a.bcur[dg], (u32)__popc(same));
        pos = __shfl_sync(same, pos, leader) + __popc(same & ((1u << (tid & 31)) - 1));
        tmp_score[pos] = sc;
        tmp_id[pos] = id;
    }
    grid_barrier(st, G, bar_gen);
    stamp(st, n_stamp);
    // D4: one warp per bucket: up to 128 keys are sorted by the warp in its own shared-memory chunk (bitonic,
    //     __syncwarp only) and written to their final place; larger buckets are queued for a CTA sort
    //     (<= 4096) or the grid-wide fallback
    {
        const u32 lane = tid & 31, warp = tid >> 5;
        u64* ws = s_score + warp * 128;
        u32* wi = s_id + warp * 128;
        // warp w of CTA c takes buckets c + G*w, ...: the few thousand busy warps are spread over all SMs
        const u32 gw = warp * G + blockIdx.x, nw = (G * CWE_THREADS) >> 5;
        const u64 rec_first = __ldcg(a.brec + gw);  // speculative (gw < 65536): in flight together with the count
        const u32 n_nonempty = __ldcg(&st->n_nonempty);
        {
          for (u32 q = gw; q < n_nonempty; q += nw) {
            const u64 rec = q == gw ? rec_first : __ldcg(a.brec + q);
            const u32 d = (u32)rec & 0xFFFFu, b0 = (u32)(rec >> 32);
            u32 n = (u32)(rec >> 16) & 0xFFFFu;
            if (n == 0xFFFFu) n = __ldcg(a.boff + d + 1) - b0;  // saturated size field
            if (lane == 0) a.bhist[d] = 0;  // self-cleaning
            if (n == 1) {
                if (lane == 0) {
                    a.victims[b0] = __ldcg(tmp_id + b0);
                    if (a.victim_scores) a.victim_scores[b0] = __ldcg(tmp_score + b0);
                }
            } else if (n <= 128) {
                u32 N = 2;
                while (N < n) N <<= 1;
                __syncwarp();
                for (u32 i = lane; i < N; i += 32) {
                    ws[i] = i < n ? __ldcg(tmp_score + b0 + i) : ~0ull;
                    wi[i] = i < n ? __ldcg(tmp_id + b0 + i) : 0xFFFFFFFFu;
                }
                __syncwarp();
                for (u32 k = 2; k <= N; k <<= 1) {
                    for (u32 j = k >> 1; j > 0; j >>= 1) {
                        for (u32 t = lane; t < (N >> 1); t += 32) {
                            const u32 i = ((t & ~(j - 1)) << 1) | (t & (j - 1));
                            const u32 p = i | j;
                            const bool up = (i & k) == 0;
                            const u64 xs = ws[i], ys = ws[p];
                            const u32 xi = wi[i], yi = wi[p];
                            if (key_lt(ys, yi, xs, xi) == up) {
                                ws[i] = ys; wi[i] = yi;
                                ws[p] = xs; wi[p] = xi;
                            }
                        }
                        __syncwarp();
                    }
                }
                for (u32 i = lane; i < n; i += 32) {
                    a.victims[b0 + i] = wi[i];
                    if (a.victim_scores) a.victim_scores[b0 + i] = ws[i];
                }
            } else if (lane == 0) {
                if (n <= CWE_SORT_RUN) a.blist[atomicAdd(&st->n_medium, 1u)] = d;
                else a.blist[CWE_BUCKETS + atomicAdd(&st->n_large, 1u)] = d;
            }
          }
        }
    }
    grid_barrier(st, G, bar_gen);
    stamp(st, n_stamp);
    // D5: medium buckets, one CTA each
    const u32 n_medium = __ldcg(&st->n_medium), n_large = __ldcg(&st->n_large);
    for (u32 m = blockIdx.x; m < n_medium; m += G) {
        const u32 d = __ldcg(a.blist + m);
        const u32 b0 = __ldcg(a.boff + d), n = __ldcg(a.boff + d + 1) - b0;
        const u32 N = sort_size(n);
        __syncthreads();
        for (u32 i = tid; i < N; i += CWE_THREADS) {
            s_score[i] = i < n ? __ldcg(tmp_score + b0 + i) : ~0ull;
            s_id[i] = i < n ? __ldcg(tmp_id + b0 + i) : 0xFFFFFFFFu;
        }
        __syncthreads();
        u64* rs;
        u32* ri;
        cta_sort(s_score, s_id, t_score, t_id, N, rs, ri);
        for (u32 i = tid; i < n; i += CWE_THREADS) {
            a.victims[b0 + i] = ri[i];
            if (a.victim_scores) a.victim_scores[b0 + i] = rs[i];
        }
    }
    // D6: fallback for a bucket of more than 4096 keys (only when the keys defeat the 16-bit split): bitonic
    //     network for arbitrary n (flip + disperse; partners beyond n count as +inf) in global memory, one grid
    //     barrier per stage
    for (u32 l = 0; l < n_large; ++l) {
        const u32 d = __ldcg(a.blist + CWE_BUCKETS + l);
        const u32 b0 = __ldcg(a.boff + d), n = __ldcg(a.boff + d + 1) - b0;
        u64* ks = tmp_score + b0;
        u32* ki = tmp_id + b0;
        u32 n_pad = 2;
        while (n_pad < n) n_pad <<= 1;
        for (u32 k = 2; k <= n_pad; k <<= 1) {
            for (u32 j = k >> 1; j > 0; j >>= 1) {
                const bool flip = j == (k >> 1);  // first stage of a merge: mirror inside the k-block
                for (u32 t = blockIdx.x * CWE_THREADS + tid; t < (n_pad >> 1); t += G * CWE_THREADS) {
                    const u32 i = ((t & ~(j - 1)) << 1) | (t & (j - 1));  // lower element of the t-th pair
                    const u32 partner = flip ? ((i & ~(k - 1)) | ((k - 1) - (i & (k - 1)))) : i + j;
                    if (partner < n) {  // i < partner; a partner beyond n is +inf: nothing to do
                        const u64 xs = __ldcg(ks + i), ys = __ldcg(ks + partner);
                        const u32 xi = __ldcg(ki + i), yi = __ldcg(ki + partner);
                        if (key_lt(ys, yi, xs, xi)) {
                            ks[i] = ys; ki[i] = yi;
                            ks[partner] = xs; ki[partner] = xi;
                        }
                    }
                }
                grid_barrier(st, G, bar_gen);
                stamp(st, n_stamp);
            }
        }
        for (u32 i = blockIdx.x * CWE_THREADS + tid; i < n; i += G * CWE_THREADS) {
            a.victims[b0 + i] = __ldcg(ki + i);
            if (a.victim_scores) a.victim_scores[b0 + i] = __ldcg(ks + i);
        }
    }
    __syncthreads();
    stamp(st, n_stamp);
    if (blockIdx.x == 0 && tid == 0) st->stamps[CWE_STAMPS - 1] = n_stamp;
}

// cw_score_evict_end: the victims of any deficit are a prefix of the (sorted) victims of the budget
__global__ void evict_trim_kernel(const u32* deficit, u32 cap, const u32* n_budget, u32* num_victims, u32* status) {
    const u32 want = min(*deficit, cap), have = *n_budget;  // have = min(cap, #evictable)
    *num_victims = min(want, have);
    if (have < want) atomicOr(status, CWS_CAPACITY);
}

}  // namespace

int32_t cwi_evict_init(cw_ctx* ctx) {
    CW_CUDA(ctx, cudaFuncSetAttribute(evict_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, CWE_SMEM_BYTES));
    int per_sm = 0;
    CW_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, evict_kernel, CWE_THREADS, CWE_SMEM_BYTES));
    if (per_sm < 1) {
        snprintf(ctx->err, sizeof(ctx->err), "evict_kernel does not fit an SM");
        return CW_E_CUDA;
    }
    ctx->evict_grid = ctx->n_sm;  // one CTA per SM: the cheapest grid barrier
    return CW_OK;
}

int32_t cwi_evict_trim(cw_ctx* ctx, const u32* d_deficit, u32 cap, u32* d_num_victims) {
    evict_trim_kernel<<<1, 1, 0, ctx->s_main>>>(d_deficit, cap, ctx->spec_n, d_num_victims, ctx->d_status);
    CW_LAUNCH_CHECK(ctx);
    return CW_OK;
}

int32_t cwi_score_evict(cw_ctx* ctx, cudaStream_t stream, u32 grid_limit, u32 tick_now, u32 S, u32 F,
                        const uint8_t* d_features, const int16_t* d_weights, i32 bias, const uint8_t* d_session_state,
                        const u32* d_tau_override, const u32* d_deficit, u32 tier, u32* d_victims, u64* d_victim_scores,
                        u32* d_num_victims, u32 cap) {
    EvictArgs a;
    a.features = d_features;
    a.weights = d_weights;
    a.session_state = d_session_state;
    a.tau_override = d_tau_override;
    a.deficit = d_deficit;
    a.m_session = ctx->meta_session[tier];
    a.m_last = ctx->meta_last_access[tier];
    a.m_depth = ctx->meta_depth[tier];
    a.m_ref = ctx->meta_ref_flags[tier];
    a.tick_now = tick_now;
    a.S = S;
    a.F = F;
    a.M = ctx->tier_size[tier];
    a.cap = cap;
    a.bias = bias;
    a.tau_q = ctx->tau_q;
    a.cand_score[0] = ctx->cand_score[0];
    a.cand_score[1] = ctx->cand_score[1];
    a.cand_id[0] = ctx->cand_id[0];
    a.cand_id[1] = ctx->cand_id[1];
    a.out_score = ctx->out_score;
    a.out_id = ctx->out_id;
    a.bhist = ctx->ev_bhist;
    a.brec = ctx->ev_brec;
    a.boff = ctx->ev_boff;
    a.bcur = ctx->ev_bcur;
    a.blist = ctx->ev_blist;
    a.hist = ctx->hist;
    a.st = ctx->ev;
    a.status = ctx->d_status;
    a.victims = d_victims;
    a.victim_scores = d_victim_scores;
    a.num_victims = d_num_victims;
    // small pools do not need the whole machine (and the grid barrier gets cheaper)
    u32 tiles = (u32)(((u64)a.M + CWE_MTILE - 1) / CWE_MTILE);
    int grid = ctx->evict_grid;
    if (grid_limit && (u32)grid > grid_limit) grid = (int)grid_limit;
    if ((u32)grid > tiles) grid = tiles ? (int)tiles : 1;
    // cooperative launch: the CTAs wait on one another at the grid barriers, so co-residency must be guaranteed
    void* kargs[] = {&a};
    CW_CUDA(ctx, cudaLaunchCooperativeKernel(reinterpret_cast<const void*>(evict_kernel), dim3(grid), dim3(CWE_THREADS),
                                             kargs, CWE_SMEM_BYTES, stream));
    CW_LAUNCH_CHECK(ctx);
    return CW_OK;
}
