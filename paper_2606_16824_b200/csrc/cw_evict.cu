// Stage 3 — reuse-aware eviction (cw_score_evict).  DESIGN.md R4 / "Kernels: evict".
//
// ONE persistent kernel (grid = resident CTAs, hand-rolled grid barrier), phases:
//   A  tau_q[s] per session: int32 dot product of uint8 features and int16 weights (PAPER.md 5.2 L217-219:
//      one predicted time-to-next-reuse per session, L252), state overrides (L181, L277)
//   B  per block: evictable? -> 64-bit fixed-point score -> compacted candidate list + histogram of the
//      top 11 bits
//   C  exact k-smallest of the 96-bit key (score : block id) by MSD radix select, 11 bits per pass: bins
//      below the threshold bin are victims, the threshold bin becomes the next candidate list; stops as
//      soon as the candidate list fits one CTA (<= 4096), which sorts it and takes what is still needed
//   D  victims are sorted: 4096-element bitonic runs in shared memory, then a rank merge (each element's
//      final position = its rank in its run + the number of smaller keys in every other run)
//   E  scratch is re-zeroed for the next call (the kernel is self-cleaning => graph-capturable)
// This replaces the paper's eviction heap + rebuild every N_rebuild=3 iterations (L252-254): a full
// re-score and exact selection per call equals popping a heap rebuilt at this instant.
#include <stdio.h>

#include "cw_internal.cuh"

namespace {

#define CWE_THREADS 512
#define CWE_ITEMS 4
#define CWE_TILE (CWE_THREADS * CWE_ITEMS)
#define CWE_SMEM_BYTES (CWE_SORT_RUN * 12)

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
    u32* hist;       // [CWE_PASSES][CWE_BINS]
    u32* counters;   // [0] n_out, [1] barrier count, [2] barrier generation, [4 + p] n_cand of pass p
    u32* status;
    // outputs
    u32* victims;
    u64* victim_scores;
    u32* num_victims;
};

__device__ __forceinline__ void grid_barrier(u32* count, u32* gen, u32 nblocks) {
    __syncthreads();
    if (threadIdx.x == 0) {
        const u32 g = ld_acquire_u32(gen);
        __threadfence();
        if (atomicAdd(count, 1u) == nblocks - 1) {
            *count = 0;
            __threadfence();
            st_release_u32(gen, g + 1);
        } else {
            while (ld_acquire_u32(gen) == g) {
            }
        }
        __threadfence();
    }
    __syncthreads();
}

__device__ __forceinline__ u32 key_digit(u64 score, u32 id, int p) {
    int sh = 96 - CWE_DIGIT_BITS * (p + 1);
    u32 width = CWE_DIGIT_BITS;
    if (sh < 0) {
        width = CWE_DIGIT_BITS + sh;
        sh = 0;
    }
    u64 v;
    if (sh >= 32) v = score >> (sh - 32);
    else v = (score << (32 - sh)) | (u64)(id >> sh);
    return (u32)v & ((1u << width) - 1);
}

__device__ __forceinline__ bool key_lt(u64 s1, u32 i1, u64 s2, u32 i2) { return s1 < s2 || (s1 == s2 && i1 < i2); }

// bitonic sort of N (power of two) (score,id) keys in shared memory, ascending
__device__ void smem_sort(u64* ss, u32* si, u32 N) {
    for (u32 k = 2; k <= N; k <<= 1) {
        for (u32 j = k >> 1; j > 0; j >>= 1) {
            for (u32 t = threadIdx.x; t < (N >> 1); t += CWE_THREADS) {
                const u32 i = ((t & ~(j - 1)) << 1) | (t & (j - 1));
                const u32 p = i | j;
                const bool up = (i & k) == 0;
                const u64 xs = ss[i], ys = ss[p];
                const u32 xi = si[i], yi = si[p];
                if (key_lt(ys, yi, xs, xi) == up) {
                    ss[i] = ys; si[i] = yi;
                    ss[p] = xs; si[p] = xi;
                }
            }
            __syncthreads();
        }
    }
}

// Block-cooperative compaction of one tile: flags f0 (-> list 0) and f1 (-> list 1) per item.
struct TileOffsets {
    u32 base0, base1;
};
__device__ __forceinline__ void tile_append(const bool (&f0)[CWE_ITEMS], const bool (&f1)[CWE_ITEMS],
                                            u32 (&pos0)[CWE_ITEMS], u32 (&pos1)[CWE_ITEMS], u32* ctr0, u32* ctr1,
                                            u32* s_w0, u32* s_w1, u32* s_base) {
    const u32 lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    u32 c0 = 0, c1 = 0;
    u32 r0[CWE_ITEMS], r1[CWE_ITEMS];
#pragma unroll
    for (int k = 0; k < CWE_ITEMS; ++k) {
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
        u32 v0 = lane < CWE_THREADS / 32 ? s_w0[lane] : 0, v1 = lane < CWE_THREADS / 32 ? s_w1[lane] : 0;
        u32 i0 = v0, i1 = v1;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            u32 y0 = __shfl_up_sync(0xffffffffu, i0, d), y1 = __shfl_up_sync(0xffffffffu, i1, d);
            if (lane >= d) {
                i0 += y0;
                i1 += y1;
            }
        }
        if (lane < CWE_THREADS / 32) {
            s_w0[lane] = i0 - v0;
            s_w1[lane] = i1 - v1;
        }
        if (lane == 31) {
            s_base[0] = i0 ? atomicAdd(ctr0, i0) : 0;
            s_base[1] = i1 ? atomicAdd(ctr1, i1) : 0;
        }
    }
    __syncthreads();
    const u32 o0 = s_base[0] + s_w0[warp], o1 = s_base[1] + s_w1[warp];
#pragma unroll
    for (int k = 0; k < CWE_ITEMS; ++k) {
        pos0[k] = o0 + r0[k];
        pos1[k] = o1 + r1[k];
    }
    __syncthreads();  // s_w*/s_base are reused by the next tile
}

__global__ void __launch_bounds__(CWE_THREADS, 2) evict_kernel(const EvictArgs a) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    u32* s_hist = reinterpret_cast<u32*>(smem_raw);                       // phases B/C
    u64* s_score = reinterpret_cast<u64*>(smem_raw);                      // sorts
    u32* s_id = reinterpret_cast<u32*>(smem_raw + CWE_SORT_RUN * 8);
    __shared__ u32 s_w0[CWE_THREADS / 32], s_w1[CWE_THREADS / 32], s_base[2];
    __shared__ u32 s_scan[CWE_THREADS / 32];
    __shared__ u32 s_thr[3];  // threshold bin, count before it, count inside it
    const u32 tid = threadIdx.x, G = gridDim.x;
    u32* n_out = a.counters + 0;
    u32* bar_count = a.counters + 1;
    u32* bar_gen = a.counters + 2;
    u32* n_cand = a.counters + 4;

    // ---------------------------------------------------------------- A: per-session tau
    for (u32 s = blockIdx.x * CWE_THREADS + tid; s < a.S; s += G * CWE_THREADS) {
        const u32 st = a.session_state[s];
        u32 tau;
        if (st == CW_SESSION_QUEUED || st == CW_SESSION_RUNNING) {
            tau = 0;
        } else if (st >= CW_SESSION_IDLE) {
            tau = CW_TAU_MAX;
        } else if (a.tau_override) {
            tau = min(a.tau_override[s], CW_TAU_MAX - 1);
        } else {
            i32 raw = a.bias;
            for (u32 f = 0; f < a.F; ++f) raw += (i32)a.weights[f] * (i32)a.features[(u64)s * a.F + f];
            tau = (u32)min(max(raw, 0), (i32)(CW_TAU_MAX - 1));
        }
        a.tau_q[s] = tau;
    }
    grid_barrier(bar_count, bar_gen, G);

    // ---------------------------------------------------------------- B: score + compact + histogram
    for (u32 i = tid; i < CWE_BINS; i += CWE_THREADS) s_hist[i] = 0;
    __syncthreads();
    for (u32 tile = blockIdx.x; (u64)tile * CWE_TILE < a.M; tile += G) {
        bool f0[CWE_ITEMS], f1[CWE_ITEMS];
        u32 p0[CWE_ITEMS], p1[CWE_ITEMS];
        u64 sc[CWE_ITEMS];
#pragma unroll
        for (int k = 0; k < CWE_ITEMS; ++k) {
            const u32 b = tile * CWE_TILE + k * CWE_THREADS + tid;
            f0[k] = false;
            f1[k] = false;
            sc[k] = 0;
            if (b < a.M) {
                const u32 rf = a.m_ref[b];
                if ((rf & CW_REF_VALID) && !(rf & CW_REF_PINNED) && (rf & 0x3FFFFFFFu) == 0) {
                    const u32 sess = a.m_session[b];
                    const u32 tau = sess < a.S ? a.tau_q[sess] : CW_TAU_MAX;
                    const u32 la = a.m_last[b];
                    const u32 age = min(a.tick_now >= la ? a.tick_now - la : 0u, 0xFFFFFu);
                    const u32 dp = min(a.m_depth[b], 0xFFFFFu);
                    sc[k] = ((u64)(CW_TAU_MAX - tau) << 40) | ((u64)(0xFFFFFu - age) << 20) | (u64)(0xFFFFFu - dp);
                    f0[k] = true;
                    atomicAdd(&s_hist[key_digit(sc[k], b, 0)], 1u);
                }
            }
        }
        tile_append(f0, f1, p0, p1, &n_cand[0], &n_cand[0], s_w0, s_w1, s_base);
#pragma unroll
        for (int k = 0; k < CWE_ITEMS; ++k)
            if (f0[k]) {
                a.cand_score[0][p0[k]] = sc[k];
                a.cand_id[0][p0[k]] = tile * CWE_TILE + k * CWE_THREADS + tid;
            }
    }
    __syncthreads();
    for (u32 i = tid; i < CWE_BINS; i += CWE_THREADS)
        if (s_hist[i]) atomicAdd(&a.hist[i], s_hist[i]);
    grid_barrier(bar_count, bar_gen, G);

    // ---------------------------------------------------------------- C: radix select
    const u32 n_evictable = n_cand[0];
    const u32 asked = min(*a.deficit, a.cap);
    const u32 want = min(asked, n_evictable);
    if (blockIdx.x == 0 && tid == 0) {
        if (n_evictable < asked) atomicOr(a.status, CWS_CAPACITY);
        *a.num_victims = want;
    }
    u32 remaining = want;
    u32 n_cur = n_evictable;
    if (want > 0) {
        for (int p = 0;; ++p) {
            const u64* cs = a.cand_score[p & 1];
            const u32* ci = a.cand_id[p & 1];
            if (n_cur <= CWE_SMALL || p >= CWE_PASSES) {
                // finish in one CTA: sort the candidates, take the first `remaining`
                if (blockIdx.x == 0) {
                    const u32 base = *n_out;
                    for (u32 i = tid; i < CWE_SORT_RUN; i += CWE_THREADS) {
                        s_score[i] = i < n_cur ? cs[i] : ~0ull;
                        s_id[i] = i < n_cur ? ci[i] : 0xFFFFFFFFu;
                    }
                    __syncthreads();
                    smem_sort(s_score, s_id, CWE_SORT_RUN);
                    for (u32 i = tid; i < remaining; i += CWE_THREADS) {
                        a.out_score[base + i] = s_score[i];
                        a.out_id[base + i] = s_id[i];
                    }
                }
                break;
            }
            // threshold bin of this pass (every CTA computes it redundantly from the global histogram)
            {
                const u32* h = a.hist + p * CWE_BINS;
                constexpr int PER = CWE_BINS / CWE_THREADS;
                u32 v[PER], sum = 0;
#pragma unroll
                for (int k = 0; k < PER; ++k) {
                    v[k] = h[tid * PER + k];
                    sum += v[k];
                }
                const u32 lane = tid & 31, warp = tid >> 5;
                u32 inc = sum;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) {
                    u32 y = __shfl_up_sync(0xffffffffu, inc, d);
                    if (lane >= d) inc += y;
                }
                if (lane == 31) s_scan[warp] = inc;
                __syncthreads();
                if (warp == 0) {
                    u32 w = lane < CWE_THREADS / 32 ? s_scan[lane] : 0, wi = w;
#pragma unroll
                    for (int d = 1; d < 32; d <<= 1) {
                        u32 y = __shfl_up_sync(0xffffffffu, wi, d);
                        if (lane >= d) wi += y;
                    }
                    if (lane < CWE_THREADS / 32) s_scan[lane] = wi - w;
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
            const u32 thr = s_thr[0], before = s_thr[1], inside = s_thr[2];
            const u32 need_here = remaining - before;
            const bool take_all = need_here == inside;
            // filter
            for (u32 i = tid; i < CWE_BINS; i += CWE_THREADS) s_hist[i] = 0;
            __syncthreads();
            u64* ns = a.cand_score[(p + 1) & 1];
            u32* ni = a.cand_id[(p + 1) & 1];
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
                        sc[k] = cs[e];
                        id[k] = ci[e];
                        const u32 dg = key_digit(sc[k], id[k], p);
                        if (dg < thr || (take_all && dg == thr)) f0[k] = true;
                        else if (dg == thr) {
                            f1[k] = true;
                            if (p + 1 < CWE_PASSES) atomicAdd(&s_hist[key_digit(sc[k], id[k], p + 1)], 1u);
                        }
                    }
                }
                tile_append(f0, f1, p0, p1, n_out, &n_cand[p + 1], s_w0, s_w1, s_base);
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
            __syncthreads();
            if (p + 1 < CWE_PASSES)
                for (u32 i = tid; i < CWE_BINS; i += CWE_THREADS)
                    if (s_hist[i]) atomicAdd(&a.hist[(p + 1) * CWE_BINS + i], s_hist[i]);
            grid_barrier(bar_count, bar_gen, G);
            if (take_all) {
                remaining = 0;
                break;
            }
            remaining = need_here;
            n_cur = inside;
        }
    }
    grid_barrier(bar_count, bar_gen, G);

    // ---------------------------------------------------------------- E (early): re-zero scratch
    // (nothing reads hist / n_cand / n_out any more: every CTA carries `want` in registers)
    for (u32 i = blockIdx.x * CWE_THREADS + tid; i < CWE_PASSES * CWE_BINS; i += G * CWE_THREADS) a.hist[i] = 0;
    if (blockIdx.x == 0 && tid < 4 + CWE_PASSES + 1 && tid != 1 && tid != 2) a.counters[tid] = 0;

    // ---------------------------------------------------------------- D: sort the victims
    const u32 n_runs = (want + CWE_SORT_RUN - 1) / CWE_SORT_RUN;
    for (u32 run = blockIdx.x; run < n_runs; run += G) {
        const u32 lo = run * CWE_SORT_RUN, len = min((u32)CWE_SORT_RUN, want - lo);
        for (u32 i = tid; i < CWE_SORT_RUN; i += CWE_THREADS) {
            s_score[i] = i < len ? a.out_score[lo + i] : ~0ull;
            s_id[i] = i < len ? a.out_id[lo + i] : 0xFFFFFFFFu;
        }
        __syncthreads();
        smem_sort(s_score, s_id, CWE_SORT_RUN);
        if (n_runs == 1) {
            for (u32 i = tid; i < len; i += CWE_THREADS) {
                a.victims[i] = s_id[i];
                if (a.victim_scores) a.victim_scores[i] = s_score[i];
            }
        } else {
            for (u32 i = tid; i < len; i += CWE_THREADS) {
                a.out_score[lo + i] = s_score[i];
                a.out_id[lo + i] = s_id[i];
            }
        }
        __syncthreads();
    }
    if (n_runs > 1) {
        grid_barrier(bar_count, bar_gen, G);
        for (u32 e = blockIdx.x * CWE_THREADS + tid; e < want; e += G * CWE_THREADS) {
            const u64 s = a.out_score[e];
            const u32 id = a.out_id[e];
            const u32 my_run = e / CWE_SORT_RUN;
            u32 rank = e - my_run * CWE_SORT_RUN;
            for (u32 r = 0; r < n_runs; ++r) {
                if (r == my_run) continue;
                const u32 lo = r * CWE_SORT_RUN, len = min((u32)CWE_SORT_RUN, want - lo);
                u32 l = 0, h = len;  // number of keys of run r below (s,id)
                while (l < h) {
                    const u32 m = (l + h) >> 1;
                    if (key_lt(a.out_score[lo + m], a.out_id[lo + m], s, id)) l = m + 1;
                    else h = m;
                }
                rank += l;
            }
            a.victims[rank] = id;
            if (a.victim_scores) a.victim_scores[rank] = s;
        }
    }
}

int g_evict_grid = 0;

}  // namespace

int32_t cwi_score_evict(cw_ctx* ctx, u32 tick_now, u32 S, u32 F, const uint8_t* d_features, const int16_t* d_weights,
                        i32 bias, const uint8_t* d_session_state, const u32* d_tau_override, const u32* d_deficit,
                        u32 tier, u32* d_victims, u64* d_victim_scores, u32* d_num_victims, u32 cap) {
    if (!g_evict_grid) {
        CW_CUDA(ctx, cudaFuncSetAttribute(evict_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, CWE_SMEM_BYTES));
        int per_sm = 0;
        CW_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, evict_kernel, CWE_THREADS, CWE_SMEM_BYTES));
        if (per_sm < 1) per_sm = 1;
        if (per_sm > 2) per_sm = 2;
        g_evict_grid = per_sm * ctx->n_sm;
    }
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
    a.hist = ctx->hist;
    a.counters = reinterpret_cast<u32*>(ctx->ev);
    a.status = ctx->d_status;
    a.victims = d_victims;
    a.victim_scores = d_victim_scores;
    a.num_victims = d_num_victims;
    // small pools do not need the whole machine (and the grid barrier gets cheaper)
    u32 tiles = (a.M + CWE_TILE - 1) / CWE_TILE;
    int grid = g_evict_grid;
    if ((u32)grid > tiles) grid = tiles ? (int)tiles : 1;
    // cooperative launch: the CTAs wait on one another at the grid barriers, so co-residency must be guaranteed
    void* kargs[] = {&a};
    CW_CUDA(ctx, cudaLaunchCooperativeKernel(reinterpret_cast<const void*>(evict_kernel), dim3(grid), dim3(CWE_THREADS),
                                             kargs, CWE_SMEM_BYTES, ctx->s_main));
    CW_LAUNCH_CHECK(ctx);
    return CW_OK;
}
