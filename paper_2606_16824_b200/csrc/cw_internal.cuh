// Internal definitions shared by the CUDA translation units of libcachewise.so (sm_100a only).
// Nothing here is shared with oracle/ (the CPU checker): constants are restated from DESIGN.md R1-R5.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/cachewise.h"

typedef uint64_t u64;
typedef uint32_t u32;
typedef int32_t i32;

// ---- latched device status bits (cw_sync translates them) --------------------------------------------
#define CWS_INVAL 1u
#define CWS_CAPACITY 2u

// ---- stage 1 constants (R1) -------------------------------------------------------------
#define CW_A 0x9E3779B97F4A7C15ull
#define CW_K2 0x6A09E667F3BCC909ull
#define CW_K3 0xBB67AE8584CAA73Bull
#define CW_K5 0x3C6EF372FE94F82Bull
#define CW_K7 0xA54FF53A5F1D36F1ull
#define CW_K11 0x510E527FADE682D1ull

__host__ __device__ constexpr u64 cw_fin(u64 x) {
    x ^= x >> 32;
    x *= CW_K2;
    x ^= x >> 29;
    x *= CW_K3;
    x ^= x >> 32;
    return x;
}
__host__ __device__ constexpr u64 cw_pow(u64 base, u64 e) {
    u64 r = 1;
    while (e) {
        if (e & 1) r *= base;
        base *= base;
        e >>= 1;
    }
    return r;
}

// ---- table (R2): open addressing, linear probing, 16-byte slots -----------------------------
struct __align__(16) cw_slot {
    u64 key;  // 0 = EMPTY, 2^64-1 = TOMBSTONE
    u32 loc;
    u32 idx;  // 0xFFFFFFFF except inside an insert batch (lowest input index of the key)
};
#define CW_KEY_EMPTY 0ull
#define CW_KEY_TOMB 0xFFFFFFFFFFFFFFFFull
#define CW_LOC_PENDING 0xFFFFFFFEu
#define CWT_HIST_BINS 1024  // probe-length histogram of cw_table_stats (longer probes land in the last bin)

__host__ __device__ __forceinline__ u64 cw_remap_key(u64 k) {
    if (k == CW_KEY_EMPTY) return 1ull;
    if (k == CW_KEY_TOMB) return CW_KEY_TOMB - 1;
    return k;
}

// ---- stage 1 launch geometry ---------------------------------------------------------------------------
#define CWH_WARPS 4                   // consumer warps per CTA; each takes a whole unit at a time
#define CWH_K 8                       // consecutive blocks a consumer lane owns inside a unit
#define CWH_UNIT (32 * CWH_K)         // blocks per unit (one unit = one TMA copy = one consumer-warp iteration)
#define CWH_UNIT_LOG2 8
#define CWH_STAGES 4                  // smem ring depth
#define CWH_MIN_CTAS 3
#define CWH_THREADS (32 * (CWH_WARPS + 1))
#define CWH_STAGE_BYTES (CWH_UNIT * 64 + 16)

struct cw_hash_rec {  // what the CTA of one range publishes for the CTA of the next range
    u64 tail;      // chain state after the last block of the range (carry-free if the range is "dependent")
    u32 ready;     // == call epoch once the record is published
    u32 len_kind;  // bit 31: dependent (the whole range lies inside one request begun earlier); low bits: its blocks
};
#define CWH_REC_MID 1u           // the range starts in the middle of a request
#define CWH_REC_TAIL_IS_BSEG 2u  // the whole range lies inside that request
#define CWH_REC_TAIL_OPEN 4u     // the last request of the range continues in the next range

// ---- stage 3 scratch -------------------------------------------------------------------------------
#define CWE_BINS 2048          // 11-bit digits
#define CWE_DIGIT_BITS 11
#define CWE_PASSES 12          // level 0 (tau bits) + at most ceil(96/11) levels over bits that still vary
#define CWE_STAMPS 32
#define CWE_LOCAL 4096         // a candidate set this small is finished by one CTA in shared memory ...
#define CWE_SMALL 256          // ... by radix levels down to this size, then rank counting
#define CWE_SORT_RUN 4096      // victims sorted in runs of this size, then rank-merged

struct cw_evict_state {  // all zero between calls, except the barrier words
    u32 bar_count, bar_gen;           // grid barrier
    u32 n_out;                        // victims emitted so far (unsorted)
    u32 pad0;
    u64 tau_masks;                    // OR of (TAU_MAX-tau) << 32 | OR of its complement (global-tau path)
    u64 all_or_hi, all_nand_hi;       // OR of the scores of ALL evictable blocks / of their complements (level-1 plan)
    u32 all_or_lo, all_nand_lo;       // same for the ids
    u32 cursor0, tile_cursor;         // append cursor of the small-pool materialisation pass; tile tickets of the filter pass
    u32 n_cand[CWE_PASSES + 1];       // candidates of every level
    u32 pad1;
    u32 or_lo[CWE_PASSES + 1], nand_lo[CWE_PASSES + 1];  // OR of the ids / of their complements, per level
    u64 or_hi[CWE_PASSES + 1], nand_hi[CWE_PASSES + 1];  // same for the scores
    // ---- not covered by the early re-zeroing (used by the ordering phase)
    u64 vic_or_hi, vic_nand_hi;       // OR of the victims' scores / of their complements
    u32 vic_or_lo, vic_nand_lo;       // same for the ids
    u32 n_medium, n_large;            // buckets that need a CTA sort / the grid-wide fallback
    u32 n_nonempty, pad2;             // non-empty buckets
    u64 stamps[CWE_STAMPS];           // %globaltimer of CTA 0 after every grid barrier; [last] = how many
};

struct cw_ctx {
    cw_config cfg;
    cudaStream_t s_main, s_copy;
    bool own_copy_stream;
    u64 page_bytes;
    // table
    cw_slot* table;
    u64 n_slots;
    u32* ins_slot;   // scratch: slot index per input of an insert batch
    u32 ins_cap;
    cw_slot* table2;  // second buffer of a compaction (allocated by the first one)
    u32* tbl_cnt;     // device: [0] live keys, [1] tombstones, [2] longest probe of the last stats pass, [3] spare
    u32* tbl_hist;    // device: probe-length histogram of cw_table_stats (CWT_HIST_BINS)
    u64 live_ub;      // host upper bound of the live keys (exact after a refresh)
    u64 tomb_ub;      // host upper bound of the tombstones created since the last compaction
    u64 compactions;
    // metadata SoA, per tier
    u32* meta_session[2];
    u32* meta_last_access[2];
    u32* meta_depth[2];
    u32* meta_ref_flags[2];
    u32 tier_size[2];
    // status
    u32* d_status;
    u32* h_status;  // pinned
    // stage 1
    u64* hash_plan;
    cw_hash_rec* hash_rec;  // hash_grid
    int hash_grid;
    // stage 2a
    u32* m_first_miss;
    u32* m_max_hit;
    u32* m_host_hits;
    u32* m_shared;  // cw_match_prefix_shared: first_miss, max_hit, host_hits, lcp [max_requests each], list length [1]
    u32* m_list;  // cw_match_prefix_shared: (task, request) pairs of the 128-position tasks that hold something to probe
    // stage 2b
    u32* sched_a;       // a of every request in dispatch order (max_requests)
    // stage 3
    u32* tau_q;
    u64* cand_score[2];
    u32* cand_id[2];
    u64* out_score;
    u32* out_id;
    u32* hist;  // CWE_PASSES * CWE_BINS
    cw_evict_state* ev;
    u32* ev_bhist;   // victims per bucket (CWE_BUCKETS) + per slice of 512 buckets (128)
    u32* ev_boff;    // exclusive scan (CWE_BUCKETS + 1)
    u64* ev_brec;    // one record per non-empty bucket (CWE_BUCKETS)
    u32* ev_bcur;    // scatter cursors (CWE_BUCKETS)
    u32* ev_blist;   // [0, 65536): medium buckets, [65536, 131072): large, [131072, 196608): non-empty
    u32 ev_cap;
    int evict_grid;  // CTAs of the cooperative evict launch on THIS device (cw_create)
    // stage 3, speculative form: side stream + fork / join events, victims of the budget, open flag
    cudaStream_t s_side;
    cudaEvent_t ev_fork, ev_spec;
    u32* spec_n;     // device: victims the speculative selection produced (= min(cap, #evictable))
    u32 spec_cap;
    bool spec_open;
    u32* dup_bits;   // CW_DEBUG: one bit per pool block (duplicate check of the gather)
    u64* dbg_stamps; // CW_DEBUG: %globaltimer values written by cw_debug_stamp (32 slots)
    // stage 4
    uint8_t* staging;
    cudaEvent_t ev_gather[2], ev_copy[2], ev_join;
    int copy_grid;
    int n_sm;
    u64 launches;
    char err[256];
};

#define CW_CUDA(ctx, call)                                                                              \
    do {                                                                                                \
        cudaError_t e__ = (call);                                                                       \
        if (e__ != cudaSuccess) {                                                                       \
            snprintf((ctx)->err, sizeof((ctx)->err), "%s:%d %s: %s", __FILE__, __LINE__, #call,         \
                     cudaGetErrorString(e__));                                                          \
            return CW_E_CUDA;                                                                           \
        }                                                                                               \
    } while (0)

#define CW_LAUNCH_CHECK(ctx)                                                                            \
    do {                                                                                                \
        (ctx)->launches++;                                                                              \
        cudaError_t e__ = cudaGetLastError();                                                           \
        if (e__ != cudaSuccess) {                                                                       \
            snprintf((ctx)->err, sizeof((ctx)->err), "%s:%d launch: %s", __FILE__, __LINE__,            \
                     cudaGetErrorString(e__));                                                          \
            return CW_E_CUDA;                                                                           \
        }                                                                                               \
    } while (0)

static inline bool cw_aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; }

// ---- small device helpers ------------------------------------------------------------------------------
__device__ __forceinline__ u64 shfl64(u64 v, int src) {
    u32 lo = __shfl_sync(0xffffffffu, (u32)v, src);
    u32 hi = __shfl_sync(0xffffffffu, (u32)(v >> 32), src);
    return ((u64)hi << 32) | lo;
}
__device__ __forceinline__ u64 shfl64_xor(u64 v, int m) {
    u32 lo = __shfl_xor_sync(0xffffffffu, (u32)v, m);
    u32 hi = __shfl_xor_sync(0xffffffffu, (u32)(v >> 32), m);
    return ((u64)hi << 32) | lo;
}
__device__ __forceinline__ u64 shfl64_up(u64 v, int d) {
    u32 lo = __shfl_up_sync(0xffffffffu, (u32)v, d);
    u32 hi = __shfl_up_sync(0xffffffffu, (u32)(v >> 32), d);
    return ((u64)hi << 32) | lo;
}
__device__ __forceinline__ u32 smem_u32(const void* p) { return (u32)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(u32 bar, u32 count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(u32 bar, u32 bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(u32 bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(u32 bar, u32 parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}
// TMA 1-D bulk copy global -> shared, completion on an mbarrier, L2 evict-first hint for streamed inputs
__device__ __forceinline__ void bulk_g2s(u32 dst, const void* src, u32 bytes, u32 bar, u64 policy) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(dst),
        "l"(src), "r"(bytes), "r"(bar), "l"(policy)
        : "memory");
}
__device__ __forceinline__ void bulk_g2s_plain(u32 dst, const void* src, u32 bytes, u32 bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void bulk_s2g(void* dst, u32 src, u32 bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait_read() {
    asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory");
}
template <int N>
__device__ __forceinline__ void bulk_wait_all() {
    asm volatile("cp.async.bulk.wait_group %0;" ::"n"(N) : "memory");
}
__device__ __forceinline__ u64 policy_evict_first() {
    u64 p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ u32 ld_acquire_u32(const u32* p) {
    u32 v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_u32(u32* p, u32 v) {
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ u64 ld_relaxed_u64(const u64* p) {
    u64 v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}

// per-TU entry points (host side), called from cw_api.cu
int32_t cwi_hash_blocks(cw_ctx*, const i32*, const u64*, const u32*, const u64*, const u64*, const u64*, u32, u64*);
int32_t cwi_match_prefix(cw_ctx*, const u64*, const u64*, u32, u32*, u32*, u32*);
int32_t cwi_match_prefix_shared(cw_ctx*, const u64*, const u64*, u32, const u32*, u32*, u32*, u32*);
int32_t cwi_table_insert(cw_ctx*, const u64*, const u32*, u32, u32*);
int32_t cwi_table_erase(cw_ctx*, const u64*, u32);
int32_t cwi_table_retag(cw_ctx*, const u64*, const u32*, u32);
int32_t cwi_table_lookup(cw_ctx*, const u64*, u32, u32*);
int32_t cwi_schedule(cw_ctx*, u32, const u32*, const u32*, const u64*, const u32*, u32, u32, u32, u32, u32*, u32*,
                     u32*);
// stream: where the kernel runs; grid_limit: CTAs it may use (0 = one per SM); d_deficit == NULL: speculative
// (deficit = cap, no capacity status, *d_num_victims = min(cap, #evictable))
int32_t cwi_score_evict(cw_ctx*, cudaStream_t stream, u32 grid_limit, u32, u32, u32, const uint8_t*, const int16_t*, i32,
                        const uint8_t*, const u32*, const u32*, u32, u32*, u64*, u32*, u32);
int32_t cwi_admit_chunked(cw_ctx*, u32, const u32*, const u32*, const u32*, const u32*, u32, u32, u32, u64, u32*, u32*,
                          u32*);
int32_t cwi_evict_trim(cw_ctx*, const u32* d_deficit, u32 cap, u32* d_num_victims);
int32_t cwi_copy_pages(cw_ctx*, cudaStream_t, const u32* d_ids, const u32* d_num, u32 first, u32 cap, void* d_staged,
                       bool gather);
int32_t cwi_blocks_update(cw_ctx*, u32, const u32*, u32, const u32*, const u32*, const u32*, const u32*);
int32_t cwi_predict_tau(cw_ctx*, u32, const u32*, const u32*, u32, const u64*, const u32*, u32*);
int32_t cwi_table_compact(cw_ctx*);
int32_t cwi_table_stats(cw_ctx*, u64* h_out8);
int cwi_hash_grid(int n_sm);
int cwi_copy_grid(int n_sm);
int32_t cwi_evict_init(cw_ctx*);     // per-device function attributes + cooperative grid size (cw_create)
int32_t cwi_schedule_init(cw_ctx*);  // per-device function attributes (cw_create)
