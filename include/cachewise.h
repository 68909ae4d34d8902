/* cachewise.h — C ABI of the B200-native block-management pass of CacheWise (arxiv/paper_2606_16824).
 *
 * One scheduling step = hash -> match -> schedule -> score/select -> swap (BASELINE.json
 * north_star).  The paper's own implementation of this path is CPU-side Python inside vLLM (PAPER.md L235,
 * 5.3 L250-254, 6.6 L359-365); this library is its data-parallel restatement as sm_100a CUDA kernels.
 *
 * Conventions
 *   - Every call returns int32_t: CW_OK, or a negative CW_E_* code.  No exceptions, no abort.
 *   - `d_*` arguments are DEVICE pointers owned by the caller (16-byte aligned unless stated otherwise);
 *     `h_*` arguments are HOST pointers owned by the caller (page-locked where the comment says "pinned").
 *     The ctx owns only its table, block metadata, scratch and device staging ring.
 *   - Argument checks that need no device data (NULL, alignment, ranges against cw_config) run on the host
 *     before any launch and return CW_E_INVAL with no side effect.
 *   - All work is ASYNCHRONOUS on cfg.stream_main (and cfg.stream_copy for PCIe copies).  Outputs are
 *     valid after cw_sync().  Conditions only the device can detect (table full, fewer evictable blocks
 *     than the deficit, inconsistent offsets) are latched in a device status word and returned — once — by
 *     the next cw_sync() (CW_E_CAPACITY / CW_E_INVAL); outputs are still well defined (see each call).
 *   - The launch sequence of every call is fixed (no host read-back, no data-dependent launch), so a
 *     sequence of calls can be captured into a CUDA graph on stream_main.
 *   - One ctx per host thread; calls on one ctx must not run concurrently.
 */
#ifndef CACHEWISE_H
#define CACHEWISE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CW_OK 0
#define CW_E_INVAL (-1)    /* NULL / misaligned / out-of-range argument, or inconsistent device offsets      */
#define CW_E_CAPACITY (-2) /* table full, or fewer evictable blocks than the requested deficit              */
#define CW_E_CUDA (-3)     /* a CUDA runtime call failed; sticky; text via cw_last_error()                  */
#define CW_E_STATE (-4)    /* ctx misuse (NULL ctx, tier without metadata, staging too small)               */

#define CW_MISS 0xFFFFFFFFu     /* hit_loc / winner_loc value for "not resident"                             */
#define CW_HOST_BIT 0x80000000u /* loc = host-tier slot | CW_HOST_BIT; otherwise loc = HBM block id          */
#define CW_TAU_MAX 0x00FFFFFFu  /* 2^24-1, predictor output range in ms (2.6 h session tail)   */
#define CW_REF_VALID 0x80000000u  /* ref_flags bit 31: block holds a resident page                           */
#define CW_REF_PINNED 0x40000000u /* ref_flags bit 30: pinned (never evictable); bits 0..29 = refcount       */

/* session_state codes (PAPER.md L181 j != i, L277 idle sessions first) */
#define CW_SESSION_TOOL_WAIT 0
#define CW_SESSION_QUEUED 1
#define CW_SESSION_RUNNING 2
#define CW_SESSION_IDLE 3

/* cw_schedule policies (PAPER.md 5.1 L207 / L45+L223 / L281) */
#define CW_POLICY_MIN_ADDITIONAL 0
#define CW_POLICY_OVERLAP_FIRST 1
#define CW_POLICY_FCFS 2

typedef struct cw_ctx cw_ctx;

typedef struct {
    uint32_t num_blocks;       /* M: HBM pool capacity in blocks ("M")                         */
    uint32_t host_slots;       /* host-tier capacity in blocks (0 = no tier)                  */
    uint32_t table_log2_slots; /* >= ceil(log2(2*(M+host_slots))) so that the load factor stays <= 0.5       */
    uint32_t block_tokens;     /* must be 16                                                                */
    uint32_t n_chunks;         /* chunks per KV page = 2*layers (K and V of each layer); 0 = no pool          */
    uint64_t chunk_bytes;      /* block_tokens*kv_heads*head_dim*elt_bytes; multiple of 16                   */
    uint64_t chunk_stride;     /* pool bytes between chunk c and c+1 of one block; multiple of 16            */
    uint64_t block_stride;     /* pool bytes between block b and b+1 inside one chunk; multiple of 16        */
    void* d_pool;              /* caller-owned HBM pool (may be NULL if the swap calls are never used)       */
    uint32_t max_requests;     /* largest R of any call                                                     */
    uint32_t max_sessions;     /* largest S of cw_score_evict                                               */
    uint32_t max_features;     /* largest F of cw_score_evict (<= 16)                                       */
    uint64_t max_hashed_blocks; /* largest hash_off[R] (sum of floor(len_r/16)) of any call                  */
    uint64_t staging_bytes;    /* device staging ring owned by the ctx for cw_swap_out / cw_swap_in
                                  (two halves, each >= one page); 0 = swap calls unavailable                */
    void* stream_main;         /* cudaStream_t, caller-owned; NULL = legacy default stream                   */
    void* stream_copy;         /* cudaStream_t for the PCIe copies; NULL = created and owned by the ctx      */
} cw_config; /* page_bytes = n_chunks*chunk_bytes; byte address of chunk c of block b =
                d_pool + b*block_stride + c*chunk_stride                                                    */

int32_t cw_create(const cw_config* cfg, cw_ctx** out);
int32_t cw_destroy(cw_ctx* ctx);
/* Waits for stream_main and stream_copy, then returns (and clears) the latched device status. */
int32_t cw_sync(cw_ctx* ctx);
/* Orders stream_main after every PCIe copy issued so far on stream_copy (event wait on the device, no host
 * sync): work queued on stream_main afterwards — e.g. the next step's kernels, or a timing event — sees the
 * swap-out data on the host. */
int32_t cw_join_copy(cw_ctx* ctx);
/* Text of the last CW_E_CUDA failure ("" if none).  Valid until the next call on this ctx. */
const char* cw_last_error(cw_ctx* ctx);
#ifdef CW_DEBUG
/* Debug builds only (libcachewise_debug.so, -DCW_DEBUG; not part of the product ABI).  Waits for stream_main, then
 * copies the 32 device timestamps (ns, %globaltimer) that CTA 0 of the last cw_score_evict took after each of its
 * grid-wide phases; h_out32[31] = how many are valid.  Debug builds also reject duplicate block ids in
 * cw_swap_out / cw_gather_pages (CW_E_INVAL at cw_sync; SURVEY.md 8c stage 4). */
int32_t cw_debug_evict_times(cw_ctx* ctx, uint64_t* h_out32);
/* cw_debug_stamp queues a one-thread kernel on stream_main that stores %globaltimer in slot i (< 32); cw_debug_stamps
 * waits and copies the 32 slots: with cw_debug_evict_times (same clock) this gives the timeline of a step's branches. */
int32_t cw_debug_stamp(cw_ctx* ctx, uint32_t i);
int32_t cw_debug_stamps(cw_ctx* ctx, uint64_t* h_out32);
#endif
/* Number of kernels this ctx has launched so far (bench.py's gpu_launches). */
uint64_t cw_launch_count(const cw_ctx* ctx);

/* Stage 1 — chained prefix hashing of every full 16-token block (BASELINE.json stage 1; the paper relies on
 * it, "persist KVCache from previous requests" L60, but never describes it: DESIGN.md reading R1).
 *   d_tokens      int32[tok_off[R]]  token ids, request r = [tok_off[r], tok_off[r+1]); 16-byte aligned base,
 *                 readable up to the next 16-byte boundary past its end (any cudaMalloc allocation is)
 *   d_tok_off     uint64[R+1]
 *   d_start_block uint32[R] or NULL (=0): first block to hash; lower entries of d_hashes are left untouched
 *   d_start_state uint64[R] or NULL: hash of block start_block-1; read only where start_block > 0
 *   d_salt        uint64[R] or NULL (=0): per-request chain seed (e.g. model / LoRA id)
 *   d_hash_off    uint64[R+1]: hash_off[r+1]-hash_off[r] must equal floor(len_r/16)
 *   d_hashes      uint64[hash_off[R]], in-out
 * Device-detected: hash_off inconsistent with tok_off, start_block > n_r, or hash_off[R] > max_hashed_blocks
 * -> CW_E_INVAL at cw_sync; the offending request is skipped. */
int32_t cw_hash_blocks(cw_ctx* ctx, const int32_t* d_tokens, const uint64_t* d_tok_off,
                       const uint32_t* d_start_block, const uint64_t* d_start_state, const uint64_t* d_salt,
                       const uint64_t* d_hash_off, uint32_t R, uint64_t* d_hashes);

/* cw_hash_blocks without a ctx and WITHOUT ANY ALLOCATION — for callers that cannot call cudaMalloc (code under CUDA
 * graph capture, tight serving loops, harnesses that forbid it) and therefore cannot cw_create.  Same operation, same
 * kernel and same argument meaning as cw_hash_blocks (stage 1, reading R1); the scratch a ctx would own
 * (ticket / epoch words, per-CTA hand-over records) is a fixed file-scope device array of about 32 KiB that every
 * GPU loading the library holds until the process exits.  The call issues one 16-byte cudaMemsetAsync and one
 * kernel on `stream`, on the CURRENT device; it calls no cudaMalloc / cudaFree / allocating routine.
 *   R                  at most CW_HASH_STATIC_MAX_REQUESTS, else CW_E_INVAL (and a line on stderr); 0 = no-op
 *   max_hashed_blocks  capacity of d_hashes in blocks: hash_off[R]-hash_off[0] beyond it is reported, nothing written
 *   d_status           uint32 device word or NULL: device-detected conditions (the ones cw_hash_blocks reports at
 *                      cw_sync) are OR-ed into it as a non-zero value; the caller clears and reads it
 *   stream             cudaStream_t; NULL = legacy default stream
 * All calls share the one scratch array: calls that OVERLAP on the GPU (two streams, two graph branches, two host
 * threads) race — serialise them.  The array keeps the last call's contents; the call clears what must start at
 * zero itself. */
#define CW_HASH_STATIC_MAX_REQUESTS 16384u
int32_t cw_hash_blocks_static(const int32_t* d_tokens, const uint64_t* d_tok_off, const uint32_t* d_start_block,
                              const uint64_t* d_start_state, const uint64_t* d_salt, const uint64_t* d_hash_off,
                              uint32_t R, uint64_t max_hashed_blocks, uint64_t* d_hashes, uint32_t* d_status,
                              void* stream);

/* Stage 2a — prefix overlap k_i(t) ("k_i(t) ... already reside in memory", L173 contiguous
 * prefix, Fig. 11B "overlap with KVCache resident on the XPU").  DESIGN.md reading R2.
 *   d_k_total uint32[R]: length of the LEADING run of resident hashes (either tier)
 *   d_n_gpu   uint32[R]: how many blocks of that run are in HBM (= the paper's k_i)
 *   d_hit_loc uint32[hash_off[R]] or NULL: loc of each block of the run; CW_MISS from the first miss on
 * hash_off may be a slice of a longer CSR array (absolute offsets); at most 2^32-1 hashes per call (more ->
 * CW_E_INVAL at cw_sync, outputs untouched). */
int32_t cw_match_prefix(cw_ctx* ctx, const uint64_t* d_hashes, const uint64_t* d_hash_off, uint32_t R,
                        uint32_t* d_k_total, uint32_t* d_n_gpu, uint32_t* d_hit_loc);

/* cw_match_prefix for a queue whose requests SHARE PREFIXES (an agent workload queues many requests of one session:
 * PAPER.md L173 "contiguous prefix", Fig. 11B; configs[2] repeats 5.4 M of its 6.6 M lookups).  Same outputs
 * as cw_match_prefix, bit for bit, under the precondition below; the shared part of a request is looked up once.
 *   d_leader uint32[R]: for request r the index of a request of the same call that is expected to start with the same
 *            hashes (e.g. the longest queued request of r's session; the scheduler knows the session of a request);
 *            d_leader[r] = r for a request that probes on its own.  A hint is only a hint: an index >= R, a
 *            leader that is not its own leader, or a leader that shares nothing costs one search and the request is
 *            probed on its own.
 * PRECONDITION: d_hashes are CHAIN hashes as cw_hash_blocks writes them (the hash of block p is a function of the
 * whole token prefix), so two requests whose hashes agree at position p agree at every position before p.  The
 * length of the shared prefix is found by a search that relies on it; hashes without that property give unspecified
 * (but memory-safe) results — use cw_match_prefix for those. */
int32_t cw_match_prefix_shared(cw_ctx* ctx, const uint64_t* d_hashes, const uint64_t* d_hash_off, uint32_t R,
                               const uint32_t* d_leader, uint32_t* d_k_total, uint32_t* d_n_gpu, uint32_t* d_hit_loc);

/* Stage 2b — prefix-aware scheduling (PAPER.md 5.1 L207 "fewest additional blocks a_i(t)", L177 a_i = d_i-k_i
 * and admission W+a_i <= M, L281 FCFS baseline).  DESIGN.md reading R3.
 *   d_need uint32[R] = d_r = ceil(len_r/16);  a_r = max(d_r - n_gpu_r, 0)
 *   policy 0: (a asc, n_gpu desc, arrival_seq asc, req_id asc); 1: (n_gpu desc, a asc, arrival, req_id);
 *          2: (arrival_seq, req_id).  Remaining ties: input index ascending.
 *   d_order uint32[R]: the permutation (input indices in dispatch order)
 *   d_num_admit, d_deficit: device scalars.  Walk d_order; admit while count < max_admit and
 *          need + a <= free_blocks + evictable; stop at the first misfit; deficit = max(0, need - free_blocks).
 * R must be <= max_requests (the rank sort costs R^2 key comparisons: meant for queues of a few thousand). */
int32_t cw_schedule(cw_ctx* ctx, uint32_t R, const uint32_t* d_need, const uint32_t* d_n_gpu,
                    const uint64_t* d_arrival_seq, const uint32_t* d_req_id, uint32_t policy,
                    uint32_t free_blocks, uint32_t evictable, uint32_t max_admit, uint32_t* d_order,
                    uint32_t* d_num_admit, uint32_t* d_deficit);

/* NEXT-3 — admission under a chunked-prefill token budget (PAPER.md 6.1 L271 "chunked-prefill enabled
 * ... max. 512 tokens per chunk"; reading R8: an engine iteration prefills at most token_budget new tokens).
 * Re-runs the admission walk of cw_schedule over its output d_order: request i (a_i = max(d_i - n_gpu_i, 0) more
 * blocks, d_new_tokens[i] tokens to prefill) is admitted while count < max_admit, need + a_i <= free_blocks +
 * evictable and tokens handed out so far < token_budget; it receives min(d_new_tokens[i], budget left).  Stops at the
 * first request that does not fit.
 *   d_chunk_tokens uint32[R], by INPUT index: tokens each request may prefill this iteration (0 = not admitted, or
 *   nothing to prefill); d_num_admit / d_deficit as in cw_schedule.  d_order[p] >= R -> CW_E_INVAL at cw_sync. */
int32_t cw_admit_chunked(cw_ctx* ctx, uint32_t R, const uint32_t* d_order, const uint32_t* d_need,
                         const uint32_t* d_n_gpu, const uint32_t* d_new_tokens, uint32_t free_blocks,
                         uint32_t evictable, uint32_t max_admit, uint64_t token_budget, uint32_t* d_chunk_tokens,
                         uint32_t* d_num_admit, uint32_t* d_deficit);

/* Stage 3 — reuse-aware eviction (PAPER.md 5.2 L215-219 evict in decreasing predicted time-to-next-reuse,
 * L181 j* = argmax_{j != i} tau_j, L252 unreferenced blocks only and one prediction per session, L277 idle
 * sessions first, L281 LRU fallback).  DESIGN.md reading R4.
 *   tau_q[s]: TOOL_WAIT -> clamp(bias + sum_f w[f]*x[s][f], 0, CW_TAU_MAX-1), or min(tau_override[s],
 *             CW_TAU_MAX-1) when d_tau_override != NULL (CacheWise* "Hint", L285);
 *             QUEUED/RUNNING -> 0;  IDLE (>=3), or a block whose session id >= S -> CW_TAU_MAX
 *   block b of `tier` (metadata set by cw_blocks_update) is evictable iff VALID && !PINNED && refcount==0
 *   score = (CW_TAU_MAX - tau)<<40 | (0xFFFFF - min(tick_now - last_access, 0xFFFFF))<<20
 *           | (0xFFFFF - min(depth, 0xFFFFF))            (tick_now < last_access counts as age 0)
 *   victims = the min(*d_deficit, cap, #evictable) smallest by (score, block id), SORTED ascending.
 *   d_features uint8[S*F] row-major, d_weights int16[F], |bias| <= 2^30, F <= max_features <= 16
 *   d_victims uint32[cap], d_victim_scores uint64[cap] or NULL, d_num_victims device scalar.
 * Device-detected: #evictable < min(*d_deficit, cap) -> all evictable blocks are returned and cw_sync
 * reports CW_E_CAPACITY. */
int32_t cw_score_evict(cw_ctx* ctx, uint32_t tick_now, uint32_t S, uint32_t F, const uint8_t* d_features,
                       const int16_t* d_weights, int32_t bias, const uint8_t* d_session_state,
                       const uint32_t* d_tau_override, const uint32_t* d_deficit, uint32_t tier,
                       uint32_t* d_victims, uint64_t* d_victim_scores, uint32_t* d_num_victims, uint32_t cap);

/* Stage 3, speculative form.  The victims come out SORTED by (score, id), so the victims for any
 * deficit are a PREFIX of the victims for the step's eviction budget `cap`; the selection therefore does not have to
 * wait for cw_schedule's deficit.  cw_score_evict_begin forks: the same kernel as cw_score_evict, with deficit = cap,
 * is launched on a side stream owned by the ctx, ordered after everything queued on stream_main so far; whatever the
 * caller queues on stream_main next (cw_hash_blocks -> cw_match_prefix -> cw_schedule) runs BESIDE it.
 * cw_score_evict_end joins: stream_main waits for the side stream, then
 *     *d_num_victims = min(*d_deficit, cap, #evictable)      (CW_E_CAPACITY latched iff #evictable < min(*d_deficit, cap))
 * i.e. d_victims[0..*d_num_victims), d_victim_scores and the status are exactly those of cw_score_evict; entries of
 * d_victims behind *d_num_victims hold the rest of the budget's victims.  Block metadata, the predictor inputs and
 * the output arrays must not be touched between begin and end.  One begin may be outstanding per ctx (a second one,
 * or an end without a begin, returns CW_E_STATE).  Both calls can be captured into one CUDA graph on stream_main (the
 * side stream joins the capture as a parallel branch).
 *   n_ctas: how many CTAs (= SMs) the speculative kernel may occupy; 0 = library default (a third of the SMs:
 *   measured on configs[2], 44 to 56 of 148 CTAs is where the steady step is shortest — the kernels on stream_main
 *   keep the other two thirds of the machine and both branches end together). */
int32_t cw_score_evict_begin(cw_ctx* ctx, uint32_t tick_now, uint32_t S, uint32_t F, const uint8_t* d_features,
                             const int16_t* d_weights, int32_t bias, const uint8_t* d_session_state,
                             const uint32_t* d_tau_override, uint32_t tier, uint32_t* d_victims,
                             uint64_t* d_victim_scores, uint32_t cap, uint32_t n_ctas);
int32_t cw_score_evict_end(cw_ctx* ctx, const uint32_t* d_deficit, uint32_t* d_num_victims);

/* The paper's own predictor (PAPER.md 5.2 L219-225 "expected remaining time for the tool call to complete",
 * L227 per-cluster distributions of historical tool durations).  DESIGN.md reading R7.
 *   d_cluster    uint32[S]: cluster of the tool call each session is waiting on (its metadata class)
 *   d_elapsed_ms uint32[S]: t - T_i, time since that call was issued
 *   d_sample_off uint64[C+1], d_samples uint32[sample_off[C]]: historical durations (ms) of every cluster, ASCENDING
 *                inside a cluster
 *   d_tau_out    uint32[S]: clamp(floor(mean of the cluster's samples > elapsed) - elapsed, 0, CW_TAU_MAX-1); if no
 *                sample exceeds elapsed (or the cluster is empty): min(elapsed, CW_TAU_MAX-1)
 * The result is meant for cw_score_evict's d_tau_override.  cluster >= C -> tau 0 and CW_E_INVAL at cw_sync. */
int32_t cw_predict_tau(cw_ctx* ctx, uint32_t S, const uint32_t* d_cluster, const uint32_t* d_elapsed_ms, uint32_t C,
                       const uint64_t* d_sample_off, const uint32_t* d_samples, uint32_t* d_tau_out);

/* Stage 4 — paged KV swap (PAPER.md 6.4 L345 "transferred from GPU memory to CPU DRAM and swapped back on
 * demand", Fig. 18).  DESIGN.md reading R5.  A staged page = chunks 0..n_chunks-1 contiguous.
 *
 * cw_swap_out: gather the pages of d_victims[0..n) from the pool into the ctx staging ring (TMA bulk-copy
 * kernel on stream_main) and copy them to pinned host memory (cudaMemcpyAsync on stream_copy), slice by
 * slice so that gather k+1 overlaps copy k.
 *   n = cap if d_num_victims == NULL, else min(*d_num_victims, cap) for the gather while the PCIe copy still
 *   moves cap pages (pages >= n of h_dst are unspecified).
 *   h_host_slots uint32[cap] HOST array or NULL: victim j lands at h_dst + h_host_slots[j]*page_bytes
 *   (NULL: at h_dst + j*page_bytes).  h_dst: pinned. */
int32_t cw_swap_out(cw_ctx* ctx, const uint32_t* d_victims, const uint32_t* d_num_victims, uint32_t cap,
                    const uint32_t* h_host_slots, void* h_dst);
/* cw_swap_in: the exact inverse — page j is read from h_src + (h_host_slots ? h_host_slots[j] : j)*page_bytes
 * and scattered into pool block d_dst_blocks[j]. */
int32_t cw_swap_in(cw_ctx* ctx, const uint32_t* h_host_slots, const void* h_src, const uint32_t* d_dst_blocks,
                   uint32_t n);
/* The device halves of stage 4 alone (HBM-roofline measurement; also what the swap calls launch):
 * d_staged is caller-owned device memory of cap*page_bytes, page j = block d_ids[j]. */
int32_t cw_gather_pages(cw_ctx* ctx, const uint32_t* d_ids, const uint32_t* d_num, uint32_t cap, void* d_staged);
int32_t cw_scatter_pages(cw_ctx* ctx, const uint32_t* d_ids, const uint32_t* d_num, uint32_t cap,
                         const void* d_staged);

/* Support calls (used by the host-driven replay).
 * cw_table_insert: keys 0 and 2^64-1 are remapped to 1 and 2^64-2.  A key already present keeps its loc;
 * among duplicates inside the batch the LOWEST input index wins.  d_winner_loc[i] (may be NULL) = the loc
 * that survives for input i, CW_MISS if the table is full (CW_E_CAPACITY at cw_sync).  When the table fills up
 * the keys that still find a slot are the first ones by input index (a batch that could fill the table is
 * inserted sequentially; deciding that costs one host sync, so such a call cannot be captured: CW_E_STATE).
 * cw_table_erase: absent keys are a no-op.  cw_table_retag: sets loc of present keys (keys must be distinct).
 * cw_table_lookup: d_loc[i] = loc or CW_MISS. */
int32_t cw_table_insert(cw_ctx* ctx, const uint64_t* d_keys, const uint32_t* d_loc, uint32_t n,
                        uint32_t* d_winner_loc);
int32_t cw_table_erase(cw_ctx* ctx, const uint64_t* d_keys, uint32_t n);
int32_t cw_table_retag(cw_ctx* ctx, const uint64_t* d_keys, const uint32_t* d_new_loc, uint32_t n);
int32_t cw_table_lookup(cw_ctx* ctx, const uint64_t* d_keys, uint32_t n, uint32_t* d_loc);
/* Table maintenance (R2b).  Erases leave tombstones; cw_table_erase compacts the table on its own once
 * the erases since the last compaction could have turned a quarter of the slots into tombstones (not while
 * stream_main is being captured).  cw_table_compact forces it: live entries are re-inserted into a second buffer
 * and copied back (the table keeps its address).
 * cw_table_stats: waits for stream_main; h_out8 = { live keys, tombstones, slots, longest probe, median probe, p99
 * probe, compactions so far, sum of probe lengths }, a probe length being the slots examined to find a resident key
 * (lengths above 1024 are counted as 1024 in the median / p99 / sum). */
int32_t cw_table_compact(cw_ctx* ctx);
int32_t cw_table_stats(cw_ctx* ctx, uint64_t* h_out8);
/* cw_blocks_update: scatter per-block metadata of `tier` (0 = HBM blocks, 1 = host slots) at d_ids[0..n);
 * any of the four value arrays may be NULL (= leave unchanged).  PAPER.md 5.3 L250 per-block metadata. */
int32_t cw_blocks_update(cw_ctx* ctx, uint32_t tier, const uint32_t* d_ids, uint32_t n, const uint32_t* d_session,
                         const uint32_t* d_depth, const uint32_t* d_last_access, const uint32_t* d_ref_flags);

#ifdef __cplusplus
}
#endif
#endif /* CACHEWISE_H */
