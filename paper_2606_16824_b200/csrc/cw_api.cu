// C-ABI entry points of libcachewise.so: ctx lifetime, host-side argument checks, and the PCIe legs of
// stage 4.  Every check that needs no device data happens here, before any launch (include/cachewise.h).
#include <stddef.h>
#include <stdio.h>
#include <string.h>

#include <new>

#include "cw_internal.cuh"

namespace {

template <typename T>
cudaError_t dalloc_zero(T** p, size_t n, cudaStream_t s, int fill = 0) {
    *p = nullptr;
    if (n == 0) return cudaSuccess;
    cudaError_t e = cudaMalloc(reinterpret_cast<void**>(p), n * sizeof(T));
    if (e != cudaSuccess) return e;
    return cudaMemsetAsync(*p, fill, n * sizeof(T), s);
}

void free_all(cw_ctx* c) {
    cudaFree(c->table);
    cudaFree(c->table2);
    cudaFree(c->tbl_cnt);
    cudaFree(c->tbl_hist);
    cudaFree(c->ins_slot);
    for (int t = 0; t < 2; ++t) {
        cudaFree(c->meta_session[t]);
        cudaFree(c->meta_last_access[t]);
        cudaFree(c->meta_depth[t]);
        cudaFree(c->meta_ref_flags[t]);
        cudaFree(c->cand_score[t]);
        cudaFree(c->cand_id[t]);
        if (c->ev_gather[t]) cudaEventDestroy(c->ev_gather[t]);
        if (c->ev_copy[t]) cudaEventDestroy(c->ev_copy[t]);
    }
    if (c->ev_join) cudaEventDestroy(c->ev_join);
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    if (c->ev_spec) cudaEventDestroy(c->ev_spec);
    if (c->s_side) cudaStreamDestroy(c->s_side);
    cudaFree(c->spec_n);
    cudaFree(c->dup_bits);
    cudaFree(c->dbg_stamps);
    cudaFree(c->d_status);
    if (c->h_status) cudaFreeHost(c->h_status);
    cudaFree(c->hash_plan);
    cudaFree(c->hash_rec);
    cudaFree(c->m_first_miss);
    cudaFree(c->m_max_hit);
    cudaFree(c->m_host_hits);
    cudaFree(c->m_shared);
    cudaFree(c->m_list);
    cudaFree(c->sched_a);
    cudaFree(c->tau_q);
    cudaFree(c->out_score);
    cudaFree(c->out_id);
    cudaFree(c->hist);
    cudaFree(c->ev);
    cudaFree(c->ev_bhist);
    cudaFree(c->ev_boff);
    cudaFree(c->ev_brec);
    cudaFree(c->ev_bcur);
    cudaFree(c->ev_blist);
    cudaFree(c->staging);
    if (c->own_copy_stream && c->s_copy) cudaStreamDestroy(c->s_copy);
}

}  // namespace

extern "C" {
#pragma GCC visibility push(default)

int32_t cw_create(const cw_config* cfg, cw_ctx** out) {
    if (!cfg || !out) return CW_E_INVAL;
    *out = nullptr;
    if (cfg->block_tokens != 16 || cfg->num_blocks == 0 || cfg->table_log2_slots < 4 || cfg->table_log2_slots > 31 ||
        cfg->max_features > 16 || cfg->max_requests == 0)
        return CW_E_INVAL;
    if ((1ull << cfg->table_log2_slots) < 2ull * ((u64)cfg->num_blocks + cfg->host_slots)) return CW_E_INVAL;
    if (cfg->n_chunks) {
        if (cfg->chunk_bytes == 0 || (cfg->chunk_bytes & 15) || (cfg->chunk_stride & 15) || (cfg->block_stride & 15) ||
            !cfg->d_pool || !cw_aligned16(cfg->d_pool))
            return CW_E_INVAL;
    }
    cw_ctx* c = new (std::nothrow) cw_ctx();
    if (!c) return CW_E_CUDA;
    memset(c, 0, sizeof(*c));
    c->cfg = *cfg;
    c->s_main = static_cast<cudaStream_t>(cfg->stream_main);
    c->page_bytes = (u64)cfg->n_chunks * cfg->chunk_bytes;
    *out = c;  // handed out even on failure so that cw_last_error / cw_destroy work
    int dev = 0;
    cudaDeviceProp prop;
    CW_CUDA(c, cudaGetDevice(&dev));
    CW_CUDA(c, cudaGetDeviceProperties(&prop, dev));
    if (prop.major < 10) {
        snprintf(c->err, sizeof(c->err), "libcachewise is built for sm_100a only; device is sm_%d%d", prop.major,
                 prop.minor);
        return CW_E_CUDA;
    }
    c->n_sm = prop.multiProcessorCount;
    if (cfg->stream_copy) {
        c->s_copy = static_cast<cudaStream_t>(cfg->stream_copy);
    } else {
        CW_CUDA(c, cudaStreamCreateWithFlags(&c->s_copy, cudaStreamNonBlocking));
        c->own_copy_stream = true;
    }
    cudaStream_t s = c->s_main;
    c->n_slots = 1ull << cfg->table_log2_slots;
    CW_CUDA(c, cudaMalloc(reinterpret_cast<void**>(&c->table), c->n_slots * sizeof(cw_slot)));
    {  // EMPTY slots: key 0, loc 0, idx 0xFFFFFFFF
        CW_CUDA(c, cudaMemsetAsync(c->table, 0, c->n_slots * sizeof(cw_slot), s));
        CW_CUDA(c, cudaMemset2DAsync(reinterpret_cast<uint8_t*>(c->table) + 12, sizeof(cw_slot), 0xFF, 4, c->n_slots, s));
    }
    CW_CUDA(c, dalloc_zero(&c->tbl_cnt, 4, s));
    CW_CUDA(c, dalloc_zero(&c->tbl_hist, CWT_HIST_BINS, s));
    c->tier_size[0] = cfg->num_blocks;
    c->tier_size[1] = cfg->host_slots;
    for (int t = 0; t < 2; ++t) {
        CW_CUDA(c, dalloc_zero(&c->meta_session[t], c->tier_size[t], s));
        CW_CUDA(c, dalloc_zero(&c->meta_last_access[t], c->tier_size[t], s));
        CW_CUDA(c, dalloc_zero(&c->meta_depth[t], c->tier_size[t], s));
        CW_CUDA(c, dalloc_zero(&c->meta_ref_flags[t], c->tier_size[t], s));
    }
    CW_CUDA(c, dalloc_zero(&c->d_status, 1, s));
    CW_CUDA(c, cudaHostAlloc(reinterpret_cast<void**>(&c->h_status), sizeof(u32), cudaHostAllocDefault));
    *c->h_status = 0;
    // stage 1
    c->hash_grid = cwi_hash_grid(c->n_sm);
    CW_CUDA(c, dalloc_zero(&c->hash_plan, 4, s));
    CW_CUDA(c, dalloc_zero(&c->hash_rec, (size_t)c->hash_grid, s));
    // stage 2a
    CW_CUDA(c, dalloc_zero(&c->m_first_miss, cfg->max_requests, s, 0xFF));
    CW_CUDA(c, dalloc_zero(&c->m_max_hit, cfg->max_requests, s));
    CW_CUDA(c, dalloc_zero(&c->m_host_hits, cfg->max_requests, s));
    CW_CUDA(c, dalloc_zero(&c->m_shared, 4 * (size_t)cfg->max_requests + 1, s));
    CW_CUDA(c, dalloc_zero(&c->m_list, 2 * ((size_t)(cfg->max_hashed_blocks / 128) + cfg->max_requests + 2), s));
    // stage 2b
    CW_CUDA(c, dalloc_zero(&c->sched_a, cfg->max_requests, s));
    // stage 3
    c->ev_cap = cfg->num_blocks > cfg->host_slots ? cfg->num_blocks : cfg->host_slots;
    CW_CUDA(c, dalloc_zero(&c->tau_q, cfg->max_sessions ? cfg->max_sessions : 1, s));
    for (int t = 0; t < 2; ++t) {
        CW_CUDA(c, dalloc_zero(&c->cand_score[t], c->ev_cap, s));
        CW_CUDA(c, dalloc_zero(&c->cand_id[t], c->ev_cap, s));
    }
    CW_CUDA(c, dalloc_zero(&c->out_score, c->ev_cap, s));
    CW_CUDA(c, dalloc_zero(&c->out_id, c->ev_cap, s));
    CW_CUDA(c, dalloc_zero(&c->hist, (size_t)CWE_PASSES * CWE_BINS, s));
    CW_CUDA(c, dalloc_zero(&c->ev, 1, s));
    CW_CUDA(c, dalloc_zero(&c->ev_bhist, 65536 + 128, s));
    CW_CUDA(c, dalloc_zero(&c->ev_boff, 65537, s));
    CW_CUDA(c, dalloc_zero(&c->ev_brec, 65536, s));
    CW_CUDA(c, dalloc_zero(&c->ev_bcur, 65536, s));
    CW_CUDA(c, dalloc_zero(&c->ev_blist, 196608, s));
    CW_CUDA(c, dalloc_zero(&c->spec_n, 1, s));
    {   // function attributes and launch geometry are per DEVICE: set for the device this ctx lives on
        int32_t st = cwi_evict_init(c);
        if (st) return st;
        st = cwi_schedule_init(c);
        if (st) return st;
    }
    CW_CUDA(c, cudaStreamCreateWithFlags(&c->s_side, cudaStreamNonBlocking));
    CW_CUDA(c, cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming));
    CW_CUDA(c, cudaEventCreateWithFlags(&c->ev_spec, cudaEventDisableTiming));
#ifdef CW_DEBUG
    CW_CUDA(c, dalloc_zero(&c->dup_bits, ((size_t)cfg->num_blocks + 31) / 32, s));
    CW_CUDA(c, dalloc_zero(&c->dbg_stamps, 32, s));
#endif
    // stage 4
    if (cfg->staging_bytes) {
        if (!cfg->n_chunks || cfg->staging_bytes / 2 < c->page_bytes) {
            snprintf(c->err, sizeof(c->err), "staging_bytes must hold two pages");
            return CW_E_STATE;
        }
        CW_CUDA(c, cudaMalloc(reinterpret_cast<void**>(&c->staging), cfg->staging_bytes));
    }
    for (int t = 0; t < 2; ++t) {
        CW_CUDA(c, cudaEventCreateWithFlags(&c->ev_gather[t], cudaEventDisableTiming));
        CW_CUDA(c, cudaEventCreateWithFlags(&c->ev_copy[t], cudaEventDisableTiming));
    }
    CW_CUDA(c, cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming));
    c->copy_grid = cwi_copy_grid(c->n_sm);
    CW_CUDA(c, cudaStreamSynchronize(s));
    CW_CUDA(c, cudaGetLastError());
    return CW_OK;
}

int32_t cw_destroy(cw_ctx* ctx) {
    if (!ctx) return CW_E_STATE;
    cudaStreamSynchronize(ctx->s_main);
    if (ctx->s_copy) cudaStreamSynchronize(ctx->s_copy);
    if (ctx->s_side) cudaStreamSynchronize(ctx->s_side);
    free_all(ctx);
    delete ctx;
    return CW_OK;
}

int32_t cw_sync(cw_ctx* ctx) {
    if (!ctx) return CW_E_STATE;
    CW_CUDA(ctx, cudaStreamSynchronize(ctx->s_copy));
    CW_CUDA(ctx, cudaStreamSynchronize(ctx->s_side));
    CW_CUDA(ctx, cudaMemcpyAsync(ctx->h_status, ctx->d_status, sizeof(u32), cudaMemcpyDeviceToHost, ctx->s_main));
    CW_CUDA(ctx, cudaMemsetAsync(ctx->d_status, 0, sizeof(u32), ctx->s_main));
    CW_CUDA(ctx, cudaStreamSynchronize(ctx->s_main));
    CW_CUDA(ctx, cudaStreamSynchronize(ctx->s_copy));
    const u32 st = *ctx->h_status;
    if (st & CWS_INVAL) return CW_E_INVAL;
    if (st & CWS_CAPACITY) return CW_E_CAPACITY;
    return CW_OK;
}

int32_t cw_join_copy(cw_ctx* ctx) {
    if (!ctx) return CW_E_STATE;
    CW_CUDA(ctx, cudaEventRecord(ctx->ev_join, ctx->s_copy));
    CW_CUDA(ctx, cudaStreamWaitEvent(ctx->s_main, ctx->ev_join, 0));
    return CW_OK;
}

#ifdef CW_DEBUG
__global__ void debug_stamp_kernel(u64* slot) {
    u64 t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    *slot = t;
}
int32_t cw_debug_stamp(cw_ctx* ctx, uint32_t i) {
    if (!ctx) return CW_E_STATE;
    if (i >= 32) return CW_E_INVAL;
    debug_stamp_kernel<<<1, 1, 0, ctx->s_main>>>(ctx->dbg_stamps + i);
    return CW_OK;
}
int32_t cw_debug_stamps(cw_ctx* ctx, uint64_t* h_out32) {
    if (!ctx) return CW_E_STATE;
    if (!h_out32) return CW_E_INVAL;
    CW_CUDA(ctx, cudaStreamSynchronize(ctx->s_main));
    CW_CUDA(ctx, cudaStreamSynchronize(ctx->s_side));
    CW_CUDA(ctx, cudaMemcpy(h_out32, ctx->dbg_stamps, 32 * sizeof(u64), cudaMemcpyDeviceToHost));
    return CW_OK;
}
int32_t cw_debug_evict_times(cw_ctx* ctx, uint64_t* h_out32) {
    if (!ctx) return CW_E_STATE;
    if (!h_out32) return CW_E_INVAL;
    CW_CUDA(ctx, cudaStreamSynchronize(ctx->s_main));
    CW_CUDA(ctx, cudaStreamSynchronize(ctx->s_side));
    CW_CUDA(ctx, cudaMemcpy(h_out32, reinterpret_cast<uint8_t*>(ctx->ev) + offsetof(cw_evict_state, stamps),
                            CWE_STAMPS * sizeof(u64), cudaMemcpyDeviceToHost));
    return CW_OK;
}
#endif

const char* cw_last_error(cw_ctx* ctx) { return ctx ? ctx->err : "null ctx"; }
uint64_t cw_launch_count(const cw_ctx* ctx) { return ctx ? ctx->launches : 0; }

int32_t cw_hash_blocks(cw_ctx* ctx, const int32_t* d_tokens, const uint64_t* d_tok_off, const uint32_t* d_start_block,
                       const uint64_t* d_start_state, const uint64_t* d_salt, const uint64_t* d_hash_off, uint32_t R,
                       uint64_t* d_hashes) {
    if (!ctx) return CW_E_STATE;
    if (R == 0) return CW_OK;
    if (!d_tokens || !d_tok_off || !d_hash_off || !d_hashes || R > ctx->cfg.max_requests) return CW_E_INVAL;
    if (d_start_block && !d_start_state) return CW_E_INVAL;
    if (!cw_aligned16(d_tokens) || (reinterpret_cast<uintptr_t>(d_tok_off) & 7) ||
        (reinterpret_cast<uintptr_t>(d_hash_off) & 7) || (reinterpret_cast<uintptr_t>(d_hashes) & 7))
        return CW_E_INVAL;
    return cwi_hash_blocks(ctx, d_tokens, d_tok_off, d_start_block, d_start_state, d_salt, d_hash_off, R, d_hashes);
}

int32_t cw_match_prefix(cw_ctx* ctx, const uint64_t* d_hashes, const uint64_t* d_hash_off, uint32_t R,
                        uint32_t* d_k_total, uint32_t* d_n_gpu, uint32_t* d_hit_loc) {
    if (!ctx) return CW_E_STATE;
    if (R == 0) return CW_OK;
    if (!d_hashes || !d_hash_off || !d_k_total || !d_n_gpu || R > ctx->cfg.max_requests) return CW_E_INVAL;
    return cwi_match_prefix(ctx, d_hashes, d_hash_off, R, d_k_total, d_n_gpu, d_hit_loc);
}

int32_t cw_match_prefix_shared(cw_ctx* ctx, const uint64_t* d_hashes, const uint64_t* d_hash_off, uint32_t R,
                               const uint32_t* d_leader, uint32_t* d_k_total, uint32_t* d_n_gpu, uint32_t* d_hit_loc) {
    if (!ctx) return CW_E_STATE;
    if (R == 0) return CW_OK;
    if (!d_hashes || !d_hash_off || !d_leader || !d_k_total || !d_n_gpu || R > ctx->cfg.max_requests) return CW_E_INVAL;
    return cwi_match_prefix_shared(ctx, d_hashes, d_hash_off, R, d_leader, d_k_total, d_n_gpu, d_hit_loc);
}

int32_t cw_schedule(cw_ctx* ctx, uint32_t R, const uint32_t* d_need, const uint32_t* d_n_gpu,
                    const uint64_t* d_arrival_seq, const uint32_t* d_req_id, uint32_t policy, uint32_t free_blocks,
                    uint32_t evictable, uint32_t max_admit, uint32_t* d_order, uint32_t* d_num_admit,
                    uint32_t* d_deficit) {
    if (!ctx) return CW_E_STATE;
    if (policy > 2 || !d_num_admit || !d_deficit || R > ctx->cfg.max_requests) return CW_E_INVAL;
    if (R && (!d_need || !d_n_gpu || !d_arrival_seq || !d_req_id || !d_order)) return CW_E_INVAL;
    return cwi_schedule(ctx, R, d_need, d_n_gpu, d_arrival_seq, d_req_id, policy, free_blocks, evictable, max_admit,
                        d_order, d_num_admit, d_deficit);
}

int32_t cw_admit_chunked(cw_ctx* ctx, uint32_t R, const uint32_t* d_order, const uint32_t* d_need,
                         const uint32_t* d_n_gpu, const uint32_t* d_new_tokens, uint32_t free_blocks,
                         uint32_t evictable, uint32_t max_admit, uint64_t token_budget, uint32_t* d_chunk_tokens,
                         uint32_t* d_num_admit, uint32_t* d_deficit) {
    if (!ctx) return CW_E_STATE;
    if (!d_num_admit || !d_deficit || R > ctx->cfg.max_requests) return CW_E_INVAL;
    if (R && (!d_order || !d_need || !d_n_gpu || !d_new_tokens || !d_chunk_tokens)) return CW_E_INVAL;
    return cwi_admit_chunked(ctx, R, d_order, d_need, d_n_gpu, d_new_tokens, free_blocks, evictable, max_admit,
                             token_budget, d_chunk_tokens, d_num_admit, d_deficit);
}

static int32_t check_evict_args(cw_ctx* ctx, uint32_t S, uint32_t F, const uint8_t* d_features,
                                const int16_t* d_weights, int32_t bias, const uint8_t* d_session_state,
                                const uint32_t* d_tau_override, uint32_t tier, const uint32_t* d_victims) {
    if (!ctx) return CW_E_STATE;
    if (tier > 1 || !d_victims) return CW_E_INVAL;
    if (ctx->tier_size[tier] == 0) return CW_E_STATE;
    if (S > ctx->cfg.max_sessions || F > ctx->cfg.max_features || F > 16) return CW_E_INVAL;
    if (bias > (1 << 30) || bias < -(1 << 30)) return CW_E_INVAL;
    if (S && (!d_session_state || (F && !d_tau_override && (!d_features || !d_weights)))) return CW_E_INVAL;
    return CW_OK;
}

int32_t cw_score_evict(cw_ctx* ctx, uint32_t tick_now, uint32_t S, uint32_t F, const uint8_t* d_features,
                       const int16_t* d_weights, int32_t bias, const uint8_t* d_session_state,
                       const uint32_t* d_tau_override, const uint32_t* d_deficit, uint32_t tier, uint32_t* d_victims,
                       uint64_t* d_victim_scores, uint32_t* d_num_victims, uint32_t cap) {
    int32_t st = check_evict_args(ctx, S, F, d_features, d_weights, bias, d_session_state, d_tau_override, tier, d_victims);
    if (st) return st;
    if (!d_deficit || !d_num_victims) return CW_E_INVAL;
    if (ctx->spec_open) return CW_E_STATE;  // the scratch is in use by a speculative selection
    if (cap > ctx->tier_size[tier]) cap = ctx->tier_size[tier];
    return cwi_score_evict(ctx, ctx->s_main, 0, tick_now, S, F, d_features, d_weights, bias, d_session_state,
                           d_tau_override, d_deficit, tier, d_victims, d_victim_scores, d_num_victims, cap);
}

int32_t cw_score_evict_begin(cw_ctx* ctx, uint32_t tick_now, uint32_t S, uint32_t F, const uint8_t* d_features,
                             const int16_t* d_weights, int32_t bias, const uint8_t* d_session_state,
                             const uint32_t* d_tau_override, uint32_t tier, uint32_t* d_victims,
                             uint64_t* d_victim_scores, uint32_t cap, uint32_t n_ctas) {
    int32_t st = check_evict_args(ctx, S, F, d_features, d_weights, bias, d_session_state, d_tau_override, tier, d_victims);
    if (st) return st;
    if (ctx->spec_open) return CW_E_STATE;
    if (cap > ctx->tier_size[tier]) cap = ctx->tier_size[tier];
    // fork: the side stream starts after everything queued on stream_main so far
    CW_CUDA(ctx, cudaEventRecord(ctx->ev_fork, ctx->s_main));
    CW_CUDA(ctx, cudaStreamWaitEvent(ctx->s_side, ctx->ev_fork, 0));
    st = cwi_score_evict(ctx, ctx->s_side, n_ctas ? n_ctas : (u32)(ctx->n_sm + 2) / 3, tick_now, S, F, d_features,
                         d_weights, bias, d_session_state, d_tau_override, nullptr, tier, d_victims, d_victim_scores,
                         ctx->spec_n, cap);
    if (st) return st;
    CW_CUDA(ctx, cudaEventRecord(ctx->ev_spec, ctx->s_side));
    ctx->spec_open = true;
    ctx->spec_cap = cap;
    return CW_OK;
}

int32_t cw_score_evict_end(cw_ctx* ctx, const uint32_t* d_deficit, uint32_t* d_num_victims) {
    if (!ctx) return CW_E_STATE;
    if (!ctx->spec_open) return CW_E_STATE;
    if (!d_deficit || !d_num_victims) return CW_E_INVAL;
    CW_CUDA(ctx, cudaStreamWaitEvent(ctx->s_main, ctx->ev_spec, 0));  // join
    ctx->spec_open = false;
    return cwi_evict_trim(ctx, d_deficit, ctx->spec_cap, d_num_victims);
}

int32_t cw_predict_tau(cw_ctx* ctx, uint32_t S, const uint32_t* d_cluster, const uint32_t* d_elapsed_ms, uint32_t C,
                       const uint64_t* d_sample_off, const uint32_t* d_samples, uint32_t* d_tau_out) {
    if (!ctx) return CW_E_STATE;
    if (S == 0) return CW_OK;
    if (!d_cluster || !d_elapsed_ms || !d_sample_off || !d_tau_out || (C && !d_samples)) return CW_E_INVAL;
    return cwi_predict_tau(ctx, S, d_cluster, d_elapsed_ms, C, d_sample_off, d_samples, d_tau_out);
}

int32_t cw_gather_pages(cw_ctx* ctx, const uint32_t* d_ids, const uint32_t* d_num, uint32_t cap, void* d_staged) {
    if (!ctx) return CW_E_STATE;
    if (!ctx->cfg.n_chunks) return CW_E_STATE;
    if (cap == 0) return CW_OK;
    if (!d_ids || !d_staged || !cw_aligned16(d_staged)) return CW_E_INVAL;
    return cwi_copy_pages(ctx, ctx->s_main, d_ids, d_num, 0, cap, d_staged, true);
}

int32_t cw_scatter_pages(cw_ctx* ctx, const uint32_t* d_ids, const uint32_t* d_num, uint32_t cap,
                         const void* d_staged) {
    if (!ctx) return CW_E_STATE;
    if (!ctx->cfg.n_chunks) return CW_E_STATE;
    if (cap == 0) return CW_OK;
    if (!d_ids || !d_staged || !cw_aligned16(d_staged)) return CW_E_INVAL;
    return cwi_copy_pages(ctx, ctx->s_main, d_ids, d_num, 0, cap, const_cast<void*>(d_staged), false);
}

// One PCIe leg of a slice: pages [first, first+cnt) between the staging half and host memory.
static int32_t pcie_slice(cw_ctx* ctx, uint8_t* half, const uint32_t* h_slots, uint8_t* h_base, u32 first, u32 cnt,
                          bool to_host) {
    const u64 page = ctx->page_bytes;
    u32 j = 0;
    while (j < cnt) {
        u32 run = 1;  // coalesce consecutive host slots into one copy
        if (!h_slots) run = cnt;
        else
            while (j + run < cnt && h_slots[first + j + run] == h_slots[first + j] + run) ++run;
        uint8_t* h = h_base + (u64)(h_slots ? h_slots[first + j] : first + j) * page;
        uint8_t* d = half + (u64)j * page;
        if (to_host) CW_CUDA(ctx, cudaMemcpyAsync(h, d, (u64)run * page, cudaMemcpyDeviceToHost, ctx->s_copy));
        else CW_CUDA(ctx, cudaMemcpyAsync(d, h, (u64)run * page, cudaMemcpyHostToDevice, ctx->s_copy));
        j += run;
    }
    return CW_OK;
}

int32_t cw_swap_out(cw_ctx* ctx, const uint32_t* d_victims, const uint32_t* d_num_victims, uint32_t cap,
                    const uint32_t* h_host_slots, void* h_dst) {
    if (!ctx) return CW_E_STATE;
    if (!ctx->cfg.n_chunks) return CW_E_STATE;
    if (cap == 0) return CW_OK;
    if (!d_victims || !h_dst) return CW_E_INVAL;
    if (d_num_victims) {
        // device count: the page count is unknown to the host, so no copy-engine transfer can be sized for it.  The
        // gather kernel stores straight into the (mapped, pinned) destination: exactly n pages cross PCIe.
        if (h_host_slots || !cw_aligned16(h_dst)) return CW_E_INVAL;
        cudaPointerAttributes at;
        if (cudaPointerGetAttributes(&at, h_dst) != cudaSuccess || at.type != cudaMemoryTypeHost || !at.devicePointer) {
            cudaGetLastError();
            return CW_E_INVAL;
        }
        return cwi_copy_pages(ctx, ctx->s_main, d_victims, d_num_victims, 0, cap, at.devicePointer, true);
    }
    if (!ctx->staging) return CW_E_STATE;
    const u64 page = ctx->page_bytes, half_bytes = (ctx->cfg.staging_bytes / 2) & ~15ull;
    const u32 pps = (u32)(half_bytes / page < 0xFFFFFFFFull ? half_bytes / page : 0xFFFFFFFFull);
    for (u32 first = 0, k = 0; first < cap; first += pps, ++k) {
        const u32 cnt = cap - first < pps ? cap - first : pps;
        const int b = k & 1;
        uint8_t* half = ctx->staging + (u64)b * half_bytes;
        CW_CUDA(ctx, cudaStreamWaitEvent(ctx->s_main, ctx->ev_copy[b], 0));  // PCIe done with this half
        int32_t st = cwi_copy_pages(ctx, ctx->s_main, d_victims, nullptr, first, first + cnt,
                                    half - (u64)first * page, true);
        if (st) return st;
        CW_CUDA(ctx, cudaEventRecord(ctx->ev_gather[b], ctx->s_main));
        CW_CUDA(ctx, cudaStreamWaitEvent(ctx->s_copy, ctx->ev_gather[b], 0));
        st = pcie_slice(ctx, half, h_host_slots, static_cast<uint8_t*>(h_dst), first, cnt, true);
        if (st) return st;
        CW_CUDA(ctx, cudaEventRecord(ctx->ev_copy[b], ctx->s_copy));
    }
    return CW_OK;
}

int32_t cw_swap_in(cw_ctx* ctx, const uint32_t* h_host_slots, const void* h_src, const uint32_t* d_dst_blocks,
                   uint32_t n) {
    if (!ctx) return CW_E_STATE;
    if (!ctx->cfg.n_chunks || !ctx->staging) return CW_E_STATE;
    if (n == 0) return CW_OK;
    if (!d_dst_blocks || !h_src) return CW_E_INVAL;
    const u64 page = ctx->page_bytes, half_bytes = (ctx->cfg.staging_bytes / 2) & ~15ull;
    const u32 pps = (u32)(half_bytes / page < 0xFFFFFFFFull ? half_bytes / page : 0xFFFFFFFFull);
    for (u32 first = 0, k = 0; first < n; first += pps, ++k) {
        const u32 cnt = n - first < pps ? n - first : pps;
        const int b = k & 1;
        uint8_t* half = ctx->staging + (u64)b * half_bytes;
        CW_CUDA(ctx, cudaStreamWaitEvent(ctx->s_copy, ctx->ev_gather[b], 0));  // kernels done with this half
        int32_t st = pcie_slice(ctx, half, h_host_slots, const_cast<uint8_t*>(static_cast<const uint8_t*>(h_src)),
                                first, cnt, false);
        if (st) return st;
        CW_CUDA(ctx, cudaEventRecord(ctx->ev_copy[b], ctx->s_copy));
        CW_CUDA(ctx, cudaStreamWaitEvent(ctx->s_main, ctx->ev_copy[b], 0));
        st = cwi_copy_pages(ctx, ctx->s_main, d_dst_blocks, nullptr, first, first + cnt, half - (u64)first * page,
                            false);
        if (st) return st;
        CW_CUDA(ctx, cudaEventRecord(ctx->ev_gather[b], ctx->s_main));
    }
    return CW_OK;
}

int32_t cw_table_insert(cw_ctx* ctx, const uint64_t* d_keys, const uint32_t* d_loc, uint32_t n,
                        uint32_t* d_winner_loc) {
    if (!ctx) return CW_E_STATE;
    if (n == 0) return CW_OK;
    if (!d_keys || !d_loc) return CW_E_INVAL;
    return cwi_table_insert(ctx, d_keys, d_loc, n, d_winner_loc);
}
int32_t cw_table_erase(cw_ctx* ctx, const uint64_t* d_keys, uint32_t n) {
    if (!ctx) return CW_E_STATE;
    if (n == 0) return CW_OK;
    if (!d_keys) return CW_E_INVAL;
    return cwi_table_erase(ctx, d_keys, n);
}
int32_t cw_table_retag(cw_ctx* ctx, const uint64_t* d_keys, const uint32_t* d_new_loc, uint32_t n) {
    if (!ctx) return CW_E_STATE;
    if (n == 0) return CW_OK;
    if (!d_keys || !d_new_loc) return CW_E_INVAL;
    return cwi_table_retag(ctx, d_keys, d_new_loc, n);
}
int32_t cw_table_lookup(cw_ctx* ctx, const uint64_t* d_keys, uint32_t n, uint32_t* d_loc) {
    if (!ctx) return CW_E_STATE;
    if (n == 0) return CW_OK;
    if (!d_keys || !d_loc) return CW_E_INVAL;
    return cwi_table_lookup(ctx, d_keys, n, d_loc);
}
int32_t cw_table_compact(cw_ctx* ctx) {
    if (!ctx) return CW_E_STATE;
    return cwi_table_compact(ctx);
}
int32_t cw_table_stats(cw_ctx* ctx, uint64_t* h_out8) {
    if (!ctx) return CW_E_STATE;
    if (!h_out8) return CW_E_INVAL;
    return cwi_table_stats(ctx, h_out8);
}
int32_t cw_blocks_update(cw_ctx* ctx, uint32_t tier, const uint32_t* d_ids, uint32_t n, const uint32_t* d_session,
                         const uint32_t* d_depth, const uint32_t* d_last_access, const uint32_t* d_ref_flags) {
    if (!ctx) return CW_E_STATE;
    if (tier > 1) return CW_E_INVAL;
    if (n == 0) return CW_OK;
    if (ctx->tier_size[tier] == 0) return CW_E_STATE;
    if (!d_ids) return CW_E_INVAL;
    return cwi_blocks_update(ctx, tier, d_ids, n, d_session, d_depth, d_last_access, d_ref_flags);
}

#pragma GCC visibility pop
}  // extern "C"
