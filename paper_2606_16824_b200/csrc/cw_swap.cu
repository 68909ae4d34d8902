// Stage 4 — paged KV gather / scatter (device halves of cw_swap_out / cw_swap_in).  DESIGN.md R5.
//
// A pure byte permutation, HBM-bound: 2 bytes of traffic per byte moved.  Each CTA is ONE elected thread
// driving a shared-memory ring with the TMA engine: cp.async.bulk global->shared (mbarrier complete_tx),
// then cp.async.bulk shared->global (bulk_group), CWC_AHEAD loads in flight ahead of the stores.  No data
// ever passes through registers.  Work item = (page j, chunk c, piece) of <= CWC_PIECE bytes; items are
// dealt round-robin to the CTAs so that every SM streams the same amount.  A block-major pool (chunk_stride ==
// chunk_bytes: the page is contiguous) is moved as ONE chunk per page, so small chunks still travel in 16 KiB pieces.
#include <stdio.h>

#include "cw_internal.cuh"

namespace {

#define CWC_PIECE 16384u
#define CWC_STAGES 6
#define CWC_AHEAD 4
#define CWC_CTAS_PER_SM 2

struct CopyArgs {
    uint8_t* pool;
    uint8_t* staged;
    const u32* ids;
    const u32* num;  // device scalar or NULL
    u32 first, cap;
    u32 n_chunks;
    u32 pieces_per_chunk;
    u64 chunk_bytes, chunk_stride, block_stride;
    u32 pool_blocks;
    u32* status;
};

template <bool GATHER>
__global__ void __launch_bounds__(32) copy_pages_kernel(const CopyArgs a) {
    extern __shared__ __align__(128) uint8_t ring[];
    __shared__ u64 full[CWC_STAGES];
    if (threadIdx.x != 0) return;
    for (int s = 0; s < CWC_STAGES; ++s) mbar_init(smem_u32(&full[s]), 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");

    u32 n = a.cap;
    if (a.num) n = min(n, *a.num);
    n = n > a.first ? n - a.first : 0;
    const u64 per_page = (u64)a.n_chunks * a.pieces_per_chunk;
    const u64 items = (u64)n * per_page;
    // items of this CTA: blockIdx.x, blockIdx.x + G, ...
    const u64 G = gridDim.x;
    const u64 mine = items > blockIdx.x ? (items - blockIdx.x + G - 1) / G : 0;

    auto locate = [&](u64 local, const uint8_t*& src, uint8_t*& dst, u32& bytes) {
        const u64 it = blockIdx.x + local * G;
        const u64 j = it / per_page;
        const u32 rem = (u32)(it - j * per_page);
        const u32 c = rem / a.pieces_per_chunk, pc = rem - c * a.pieces_per_chunk;
        const u64 off = (u64)pc * CWC_PIECE;
        bytes = (u32)min((u64)CWC_PIECE, a.chunk_bytes - off);
        u32 b = a.ids[a.first + j];
        if (b >= a.pool_blocks) {  // never touch memory outside the pool
            atomicOr(a.status, CWS_INVAL);
            bytes = 0;
            b = 0;
        }
        uint8_t* in_pool = a.pool + (u64)b * a.block_stride + (u64)c * a.chunk_stride + off;
        uint8_t* in_stage = a.staged + ((a.first + j) * (u64)a.n_chunks + c) * a.chunk_bytes + off;
        src = GATHER ? in_pool : in_stage;
        dst = GATHER ? in_stage : in_pool;
    };
    auto issue_load = [&](u64 local) {
        const uint8_t* src;
        uint8_t* dst;
        u32 bytes;
        locate(local, src, dst, bytes);
        const u32 s = (u32)(local % CWC_STAGES);
        const u32 bar = smem_u32(&full[s]);
        if (bytes) {
            mbar_expect_tx(bar, bytes);
            bulk_g2s_plain(smem_u32(ring + (u64)s * CWC_PIECE), src, bytes, bar);
        } else {
            mbar_arrive(bar);
        }
    };

    const u64 pre = mine < CWC_AHEAD ? mine : CWC_AHEAD;
    for (u64 l = 0; l < pre; ++l) issue_load(l);
    for (u64 l = 0; l < mine; ++l) {
        if (l + CWC_AHEAD < mine) {
            // stage of item l+AHEAD was last used by item l+AHEAD-STAGES: its store must have read smem
            bulk_wait_read<CWC_STAGES - CWC_AHEAD - 1>();
            issue_load(l + CWC_AHEAD);
        }
        const u32 s = (u32)(l % CWC_STAGES);
        mbar_wait(smem_u32(&full[s]), (u32)(l / CWC_STAGES) & 1);
        const uint8_t* src;
        uint8_t* dst;
        u32 bytes;
        locate(l, src, dst, bytes);
        if (bytes) bulk_s2g(dst, smem_u32(ring + (u64)s * CWC_PIECE), bytes);
        bulk_commit();
    }
    bulk_wait_all<0>();
}

#ifdef CW_DEBUG
// debug builds: a block id that occurs twice in a gather list is a caller bug (SURVEY.md 8c stage 4)
__global__ void dup_check_kernel(const u32* ids, const u32* num, u32 first, u32 cap, u32 pool_blocks, u32* bits,
                                 u32* status, bool clear) {
    u32 n = cap;
    if (num) n = min(n, *num);
    const u32 j = first + blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    const u32 b = ids[j];
    if (b >= pool_blocks) return;  // reported by the copy kernel itself
    if (clear) {
        bits[b >> 5] = 0;
    } else if (atomicOr(&bits[b >> 5], 1u << (b & 31)) & (1u << (b & 31))) {
        atomicOr(status, CWS_INVAL);
    }
}
#endif

}  // namespace

int cwi_copy_grid(int n_sm) {
    cudaFuncSetAttribute(copy_pages_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                         CWC_STAGES * CWC_PIECE);
    cudaFuncSetAttribute(copy_pages_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                         CWC_STAGES * CWC_PIECE);
    return n_sm * CWC_CTAS_PER_SM;
}

int32_t cwi_copy_pages(cw_ctx* ctx, cudaStream_t stream, const u32* d_ids, const u32* d_num, u32 first, u32 cap,
                       void* d_staged, bool gather) {
    if (cap <= first) return CW_OK;
    CopyArgs a;
    a.pool = static_cast<uint8_t*>(ctx->cfg.d_pool);
    a.staged = static_cast<uint8_t*>(d_staged);
    a.ids = d_ids;
    a.num = d_num;
    a.first = first;
    a.cap = cap;
    a.n_chunks = ctx->cfg.n_chunks;
    a.chunk_bytes = ctx->cfg.chunk_bytes;
    a.chunk_stride = ctx->cfg.chunk_stride;
    a.block_stride = ctx->cfg.block_stride;
    if (a.chunk_stride == a.chunk_bytes) {  // block-major pool: a page is contiguous, move it as one chunk
        a.chunk_bytes *= a.n_chunks;
        a.chunk_stride = a.chunk_bytes;
        a.n_chunks = 1;
    }
    a.pieces_per_chunk = (u32)((a.chunk_bytes + CWC_PIECE - 1) / CWC_PIECE);
    a.pool_blocks = ctx->cfg.num_blocks;
    a.status = ctx->d_status;
#ifdef CW_DEBUG
    if (gather && ctx->dup_bits) {
        const u32 nb = (cap - first + 255) / 256;
        dup_check_kernel<<<nb, 256, 0, stream>>>(d_ids, d_num, first, cap, a.pool_blocks, ctx->dup_bits, a.status, false);
        dup_check_kernel<<<nb, 256, 0, stream>>>(d_ids, d_num, first, cap, a.pool_blocks, ctx->dup_bits, a.status, true);
    }
#endif
    const u64 items = (u64)(cap - first) * a.n_chunks * a.pieces_per_chunk;  // a.n_chunks: after coalescing
    u64 grid = (u64)ctx->copy_grid;
    if (grid > items) grid = items;
    if (gather)
        copy_pages_kernel<true><<<(u32)grid, 32, CWC_STAGES * CWC_PIECE, stream>>>(a);
    else
        copy_pages_kernel<false><<<(u32)grid, 32, CWC_STAGES * CWC_PIECE, stream>>>(a);
    CW_LAUNCH_CHECK(ctx);
    return CW_OK;
}
