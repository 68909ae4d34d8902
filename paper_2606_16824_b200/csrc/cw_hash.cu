// Stage 1 — chained prefix hashing (cw_hash_blocks).  DESIGN.md R1 / "Kernels: hash".
//
//   digest  c_j = fin( (sum_{m<8} u64(u32(t[2m]+ka_m)) * u64(u32(t[2m+1]+kb_m))) ^ K5 )
//   chain   H_j = A*H_{j-1} + c_j  (mod 2^64),  H_{-1} = fin(salt ^ K7)  or  start_state
//
// The chain is an affine recurrence whose multiplier is always a power of A, so it is a SCAN:
//   warp   : inclusive scan over 32 blocks, step d uses the constant A^d
//   CTA    : 8 warp aggregates combined by Horner with A^32
//   request: units of 256 blocks; unit t's carry-in = A^(256 t)*seed + sum_{v<t} A^(256 (t-1-v)) * agg_v,
//            where agg_v is unit v's carry-free aggregate — published to global memory as soon as it is
//            known, so no unit ever waits on another unit's look-back (no serial chain across units).
//
// Data movement: one producer warp per CTA takes unit tickets (atomic counter => forward progress without
// any co-residency assumption), locates the request with a warp-wide 32-ary search over hash_off, and
// issues ONE TMA bulk copy (cp.async.bulk, L2 evict-first) of the unit's 16 KiB of token ids into a
// 3-stage shared-memory ring.  Requests start at arbitrary 4-byte alignment: the copy starts at the
// 16-byte boundary below and the consumers funnel the `mis` leading words away in registers.
// Consumers read shared memory conflict-free (lane = 16-byte quarter of a block, 512 contiguous bytes per
// LDS.128), form quarter sums, and transpose-reduce them with 6 shuffles so that each lane owns one block.
#include <stdio.h>

#include "cw_internal.cuh"

namespace {

__host__ __device__ constexpr u32 key_a(int m) { return (u32)(cw_fin(CW_K11 * (u64)(m + 1)) >> 32) | 0x80000000u; }
__host__ __device__ constexpr u32 key_b(int m) {
    return (u32)(cw_fin(CW_K11 * (u64)(m + 1)) & 0xffffffffull) | 0x80000000u;
}

struct HashArgs {
    const i32* tokens;
    const u64* tok_off;
    const u32* start_block;
    const u64* start_state;
    const u64* salt;
    const u64* hash_off;
    u64* hashes;
    cw_hash_ctl* ctl;
    u64* agg;
    u32* flag;
    u32* status;
    u64 agg_slots;
    u64 max_hashed;
    u32 R;
};

struct UnitInfo {
    u64 out_base;  // index in hashes[] of the unit's first block
    u64 slot;      // aggregate slot of this unit
    u64 seed;      // H_{-1} or start_state of the request
    u32 valid;
    u32 t;         // unit index inside the request
    u32 nblk;      // blocks in this unit (<= CWH_UNIT)
    u32 mis;       // leading words to skip in the staged copy (0..3)
    u32 publish;   // 1 if a later unit of the same request exists
    u32 pad[3];
};

struct __align__(128) HashSmem {
    uint8_t stage[CWH_STAGES][CWH_STAGE_BYTES + 112];  // keeps every stage 128-byte aligned
    UnitInfo info[CWH_STAGES];
    u64 full[CWH_STAGES];
    u64 empty[CWH_STAGES];
    u64 wagg[2][CWH_WARPS];
    u64 carry[2];
};

// unit slots are numbered relative to the call's first hash (hash_off may be a slice of a longer CSR array)
__device__ __forceinline__ u64 slot_base(const u64* hash_off, u64 h_first, u32 r) {
    return ((hash_off[r] - h_first) >> CWH_UNIT_LOG2) + r;
}

__device__ __forceinline__ u64 pow_u64(u64 base, u32 e) {
    u64 r = 1;
    while (e) {
        if (e & 1) r *= base;
        base *= base;
        e >>= 1;
    }
    return r;
}

__device__ __forceinline__ void consumer_bar() { asm volatile("bar.sync 1, %0;" ::"n"(CWH_UNIT) : "memory"); }

__global__ void __launch_bounds__(CWH_UNIT + 32, 4) hash_kernel(const HashArgs a) {
    extern __shared__ __align__(128) uint8_t smem_raw[];
    HashSmem& sm = *reinterpret_cast<HashSmem*>(smem_raw);
    const u32 tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const u32 cur_epoch = a.ctl->epoch + 1;

    if (tid == 0) {
        for (int s = 0; s < CWH_STAGES; ++s) {
            mbar_init(smem_u32(&sm.full[s]), 1);
            mbar_init(smem_u32(&sm.empty[s]), 1);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == CWH_WARPS) {
        // ------------------------------------------------------------------ producer warp
        const u32 R = a.R;
        const u64 h_first = R ? a.hash_off[0] : 0;
        u64 total_blocks = R ? a.hash_off[R] - h_first : 0;
        u64 total_slots = 0;
        if (R) {
            if (a.hash_off[R] < h_first || total_blocks > a.max_hashed ||
                (total_blocks >> CWH_UNIT_LOG2) + R > a.agg_slots) {
                if (lane == 0 && blockIdx.x == 0) atomicOr(a.status, CWS_INVAL);
            } else {
                total_slots = (total_blocks >> CWH_UNIT_LOG2) + R;
            }
        }
        const u64 policy = policy_evict_first();
        for (u32 it = 0;; ++it) {
            const u32 s = it % CWH_STAGES;
            if (it >= CWH_STAGES) mbar_wait(smem_u32(&sm.empty[s]), ((it / CWH_STAGES) - 1) & 1);
            UnitInfo ui;
            ui.valid = 0;
            const i32* src = nullptr;
            u32 bytes = 0;
            for (;;) {
                u64 tk = 0;
                if (lane == 0) tk = atomicAdd(&a.ctl->ticket, 1u);
                tk = shfl64(tk, 0);
                if (tk >= total_slots) break;
                // largest r with slot_base(r) <= tk, by 32-ary search (slot_base is strictly increasing)
                u32 lo = 0, hi = R;
                while (hi - lo > 1) {
                    u32 step = (hi - lo + 31) >> 5;
                    u32 p = lo + lane * step;
                    bool ok = p < hi && slot_base(a.hash_off, h_first, p) <= tk;
                    u32 cnt = __popc(__ballot_sync(0xffffffffu, ok));
                    u32 nlo = lo + (cnt - 1) * step;
                    hi = min(hi, nlo + step);
                    lo = nlo;
                }
                const u32 r = lo;
                const u64 h0 = a.hash_off[r], n_r = a.hash_off[r + 1] - h0;
                const u64 t0 = a.tok_off[r], len = a.tok_off[r + 1] - t0;
                const u64 sb = a.start_block ? a.start_block[r] : 0;
                const u64 t = tk - slot_base(a.hash_off, h_first, r);
                if (a.tok_off[r + 1] < t0 || n_r != (len >> 4) || sb > n_r) {
                    if (lane == 0 && t == 0) atomicOr(a.status, CWS_INVAL);
                    continue;
                }
                const u64 todo = n_r - sb;
                const u64 T = (todo + CWH_UNIT - 1) >> CWH_UNIT_LOG2;
                if (t >= T) continue;  // unused slot of the sparse numbering
                const u64 j0 = sb + (t << CWH_UNIT_LOG2);
                ui.valid = 1;
                ui.t = (u32)t;
                ui.nblk = (u32)min((u64)CWH_UNIT, n_r - j0);
                ui.mis = (u32)(t0 & 3);
                ui.publish = (t + 1 < T) ? 1u : 0u;
                ui.out_base = h0 + j0;
                ui.slot = tk;
                ui.seed = sb > 0 ? a.start_state[r] : cw_fin((a.salt ? a.salt[r] : 0ull) ^ CW_K7);
                src = a.tokens + (t0 + 16 * j0 - ui.mis);
                bytes = ui.nblk * 64 + (ui.mis ? 16u : 0u);
                break;
            }
            if (lane == 0) {
                sm.info[s] = ui;
                const u32 bar = smem_u32(&sm.full[s]);
                if (ui.valid) {
                    mbar_expect_tx(bar, bytes);
                    bulk_g2s(smem_u32(&sm.stage[s][0]), src, bytes, bar, policy);
                } else {
                    mbar_arrive(bar);
                }
            }
            __syncwarp();
            if (!ui.valid) break;
        }
    } else {
        // ------------------------------------------------------------------ consumer warps
        const u32 q = lane & 3;
        const u32 ka0 = q == 0 ? key_a(0) : q == 1 ? key_a(2) : q == 2 ? key_a(4) : key_a(6);
        const u32 kb0 = q == 0 ? key_b(0) : q == 1 ? key_b(2) : q == 2 ? key_b(4) : key_b(6);
        const u32 ka1 = q == 0 ? key_a(1) : q == 1 ? key_a(3) : q == 2 ? key_a(5) : key_a(7);
        const u32 kb1 = q == 0 ? key_b(1) : q == 1 ? key_b(3) : q == 2 ? key_b(5) : key_b(7);
        const u64 a_lane1 = pow_u64(CW_A, lane + 1);  // A^(lane+1)
        // after the transposed reduction lane i owns block 8*k(i) + (i>>2), k(i) = 2*bit0 + bit1;
        // the lane that owns block b is 4*(b&7) | ((b>>3)&1)<<1 | (b>>4)
        const u32 owner = ((lane & 7) << 2) | (((lane >> 3) & 1) << 1) | (lane >> 4);
        constexpr u64 A2 = cw_pow(CW_A, 2), A4 = cw_pow(CW_A, 4), A8 = cw_pow(CW_A, 8), A16 = cw_pow(CW_A, 16),
                      A32 = cw_pow(CW_A, 32), AC = cw_pow(CW_A, CWH_UNIT);

        for (u32 it = 0;; ++it) {
            const u32 s = it % CWH_STAGES;
            mbar_wait(smem_u32(&sm.full[s]), (it / CWH_STAGES) & 1);
            const UnitInfo ui = sm.info[s];
            if (!ui.valid) break;

            // ---- quarter sums of 4 x 8 blocks
            const uint8_t* base = &sm.stage[s][0] + warp * (32 * 64) + (lane >> 2) * 64 + q * 16;
            u64 p[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const uint4 w0 = *reinterpret_cast<const uint4*>(base + k * 512);
                u32 t0, t1, t2, t3;
                if (ui.mis == 0) {
                    t0 = w0.x; t1 = w0.y; t2 = w0.z; t3 = w0.w;
                } else {
                    const uint4 w1 = *reinterpret_cast<const uint4*>(base + k * 512 + 16);
                    if (ui.mis == 1) {
                        t0 = w0.y; t1 = w0.z; t2 = w0.w; t3 = w1.x;
                    } else if (ui.mis == 2) {
                        t0 = w0.z; t1 = w0.w; t2 = w1.x; t3 = w1.y;
                    } else {
                        t0 = w0.w; t1 = w1.x; t2 = w1.y; t3 = w1.z;
                    }
                }
                p[k] = (u64)(t0 + ka0) * (u64)(t1 + kb0) + (u64)(t2 + ka1) * (u64)(t3 + kb1);
            }
            // ---- transposed reduction over the 4 lanes of a block (6 shuffles)
            const bool b0 = lane & 1, b1 = lane & 2;
            u64 keep0 = b0 ? p[2] : p[0], keep1 = b0 ? p[3] : p[1];
            u64 send0 = b0 ? p[0] : p[2], send1 = b0 ? p[1] : p[3];
            keep0 += shfl64_xor(send0, 1);
            keep1 += shfl64_xor(send1, 1);
            u64 keep = b1 ? keep1 : keep0, send = b1 ? keep0 : keep1;
            keep += shfl64_xor(send, 2);
            const u64 ssum = shfl64(keep, owner);  // lane = block index inside the warp
            u64 x = cw_fin(ssum ^ CW_K5);

            // ---- warp scan of the affine chain (carry-free)
            u64 y;
            y = shfl64_up(x, 1);  if (lane >= 1) x += CW_A * y;
            y = shfl64_up(x, 2);  if (lane >= 2) x += A2 * y;
            y = shfl64_up(x, 4);  if (lane >= 4) x += A4 * y;
            y = shfl64_up(x, 8);  if (lane >= 8) x += A8 * y;
            y = shfl64_up(x, 16); if (lane >= 16) x += A16 * y;
            const u32 buf = it & 1;
            if (lane == 31) sm.wagg[buf][warp] = x;
            consumer_bar();
            if (tid == 0) mbar_arrive(smem_u32(&sm.empty[s]));  // every consumer has read stage s

            if (warp == 0) {
                if (ui.publish) {  // full unit: aggregate = sum_w A^(32 (W-1-w)) * wagg[w]
                    u64 v = 0;
                    if (lane < CWH_WARPS) v = sm.wagg[buf][lane] * pow_u64(A32, CWH_WARPS - 1 - lane);
#pragma unroll
                    for (int m = 1; m < CWH_WARPS; m <<= 1) v += shfl64_xor(v, m);
                    if (lane == 0) {
                        a.agg[ui.slot] = v;
                        st_release_u32(&a.flag[ui.slot], cur_epoch);
                    }
                }
                u64 carry = 0;
                if (ui.t == 0) {
                    carry = ui.seed;
                } else {
                    for (u32 b = 0; b < ui.t; b += 32) {
                        const u32 v = b + lane;
                        if (v < ui.t) {
                            const u64 slot = ui.slot - ui.t + v;
                            while (ld_acquire_u32(&a.flag[slot]) != cur_epoch) {
                            }
                            carry += ld_relaxed_u64(&a.agg[slot]) * pow_u64(AC, ui.t - 1 - v);
                        }
                    }
                    if (lane == 0) carry += pow_u64(AC, ui.t) * ui.seed;
#pragma unroll
                    for (int m = 1; m < 32; m <<= 1) carry += shfl64_xor(carry, m);
                }
                if (lane == 0) sm.carry[buf] = carry;
            }
            consumer_bar();
            u64 cin = sm.carry[buf];
            for (u32 v = 0; v < warp; ++v) cin = A32 * cin + sm.wagg[buf][v];
            const u64 h = x + a_lane1 * cin;
            const u32 bi = warp * 32 + lane;
            if (bi < ui.nblk) a.hashes[ui.out_base + bi] = h;
        }
    }

    __syncthreads();
    if (tid == 0) {
        __threadfence();
        const u32 prev = atomicAdd(&a.ctl->done, 1u);
        if (prev == gridDim.x - 1) {  // last CTA: leave the control block ready for the next call
            a.ctl->ticket = 0;
            a.ctl->done = 0;
            a.ctl->epoch = cur_epoch;
            __threadfence();
        }
    }
}

}  // namespace

int cwi_hash_grid(int n_sm) {
    int per_sm = 0;
    cudaFuncSetAttribute(hash_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(HashSmem));
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, hash_kernel, CWH_UNIT + 32, sizeof(HashSmem));
    if (per_sm < 1) per_sm = 1;
    return per_sm * n_sm;
}

int32_t cwi_hash_blocks(cw_ctx* ctx, const i32* d_tokens, const u64* d_tok_off, const u32* d_start_block,
                        const u64* d_start_state, const u64* d_salt, const u64* d_hash_off, u32 R, u64* d_hashes) {
    if (R == 0) return CW_OK;
    HashArgs a;
    a.tokens = d_tokens;
    a.tok_off = d_tok_off;
    a.start_block = d_start_block;
    a.start_state = d_start_state;
    a.salt = d_salt;
    a.hash_off = d_hash_off;
    a.hashes = d_hashes;
    a.ctl = ctx->hash_ctl;
    a.agg = ctx->hash_agg;
    a.flag = ctx->hash_flag;
    a.status = ctx->d_status;
    a.agg_slots = ctx->hash_slots;
    a.max_hashed = ctx->cfg.max_hashed_blocks;
    a.R = R;
    // never more CTAs than units could exist; small calls stay small
    u64 max_units = (ctx->cfg.max_hashed_blocks >> CWH_UNIT_LOG2) + R;
    int grid = (int)((u64)ctx->hash_grid < max_units ? (u64)ctx->hash_grid : max_units);
    if (grid < 1) grid = 1;
    hash_kernel<<<grid, CWH_UNIT + 32, sizeof(HashSmem), ctx->s_main>>>(a);
    CW_LAUNCH_CHECK(ctx);
    return CW_OK;
}
