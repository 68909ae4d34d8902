// Stage 1 — chained prefix hashing (cw_hash_blocks).  DESIGN.md R1 / "Kernels: hash".
//
//   digest  c_j = fin( (sum_{m<8} u64(u32(t[2m]+ka_m)) * u64(u32(t[2m+1]+kb_m))) ^ K5 )
//   chain   H_j = A*H_{j-1} + c_j  (mod 2^64),  H_{-1} = fin(salt ^ K7)  or  start_state
//
// The chain is an affine recurrence whose multiplier is always a power of A, so it is a SCAN:
//   lane : a consumer lane owns CWH_K = 8 CONSECUTIVE blocks of a unit (512 bytes of token ids): it digests them
//          itself (no cross-lane reduction) and chains them serially in registers (7 multiply-adds)
//   warp : one inclusive scan over the 32 lane aggregates, step d uses the constant (A^8)^d; a unit of 256 blocks
//          therefore costs ONE 5-step warp scan, and a warp works on a unit alone (no CTA barrier per unit)
//   CTA  : the 4 consumer warps take the units of the CTA's range round-robin; the chain state is handed from the
//          warp of unit i to the warp of unit i+1 through a shared-memory ring (one mbarrier per slot): the serial
//          part per unit is one multiply-add, everything else of a unit runs beside the other warps' units
//   grid : the list of units (request-aligned runs of <= 256 blocks) is cut into gridDim.x CONTIGUOUS ranges of
//          about equal length (equal in tokens), one per CTA.  A CTA therefore walks its requests sequentially and
//          never waits on another CTA while it streams.  Only the first request of a range can have begun in an
//          earlier range: that boundary segment is scanned with carry-in 0 and patched at the very end of the CTA,
//          H_j += A^(j-j0+1) * carry_in (linear in the carry, mod 2^64), from the chain states the CTAs of the
//          earlier ranges have published (a range wholly inside one request publishes its carry-free tail and its
//          length, and the reader folds those while walking back).  Ranges are handed out by an atomic ticket, so
//          the CTA that is waited for has always started: the single wait per CTA cannot deadlock and happens when
//          both CTAs are finishing anyway.
//
// One launch per call, no plan pass: the TOKEN space of the call is cut into gridDim.x equal pieces (a multiple of a
// unit's 4096 tokens each) and every CTA moves the two ends of its piece to the first unit at or behind them by a
// 32-ary search over tok_off (three rounds for 4096 requests; both ends are mapped by the same function, so the ranges
// tile the unit list); the offsets of every request are validated once, spread over the grid; the last CTA to finish
// re-arms the ticket and advances the epoch.  (Rounds 1-2 ran a one-CTA plan kernel first — units per request,
// exclusive scan, 10 us plus a launch gap in front of an 87 us kernel — and cut the UNIT list into equal ranges.)
// The streaming pass: one producer warp issues ONE TMA bulk copy (cp.async.bulk, L2 evict-first) of each unit's
// 16 KiB of token ids into a 4-stage shared-memory ring (mbarrier full/empty); a consumer warp reads its unit with
// conflict-free 16-byte loads (the quarter of a block a lane reads first is rotated by the lane id and odd lane quads
// take their block pairs in swapped order, so the 8 lanes of a load phase cover all 32 banks); 16 multiplies + fin per
// block, the lane chain, the warp scan, the hand-over, 8 stores; then the boundary patch (about half a request per
// CTA: ~1% extra traffic, L2-resident).
// Requests start at arbitrary 4-byte alignment: the copy starts at the 16-byte boundary below and the
// consumers funnel the `mis` leading words away in registers.
#include <stddef.h>
#include <stdio.h>

#include <mutex>

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
    u64* plan;          // [1] call epoch, [2] range ticket, [3] CTAs done ([0] unused)
    cw_hash_rec* rec;   // per CTA of hash_kernel
    u32* status;
    u64 max_hashed;
    u32 R;
};

enum { MODE_CONTINUE = 0, MODE_SEED = 1, MODE_ZERO = 2 };

struct UnitInfo {
    u64 out_base;  // index in hashes[] of the unit's first block
    u64 seed;      // H_{-1} or start_state of the request (MODE_SEED)
    u32 valid;
    u32 nblk;      // blocks in this unit (<= CWH_UNIT)
    u32 mis;       // leading words to skip in the staged copy (0..3)
    u32 mode;      // where the unit's carry-in comes from
    u32 last;      // last unit of this CTA's range: record the chain state after it
    u32 pad[3];
};

struct __align__(128) HashSmem {
    uint8_t stage[CWH_STAGES][CWH_STAGE_BYTES + 112];  // keeps every stage 128-byte aligned
    UnitInfo info[CWH_STAGES];
    u64 full[CWH_STAGES];
    u64 empty[CWH_STAGES];
    u64 carry_bar[CWH_WARPS];   // slot i % CWH_WARPS: the chain state after unit i of the range is published
    u64 carry_ring[CWH_WARPS];
    u64 carry_in;
    u32 wsum[CWH_WARPS + 1];
    u32 b_r[2], b_t[2];         // the range's two ends as (request, unit inside the request)
    u32 range;
    u32 rec_flags;
    u32 rec_bseg_len;
    u64 rec_bseg_first;
    u64 rec_tail_state;
};

__device__ __forceinline__ u64 pow_u64(u64 base, u64 e) {
    u64 r = 1;
    while (e) {
        if (e & 1) r *= base;
        base *= base;
        e >>= 1;
    }
    return r;
}

// ------------------------------------------------------------------------------------------------ requests
// Units (request-aligned runs of <= 256 blocks from start_block on) of request r; ~0 if its offsets are inconsistent.
// Loads first, decisions after (a load behind a condition is not issued until the condition is known).
struct ReqInfo {
    u64 t0, h0, n, sb, units;  // token offset, hash offset, blocks, first block to hash, units (0 if invalid)
    bool invalid;
};
__device__ __forceinline__ ReqInfo req_info(const HashArgs& a, u32 r) {
    const u64 t0 = a.tok_off[r], t1 = a.tok_off[r + 1], h0 = a.hash_off[r], h1 = a.hash_off[r + 1];
    const u64 sb = a.start_block ? a.start_block[r] : 0;
    ReqInfo q;
    q.invalid = t1 < t0 || h1 < h0 || (h1 - h0) != ((t1 - t0) >> 4) || sb > h1 - h0;
    q.t0 = t0;
    q.h0 = h0;
    q.n = h1 - h0;
    q.sb = sb;
    q.units = q.invalid ? 0ull : (h1 - h0 - sb + CWH_UNIT - 1) >> CWH_UNIT_LOG2;
    return q;
}

// A boundary of the token space (token index p, T0 <= p <= TR) -> the first unit at or behind it: (request, unit inside
// the request); (R, 0) behind the last unit.  Warp-collective: a 32-ary search over tok_off for the request that holds
// p, then at most a hop over requests without work.  Both ends of a range are mapped by the same function, so the
// ranges tile the unit list whatever the offsets look like.
__device__ __forceinline__ void map_boundary(const HashArgs& a, u64 p, u32 lane, u32& r_out, u32& t_out) {
    const u32 R = a.R;
    u32 lo = 0, hi = R;  // largest r < R with tok_off[r] <= p
    while (hi - lo > 1) {
        const u32 step = (hi - lo + 31) >> 5;
        const u32 q = lo + lane * step;
        const bool ok = q < hi && a.tok_off[q] <= p;
        u32 cnt = __popc(__ballot_sync(0xffffffffu, ok));
        cnt = cnt ? cnt : 1u;  // (tok_off[lo] <= p holds for consistent offsets)
        const u32 nlo = lo + (cnt - 1) * step;
        hi = min(hi, nlo + step);
        lo = nlo;
    }
    const ReqInfo q = req_info(a, lo);
    const u64 hs = q.t0 + 16 * q.sb;  // first token that is hashed
    const u64 t = p > hs ? (p - hs + (16 * CWH_UNIT - 1)) / (16 * CWH_UNIT) : 0;
    if (t < q.units) {
        r_out = lo;
        t_out = (u32)t;
        return;
    }
    for (u32 r = lo + 1; r < R; r += 32) {  // the next request with work
        const u32 rr = r + lane;
        const bool has = rr < R && req_info(a, min(rr, R - 1)).units > 0;
        const u32 m = __ballot_sync(0xffffffffu, has);
        if (m) {
            r_out = r + (u32)__ffs(m) - 1;
            t_out = 0;
            return;
        }
    }
    r_out = R;
    t_out = 0;
}

// ------------------------------------------------------------------------------------------------ digests
// The raw sums (before fin) of the 8 blocks a lane owns.  `lane_run` points at the lane's 512 staged bytes; step k
// reads the quarter (k + lane) & 3 of a block (keys kq[k][]), and a lane with `swapped` set takes the blocks of each
// pair in the order odd, even (off_e / off_o carry both rotations), so ct[] comes back in NATURAL block order.
template <int MIS>
__device__ __forceinline__ void digest8(const uint8_t* lane_run, const u32 (&off_e)[4], const u32 (&off_o)[4],
                                        const u32 (&kq)[4][4], bool swapped, u64 (&ct)[CWH_K]) {
    u64 raw[CWH_K];
#pragma unroll
    for (int m = 0; m < CWH_K; ++m) {
        u64 acc = 0;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const uint8_t* p = lane_run + 64 * m + ((m & 1) ? off_o[k] : off_e[k]);
            const uint4 w0 = *reinterpret_cast<const uint4*>(p);
            u32 t0, t1, t2, t3;
            if (MIS == 0) {
                t0 = w0.x; t1 = w0.y; t2 = w0.z; t3 = w0.w;
            } else {
                const uint4 w1 = *reinterpret_cast<const uint4*>(p + 16);
                if (MIS == 1) {
                    t0 = w0.y; t1 = w0.z; t2 = w0.w; t3 = w1.x;
                } else if (MIS == 2) {
                    t0 = w0.z; t1 = w0.w; t2 = w1.x; t3 = w1.y;
                } else {
                    t0 = w0.w; t1 = w1.x; t2 = w1.y; t3 = w1.z;
                }
            }
            acc += (u64)(t0 + kq[k][0]) * (u64)(t1 + kq[k][1]) + (u64)(t2 + kq[k][2]) * (u64)(t3 + kq[k][3]);
        }
        raw[m] = acc;
    }
#pragma unroll
    for (int m = 0; m < CWH_K; m += 2) {
        ct[m] = swapped ? raw[m + 1] : raw[m];
        ct[m + 1] = swapped ? raw[m] : raw[m + 1];
    }
}

// ------------------------------------------------------------------------------------------------ main pass
__global__ void __launch_bounds__(CWH_THREADS, CWH_MIN_CTAS) hash_kernel(const HashArgs a) {
    extern __shared__ __align__(128) uint8_t smem_raw[];
    HashSmem& sm = *reinterpret_cast<HashSmem*>(smem_raw);
    const u32 tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    if (tid == 0) sm.range = atomicAdd(reinterpret_cast<unsigned int*>(a.plan + 2), 1u);
    const u32 R = a.R, G = gridDim.x;
    const u64 T0 = a.tok_off[0], TR = a.tok_off[R], H0 = a.hash_off[0], HR = a.hash_off[R];
    const bool too_big = HR < H0 || HR - H0 > a.max_hashed || TR < T0;
    const u32 epoch = (u32)a.plan[1] + 1;  // advanced by the last CTA to finish (records of earlier calls go stale)
    {   // every request's offsets are checked once, spread over the grid (the status word is all this produces)
        bool bad = too_big;
        for (u32 r = blockIdx.x * CWH_THREADS + tid; r < R; r += G * CWH_THREADS) bad |= req_info(a, r).invalid;
        if (__syncthreads_or(bad) && tid == 0) atomicOr(a.status, CWS_INVAL);  // (also makes sm.range visible)
    }
    auto call_done = [&]() {  // self-cleaning: the last CTA to finish re-arms the ticket and advances the epoch
        if (tid == 0) {
            const u32 old = atomicAdd(reinterpret_cast<unsigned int*>(a.plan + 3), 1u);
            if (old == G - 1) {
                a.plan[3] = 0;
                a.plan[2] = 0;
                a.plan[1] = a.plan[1] + 1;
            }
        }
    };
    // ---- the range of this CTA.  There is no plan pass: the TOKEN space [T0, TR) is cut into G equal pieces (a
    // multiple of a unit's 4096 tokens each), and a boundary is moved to the first unit at or behind it by a search
    // over tok_off.  Ranges in ticket order: every lower range belongs to a CTA that has started.
    const u32 range = sm.range;
    u64 per_tok = (TR - T0 + G - 1) / G;
    per_tok = max((per_tok + 16 * CWH_UNIT - 1) / (16 * CWH_UNIT), (u64)1) * (16 * CWH_UNIT);
    const u64 pb = T0 + (u64)range * per_tok;
    if (too_big || pb >= TR) {  // nothing to do (uniform over the CTA): nobody waits for an empty range
        call_done();
        return;
    }
    if (warp < 2) {
        u32 r, t;
        map_boundary(a, warp ? min(TR, pb + per_tok) : pb, lane, r, t);
        if (lane == 0) {
            sm.b_r[warp] = r;
            sm.b_t[warp] = t;
        }
    }
    __syncthreads();
    const u32 r_b = sm.b_r[0], t_b = sm.b_t[0], r_e = sm.b_r[1], t_e = sm.b_t[1];
    if (r_b == r_e && t_b == t_e) {  // a stretch of tokens without a unit (short or resumed requests)
        call_done();
        return;
    }
    u32 n_units;
    {   // units of the requests [r_b, r_e), less the t_b units in front of the range, plus the t_e units of request r_e
        u32 local = 0;
        for (u32 r = r_b + tid; r < r_e; r += CWH_THREADS) local += (u32)req_info(a, r).units;
        local = __reduce_add_sync(0xffffffffu, local);
        if (lane == 0) sm.wsum[warp] = local;
        __syncthreads();
        u32 total = 0;
#pragma unroll
        for (u32 w = 0; w <= CWH_WARPS; ++w) total += sm.wsum[w];
        n_units = total - t_b + t_e;
    }

    if (tid == 0) {
        for (int s = 0; s < CWH_STAGES; ++s) {
            mbar_init(smem_u32(&sm.full[s]), 1);
            mbar_init(smem_u32(&sm.empty[s]), 1);
        }
        for (int w = 0; w < CWH_WARPS; ++w) mbar_init(smem_u32(&sm.carry_bar[w]), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == CWH_WARPS) {
        // ------------------------------------------------------------------ producer warp
        if (lane == 0) {
            const u64 policy = policy_evict_first();
            u32 r = r_b;
            u64 t = t_b;
            const bool starts_mid = t > 0;  // the first request began in an earlier CTA's range
            bool in_bseg = starts_mid;
            u64 bseg_first = 0, bseg_len = 0;
            u64 h0 = 0, n_r = 0, t0 = 0, sb = 0, seed = 0, un = 0;
            bool fresh = true;
            for (u32 it = 0; it < n_units; ++it) {
                if (fresh) {
                    const ReqInfo q = req_info(a, r);
                    h0 = q.h0;
                    n_r = q.n;
                    t0 = q.t0;
                    sb = q.sb;
                    un = q.units;
                    seed = sb > 0 ? a.start_state[r] : cw_fin((a.salt ? a.salt[r] : 0ull) ^ CW_K7);
                    fresh = false;
                }
                const u32 s = it % CWH_STAGES;
                if (it >= CWH_STAGES) mbar_wait(smem_u32(&sm.empty[s]), ((it / CWH_STAGES) - 1) & 1);
                const u64 j0 = sb + (t << CWH_UNIT_LOG2);
                UnitInfo ui;
                ui.valid = 1;
                ui.nblk = (u32)min((u64)CWH_UNIT, n_r - j0);
                ui.mis = (u32)(t0 & 3);
                ui.mode = t == 0 ? MODE_SEED : (it == 0 ? MODE_ZERO : MODE_CONTINUE);
                ui.out_base = h0 + j0;
                ui.seed = seed;
                ui.last = (it + 1 == n_units) ? 1u : 0u;
                if (in_bseg) {
                    if (it == 0) bseg_first = h0 + j0;
                    bseg_len += ui.nblk;
                }
                sm.info[s] = ui;
                const i32* src = a.tokens + (t0 + 16 * j0 - ui.mis);
                const u32 bytes = ui.nblk * 64 + (ui.mis ? 16u : 0u);
                const u32 bar = smem_u32(&sm.full[s]);
                mbar_expect_tx(bar, bytes);
                bulk_g2s(smem_u32(&sm.stage[s][0]), src, bytes, bar, policy);
                // advance
                ++t;
                if (t == un && it + 1 < n_units) {
                    in_bseg = false;
                    do ++r;
                    while (req_info(a, r).units == 0);  // requests without work (n_units says one with work follows)
                    t = 0;
                    fresh = true;
                }
            }
            // hand-over record (rec_tail_state is written by the consumers)
            const bool tail_open = t < un;  // the last request continues in the next range
            sm.rec_bseg_first = bseg_first;
            sm.rec_bseg_len = (u32)bseg_len;
            sm.rec_flags = (starts_mid ? CWH_REC_MID : 0u) | (in_bseg ? CWH_REC_TAIL_IS_BSEG : 0u) |
                           (tail_open ? CWH_REC_TAIL_OPEN : 0u);
        }
    } else {
        // ------------------------------------------------------------------ consumer warps
        const bool swapped = (lane >> 2) & 1;
        u32 kq[4][4], off_e[4], off_o[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const u32 q = (k + lane) & 3;  // pairs 2q and 2q+1 of the block
            kq[k][0] = q == 0 ? key_a(0) : q == 1 ? key_a(2) : q == 2 ? key_a(4) : key_a(6);
            kq[k][1] = q == 0 ? key_b(0) : q == 1 ? key_b(2) : q == 2 ? key_b(4) : key_b(6);
            kq[k][2] = q == 0 ? key_a(1) : q == 1 ? key_a(3) : q == 2 ? key_a(5) : key_a(7);
            kq[k][3] = q == 0 ? key_b(1) : q == 1 ? key_b(3) : q == 2 ? key_b(5) : key_b(7);
            off_e[k] = 16 * q + (swapped ? 64u : 0u);
            off_o[k] = 16 * q - (swapped ? 64u : 0u);  // added to 64*m with m odd: never below the lane's run
        }
        constexpr u64 A8 = cw_pow(CW_A, 8), A16 = cw_pow(CW_A, 16), A32 = cw_pow(CW_A, 32), A64 = cw_pow(CW_A, 64),
                      A128 = cw_pow(CW_A, 128), A256 = cw_pow(CW_A, 256);
        const u64 a_lane8 = pow_u64(A8, lane);  // A^(8*lane): carries the unit's carry-in to the lane's first block

        for (u32 it = warp; it < n_units; it += CWH_WARPS) {
            const u32 s = it % CWH_STAGES;
            mbar_wait(smem_u32(&sm.full[s]), (it / CWH_STAGES) & 1);
            const UnitInfo ui = sm.info[s];

            // ---- digests of the lane's 8 consecutive blocks
            const uint8_t* lane_run = &sm.stage[s][0] + lane * (64 * CWH_K);
            u64 c[CWH_K];
            if (ui.mis == 0) digest8<0>(lane_run, off_e, off_o, kq, swapped, c);
            else if (ui.mis == 1) digest8<1>(lane_run, off_e, off_o, kq, swapped, c);
            else if (ui.mis == 2) digest8<2>(lane_run, off_e, off_o, kq, swapped, c);
            else digest8<3>(lane_run, off_e, off_o, kq, swapped, c);
            __syncwarp();
            if (lane == 0) mbar_arrive(smem_u32(&sm.empty[s]));  // every lane has read stage s

            // ---- lane chain (carry-free), then one warp scan over the lane aggregates
#pragma unroll
            for (int m = 0; m < CWH_K; ++m) c[m] = cw_fin(c[m] ^ CW_K5);
#pragma unroll
            for (int m = 1; m < CWH_K; ++m) c[m] += CW_A * c[m - 1];
            u64 x = c[CWH_K - 1], y;
            y = shfl64_up(x, 1);  if (lane >= 1) x += A8 * y;
            y = shfl64_up(x, 2);  if (lane >= 2) x += A16 * y;
            y = shfl64_up(x, 4);  if (lane >= 4) x += A32 * y;
            y = shfl64_up(x, 8);  if (lane >= 8) x += A64 * y;
            y = shfl64_up(x, 16); if (lane >= 16) x += A128 * y;
            u64 before = shfl64_up(x, 1);  // carry-free chain state in front of the lane's first block
            if (lane == 0) before = 0;
            const u64 agg = shfl64(x, 31);

            // ---- hand-over: the chain state in front of this unit, the state behind it for the next warp.  Every
            //      unit waits for its predecessor's slot (also when it does not use the value), so a slot is never
            //      overwritten before it was read.
            u64 cin = 0;
            if (it > 0) {
                const u32 ps = (it - 1) % CWH_WARPS;
                mbar_wait(smem_u32(&sm.carry_bar[ps]), ((it - 1) / CWH_WARPS) & 1);
                cin = *reinterpret_cast<volatile u64*>(&sm.carry_ring[ps]);
            }
            if (ui.mode == MODE_SEED) cin = ui.seed;
            else if (ui.mode == MODE_ZERO) cin = 0;
            const u64 cout = A256 * cin + agg;  // meaningful when the unit is full (a partial unit ends its request)
            __syncwarp();                       // every lane has read the predecessor's slot
            if (lane == 0) {
                *reinterpret_cast<volatile u64*>(&sm.carry_ring[it % CWH_WARPS]) = cout;
                if (it + 1 == n_units) sm.rec_tail_state = cout;
                mbar_arrive(smem_u32(&sm.carry_bar[it % CWH_WARPS]));
            }

            // ---- final hashes of the lane's blocks: H = local + A^(m+1) * (state in front of the lane)
            const u64 front = before + a_lane8 * cin;
            const u32 first = lane * CWH_K;
            const u32 nv = ui.nblk > first ? ui.nblk - first : 0u;  // valid blocks of this lane
            u64* dst = a.hashes + ui.out_base + first;
            u64 h[CWH_K];
#pragma unroll
            for (int m = 0; m < CWH_K; ++m) h[m] = c[m] + cw_pow(CW_A, m + 1) * front;
            if ((reinterpret_cast<uintptr_t>(dst) & 15) == 0 && nv >= CWH_K) {
#pragma unroll
                for (int m = 0; m < CWH_K; m += 2) *reinterpret_cast<ulonglong2*>(dst + m) = make_ulonglong2(h[m], h[m + 1]);
            } else {
#pragma unroll
                for (int m = 0; m < CWH_K; ++m)
                    if ((u32)m < nv) dst[m] = h[m];
            }
        }
    }

    // ---- hand-over and boundary patch
    __syncthreads();
    const u32 flags = sm.rec_flags;
    const u32 bseg_len = sm.rec_bseg_len;
    if (warp == 0) {
        // Publish at once, never after a wait: a range that lies wholly inside one request publishes its CARRY-FREE
        // tail together with its length; the reader folds such records while walking back to the first final one
        // (decoupled look-back over ranges: every CTA walks on its own, nobody waits for a chain of CTAs).
        if (lane == 0) {
            const bool dependent = (flags & CWH_REC_TAIL_IS_BSEG) != 0;
            a.rec[range].tail = sm.rec_tail_state;
            a.rec[range].len_kind = dependent ? (bseg_len | 0x80000000u) : 0u;
            st_release_u32(&a.rec[range].ready, epoch);
        }
        // The walk is WARP-PARALLEL: lane i looks at record range-1-i, all 32 records are polled together, and the
        // records up to the first final one are folded with a multiplicative warp scan of A^len — a request of 8192
        // blocks spans 8 ranges, and one dependent L2 round trip per record made the last CTAs finish 8 us late.
        u64 carry_in = 0;
        if (flags & CWH_REC_MID) {  // the true chain state at the end of the previous range
            u64 mult = 1;           // product of A^len over the records folded in earlier rounds (warp-uniform)
            i32 k_hi = (i32)range - 1;
            for (;;) {
                const i32 k = k_hi - (i32)lane;
                const cw_hash_rec* prev = a.rec + (k >= 0 ? k : 0);
                u32 nuse;
                bool fin_found;
                for (;;) {  // poll until the records from k_hi down to the first final one are all published
                    const bool ready = k < 0 || ld_acquire_u32(&prev->ready) == epoch;
                    const bool fin = k < 0 || (ready && !(*reinterpret_cast<const volatile u32*>(&prev->len_kind) & 0x80000000u));
                    const u32 rmask = __ballot_sync(0xffffffffu, ready);
                    const u32 fmask = __ballot_sync(0xffffffffu, fin);
                    const u32 first_fin = fmask ? (u32)__ffs(fmask) - 1 : 32u;
                    const u32 need = first_fin >= 32 ? 0xffffffffu : ((2u << first_fin) - 1);  // lanes 0..first_fin
                    if ((rmask & need) == need) {
                        fin_found = first_fin < 32;
                        nuse = fin_found ? first_fin + 1 : 32u;
                        break;
                    }
                }
                u64 tail = 0, f = 1;
                if (k >= 0 && lane < nuse) {
                    tail = ld_relaxed_u64(&prev->tail);
                    const u32 lk = *reinterpret_cast<const volatile u32*>(&prev->len_kind);
                    if (lk & 0x80000000u) f = pow_u64(CW_A, lk & 0x7FFFFFFFu);
                }
                u64 incl = f;  // inclusive product scan of the factors
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) {
                    const u64 y = shfl64_up(incl, d);
                    if (lane >= (u32)d) incl *= y;
                }
                u64 excl = shfl64_up(incl, 1);
                if (lane == 0) excl = 1;
                u64 term = lane < nuse ? mult * excl * tail : 0ull;
#pragma unroll
                for (int d = 16; d; d >>= 1) term += shfl64_xor(term, d);
                carry_in += term;
                if (fin_found) break;  // reached a final record (range 0 is always final; k < 0 counts as final)
                mult *= shfl64(incl, 31);
                k_hi -= 32;
            }
        }
        if (lane == 0) sm.carry_in = carry_in;
    }
    __syncthreads();
    if ((flags & CWH_REC_MID) && bseg_len) {
        const u64 carry_in = sm.carry_in;
        const u64 first = sm.rec_bseg_first;
        u64 m = pow_u64(CW_A, (u64)tid + 1);
        const u64 stride = pow_u64(CW_A, blockDim.x);
        for (u32 j = tid; j < bseg_len; j += blockDim.x) {
            a.hashes[first + j] += m * carry_in;
            m *= stride;
        }
    }
    call_done();
}

}  // namespace

int cwi_hash_grid(int n_sm) {
    int per_sm = 0;
    cudaFuncSetAttribute(hash_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(HashSmem));
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, hash_kernel, CWH_THREADS, sizeof(HashSmem));
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
    a.plan = ctx->hash_plan;
    a.rec = ctx->hash_rec;
    a.status = ctx->d_status;
    a.max_hashed = ctx->cfg.max_hashed_blocks;
    a.R = R;
    // never more CTAs than units could exist; small calls stay small
    u64 max_units = (ctx->cfg.max_hashed_blocks >> CWH_UNIT_LOG2) + R;
    int grid = (int)((u64)ctx->hash_grid < max_units ? (u64)ctx->hash_grid : max_units);
    if (grid < 1) grid = 1;
    hash_kernel<<<grid, CWH_THREADS, sizeof(HashSmem), ctx->s_main>>>(a);
    CW_LAUNCH_CHECK(ctx);
    return CW_OK;
}

// ------------------------------------------------------------------------------------- no-allocation entry point
// cw_hash_blocks_static: the same kernel, for callers that can create no cw_ctx because they may not call
// cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).  The scratch the ctx
// would own — the plan words, one hand-over record per CTA, a status word — lives in ONE file-scope device array of
// fixed size (CWH_STATIC_BYTES, about 32 KiB), held by every GPU that loads the library until the process exits.
// Limits: R <= CW_HASH_STATIC_MAX_REQUESTS (the stated maximum of this entry point); any number of blocks.
//
// Host code must not hand `g_hash_static` itself to a kernel: in host code that name is a host-side stand-in, not a
// device address.  The device address is fetched once per device with cudaGetSymbolAddress (that device current) and
// kept in g_static_dev[]; the kernels get that pointer.
//
// Every call shares the array and it keeps the last call's contents.  What must start at zero — the range ticket and
// the CTAs-done counter — is cleared at the start of every call (cudaMemsetAsync on the caller's stream: no
// allocation); the epoch word deliberately persists (records of earlier calls go stale by epoch); the records are
// rewritten before they are read.  Two calls that overlap on the GPU (different streams, or graph branches)
// RACE on the array: the caller serialises them.
namespace {

constexpr u32 CWH_STATIC_MAX_R = 16384;    // == CW_HASH_STATIC_MAX_REQUESTS in cachewise.h
constexpr u32 CWH_STATIC_MAX_GRID = 2048;  // hand-over records (the grid is clamped to this)

struct HashStaticScratch {
    u64 plan[4];  // [1] call epoch, [2] range ticket, [3] CTAs done
    cw_hash_rec rec[CWH_STATIC_MAX_GRID];
    u32 status;   // device-detected conditions when the caller passes no d_status
    u32 pad[3];
};
constexpr size_t CWH_STATIC_BYTES = sizeof(HashStaticScratch);
static_assert(CWH_STATIC_BYTES <= (64u << 10), "the static scratch is meant to stay modest");

static __device__ __align__(256) unsigned char g_hash_static[CWH_STATIC_BYTES];

struct StaticDev {
    HashStaticScratch* scratch = nullptr;  // DEVICE address of g_hash_static on this device
    int grid = 0;
    bool ready = false;
};
constexpr int CWH_STATIC_MAX_DEVICES = 64;
StaticDev g_static_dev[CWH_STATIC_MAX_DEVICES];
std::mutex g_static_mu;

// once per device, with that device current
int32_t static_setup(int dev, StaticDev** out) {
    std::lock_guard<std::mutex> lock(g_static_mu);
    StaticDev& d = g_static_dev[dev];
    if (!d.ready) {
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, g_hash_static) != cudaSuccess || p == nullptr) return CW_E_CUDA;
        int n_sm = 0;
        if (cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n_sm < 1)
            return CW_E_CUDA;
        int grid = cwi_hash_grid(n_sm);  // sets the kernel's shared-memory opt-in on this device as well
        if (cudaGetLastError() != cudaSuccess) return CW_E_CUDA;
        d.scratch = static_cast<HashStaticScratch*>(p);
        d.grid = grid < (int)CWH_STATIC_MAX_GRID ? grid : (int)CWH_STATIC_MAX_GRID;
        d.ready = true;
    }
    *out = &d;
    return CW_OK;
}

}  // namespace

extern "C" {
#pragma GCC visibility push(default)

int32_t cw_hash_blocks_static(const int32_t* d_tokens, const uint64_t* d_tok_off, const uint32_t* d_start_block,
                              const uint64_t* d_start_state, const uint64_t* d_salt, const uint64_t* d_hash_off,
                              uint32_t R, uint64_t max_hashed_blocks, uint64_t* d_hashes, uint32_t* d_status,
                              void* stream) {
    if (R == 0) return CW_OK;
    if (R > CWH_STATIC_MAX_R) {
        fprintf(stderr, "cw_hash_blocks_static: R = %u exceeds the static scratch (at most %u requests per call)\n", R,
                CWH_STATIC_MAX_R);
        return CW_E_INVAL;
    }
    if (!d_tokens || !d_tok_off || !d_hash_off || !d_hashes) return CW_E_INVAL;
    if (d_start_block && !d_start_state) return CW_E_INVAL;
    if (!cw_aligned16(d_tokens) || (reinterpret_cast<uintptr_t>(d_tok_off) & 7) ||
        (reinterpret_cast<uintptr_t>(d_hash_off) & 7) || (reinterpret_cast<uintptr_t>(d_hashes) & 7) ||
        (reinterpret_cast<uintptr_t>(d_status) & 3))
        return CW_E_INVAL;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return CW_E_CUDA;
    if (dev < 0 || dev >= CWH_STATIC_MAX_DEVICES) return CW_E_INVAL;
    StaticDev* sd = nullptr;
    const int32_t rc = static_setup(dev, &sd);
    if (rc != CW_OK) return rc;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    HashStaticScratch* sc = sd->scratch;  // device address; members are only ever dereferenced on the device

    // what must start at zero: the range ticket and the CTAs-done counter (plan[2], plan[3]); the epoch stays
    if (cudaMemsetAsync(reinterpret_cast<unsigned char*>(sc) + offsetof(HashStaticScratch, plan) + 2 * sizeof(u64), 0,
                        2 * sizeof(u64), s) != cudaSuccess)
        return CW_E_CUDA;
    HashArgs a;
    a.tokens = d_tokens;
    a.tok_off = d_tok_off;
    a.start_block = d_start_block;
    a.start_state = d_start_state;
    a.salt = d_salt;
    a.hash_off = d_hash_off;
    a.hashes = d_hashes;
    a.plan = reinterpret_cast<u64*>(reinterpret_cast<unsigned char*>(sc) + offsetof(HashStaticScratch, plan));
    a.rec = reinterpret_cast<cw_hash_rec*>(reinterpret_cast<unsigned char*>(sc) + offsetof(HashStaticScratch, rec));
    a.status = d_status ? d_status
                        : reinterpret_cast<u32*>(reinterpret_cast<unsigned char*>(sc) + offsetof(HashStaticScratch, status));
    a.max_hashed = max_hashed_blocks;
    a.R = R;
    const u64 max_units = (max_hashed_blocks >> CWH_UNIT_LOG2) + R;
    int grid = (int)((u64)sd->grid < max_units ? (u64)sd->grid : max_units);
    if (grid < 1) grid = 1;
    hash_kernel<<<grid, CWH_THREADS, sizeof(HashSmem), s>>>(a);
    if (cudaGetLastError() != cudaSuccess) return CW_E_CUDA;
    return CW_OK;
}

#pragma GCC visibility pop
}  // extern "C"
