// Stage 2a — resident-block table and prefix match (cw_match_prefix, cw_table_*).  DESIGN.md R2.
//
// Table: 2^t slots of 16 bytes {key u64, loc u32, idx u32}, linear probing from slot (key & mask).  Two
// slots share a 32-byte sector, eight a 128-byte line, so a probe sequence walks one line before it
// touches the next ("coalesced buckets").  Lookups are wait-free reads (one LDG.128 per slot).
//
// Insert is lock-free and DETERMINISTIC (result independent of CAS order):
//   pass 1  walk to the key or to the end of the cluster; claim the first reusable slot with a 64-bit CAS on
//           the key; every thread of the same key then atomicMin's its input index into slot.idx
//   pass 2  slot.loc == PENDING  <=> the key was claimed in this batch: input idx wins and writes its loc;
//           every input reports the surviving loc
//   pass 3  the winners restore slot.idx = 0xFFFFFFFF
// (All same-key threads follow one probe sequence whose slots only go from reusable to occupied during the
// batch, so they converge on the same slot.)
// A batch that could fill the table (live keys + batch > slots, decided on the host from an exact device counter)
// is inserted by ONE thread in input order instead: which keys still find a slot is then the oracle's rule
// (first come by input index), and the parallel path can never meet a full table.
//
// Erase leaves a TOMBSTONE (or EMPTY when the next slot is EMPTY: the cluster ends there, nothing can lie behind).
// Tombstones are reclaimed by inserts that pass them and by COMPACTION: once the erases since the last compaction
// could have turned a quarter of the slots into tombstones, the live entries are re-inserted into a second buffer
// and copied back (the table address never changes, so captured graphs stay valid).  Every probe loop is bounded
// by one full cycle: a table without EMPTY slots answers MISS for an absent key instead of spinning.
//
// Match: flat over hashes[]; a warp task is 128 consecutive hashes (one 32-ary search over hash_off for its first
// request).  A task inside one request is probed LANE-INDEPENDENTLY: lane l owns hashes l + 32k, keys and results are
// staged per warp in shared memory, every iteration of a warp-synchronous loop issues one slot load per live lane and
// each lane walks its own keys front to back; the first missing position is min-reduced over the warp and lanes stop
// at it.  Tasks that cross a request boundary walk round by round (32 hashes, one lane per hash); rounds that lie behind
// a miss already seen for their request are answered without a probe.  Per request: first_miss = atomicMin, max_hit =
// atomicMax over hits that are not already behind a miss of their own task / round; a small per-request kernel then
// writes k_total / n_gpu and blanks hits that lie behind the first miss (rare), and re-arms the scratch for the next
// call.  hit_loc is written with streaming stores and the hashes are read with streaming loads: neither is re-read
// by this pass, and the table should own the L2.
#include <stdio.h>

#include <algorithm>

#include "cw_internal.cuh"

namespace {

__device__ __forceinline__ uint4 ld_slot(const cw_slot* s) { return *reinterpret_cast<const uint4*>(s); }
__device__ __forceinline__ u64 slot_key(const uint4& v) { return ((u64)v.y << 32) | v.x; }

// returns slot index of `key` (already remapped) or ~0 if absent
__device__ __forceinline__ u64 table_find(const cw_slot* table, u64 mask, u64 key, u32* loc) {
    u64 i = key & mask & ~1ull;  // homes are even slots: a home PAIR is one 32-byte sector
    for (u64 n = 0; n <= mask; ++n) {
        const uint4 v = ld_slot(table + i);
        const u64 k = slot_key(v);
        if (k == key) {
            *loc = v.z;
            return i;
        }
        if (k == CW_KEY_EMPTY) break;
        i = (i + 1) & mask;
    }
    *loc = CW_MISS;
    return ~0ull;
}

// Probe of the match pass: ONE 128-bit load per slot (the generic ld_slot is split by the compiler into a key load
// and a dependent loc load: a second memory latency on every hit), 32-bit index arithmetic.
__device__ __forceinline__ u32 table_probe(const cw_slot* __restrict__ table, u32 mask, u64 key) {
    u32 i = (u32)key & mask & ~1u;
    for (u32 n = 0; n <= mask; ++n) {
        uint4 v;
        asm volatile("ld.global.nc.v4.u32 {%0, %1, %2, %3}, [%4];"
                     : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
                     : "l"(table + i));
        const u64 k = slot_key(v);
        if (k == key) return v.z;
        if (k == CW_KEY_EMPTY) break;
        i = (i + 1) & mask;
    }
    return CW_MISS;
}

__global__ void lookup_kernel(const cw_slot* table, u64 mask, const u64* keys, u32 n, u32* loc) {
    u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    u32 l;
    table_find(table, mask, cw_remap_key(keys[i]), &l);
    loc[i] = l;
}

// one counter update per warp: live keys, tombstones
__device__ __forceinline__ void count_add(u32* cnt, bool live_up, bool live_down, bool tomb_up, bool tomb_down) {
    const u32 lu = __popc(__ballot_sync(0xffffffffu, live_up)), ld = __popc(__ballot_sync(0xffffffffu, live_down));
    const u32 tu = __popc(__ballot_sync(0xffffffffu, tomb_up)), td = __popc(__ballot_sync(0xffffffffu, tomb_down));
    if ((threadIdx.x & 31) == 0) {
        if (lu != ld) atomicAdd(&cnt[0], lu - ld);  // wraps for a negative difference: the sum stays exact
        if (tu != td) atomicAdd(&cnt[1], tu - td);
    }
}

__global__ void erase_kernel(cw_slot* table, u64 mask, const u64* keys, u32 n, u32* cnt) {
    u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    bool erased = false, tomb = false;
    if (i < n) {
        const u64 key = cw_remap_key(keys[i]);
        u32 l;
        u64 s = table_find(table, mask, key, &l);
        if (s != ~0ull) {
            // duplicates of a key inside the batch: exactly one thread wins the CAS and counts the erase
            const u64 old = atomicCAS(reinterpret_cast<unsigned long long*>(&table[s].key), (unsigned long long)key,
                                      (unsigned long long)CW_KEY_TOMB);  // idx stays 0xFFFFFFFF, loc is dead
            if (old == key) {
                erased = true;
                // the cluster ends behind this slot: no probe sequence continues past it, so it can be EMPTY again
                // (EMPTY slots never change during an erase batch; a neighbour erased concurrently is seen either as
                // a key or as a tombstone -> this slot keeps its tombstone, which is still correct)
                const u64 next = *reinterpret_cast<volatile unsigned long long*>(&table[(s + 1) & mask].key);
                if (next == CW_KEY_EMPTY) *reinterpret_cast<volatile unsigned long long*>(&table[s].key) = CW_KEY_EMPTY;
                else tomb = true;
            }
        }
    }
    count_add(cnt, false, erased, tomb, false);
}

__global__ void retag_kernel(cw_slot* table, u64 mask, const u64* keys, const u32* new_loc, u32 n) {
    u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    u32 l;
    u64 s = table_find(table, mask, cw_remap_key(keys[i]), &l);
    if (s != ~0ull) table[s].loc = new_loc[i];
}

__global__ void insert_claim_kernel(cw_slot* table, u64 mask, const u64* keys, u32 n, u32* ins_slot, u32* status,
                                    u32* cnt) {
    u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    bool claimed = false, from_tomb = false;
    if (i < n) {
        const u64 key = cw_remap_key(keys[i]);
        const u64 home = key & mask & ~1ull;
        u64 pos = home, steps = 0;
        u64 found = ~0ull;
        for (;;) {
            // walk until the key, the end of the cluster (EMPTY) or a full cycle; remember the first reusable slot
            u64 cand = ~0ull, cand_expect = 0;
            while (steps <= mask) {
                const u64 k = *reinterpret_cast<volatile unsigned long long*>(&table[pos].key);
                if (k == key) {
                    found = pos;
                    break;
                }
                if (k == CW_KEY_TOMB && cand == ~0ull) {
                    cand = pos;
                    cand_expect = CW_KEY_TOMB;
                }
                if (k == CW_KEY_EMPTY) {
                    if (cand == ~0ull) {
                        cand = pos;
                        cand_expect = CW_KEY_EMPTY;
                    }
                    break;
                }
                pos = (pos + 1) & mask;
                ++steps;
            }
            if (found != ~0ull || cand == ~0ull) break;  // present, or table full
            const u64 old = atomicCAS(reinterpret_cast<unsigned long long*>(&table[cand].key),
                                      (unsigned long long)cand_expect, (unsigned long long)key);
            if (old == cand_expect) {
                table[cand].loc = CW_LOC_PENDING;
                found = cand;
                claimed = true;
                from_tomb = cand_expect == CW_KEY_TOMB;
                break;
            }
            if (old == key) {
                found = cand;
                break;
            }
            // another key took the slot: every slot before it is occupied by other keys for the rest of the
            // batch, so the walk resumes there
            pos = cand;
            steps = (cand - home) & mask;
        }
        if (found != ~0ull) {
            atomicMin(&table[found].idx, i);
            ins_slot[i] = (u32)found;
        } else {
            ins_slot[i] = 0xFFFFFFFFu;
            atomicOr(status, CWS_CAPACITY);
        }
    }
    count_add(cnt, claimed, false, false, from_tomb);
}

// A batch that could fill the table: ONE thread inserts in input order, so the keys that still find a slot are the
// first ones by input index (the oracle's rule; R2).  Misuse path (cw_create sizes the table for a load
// factor <= 0.5): speed is irrelevant.
__global__ void insert_seq_kernel(cw_slot* table, u64 mask, const u64* keys, const u32* loc, u32 n, u32* winner_loc,
                                  u32* status, u32* cnt) {
    if (blockIdx.x || threadIdx.x) return;
    u32 live = cnt[0], tombs = cnt[1];
    for (u32 i = 0; i < n; ++i) {
        const u64 key = cw_remap_key(keys[i]);
        u64 pos = key & mask & ~1ull, cand = ~0ull, found = ~0ull;
        for (u64 steps = 0; steps <= mask; ++steps) {
            const u64 k = table[pos].key;
            if (k == key) {
                found = pos;
                break;
            }
            if (k == CW_KEY_TOMB && cand == ~0ull) cand = pos;
            if (k == CW_KEY_EMPTY) {
                if (cand == ~0ull) cand = pos;
                break;
            }
            pos = (pos + 1) & mask;
        }
        u32 w = CW_MISS;
        if (found != ~0ull) {
            w = table[found].loc;
        } else if (cand != ~0ull) {
            if (table[cand].key == CW_KEY_TOMB) --tombs;
            ++live;
            w = loc[i];
            table[cand].key = key;
            table[cand].loc = w;
            table[cand].idx = 0xFFFFFFFFu;
        } else {
            atomicOr(status, CWS_CAPACITY);
        }
        if (winner_loc) winner_loc[i] = w;
    }
    cnt[0] = live;
    cnt[1] = tombs;
}

// Compaction: every live entry of `src` is re-inserted into the (cleared) second buffer; keys are unique, so one
// CAS on the key decides the slot.
__global__ void rebuild_kernel(const cw_slot* __restrict__ src, cw_slot* dst, u64 n_slots) {
    const u64 mask = n_slots - 1;
    for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < n_slots; i += (u64)gridDim.x * blockDim.x) {
        const uint4 v = ld_slot(src + i);
        const u64 key = slot_key(v);
        if (key == CW_KEY_EMPTY || key == CW_KEY_TOMB) continue;
        u64 pos = key & mask & ~1ull;
        for (u64 steps = 0; steps <= mask; ++steps) {
            const u64 old = atomicCAS(reinterpret_cast<unsigned long long*>(&dst[pos].key),
                                      (unsigned long long)CW_KEY_EMPTY, (unsigned long long)key);
            if (old == CW_KEY_EMPTY) {
                dst[pos].loc = v.z;
                break;
            }
            pos = (pos + 1) & mask;
        }
    }
}

// cw_table_stats: exact recount of live keys / tombstones and the histogram of probe lengths (slots examined to
// find each resident key = its distance from the home slot + 1).
__global__ void stats_kernel(const cw_slot* __restrict__ table, u64 n_slots, u32* cnt, u32* hist) {
    const u64 mask = n_slots - 1;
    u32 live = 0, tombs = 0, longest = 0;
    for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < n_slots; i += (u64)gridDim.x * blockDim.x) {
        const u64 key = slot_key(ld_slot(table + i));
        if (key == CW_KEY_TOMB) ++tombs;
        else if (key != CW_KEY_EMPTY) {
            ++live;
            const u64 d = ((i - (key & mask & ~1ull)) & mask) + 1;
            longest = max(longest, (u32)min(d, (u64)0xFFFFFFFFull));
            atomicAdd(&hist[min(d, (u64)CWT_HIST_BINS) - 1], 1u);
        }
    }
    live = __reduce_add_sync(0xffffffffu, live);
    tombs = __reduce_add_sync(0xffffffffu, tombs);
    longest = __reduce_max_sync(0xffffffffu, longest);
    if ((threadIdx.x & 31) == 0) {
        if (live) atomicAdd(&cnt[0], live);
        if (tombs) atomicAdd(&cnt[1], tombs);
        if (longest) atomicMax(&cnt[2], longest);
    }
}

__global__ void insert_resolve_kernel(cw_slot* table, const u32* loc, u32 n, const u32* ins_slot, u32* winner_loc) {
    u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const u32 s = ins_slot[i];
    if (s == 0xFFFFFFFFu) {
        if (winner_loc) winner_loc[i] = CW_MISS;
        return;
    }
    const u32 w = table[s].idx;
    u32 l = *reinterpret_cast<volatile u32*>(&table[s].loc);
    if (l == CW_LOC_PENDING) {  // claimed in this batch: the lowest input index owns it
        l = loc[w];
        if (w == i) table[s].loc = l;
    }
    if (winner_loc) winner_loc[i] = l;
}

__global__ void insert_reset_kernel(cw_slot* table, u32 n, const u32* ins_slot) {
    u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const u32 s = ins_slot[i];
    if (s != 0xFFFFFFFFu && table[s].idx == i) table[s].idx = 0xFFFFFFFFu;
}

// ---------------------------------------------------------------------------------------------- match
// full occupancy (<= 32 registers, 2048 threads per SM): the probe is bound by resident warps x latency (93 us vs 107 us
// at 6 CTAs/SM on configs[2])
#define MATCH_THREADS 64  // measured on configs[2]: 256 -> 66.1 us, 128 -> 65.9, 64 -> 64.6 (CTA slots turn over per 2 tasks)
#define MATCH_MIN_CTAS (2048 / MATCH_THREADS)
#define CWM_CHUNK 128  // consecutive hashes handled by one warp task (4 rounds of 32): measured optimum on configs[2]
                       // (64: 89 us, 128: 75, 256: 79, 512: ~85, 1024: ~100, 2048: ~170 — long tasks are bound by the
                       // dependent probe chain of the slowest warp, short ones by the per-task search and set-up)

__global__ void __launch_bounds__(MATCH_THREADS, MATCH_MIN_CTAS) match_probe_kernel(const cw_slot* __restrict__ table, u32 mask,
                                                          const u64* __restrict__ hashes,
                                                          const u64* __restrict__ hash_off, u32 R, u32* first_miss,
                                                          u32* max_hit, u32* host_hits, u32* hit_loc, u32* status,
                                                          const uint2* __restrict__ list,
                                                          const u32* __restrict__ list_n) {
    // list (cw_match_prefix_shared only, else NULL): the tasks to probe, in no particular order, as (request, first
    // position inside the request) pairs: up to CWM_CHUNK positions of ONE request each, so every task takes the
    // lane-independent path below; the plain call walks the flat CSR in CWM_CHUNK-aligned tasks instead
    __shared__ u64 s_key[MATCH_THREADS / 32][CWM_CHUNK];
    __shared__ u32 s_loc[MATCH_THREADS / 32][CWM_CHUNK];
    // hash_off may be a slice of a longer CSR array: positions below are 32-bit offsets from its first hash
    const u64 h_first = hash_off[0];
    if (hash_off[R] - h_first > 0xFFFFFFFFull) {  // more than 2^32 hashes in one call: not supported
        if (blockIdx.x == 0 && threadIdx.x == 0) atomicOr(status, CWS_INVAL);
        return;
    }
    const u32 total = (u32)(hash_off[R] - h_first);
    const u64* __restrict__ hs = hashes + h_first;
    u32* hl = hit_loc ? hit_loc + h_first : nullptr;
    const u32 lane = threadIdx.x & 31;
    const u32 nwarps = (gridDim.x * blockDim.x) >> 5;
    const u32 n_tasks = list ? *list_n : (total + CWM_CHUNK - 1) / CWM_CHUNK;
    // a warp walks its task front to back, so once it has seen a miss of a request the rest of that request is
    // answered without touching the table (the leading run is over); a miss recorded by an earlier task of the
    // same request is honoured too when the warp enters that request
    for (u32 wi = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; wi < n_tasks; wi += nwarps) {
        uint2 le = make_uint2(0u, 0u);
        if (list) le = list[wi];
        u32 c0 = wi * CWM_CHUNK;
        // largest r with hash_off[r] <= c0 (r < R), 32-ary search, warp-uniform, once per task (a listed task names it)
        u32 lo = le.x, hi = list ? lo + 1 : R;
        while (hi - lo > 1) {
            u32 step = (hi - lo + 31) >> 5;
            u32 p = lo + lane * step;
            bool ok = p < hi && (u32)(hash_off[p] - h_first) <= c0;
            u32 cnt = __popc(__ballot_sync(0xffffffffu, ok));
            u32 nlo = lo + (cnt - 1) * step;
            hi = min(hi, nlo + step);
            lo = nlo;
        }
        u32 r_base = lo;  // request of the first hash of the current round (kept up to date below)
        u32 req_start = (u32)(hash_off[lo] - h_first), req_end = (u32)(hash_off[lo + 1] - h_first);
        u32 dead_r = 0xFFFFFFFFu, checked_r = 0xFFFFFFFFu;  // request known to have missed / whose global state was read
        if (list) c0 = req_start + le.y;
        const u32 c1 = list ? min(req_end, c0 + CWM_CHUNK) : min(total, c0 + CWM_CHUNK);
        if (c1 <= req_end) {
            // ---- the whole task lies inside request r_base (the common case): LANE-INDEPENDENT probing.  Lane l
            // owns the hashes c0 + l + 32k (coalesced) and walks them front to back on its own, one slot load per
            // iteration of a warp-synchronous loop, so the warp waits for the longest SUM of probe lengths over a
            // lane's keys instead of the sum over rounds of the longest probe of the round.
            const u32 j0 = c0 - req_start;
            if (j0 > 0 && __ldcg(first_miss + r_base) < j0) {  // an earlier task of the request already missed
                if (hl)
                    for (u32 g = c0 + lane; g < c1; g += 32) __stcs(hl + g, CW_MISS);
                continue;
            }
            constexpr int KPL = CWM_CHUNK / 32;  // keys per lane
            const u32 n_task = c1 - c0;
            u64* wkey = s_key[threadIdx.x >> 5];  // this warp's staged (remapped) keys and resolved locations
            u32* wloc = s_loc[threadIdx.x >> 5];
            {
                u64 kk[KPL];
                // UNCONDITIONAL loads at clamped positions: a predicated load followed by its own use is not hoisted by
                // the compiler, and the four loads then complete one after the other
#pragma unroll
                for (int q = 0; q < KPL; ++q)  // in flight together; streaming (evict-first): the table stays in L2
                    kk[q] = __ldcs(hs + c0 + min(lane + 32 * q, n_task - 1));
#pragma unroll
                for (int q = 0; q < KPL; ++q) wkey[lane + 32 * q] = cw_remap_key(kk[q]);  // read back by this lane only
            }
            u32 pos = lane;          // position of this lane's current key inside the task
            u32 limit = n_task;      // warp-uniform: min(n_task, first missing position seen so far)
            uint2 key = *reinterpret_cast<const uint2*>(wkey + pos);
            const u32 pmask = mask >> 1;          // the table as pairs of slots: one 32-byte sector each
            u32 pair = (key.x & mask) >> 1;       // homes are even slots
            for (;;) {
                const bool live = pos < limit;
                if (!__any_sync(0xffffffffu, live)) break;
                u32 miss_at = 0xFFFFFFFFu;
                if (live) {
                    // ONE 256-bit load examines both slots of the sector (LDG.E.ENL2.256): the same load wavefront and
                    // the same L2 sector as a single slot, and 1.2 instead of 1.5 dependent steps per resident key
                    u64 a0, a1, b0, b1;
                    asm volatile("ld.global.nc.v4.u64 {%0, %1, %2, %3}, [%4];"
                                 : "=l"(a0), "=l"(a1), "=l"(b0), "=l"(b1)
                                 : "l"(table + 2 * (u64)pair));
                    const u64 k64 = ((u64)key.y << 32) | key.x;
                    const bool hit_a = a0 == k64, end_a = a0 == CW_KEY_EMPTY;
                    const bool hit_b = !hit_a && !end_a && b0 == k64;
                    const bool end_b = !hit_a && !end_a && !hit_b && b0 == CW_KEY_EMPTY;
                    pair = (pair + 1) & pmask;
                    const bool hit = hit_a || hit_b;
                    // EMPTY ends the cluster; so does a full cycle (a table without EMPTY slots must not spin)
                    const bool empty = end_a || end_b || (!hit && pair == ((key.x & mask) >> 1));
                    if (hit || empty) {  // resolved: record, next key of this lane
                        wloc[pos] = hit ? (u32)(hit_a ? a1 : b1) : CW_MISS;
                        if (empty) miss_at = pos;
                        pos += 32;
                        key = *reinterpret_cast<const uint2*>(wkey + (pos & (CWM_CHUNK - 1)));
                        pair = (key.x & mask) >> 1;
                    }
                }
                if (__any_sync(0xffffffffu, miss_at != 0xFFFFFFFFu)) limit = min(limit, __reduce_min_sync(0xffffffffu, miss_at));
            }
            __syncwarp();
            // hits behind the first miss are not part of the prefix
            u32 host = 0;
#pragma unroll
            for (int q = 0; q < KPL; ++q) {
                const u32 p = lane + 32 * q;
                const u32 l = p < limit ? wloc[p] : CW_MISS;
                host += (l != CW_MISS && (l & CW_HOST_BIT)) ? 1u : 0u;
                if (hl && p < n_task) __stcs(hl + c0 + p, l);  // streaming: hit_loc is not re-read by this kernel
            }
            host = __reduce_add_sync(0xffffffffu, host);
            if (lane == 0) {
                if (limit < n_task) atomicMin(&first_miss[r_base], j0 + limit);
                if (limit) atomicMax(&max_hit[r_base], j0 + limit);
                if (host) atomicAdd(&host_hits[r_base], host);
            }
            __syncwarp();  // the staging rows are reused by the next task of this warp
            continue;
        }
        u64 key_next = c0 + lane < c1 ? hs[c0 + lane] : 0;
        for (u32 g0 = c0; g0 < c1; g0 += 32) {
            while (g0 >= req_end) {  // warp-uniform; also skips empty requests
                ++r_base;
                req_start = req_end;
                req_end = (u32)(hash_off[r_base + 1] - h_first);
            }
            const u32 g = g0 + lane;
            const bool active = g < c1;
            const u64 key = key_next;
            if (g + 32 < c1) key_next = hs[g + 32];  // prefetch the next round
            u32 r = r_base;
            u32 j = g - req_start;
            bool uniform = true;
            if (min(g0 + 32, c1) > req_end) {  // the round crosses into the next request(s): per-lane walk (rare)
                if (active)
                    while (g >= (u32)(hash_off[r + 1] - h_first)) ++r;
                j = active ? g - (u32)(hash_off[r] - h_first) : 0;
                uniform = __all_sync(0xffffffffu, !active || r == r_base);
            }
            if (uniform) {
                if (r_base != checked_r && r_base != dead_r) {  // entering a request: did an earlier task miss?
                    checked_r = r_base;
                    const u32 j0 = g0 - req_start;
                    if (j0 > 0 && __ldcg(first_miss + r_base) < j0) dead_r = r_base;
                }
                if (r_base == dead_r) {  // the whole round lies behind a known miss
                    if (active && hl) __stcs(hl + g, CW_MISS);
                    continue;
                }
            }
            u32 loc = CW_MISS;
            if (active) loc = table_probe(table, mask, cw_remap_key(key));
            if (uniform) {
                const u32 act_mask = __ballot_sync(0xffffffffu, active);
                const u32 miss_mask = __ballot_sync(0xffffffffu, active && loc == CW_MISS);
                const u32 first = miss_mask ? (u32)__ffs(miss_mask) - 1 : 32;
                if (lane > first) loc = CW_MISS;
                const u32 hit_mask = act_mask & (first >= 32 ? 0xffffffffu : ((1u << first) - 1));
                const u32 host_mask = __ballot_sync(0xffffffffu, active && loc != CW_MISS && (loc & CW_HOST_BIT));
                if (miss_mask) dead_r = r_base;
                if (lane == 0) {
                    if (miss_mask) atomicMin(&first_miss[r], j + first);
                    if (hit_mask) atomicMax(&max_hit[r], j + (32 - __clz(hit_mask)));
                    if (host_mask) atomicAdd(&host_hits[r], __popc(host_mask));
                }
            } else if (active) {
                if (loc == CW_MISS) {
                    atomicMin(&first_miss[r], j);
                } else {
                    atomicMax(&max_hit[r], j + 1);
                    if (loc & CW_HOST_BIT) atomicAdd(&host_hits[r], 1u);
                }
            }
            if (active && hl) __stcs(hl + g, loc);
        }
    }
}

// one warp per request
__global__ void __launch_bounds__(256) match_finish_kernel(const u64* __restrict__ hash_off, u32 R, u32* first_miss,
                                                           u32* max_hit, u32* host_hits, u32* k_total, u32* n_gpu,
                                                           u32* hit_loc, const cw_slot* __restrict__ table, u64 mask,
                                                           const u64* __restrict__ hashes) {
    const u32 lane = threadIdx.x & 31;
    const u32 r = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (r >= R) return;
    if (hash_off[R] - hash_off[0] > 0xFFFFFFFFull) return;  // rejected by the probe kernel: outputs untouched
    const u64 h0 = hash_off[r];
    const u32 n_r = (u32)(hash_off[r + 1] - h0);
    const u32 k = min(first_miss[r], n_r);
    const u32 mh = max_hit[r];
    const u32 hh = host_hits[r];
    u32 host_in_run = 0;
    if (hh) {  // count host-tier blocks inside the run (re-probe when the caller did not ask for hit_loc)
        for (u32 j = lane; j < k; j += 32) {
            u32 loc;
            if (hit_loc) loc = hit_loc[h0 + j];
            else table_find(table, mask, cw_remap_key(hashes[h0 + j]), &loc);
            host_in_run += (loc != CW_MISS && (loc & CW_HOST_BIT)) ? 1 : 0;
        }
#pragma unroll
        for (int m = 16; m; m >>= 1) host_in_run += __shfl_xor_sync(0xffffffffu, host_in_run, m);
    }
    if (hit_loc && mh > k)  // resident blocks behind the first miss are not part of the prefix
        for (u32 j = k + lane; j < mh; j += 32) hit_loc[h0 + j] = CW_MISS;
    if (lane == 0) {
        k_total[r] = k;
        n_gpu[r] = k - host_in_run;
        first_miss[r] = 0xFFFFFFFFu;  // re-arm
        max_hit[r] = 0;
        host_hits[r] = 0;
    }
}

// ---------------------------------------------------------------------------------- match with shared prefixes
// cw_match_prefix_shared.  The queue of an agent workload holds many requests of one session, and they repeat the
// session's first thousands of hashes (configs[2]: 5.4 M of 6.6 M lookups).  The caller names, per request, a LEADER
// (say the longest queued request of the session).  Because the hashes are CHAIN hashes (stage 1: H_j is a function of
// the whole token prefix), two requests that agree at position p agree at every position before p, so
//   match_lcp_kernel    finds L_r = number of leading hashes request r shares with its leader by a 32-ary search
//                       (three rounds for 8192 blocks) without touching the table, and appends the request's tasks
//                       (128 positions each, from position 0 of a leader, from L_r of a follower) to a compact list,
//   match_probe_kernel  walks that list: leaders in full, every other request from position L_r on (its own tail);
//                       a listed task lies inside one request, so all of them take the lane-independent path,
//   match_share_kernel  (one CTA per request) answers positions [0, L_r) of a follower from the leader's results,
//                       computes k_total / n_gpu and resets the list counter.
// A hint that shares nothing (or is not itself a leader) only costs the search: the request is probed on its own.
#define SHARE_THREADS 128
#define SHARE_UNROLL 8  // loads in flight per thread: a follower of 8192 shared blocks is copied in 8 rounds

// one warp per request
__global__ void __launch_bounds__(256) match_lcp_kernel(const u64* __restrict__ hashes, const u64* __restrict__ hash_off,
                                                        u32 R, const u32* __restrict__ leader, u32* lcp, uint2* list,
                                                        u32* list_n, u32* first_miss, u32* max_hit, u32* host_hits) {
    const u32 lane = threadIdx.x & 31;
    const u32 r = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (r >= R) return;
    const u64 h_first = hash_off[0];
    if (hash_off[R] - h_first > 0xFFFFFFFFull) return;  // the probe kernel rejects the call: scratch stays armed
    const u64 a0 = hash_off[r], a1 = hash_off[r + 1];
    const u32 l = leader[r];
    u32 out = 0xFFFFFFFFu;
    if (l < R && l != r && leader[l] == l) {
        const u64 b0 = hash_off[l];
        const u64 n = min(a1 - a0, hash_off[l + 1] - b0);
        const u64* __restrict__ ha = hashes + a0;
        const u64* __restrict__ hb = hashes + b0;
        u64 lo = 0, hi = n;  // every position below lo agrees; position hi (if < n) differs
        while (lo < hi) {
            const u64 step = (hi - lo + 31) >> 5;
            const u64 p = lo + lane * step;
            const bool tested = p < hi;
            const bool differs = tested && ha[p] != hb[p];
            const u32 dmask = __ballot_sync(0xffffffffu, differs);
            const u32 tmask = __ballot_sync(0xffffffffu, tested);
            if (dmask) {
                const u32 first = (u32)__ffs(dmask) - 1;  // positions up to lane first-1 agree, lane first differs
                hi = lo + first * step;
                if (first) lo = lo + (first - 1) * step + 1;
            } else {
                lo = min(hi, lo + (u64)(32 - __clz(tmask) - 1) * step + 1);  // the last tested position agrees
            }
        }
        if (lo > 0 && lo <= 0xFFFFFFFEull) out = (u32)lo;
    }
    if (lane == 0) {
        lcp[r] = out;
        // this path has its own per-request scratch and arms it here, in front of the probe kernel (the plain call's
        // scratch is re-armed by its finish kernel; a grid-wide "last CTA re-arms" costs one contended atomic per CTA)
        first_miss[r] = 0xFFFFFFFFu;
        max_hit[r] = 0;
        host_hits[r] = 0;
    }
    // the tasks of this request: CWM_CHUNK positions each, from position 0 (leader) or L (follower: its own tail) on
    const u32 n_r = (u32)(a1 - a0);
    const u32 from = out == 0xFFFFFFFFu ? 0u : out;
    const u32 n_t = (n_r - from + CWM_CHUNK - 1) / CWM_CHUNK;
    if (n_t) {
        u32 base = 0;
        if (lane == 0) base = atomicAdd(list_n, n_t);
        base = __shfl_sync(0xffffffffu, base, 0);
        for (u32 i = lane; i < n_t; i += 32) list[base + i] = make_uint2(r, from + i * CWM_CHUNK);
    }
}

// one CTA per request
__global__ void __launch_bounds__(SHARE_THREADS) match_share_kernel(
    const u64* __restrict__ hash_off, u32 R, const u32* __restrict__ leader, const u32* __restrict__ lcp, u32* first_miss,
    u32* max_hit, u32* host_hits, u32* k_total, u32* n_gpu, u32* hit_loc, const cw_slot* __restrict__ table, u64 mask,
    const u64* __restrict__ hashes, u32* list_n) {
    if (hash_off[R] - hash_off[0] > 0xFFFFFFFFull) return;  // rejected by the probe kernel: outputs and scratch untouched
    const u32 tid = threadIdx.x, lane = tid & 31;
    const u32 r = blockIdx.x;
    const u64 h0 = hash_off[r];
    const u32 n_r = (u32)(hash_off[r + 1] - h0);
    const u32 L = lcp[r];
    const bool follower = L != 0xFFFFFFFFu;
    u64 lh0 = 0;
    u32 k_l = 0;
    if (follower) {
        const u32 l = leader[r];
        lh0 = hash_off[l];
        k_l = min(first_miss[l], (u32)(hash_off[l + 1] - lh0));
    }
    // ---- (1) k_total / n_gpu (warp 0)
    if (tid < 32) {
        // the leader's run ends inside the shared prefix: so does this one; else it goes on into the own tail
        const u32 k = !follower ? min(first_miss[r], n_r) : (k_l < L ? k_l : min(first_miss[r], n_r));
        const u32 own_from = follower ? L : 0u;
        u32 hh = host_hits[r];
        if (follower) hh |= host_hits[leader[r]];
        u32 host_in_run = 0;
        if (hh) {  // count host-tier blocks inside the run (re-probe when the caller did not ask for hit_loc)
            for (u32 j = lane; j < k; j += 32) {
                u32 loc;
                const u64 at = j < own_from ? lh0 + j : h0 + j;
                if (hit_loc) loc = hit_loc[at];
                else table_find(table, mask, cw_remap_key(hashes[at]), &loc);
                host_in_run += (loc != CW_MISS && (loc & CW_HOST_BIT)) ? 1 : 0;
            }
#pragma unroll
            for (int m = 16; m; m >>= 1) host_in_run += __shfl_xor_sync(0xffffffffu, host_in_run, m);
        }
        const u32 mh = max_hit[r];
        if (hit_loc && mh > max(k, own_from))  // resident blocks of the probed part behind the run's end
            for (u32 j = max(k, own_from) + lane; j < mh; j += 32) hit_loc[h0 + j] = CW_MISS;
        if (lane == 0) {
            k_total[r] = k;
            n_gpu[r] = k - host_in_run;
        }
    }
    // ---- (2) positions [0, L) of a follower: the leader's locations up to the end of the leader's run, MISS behind
    if (follower && hit_loc) {
        const u32* src = hit_loc + lh0;
        u32* dst = hit_loc + h0;
        for (u32 j0 = 0; j0 < L; j0 += SHARE_UNROLL * SHARE_THREADS) {
            u32 v[SHARE_UNROLL];
#pragma unroll
            for (int q = 0; q < SHARE_UNROLL; ++q)  // unconditional loads at clamped positions, in flight together
                v[q] = __ldcg(src + min(j0 + tid + q * SHARE_THREADS, L - 1));
#pragma unroll
            for (int q = 0; q < SHARE_UNROLL; ++q) {
                const u32 j = j0 + tid + q * SHARE_THREADS;
                if (j < L) __stcs(dst + j, j < k_l ? v[q] : CW_MISS);
            }
        }
    }
    // ---- (3) the list is consumed (by the probe kernel, in front of this one): empty it for the next call
    if (r == 0 && tid == 0) *list_n = 0;
}

__global__ void blocks_update_kernel(const u32* ids, u32 n, u32 size, const u32* session, const u32* depth,
                                     const u32* last_access, const u32* ref_flags, u32* m_session, u32* m_depth,
                                     u32* m_last, u32* m_ref, u32* status) {
    u32 i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const u32 b = ids[i];
    if (b >= size) {
        atomicOr(status, CWS_INVAL);
        return;
    }
    if (session) m_session[b] = session[i];
    if (depth) m_depth[b] = depth[i];
    if (last_access) m_last[b] = last_access[i];
    if (ref_flags) m_ref[b] = ref_flags[i];
}

inline u32 cdiv(u64 a, u32 b) { return (u32)((a + b - 1) / b); }

}  // namespace

int32_t cwi_table_lookup(cw_ctx* ctx, const u64* d_keys, u32 n, u32* d_loc) {
    if (!n) return CW_OK;
    lookup_kernel<<<cdiv(n, 256), 256, 0, ctx->s_main>>>(ctx->table, ctx->n_slots - 1, d_keys, n, d_loc);
    CW_LAUNCH_CHECK(ctx);
    return CW_OK;
}
static bool stream_capturing(cudaStream_t s) {
    cudaStreamCaptureStatus st = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(s, &st) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return st != cudaStreamCaptureStatusNone;
}

int32_t cwi_table_compact(cw_ctx* ctx) {
    const size_t bytes = ctx->n_slots * sizeof(cw_slot);
    if (!ctx->table2) CW_CUDA(ctx, cudaMalloc(reinterpret_cast<void**>(&ctx->table2), bytes));
    cudaStream_t s = ctx->s_main;
    CW_CUDA(ctx, cudaMemsetAsync(ctx->table2, 0, bytes, s));
    CW_CUDA(ctx, cudaMemset2DAsync(reinterpret_cast<uint8_t*>(ctx->table2) + 12, sizeof(cw_slot), 0xFF, 4, ctx->n_slots, s));
    const u32 grid = (u32)std::min<u64>((ctx->n_slots + 255) / 256, (u64)ctx->n_sm * 16);
    rebuild_kernel<<<grid, 256, 0, s>>>(ctx->table, ctx->table2, ctx->n_slots);
    CW_LAUNCH_CHECK(ctx);
    // copied back: the table address is baked into captured graphs and must not change
    CW_CUDA(ctx, cudaMemcpyAsync(ctx->table, ctx->table2, bytes, cudaMemcpyDeviceToDevice, s));
    CW_CUDA(ctx, cudaMemsetAsync(ctx->tbl_cnt + 1, 0, sizeof(u32), s));
    ctx->tomb_ub = 0;
    ctx->compactions++;
    return CW_OK;
}

int32_t cwi_table_stats(cw_ctx* ctx, u64* h_out8) {
    cudaStream_t s = ctx->s_main;
    CW_CUDA(ctx, cudaMemsetAsync(ctx->tbl_cnt, 0, 4 * sizeof(u32), s));
    CW_CUDA(ctx, cudaMemsetAsync(ctx->tbl_hist, 0, CWT_HIST_BINS * sizeof(u32), s));
    const u32 grid = (u32)std::min<u64>((ctx->n_slots + 255) / 256, (u64)ctx->n_sm * 16);
    stats_kernel<<<grid, 256, 0, s>>>(ctx->table, ctx->n_slots, ctx->tbl_cnt, ctx->tbl_hist);
    CW_LAUNCH_CHECK(ctx);
    u32 cnt[4];
    static thread_local u32 hist[CWT_HIST_BINS];
    CW_CUDA(ctx, cudaMemcpyAsync(cnt, ctx->tbl_cnt, sizeof(cnt), cudaMemcpyDeviceToHost, s));
    CW_CUDA(ctx, cudaMemcpyAsync(hist, ctx->tbl_hist, sizeof(hist), cudaMemcpyDeviceToHost, s));
    CW_CUDA(ctx, cudaStreamSynchronize(s));
    ctx->live_ub = cnt[0];  // exact again
    u64 sum = 0, p50 = 0, p99 = 0, acc = 0;
    for (u32 b = 0; b < CWT_HIST_BINS; ++b) sum += (u64)hist[b] * (b + 1);  // the last bin counts its lower edge
    for (u32 b = 0; b < CWT_HIST_BINS; ++b) {
        acc += hist[b];
        if (!p50 && cnt[0] && acc * 2 >= cnt[0]) p50 = b + 1;
        if (!p99 && cnt[0] && acc * 100 >= (u64)cnt[0] * 99) p99 = b + 1;
    }
    h_out8[0] = cnt[0];
    h_out8[1] = cnt[1];
    h_out8[2] = ctx->n_slots;
    h_out8[3] = cnt[2];
    h_out8[4] = p50;
    h_out8[5] = p99;
    h_out8[6] = ctx->compactions;
    h_out8[7] = sum;
    return CW_OK;
}

int32_t cwi_table_erase(cw_ctx* ctx, const u64* d_keys, u32 n) {
    if (!n) return CW_OK;
    erase_kernel<<<cdiv(n, 256), 256, 0, ctx->s_main>>>(ctx->table, ctx->n_slots - 1, d_keys, n, ctx->tbl_cnt);
    CW_LAUNCH_CHECK(ctx);
    // tombstones are bounded from the host (no read-back): once the erases since the last compaction could have
    // turned a quarter of the slots into tombstones, rebuild (never inside a graph capture: the launch sequence of
    // a captured call must not depend on the table's history)
    ctx->tomb_ub += n;
    if (ctx->tomb_ub > ctx->n_slots / 4 && !stream_capturing(ctx->s_main)) return cwi_table_compact(ctx);
    return CW_OK;
}
int32_t cwi_table_retag(cw_ctx* ctx, const u64* d_keys, const u32* d_new_loc, u32 n) {
    if (!n) return CW_OK;
    retag_kernel<<<cdiv(n, 256), 256, 0, ctx->s_main>>>(ctx->table, ctx->n_slots - 1, d_keys, d_new_loc, n);
    CW_LAUNCH_CHECK(ctx);
    return CW_OK;
}
int32_t cwi_table_insert(cw_ctx* ctx, const u64* d_keys, const u32* d_loc, u32 n, u32* d_winner_loc) {
    if (!n) return CW_OK;
    const u64 mask = ctx->n_slots - 1;
    if (ctx->live_ub + n > ctx->n_slots) {
        // the batch might fill the table: replace the host bound by the exact device count (one sync, misuse path)
        if (stream_capturing(ctx->s_main)) {
            snprintf(ctx->err, sizeof(ctx->err), "cw_table_insert near a full table cannot be captured");
            return CW_E_STATE;
        }
        u32 live = 0;
        CW_CUDA(ctx, cudaMemcpyAsync(&live, ctx->tbl_cnt, sizeof(u32), cudaMemcpyDeviceToHost, ctx->s_main));
        CW_CUDA(ctx, cudaStreamSynchronize(ctx->s_main));
        ctx->live_ub = live;
    }
    if (ctx->live_ub + n > ctx->n_slots) {  // first come by input index, like the oracle
        insert_seq_kernel<<<1, 32, 0, ctx->s_main>>>(ctx->table, mask, d_keys, d_loc, n, d_winner_loc, ctx->d_status,
                                                     ctx->tbl_cnt);
        CW_LAUNCH_CHECK(ctx);
        ctx->live_ub = ctx->n_slots;
        return CW_OK;
    }
    ctx->live_ub += n;
    if (n > ctx->ins_cap) {  // grow the per-batch scratch (outside of graph capture)
        if (ctx->ins_slot) CW_CUDA(ctx, cudaFree(ctx->ins_slot));
        ctx->ins_slot = nullptr;
        ctx->ins_cap = 0;
        CW_CUDA(ctx, cudaMalloc(&ctx->ins_slot, (size_t)n * sizeof(u32)));
        ctx->ins_cap = n;
    }
    insert_claim_kernel<<<cdiv(n, 256), 256, 0, ctx->s_main>>>(ctx->table, mask, d_keys, n, ctx->ins_slot,
                                                               ctx->d_status, ctx->tbl_cnt);
    CW_LAUNCH_CHECK(ctx);
    insert_resolve_kernel<<<cdiv(n, 256), 256, 0, ctx->s_main>>>(ctx->table, d_loc, n, ctx->ins_slot, d_winner_loc);
    CW_LAUNCH_CHECK(ctx);
    insert_reset_kernel<<<cdiv(n, 256), 256, 0, ctx->s_main>>>(ctx->table, n, ctx->ins_slot);
    CW_LAUNCH_CHECK(ctx);
    return CW_OK;
}

int32_t cwi_match_prefix(cw_ctx* ctx, const u64* d_hashes, const u64* d_hash_off, u32 R, u32* d_k_total,
                         u32* d_n_gpu, u32* d_hit_loc) {
    if (!R) return CW_OK;
    const u64 mask = ctx->n_slots - 1;
    // enough warps to cover max_hashed_blocks once, capped at a few waves; the kernel grid-strides
    u64 warps = (ctx->cfg.max_hashed_blocks + CWM_CHUNK - 1) / CWM_CHUNK;
    u64 blocks = (warps + MATCH_THREADS / 32 - 1) / (MATCH_THREADS / 32);
    u64 cap = (u64)ctx->n_sm * MATCH_MIN_CTAS * 4;
    if (blocks > cap) blocks = cap;
    if (blocks < 1) blocks = 1;
    match_probe_kernel<<<(u32)blocks, MATCH_THREADS, 0, ctx->s_main>>>(ctx->table, (u32)mask, d_hashes, d_hash_off, R,
                                                             ctx->m_first_miss, ctx->m_max_hit, ctx->m_host_hits,
                                                             d_hit_loc, ctx->d_status, nullptr, nullptr);
    CW_LAUNCH_CHECK(ctx);
    match_finish_kernel<<<cdiv((u64)R * 32, 256), 256, 0, ctx->s_main>>>(d_hash_off, R, ctx->m_first_miss,
                                                                         ctx->m_max_hit, ctx->m_host_hits, d_k_total,
                                                                         d_n_gpu, d_hit_loc, ctx->table, mask,
                                                                         d_hashes);
    CW_LAUNCH_CHECK(ctx);
    return CW_OK;
}

int32_t cwi_match_prefix_shared(cw_ctx* ctx, const u64* d_hashes, const u64* d_hash_off, u32 R, const u32* d_leader,
                                u32* d_k_total, u32* d_n_gpu, u32* d_hit_loc) {
    if (!R) return CW_OK;
    const u64 mask = ctx->n_slots - 1;
    const u32 mr = ctx->cfg.max_requests;
    u32 *first_miss = ctx->m_shared, *max_hit = ctx->m_shared + mr, *host_hits = ctx->m_shared + 2 * (size_t)mr;
    u32 *lcp = ctx->m_shared + 3 * (size_t)mr, *list_n = ctx->m_shared + 4 * (size_t)mr;
    uint2* list = reinterpret_cast<uint2*>(ctx->m_list);
    match_lcp_kernel<<<cdiv((u64)R * 32, 256), 256, 0, ctx->s_main>>>(d_hashes, d_hash_off, R, d_leader, lcp, list, list_n,
                                                                      first_miss, max_hit, host_hits);
    CW_LAUNCH_CHECK(ctx);
    // one resident wave: the list is short (the leaders' tasks and one tail task per follower) and its length is
    // known to the device only
    u64 warps = (ctx->cfg.max_hashed_blocks + CWM_CHUNK - 1) / CWM_CHUNK;
    u64 blocks = (warps + MATCH_THREADS / 32 - 1) / (MATCH_THREADS / 32);
    u64 cap = (u64)ctx->n_sm * MATCH_MIN_CTAS;
    if (blocks > cap) blocks = cap;
    if (blocks < 1) blocks = 1;
    match_probe_kernel<<<(u32)blocks, MATCH_THREADS, 0, ctx->s_main>>>(ctx->table, (u32)mask, d_hashes, d_hash_off, R,
                                                                       first_miss, max_hit, host_hits, d_hit_loc,
                                                                       ctx->d_status, list, list_n);
    CW_LAUNCH_CHECK(ctx);
    match_share_kernel<<<R, SHARE_THREADS, 0, ctx->s_main>>>(d_hash_off, R, d_leader, lcp, first_miss, max_hit, host_hits,
                                                             d_k_total, d_n_gpu, d_hit_loc, ctx->table, mask, d_hashes,
                                                             list_n);
    CW_LAUNCH_CHECK(ctx);
    return CW_OK;
}

int32_t cwi_blocks_update(cw_ctx* ctx, u32 tier, const u32* d_ids, u32 n, const u32* d_session, const u32* d_depth,
                          const u32* d_last_access, const u32* d_ref_flags) {
    if (!n) return CW_OK;
    blocks_update_kernel<<<cdiv(n, 256), 256, 0, ctx->s_main>>>(
        d_ids, n, ctx->tier_size[tier], d_session, d_depth, d_last_access, d_ref_flags, ctx->meta_session[tier],
        ctx->meta_depth[tier], ctx->meta_last_access[tier], ctx->meta_ref_flags[tier], ctx->d_status);
    CW_LAUNCH_CHECK(ctx);
    return CW_OK;
}
