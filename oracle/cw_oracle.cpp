// ORACLE — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, single-threaded C++17 restatement of what CacheWise's per-step block-management
// pass computes (hash -> match -> schedule -> score/select -> swap), written from PAPER.md and the
// readings listed in DESIGN.md ("Readings of the paper").  It shares no code, header, table or
// constant generator with paper_2606_16824_b200/csrc (the CUDA path); only tests/, bench.py's
// cpu_baseline / --impl reference legs and __graft_entry__.smoke() may load it.
//
// Parity pins (tests/test_oracle_*.py, all `-m "not gpu"`): every function below is pinned to
// something other than itself — closed forms, brute force on tiny inputs, textbook special cases
// (LRU, Belady, FCFS), invariants.  Nothing here is "parity unpinned"; note however that PAPER.md
// prints no worked numeric example for any stage, so no pin is a value printed by the paper.
//
// Every function takes HOST pointers.  Status codes mirror the paper-facing boundary:
//   0 ok, -1 invalid argument, -2 capacity (table full / fewer evictable blocks than the deficit).

#include <algorithm>
#include <cstdint>
#include <cstring>
#include <tuple>
#include <unordered_map>
#include <vector>

typedef uint64_t u64;
typedef uint32_t u32;
typedef int32_t i32;

// ------------------------------------------------------------------------------------------------
// Stage 1 — chained prefix hashing.  PAPER.md never describes the hash (L60 "persist KVCache from
// previous requests", L235 vLLM base); reading R1 fixes it:
//   fin(x): x^=x>>32; x*=K2; x^=x>>29; x*=K3; x^=x>>32                       (mod 2^64)
//   keys  : x=fin(K11*(m+1)); ka_m=(x>>32)|2^31; kb_m=(x&0xffffffff)|2^31      m=0..7
//   digest: s=sum_m u64(u32(t[2m]+ka_m))*u64(u32(t[2m+1]+kb_m)); c=fin(s^K5)
//   chain : H_{-1}=fin(salt^K7); H_j=A*H_{j-1}+c_j
// ------------------------------------------------------------------------------------------------
static const u64 CW_A = 0x9E3779B97F4A7C15ull;    // floor(2^64*(sqrt5-1)/2)
static const u64 CW_K2 = 0x6A09E667F3BCC909ull;   // floor(2^64*frac(sqrt 2))|1
static const u64 CW_K3 = 0xBB67AE8584CAA73Bull;   // floor(2^64*frac(sqrt 3))|1
static const u64 CW_K5 = 0x3C6EF372FE94F82Bull;   // floor(2^64*frac(sqrt 5))|1
static const u64 CW_K7 = 0xA54FF53A5F1D36F1ull;   // floor(2^64*frac(sqrt 7))|1
static const u64 CW_K11 = 0x510E527FADE682D1ull;  // floor(2^64*frac(sqrt 11))|1

static u64 fin(u64 x) {
    x ^= x >> 32;
    x *= CW_K2;
    x ^= x >> 29;
    x *= CW_K3;
    x ^= x >> 32;
    return x;
}

static u64 block_digest(const i32* tok) {
    u64 s = 0;
    for (int m = 0; m < 8; ++m) {
        u64 x = fin(CW_K11 * (u64)(m + 1));
        u32 ka = (u32)(x >> 32) | 0x80000000u;
        u32 kb = (u32)(x & 0xffffffffull) | 0x80000000u;
        u32 a = (u32)tok[2 * m] + ka;
        u32 b = (u32)tok[2 * m + 1] + kb;
        s += (u64)a * (u64)b;
    }
    return fin(s ^ CW_K5);
}

extern "C" {

u64 cwo_fin(u64 x) { return fin(x); }
u64 cwo_block_digest(const i32* tok16) { return block_digest(tok16); }

// Hash every full 16-token block j >= start_block[r] of request r (R1).
// tokens: int32[sum T] CSR by tok_off[R+1]; hashes: u64[sum N] CSR by hash_off[R+1], in-out:
// entries below start_block are left untouched.  The chain resumes from start_state[r] (= the hash
// of block start_block-1) when start_block[r] > 0, else from fin(salt ^ K7).
int cwo_hash_blocks(const i32* tokens, const u64* tok_off, const u32* start_block, const u64* start_state,
                    const u64* salt, const u64* hash_off, u32 R, u64* hashes) {
    if (!tokens || !tok_off || !hash_off || !hashes) return -1;
    for (u32 r = 0; r < R; ++r) {
        u64 len = tok_off[r + 1] - tok_off[r];
        u64 n = len / 16;
        if (hash_off[r + 1] - hash_off[r] != n) return -1;
        u32 sb = start_block ? start_block[r] : 0;
        if (sb > n) return -1;
        if (sb > 0 && !start_state) return -1;
        u64 h = sb > 0 ? start_state[r] : fin((salt ? salt[r] : 0) ^ CW_K7);
        for (u64 j = sb; j < n; ++j) {
            h = CW_A * h + block_digest(tokens + tok_off[r] + 16 * j);
            hashes[hash_off[r] + j] = h;
        }
    }
    return 0;
}

// ------------------------------------------------------------------------------------------------
// Stage 2a — resident-block table (exact map) and prefix match.  PAPER.md L177 (k_i(t) blocks
// "already reside in memory (the reusable prefix overlap)"), L173 ("contiguous ... prefix"), Fig.
// 11B L223 ("overlap with KVCache resident on the XPU memory").  DESIGN.md reading R2.
// ------------------------------------------------------------------------------------------------
struct cwo_table {
    std::unordered_map<u64, u32> map;
    u64 capacity;
};

static u64 remap(u64 k) {  // keys 0 and 2^64-1 are reserved by the product's open-addressing table
    if (k == 0) return 1;
    if (k == ~0ull) return ~0ull - 1;
    return k;
}

cwo_table* cwo_table_create(u32 log2_slots) {
    cwo_table* t = new cwo_table();
    t->capacity = 1ull << log2_slots;
    return t;
}
void cwo_table_destroy(cwo_table* t) { delete t; }
u64 cwo_table_size(const cwo_table* t) { return t->map.size(); }

// Insert in input order: an already-present key keeps its loc, else the lowest input index wins.
int cwo_table_insert(cwo_table* t, const u64* keys, const u32* loc, u32 n, u32* winner_loc) {
    int status = 0;
    for (u32 i = 0; i < n; ++i) {
        u64 k = remap(keys[i]);
        auto it = t->map.find(k);
        if (it != t->map.end()) {
            if (winner_loc) winner_loc[i] = it->second;
        } else if (t->map.size() >= t->capacity) {
            status = -2;
            if (winner_loc) winner_loc[i] = 0xFFFFFFFFu;
        } else {
            t->map.emplace(k, loc[i]);
            if (winner_loc) winner_loc[i] = loc[i];
        }
    }
    return status;
}
int cwo_table_erase(cwo_table* t, const u64* keys, u32 n) {
    for (u32 i = 0; i < n; ++i) t->map.erase(remap(keys[i]));
    return 0;
}
int cwo_table_retag(cwo_table* t, const u64* keys, const u32* new_loc, u32 n) {
    for (u32 i = 0; i < n; ++i) {
        auto it = t->map.find(remap(keys[i]));
        if (it != t->map.end()) it->second = new_loc[i];
    }
    return 0;
}
int cwo_table_lookup(const cwo_table* t, const u64* keys, u32 n, u32* loc) {
    for (u32 i = 0; i < n; ++i) {
        auto it = t->map.find(remap(keys[i]));
        loc[i] = it == t->map.end() ? 0xFFFFFFFFu : it->second;
    }
    return 0;
}

// k_total[r] = length of the LEADING run of present hashes (either tier); n_gpu[r] = how many of those
// have an HBM location (bit 31 of loc clear) = the paper's k_i(t); hit_loc past the run is MISS.
int cwo_match_prefix(const cwo_table* t, const u64* hashes, const u64* hash_off, u32 R, u32* k_total,
                     u32* n_gpu, u32* hit_loc) {
    for (u32 r = 0; r < R; ++r) {
        u64 lo = hash_off[r], hi = hash_off[r + 1];
        u32 k = 0, g = 0;
        bool run = true;
        for (u64 j = lo; j < hi; ++j) {
            u32 loc = 0xFFFFFFFFu;
            if (run) {
                auto it = t->map.find(remap(hashes[j]));
                if (it == t->map.end()) {
                    run = false;
                } else {
                    loc = it->second;
                    ++k;
                    if (!(loc & 0x80000000u)) ++g;
                }
            }
            if (hit_loc) hit_loc[j] = loc;
        }
        k_total[r] = k;
        n_gpu[r] = g;
    }
    return 0;
}

// ------------------------------------------------------------------------------------------------
// Stage 2b — prefix-aware scheduling.  PAPER.md 5.1 L207 ("selects request r_i which requires fewest
// additional blocks a_i(t)"), L177 (a_i = d_i - k_i; admit if it fits, else evict), L281 (FCFS
// baseline).  DESIGN.md reading R3: three total orders + stop-at-first-misfit admission.
// ------------------------------------------------------------------------------------------------
int cwo_schedule(u32 R, const u32* need_d, const u32* n_gpu, const u64* arrival_seq, const u32* req_id,
                 u32 policy, u32 free_blocks, u32 evictable, u32 max_admit, u32* order, u32* num_admit,
                 u32* deficit) {
    if (policy > 2) return -1;
    typedef std::tuple<u64, u64, u64, u64, u32> key_t;  // last = input index (stable tie-break)
    std::vector<key_t> keys(R);
    std::vector<u64> a(R);
    for (u32 i = 0; i < R; ++i) {
        a[i] = need_d[i] > n_gpu[i] ? (u64)(need_d[i] - n_gpu[i]) : 0;
        u64 inv_overlap = 0xFFFFFFFFull - n_gpu[i];  // descending overlap
        if (policy == 0)
            keys[i] = key_t(a[i], inv_overlap, arrival_seq[i], req_id[i], i);
        else if (policy == 1)
            keys[i] = key_t(inv_overlap, a[i], arrival_seq[i], req_id[i], i);
        else
            keys[i] = key_t(arrival_seq[i], req_id[i], 0, 0, i);
    }
    std::stable_sort(keys.begin(), keys.end());
    u64 need = 0, budget = (u64)free_blocks + (u64)evictable;
    u32 count = 0;
    bool open = true;
    for (u32 p = 0; p < R; ++p) {
        u32 i = std::get<4>(keys[p]);
        order[p] = i;
        if (open) {
            if (count >= max_admit || need + a[i] > budget) {
                open = false;  // stop at the first request that does not fit: no back-filling
            } else {
                need += a[i];
                ++count;
            }
        }
    }
    *num_admit = count;
    *deficit = need > free_blocks ? (u32)(need - free_blocks) : 0;
    return 0;
}

// NEXT-3 — admission under a chunked-prefill token budget.  PAPER.md 6.1 L271: "All experiments run
// with chunked-prefill enabled and we use the default value of max. 512 tokens per chunk".  DESIGN.md reading R8: an
// engine iteration prefills at most `token_budget` new tokens.  Walk the dispatch order of cwo_schedule; request i
// (needing a_i = d_i - k_i more blocks and t_i new tokens) is admitted while count < max_admit, the blocks fit
// (need + a_i <= free + evictable, L177) and budget is left (used < token_budget); it gets the chunk
// min(t_i, token_budget - used).  Stop at the first request that does not fit (no back-filling).  chunk_tokens is in
// INPUT-index order, 0 for everybody who was not admitted; deficit = max(0, need - free_blocks) as in cwo_schedule.
int cwo_admit_chunked(u32 R, const u32* order, const u32* need_d, const u32* n_gpu, const u32* new_tokens,
                      u32 free_blocks, u32 evictable, u32 max_admit, u64 token_budget, u32* chunk_tokens,
                      u32* num_admit, u32* deficit) {
    for (u32 i = 0; i < R; ++i) chunk_tokens[i] = 0;
    u64 need = 0, used = 0, budget = (u64)free_blocks + (u64)evictable;
    u32 count = 0;
    for (u32 p = 0; p < R; ++p) {
        u32 i = order[p];
        if (i >= R) return -1;
        u64 a = need_d[i] > n_gpu[i] ? (u64)(need_d[i] - n_gpu[i]) : 0;
        if (count >= max_admit || need + a > budget || used >= token_budget) break;
        u64 chunk = std::min<u64>(new_tokens[i], token_budget - used);
        chunk_tokens[i] = (u32)chunk;
        used += chunk;
        need += a;
        ++count;
    }
    *num_admit = count;
    *deficit = need > free_blocks ? (u32)std::min<u64>(need - free_blocks, 0xFFFFFFFFull) : 0;
    return 0;
}

// ------------------------------------------------------------------------------------------------
// Stage 3 — reuse-aware eviction.  PAPER.md 5.2 L215-219 (evict in decreasing tau; Belady with true
// tau), L181 (j* = argmax_{j != i} tau_j), L252 (unreferenced blocks only; one prediction per
// session), L277 (idle sessions first), L281 (LRU fallback).  DESIGN.md reading R4:
//   raw = bias + sum_f w[f]*x[s][f];  TOOL_WAIT(0): tau = clamp(raw,0,TAU_MAX-1) (or override);
//   QUEUED(1)/RUNNING(2): tau = 0;  IDLE(>=3) or unknown session: tau = TAU_MAX = 2^24-1
//   evictable <=> VALID(bit31) && !PINNED(bit30) && refcount(bits 0..29)==0
//   score = (TAU_MAX - tau)<<40 | (0xFFFFF - min(age,0xFFFFF))<<20 | (0xFFFFF - min(depth,0xFFFFF))
//   victims = the min(deficit, #evictable) smallest by (score, block id), sorted ascending.
// ------------------------------------------------------------------------------------------------
static const u32 TAU_MAX = (1u << 24) - 1;

int cwo_session_tau(u32 S, u32 F, const uint8_t* features, const int16_t* weights, i32 bias,
                    const uint8_t* session_state, const u32* tau_override, u32* tau_q) {
    if (bias > (1 << 30) || bias < -(1 << 30) || F > 16) return -1;
    for (u32 s = 0; s < S; ++s) {
        u32 st = session_state[s];
        u32 tau;
        if (st == 1 || st == 2) {
            tau = 0;
        } else if (st >= 3) {
            tau = TAU_MAX;
        } else if (tau_override) {
            tau = std::min(tau_override[s], TAU_MAX - 1);
        } else {
            int64_t raw = bias;
            for (u32 f = 0; f < F; ++f) raw += (int64_t)weights[f] * (int64_t)features[(u64)s * F + f];
            tau = (u32)std::min<int64_t>(std::max<int64_t>(raw, 0), TAU_MAX - 1);
        }
        tau_q[s] = tau;
    }
    return 0;
}

u64 cwo_block_score(u32 tau, u32 tick_now, u32 last_access, u32 depth) {
    u64 age = tick_now >= last_access ? tick_now - last_access : 0;
    if (age > 0xFFFFF) age = 0xFFFFF;
    u64 dp = depth > 0xFFFFF ? 0xFFFFF : depth;
    return ((u64)(TAU_MAX - tau) << 40) | ((0xFFFFFull - age) << 20) | (0xFFFFFull - dp);
}

int cwo_score_evict(u32 tick_now, u32 S, u32 F, const uint8_t* features, const int16_t* weights, i32 bias,
                    const uint8_t* session_state, const u32* tau_override, u32 deficit, u32 M,
                    const u32* blk_session, const u32* blk_last_access, const u32* blk_depth,
                    const u32* blk_ref_flags, u32* victims, u64* victim_scores, u32* num_victims, u32 cap) {
    std::vector<u32> tau(S);
    int st = cwo_session_tau(S, F, features, weights, bias, session_state, tau_override, tau.data());
    if (st) return st;
    std::vector<std::pair<u64, u32>> all;
    for (u32 b = 0; b < M; ++b) {
        u32 rf = blk_ref_flags[b];
        bool evictable = (rf & 0x80000000u) && !(rf & 0x40000000u) && (rf & 0x3FFFFFFFu) == 0;
        if (!evictable) continue;
        u32 t = blk_session[b] < S ? tau[blk_session[b]] : TAU_MAX;
        all.emplace_back(cwo_block_score(t, tick_now, blk_last_access[b], blk_depth[b]), b);
    }
    std::sort(all.begin(), all.end());  // full sort by (score, id): exhaustive, no selection shortcut
    u32 want = std::min(deficit, cap);
    u32 n = (u32)std::min<u64>(want, all.size());
    for (u32 i = 0; i < n; ++i) {
        victims[i] = all[i].second;
        if (victim_scores) victim_scores[i] = all[i].first;
    }
    *num_victims = n;
    return n < want ? -2 : 0;
}

// ------------------------------------------------------------------------------------------------
// Stage 4 — paged KV swap.  PAPER.md 6.4 L345 ("transferred from GPU memory to CPU DRAM and swapped
// back on demand").  DESIGN.md reading R5: chunk c of block b lives at pool + b*block_stride +
// c*chunk_stride; a staged page is chunks 0..n_chunks-1 contiguous; victim j -> slot j (or slots[j]).
// ------------------------------------------------------------------------------------------------
int cwo_swap_out(const uint8_t* pool, u32 n_chunks, u64 chunk_bytes, u64 chunk_stride, u64 block_stride,
                 const u32* victims, u32 n, const u32* slots, uint8_t* dst) {
    u64 page = (u64)n_chunks * chunk_bytes;
    for (u32 j = 0; j < n; ++j) {
        uint8_t* out = dst + (u64)(slots ? slots[j] : j) * page;
        for (u32 c = 0; c < n_chunks; ++c)
            std::memcpy(out + c * chunk_bytes, pool + victims[j] * block_stride + c * chunk_stride, chunk_bytes);
    }
    return 0;
}
int cwo_swap_in(uint8_t* pool, u32 n_chunks, u64 chunk_bytes, u64 chunk_stride, u64 block_stride,
                const u32* slots, const uint8_t* src, const u32* dst_blocks, u32 n) {
    u64 page = (u64)n_chunks * chunk_bytes;
    for (u32 j = 0; j < n; ++j) {
        const uint8_t* in = src + (u64)(slots ? slots[j] : j) * page;
        for (u32 c = 0; c < n_chunks; ++c)
            std::memcpy(pool + dst_blocks[j] * block_stride + c * chunk_stride, in + c * chunk_bytes, chunk_bytes);
    }
    return 0;
}

// ------------------------------------------------------------------------------------------------
// NEXT-1 — the paper's own predictor.  PAPER.md 5.2 L219-225: "at time t, CacheWise estimates
// the expected remaining time for the tool call to complete, i.e. E[tau_i(t) | tau_i(t) - T_i > t - T_i], by
// analyzing distributions of tool execution durations with similar metadata m"; L227: per-cluster empirical
// distributions.  DESIGN.md reading R7: with the historical durations d_0..d_{n-1} (ms) of the session's
// cluster and the elapsed time e = t - T_i,
//     tau = clamp( floor( sum_{d_k > e} d_k / #{d_k > e} ) - e , 0, TAU_MAX-1 )
// and, when no historical call of the cluster ran longer than e (or the cluster is empty), tau = min(e,
// TAU_MAX-1) (the call has outlived all history: expect it to take as long again).  cluster >= C -> tau = 0, status -1.
// ------------------------------------------------------------------------------------------------
int cwo_predict_tau(u32 S, const u32* cluster, const u32* elapsed_ms, u32 C, const u64* sample_off,
                    const u32* samples, u32* tau_out) {
    int status = 0;
    for (u32 s = 0; s < S; ++s) {
        u32 c = cluster[s];
        if (c >= C) {
            tau_out[s] = 0;
            status = -1;
            continue;
        }
        u64 e = elapsed_ms[s], sum = 0, cnt = 0;
        for (u64 k = sample_off[c]; k < sample_off[c + 1]; ++k)
            if (samples[k] > e) {
                sum += samples[k];
                ++cnt;
            }
        u64 tau = cnt ? sum / cnt - e : e;
        tau_out[s] = (u32)std::min<u64>(tau, TAU_MAX - 1);
    }
    return status;
}

}  // extern "C"
