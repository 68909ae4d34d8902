// NEXT-1 — the paper's own predictor on the device (cw_predict_tau).  DESIGN.md R7.
//
// PAPER.md 5.2 L219-225: the expected REMAINING time of the session's tool call given that it is still running
// e = t - T_i after it was issued, from the empirical distribution of the durations of historical calls with
// similar metadata (per-cluster distributions, L227).  One warp per session: a binary search finds the first
// historical duration above e in the cluster's sorted samples, the lanes sum the tail with coalesced loads,
//     tau = clamp( floor( sum_{d > e} d / #{d > e} ) - e, 0, TAU_MAX-1 ),    none above e  ->  tau = min(e, TAU_MAX-1).
// The output feeds cw_score_evict's d_tau_override, so one launch per scheduling step refreshes every session —
// the paper re-evaluates the predictor only every N_rebuild iterations because it costs CPU time (L254).
#include <stdio.h>

#include "cw_internal.cuh"

namespace {

__global__ void __launch_bounds__(256) predict_kernel(u32 S, const u32* __restrict__ cluster,
                                                      const u32* __restrict__ elapsed, u32 C,
                                                      const u64* __restrict__ sample_off,
                                                      const u32* __restrict__ samples, u32* tau_out, u32* status) {
    const u32 lane = threadIdx.x & 31;
    const u32 s = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (s >= S) return;
    const u32 c = cluster[s];
    if (c >= C) {
        if (lane == 0) {
            tau_out[s] = 0;
            atomicOr(status, CWS_INVAL);
        }
        return;
    }
    const u64 e = elapsed[s];
    const u64 lo0 = sample_off[c], hi0 = sample_off[c + 1];
    u64 lo = lo0, hi = hi0;  // first index with samples[idx] > e (samples ascending inside a cluster)
    while (lo < hi) {
        const u64 mid = (lo + hi) >> 1;
        if ((u64)samples[mid] > e) hi = mid;
        else lo = mid + 1;
    }
    u64 sum = 0;
    for (u64 k = lo + lane; k < hi0; k += 32) sum += samples[k];
#pragma unroll
    for (int m = 16; m; m >>= 1) sum += shfl64_xor(sum, m);
    if (lane == 0) {
        const u64 cnt = hi0 - lo;
        const u64 tau = cnt ? sum / cnt - e : e;
        tau_out[s] = (u32)min(tau, (u64)(CW_TAU_MAX - 1));
    }
}

}  // namespace

int32_t cwi_predict_tau(cw_ctx* ctx, u32 S, const u32* d_cluster, const u32* d_elapsed, u32 C, const u64* d_sample_off,
                        const u32* d_samples, u32* d_tau_out) {
    if (!S) return CW_OK;
    predict_kernel<<<(u32)(((u64)S * 32 + 255) / 256), 256, 0, ctx->s_main>>>(S, d_cluster, d_elapsed, C, d_sample_off,
                                                                           d_samples, d_tau_out, ctx->d_status);
    CW_LAUNCH_CHECK(ctx);
    return CW_OK;
}
