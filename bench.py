#!/usr/bin/env python
"""bench.py — the block-management pass of CacheWise (arxiv/paper_2606_16824) on B200, measured.

A "step" is one pass of the whole hot path (hash -> match -> schedule -> score/select -> swap-out
-> swap-in) over BASELINE.json configs[2] (4096 queued requests, 256 sessions, 2^20-block resident table at load
0.5, 20% pinned, eviction budget 5% of the pool, 16-feature predictor).  DESIGN.md "Measurement" defines every
number printed here.

  python bench.py [--gpus N] [--steps K] [--warmup W]      the CUDA path (libcachewise.so), ONE JSON line
  python bench.py --impl reference ...                      the CPU oracle on a bounded sample of the same workload

N > 1 (launched by torch.distributed.run): independent replicas, one per GPU, no data-path collective
 — value = all ranks' blocks / the slowest rank's device time.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "kv_mgmt_step_blocks_per_s"
UNIT = "blocks/s"
WORKLOAD = ("BASELINE.json configs[2]: 4096 queued requests, 256 sessions x 131072-token streams, 2^20 resident "
            "blocks in a 2^21-slot table, 20% ref-pinned, eviction budget 5% of the pool, F=16")
PCIE_GEN5_X16_GBS = 63.0  # 32 GT/s x 16 lanes x 128/130 / 8 per direction

# dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full` captures
# (profiles/r1_full_step_kernels.md), full-size configs[2] step.
NCU_TRAFFIC_BYTES = {"hash": 434_067_199, "match": 94_296_064, "score_evict": 17_158_912, "gather": 1_660_988_672,
                     "scatter": 1_659_497_727, "schedule": 126_976}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


# ------------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """Samples SM clock + throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period_s: float = 0.01):
        self.index, self.period, self.samples, self._stop = index, period_s, [], threading.Event()
        self._thread, self.ok, self.sm_max = None, False, None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.sm_max = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                mhz = int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    reasons = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    reasons = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                self.samples.append((time.perf_counter(), mhz, reasons))
            except Exception:
                pass
            time.sleep(self.period)

    def start(self):
        if self.ok:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()

    def stop(self, t0=None, t1=None):
        self._stop.set()
        if self._thread:
            self._thread.join()
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": ["unavailable"]}
        sel = [s for s in self.samples if t0 is None or (t0 <= s[0] <= t1)] or self.samples
        names = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
                 0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
                 0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}
        bits = 0
        for _, _, r in sel:
            bits |= r
        reasons = [n for b, n in names.items() if bits & b and n != "gpu_idle"]
        return {"sm_mhz": int(statistics.median(s[1] for s in sel)), "sm_max_mhz": self.sm_max, "reasons": reasons,
                "samples": len(sel)}


# ------------------------------------------------------------------------------------------------ CUDA arm
def make_snapshot(seed: int, scale: int):
    from harness import gen
    if scale <= 1:
        return gen.stress_snapshot(seed=seed)
    # debugging aid only (--scale): the same recipe with fewer sessions; NOT a benchmark configuration
    return gen.stress_snapshot(seed=seed, S=max(256 // scale, 2))


def time_region(torch, stream, fns, steps):
    """Runs `steps` x all fns on `stream` with a CUDA event before/after every fn.  Returns (total_ms,
    per-fn list of mean ms)."""
    n = len(fns)
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(n + 1)] for _ in range(steps)]
    for k in range(steps):
        ev[k][0].record(stream)
        for i, f in enumerate(fns):
            f()
            ev[k][i + 1].record(stream)
    stream.synchronize()
    total = ev[0][0].elapsed_time(ev[-1][n])
    per = [statistics.fmean(ev[k][i].elapsed_time(ev[k][i + 1]) for k in range(steps)) for i in range(n)]
    return total, per


def graph_latency(torch, stream, fn, reps=100, warm=10, flush=None):
    """Median / p99 device time (us) of ONE CUDA-graph launch of fn's kernels; `flush` (optional) runs between
    launches, outside the timed events."""
    g = torch.cuda.CUDAGraph()
    fn()
    stream.synchronize()
    with torch.cuda.graph(g, stream=stream):
        fn()
    ts = []
    with torch.cuda.stream(stream):
        for i in range(warm + reps):
            if flush is not None:
                flush()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            g.replay()
            e1.record(stream)
            stream.synchronize()
            if i >= warm:
                ts.append(e0.elapsed_time(e1) * 1e3)
    ts.sort()
    return {"median_us": round(ts[len(ts) // 2], 2), "p99_us": round(ts[min(len(ts) - 1, int(len(ts) * 0.99))], 2),
            "min_us": round(ts[0], 2)}


def pcie_peak(torch, stream, gib=1, reps=5):
    n = gib << 30
    h = torch.empty(n, dtype=torch.uint8).pin_memory()
    d = torch.empty(n, dtype=torch.uint8, device="cuda")
    out = {}
    with torch.cuda.stream(stream):
        for name, (dst, src) in {"h2d": (d, h), "d2h": (h, d)}.items():
            best = 1e30
            for _ in range(reps + 1):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                dst.copy_(src, non_blocking=True)
                e1.record(stream)
                stream.synchronize()
                best = min(best, e0.elapsed_time(e1))
            out[name + "_gbs"] = round(n / best / 1e6, 2)
    del h, d
    return out


def swap_sweep(torch, cw, gen, stream, hbm_peak, pcie, ns):
    """BASELINE.json configs[3]: Llama-3-70B-shaped pages (160 chunks x 32 KiB = 5 MiB) scattered over a 60 GiB
    layer-major pool; n victims gathered to pinned host and restored; both directions and both kernels timed."""
    n_chunks, chunk_bytes, M = 160, 32768, 12288
    page = n_chunks * chunk_bytes
    rows = []
    with torch.cuda.stream(stream):
        pool = torch.empty(M * page, dtype=torch.uint8, device="cuda")
        ctx = cw.Context(num_blocks=M, table_log2_slots=15, max_requests=1, max_hashed_blocks=1, n_chunks=n_chunks,
                         chunk_bytes=chunk_bytes, chunk_stride=M * chunk_bytes, block_stride=chunk_bytes, pool=pool,
                         staging_bytes=2 * (320 << 20), stream_main=stream)
        nmax = max(ns)
        h = torch.empty(nmax * page, dtype=torch.uint8).pin_memory()
        staged = torch.empty(nmax * page, dtype=torch.uint8, device="cuda")

        def timed(fn, reps):
            ts = []
            for i in range(reps + 1):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                fn()
                e1.record(stream)
                ctx.sync()
                if i:
                    ts.append(e0.elapsed_time(e1))
            return statistics.median(ts)

        for n in ns:
            vic = torch.from_numpy(gen.swap_victims(4, M, n).astype(np.int32)).cuda()
            reps = 20 if n <= 64 else (8 if n <= 512 else 3)
            nbytes = n * page
            # cw_swap_out's last D2H runs on stream_copy: make stream_main wait for it through an empty swap-in join
            t_g = timed(lambda: ctx.gather_pages(vic, None, n, staged), reps)
            t_s = timed(lambda: ctx.scatter_pages(vic, None, n, staged), reps)

            def out_fn():
                ctx.swap_out(vic, None, n, None, h)
                ctx.join_copy()

            t_o = timed(out_fn, reps)
            t_i = timed(lambda: ctx.swap_in(None, h, vic, n), reps)
            rows.append({
                "n_blocks": n, "mib": round(nbytes / 2**20, 1),
                "gather_us": round(t_g * 1e3, 1), "gather_gbs": round(2 * nbytes / t_g / 1e6, 1),
                "gather_frac_hbm": round(2 * nbytes / t_g / 1e6 / hbm_peak, 3),
                "scatter_us": round(t_s * 1e3, 1), "scatter_gbs": round(2 * nbytes / t_s / 1e6, 1),
                "scatter_frac_hbm": round(2 * nbytes / t_s / 1e6 / hbm_peak, 3),
                "swap_out_us": round(t_o * 1e3, 1), "swap_out_gbs": round(nbytes / t_o / 1e6, 2),
                "swap_out_frac_pcie_measured": round(nbytes / t_o / 1e6 / pcie["d2h_gbs"], 3),
                "swap_out_frac_pcie_gen5x16": round(nbytes / t_o / 1e6 / PCIE_GEN5_X16_GBS, 3),
                "swap_in_us": round(t_i * 1e3, 1), "swap_in_gbs": round(nbytes / t_i / 1e6, 2),
                "swap_in_frac_pcie_measured": round(nbytes / t_i / 1e6 / pcie["h2d_gbs"], 3),
                "swap_in_frac_pcie_gen5x16": round(nbytes / t_i / 1e6 / PCIE_GEN5_X16_GBS, 3),
            })
        ctx.close()
        del pool, h, staged
    torch.cuda.empty_cache()
    return rows


def oracle_step(snap, table, pool, page, n_chunks, chunk_bytes, stage4=True):
    """One block-management step on the CPU oracle (as it stands).  Returns (seconds, blocks hashed)."""
    import oracle
    t0 = time.perf_counter()
    h, ho = oracle.hash_blocks(snap.tokens, snap.tok_off)
    k, g, loc = table.match_prefix(h, ho)
    order, na, de = oracle.schedule(snap.need_d, g, snap.arrival_seq, snap.req_id, 0, 0, snap.deficit, snap.need_d.size)
    vic, sc, _ = oracle.score_evict(snap.tick_now, snap.features, snap.weights, snap.bias, snap.session_state, None,
                                    de, snap.blk_session, snap.blk_last_access, snap.blk_depth, snap.blk_ref_flags,
                                    cap=max(snap.deficit, 1))
    if stage4 and pool is not None and vic.size:
        dst = np.empty(vic.size * page, np.uint8)
        oracle.swap_out(pool, n_chunks, chunk_bytes, chunk_bytes, page, vic, dst)
        oracle.swap_in(pool, n_chunks, chunk_bytes, chunk_bytes, page, dst, vic)
    return time.perf_counter() - t0, int(ho[-1])


def oracle_setup(snap, page, with_pool=True):
    import oracle
    S, L = snap.streams.shape
    sh, _ = oracle.hash_blocks(snap.streams.reshape(-1), np.arange(S + 1, dtype=np.uint64) * np.uint64(L))
    keys = sh.reshape(S, L // 16)[:, :snap.resident_blocks].reshape(-1)
    t = oracle.Table(snap.table_log2)
    t.insert(keys, np.arange(snap.M, dtype=np.uint32))
    pool = None
    if with_pool:
        try:
            pool = np.zeros(snap.M * page, np.uint8)  # lazily mapped; only victim pages are ever touched
        except MemoryError:
            pool = None
    return t, pool


def sample_snapshot(seed, sessions):
    """A bounded sample of configs[2] for the CPU oracle: the same recipe with `sessions` of the 256 sessions
    (16 requests, 4096 resident blocks and 5% eviction budget per session's share)."""
    from harness import gen
    return gen.stress_snapshot(seed=seed, S=sessions)


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on host cores; rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from harness import stress
    total_steps = args.steps + args.warmup
    # about 1 s per full-size step on one core (measured) => size the per-step sample for ~90 s in total
    sessions = int(min(256, max(2, 2 ** int(np.floor(np.log2(max(90.0 / (total_steps * 1.0), 1 / 128) * 256))))))
    snap = sample_snapshot(3, sessions)
    page = stress.STEP_N_CHUNKS * stress.STEP_CHUNK_BYTES
    table, pool = oracle_setup(snap, page)
    for _ in range(args.warmup):
        oracle_step(snap, table, pool, page, stress.STEP_N_CHUNKS, stress.STEP_CHUNK_BYTES)
    t = 0.0
    blocks = 0
    for _ in range(args.steps):
        dt, nb = oracle_step(snap, table, pool, page, stress.STEP_N_CHUNKS, stress.STEP_CHUNK_BYTES)
        t += dt
        blocks += nb
    value = blocks / t
    sample = (f"{sessions}/256 sessions of configs[2] per step ({snap.tok_off.size - 1} requests, {snap.M} resident "
              f"blocks, budget {snap.deficit}; stage 4 {'included' if pool is not None else 'skipped: no host RAM'})")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": t / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u64", "data": "synthetic",
        "config": {"workload": WORKLOAD, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def run_cuda(args):
    import torch

    import paper_2606_16824_b200 as cw
    from harness import dist as hdist
    from harness import gen, stress

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the CUDA path has no CPU fallback)")
    rank, local_rank, world = hdist.init("nccl")
    torch.cuda.set_device(local_rank)
    cw.lib()  # fails loudly if libcachewise.so is missing
    hbm_peak, peak_src = measured_peaks()
    stream = torch.cuda.Stream()
    snap = make_snapshot(3 + rank, args.scale)
    st = stress.StressStep(snap, stream)
    K, W = args.steps, max(args.warmup, 3)

    # ---- device-resident step: warm-up, then EXACTLY K timed steps
    with torch.cuda.stream(stream):
        for _ in range(W):
            st.step()
        stream.synchronize()
        res = st.results()
        nv = res["num_victims"]
        sampler = ClockSampler(local_rank)
        sampler.start()
        hdist.barrier()
        torch.cuda.synchronize()
        l0 = st.ctx.launches
        t_host0 = time.perf_counter()
        total_ms, per = time_region(torch, stream, st.stage_fns(), K)
        torch.cuda.synchronize()
        t_host1 = time.perf_counter()
        hdist.barrier()
        launches = st.ctx.launches - l0
        clocks = sampler.stop(t_host0, t_host1)
    status = st.ctx.sync(check=False)
    units = float(st.n_hashed) * K
    g_units, g_ms = hdist.aggregate(units, total_ms, "cuda")
    value = g_units / (g_ms * 1e-3)
    stage_ms = dict(zip(st.STAGES, per))
    alg = st.algorithmic_bytes(nv)
    rooflines = {}
    for name in st.STAGES:
        if name in stage_ms and stage_ms[name] > 0:
            ach = alg[name] / stage_ms[name] / 1e6
            rooflines[name] = {"bound": "hbm", "achieved": round(ach, 1), "peak": hbm_peak, "unit": "GB/s",
                               "frac": round(ach / hbm_peak, 4), "traffic": NCU_TRAFFIC_BYTES.get(name) if args.scale <= 1 else None,
                               "algorithmic_bytes": alg[name], "us": round(stage_ms[name] * 1e3, 2)}
    dominant = max(stage_ms, key=stage_ms.get)
    roofline = dict(rooflines[dominant], kernel=dominant, peak_source=peak_src)

    extra = {}
    if rank == 0 or world > 1:
        # ---- end to end: host buffers in, host buffers out, through the C ABI (every rank, same K)
        with torch.cuda.stream(stream):
            T = int(snap.tok_off[-1])
            h_tok = stress.as_torch(snap.tokens, pin=True)
            h_small = [(st.d_tok_off, stress.as_torch(snap.tok_off, pin=True)),
                       (st.d_hash_off, stress.as_torch(st.hash_off, pin=True)),
                       (st.d_need, stress.as_torch(snap.need_d, pin=True)),
                       (st.d_arr, stress.as_torch(snap.arrival_seq, pin=True)),
                       (st.d_rid, stress.as_torch(snap.req_id, pin=True)),
                       (st.d_feat, stress.as_torch(snap.features, pin=True)),
                       (st.d_state, stress.as_torch(snap.session_state, pin=True))]
            h_swap = torch.empty(st.cap * st.page, dtype=torch.uint8).pin_memory()
            h_scal = torch.zeros(3, dtype=torch.int32).pin_memory()
            h_order, h_k, h_g = (torch.zeros(st.R, dtype=torch.int32).pin_memory() for _ in range(3))
            h_vic = torch.zeros(st.cap, dtype=torch.int32).pin_memory()
            h2d = T * 4 + sum(h.numel() * h.element_size() for _, h in h_small)
            d2h = 12 + 3 * st.R * 4

            # The token ids of step i+1 travel host->device on a side stream while step i's victims travel
            # device->host (PCIe is full duplex): two device token buffers, one upload per step, all inside the
            # timed region.  Everything else of a step stays in order on `stream`.
            up_stream = torch.cuda.Stream()
            tok_bufs = [st.d_tok, torch.empty_like(st.d_tok)]
            tok_bufs[1][T:].zero_()
            up_done = [torch.cuda.Event(), torch.cuda.Event()]
            e2e_i = [0]

            def upload(k):
                up_stream.wait_stream(stream)          # the decide that last read this buffer has been enqueued
                with torch.cuda.stream(up_stream):
                    tok_bufs[k][:T].copy_(h_tok, non_blocking=True)
                    up_done[k].record(up_stream)

            upload(0)

            def e2e_step():
                k = e2e_i[0] & 1
                e2e_i[0] += 1
                st.d_tok = tok_bufs[k]
                stream.wait_event(up_done[k])          # this step's token ids are on the device
                for d, h in h_small:
                    d.copy_(h, non_blocking=True)
                st.decide()
                h_scal[0:1].copy_(st.d_na, non_blocking=True)
                h_scal[1:2].copy_(st.d_def, non_blocking=True)
                h_scal[2:3].copy_(st.d_nv, non_blocking=True)
                stream.synchronize()
                upload(k ^ 1)                          # next step's token ids: overlaps this step's swap-out
                n = int(h_scal[2])
                st.ctx.swap_out(st.d_vic, None, n, None, h_swap)
                st.ctx.swap_in(None, h_swap, st.d_vic, n)
                h_order.copy_(st.d_order, non_blocking=True)
                h_k.copy_(st.d_k, non_blocking=True)
                h_g.copy_(st.d_g, non_blocking=True)
                h_vic[:n].copy_(st.d_vic[:n], non_blocking=True)
                return n

            Ke = max(3, min(K, 20))
            for _ in range(2):
                n_e2e = e2e_step()
            hdist.barrier()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(Ke):
                n_e2e = e2e_step()
            e1.record(stream)
            torch.cuda.synchronize()
            hdist.barrier()
            e2e_ms = e0.elapsed_time(e1)
            st.ctx.sync(check=False)
            st.d_tok = tok_bufs[0]
        eu, et = hdist.aggregate(float(st.n_hashed) * Ke, e2e_ms, "cuda")
        extra["e2e"] = {"value": eu / (et * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d + n_e2e * st.page,
                        "d2h_bytes_per_step": d2h + n_e2e * st.page + n_e2e * 4, "steps": Ke,
                        "ms_per_step": round(et / Ke, 4)}
        del h_tok, h_swap, tok_bufs

    if rank == 0 and not args.quick:
        # ---- the <=100 us target: stages 1-3 as ONE CUDA-graph launch, cold (all requests hashed) and steady
        big = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

        def flush():
            big.zero_()

        with torch.cuda.stream(stream):
            dec = {}
            for name, steady in (("cold", False), ("steady", True)):
                dec[name + "_l2_warm"] = graph_latency(torch, stream, lambda: st.decide(steady))
                dec[name + "_l2_flushed"] = graph_latency(torch, stream, lambda: st.decide(steady), flush=flush)
        del big
        with torch.cuda.stream(stream):  # the steady-state hash call alone (CUDA events, median of 20)
            ts = []
            for _ in range(23):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                st.hash(True)
                e1.record(stream)
                stream.synchronize()
                ts.append(e0.elapsed_time(e1) * 1e3)
            dec["steady_hash_us"] = round(sorted(ts[3:])[10], 2)
        dec["note"] = ("stages 1-3 (hash, match, schedule, score/select) as one CUDA graph; cold = all 4096 requests "
                       f"hashed ({st.n_hashed} blocks), steady = hashes persist and the {st.new_requests} newest "
                       f"requests ({st.n_hashed_new} blocks) are hashed; target <= 100 us")
        extra["decision_step"] = dec

    st.close()
    del st
    torch.cuda.empty_cache()

    if rank == 0:
        pcie = pcie_peak(torch, stream)
        extra["pcie_peak"] = dict(pcie, gen5_x16_raw_gbs=PCIE_GEN5_X16_GBS)
        if not args.quick and not args.no_swap_sweep:
            try:
                avail_gib = 0
                for line in open("/proc/meminfo"):
                    if line.startswith("MemAvailable"):
                        avail_gib = int(line.split()[1]) / 2**20
                free_gib = torch.cuda.mem_get_info()[0] / 2**30
                ns = [1, 8, 64, 512]
                if avail_gib > 48 and free_gib > 90:
                    ns.append(4096)
                extra["swap_sweep"] = {"config": "BASELINE.json configs[3]: 160 x 32 KiB chunks (5 MiB page), 60 GiB "
                                                 "layer-major pool, random distinct victims",
                                       "rows": swap_sweep(torch, cw, gen, stream, hbm_peak, pcie, ns)}
            except Exception as e:  # the sweep is additional evidence; the step numbers above stand without it
                extra["swap_sweep"] = {"error": repr(e)[:300]}
        # ---- CPU baseline: the oracle as it stands, one core, bounded sample of the same workload
        if not args.no_cpu_baseline:
            sessions = 256 if args.scale <= 1 else max(256 // args.scale, 2)
            osnap = snap if args.scale <= 1 else sample_snapshot(3, sessions)
            page = stress.STEP_N_CHUNKS * stress.STEP_CHUNK_BYTES
            table, pool = oracle_setup(osnap, page)
            reps, t, nb = 0, 0.0, 0
            while reps < 3 and t < 20.0:
                dt, b = oracle_step(osnap, table, pool, page, stress.STEP_N_CHUNKS, stress.STEP_CHUNK_BYTES)
                t += dt
                nb += b
                reps += 1
            extra["cpu_baseline"] = {"value": nb / t, "unit": UNIT, "cores": 1, "kind": "oracle",
                                     "sample": f"{reps} full step(s) of the same configs[2] snapshot "
                                               f"({'with' if pool is not None else 'without'} stage 4), "
                                               f"{t / reps:.2f} s per step, host has {os.cpu_count()} cores",
                                     "ms_per_step": round(t / reps * 1e3, 1)}
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": g_ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u64",
            "data": "synthetic",
            "config": {"workload": WORKLOAD, "requests": st_R(snap), "blocks_hashed_per_step": int(units / K),
                       "tokens_per_step": int(snap.tok_off[-1]), "victims_per_step": nv,
                       "kv_page_bytes": stress.STEP_N_CHUNKS * stress.STEP_CHUNK_BYTES,
                       "l2": "inputs larger than L2 (token ids + swap traffic per step >> 126 MB); no flush",
                       "parallelism": f"replicas x{world} (no collective)", "status": status, "scale": args.scale},
            "roofline": roofline, "rooflines": rooflines,
            "stages_us": {k: round(v * 1e3, 2) for k, v in stage_ms.items()},
            "gpu_launches": int(launches), "clocks": clocks,
        }
        out.update(extra)
        print(json.dumps(out))
    hdist.finalize()


def st_R(snap):
    return int(snap.tok_off.size - 1)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--scale", type=int, default=1, help="debug only: shrink configs[2] by this factor")
    ap.add_argument("--quick", action="store_true", help="skip the graph-latency and swap-sweep sections")
    ap.add_argument("--no-swap-sweep", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
