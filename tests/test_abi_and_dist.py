"""CPU-only checks of the boundary and of the host logic around it (no compute calls: there is no GPU here).

* libcachewise.so builds for sm_100a, loads, and exports every symbol include/cachewise.h declares;
* the Python binding declares the same set; the cw_config struct layouts agree (field by field);
* host-side argument checks that need no device answer before any CUDA call;
* bench.py's multi-rank aggregation (replicas, max-over-ranks time) on gloo, world_size 2.
"""
import ctypes as C
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "cachewise.h")


def _declared():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    src = re.sub(r"#ifdef CW_DEBUG.*?#endif", "", src, flags=re.S)  # debug-build-only diagnostics
    return sorted(set(re.findall(r"\b(cw_[a-z_0-9]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    from paper_2606_16824_b200 import build
    import paper_2606_16824_b200 as cw
    build.build()
    return cw.lib()


def test_library_exports_every_declared_symbol(lib):
    import paper_2606_16824_b200 as cw
    names = _declared()
    assert len(names) >= 19 and "cw_hash_blocks" in names and "cw_swap_in" in names
    for n in names:
        assert hasattr(lib, n), f"{n} declared in cachewise.h but not exported"
    assert sorted(cw.EXPORTS) == names, "binding and header disagree"
    out = subprocess.check_output(["nm", "-D", "--defined-only", cw.LIB_PATH], text=True)
    exported = sorted(l.split()[-1] for l in out.splitlines() if " T " in l)
    assert [e for e in exported if e.startswith("cw_")] == names
    assert not [e for e in exported if not e.startswith("cw_") and not e.startswith("_")], "stray exports"


def test_config_struct_layout_matches_the_header():
    """Compile a tiny C program against the header and compare offsets with the ctypes mirror."""
    import paper_2606_16824_b200 as cw
    fields = [f for f, _ in cw.CwConfig._fields_]
    prog = "#include <stdio.h>\n#include <stddef.h>\n#include \"cachewise.h\"\nint main(){"
    for f in fields:
        prog += f'printf("%zu\\n", offsetof(cw_config, {f}));'
    prog += 'printf("%zu\\n", sizeof(cw_config));return 0;}'
    exe = os.path.join("/tmp", f"cw_layout_{os.getpid()}")
    subprocess.run(["gcc", "-x", "c", "-", "-I", os.path.join(ROOT, "include"), "-o", exe], input=prog, text=True,
                   check=True)
    got = [int(x) for x in subprocess.check_output([exe], text=True).split()]
    os.unlink(exe)
    want = [getattr(cw.CwConfig, f).offset for f in fields] + [C.sizeof(cw.CwConfig)]
    assert got == want


def test_null_ctx_and_bad_config_are_rejected_without_a_device(lib):
    import paper_2606_16824_b200 as cw
    assert lib.cw_sync(None) == cw.CW_E_STATE
    assert lib.cw_destroy(None) == cw.CW_E_STATE
    assert lib.cw_join_copy(None) == cw.CW_E_STATE
    assert lib.cw_hash_blocks(None, None, None, None, None, None, None, 1, None) == cw.CW_E_STATE
    assert lib.cw_swap_in(None, None, None, None, 1) == cw.CW_E_STATE
    assert lib.cw_launch_count(None) == 0
    h = C.c_void_p()
    assert lib.cw_create(None, C.byref(h)) == cw.CW_E_INVAL
    bad = cw.CwConfig(num_blocks=16, table_log2_slots=4, block_tokens=32, max_requests=1)   # block_tokens != 16
    assert lib.cw_create(C.byref(bad), C.byref(h)) == cw.CW_E_INVAL and not h
    bad = cw.CwConfig(num_blocks=1024, table_log2_slots=10, block_tokens=16, max_requests=1)  # load factor > 0.5
    assert lib.cw_create(C.byref(bad), C.byref(h)) == cw.CW_E_INVAL and not h
    bad = cw.CwConfig(num_blocks=16, table_log2_slots=6, block_tokens=16, max_requests=1, n_chunks=2, chunk_bytes=24,
                      chunk_stride=24, block_stride=48, d_pool=4096)                       # chunk_bytes % 16 != 0
    assert lib.cw_create(C.byref(bad), C.byref(h)) == cw.CW_E_INVAL and not h


_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
from harness import dist as hdist
rank, local, world = hdist.init("gloo")
assert world == 2
hdist.barrier()
# rank r processed (r+1)*1000 units in (r+1)*10 ms: whole job = 3000 units / 20 ms
u, t = hdist.aggregate((rank + 1) * 1000, (rank + 1) * 10.0)
assert (u, t) == (3000.0, 20.0), (u, t)
v = hdist.throughput((rank + 1) * 1000, (rank + 1) * 10.0)
assert abs(v - 150000.0) < 1e-6, v
hdist.finalize()
print("ok", rank)
"""


def test_replica_aggregation_world_size_2_gloo(tmp_path):
    script = tmp_path / "w.py"
    script.write_text(_WORKER.format(root=ROOT))
    port = 29600 + os.getpid() % 300
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    for p in procs:
        out, _ = p.communicate(timeout=120)
        assert p.returncode == 0 and "ok" in out, out


def test_reference_arm_other_ranks_exit_without_work():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                         env=env, capture_output=True, text=True, timeout=120)
    assert out.returncode == 0 and out.stdout.strip() == ""


def test_bench_gpus_2_launches_two_ranks():
    """`python bench.py --gpus 2` (no torchrun around it) must start two ranks itself and report
    n_gpus 2; --dist-check stops after the rendezvous, the barrier and the max-over-ranks aggregation (gloo here)."""
    import json
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_PORT")}
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--dist-check"], env=env,
                         capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stdout + out.stderr
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    d = json.loads(line)
    assert d["n_gpus"] == 2 and d["units"] == 3000.0 and d["max_ms"] == 20.0


def test_tp_head_slices_partition_the_page_and_reassemble_through_the_oracle():
    """SURVEY.md 8f NEXT-4 (TP=2): stage 4 shards by KV head with no exchange.  Host logic only (the
    GPU halves are in test_gpu_evict_swap.py): the slices partition every chunk, and the ranks' oracle swap-outs of
    their shards, re-interleaved, are the oracle's swap-out of the unsharded pool, for both pool layouts."""
    import numpy as np
    import oracle
    from harness import gen, tp as htp
    M, n_chunks, cb, n = 24, 4, 256, 9
    g = gen.rng(91, 0)
    full = g.integers(0, 256, size=(n_chunks, M, cb), dtype=np.uint8)
    vic = g.permutation(M)[:n].astype(np.uint32)
    exp = oracle.swap_out(full.reshape(-1).copy(), n_chunks, cb, M * cb, cb, vic, np.zeros(n * n_chunks * cb, np.uint8))
    for tp in (1, 2, 4, 8):
        cover = np.zeros(cb, np.int32)
        pages = []
        for r in range(tp):
            off, sb = htp.head_slice(cb, tp, r)
            cover[off:off + sb] += 1
            for layout in ("layer", "block"):
                shard = htp.shard_pool(full, tp, r, layout)
                cs, bs = (M * sb, sb) if layout == "layer" else (sb, n_chunks * sb)
                out = oracle.swap_out(shard, n_chunks, sb, cs, bs, vic, np.zeros(n * n_chunks * sb, np.uint8))
                if layout == "layer":
                    pages.append(out)
                else:
                    assert np.array_equal(out, pages[-1])          # the layout does not change the staged page
        assert (cover == 1).all()
        assert np.array_equal(htp.interleave_pages(pages, n, n_chunks).reshape(-1), exp)
    with pytest.raises(ValueError):
        htp.head_slice(cb, 3, 0)
    with pytest.raises(ValueError):
        htp.head_slice(cb, 2, 2)


def test_bench_reads_roofline_traffic_from_the_committed_ncu_export():
    """roofline.traffic is not a constant in bench.py; it is parsed from the raw `ncu --set full`
    export under profiles/ (dram__bytes_read.sum + dram__bytes_write.sum of each stage's kernel)."""
    sys.path.insert(0, ROOT)
    import bench
    assert "NCU_TRAFFIC_BYTES" not in open(os.path.join(ROOT, "bench.py")).read()
    t = bench.ncu_traffic()
    assert set(t) == {"hash", "match", "schedule", "score_evict", "gather", "scatter"}
    assert 0.9 * 2 * 16384 * 52352 < t["gather"] < 1.1 * 2 * 16384 * 52352      # read + write of every victim page
    assert 0.85 * 421e6 < t["hash"] < 1.15 * 475e6                              # the token ids, once
    md = open(os.path.join(ROOT, "profiles", "r2_step_kernels_raw.md")).read()
    assert "ncu --set full" in md and "bench.py" in md                            # the export names its command
    us = bench.ncu_kernel_us()                                                    # the main kernel of each stage alone
    assert set(us) == set(t) and 64 < us["hash"] < 130 and 200 < us["gather"] < 320
