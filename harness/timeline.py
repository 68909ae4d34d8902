"""Two-branch timeline of the decision step (debug build only): %globaltimer stamps on stream_main between the calls,
and the phase stamps of the speculative evict kernel on the side stream, on one clock.

    python -m paper_2606_16824_b200.build --debug
    CACHEWISE_DEBUG=1 python -m harness.timeline

Eager launches with a one-thread stamp kernel between the calls: the absolute times are longer than inside a CUDA graph
(bench.py's decision_step); what the listing shows is WHICH kernels run beside each other.
"""
import torch
import paper_2606_16824_b200 as cw
from harness import gen, stress


def main():
    assert cw.DEBUG
    snap = gen.stress_snapshot(seed=3)
    stream = torch.cuda.Stream()
    st = stress.StressStep(snap, stream, with_pool=False)
    with torch.cuda.stream(stream):
        st.decide(False); st.decide(True); stream.synchronize()
        for name, steady in (("steady", True), ("cold", False)):
            for rep in range(3):
                fns = [st.score_evict_begin, lambda: st.hash(steady), st.match, st.schedule, st.score_evict_end]
                labels = ["begin (fork)", "hash (256 new requests)" if steady else "hash (all 4096 requests)", "match",
                          "schedule", "end (join + trim)"]
                main, ev = st.ctx.debug_timeline(fns)
            t0 = main[0]
            print(f"== {name} step, us from the first stamp on stream_main")
            for i, l in enumerate(labels):
                print(f"main  after {l:28s} {(main[i + 1] - t0) / 1e3:8.1f}")
            print(f"side  evict_kernel first stamp     {(ev[0] - t0) / 1e3:8.1f}")
            print(f"side  evict_kernel phase stamps    {[round((x - t0) / 1e3, 1) for x in ev[1:]]}")


if __name__ == "__main__":
    main()
