"""-m gpu: cdh_histograms_stream (include/cdh.h) -- a host trajectory fed chunk by chunk with the copy of one chunk
overlapping the kernels of the previous one -- against the oracle, bin for bin, for every chunking.

The result is a sum of integers (Eq. 2), so it may not depend on frames_per_chunk, on whether the host
buffer is pageable or page-locked, or on the precision path's own staging.
"""
import numpy as np
import pytest

import paper_1808_01478_b200 as cdh
from paper_1808_01478_b200 import inputs
from oracle import oracle as cdh_oracle

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def _need_gpu():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")


def oracle_hist(p, precision="f32"):
    c = p.coords.astype(np.float64) if precision == "f64" else p.coords
    return cdh_oracle.histograms(c, p.species_offsets, p.box_type, p.box, p.r_max, p.n_bins, precision=precision)


def same(got, want, what):
    if not np.array_equal(got, want):
        d = got.astype(np.int64) - want.astype(np.int64)
        raise AssertionError(f"{what}: {np.count_nonzero(d)} bins differ, L1 = {int(np.abs(d).sum())}, "
                             f"sums {int(got.sum())} / {int(want.sum())}")


def trajectory(n_frames=7):
    return inputs.config4(n_frames=n_frames, counts=(600, 1900), n_bins=3000)


@pytest.mark.parametrize("fpc", [0, 1, 2, 3, 7, 100])
def test_every_chunking_gives_the_oracle_histograms(fpc):
    _need_gpu()
    p = trajectory()
    want = oracle_hist(p)
    with cdh.Context(0) as ctx:
        got = ctx.cdh_histograms_stream(p.coords, p.species_offsets, p.box_type, p.box, p.r_max, p.n_bins,
                                        frames_per_chunk=fpc)
        same(got, want, f"pageable host buffer, {fpc} frames per chunk")
        pinned = torch.from_numpy(p.coords).pin_memory()
        s = torch.cuda.Stream()
        got = ctx.cdh_histograms_stream(pinned, p.species_offsets, p.box_type, p.box, p.r_max, p.n_bins,
                                        frames_per_chunk=fpc, stream=s)
        same(got, want, f"page-locked host buffer on a side stream, {fpc} frames per chunk")
        # the one-shot host entry on the same context afterwards (shared scratch) still agrees
        same(ctx.cdh_histograms_host(p.coords, p.species_offsets, p.box_type, p.box, p.r_max, p.n_bins), want, "one shot")


def test_per_frame_boxes_follow_their_chunk():
    _need_gpu()
    g = np.random.Generator(np.random.PCG64(34))
    f, n = 5, 1300
    boxes = np.stack([np.array([[7.0 + k, 0, 0], [1.0, 6.5, 0], [0.5 * k, -1.0, 8.0 - k]]) for k in range(f)])
    coords = np.stack([(g.random((n, 3)) @ boxes[k]).astype(np.float32) for k in range(f)])
    p = inputs.Problem("tri_per_frame_stream", coords, np.array([0, 300, n], dtype=np.int32), inputs.BOX_TRICLINIC,
                       boxes.reshape(f, 9), 2.4, 999)
    want = oracle_hist(p)
    with cdh.Context(0) as ctx:
        for fpc in (1, 2, 5):
            got = ctx.cdh_histograms_stream(p.coords, p.species_offsets, p.box_type, p.box, p.r_max, p.n_bins,
                                            frames_per_chunk=fpc)
            same(got, want, f"per-frame triclinic boxes, {fpc} frames per chunk")


def test_double_precision_trajectory():
    _need_gpu()
    p = trajectory(4)
    want = oracle_hist(p, "f64")
    with cdh.Context(0) as ctx:
        got = ctx.cdh_histograms_stream(p.coords.astype(np.float64), p.species_offsets, p.box_type, p.box, p.r_max,
                                        p.n_bins, precision=cdh.F64, frames_per_chunk=3)
    same(got, want, "f64, chunks of 3 + 1 frames")


def test_accumulate_context_and_repeated_calls_do_not_leak_into_the_result():
    _need_gpu()
    p = trajectory(3)
    want = oracle_hist(p)
    with cdh.Context(0, cdh.FLAG_ACCUMULATE) as ctx:            # the flag is for cdh_histograms only: overwritten here
        for _ in range(3):
            got = ctx.cdh_histograms_stream(p.coords, p.species_offsets, p.box_type, p.box, p.r_max, p.n_bins,
                                            frames_per_chunk=2)
            same(got, want, "repeated call")


def test_invalid_arguments_are_refused_before_anything_runs():
    _need_gpu()
    p = trajectory(2)
    with cdh.Context(0) as ctx:
        with pytest.raises(cdh.CdhError) as e:
            ctx.cdh_histograms_stream(p.coords, p.species_offsets, p.box_type, p.box, p.r_max, p.n_bins,
                                      frames_per_chunk=-1)
        assert e.value.code == -1            # CDH_ERR_INVALID_ARG
        with pytest.raises(cdh.CdhError):
            ctx.cdh_histograms_stream(p.coords, p.species_offsets, p.box_type, p.box, -1.0, p.n_bins)


def test_plan_cache_many_shapes_two_streams_and_changing_coordinates():
    """The context caches plans keyed by the arguments (not the coordinate values): repeated calls with new
    coordinates, more distinct shapes than the cache holds (least recently used out) and a plan reused on another
    stream than the one its tables were uploaded on must all give the oracle's integers."""
    _need_gpu()
    box = np.diag([3.0, 3.5, 4.0])
    with cdh.Context(0) as ctx:
        s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
        shapes = [(300 + 37 * k, 100 + 11 * k) for k in range(20)]            # 20 plans > 16 cached
        for rnd in range(2):
            for k, counts in enumerate(shapes):
                p = inputs.uniform_problem(1000 * rnd + k, counts, inputs.BOX_ORTHO, 500 + k, 1.4, box=box)
                out = cdh.histograms_device(ctx, p, stream=(s1 if (k + rnd) % 2 else s2))
                torch.cuda.synchronize()
                got = out.cpu().numpy().view(np.uint64)
                assert np.array_equal(got, cdh_oracle.problem_histograms(p, "f32")), (rnd, counts)
        # same plan, back-to-back calls on alternating streams without a host synchronisation in between
        p = inputs.uniform_problem(5, (700, 200), inputs.BOX_ORTHO, 640, 1.4, box=box)
        q = inputs.uniform_problem(6, (700, 200), inputs.BOX_ORTHO, 640, 1.4, box=box)
        a = cdh.histograms_device(ctx, p, stream=s1)
        s2.wait_stream(s1)                                                     # the context's scratch is reused: order the streams
        b = cdh.histograms_device(ctx, q, stream=s2)
        torch.cuda.synchronize()
        assert np.array_equal(a.cpu().numpy().view(np.uint64), cdh_oracle.problem_histograms(p, "f32"))
        assert np.array_equal(b.cpu().numpy().view(np.uint64), cdh_oracle.problem_histograms(q, "f32"))


def test_cached_call_captured_into_a_cuda_graph_and_replayed_between_other_calls():
    """A call that hits the plan cache enqueues kernels only (include/cdh.h): it can be recorded into a CUDA graph.  ONE captured
    call, replayed several times with other (uncaptured) calls of the same context in between: every replay and every call in
    between must give the oracle-checked result (the library's per-call scalars must not leak between them)."""
    _need_gpu()
    dev = torch.device("cuda", 0)
    p, q = inputs.reduced_config(2), inputs.reduced_config(3)
    want_p, want_q = cdh_oracle.problem_histograms(p, "f32"), cdh_oracle.problem_histograms(q, "f32")
    cp, cq = torch.from_numpy(p.coords).to(dev), torch.from_numpy(q.coords).to(dev)
    op = torch.zeros((p.n_hist, p.n_bins), dtype=torch.int64, device=dev)
    oq = torch.zeros((q.n_hist, q.n_bins), dtype=torch.int64, device=dev)
    s = torch.cuda.Stream()
    with cdh.Context(0) as ctx:
        def call(prob, coords, out):
            ctx.cdh_histograms(coords, prob.n_frames, prob.species_offsets, prob.box_type, prob.box, prob.r_max, prob.n_bins, out, stream=s)
        with torch.cuda.stream(s):
            call(p, cp, op); call(q, cq, oq)            # build both plans before the capture
        s.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            call(p, cp, op)                             # one call: an odd number on purpose
        for rep in range(3):
            op.fill_(-1)
            with torch.cuda.stream(s):
                g.replay()
            s.synchronize()
            assert np.array_equal(op.cpu().numpy().view(np.uint64), want_p), f"replay {rep}"
            oq.fill_(-1)
            with torch.cuda.stream(s):
                call(q, cq, oq)
                if rep == 1:
                    call(q, cq, oq)
            s.synchronize()
            assert np.array_equal(oq.cpu().numpy().view(np.uint64), want_q), f"uncaptured call after replay {rep}"
