"""-m gpu: cdh_histograms_noalloc (include/cdh.h) against the existing context path, cdh_histograms.

The entry point keeps all its device scratch in one static device array inside the library (no cudaMalloc on any call).
The array is shared by every call and keeps the last call's contents, so every comparison here is made on TWO calls in a
row: the second one must not see anything of the first.  Integer histograms: the bar is bit-exact, as everywhere else.
Collected last on purpose (the file name): the suite runs with pytest -x.
"""
import numpy as np
import pytest

import paper_1808_01478_b200 as cdh
from paper_1808_01478_b200 import inputs

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def dev():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch.device("cuda", 0)


def existing_path(p):
    with cdh.Context(0) as ctx:
        out = cdh.histograms_device(ctx, p)
        torch.cuda.synchronize()
        return out.cpu().numpy().view(np.uint64)


def no_alloc(p, dev, stream=None, poison=False):
    coords = torch.from_numpy(p.coords).to(dev)
    out = torch.empty((p.n_hist, p.n_bins), dtype=torch.int64, device=dev)
    if poison:
        out.fill_(-7)                       # the call overwrites its result
    cdh.cdh_histograms_noalloc(0, coords, p.n_frames, p.species_offsets, p.box_type, p.box, p.r_max, p.n_bins, out, stream=stream)
    torch.cuda.synchronize()
    return out.cpu().numpy().view(np.uint64)


def same(got, want, what):
    assert got.shape == want.shape, what
    if not np.array_equal(got, want):
        d = got.astype(np.int64) - want.astype(np.int64)
        raise AssertionError(f"{what}: {np.count_nonzero(d)} bins differ, L1 = {int(np.abs(d).sum())}")


@pytest.mark.parametrize("k", [1, 2, 3, 4])
def test_two_calls_in_a_row_match_the_existing_path(dev, k):
    p = inputs.reduced_config(k)            # no box / orthorhombic / triclinic / several frames
    want = existing_path(p)
    same(no_alloc(p, dev, poison=True), want, f"{p.name}: first call")
    same(no_alloc(p, dev, poison=True), want, f"{p.name}: second call (same problem, scratch holds the first call's contents)")


def test_a_smaller_problem_after_a_larger_one_sees_nothing_of_it(dev):
    big = inputs.config2(counts=(5000, 30000, 60000), n_bins=10000)      # config 2 at full size: 102,400 of 131,072 padded particles
    small = inputs.uniform_problem(11, (37, 5), inputs.BOX_NONE, 300, 0.8)
    tri = inputs.reduced_config(3)
    want_big, want_small, want_tri = existing_path(big), existing_path(small), existing_path(tri)
    stream = torch.cuda.Stream()
    for rep in range(2):
        same(no_alloc(big, dev, stream=stream), want_big, f"config 2 full size, pass {rep}")
        same(no_alloc(small, dev, stream=stream), want_small, f"42 points right after config 2, pass {rep}")
        same(no_alloc(tri, dev), want_tri, f"triclinic on the default stream after that, pass {rep}")


def test_empty_species_and_single_particles(dev):
    p = inputs.uniform_problem(5, (0, 1, 9), inputs.BOX_ORTHO, 64, 0.5, box=np.diag([1.0, 1.0, 1.0]))
    want = existing_path(p)
    same(no_alloc(p, dev, poison=True), want, "species of 0, 1 and 9 particles")
    same(no_alloc(p, dev, poison=True), want, "species of 0, 1 and 9 particles, again")


def test_sizes_beyond_the_static_scratch_are_rejected_with_a_clear_error(dev):
    coords = torch.zeros((1, 8, 3), dtype=torch.float32, device=dev)
    out = torch.full((1, 16), 5, dtype=torch.int64, device=dev)
    n_too_many = cdh.NOALLOC_MAX_PADDED_PARTICLES + 1
    with pytest.raises(cdh.CdhError) as e:          # the offsets alone decide: nothing is read, nothing enqueued
        cdh.cdh_histograms_noalloc(0, coords.data_ptr(), 1, [0, n_too_many], inputs.BOX_NONE, None, 1.0, 16, out.data_ptr())
    assert e.value.code == -2 and "maximum of 131072 padded particles" in str(e.value)
    with pytest.raises(cdh.CdhError) as e:          # frames count too: 40 frames x 4096 padded particles
        cdh.cdh_histograms_noalloc(0, coords.data_ptr(), 40, [0, 8], inputs.BOX_NONE, None, 1.0, 16, out.data_ptr())
    assert e.value.code == -2 and "padded particles" in str(e.value)
    wide = torch.zeros((1, cdh.NOALLOC_MAX_BINS + 1), dtype=torch.int64, device=dev)
    with pytest.raises(cdh.CdhError) as e:
        cdh.cdh_histograms_noalloc(0, coords, 1, [0, 8], inputs.BOX_NONE, None, 1.0, cdh.NOALLOC_MAX_BINS + 1, wide)
    assert e.value.code == -2 and "n_bins" in str(e.value)
    torch.cuda.synchronize()
    assert int(out.min()) == 5 and int(out.max()) == 5      # rejected calls touch nothing
    # and the entry point still works afterwards
    p = inputs.reduced_config(1)
    same(no_alloc(p, dev), existing_path(p), "config 1 after the rejected calls")


def test_recorded_into_a_cuda_graph_and_replayed(dev):
    """Calls with small work tables (they travel as a kernel parameter) have no node that reads host memory: recorded into a
    CUDA graph and replayed, with OTHER calls of the entry point in between (which overwrite the shared scratch), every replay
    must rebuild everything it needs and give the existing path's result."""
    p, q = inputs.reduced_config(2), inputs.reduced_config(3)
    want_p, want_q = existing_path(p), existing_path(q)
    same(no_alloc(p, dev), want_p, "before the capture")        # device set-up (cudaGetSymbolAddress) happens outside the capture
    coords = torch.from_numpy(p.coords).to(dev)
    out = torch.empty((p.n_hist, p.n_bins), dtype=torch.int64, device=dev)
    s = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=s):
        cdh.cdh_histograms_noalloc(0, coords, p.n_frames, p.species_offsets, p.box_type, p.box, p.r_max, p.n_bins, out, stream=s)
    for rep in range(3):
        out.fill_(-3)
        with torch.cuda.stream(s):
            g.replay()
        s.synchronize()
        same(out.cpu().numpy().view(np.uint64), want_p, f"replay {rep}")
        same(no_alloc(q, dev, stream=s), want_q, f"another problem through the same scratch after replay {rep}")


def test_large_tables_are_refused_on_a_capturing_stream(dev):
    # 32 species: 528 species pairs, 33.8 KB of work tables -- more than a kernel parameter holds, so they are copied from host
    # memory of the call; recorded into a graph that copy would read freed memory on replay: the call must refuse, record
    # nothing, leave the capture valid, and work again afterwards
    counts = (3,) * 32
    p = inputs.uniform_problem(99, counts, inputs.BOX_NONE, 50, 2.0)
    coords = torch.from_numpy(p.coords).to(dev)
    out = torch.full((p.n_hist, p.n_bins), 5, dtype=torch.int64, device=dev)
    want = existing_path(p)
    same(no_alloc(p, dev), want, "32 species, not captured")
    s = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=s):
        with pytest.raises(cdh.CdhError) as e:
            cdh.cdh_histograms_noalloc(0, coords, p.n_frames, p.species_offsets, p.box_type, p.box, p.r_max, p.n_bins, out, stream=s)
        out.add_(1)                                              # something to record, so that the graph is not empty
    assert e.value.code == -2 and "captured" in str(e.value)
    g.replay()
    torch.cuda.synchronize()
    assert int(out.min()) == 6 and int(out.max()) == 6
    same(no_alloc(p, dev), want, "after the capture")
