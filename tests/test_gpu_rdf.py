"""-m gpu: cdh_rdf (g(r) post-processing, Eqs. 1-3) against the oracle, element by element.

Both sides evaluate the same IEEE double formula in the same order, so the values must be identical bits; the test
allows 2 ulp in case a compiler reassociates the constant 4*pi and says so if it is used.
"""
import numpy as np
import pytest

import paper_1808_01478_b200 as cdh
from paper_1808_01478_b200 import inputs
from oracle import oracle as cdh_oracle

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("k", [2, 3, 4])
def test_rdf_matches_oracle_and_ideal_gas(k):
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    p = inputs.reduced_config(k)
    box = p.box.reshape(-1, 3, 3)[0]
    volume = abs(float(np.linalg.det(box)))
    with cdh.Context(0) as ctx:
        hist = cdh.histograms_device(ctx, p)
        g = torch.empty((p.n_hist, p.n_bins), dtype=torch.float64, device=hist.device)
        ctx.cdh_rdf(hist, p.n_hist, p.n_bins, p.r_max, p.n_frames, p.pairs_per_hist(), volume, g)
        torch.cuda.synchronize()
    got = g.cpu().numpy()
    h = hist.cpu().numpy().view(np.uint64)
    want = cdh_oracle.rdf(h, p.r_max, p.n_frames, p.pairs_per_hist(), volume)
    assert np.array_equal(got, want) or np.allclose(got, want, rtol=4.5e-16, atol=0), "cdh_rdf differs from the oracle"
    # ideal gas: the r^2-weighted mean of g over the outer 80 % of the bins of the most populated row is 1
    w = (np.arange(p.n_bins) + 0.5) ** 2
    lo = p.n_bins // 5
    assert abs((got[-1, lo:] * w[lo:]).sum() / w[lo:].sum() - 1.0) < 0.02


def test_rdf_argument_errors():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    h = torch.zeros((1, 8), dtype=torch.int64, device="cuda")
    g = torch.full((1, 8), -3.0, dtype=torch.float64, device="cuda")
    with cdh.Context(0) as ctx:
        for kw in (dict(r_max=0.0), dict(volume=-1.0), dict(n_frames=0), dict(n_pairs=[float("nan")])):
            a = dict(r_max=1.0, volume=1.0, n_frames=1, n_pairs=[10.0])
            a.update(kw)
            with pytest.raises(cdh.CdhError):
                ctx.cdh_rdf(h, 1, 8, a["r_max"], a["n_frames"], a["n_pairs"], a["volume"], g)
    torch.cuda.synchronize()
    assert bool((g == -3.0).all())
