"""The allocation-free entry point rte_media_lognormal_noalloc (static in-library scratch, include/rte.h) against the
existing path rte_media_lognormal (caller scratch + cudaMalloc) on the same arguments.  Collected last on purpose (the
suite runs with pytest -x).  Run with -m gpu."""
import numpy as np
import pytest
import torch

import paper_1801_06364_b200 as rte

pytestmark = pytest.mark.gpu
DEV = "cuda:0"
TOL = 1e-5      # same kernels in the same order; only the fp64 atomics of the moments may differ in order


def both(grid, dx, seed, mean, sigma_log, corr_len, poison):
    shape = (grid[3], grid[2], grid[1])
    ref = torch.empty(shape, dtype=torch.float32, device=DEV)
    scr = torch.empty_like(ref)
    rte.rte_media_lognormal(grid, dx, seed, mean, sigma_log, corr_len, ref, scr)
    got = torch.full(shape, poison, dtype=torch.float32, device=DEV)
    rte.rte_media_lognormal_noalloc(grid, dx, seed, mean, sigma_log, corr_len, got)
    torch.cuda.synchronize()
    return got.cpu().numpy().astype(np.float64), ref.cpu().numpy().astype(np.float64)


def test_no_alloc_lognormal_matches_existing_path_twice_in_a_row():
    # two calls in a row with different grids / seeds / parameters: the second finds the first's contents in the static
    # scratch (blur field and moments) and must not be affected by them; then the first again
    cases = [((3, 48, 32, 64), 0.25, 5, 10.0, 0.3, 2.0), ((2, 96, 128, 1), 0.05, 6364, 7.5, 0.5, 0.4),
             ((3, 48, 32, 64), 0.25, 5, 10.0, 0.3, 2.0)]
    outs = []
    for k, (grid, dx, seed, mean, sl, cl) in enumerate(cases):
        got, ref = both(grid, dx, seed, mean, sl, cl, poison=float(k) - 1.0)
        assert np.isfinite(got).all() and (got > 0).all()
        assert np.abs(got / ref - 1).max() <= TOL, (k, np.abs(got / ref - 1).max())
        lf = np.log(got)
        assert abs(lf.std() - sl) < 1e-3 and abs(lf.mean() - (np.log(mean) - 0.5 * sl * sl)) < 1e-3
        outs.append(got)
    assert np.abs(outs[0] / outs[2] - 1).max() <= TOL          # same arguments, same field, whatever ran in between


def test_no_alloc_lognormal_limit_and_arguments():
    out = torch.empty((1, 1, 16), dtype=torch.float32, device=DEV)
    with pytest.raises(rte.RteError) as e:                     # 256 * 128 * 128 = 4 194 304 cells > 2 097 152
        rte.rte_media_lognormal_noalloc((3, 256, 128, 128), 0.1, 1, 10.0, 0.3, 2.0, out)
    assert e.value.code == rte.RTE_EUNSUPPORTED and "2097152" in str(e.value)
    with pytest.raises(rte.RteError) as e:
        rte.rte_media_lognormal_noalloc((3, 16, 16, 16), 0.1, 1, -1.0, 0.3, 2.0, out)
    assert e.value.code == rte.RTE_EINVAL
    full = torch.empty((128, 128, 128), dtype=torch.float32, device=DEV)      # exactly the maximum is accepted
    rte.rte_media_lognormal_noalloc((3, 128, 128, 128), 0.8, 2018, 10.0, 0.3, 2.0, full)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(full).all())
