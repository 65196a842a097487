"""Matched replay (bench.py --mode replay; Table 3): the protocol's qualitative expectation on a twin of
config 2 -- the same inactive systems, zero initial guesses, the same reference: direct restriction never needs more
iterations in total than zero-extension, and every replayed solve is verified at 1e-8."""
import argparse

import pytest

pytestmark = pytest.mark.gpu


def test_matched_replay_direct_restriction_beats_zero_extension():
    import torch

    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import bench

    args = argparse.Namespace(config=2, twin="c2_48", steps=2, alg1_variant=0, reference="sine", ref_tol=1e-3)
    out = bench.run_replay(args)
    m = out["methods"]
    assert out["config"]["systems"] >= 10
    for name in ("refdef", "zeroext", "jacobi"):
        assert m[name]["worst_rel_resid"] <= 1e-8
    assert m["refdef"]["cg_iters"] <= m["zeroext"]["cg_iters"] <= 1.02 * m["jacobi"]["cg_iters"]
    assert m["refdef"]["mean_rank"] >= m["zeroext"]["mean_rank"]
    assert out["iteration_ratio_zeroext_over_direct"] >= 1.0
    # eq. (24): a fraction; zero for rank zero; direct restriction keeps the larger coarse space here
    assert m["jacobi"]["mean_chi"] == 0.0
    assert 0.0 < m["zeroext"]["min_chi"] <= m["zeroext"]["mean_chi"] < 1.0
    assert 0.0 < m["refdef"]["min_chi"] <= m["refdef"]["mean_chi"] < 1.0
    assert m["refdef"]["mean_chi"] >= m["zeroext"]["mean_chi"]
