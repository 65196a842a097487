"""rd_apply_H_noalloc (include/refdef.h): S3 with its scratch in a static device array, for callers that cannot allocate.

Collected LAST on purpose (the file name sorts after every other test file): the suite runs with `pytest -x`, and a
failure here must not hide the parity tests.  The test passes alone in a fresh process and after the other tests: it
uses its own contexts and relies on nothing another test left behind (the static array keeps the last call's
contents; every call rewrites what it reads).

Checked against the existing path rd_apply_H (which the parity tests compare with the oracle) on the same inputs, on
two calls in a row with different inputs and masks; both paths do the same sums in the same order, so the comparison
is exact, well inside the 1e-12 relative tolerance of the operator parity tests.
"""
import numpy as np
import pytest

from workloads import make_config

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def rd():
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2606_17971_b200 as pkg

    pkg.load_library()
    return pkg


def test_apply_H_noalloc_matches_apply_H_on_two_calls_in_a_row(rd):
    import torch

    w = make_config(twin="c3_32")  # N = 32,768: 1024 slices, several waves of the grid; 3-D operator, 7-13 entries per row
    g = rd.RefDef.from_workload(w)
    try:
        assert w.N <= rd.NOALLOC_MAX_N
        rng = np.random.default_rng(2024)
        out = torch.full((w.N,), float("nan"), dtype=torch.float64, device="cuda")
        for call in range(2):
            v = torch.from_numpy(rng.standard_normal(w.N)).cuda()
            act = None if call == 0 else torch.from_numpy((rng.random(w.N) < 0.4).astype(np.uint8)).cuda()
            ref = g.apply_H(v, act)  # the existing path (synchronises)
            before = torch.cuda.memory_allocated()
            g.apply_H_noalloc(v, act, out)  # asynchronous on the context's stream
            torch.cuda.synchronize()
            assert torch.cuda.memory_allocated() == before
            scale = float(ref.abs().max())
            assert torch.isfinite(out).all()
            err = float((out - ref).abs().max())
            assert err <= 1e-12 * scale, (call, err, scale)
            assert torch.equal(out, ref), "same kernels' order of sums: bit-identical"
            if act is not None:
                assert float(out[act.bool()].abs().max()) == 0.0
        # the second call's result does not depend on what the first left in the scratch: repeat the first input
        v0 = torch.from_numpy(np.random.default_rng(2024).standard_normal(w.N)).cuda()
        g.apply_H_noalloc(v0, None, out)
        torch.cuda.synchronize()
        assert torch.equal(out, g.apply_H(v0, None))
    finally:
        g.close()


def test_apply_H_noalloc_a_second_context_shares_the_scratch(rd):
    """A smaller operator after a larger one: the stale tail of the shared array is never read."""
    import torch

    big, small = make_config(twin="c2_128"), make_config(1)
    for w in (big, small):
        g = rd.RefDef.from_workload(w)
        try:
            rng = np.random.default_rng(w.N)
            v = torch.from_numpy(rng.standard_normal(w.N)).cuda()
            act = torch.from_numpy((rng.random(w.N) < 0.5).astype(np.uint8)).cuda()
            out = torch.empty_like(v)
            g.apply_H_noalloc(v, act, out)
            torch.cuda.synchronize()
            assert torch.equal(out, g.apply_H(v, act))
        finally:
            g.close()


def test_apply_H_noalloc_rejects_what_it_cannot_serve(rd):
    import torch

    w = make_config(1)
    g = rd.RefDef.from_workload(w)
    try:
        v = torch.zeros(w.N, dtype=torch.float64, device="cuda")
        out = torch.empty_like(v)
        with pytest.raises(rd.RefDefError, match="device pointers"):
            g.apply_H_noalloc(np.zeros(w.N), None, out)  # host input
        with pytest.raises(rd.RefDefError, match="device pointers"):
            g.apply_H_noalloc(v, np.zeros(w.N, dtype=np.uint8), out)  # host mask
        with pytest.raises(rd.RefDefError, match="alias"):
            g.apply_H_noalloc(v, None, v)
    finally:
        g.close()
    # beyond the static maximum: a clear error, nothing launched (a diagonal operator one row too large)
    N = rd.NOALLOC_MAX_N + 1
    rowptr = np.arange(N + 1, dtype=np.int64)
    colidx = np.arange(N, dtype=np.int32)
    g = rd.RefDef(rowptr, colidx, np.ones(N), np.ones(N), 1e-4)
    try:
        v = torch.ones(N, dtype=torch.float64, device="cuda")
        out = torch.empty_like(v)
        n0 = g.kernel_launches()
        with pytest.raises(rd.RefDefError, match="RD_NOALLOC_MAX_N"):
            g.apply_H_noalloc(v, None, out)
        assert g.kernel_launches() == n0
        assert torch.allclose(g.apply_H(v, None), torch.full_like(v, 1.0 + 1e-4))  # the existing path has no such limit
    finally:
        g.close()
