"""bd_grid_filter_spline_static: step a2 (grid median filter + spline prefilter) for callers that cannot allocate.

Some users of libbkgdet run where cudaMalloc is off limits: a plug-in that lives inside another application's memory
budget and only gets the buffers it is handed, or a real-time acquisition loop that must never enter the CUDA allocator.
bd_grid_filter_spline needs a caller-allocated workspace for its Thomas factors; the _static entry point keeps that
scratch in a 256 KiB array built into the library (one per GPU, shared by every call, never cleared between calls).

What is checked, on a B200: its outputs equal the workspace path's on the same inputs, on two calls in a row that use
the array differently (so the second call runs on whatever the first left behind), and a batch beyond the array's
size is refused with a message instead of overrunning it.  The file name sorts last on purpose: `pytest -x` stops at
the first failure, and a failure here should not hide the parity tests.  It makes its own context, so it passes alone
in a fresh process (where its first call is also the one-time address look-up) as well as after the other tests.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def _grids(seed, B, ny, nx):
    rng = np.random.default_rng(seed)
    raw_b = torch.from_numpy(rng.normal(1000, 30, size=(B, ny, nx))).cuda()
    raw_r = torch.from_numpy(rng.uniform(5, 40, size=(B, ny, nx))).cuda()
    return raw_b, raw_r


def _assert_same(got, want):
    """Tolerances of test_k2_filter_and_prefilter: filtered grids bit-equal, coefficients to 1e-11 of their range."""
    bm, rm, cb, cr = got
    bm0, rm0, cb0, cr0 = want
    assert torch.equal(bm, bm0) and torch.equal(rm, rm0)
    for c, c0 in ((cb, cb0), (cr, cr0)):
        assert torch.isfinite(c).all()
        assert float((c - c0).abs().max()) <= 1e-11 * float(c0.abs().max())


def test_static_scratch_matches_workspace_path_on_two_calls_in_a_row():
    import paper_2502_10783_b200 as bd
    ctx = bd.Context(0)
    try:
        # Shapes that send the prefilter to global memory, i.e. really use the scratch array (a line longer than 160 cells,
        # or more cells than fit in shared memory), with different layouts of the factors inside the array; then a
        # grid that fits shared memory and leaves the array alone.  No synchronisation between consecutive static calls:
        # they are on one stream, which is the documented way to share the array.
        cases = [(3, 40, 300, 11, 7), (2, 161, 40, 3, 3), (1, 200, 180, 5, 5), (64, 32, 32, 3, 3), (3, 37, 36, 5, 5)]
        inputs = [_grids(10 * i + 1, B, ny, nx) for i, (B, ny, nx, _, _) in enumerate(cases)]
        for rep in range(2):   # the whole sequence twice: every call after the first starts from a used array
            got = [bd.grid_filter_spline_static(ctx, rb, rr, fh, fw) for (rb, rr), (_, _, _, fh, fw) in zip(inputs, cases)]
            torch.cuda.synchronize()
            for (rb, rr), (_, _, _, fh, fw), g in zip(inputs, cases, got):
                want = bd.grid_filter_spline(ctx, rb, rr, fh, fw)
                torch.cuda.synchronize()
                _assert_same(g, want)
        # caller-owned outputs (what a caller that cannot allocate passes): same numbers, written in place
        rb, rr = inputs[0]
        B, ny, nx, fh, fw = cases[0]
        out = (torch.full((B, ny, nx), -1.0, dtype=torch.float32, device="cuda"), torch.full((B, ny, nx), -1.0, dtype=torch.float32, device="cuda"),
               torch.full((B, ny, nx), -1.0, dtype=torch.float64, device="cuda"), torch.full((B, ny, nx), -1.0, dtype=torch.float64, device="cuda"))
        ret = bd.grid_filter_spline_static(ctx, rb, rr, fh, fw, out=out)
        torch.cuda.synchronize()
        assert all(a.data_ptr() == b.data_ptr() for a, b in zip(ret, out))
        _assert_same(out, bd.grid_filter_spline(ctx, rb, rr, fh, fw))
    finally:
        ctx.close()


def test_static_scratch_refuses_what_does_not_fit():
    import paper_2502_10783_b200 as bd
    ctx = bd.Context(0)
    try:
        # exactly at the limit: 4 * 64 * (64 + 64) = 32768 doubles
        assert 4 * 64 * (64 + 64) == bd.GRID_STATIC_MAX_DOUBLES
        rb, rr = _grids(5, 64, 64, 64)
        _assert_same(bd.grid_filter_spline_static(ctx, rb, rr, 3, 3), bd.grid_filter_spline(ctx, rb, rr, 3, 3))
        # one frame more: refused before anything is launched, outputs untouched
        rb, rr = _grids(6, 65, 64, 64)
        out = tuple(torch.full((65, 64, 64), -7.0, dtype=dt, device="cuda") for dt in (torch.float32, torch.float32, torch.float64, torch.float64))
        with pytest.raises(bd.BkgdetError, match=r"33280 doubles.*holds 32768"):
            bd.grid_filter_spline_static(ctx, rb, rr, 3, 3, out=out)
        torch.cuda.synchronize()
        assert all(bool((o == -7.0).all()) for o in out)
        # the call after a refusal still works
        rb, rr = _grids(7, 2, 161, 40)
        _assert_same(bd.grid_filter_spline_static(ctx, rb, rr, 3, 3), bd.grid_filter_spline(ctx, rb, rr, 3, 3))
    finally:
        ctx.close()
