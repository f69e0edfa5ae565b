"""bsh_post_coincidences_static -- the coincidence step of the post-processing (section V.E, Eq. 44) for callers
that cannot allocate device memory: a job whose GPU memory is all in its own pool, a sweep whose other patches must not be
stalled by a cudaMalloc, a consumer that needs the pairs in bounded time.  Its work area is a fixed array inside the loaded
library instead of buffers a context grows, so what has to be shown is (1) that it returns exactly what the allocating
call bsh_post_coincidences returns -- the comparison is bit for bit, as in tests/test_gpu_post.py, because both run the same
FP64 operations in the same order --, (2) that a call is not disturbed by what the call before it left in that shared
array (several calls in a row, on lists of different lengths), and (3) that lists beyond the fixed limit are refused with a
message instead of overrunning the array.

The file name makes pytest collect it last: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It sets up everything it uses itself, so it passes alone in a fresh process (where its first call is also the
one that looks up the array's device address) as well as after the rest of the suite.  Needs a B200: -m gpu."""
import numpy as np
import pytest

import synth

pytestmark = pytest.mark.gpu


def _lists(na, nb, seed):
    a = synth.candidate_list(seed, n_background=na)
    b = synth.candidate_list(seed + 1, n_background=nb)
    m = min(a.n, b.n, 60)                         # some of b's candidates sit next to a's, so that pairs exist
    b.param[:m] = a.param[:m] + 0.7 * a.res[:m] * np.random.default_rng(seed).standard_normal((m, 6))
    b.res[:m] = synth.resolutions(b.param[:m, 0], b.param[:m, 3], b.param[:m, 4])
    return a, b


def _dev(torch, c):
    return tuple(torch.from_numpy(np.ascontiguousarray(x)).cuda() for x in (c.param, c.res, c.sig))


def _out(torch, cap):
    return (torch.full((cap,), -7, dtype=torch.int32, device="cuda"), torch.full((cap,), -7, dtype=torch.int32, device="cuda"),
            torch.full((cap, 6), -7.0, dtype=torch.float64, device="cuda"), torch.full((cap,), -7.0, dtype=torch.float64, device="cuda"))


def test_static_scratch_coincidences_equal_the_allocating_path_call_after_call():
    import torch
    import paper_1904_04873_b200 as bsh
    ctx = bsh.Context(0)
    try:
        # a long pair of lists, then a short one (its rows and counts lie inside what the long one wrote), then a pair with
        # other row lengths, then the first again on a side stream
        cases = [(1000, 777, 3.0, 11), (65, 31, 10.0, 12), (300, 300, 3.0, 13), (1000, 777, 3.0, 11)]
        side = torch.cuda.Stream()
        for call, (na, nb, window, seed) in enumerate(cases):
            a, b = _lists(na, nb, seed)
            da, db = _dev(torch, a), _dev(torch, b)
            want_a, want_b, want_cen, want_sig = ctx.post_coincidences(da, db, window)        # the existing path
            assert want_a.numel() >= 20
            cap = want_a.numel() + 5
            out = _out(torch, cap)
            torch.cuda.synchronize()
            stream = side if call == len(cases) - 1 else None
            n = bsh.post_coincidences_static(da, db, window, out, device=0, stream=stream)
            assert n == want_a.numel(), f"call {call}"
            got_a, got_b, got_cen, got_sig = (t[:n] for t in out)
            assert torch.equal(got_a, want_a) and torch.equal(got_b, want_b), f"call {call}: pair list"
            assert torch.equal(got_cen, want_cen) and torch.equal(got_sig, want_sig), f"call {call}: centroids"
            assert bool((out[0][n:] == -7).all()) and bool((out[3][n:] == -7.0).all()), "nothing written past the last pair"
            # a result buffer that is too small: the full count is reported, what fits is filled
            small = _out(torch, 5)
            assert bsh.post_coincidences_static(da, db, window, small, device=0) == n
            assert torch.equal(small[0], want_a[:5]) and torch.equal(small[1], want_b[:5])
    finally:
        ctx.close()


def test_static_scratch_limit_and_empty_lists():
    import torch
    import paper_1904_04873_b200 as bsh
    a, b = _lists(40, 40, 5)
    da, db = _dev(torch, a), _dev(torch, b)
    out = _out(torch, 16)
    n_big = bsh.binding.STATIC_MAX_CANDS + 1
    big = (torch.zeros((n_big, 6), dtype=torch.float64, device="cuda"), torch.ones((n_big, 6), dtype=torch.float64, device="cuda"),
           torch.ones(n_big, dtype=torch.float64, device="cuda"))
    for pair in ((big, db), (da, big)):
        with pytest.raises(bsh.BshError, match=r"bsh error -6: .*at most 8192 per list"):
            bsh.post_coincidences_static(*pair, 3.0, out)
    assert bool((out[0] == -7).all())                                # refused before anything ran
    with pytest.raises(bsh.BshError, match="bsh error -1"):
        bsh.post_coincidences_static(da, db, 0.0, out)               # window must be positive, as in the allocating call
    empty = tuple(t[:0] for t in da)
    assert bsh.post_coincidences_static(da, empty, 3.0, out) == 0 and bsh.post_coincidences_static(empty, db, 3.0, out) == 0
    # lists of exactly the limit are accepted (every row of the array in use); spot-check against the allocating path
    n_max = bsh.binding.STATIC_MAX_CANDS
    full = synth.candidate_list(77, n_background=n_max)
    sel = np.arange(n_max)
    full_dev = tuple(torch.from_numpy(np.ascontiguousarray(x[sel])).cuda() for x in (full.param, full.res, full.sig))
    assert full_dev[0].shape[0] == n_max
    ctx = bsh.Context(0)
    try:
        want = ctx.post_coincidences(full_dev, full_dev, 3.0)
        outs = _out(torch, want[0].numel())
        assert bsh.post_coincidences_static(full_dev, full_dev, 3.0, outs) == want[0].numel() >= n_max   # every a pairs with itself
        assert all(torch.equal(g, w) for g, w in zip(outs, want))
    finally:
        ctx.close()
