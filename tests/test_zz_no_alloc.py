"""rift_ile_reduce_static, the allocation-free entry point (include/rift_ile.h): the reduce kernels of step a8 (Eq. (3),
PAPER.md:55; App. B) run with their scratch in a file-scope device array instead of buffers owned by a handle.  Checked
against the existing path, rift_ile_reduce(merge=0), on two calls in a row whose shapes differ (the shared array keeps the
first call's contents), and against the oracle's reduce.  Collected last on purpose (pytest -x)."""
import numpy as np
import pytest

import paper_2210_07912_b200 as rift
from paper_2210_07912_b200 import synth

from helpers import build, create

pytestmark = pytest.mark.gpu

TOL_FP64_REL = 1e-10         # BASELINE.json north_star, fp64 mode (the two paths run the same kernels: observed bit-identical)


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available(), "GPU tests need a CUDA device"
    rift.lib()
    return t


def _close(a, b):
    a, b = np.asarray(a, dtype=np.float64), np.asarray(b, dtype=np.float64)
    both_nan = np.isnan(a) & np.isnan(b)
    return np.all(both_nan | (np.abs(a - b) <= TOL_FP64_REL * np.maximum(1.0, np.abs(b))))


def test_reduce_static_matches_reduce_on_two_calls_in_a_row(torch, oracle):
    cfg = synth.with_overrides(synth.CONFIGS[0], n_points=1)
    inp = build(oracle, cfg, n_points=1)
    h = create(rift, inp, rift.RIFT_PREC_FP64)
    stream = torch.cuda.current_stream().cuda_stream
    # call 1: 3 segments x 5000 real lnL values with importance weights; call 2: 7 segments x 1237, no weights, and one
    # segment holding a NaN (its outputs are NaN on both paths) -- another shape, so stale scratch contents would show
    shapes = [(3, 5000, True), (7, 1237, False)]
    free_before = None
    for call, (n_seg, n, weighted) in enumerate(shapes):
        params = np.concatenate([synth.draw_samples(cfg, 400 + 10 * call + s, n)[0] for s in range(n_seg)], axis=1)
        p = torch.from_numpy(np.ascontiguousarray(params)).cuda()
        lnL = torch.full((n_seg * n,), float("nan"), dtype=torch.float64, device="cuda")
        rift.rift_ile_eval_batch(h, [0] * n_seg, n, p, lnL, None, stream)
        rng = np.random.default_rng(77 + call)
        ln_w = torch.from_numpy(rng.normal(0.0, 1.5, n_seg * n)).cuda() if weighted else None
        if call == 1:
            lnL[2 * n + 17] = float("nan")
        out = torch.full((4, n_seg), -1.0, dtype=torch.float64, device="cuda")
        torch.cuda.synchronize()
        if call == 1:
            free_before = torch.cuda.mem_get_info()[0]
        rift.rift_ile_reduce_static(n_seg, n, lnL, ln_w, out, stream)
        torch.cuda.synchronize()
        if call == 1:                                   # the second call found everything set up: no device memory moved
            assert torch.cuda.mem_get_info()[0] == free_before
        got = out.cpu().numpy()
        ref = rift.rift_ile_reduce(h, n_seg, n, lnL, ln_w, merge=0, cuda_stream=stream)
        for row, key in enumerate(("lnZ", "rel_err", "n_eff", "n_ess")):
            assert _close(got[row], ref[key]), (call, key, got[row], ref[key])
        if call == 1:
            assert np.all(np.isnan(got[:, 2])) and not np.any(np.isnan(np.delete(got, 2, axis=1)))
        # and against the oracle's own reduce, segment by segment
        l_host = lnL.cpu().numpy().reshape(n_seg, n)
        w_host = None if ln_w is None else ln_w.cpu().numpy().reshape(n_seg, n)
        for s in range(n_seg):
            if np.any(np.isnan(l_host[s])):
                continue
            rr = oracle.reduce(l_host[s], None if w_host is None else w_host[s])
            assert abs(got[0, s] - rr["lnZ"]) <= TOL_FP64_REL * max(1.0, abs(rr["lnZ"]))
            assert abs(got[2, s] - rr["n_eff"]) <= 1e-8 * abs(rr["n_eff"])
            assert abs(got[3, s] - rr["n_ess"]) <= 1e-8 * abs(rr["n_ess"])
    rift.rift_ile_destroy(h)


def test_reduce_static_rejects_sizes_beyond_the_static_array(torch):
    n_seg = rift.RIFT_REDUCE_STATIC_MAX_SEG + 1
    lnL = torch.zeros(n_seg * 4, dtype=torch.float64, device="cuda")
    out = torch.full((4, n_seg), -1.0, dtype=torch.float64, device="cuda")
    with pytest.raises(rift.RiftError) as e:
        rift.rift_ile_reduce_static(n_seg, 4, lnL, None, out)
    assert e.value.code == rift.RIFT_EINVAL and "RIFT_REDUCE_STATIC_MAX_SEG" in str(e.value)
    torch.cuda.synchronize()
    assert torch.all(out == -1.0)                      # outputs untouched on error
    # the largest accepted size works (one block per segment): lnZ of equal lnL = 0 is 0, n_eff = n_ess = N
    n_seg = rift.RIFT_REDUCE_STATIC_MAX_SEG
    lnL = torch.zeros(n_seg * 4, dtype=torch.float64, device="cuda")
    out = torch.full((4, n_seg), -1.0, dtype=torch.float64, device="cuda")
    rift.rift_ile_reduce_static(n_seg, 4, lnL, None, out)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    assert np.all(got[0] == 0.0) and np.all(got[2] == 4.0) and np.all(got[3] == 4.0) and np.all(got[1] == 0.0)
