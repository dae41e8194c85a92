"""heget_eval_me2_static -- the entry point that allocates nothing (include/heget.h) -- against the existing heget_eval_me2 path.

Collected last on purpose (pytest -x: a failure here must not hide other tests).  The scratch between the three kernels
(rows of J, row forms; eqs. 8-12) is a file-scope device array inside libheget.so; the call itself must perform no
cudaMalloc / cudaFree, so the test also watches the allocator of the device through cudaMemGetInfo."""
import numpy as np
import pytest
import torch

import paper_0909_5257_b200 as hg

pytestmark = pytest.mark.gpu

TOL64 = 1e-11                       # the tolerances of tests/test_gpu_parity.py (BASELINE.json north_star)
TOL32_MEDIAN, TOL32_MAX = 1e-5, 1e-3


def rel_err(a, b):
    return np.abs(a - b) / np.maximum(np.abs(b), 1e-300)


@pytest.mark.parametrize("precision", ["fp64", "fp32"])
@pytest.mark.parametrize("name,sqrt_s,seed,n", [("u u~ > g g g g g", 2000.0, 4, 515), ("g g > g g g g", 1500.0, 3, 1031)])
def test_static_entry_point_matches_existing_path_twice(name, sqrt_s, seed, n, precision):
    torch.cuda.set_device(0)
    # the existing path: table back end with its default colour stage, its own handle
    ref_p = hg.Process(name, sqrt_s, precision=precision, kernel="table")
    moms = [ref_p.sample_momenta(seed, n), ref_p.sample_momenta(seed + 100, n - 7)]        # two different batches, the second one smaller and ragged
    refs = [ref_p.eval_me2(m).cpu().numpy().astype(np.float64) for m in moms]

    P = hg.Process(name, sqrt_s, precision=precision, kernel="table")
    with pytest.raises(hg.HegetError):                       # not prepared: a clear error, nothing launched
        P.eval_me2_static(moms[0], torch.empty(n, dtype=P.dtype, device="cuda"))
    P.set_colour_stage("tensor")
    P.static_prepare()                                       # set-up: the only place that allocates
    nmax = P.static_max_events
    assert nmax >= n
    outs = [torch.full((m.shape[-1],), float("nan"), dtype=P.dtype, device="cuda") for m in moms]
    P.eval_me2_static(moms[1], outs[1])                      # leaves its rows in the array (and, with lazy module loading, has the kernels' code on the device)
    outs[1].fill_(float("nan"))
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for m, o in zip(moms, outs):                             # two calls in a row share the array; the second must not see the first one's leftovers
        P.eval_me2_static(m, o)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0, "device memory in use changed during heget_eval_me2_static"
    for o, ref in zip(outs, refs):
        err = rel_err(o.cpu().numpy().astype(np.float64), ref)
        assert np.all(np.isfinite(err))
        if precision == "fp64":
            assert err.max() <= TOL64, "max rel err %.3e" % err.max()
        else:
            assert np.median(err) <= TOL32_MEDIAN and err.max() <= TOL32_MAX, "median %.3e max %.3e" % (np.median(err), err.max())
    # the same batch again gives the same bits (nothing depends on what the array held)
    again = torch.empty_like(outs[0])
    P.eval_me2_static(moms[0], again)
    assert torch.equal(again, outs[0])
    # beyond the maximum: rejected with the limit in the message, output untouched
    big = torch.zeros(P.n_ext * 4 * (nmax + 1), dtype=torch.float64, device="cuda")
    sentinel = torch.full((nmax + 1,), -1.0, dtype=P.dtype, device="cuda")
    with pytest.raises(hg.HegetError) as ei:
        P.eval_me2_static(big.view(P.n_ext, 4, nmax + 1), sentinel)
    assert str(nmax) in str(ei.value)
    torch.cuda.synchronize()
    assert bool((sentinel == -1.0).all())
    # changing the colour stage undoes the preparation
    P.set_colour_stage("symmetric")
    assert P.static_max_events == 0
    with pytest.raises(hg.HegetError):
        P.eval_me2_static(moms[0], again)
