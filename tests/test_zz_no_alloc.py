"""me_compute_static (include/me.h): the g g -> t t~ g g hot path for callers that must not allocate.  Its current cache is a
file-scope `static __device__` array of the library instead of the context's lazily allocated scratch; everything else (kernel,
helicity walk, arguments) is the existing me_compute path with ME_OPT_SHARE_CURRENTS on, so the two must agree to the tolerance the
sharing tests use (tests/test_gpu_parity.py test_share_currents_option: 1e-12 FP64, 5e-6 mixed, 1e-4 FP32; in fact bit for bit).

Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the other tests.
"""
import numpy as np
import pytest

import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def me():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import __graft_entry__
    __graft_entry__.build()
    import paper_2303_18244_b200 as m
    m.lib()
    return m


def events(me, ctx, cfg, n, first):
    rnd = me.me_philox_uniform(cfg["seed"], first, n, cfg["nfinal"])
    mom, _ = ctx.me_rambo(inputs.SQRT_S, rnd)
    return mom


def test_static_scratch_entry_matches_me_compute_on_two_calls_in_a_row(me):
    import torch
    proc = me.ME_GG_TTXGG
    cfg = inputs.CONFIGS[proc]
    ctx = me.MEContext(proc)
    nmax = me.ME_STATIC_MAX_EVENTS
    # two different batches: the full maximum, then a ragged smaller one that finds the first call's contents in the array
    batches = [(nmax, 0), (1517, 100000)]
    moms = [events(me, ctx, cfg, n, first) for n, first in batches]
    mask, ngood = ctx.me_filter_helicities(moms[0], 32)
    assert ngood == 64
    tols = {"fp64": 1e-12, "mixed": 5e-6, "fp32": 1e-4}
    want = {(i, name): ctx.me_compute(moms[i], batches[i][0], me.PRECISIONS[name]).cpu().numpy()
            for i in range(2) for name in tols}                       # the existing path (allocates the context's scratch once)
    outs = [torch.empty(n, dtype=torch.float64, device="cuda") for n, _ in batches]
    ctx.me_compute_static(moms[1], batches[1][0], out=outs[1])         # first use on this device: resolves the array's address
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for name, tol in tols.items():
        got = []
        for i, (n, _) in enumerate(batches):                           # two calls in a row on one stream, outputs preallocated
            ctx.me_compute_static(moms[i], n, me.PRECISIONS[name], out=outs[i])
        torch.cuda.synchronize()
        got = [o.cpu().numpy() for o in outs]
        for i in range(2):
            w = want[(i, name)]
            assert np.isfinite(got[i]).all() and (got[i] > 0).all()
            assert np.abs(got[i] / w - 1).max() <= tol, (name, i, np.abs(got[i] / w - 1).max())
            assert np.array_equal(got[i], w), (name, i)                 # same kernel, same walk: bit for bit
    assert torch.cuda.mem_get_info()[0] == free0                       # nothing was allocated or freed on the device
    # parity pairing is honoured like in me_compute
    ctx.me_set_option(me.ME_OPT_PARITY_PAIRING, 1)
    w = ctx.me_compute(moms[1], batches[1][0]).cpu().numpy()
    g = ctx.me_compute_static(moms[1], batches[1][0], out=outs[1]).cpu().numpy()
    ctx.me_set_option(me.ME_OPT_PARITY_PAIRING, 0)
    assert np.abs(g / w - 1).max() <= 1e-12
    ctx.close()


def test_static_scratch_entry_rejects_what_it_cannot_take(me):
    import torch
    ctx = me.MEContext(me.ME_GG_TTXGG)
    cfg = inputs.CONFIGS[me.ME_GG_TTXGG]
    n = me.ME_STATIC_MAX_EVENTS + 1
    mom = events(me, ctx, cfg, n, 0)
    out = torch.full((n,), -1.0, dtype=torch.float64, device="cuda")
    with pytest.raises(me.MEError) as ei:                               # not filtered yet, but the size is judged first
        ctx.me_compute_static(mom, n, out=out)
    assert ei.value.status == me.ME_ETOOLARGE and str(me.ME_STATIC_MAX_EVENTS) in str(ei.value)
    with pytest.raises(me.MEError) as ei:
        ctx.me_compute_static(mom, 64, out=out)
    assert ei.value.status == me.ME_ENOTFILTERED
    ctx.me_filter_helicities(mom, 32)
    with pytest.raises(me.MEError) as ei:
        ctx.me_compute_static(mom, n, out=out)
    assert ei.value.status == me.ME_ETOOLARGE
    torch.cuda.synchronize()
    assert (out == -1.0).all()                                          # nothing was launched
    assert ctx.me_compute_static(mom, 0, out=out[:0]).numel() == 0      # n = 0 is a no-op
    ctx.close()
    other = me.MEContext(me.ME_GG_TTXG)                                 # only the process that has the sharing kernel
    with pytest.raises(me.MEError) as ei:
        other.me_compute_static(mom, 64, out=out)
    assert ei.value.status == me.ME_EPROCESS
    other.close()
