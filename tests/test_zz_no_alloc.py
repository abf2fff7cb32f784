"""dmx_rollout_backward_noalloc (include/dmx.h): the reverse sweep with its scratch in a static device array, for callers
that must not allocate at call time.  Collected last on purpose (the suite runs with pytest -x).  Runs alone in a fresh
process and after the other tests: it builds its own model and depends on no state they leave."""
import numpy as np
import pytest

from paper_2506_14186_b200 import workloads as W

pytestmark = pytest.mark.gpu


def test_noalloc_reverse_sweep_matches_the_regular_path_on_two_calls_in_a_row():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2506_14186_b200 import binding as B
    L = B.load()
    limit = int(L.dmx_noalloc_scratch_bytes())
    assert limit == 16 << 20
    w = W.make("C2", nenv=300, horizon=0.2)
    nenv = w["nenv"]
    m = B.Model(w["model"])
    x0, ctrl = m.dev(w["x0"]), m.dev(w["ctrl"])
    st = m.alloc_stats(nenv)
    tape = m.alloc_tape(nenv, 400)
    xT = m.rollout(x0, ctrl, w["nknot"], w["knot_dt"], None, w["horizon"], w["opts"], stats=st, tape=tape)
    assert (st["status"] == 0).all()
    rng = np.random.default_rng(3)
    mk = lambda: dict(dLdx0=torch.full((nenv, 2 * m.nv), float("nan"), dtype=m.dtype, device=m.device),
                      dLdctrl=torch.full_like(ctrl, float("nan")),
                      dLdparams=torch.full((nenv, m.np_), float("nan"), dtype=m.dtype, device=m.device))
    for call, cfd in enumerate((True, False)):              # two calls in a row; the second sees the first one's leftovers
        g = m.dev(rng.normal(size=w["x0"].shape))
        ref = m.rollout_backward(ctrl, w["nknot"], None, w["opts"], xT, g, cfd, tape, want_params=True)
        torch.cuda.synchronize()
        before = torch.cuda.memory_allocated()
        out = m.rollout_backward_noalloc(ctrl, w["nknot"], None, w["opts"], xT, g, cfd, tape, mk() if call == 0 else out)
        torch.cuda.synchronize()
        if call == 1:
            assert torch.cuda.memory_allocated() == before   # the wrapper reused `out`: nothing was allocated through torch either
        for k in ("dLdx0", "dLdctrl", "dLdparams"):
            a, b = out[k].cpu().numpy().reshape(nenv, -1), ref[k].cpu().numpy().reshape(nenv, -1)
            assert np.isfinite(a).all(), k
            scale = np.maximum(np.abs(b).max(axis=1), 1e-300)
            assert (np.abs(a - b).max(axis=1) / scale).max() <= 1e-6, (call, k)      # the fp64 gradient tolerance of the parity tests
            assert np.array_equal(a, b), (call, k)           # same kernel, same order of operations: in fact bit-identical
        assert float(out["dLdctrl"].abs().max()) > 0
    # a batch whose scratch need exceeds the static array is rejected with a clear error, before anything is launched
    wb = W.make("C2", nenv=8192, horizon=0.004)       # 4736 resident lane groups x 4240 B = 20.1 MB > 16 MiB
    xb, cb = m.dev(wb["x0"]), m.dev(wb["ctrl"])
    tb = m.alloc_tape(8192, 8)
    xTb = m.rollout(xb, cb, wb["nknot"], wb["knot_dt"], None, wb["horizon"], wb["opts"], tape=tb)
    big = dict(dLdx0=torch.zeros((8192, 2 * m.nv), dtype=m.dtype, device=m.device), dLdctrl=torch.zeros_like(cb), dLdparams=None)
    with pytest.raises(RuntimeError, match="DMX_NOALLOC_SCRATCH_BYTES"):
        m.rollout_backward_noalloc(cb, wb["nknot"], None, wb["opts"], xTb, torch.ones_like(xb), True, tb, big)
    ok = m.rollout_backward(cb, wb["nknot"], None, wb["opts"], xTb, torch.ones_like(xb), True, tb, want_params=False)   # the regular path takes it
    assert bool(torch.isfinite(ok["dLdx0"]).all())
