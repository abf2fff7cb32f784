"""The parameter values the paper prints for this path (tests/golden/paper_params.txt, each with its citation) are the ones
the synthetic workloads and default solver options use."""
import os

import numpy as np

from paper_2506_14186_b200 import workloads as W

HERE = os.path.dirname(os.path.abspath(__file__))


def _golden():
    out = {}
    for line in open(os.path.join(HERE, "golden", "paper_params.txt")):
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split("=")
            out[k.strip()] = [float(x) for x in v.split()]
    return out


def test_paper_parameter_values_are_used():
    g = _golden()
    o = W.default_opts()
    assert o["pcoeff"] == g["pid_pcoeff"][0] and o["icoeff"] == g["pid_icoeff"][0]
    assert o["h0"] == g["default_timestep"][0]
    assert list(W.SOLIMP_DEFAULT) == g["solimp_gradient_study"]
    assert list(W.SOLIMP_CFD) == g["solimp_cfd_mpc"]
    assert list(W.SOLIMP_CFD_SMOOTH) == g["solimp_cfd_sysid"]
    for cfg in W.CONFIGS:
        w = W.make(cfg, nenv=2)
        m = w["model"]
        assert m["newton_iters"] == g["newton_iterations"][0] and m["ls_iters"] == g["newton_ls_iterations"][0]
        assert w["opts"]["pcoeff"] == 0.2 and w["opts"]["icoeff"] == 0.4
    c2 = W.make("C2", nenv=2)["model"]
    assert np.allclose(c2["pair_solimp"].reshape(-1, 5)[:, 0], 0.1)            # CFD needs d_o = d_0 > 0
    assert np.allclose(c2["pair_solimp_cfd"].reshape(-1, 5), g["solimp_cfd_mpc"])
    c4 = W.make("C4", nenv=2)["model"]
    assert np.allclose(c4["pair_solimp"].reshape(-1, 5), g["solimp_gradient_study"])
    assert np.allclose(c4["pair_solimp_cfd"].reshape(-1, 5), g["solimp_cfd_sysid"])


def test_seeded_inputs_are_reproducible_and_counter_based():
    a, b = W.make("C3", nenv=16), W.make("C3", nenv=64)
    assert np.array_equal(a["x0"][:, 7:], a["x0"][:, 7:]) and a["x0"].shape == (16, 13)
    r1, r2 = W.SplitMix64(7), W.SplitMix64(7)
    u = r1.uniform(10)
    assert np.array_equal(u[:4], r2.uniform(4)) and np.array_equal(u[4:], r2.uniform(6))
    assert np.allclose(np.linalg.norm(b["x0"][:, 3:7], axis=1), 1.0)
