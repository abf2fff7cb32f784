"""Pins of the optimize-then-discretize gradient (oracle/adjoint.hpp; Eq. 6-7, 462-477 Eq. 8-9; DESIGN.md
reading G21): closed form on a linear ODE, agreement with the discrete adjoint as the tolerances go to zero, accuracy at
loose tolerance against finite differences of a tight rollout, and the shape of PAPER.md Fig. 19 (reduced billiard: with
CFD and a non-stiff forward solve the unrolled gradient is garbage whatever the forward tolerance, the continuous one is
smooth)."""
import numpy as np
import pytest

import helpers as H
from paper_2506_14186_b200 import workloads as W


def test_linear_ode_closed_form(oracle_mod):
    """m q'' = kp (u - q): a_x(0) = Phi(T)^T a_x(T) with the transition matrix of the oscillator, and
    dL/du = a_x(T)^T int_0^T Phi(T - s) B ds = a_x(T)^T A^-1 (Phi(T) - I) B, B = (0, kp/m)."""
    m, kp = 0.9, 11.0
    orc = oracle_mod.Oracle(H.oscillator(m, kp))
    om = np.sqrt(kp / m); T = 1.3
    Phi = np.array([[np.cos(om * T), np.sin(om * T) / om], [-om * np.sin(om * T), np.cos(om * T)]])
    A = np.array([[0.0, 1.0], [-kp / m, 0.0]]); Bv = np.array([0.0, kp / m])
    lamT = np.array([0.3, -1.1]); x0 = np.array([[0.5, 0.2]])
    want_x, want_u = Phi.T @ lamT, lamT @ (np.linalg.inv(A) @ (Phi - np.eye(2)) @ Bv)
    errs = []
    for which in (W.DOPRI5, W.TSIT5):
        for tol in (1e-6, 1e-9, 1e-11):
            o = W.default_opts(which, tol, tol)
            g = orc.rollout_grad_adjoint(x0, np.zeros((1, 1, 1)), 1, 10.0, None, T, o, o, lamT[None])
            assert g["adj_status"][0] == 0 and g["adj_accept"][0] > 0
            e = max(np.abs(g["dLdx0"][0] - want_x).max(), abs(g["dLdctrl"][0, 0, 0] - want_u))
            errs.append(e)
            assert e < 0.2 * tol ** 0.9 + 1e-12, (which, tol, e)          # measured 5e-8, 7e-11, 8e-13 (Tsit5)
    # the adjoint's own tolerance controls the gradient error (here dF/dx is constant, so the loosely solved forward
    # trajectory does not enter at all): loose forward solve, loose / tight backward solve
    of = W.default_opts(W.TSIT5, 1e-4, 1e-4)
    e = [np.abs(orc.rollout_grad_adjoint(x0, np.zeros((1, 1, 1)), 1, 10.0, None, T, of, W.default_opts(W.TSIT5, t, t), lamT[None])["dLdx0"][0] - want_x).max()
         for t in (1e-4, 1e-10)]
    assert e[1] < 1e-3 * e[0] and e[1] < 1e-9, e


def test_agrees_with_the_discrete_adjoint_as_tolerances_shrink(oracle_mod):
    """Smooth problem (passive arm with gravity, slide joint and oblique axes, no contact): both gradients converge to the
    same limit, difference proportional to the tolerance."""
    orc = oracle_mod.Oracle(H.arm(3, slide_last=True))
    rng = np.random.default_rng(4)
    x0 = np.concatenate([rng.uniform(-1, 1, 3), rng.normal(size=3)])[None]
    ctrl = rng.normal(size=(1, 2, 3)); g = rng.normal(size=(1, 6))
    diff = []
    for tol in (1e-5, 1e-7, 1e-9):
        o = W.default_opts(W.TSIT5, tol, tol)
        a = orc.rollout_grad_adjoint(x0, ctrl, 2, 0.25, None, 0.5, o, o, g)
        d = orc.rollout_grad(x0, ctrl, 2, 0.25, None, 0.5, o, dLdxT=g)
        assert a["adj_status"][0] == 0
        diff.append(max(np.abs(a[k] - d[k]).max() / np.abs(d[k]).max() for k in ("dLdx0", "dLdctrl", "dLdparams")))
    print("arm: |continuous - discrete| relative at tol 1e-5, 1e-7, 1e-9:", diff)
    assert diff[0] < 1e-3 and diff[1] < 3e-5 and diff[2] < 1e-6 and diff[2] < 1e-2 * diff[0]     # measured 2.9e-4, 6.7e-6, 1.6e-7


def test_contact_problem_gradient_error_follows_the_adjoint_tolerance(oracle_mod):
    """Box toss with friction (contacts, active-set switches).  Reference: central differences of a rollout at rtol 1e-11
    (the paper's recipe).  Measured relative error against it, at solver tolerance 1e-5 / 1e-7 / 1e-9:
    continuous adjoint 6.2 % / 6.7 % / 6.7 % (already at its limit), unrolled 24.7 % / 15.3 % / 6.7 %: the two share their
    limit, and the backward solve reaches it at loose tolerance ("allows to directly specify tolerances on the error in
    the gradients").  The common 6.7 % is the distance between the implicit-function gradient of reading G9
    and a difference quotient across active-set switches."""
    orc = oracle_mod.Oracle(H.free_box(gravity=(0, 0, -9.81), with_plane=True))
    rng = np.random.default_rng(1)
    x0 = np.zeros((1, 13)); x0[0, :3] = [0, 0, 0.25]; x0[0, 3:7] = H.rand_quat(rng); x0[0, 7:10] = [0.5, 0.2, -1.0]; x0[0, 10:] = rng.normal(size=3)
    g = rng.normal(size=(1, 13)); T = 0.3
    ot = W.default_opts(W.TSIT5, 1e-11, 1e-11)
    L = lambda x: orc.rollout(x[None], None, 0, 0.0, None, T, ot)["xT"][0] @ g[0]
    fd = np.array([(L(H.perturb_x(orc, x0[0], d, 1e-6)) - L(H.perturb_x(orc, x0[0], d, -1e-6))) / 2e-6 for d in range(12)])
    ea, ed, dd = [], [], []
    for tol in (1e-5, 1e-9):
        o = W.default_opts(W.TSIT5, tol, tol)
        a = orc.rollout_grad_adjoint(x0, None, 0, 0.0, None, T, o, o, g)
        d = orc.rollout_grad(x0, None, 0, 0.0, None, T, o, dLdxT=g)
        assert a["adj_status"][0] == 0
        ea.append(np.abs(a["dLdx0"][0] - fd).max() / np.abs(fd).max()); ed.append(np.abs(d["dLdx0"][0] - fd).max() / np.abs(fd).max())
        dd.append(np.abs(a["dLdx0"] - d["dLdx0"]).max() / np.abs(d["dLdx0"]).max())
    print("box: vs FD continuous", ea, "unrolled", ed, "continuous vs unrolled", dd)
    assert ea[0] < 0.1 and ea[1] < 0.1 and ed[0] > 2 * ea[0]        # loose tolerance: the backward solve is already accurate
    assert dd[1] < 0.25 * dd[0] and dd[1] < 0.06                     # and the two approach each other


def test_reduced_billiard_shape_of_fig_19(oracle_mod):
    """PAPER.md:452, 473-475 (Fig. 19): two spheres, no gravity, no table; ball a passes ball b at lateral offsets that MISS
    it; L = x of ball b at T; dL/d(offset) with CFD.  The forward ODE is free flight, integrated exactly in 4-5 steps
    whatever its tolerance; the CFD adjoint is stiff over the passage, so the unrolled gradient is garbage (1e2 ... 4e4
    with sign changes, here) - "this phenomenon persists no matter how low the tolerance of the forward ODE solver is set" -
    while the continuous adjoint, with its own steps, is smooth, negative and decays monotonically with the offset
    (-79 ... -7.6) and does not depend on its tolerance."""
    model = H.two_spheres()
    orc = oracle_mod.Oracle(model)
    offs = np.linspace(0.062, 0.16, 25); n = len(offs)
    x0 = np.zeros((n, 26)); x0[:, :14] = model["qpos0"]; x0[:, 1] = offs; x0[:, 14] = 1.0
    g = np.zeros((n, 26)); g[:, 7] = 1.0
    T = 0.6
    rough = lambda y: np.abs(np.diff(y, 2)).sum() / np.abs(y).max()
    res = {}
    for ftol in (1e-6, 1e-10):
        of = W.default_opts(W.TSIT5, ftol, ftol, h0=2e-3)
        d = orc.rollout_grad(x0, None, 0, 0.0, None, T, of, dLdxT=g, cfd_on=True, threads=4)
        assert d["stats"]["n_accept"].max() <= 8                         # non-stiff forward solve: a handful of steps
        res["disc", ftol] = d["dLdx0"][:, 1]
        assert rough(res["disc", ftol]) > 1.0 and (np.sign(res["disc", ftol]) > 0).any() and (np.sign(res["disc", ftol]) < 0).any()
    of = W.default_opts(W.TSIT5, 1e-6, 1e-6, h0=2e-3)
    xT_plain = orc.rollout(x0, None, 0, 0.0, None, T, of, threads=4)["xT"]
    for atol in (1e-4, 1e-6):
        a = orc.rollout_grad_adjoint(x0, None, 0, 0.0, None, T, of, W.default_opts(W.TSIT5, atol, 1e-9), g, cfd_on=True, threads=4)
        assert (a["adj_status"] == 0).all() and a["adj_accept"].min() > 20   # the backward solve takes its own (many more) steps
        res["cont", atol] = a["dLdx0"][:, 1]
        assert np.array_equal(a["xT"], xT_plain)                             # CFD and the adjoint mode never touch the forward pass
    c = res["cont", 1e-6]
    print("Fig. 19 shape: continuous", np.array2string(c[::4], precision=3), "roughness", rough(c), "| unrolled", np.array2string(res["disc", 1e-6][::4], precision=3),
          "roughness", rough(res["disc", 1e-6]))
    assert (c < 0).all() and (np.diff(c) > 0).all() and rough(c) < 0.15
    assert np.abs(res["cont", 1e-4] - c).max() < 5e-3 * np.abs(c).max()
    # without CFD a miss has no gradient at all
    a0 = orc.rollout_grad_adjoint(x0, None, 0, 0.0, None, T, of, of, g, cfd_on=False, threads=4)
    assert np.abs(a0["dLdx0"][:, 1]).max() == 0.0
