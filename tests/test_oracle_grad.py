"""Pins P7, P8, P12: oracle gradients vs central finite differences, CFD invariants."""
import numpy as np
import pytest

import helpers as H
from paper_2506_14186_b200 import workloads as W


def fd_vjp_field(orc, q, v, u, p, kappa, cfd, eps=1e-6):
    """kappa^T dF/d(q,v,u,p) by central differences of the oracle's vector field."""
    nq, nv = orc.nq, orc.nv
    x = np.concatenate([q, v])
    F = lambda x_, u_, p_: orc.vector_field(x_[:nq], x_[nq:], u_, p_, cfd)[0] @ kappa
    gx = np.array([(F(H.perturb_x(orc, x, d, eps), u, p) - F(H.perturb_x(orc, x, d, -eps), u, p)) / (2 * eps) for d in range(2 * nv)])
    gu = np.zeros(orc.nu)
    for i in range(orc.nu):
        e = np.zeros(orc.nu); e[i] = eps
        gu[i] = (F(x, u + e, p) - F(x, u - e, p)) / (2 * eps)
    gp = np.zeros(len(p))
    for i in range(len(p)):
        e = np.zeros(len(p)); e[i] = 1e-6 * max(1e-2, abs(p[i]))
        gp[i] = (F(x, u, p + e) - F(x, u, p - e)) / (2 * e[i])
    return gx[:nv], gx[nv:], gu, gp


def _contact_state(name, rng):
    """A configuration with several active contacts and generic velocities."""
    if name == "box":
        model = H.free_box(gravity=(0, 0, -9.81), with_plane=True, solimp=(0.1, 0.9, 0.01, 0.4, 2.5))
        q = np.concatenate([[0.1, 0.2, 0.075], H.rand_quat(rng) * 0 + np.array([0.98, 0.12, -0.1, 0.05])]); q[3:] /= np.linalg.norm(q[3:])
        return model, q, rng.normal(size=6), None
    if name == "arm":
        model = H.arm(3, with_contacts=True)
        return model, None, rng.normal(size=3), rng.normal(size=3)       # q searched below
    if name == "C2":
        w = W.make("C2", nenv=1); model = w["model"]
        q = w["x0"][0, :9].copy(); a = q[0] + q[1]
        tip = 0.3 * np.array([np.cos(q[0]), np.sin(q[0])]) + 0.3 * np.array([np.cos(a), np.sin(a)])
        q[2:4] = tip + 0.0695 * np.array([np.cos(a + 0.3), np.sin(a + 0.3)]); q[4] = 0.0496; q[5:9] = H.rand_quat(rng)
        return model, q, rng.normal(size=8), rng.normal(size=2)
    if name == "C5":
        w = W.make("C5", nenv=1); model = w["model"]
        q = w["x0"][0, :19].copy(); q[2] = 0.322; q[3:7] = np.array([0.995, 0.05, -0.06, 0.03]); q[3:7] /= np.linalg.norm(q[3:7])
        return model, q, rng.normal(size=18) * 0.5, q[7:19] + 0.1 * rng.normal(size=12)
    raise KeyError(name)


@pytest.mark.parametrize("name", ["box", "arm", "C2", "C5"])
@pytest.mark.parametrize("cfd", [False, True])
def test_P7_vjp_of_vector_field_vs_fd(oracle_mod, name, cfd):
    rng = np.random.default_rng(31)
    model, q, v, u = _contact_state(name, rng)
    model = dict(model); model["newton_iters"] = 30      # random (inconsistent) states need more than 4 iterations
    orc = oracle_mod.Oracle(model)
    u = np.zeros(max(orc.nu, 1)) if u is None else u
    p = orc.default_params()
    for _ in range(2000 if q is None else 0):           # arm: draw joint angles until link caps touch the plane
        qq = rng.uniform(-3, 3, size=orc.nq)
        if orc.vector_field(qq, v, u, p, False)[1] >= 4:
            q = qq
            break
    acc, nr, conv = orc.vector_field(q, v, u, p, cfd)
    assert nr >= 4 and conv, (nr, conv)
    kappa = rng.normal(size=orc.nv)
    qb, vb, ub, pb = orc.vjp_field(q, v, u, p, kappa, cfd)
    fq, fv, fu, fp = fd_vjp_field(orc, q, v, u[: orc.nu] if orc.nu else u, p, kappa, cfd)
    sc = max(1.0, np.abs(fq).max())
    assert np.abs(qb - fq).max() < 1e-5 * sc, (qb, fq)
    assert np.abs(vb - fv).max() < 2e-6 * max(1.0, np.abs(fv).max())
    if orc.nu:
        assert np.abs(ub - fu).max() < 1e-5 * sc
    # parameters: mass, friction, solref, solimp (body 0 is the world: no effect)
    assert np.abs(pb - fp).max() < 5e-5 * max(1.0, np.abs(fp).max()), (pb, fp)
    assert np.abs(fp[orc.nbody:]).max() > 0          # contact parameters matter in these states


def _frozen_fd(orc, w, x0, ctrl, p, hs, lamT, nknot, knot_dt, T, eps=1e-7):
    """Central differences of lamT . xT(x0, ctrl, p) with the recorded step-size schedule replayed."""
    nq, nv = orc.nq, orc.nv
    f = lambda x_, c_, p_: orc.rollout(x_[None], None if c_ is None else c_[None], nknot, knot_dt, p_[None], T, w["opts"], h_replay=hs)["xT"][0] @ lamT
    gx = np.array([(f(H.perturb_x(orc, x0, d, eps), ctrl, p) - f(H.perturb_x(orc, x0, d, -eps), ctrl, p)) / (2 * eps) for d in range(2 * nv)])
    gc = None
    if ctrl is not None:
        gc = np.zeros_like(ctrl)
        for idx in np.ndindex(*ctrl.shape):
            e = np.zeros_like(ctrl); e[idx] = eps
            gc[idx] = (f(x0, ctrl + e, p) - f(x0, ctrl - e, p)) / (2 * eps)
    gp = np.zeros_like(p)
    for i in range(len(p)):
        e = np.zeros_like(p); e[i] = 1e-6 * max(1e-2, abs(p[i]))
        gp[i] = (f(x0, ctrl, p + e) - f(x0, ctrl, p - e)) / (2 * e[i])
    return gx, gc, gp


def _grad_case(name):
    if name == "C1":
        w = W.ball_drop(nenv=4, horizon=0.16); return w, np.array([0.3, -1.0])      # in flight after the first bounce
    if name == "C3":
        w = W.cube_toss(nenv=4, horizon=0.12, mu=0.6); x = w["x0"][2].copy(); x[2] = 0.12; x[9] = -2.0
        w["model"]["newton_iters"] = 30; return w, x
    if name == "C2":
        w = W.planar_push(nenv=4, horizon=0.03, cfd_model=False); x = w["x0"][0].copy()
        a = x[0] + x[1]; tip = 0.3 * np.array([np.cos(x[0]), np.sin(x[0])]) + 0.3 * np.array([np.cos(a), np.sin(a)])
        # d_o = 0 here: with d_o > 0 (CFD settings) the force jumps whenever r crosses 0 (G6), the
        # frozen-step map is then discontinuous and FD is meaningless; that model is FD-checked at the VJP level above
        x[2:4] = tip + 0.0697 * np.array([np.cos(a + 0.4), np.sin(a + 0.4)]); x[4] = 0.0496; x[9:11] = [1.5, 2.0]
        w["model"]["newton_iters"] = 30; return w, x
    if name == "C5":
        w = W.quadruped(nenv=2, horizon=0.05); return w, w["x0"][1].copy()
    raise KeyError(name)


@pytest.mark.parametrize("name", ["C1", "C3", "C2", "C5"])
def test_P7a_rollout_gradient_vs_frozen_schedule_fd(oracle_mod, name):
    w, x0 = _grad_case(name)
    orc = oracle_mod.Oracle(w["model"])
    T, nknot, knot_dt = w["horizon"], w["nknot"], w["knot_dt"]
    ctrl = None if w["ctrl"] is None else w["ctrl"][0].copy()
    p = orc.default_params()
    fwd = orc.rollout(x0[None], None if ctrl is None else ctrl[None], nknot, knot_dt, p[None], T, w["opts"], n_hout=4096)
    st = fwd["stats"]
    assert st["status"][0] == 0 and st["n_newton_unconverged"][0] == 0
    n = st["n_accept"][0]; hs = fwd["h"][:, :n].copy()
    assert st["n_feval"][0] > 7 * 10 and (name in ("C5",) or st["n_reject"][0] > 0)
    rng = np.random.default_rng(41)
    lamT_amb = rng.normal(size=orc.nq + orc.nv)
    g = orc.rollout_grad(x0[None], None if ctrl is None else ctrl[None], nknot, knot_dt, p[None], T, w["opts"],
                         dLdxT=lamT_amb[None], h_replay=hs)
    assert np.array_equal(g["xT"], orc.rollout(x0[None], None if ctrl is None else ctrl[None], nknot, knot_dt, p[None], T, w["opts"], h_replay=hs)["xT"])
    assert np.abs(g["xT"] - fwd["xT"]).max() < 1e-14         # replay reproduces the free-running trajectory
    # the free-running gradient equals the replayed one (h frozen in the backward pass, G15)
    g_free = orc.rollout_grad(x0[None], None if ctrl is None else ctrl[None], nknot, knot_dt, p[None], T, w["opts"], dLdxT=lamT_amb[None])
    assert np.allclose(g_free["dLdx0"], g["dLdx0"], rtol=1e-12, atol=1e-14)
    # FD of the replayed map; ambient cotangent is constant, so use lamT . xT directly
    if ctrl is not None and ctrl.size > 40:
        ctrl_fd_idx = [(0, 0), (ctrl.shape[0] // 2, ctrl.shape[1] - 1), (ctrl.shape[0] - 1, 0)]
    else:
        ctrl_fd_idx = None
    gx = gc = gp = None
    if ctrl_fd_idx is None:
        gx, gc, gp = _frozen_fd(orc, w, x0, ctrl, p, hs, lamT_amb, nknot, knot_dt, T)
    else:               # large control arrays: FD on a few knots only
        f = lambda x_, c_, p_: orc.rollout(x_[None], c_[None], nknot, knot_dt, p_[None], T, w["opts"], h_replay=hs)["xT"][0] @ lamT_amb
        eps = 1e-7
        gx = np.array([(f(H.perturb_x(orc, x0, d, eps), ctrl, p) - f(H.perturb_x(orc, x0, d, -eps), ctrl, p)) / (2 * eps) for d in range(2 * orc.nv)])
        for idx in ctrl_fd_idx:
            e = np.zeros_like(ctrl); e[idx] = eps
            fd = (f(x0, ctrl + e, p) - f(x0, ctrl - e, p)) / (2 * eps)
            assert abs(g["dLdctrl"][0][idx] - fd) < 3e-5 * max(1.0, abs(fd)), (idx, g["dLdctrl"][0][idx], fd)
        gp = np.zeros_like(p)
        for i in range(len(p)):
            e = np.zeros_like(p); e[i] = 1e-6 * max(1e-2, abs(p[i]))
            gp[i] = (f(x0, ctrl, p + e) - f(x0, ctrl, p - e)) / (2 * e[i])
    if gc is not None:
        assert np.abs(g["dLdctrl"][0] - gc).max() < 3e-5 * max(1.0, np.abs(gc).max())
    assert np.abs(g["dLdx0"][0] - gx).max() < 3e-5 * max(1.0, np.abs(gx).max()), (g["dLdx0"][0], gx)
    assert np.abs(g["dLdparams"][0] - gp).max() < 1e-4 * max(1.0, np.abs(gp).max()), (g["dLdparams"][0], gp)
    assert np.abs(gx).max() > 1e-3


def test_P7b_free_running_fd_at_tight_tolerance(oracle_mod):
    """PAPER.md:347 ground-truth recipe: FD of an adaptive rollout at very low tolerance (continuous onset, d_o=0)."""
    w = W.ball_drop(nenv=1, horizon=0.3, gravity=0.0)      # shape of Fig. 20: no gravity, downward velocity
    orc = oracle_mod.Oracle(w["model"])
    x0 = np.array([0.3, -2.0])
    tight = W.default_opts(W.DOPRI5, 1e-12, 1e-12)
    f = lambda x: orc.rollout(x[None], None, 0, 0.0, None, 0.3, tight)["xT"][0, 0]
    eps = 1e-5
    fd = np.array([(f(x0 + [eps, 0]) - f(x0 - [eps, 0])) / (2 * eps), (f(x0 + [0, eps]) - f(x0 - [0, eps])) / (2 * eps)])
    errs = []
    for tol in (1e-6, 1e-9, 1e-11):
        g = orc.rollout_grad(x0[None], None, 0, 0.0, None, 0.3, W.default_opts(W.DOPRI5, tol, tol), loss_grad=w["loss_grad"])
        errs.append(np.abs(g["dLdx0"][0] - fd).max() / np.abs(fd).max())
    assert np.abs(fd).max() > 0.05
    # The frozen-step adjoint is the exact derivative of the discrete map (P7a) and approaches the continuous
    # gradient as the tolerance tightens — slowly and not monotonically, because the impedance
    # spline makes F only C^1 at contact onset (measured: 3e-1, 7e-3, 3e-3 relative at these tolerances).
    assert errs[0] < 1.0 and errs[1] < 5e-2 and errs[2] < 1e-2 and errs[2] < errs[0], errs


def test_P8_cfd_changes_gradients_but_not_forward_states(oracle_mod):
    """straight-through CFD leaves the rollout untouched; a miss has zero plain gradient."""
    model = H.two_spheres()
    orc = oracle_mod.Oracle(model)
    opts = W.default_opts(W.TSIT5, 1e-8, 1e-8)
    # ball A shot along +x, ball B offset so that they MISS by 2 cm (gap to surfaces)
    x0 = np.zeros(26); x0[3] = 1.0; x0[10] = 1.0
    x0[7:10] = [0.3, 0.08, 0.0]; x0[14] = 1.0
    lam = np.zeros(26); lam[7] = 1.0                      # loss = x of ball B
    g0 = orc.rollout_grad(x0[None], None, 0, 0.0, None, 0.5, opts, dLdxT=lam[None], cfd_on=False)
    g1 = orc.rollout_grad(x0[None], None, 0, 0.0, None, 0.5, opts, dLdxT=lam[None], cfd_on=True)
    assert np.array_equal(g0["xT"], g1["xT"])
    for k in ("n_accept", "n_reject", "n_feval", "status", "h_min", "h_max", "t_end"):
        assert np.array_equal(g0["stats"][k], g1["stats"][k])
    assert abs(g0["xT"][0, 7] - 0.3) < 1e-15              # B never moved
    assert g0["dLdx0"][0, 12 + 0] == 0.0                   # no contact -> zero gradient w.r.t. A's velocity
    assert g1["dLdx0"][0, 12 + 0] > 1e-6                   # CFD: pushing A harder towards B moves B forward
    # w_c -> 0 recovers the plain gradients on a trajectory WITH contact.  Head-on and starting
    # in slight penetration: with d_o > 0 an r=0 crossing under load is a force jump (G6) around which the
    # stepper takes ~1e-9 steps, so stages would land inside the (0, w_c) band however small w_c is.
    x1 = x0.copy(); x1[7:10] = [0.0595, 0.0, 0.0]
    gc0 = orc.rollout_grad(x1[None], None, 0, 0.0, None, 0.5, opts, dLdxT=lam[None], cfd_on=False)
    assert gc0["xT"][0, 7] > 0.1 and abs(gc0["dLdx0"][0, 12]) > 1e-3
    prev = None
    for wc in (1e-2, 1e-4, 1e-6):
        m2 = dict(model); m2["pair_solimp_cfd"] = np.array([0.0, 0.1, wc, 1.0, 4.0]); m2["pair_cfd_beta"] = np.array([10.0 / wc])
        o2 = oracle_mod.Oracle(m2)
        gc1 = o2.rollout_grad(x1[None], None, 0, 0.0, None, 0.5, opts, dLdxT=lam[None], cfd_on=True)
        err = np.abs(gc1["dLdx0"] - gc0["dLdx0"]).max() / np.abs(gc0["dLdx0"]).max()
        assert np.array_equal(gc1["xT"], gc0["xT"])
        assert prev is None or err <= prev
        prev = err
    assert prev < 1e-3


def test_P12_batch_independence(oracle_mod):
    w = W.make("C3", nenv=6, horizon=0.6)
    orc = oracle_mod.Oracle(w["model"])
    full = orc.rollout(w["x0"], None, 0, 0.0, None, 0.6, w["opts"])
    perm = np.array([4, 1, 5, 0])
    part = orc.rollout(w["x0"][perm], None, 0, 0.0, None, 0.6, w["opts"], threads=2)
    assert np.array_equal(part["xT"], full["xT"][perm])
    assert np.array_equal(part["stats"]["n_accept"], full["stats"]["n_accept"][perm])
    assert len(set(full["stats"]["n_accept"].tolist())) > 1      # step sizes are per environment


def test_unconverged_newton_gradient_is_flagged_and_quantified(oracle_mod):
    """Reading G9 (PAPER.md:68, 515, 539 fixed iteration counts; PAPER.md:543 implicit differentiation): the VJP is the
    implicit-function gradient at the final active set, which is the gradient of the computed F only when the fixed
    budget of Newton iterations ended on a full step inside an unchanged active set.  Otherwise the evaluation is counted
    (n_newton_unconverged, n_newton_unconverged_bwd) and this test quantifies what the count means, on a state of the
    BASELINE workload itself: C3 environment 2022 lands flat on a face at t = 0.5145 s (16 rows), where 4 iterations
    are not enough.  Measured there: F differs from the converged solution by 0.8 %; the implicit gradient differs from
    central differences of the 4-iteration map by 7.5 % (and that map is discontinuous: on neighbouring states of the same
    impact the difference quotient grows without bound as eps -> 0) and from the converged gradient by 21 %; with 50
    iterations the solve converges and the implicit gradient equals central differences to 1e-7.  The same environment
    takes 11 007 accepted steps with the 4-iteration budget and 450 with 8 iterations (step size collapses to 2e-8 s while
    F is noisy): DESIGN.md section 5."""
    w = W.make("C3")                               # the draws of an environment depend on the batch size: BASELINE batch
    x0 = w["x0"][2022:2023]
    orc = oracle_mod.Oracle(w["model"])
    r = orc.rollout(x0, None, 0, 0.0, None, 0.5145, w["opts"])
    assert r["stats"]["status"][0] == 0 and r["stats"]["n_newton_unconverged"][0] > 0        # the forward pass counts it
    x = r["xT"][0]; q, v = x[:7], x[7:]
    p = orc.default_params()
    a4, nr, conv = orc.vector_field(q, v, None, p, False)
    assert nr == 16 and not conv
    kap = np.random.default_rng(0).normal(size=6)
    g4 = np.concatenate(orc.vjp_field(q, v, None, p, kap, False)[:2])
    fd4 = np.concatenate(fd_vjp_field(orc, q, v, None, p, kap, False, eps=1e-7)[:2])
    e4 = np.abs(g4 - fd4).max() / np.abs(fd4).max()
    mdl = dict(w["model"]); mdl["newton_iters"] = 50
    o50 = oracle_mod.Oracle(mdl)
    a50, _, conv50 = o50.vector_field(q, v, None, p, False)
    g50 = np.concatenate(o50.vjp_field(q, v, None, p, kap, False)[:2])
    fd50 = np.concatenate(fd_vjp_field(o50, q, v, None, p, kap, False, eps=1e-7)[:2])
    e50 = np.abs(g50 - fd50).max() / np.abs(fd50).max()
    print("unconverged state: |F4-F50|/|F50| = %.2e, implicit gradient vs FD of the 4-iteration map %.2e, vs converged gradient %.2e; "
          "50 iterations: vs FD %.2e" % (np.abs(a4 - a50).max() / np.abs(a50).max(), e4, np.abs(g4 - g50).max() / np.abs(g50).max(), e50))
    assert conv50 and e50 < 1e-5
    assert 1e-3 < e4 < 1.0                         # a real discrepancy, of the size recorded above
    assert 1e-4 < np.abs(a4 - a50).max() / np.abs(a50).max() < 0.1
