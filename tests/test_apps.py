"""the paper's applications on top of the ABI (PAPER.md:167 gradient-based MPC; :157, :515 identification).

CPU part: pins of the oracle's Adam step against what the update rule fixes.  GPU part (-m gpu): dmx_adam_step and the
MPC plan step of paper_2506_14186_b200/apps.py against oracle/apps.py, that MPC lowers the cost of the C2 pushing task, and
that the identification loop recovers the friction coefficient that generated oracle trajectories."""
import numpy as np
import pytest

from oracle import apps as OA
from oracle import oracle as oracle_mod
from paper_2506_14186_b200 import workloads as W


# ---- oracle pins (CPU) ----------------------------------------------------------------------------------------------
def test_adam_first_step_moves_by_lr_times_sign():
    """t = 1: m^ = g, v^ = g^2, so the update is lr g / (|g| + eps) whatever the magnitude of g (Kingma & Ba 2015, sec. 2.1)"""
    rng = np.random.default_rng(1)
    g = rng.normal(size=(3, 7)) * np.array([[1e-6], [1.0], [1e6]])
    x = rng.normal(size=(3, 7)); x0 = x.copy()
    m = np.zeros_like(x); v = np.zeros_like(x)
    OA.adam_step(x, g, m, v, 1, 0.01, 0.9, 0.999, 1e-12)
    assert np.allclose(x0 - x, 0.01 * np.sign(g), rtol=1e-5, atol=0)
    assert np.allclose(m, 0.1 * g) and np.allclose(v, 0.001 * g * g)


@pytest.mark.parametrize("betas", [(0.9, 0.999), (0.5, 0.9)])
def test_adam_constant_gradient_gives_a_linear_path(betas):
    """with the same gradient at every step the bias-corrected moments equal g and g^2 at every t, so x_t = x_0 - t lr g / (|g| + eps);
    without the bias correction, or with t off by one, the first steps are shorter"""
    g = np.array([[0.3, -2.0, 1e-3]]); x = np.zeros((1, 3)); m = np.zeros_like(x); v = np.zeros_like(x)
    eps, lr = 1e-8, 0.01
    for t in range(1, 21):
        OA.adam_step(x, g, m, v, t, lr, betas[0], betas[1], eps)
        assert np.allclose(x, -t * lr * g / (np.abs(g) + eps), rtol=1e-12, atol=0)


def test_adam_clips_the_row_norm_and_skips_inactive_rows():
    g = np.array([[3.0, 4.0], [0.3, 0.4], [3.0, 4.0]])                      # norms 5, 0.5, 5
    x = np.zeros((3, 2)); m = np.zeros_like(x); v = np.zeros_like(x)
    OA.adam_step(x, g, m, v, 1, 0.01, 0.9, 0.999, 1e-8, clip=1.0, active=np.array([1, 1, 0]))
    assert np.allclose(m[0], 0.1 * np.array([0.6, 0.8]))                      # scaled to norm 1
    assert np.allclose(m[1], 0.1 * g[1])                                      # below the threshold: unchanged
    assert np.all(m[2] == 0) and np.all(x[2] == 0)                            # inactive row untouched
    assert np.all(g[0] == [3.0, 4.0])                                         # the caller's gradient is not modified


# ---- CUDA path -------------------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2506_14186_b200 import binding
    binding.load()
    return binding


@pytest.mark.gpu
@pytest.mark.parametrize("precision", [64, 32])
def test_adam_kernel_matches_the_oracle(B, precision):
    import torch
    rng = np.random.default_rng(5)
    nrow, ln = 37, 45                                                         # ragged: rows are not a multiple of the warps per CTA, len > 32
    dt = torch.float64 if precision == 64 else torch.float32
    x = rng.normal(size=(nrow, ln)); m = np.zeros_like(x); v = np.zeros_like(x)
    act = (rng.uniform(size=nrow) > 0.2).astype(np.uint8)
    xd, md, vd = (torch.tensor(a, dtype=dt, device="cuda") for a in (x, m, v))
    ad = torch.tensor(act, device="cuda")
    for t in range(1, 6):
        g = rng.normal(size=(nrow, ln)) * 10.0 ** rng.integers(-3, 3, size=(nrow, 1))
        gd = torch.tensor(g, dtype=dt, device="cuda")
        OA.adam_step(x, gd.cpu().double().numpy(), m, v, t, 0.01, 0.5, 0.9, 1e-6, clip=1.0, active=act)
        B.adam_step(xd, gd, md, vd, t, 0.01, 0.5, 0.9, 1e-6, clip=1.0, active=ad)
    tol = 1e-13 if precision == 64 else 2e-5
    assert np.abs(xd.cpu().double().numpy() - x).max() < tol
    assert np.abs(md.cpu().double().numpy() - m).max() < tol
    with pytest.raises(RuntimeError):
        B.adam_step(xd, gd, md, vd, 0, 0.01)                                  # t starts at 1


def _c2_cost_np(goal):
    def cost(xT):
        e = xT[:, 2:4] - goal
        g = np.zeros_like(xT); g[:, 2:4] = 2 * e
        return (e * e).sum(1), g
    return cost


def _c2_cost_torch(goal):
    def cost(xT):
        import torch
        e = xT[:, 2:4] - goal
        g = torch.zeros_like(xT); g[:, 2:4] = 2 * e
        return (e * e).sum(1), g
    return cost


@pytest.mark.gpu
def test_mpc_plan_step_matches_the_oracle_loop(B):
    """three Adam iterations of one plan step on C2 (CFD backward): same costs, same control iterates"""
    import torch
    from paper_2506_14186_b200 import apps
    w = W.make("C2", nenv=6, horizon=0.06)
    nknot, kdt = w["nknot"], w["knot_dt"]
    orc = oracle_mod.Oracle(w["model"])
    goal = np.array([0.6, 0.0])
    bu, bc, hist, its = OA.mpc_plan_step(orc, w["x0"], w["ctrl"], nknot, kdt, w["opts"], _c2_cost_np(goal), cfd=True, iters=3, lr=0.01, clip=1.0, threads=6)
    m = B.Model(w["model"], precision=64)
    mpc = apps.MPC(m, 6, nknot, kdt, w["opts"], _c2_cost_torch(torch.tensor(goal, device="cuda")), cfd=True, iters=3, lr=0.01, clip=1.0)
    gu, gc, ghist = mpc.plan_step(m.dev(w["x0"]), m.dev(w["ctrl"]))
    assert np.abs(ghist.cpu().numpy() - hist).max() < 1e-8 * max(1.0, np.abs(hist).max())
    assert np.abs(gc.cpu().numpy() - bc).max() < 1e-8
    # Adam divides by sqrt(v^): a control knot whose gradient is ~0 amplifies rounding, so compare in units of lr
    assert np.abs(gu.cpu().numpy() - bu).max() < 1e-4 * 0.01


def _push_task(nenv, horizon):
    """C2 with the sphere placed next to the finger tip (2 mm gap) and, per environment, a goal 0.15 m further along the
    tip -> sphere direction: a push the finger can perform.  (With the workload's fixed goal most spheres would have to be
    pulled, and the CFD gradient rightly steers the finger away.)"""
    w = W.make("C2", nenv=nenv, horizon=horizon)
    x0 = w["x0"].copy(); L = 0.3
    th1, a12 = x0[:, 0], x0[:, 0] + x0[:, 1]
    tip = np.stack([L * np.cos(th1) + L * np.cos(a12), L * np.sin(th1) + L * np.sin(a12)], 1)
    d = x0[:, 2:4] - tip; d /= np.linalg.norm(d, axis=1, keepdims=True)
    x0[:, 2:4] = tip + 0.072 * d
    return w, x0, x0[:, 2:4] + 0.15 * d


@pytest.mark.gpu
def test_mpc_lowers_the_cost_of_the_pushing_task(B):
    """64 environments, 2 plan steps of 24 Adam iterations over a 0.3 s horizon, 50 knots executed per plan step: the cost of
    the executed state is lower than that of executing the initial random plan, on average and in most environments; the
    cost over the iterations of a plan step is not monotone (why the best iterate is kept)"""
    import torch
    from paper_2506_14186_b200 import apps
    nenv = 64
    w, x0n, goaln = _push_task(nenv, 0.3)
    nknot, kdt = w["nknot"], w["knot_dt"]
    m = B.Model(w["model"], precision=64)
    cost = _c2_cost_torch(m.dev(goaln))
    mpc = apps.MPC(m, nenv, nknot, kdt, w["opts"], cost, cfd=True, iters=24, lr=0.05, clip=1.0, execute=50)
    x0, u0 = m.dev(x0n), m.dev(w["ctrl"])
    _, best, hist = mpc.plan_step(x0, u0)
    hist = hist.cpu().numpy()
    assert (best.cpu().numpy() <= hist.min(0) + 1e-15).all()                 # the kept iterate is the best evaluated one
    n_nonmono = int((np.diff(hist, axis=0) > 1e-9).any(0).sum())
    out = mpc.run(x0, u0, 2)
    x, u = x0, u0                                                            # baseline: the same executions without planning
    for _ in range(2):
        x = mpc.execute_plan(x, u); u = mpc.shift(u)
    c_mpc, c_base = out["cost"][-1].cpu().numpy(), cost(x)[0].cpu().numpy()
    print("MPC: mean cost %.5f (no planning %.5f), lower in %d / %d environments; %d environments with a non-monotone plan step"
          % (c_mpc.mean(), c_base.mean(), int((c_mpc < c_base).sum()), nenv, n_nonmono))
    assert np.isfinite(c_mpc).all()
    assert c_mpc.mean() < 0.9 * c_base.mean()
    assert (c_mpc < c_base).sum() >= 0.6 * nenv
    assert n_nonmono > 0


@pytest.mark.gpu
def test_sysid_recovers_the_friction_of_oracle_trajectories(B):
    """cube tosses released 7 cm above the plane (C3 model and velocities, mu* = 0.3), 0.2 s segments generated by the ORACLE at
    mu*; starting from mu = 0.6 the identification loop brings mu within 10 % of mu* and the loss down by 20x (PAPER.md:157
    reports ~5 % on real data after far more steps; sliding-only segments were tried first: there the loss is a sawtooth
    in mu and its gradient has the wrong sign over most of [0.3, 0.6])"""
    import torch
    from paper_2506_14186_b200 import apps
    nenv, horizon, mu_true = 48, 0.2, 0.3
    w = W.make("C3", nenv=nenv, mu=mu_true)
    x0 = w["x0"].copy(); x0[:, 2] = 0.12
    orc = oracle_mod.Oracle(w["model"])
    x1 = orc.rollout(x0, None, 0, 0.0, None, horizon, w["opts"], threads=16)["xT"]
    m = B.Model(w["model"], precision=64)
    p0 = torch.tensor(m.default_params()); i_mu = m.default_params().size - 8      # [masses | friction | solref 2 | solimp 5]
    assert abs(float(p0[i_mu]) - mu_true) < 1e-12
    p0[i_mu] = 0.6
    sid = apps.SysID(m, m.dev(x0), m.dev(x1), horizon, w["opts"], p0, free=[i_mu], lr=0.03)
    losses, mus = [], []
    for _ in range(60):
        mus.append(float(sid.params()[i_mu])); losses.append(sid.step())
    mu = float(sid.params()[i_mu])
    print("sys-ID: loss %.3e -> min %.3e (last %.3e), mu 0.6 -> %.4f (true %.2f); mu every 10 steps %s"
          % (losses[0], min(losses), losses[-1], mu, mu_true, np.round(mus[::10], 3)))
    assert min(losses) < 0.05 * losses[0]
    assert abs(mu - mu_true) < 0.1 * mu_true
