"""Pins P9, P10, P11, P4: tableaus, manifold update, linear discrete adjoint, invariants."""
import numpy as np
import pytest

import helpers as H
from paper_2506_14186_b200 import workloads as W


def order_conditions(A, b, c, order):
    """Rooted-tree order conditions of an explicit RK method up to `order` (17 for order 5)."""
    one = np.ones_like(c)
    Ac, Ac2, Ac3 = A @ c, A @ c**2, A @ c**3
    AAc = A @ Ac
    res = [b @ one - 1, b @ c - 1 / 2, b @ c**2 - 1 / 3, b @ Ac - 1 / 6,
           b @ c**3 - 1 / 4, b @ (c * Ac) - 1 / 8, b @ Ac2 - 1 / 12, b @ AAc - 1 / 24]
    if order >= 5:
        res += [b @ c**4 - 1 / 5, b @ (c**2 * Ac) - 1 / 10, b @ (Ac * Ac) - 1 / 20, b @ (c * Ac2) - 1 / 15,
                b @ Ac3 - 1 / 20, b @ (c * AAc) - 1 / 30, b @ (A @ (c * Ac)) - 1 / 40, b @ (A @ Ac2) - 1 / 60,
                b @ (A @ AAc) - 1 / 120]
    return np.array(res)


@pytest.mark.parametrize("which,tol", [(W.DOPRI5, 5e-16), (W.TSIT5, 5e-15)])
def test_P9_tableau_order_conditions(oracle_mod, which, tol):
    c, A, b, e = oracle_mod.tableau(which)
    assert np.allclose(A.sum(1), c, atol=2e-16 if which == W.DOPRI5 else 1e-15)       # rows sum to c
    assert np.all(np.triu(A) == 0)                                                     # explicit
    r5 = order_conditions(A, b, c, 5)
    assert len(r5) == 17 and np.abs(r5).max() < tol
    r4 = order_conditions(A, b - e, c, 4)                                              # embedded 4th order
    assert np.abs(r4).max() < tol
    # the embedded solution is NOT 5th order (the error estimate is non-trivial)
    assert np.abs(order_conditions(A, b - e, c, 5)[8:]).max() > 1e-5
    assert b[6] == 0 and np.allclose(A[6, :6], b[:6], atol=0)                          # FSAL


@pytest.mark.parametrize("which", [W.DOPRI5, W.TSIT5])
def test_P9_fixed_step_convergence_slope(oracle_mod, which):
    m, kp = 1.3, 7.0
    orc = oracle_mod.Oracle(H.oscillator(m, kp))
    om = np.sqrt(kp / m)
    x0 = np.array([[0.8, -0.3]]); T = 2.0
    exact = np.array([0.8 * np.cos(om * T) - 0.3 / om * np.sin(om * T), -0.8 * om * np.sin(om * T) - 0.3 * np.cos(om * T)])
    errs = []
    for n in (10, 20, 40):
        hs = np.full((1, n), T / n)
        r = orc.rollout(x0, np.zeros((1, 1, 1)), 1, 10.0, None, T, W.default_opts(which), h_replay=hs)
        assert r["stats"]["n_accept"][0] == n
        errs.append(np.abs(r["xT"][0] - exact).max())
    slopes = np.log2(np.array(errs[:-1]) / np.array(errs[1:]))
    assert np.all(slopes > 4.7) and np.all(slopes < 5.6), slopes


def test_P10_quaternion_update_exact_for_constant_body_rate(oracle_mod):
    """Constant body angular velocity (spherical inertia, no forces) is integrated exactly in ONE step."""
    mb = W.ModelBuilder(gravity=(0, 0, 0))
    b = mb.body(0, mass=2.0, inertia_unit=(0.1, 0.1, 0.1)); mb.joint(b, W.JNT_FREE)
    orc = oracle_mod.Oracle(mb.build())
    rng = np.random.default_rng(3)
    for h in (1e-3, 0.7, 5.0):
        q0 = H.rand_quat(rng); w = rng.normal(size=3) * 2; v = rng.normal(size=3)
        x0 = np.concatenate([[0.1, 0.2, 0.3], q0, v, w])[None]
        r = orc.rollout(x0, None, 0, 0.0, None, h, W.default_opts(W.TSIT5), h_replay=np.array([[h]]))
        th = np.linalg.norm(w) * h
        dq = np.concatenate([[np.cos(th / 2)], np.sin(th / 2) * w / np.linalg.norm(w)])
        a, bq = q0, dq
        expect = np.array([a[0]*bq[0]-a[1]*bq[1]-a[2]*bq[2]-a[3]*bq[3], a[0]*bq[1]+a[1]*bq[0]+a[2]*bq[3]-a[3]*bq[2],
                           a[0]*bq[2]-a[1]*bq[3]+a[2]*bq[0]+a[3]*bq[1], a[0]*bq[3]+a[1]*bq[2]-a[2]*bq[1]+a[3]*bq[0]])
        xT = r["xT"][0]
        assert np.abs(xT[3:7] - expect).max() < 1e-14 * max(1.0, th**3)      # exact up to rounding of Theta x w
        assert abs(np.linalg.norm(xT[3:7]) - 1) < 1e-15
        assert np.abs(xT[0:3] - (x0[0, 0:3] + h * v)).max() < 1e-14


def test_P11_linear_discrete_adjoint_equals_stability_polynomial(oracle_mod):
    m, kp = 0.9, 11.0
    orc = oracle_mod.Oracle(H.oscillator(m, kp))
    Amat = np.array([[0.0, 1.0], [-kp / m, 0.0]])
    for which in (W.DOPRI5, W.TSIT5):
        c, A, b, e = oracle_mod.tableau(which)
        n, h = 7, 0.13
        hs = np.full((1, n), h)
        Rz = np.eye(2); Ak = np.eye(7); one = np.ones(7); Z = np.eye(2)
        for k in range(1, 7):
            Z = Z @ (h * Amat)
            Rz = Rz + (b @ Ak @ one) * Z
            Ak = Ak @ A
        lamT = np.array([0.3, -1.1])
        g = orc.rollout_grad(np.array([[0.5, 0.2]]), np.zeros((1, 1, 1)), 1, 10.0, None, n * h, W.default_opts(which),
                             dLdxT=lamT[None], h_replay=hs)
        expect = np.linalg.matrix_power(Rz.T, n) @ lamT
        assert np.abs(g["dLdx0"][0] - expect).max() < 1e-13
        # gradient w.r.t. the (constant) PD target: dq''/du = kp/m
        xs = np.array([[0.5, 0.2]])
        f = lambda u: orc.rollout(xs, np.full((1, 1, 1), u), 1, 10.0, None, n * h, W.default_opts(which), h_replay=hs)["xT"][0] @ lamT
        assert abs(g["dLdctrl"][0, 0, 0] - (f(1e-4) - f(-1e-4)) / 2e-4) < 1e-8


def _energy_momentum(orc, x, g=0.0):
    nq = orc.nq
    k = orc.kinematics(x[:nq], x[nq:]); I = orc.world_inertia(x[:nq]); p = orc.default_params()
    T = 0.0; L = np.zeros(3); P = np.zeros(3); V = 0.0
    for b in range(1, orc.nbody):
        mb_ = p[b]
        T += 0.5 * mb_ * k["comvel"][b] @ k["comvel"][b] + 0.5 * k["angvel"][b] @ I[b] @ k["angvel"][b]
        P += mb_ * k["comvel"][b]
        L += I[b] @ k["angvel"][b] + mb_ * np.cross(k["com"][b], k["comvel"][b])
        V += mb_ * g * k["com"][b][2]
    return T, V, P, L


def test_P4_torque_free_box_invariants_and_tolerance_scaling(oracle_mod):
    orc = oracle_mod.Oracle(H.free_box())
    rng = np.random.default_rng(5)
    x0 = np.concatenate([[0, 0, 0.5], H.rand_quat(rng), rng.normal(size=3), rng.normal(size=3) * 6])[None]
    T0, _, P0, L0 = _energy_momentum(orc, x0[0])
    drift = []
    for tol in (1e-6, 1e-9):
        r = orc.rollout(x0, None, 0, 0.0, None, 1.5, W.default_opts(W.TSIT5, tol, tol))
        T1, _, P1, L1 = _energy_momentum(orc, r["xT"][0])
        drift.append(max(abs(T1 - T0) / T0, np.abs(L1 - L0).max() / np.linalg.norm(L0),
                         np.abs(P1 - P0).max() / np.linalg.norm(P0)))      # COM is offset from the body origin
        assert r["stats"]["status"][0] == 0
    assert drift[0] < 2e-5 and drift[1] < 3e-8 and drift[1] < drift[0] * 1e-2      # error ~ tolerance


def test_P4_free_fall_energy_and_parabola(oracle_mod):
    orc = oracle_mod.Oracle(H.free_box(gravity=(0, 0, -9.81)))
    rng = np.random.default_rng(6)
    x0 = np.concatenate([[0, 0, 0.5], H.rand_quat(rng), [0.3, -0.2, 1.0], rng.normal(size=3)])[None]
    r = orc.rollout(x0, None, 0, 0.0, None, 0.8, W.default_opts(W.TSIT5, 1e-9, 1e-9))
    T0, V0, _, _ = _energy_momentum(orc, x0[0], 9.81); T1, V1, _, _ = _energy_momentum(orc, r["xT"][0], 9.81)
    assert abs((T1 + V1) - (T0 + V0)) < 1e-8 * abs(T0 + V0)
    k0 = orc.kinematics(x0[0, :7], x0[0, 7:]); k1 = orc.kinematics(r["xT"][0, :7], r["xT"][0, 7:])
    expect = k0["com"][1] + 0.8 * k0["comvel"][1] + np.array([0, 0, -0.5 * 9.81 * 0.64])
    assert np.abs(k1["com"][1] - expect).max() < 1e-8


def test_P4_passive_arm_conserves_energy(oracle_mod):
    orc = oracle_mod.Oracle(H.arm(4, slide_last=True))
    rng = np.random.default_rng(7)
    x0 = np.concatenate([rng.uniform(-1, 1, 4), rng.normal(size=4)])[None]
    ctrl = np.zeros((1, 1, 4))
    E = []
    for tol in (1e-6, 1e-9):
        r = orc.rollout(x0, ctrl, 1, 10.0, None, 1.0, W.default_opts(W.TSIT5, tol, tol))
        x1 = r["xT"][0]
        e0 = 0.5 * x0[0, 4:] @ orc.mass_matrix(x0[0, :4]) @ x0[0, 4:] + _energy_momentum(orc, x0[0], 9.81)[1]
        e1 = 0.5 * x1[4:] @ orc.mass_matrix(x1[:4]) @ x1[4:] + _energy_momentum(orc, x1, 9.81)[1]
        E.append(abs(e1 - e0) / abs(e0))
    assert E[0] < 1e-4 and E[1] < 1e-7, E


def test_kinetic_energy_two_ways(oracle_mod):
    """1/2 v^T M v (joint space) equals the sum of body kinetic energies (maximal coordinates)."""
    for model in (H.arm(4, slide_last=True), W.quadruped(nenv=1)["model"]):
        orc = oracle_mod.Oracle(model)
        rng = np.random.default_rng(8)
        q = np.array(model["qpos0"]) + 0.3 * rng.normal(size=orc.nq)
        for j in range(model["njnt"]):
            if model["jnt_type"][j] == W.JNT_FREE:
                a = model["jnt_qadr"][j] + 3; q[a:a + 4] /= np.linalg.norm(q[a:a + 4])
        v = rng.normal(size=orc.nv)
        T = _energy_momentum(orc, np.concatenate([q, v]))[0]
        M = orc.mass_matrix(q)
        # armature is joint-space only
        arm_ = sum(model["jnt_armature"][j] * v[model["jnt_vadr"][j]] ** 2 * 0.5 for j in range(model["njnt"]) if model["jnt_type"][j] != W.JNT_FREE)
        assert abs(0.5 * v @ M @ v - T - arm_) < 1e-12 * max(1, T)


def _tumbling_box_case():
    """Torque-free ASYMMETRIC box (principal inertias all different, COM offset), |omega| = 6 rad/s, no contacts."""
    rng = np.random.default_rng(5)
    w = rng.normal(size=3); w *= 6.0 / np.linalg.norm(w)
    return np.concatenate([[0, 0, 0.5], H.rand_quat(rng), rng.normal(size=3), w])[None]


@pytest.mark.parametrize("which", [W.DOPRI5, W.TSIT5])
def test_chart_rate_keeps_order_five_on_a_tumbling_body(oracle_mod, which):
    """Pin of reading G10 ("exact integration of quaternions"; PAPER.md:456 order-p consistency): with
    tangent-space stages Q_i = q_n (+) Theta_i the rotational chart rate must be dexp^-1 truncated after B_2,
        Theta' = w + 1/2 Theta x w + 1/12 Theta x (Theta x w),
    for the pair to keep order 5 on a body whose angular velocity changes direction.  Fixed steps n = 20/40/80 over
    1 s against a free-running rtol = 1e-13 solution.  Measured slopes (log2 of successive error ratios), this test's
    input, oracle as committed: Dopri5 4.99 / 5.00, Tsit5 5.25 / 4.93.  With the oracle's chart_rate mutated:
        1/12 term removed        -> 3.02 / 3.00   (fails)
        1/12 replaced by 1/6     -> 3.02 / 3.01   (fails)
        1/2 term removed         -> 2.02 / 2.07   (fails)
    P10 cannot see these terms (Theta || w there) and the adaptive invariants of P4 only take smaller steps."""
    orc = oracle_mod.Oracle(H.free_box())
    x0 = _tumbling_box_case(); T = 1.0
    ref = orc.rollout(x0, None, 0, 0.0, None, T, W.default_opts(W.TSIT5, 1e-13, 1e-13, h0=1e-3))
    assert ref["stats"]["status"][0] == 0
    errs = []
    for n in (20, 40, 80):
        r = orc.rollout(x0, None, 0, 0.0, None, T, W.default_opts(which), h_replay=np.full((1, n), T / n))
        assert r["stats"]["n_accept"][0] == n
        errs.append(np.abs(r["xT"][0] - ref["xT"][0]).max())
    slopes = np.log2(np.array(errs[:-1]) / np.array(errs[1:]))
    assert np.all(slopes > 4.7) and np.all(slopes < 5.6), (errs, slopes)


def _controller_replica(A, tab, y0, T, nknot, knot_dt, o, max_attempts=400):
    """Adaptive integration of the LINEAR system y' = A y written out with NumPy from DESIGN.md G12 / G2 (not from the
    oracle's code): stages by the tableau, e = h sum (b - bhat)_i k_i, scale = atol + rtol max(|y_n|, |y_n+1|),
    E = sqrt(mean((e/scale)^2)), accept iff E <= 1, fac = clip(safety E^(-(P+I)/5) E_prev^(P/5), fac_min, fac_max),
    fac = fac_min when the attempt is not finite, E floored at 1e-30, E_prev updated on accept only, h <- h fac after
    accept and after reject EXCEPT after an accepted step that was clipped to a knot / the horizon (the proposal is
    kept), steps clipped to knot boundaries when h (1 + 1e-7) >= remaining."""
    c, a, b, e = tab
    t, y, hprop, Eprev, knot = 0.0, np.array(y0, dtype=float), o["h0"], 1.0, 0
    hs, nrej = [], 0
    for _ in range(max_attempts):
        if not t < T:
            break
        tb = min((knot + 1) * knot_dt, T) if nknot > 0 else T
        if knot + 1 >= nknot:
            tb = T
        rem = tb - t
        hits = hprop * (1 + 1e-7) >= rem
        h = rem if hits else hprop
        with np.errstate(all="ignore"):
            k = []
            for i in range(7):
                Yi = y + h * sum((a[i, l] * k[l] for l in range(i)), np.zeros(2))
                k.append(A @ Yi)
            y1 = y + h * sum((a[6, l] * k[l] for l in range(6)), np.zeros(2))
            err = h * sum((e[i] * k[i] for i in range(7)), np.zeros(2))
            finite = bool(np.all(np.isfinite(err)) and np.all(np.isfinite(np.array(k))))
            if finite:
                E = np.sqrt(np.mean((err / (o["atol"] + o["rtol"] * np.maximum(np.abs(y), np.abs(y1)))) ** 2))
                accept = E <= 1.0
                Ec = max(E, 1e-30)
                fac = o["safety"] * Ec ** (-(o["pcoeff"] + o["icoeff"]) / 5.0) * Eprev ** (o["pcoeff"] / 5.0)
            else:
                accept, Ec, fac = False, np.inf, o["fac_min"]
        fac = min(o["fac_max"], max(o["fac_min"], fac))
        if (not accept) or (not hits):
            hprop = h * fac
        if not accept:
            nrej += 1
            continue
        Eprev = Ec
        hs.append(h); y = y1
        if hits:
            t = tb
            if tb < T:
                knot += 1
        else:
            t += h
    return np.array(hs), nrej, y


@pytest.mark.parametrize("which", [W.DOPRI5, W.TSIT5])
@pytest.mark.parametrize("case", ["knots_and_rejections", "non_finite_start"])
def test_controller_step_sequence_matches_hand_computation(oracle_mod, which, case):
    """Pin of reading G12 / G2 (PAPER.md:347 fixes only P = 0.2, I = 0.4, D = 0): the oracle's accepted step sizes and
    reject count on m q'' = -kp q against the replica above.  Swapping the two exponents, dropping E_prev, updating
    E_prev on rejects, or letting a clipped accepted step overwrite the proposal changes the h sequence."""
    m, kp = 1.3, 7.0
    orc = oracle_mod.Oracle(H.oscillator(m, kp))
    A = np.array([[0.0, 1.0], [-kp / m, 0.0]])
    tab = oracle_mod.tableau(which)
    if case == "knots_and_rejections":     # h0 far too large: rejections first; 4 knots clip accepted steps
        o = W.default_opts(which, 1e-7, 1e-7, h0=0.9); T, nknot, knot_dt = 2.0, 4, 0.5
    else:                                  # h0 = 1e60 on an unreachable horizon: stages overflow -> non-finite -> fac_min until
        o = W.default_opts(which, 1e-6, 1e-6, h0=1e60, max_steps=120); T, nknot, knot_dt = 1e70, 1, 1e80   # finite; stopped by the budget
    x0 = np.array([[0.8, -0.3]])
    r = orc.rollout(x0, np.zeros((1, nknot, 1)), nknot, knot_dt, None, T, o, n_hout=400)
    hs, nrej, yT = _controller_replica(A, tab, x0[0], T, nknot, knot_dt, o, max_attempts=o["max_steps"])
    na = int(r["stats"]["n_accept"][0])
    assert r["stats"]["status"][0] == (0 if case == "knots_and_rejections" else 1)      # 1: step budget
    assert na == len(hs) and int(r["stats"]["n_reject"][0]) == nrej
    assert nrej >= (3 if case == "knots_and_rejections" else 80) and na >= 10
    # The first dozen accepted steps agree to rounding.  Later ones only to ~1e-5: a step clipped to a knot can be tiny,
    # its error estimate is then rounding noise, and that noise enters the next factors through E_prev^(P/5).
    assert np.abs(r["h"][0, :12] - hs[:12]).max() <= 1e-9 * hs.max()
    assert np.abs(r["h"][0, :na] - hs).max() <= 2e-4 * hs.max()
    assert np.abs(r["xT"][0] - yT).max() < 1e-9
    if case == "knots_and_rejections":
        # at least one accepted step was clipped to a knot and the next step resumed with the unclipped proposal
        ends = np.cumsum(hs)
        clipped = [i for i in range(len(hs) - 1) if abs(ends[i] / knot_dt - round(ends[i] / knot_dt)) < 1e-12 and hs[i + 1] > hs[i] * 1.0000001]
        assert clipped
