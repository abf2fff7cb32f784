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
