"""Pins P1, P2, P3, P5, P6 and narrow-phase geometry checks for the CPU oracle."""
import itertools
import numpy as np
import pytest
from scipy.optimize import brentq

import helpers as H
from paper_2506_14186_b200 import workloads as W


# ---------------------------------------------------------------- P3: M and ID
@pytest.mark.parametrize("name", ["arm", "C2", "C4", "C5"])
def test_P3_mass_matrix_from_inverse_dynamics(oracle_mod, name):
    model = H.arm(4, slide_last=True) if name == "arm" else W.make(name, nenv=1)["model"]
    orc = oracle_mod.Oracle(model)
    rng = np.random.default_rng(11)
    q = np.array(model["qpos0"]) + 0.4 * rng.normal(size=orc.nq)
    for j in range(model["njnt"]):
        if model["jnt_type"][j] == W.JNT_FREE:
            a = model["jnt_qadr"][j] + 3; q[a:a + 4] = H.rand_quat(rng)
    M = orc.mass_matrix(q)
    z = np.zeros(orc.nv)
    id0 = orc.inverse_dynamics(q, z, z)
    cols = np.stack([orc.inverse_dynamics(q, z, np.eye(orc.nv)[j]) - id0 for j in range(orc.nv)], axis=1)
    assert np.abs(M - cols).max() < 1e-13 * np.abs(M).max()
    assert np.abs(M - M.T).max() < 1e-14 * np.abs(M).max()
    assert np.linalg.eigvalsh(M).min() > 0
    L = np.linalg.cholesky(M)
    assert np.abs(L @ L.T - M).max() < 1e-14 * np.abs(M).max()
    # gravity bias: ID(q,0,0) = -dV/dq with V = sum m g z_com, by central differences in tangent coordinates
    g = -model["gravity"][2]
    p = orc.default_params()
    V = lambda qq: sum(p[b] * g * orc.kinematics(qq, z)["com"][b][2] for b in range(1, orc.nbody))
    x = np.concatenate([q, z])
    for d in range(orc.nv):
        fd = (V(H.perturb_x(orc, x, d, 1e-6)[: orc.nq]) - V(H.perturb_x(orc, x, d, -1e-6)[: orc.nq])) / 2e-6
        assert abs(id0[d] - fd) < 1e-7 * max(1, abs(fd))


def test_P3_coriolis_power_identity(oracle_mod):
    """d/dt (1/2 v^T M v) = v^T (M a) + 1/2 v^T Mdot v  and  v^T(c - g) = 1/2 v^T Mdot v  =>  checked via FD of M."""
    model = H.arm(4, gravity=(0, 0, 0), slide_last=True)
    orc = oracle_mod.Oracle(model)
    rng = np.random.default_rng(12)
    q, v = rng.uniform(-1, 1, 4), rng.normal(size=4)
    c = orc.inverse_dynamics(q, v, np.zeros(4))
    eps = 1e-6
    Mdot = (orc.mass_matrix(q + eps * v) - orc.mass_matrix(q - eps * v)) / (2 * eps)
    assert abs(v @ c - 0.5 * v @ Mdot @ v) < 1e-8


# ---------------------------------------------------------------- narrow phase
def test_collide_geometry(oracle_mod):
    w = W.make("C3", nenv=1)
    orc = oracle_mod.Oracle(w["model"])
    rng = np.random.default_rng(13)
    q = np.concatenate([[0.3, -0.2, 0.04], H.rand_quat(rng)])
    g = orc.collide(q)
    R = orc.kinematics(q, np.zeros(6))["mat"][1]
    corners = np.array([[sx, sy, sz] for sz in (-1, 1) for sy in (-1, 1) for sx in (-1, 1)]) * 0.05
    world = q[:3] + corners @ R.T
    assert np.allclose(np.sort(g["r"]), np.sort(world[:, 2]), atol=1e-15)          # r_i = n.(vertex - p0)
    assert np.allclose(g["n"], [0, 0, 1]) and np.allclose(g["t1"], [1, 0, 0]) and np.allclose(g["t2"], [0, 1, 0])
    assert np.allclose(g["pos"][:, 2], 0.5 * g["r"], atol=1e-15)                    # mid-surface: pos = vertex - r n / 2
    # sphere-sphere, brute force against sampled surface points
    m2 = H.two_spheres()
    o2 = oracle_mod.Oracle(m2)
    q2 = np.concatenate([[0.01, 0.02, 0.03], H.rand_quat(rng), [0.05, -0.02, 0.06], H.rand_quat(rng)])
    g2 = o2.collide(q2)
    c1, c2 = q2[0:3], q2[7:10]
    u = rng.normal(size=(200000, 3)); u /= np.linalg.norm(u, axis=1, keepdims=True)
    dmin = np.linalg.norm((c1 + 0.03 * u)[:, None, :][:2000] - (c2 + 0.03 * u)[None, :2000, :], axis=2).min()
    r = np.linalg.norm(c2 - c1) - 0.06
    assert abs(g2["r"][0] - r) < 1e-15 and r < 0 or abs(dmin - r) < 2e-3
    n = (c2 - c1) / np.linalg.norm(c2 - c1)
    assert np.allclose(g2["n"][0], n)
    assert np.allclose(g2["pos"][0], c1 + (0.03 + 0.5 * r) * n)
    F = np.stack([g2["n"][0], g2["t1"][0], g2["t2"][0]])
    assert np.allclose(F @ F.T, np.eye(3), atol=1e-14) and np.linalg.det(F) > 0.999   # right-handed orthonormal frame
    # capsule end caps vs plane (C4: 10 of the 12 candidates)
    w4 = W.make("C4", nenv=1); o4 = oracle_mod.Oracle(w4["model"])
    assert o4.nc == 12 and oracle_mod.Oracle(W.make("C5", nenv=1)["model"]).nc == 4 and orc.nc == 8
    g4 = o4.collide(w4["x0"][0, :14]); k4 = o4.kinematics(w4["x0"][0, :14], np.zeros(13))
    lens = [0.30, 0.30, 0.25, 0.25, 0.20, 0.15, 0.10]
    for i, body in enumerate(range(3, 8)):
        for s, ci in ((0, 2 * i), (1, 2 * i + 1)):
            cap = k4["pos"][body] + k4["mat"][body] @ np.array([0, 0, s * lens[body - 1]])
            assert abs(g4["r"][ci] - (cap[2] - 0.03)) < 1e-15


def test_rows_are_contact_point_velocities(oracle_mod):
    """J v = relative velocity of the two bodies at the contact point along n +- mu t."""
    w = W.make("C2", nenv=1); model = w["model"]; orc = oracle_mod.Oracle(model)
    rng = np.random.default_rng(14)
    q = w["x0"][0, :9].copy(); q[2:4] = [0.6 * np.cos(q[0] + q[1]) * 0.0 + 0.3 * np.cos(q[0]) + 0.3 * np.cos(q[0] + q[1]) + 0.05,
                                         0.3 * np.sin(q[0]) + 0.3 * np.sin(q[0] + q[1]) + 0.02]
    q[4] = 0.049; q[5:9] = H.rand_quat(rng)
    v = rng.normal(size=8)
    rows = orc.rows(q, v); g = orc.collide(q)
    assert np.all(g["r"] < 0) and rows["J"].shape == (8, 8)
    # FD of world points: velocity of the material point of each body at pos
    eps = 1e-7
    xq = np.concatenate([q, v])
    def material_point_vel(body, pos):
        k0 = orc.kinematics(q, v)
        loc = k0["mat"][body].T @ (pos - k0["pos"][body])
        qp = H.perturb_x(orc, xq, 0, 0.0)[:9]
        dq = lambda s: orc.retract(q, s * v)
        kp, km = orc.kinematics(dq(eps), v), orc.kinematics(dq(-eps), v)
        return ((kp["pos"][body] + kp["mat"][body] @ loc) - (km["pos"][body] + km["mat"][body] @ loc)) / (2 * eps)
    mu = 0.8
    for ci, (b1, b2) in enumerate(((0, 3), (2, 3))):
        pos, n, t1, t2 = g["pos"][ci], g["n"][ci], g["t1"][ci], g["t2"][ci]
        rel = material_point_vel(b2, pos) - (material_point_vel(b1, pos) if b1 else 0)
        expect = [(n + mu * t1) @ rel, (n - mu * t1) @ rel, (n + mu * t2) @ rel, (n - mu * t2) @ rel]
        assert np.allclose(rows["J"][4 * ci: 4 * ci + 4] @ v, expect, atol=1e-7)
    # rdot = n . relative velocity: FD of the signed distance along the motion
    rp, rm = orc.collide(orc.retract(q, eps * v))["r"], orc.collide(orc.retract(q, -eps * v))["r"]
    Jn = 0.5 * (rows["J"][0::4] + rows["J"][1::4])
    assert np.allclose(Jn @ v, (rp - rm) / (2 * eps), atol=1e-7)


def test_impedance_spline_values(oracle_mod):
    """Hand-computed values of the solimp spline (reading G5), monotone, continuous at the midpoint."""
    si = np.array([0.0, 0.95, 0.001, 0.5, 2.0])
    imp = lambda r: oracle_mod.impedance(si, r)
    assert imp(0.0) == 0.0
    assert abs(imp(-0.00025) - 0.95 * 0.125) < 1e-15       # x=.25: y = x^2/mid
    assert abs(imp(-0.0005) - 0.95 * 0.5) < 1e-15          # x=.5
    assert abs(imp(-0.00075) - 0.95 * 0.875) < 1e-15       # x=.75: y = 1-(1-x)^2/(1-mid)
    assert abs(imp(-0.001) - 0.95) < 1e-15 and abs(imp(-1.0) - 0.95) < 1e-15
    rs = -np.linspace(0, 0.0012, 500)
    d = np.array([imp(r) for r in rs])
    assert np.all(np.diff(d) >= -1e-16)
    si3 = np.array([0.2, 0.9, 0.01, 0.3, 3.0])
    assert abs(oracle_mod.impedance(si3, -0.003) - (0.2 + 0.7 * 0.3)) < 1e-15   # y(mid) = mid
    # CFD continuation (G16): d_0 at r=0, d_c at r=w_c, with m_c=1: d = d_0 + (d_c-d_0) (r/w_c)^p_c
    sc = np.array([0.0, 0.1, 1.0, 1.0, 4.0])
    assert abs(oracle_mod.impedance_cfd(sc, 1e-300) - 0.1) < 1e-15
    assert abs(oracle_mod.impedance_cfd(sc, 0.5) - (0.1 - 0.1 * 0.5 ** 4)) < 1e-15
    assert abs(oracle_mod.impedance_cfd(sc, 1.0 - 1e-12)) < 1e-11
    # softplus: relu limit and value at 0
    assert abs(oracle_mod.softplus(0.0, 10.0) - np.log(2) / 10) < 1e-16
    assert abs(oracle_mod.softplus(3.0, 50.0) - 3.0) < 1e-15 and oracle_mod.softplus(-3.0, 50.0) < 1e-60


# ---------------------------------------------------------------- P5 / P6: solver (Eq. 2)
def _random_problem(rng, nv, nr):
    B = rng.normal(size=(nv, nv)); M = B @ B.T + nv * np.eye(nv)
    return M, rng.normal(size=nv) * 3, rng.normal(size=(nr, nv)), rng.normal(size=nr) * 3, rng.uniform(0.5, 50, nr)


def _phi(M, a0, J, aref, D, x):
    s = np.minimum(0, J @ x - aref)
    return 0.5 * (x - a0) @ M @ (x - a0) + 0.5 * np.sum(D * s * s)


def test_P5_solver_matches_brute_force_active_set(oracle_mod):
    rng = np.random.default_rng(21)
    nconv4 = 0
    for trial in range(40):
        nv, nr = int(rng.integers(1, 7)), int(rng.integers(1, 11))
        M, a0, J, aref, D = _random_problem(rng, nv, nr)
        sol = oracle_mod.contact_solve(M, a0, J, aref, D, n_it=50, n_ls=50)
        assert sol["converged"]
        hits = []
        for A in itertools.product([0, 1], repeat=nr):
            A = np.array(A, dtype=bool)
            Hm = M + J[A].T @ (D[A, None] * J[A]); x = np.linalg.solve(Hm, M @ a0 + J[A].T @ (D[A] * aref[A]))
            s = J @ x - aref
            if np.all(s[A] < 0) and np.all(s[~A] >= 0):
                hits.append((A, x))
        assert len(hits) == 1                                    # strictly convex: unique consistent active set
        A, x = hits[0]
        assert np.abs(sol["x"] - x).max() < 1e-11 * max(1, np.abs(x).max())
        assert np.array_equal(sol["active"], A)
        s = J @ sol["x"] - aref
        grad = M @ (sol["x"] - a0) + J.T @ (D * np.minimum(0, s))
        assert np.abs(grad).max() < 1e-10 * max(1, np.abs(M @ a0).max())
        assert np.all(sol["f"] >= 0) and np.abs(sol["f"] * np.maximum(0, s)).max() == 0
        assert np.allclose(sol["f"], D * np.maximum(0, -s), atol=1e-12)
        s4 = oracle_mod.contact_solve(M, a0, J, aref, D, n_it=4, n_ls=16)
        nconv4 += s4["converged"]
        assert _phi(M, a0, J, aref, D, s4["x"]) <= _phi(M, a0, J, aref, D, a0) + 1e-12
        if s4["converged"]:
            assert np.abs(s4["x"] - x).max() < 1e-11 * max(1, np.abs(x).max())
    assert nconv4 >= 30                                          # the fixed 4-iteration budget usually suffices
    e = oracle_mod.contact_solve(M, a0, np.zeros((0, nv)), np.zeros(0), np.zeros(0))
    assert np.array_equal(e["x"], a0)                            # no rows: v' = a0, solver skipped


def test_P6_line_search_matches_exact_breakpoint_sweep(oracle_mod):
    rng = np.random.default_rng(22)
    checked = 0
    for trial in range(60):
        nv, nr = int(rng.integers(2, 7)), int(rng.integers(3, 13))
        M, a0, J, aref, D = _random_problem(rng, nv, nr)
        s = J @ a0 - aref; A = s < 0
        g = J[A].T @ (D[A] * s[A]); Hm = M + J[A].T @ (D[A, None] * J[A])
        dl = -np.linalg.solve(Hm, g); p = J @ dl
        if np.array_equal(A, (s + p) < 0):
            continue                                             # full step stays inside the active set
        # exact minimiser of the convex piecewise quadratic phi(a): sweep the breakpoints -s_i/p_i
        d1 = lambda a: a * (dl @ M @ dl) + np.sum(D * p * np.minimum(0, s + a * p))
        bps = sorted(set([0.0] + [float(-s[i] / p[i]) for i in range(nr) if p[i] != 0 and -s[i] / p[i] > 0] + [1e9]))
        alpha = None
        for lo, hi in zip(bps[:-1], bps[1:]):
            if d1(lo) <= 0 <= d1(hi):
                mid = 0.5 * (lo + hi); act = (s + mid * p) < 0
                c2 = dl @ M @ dl + np.sum(D[act] * p[act] ** 2); c1 = np.sum(D[act] * p[act] * s[act])
                alpha = -c1 / c2; break
        assert alpha is not None
        sol = oracle_mod.contact_solve(M, a0, J, aref, D, n_it=1, n_ls=60)
        assert np.abs(sol["x"] - (a0 + alpha * dl)).max() < 1e-10 * max(1, np.abs(dl).max())
        checked += 1
    assert checked >= 10


# ---------------------------------------------------------------- P1 / P2: closed forms
def _oscillator_params(dbar, tc, m=1.0):
    """C1 ball: A^ = trace/3 = 1/(3m) (G7), constant impedance -> effective impedance d' and a linear ODE."""
    eta = 3.0
    dp = eta * dbar / (1 - dbar + eta * dbar)
    b = 2.0 / (dbar * tc); k = dbar / (dbar ** 2 * tc ** 2)
    return dp, dp * b, dp * k          # r'' + cb r' + ck r = -(1-dp) g


def _closed_form_bounce(h0, v0, T, rho, dbar, tc):
    dp, cb, ck = _oscillator_params(dbar, tc)
    b, k = cb / dp, ck / dp
    t1 = (h0 - rho) / (-v0)
    lam = np.roots([1.0, cb, ck]).astype(complex)
    r = lambda t: (v0 * (np.exp(lam[0] * t) - np.exp(lam[1] * t)) / (lam[0] - lam[1])).real
    rd = lambda t: (v0 * (lam[0] * np.exp(lam[0] * t) - lam[1] * np.exp(lam[1] * t)) / (lam[0] - lam[1])).real
    aref = lambda t: -b * rd(t) - k * r(t)
    ts = np.linspace(1e-9, 20 * tc, 20001); sgn = aref(ts)
    i = np.argmax(sgn < 0); trel = brentq(aref, ts[i - 1], ts[i], xtol=1e-16, rtol=1e-15)
    return rho + r(trel) + rd(trel) * (T - t1 - trel), trel, rd(trel)


def test_P1_single_contact_damped_oscillator_closed_form(oracle_mod):
    dbar, tc, rho, T = 0.9, 0.004, 0.1, 0.5
    w = W.ball_drop(nenv=1, gravity=0.0, solref=(tc, 1.0), solimp=(dbar, dbar, 0.001, 0.5, 2.0))
    orc = oracle_mod.Oracle(w["model"])
    assert abs(orc.invweight()[1][0] - 1.0 / 3.0) < 1e-15
    opts = W.default_opts(W.DOPRI5, 1e-11, 1e-11, h0=1e-3)
    h0, v0 = 0.35, -1.7
    zT, trel, vrel = _closed_form_bounce(h0, v0, T, rho, dbar, tc)
    assert vrel > 0 and 0 < trel < 10 * tc
    x0 = np.array([[h0, v0]])
    g = orc.rollout_grad(x0, None, 0, 0.0, None, T, opts, loss_grad=w["loss_grad"])
    assert abs(g["xT"][0, 0] - zT) < 5e-9 and abs(g["xT"][0, 1] - vrel) < 5e-8
    # With constant impedance d_o>0 the force JUMPS at r=0, so the continuous sensitivity has a
    # saltation term that no discrete adjoint through frozen steps contains: the closed-form derivative
    # -v_rel/|v0| is NOT what discretize-then-optimize returns here (it returns the smooth part only).  The
    # gradient is therefore pinned by finite differences of the frozen-schedule map (test_oracle_grad.py, P7)
    # and, for continuous onset (d_o=0), by free-running FD at tight tolerance.
    dh_true = -vrel / abs(v0)
    assert abs(g["dLdx0"][0, 0] - dh_true) > 1.0
    # the general phi_d: zeta scales with the damping ratio (Eq. 3): critically damped textbook case
    # eta d/(1-d+eta d) with d -> effective; check the contact duration against the closed form for another phi_d
    w2 = W.ball_drop(nenv=1, gravity=0.0, solref=(tc, 0.5), solimp=(dbar, dbar, 0.001, 0.5, 2.0))
    o2 = oracle_mod.Oracle(w2["model"])
    dp = 3 * dbar / (1 + 2 * dbar); b = 2 / (dbar * tc); k = dbar / (dbar ** 2 * tc ** 2 * 0.25)
    lam = np.roots([1.0, dp * b, dp * k]).astype(complex)
    rd = lambda t: (v0 * (lam[0] * np.exp(lam[0] * t) - lam[1] * np.exp(lam[1] * t)) / (lam[0] - lam[1])).real
    r_ = lambda t: (v0 * (np.exp(lam[0] * t) - np.exp(lam[1] * t)) / (lam[0] - lam[1])).real
    ar = lambda t: -b * rd(t) - k * r_(t)
    ts = np.linspace(1e-9, 20 * tc, 20001); i = np.argmax(ar(ts) < 0); trel2 = brentq(ar, ts[i - 1], ts[i], xtol=1e-16)
    t1 = (h0 - rho) / (-v0)
    z2 = rho + r_(trel2) + rd(trel2) * (T - t1 - trel2)
    r2 = o2.rollout(x0, None, 0, 0.0, None, T, opts)
    assert abs(r2["xT"][0, 0] - z2) < 5e-9 and abs(r2["xT"][0, 1] - rd(trel2)) < 5e-8


def test_P2_resting_penetration_with_gravity(oracle_mod):
    """At rest: (1-d') g = d' k(r) (-r) with variable d(r); the ball settles there (restitution ~ e^-2)."""
    w = W.ball_drop(nenv=1)
    orc = oracle_mod.Oracle(w["model"])
    r = orc.rollout(np.array([[0.2, 0.0]]), None, 0, 0.0, None, 1.5, W.default_opts(W.DOPRI5, 1e-10, 1e-10))
    z, v = r["xT"][0]
    assert abs(v) < 1e-7
    tc, dw, wd, mid, pw = 0.002, 0.95, 0.001, 0.5, 2.0
    def dimp(pen):
        x = min(pen / wd, 1.0)
        y = x ** pw / mid ** (pw - 1) if x <= mid else 1 - (1 - x) ** pw / (1 - mid) ** (pw - 1)
        return y * dw
    def resid(pen):
        d = dimp(pen); dp = 3 * d / (1 + 2 * d)
        return dp * d / (dw ** 2 * tc ** 2) * pen - (1 - dp) * 9.81
    pen = brentq(resid, 1e-9, 0.001, xtol=1e-16)
    assert abs((0.1 - z) - pen) < 1e-9
    # vector field at the resting state is zero; slightly above the plane it is free fall
    acc, nr, conv = orc.vector_field([0.1 - pen], [0.0])
    assert abs(acc[0]) < 1e-6 and nr == 1 and conv
    acc, nr, _ = orc.vector_field([0.1001], [0.0])
    assert abs(acc[0] + 9.81) < 1e-14 and nr == 0
