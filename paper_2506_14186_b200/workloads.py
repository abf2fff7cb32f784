"""Seeded synthetic workloads shaped like the paper's (BASELINE.json configs).

This module holds INPUT GENERATION only — model descriptions (plain arrays), initial states,
control sequences, solver options and the caller-side loss — and none of the method's
arithmetic.  It is the one module that both the CUDA binding and the CPU oracle are fed from
(neither imports the other).  No paper dataset is in the container (ContactNets, MyoSuite:
PAPER.md:157, 173); these inputs stand in for them.

Random draws: SplitMix64 counter-based generator -> 53-bit uniforms -> Box-Muller normals,
seed 250614186 + config index, drawn env-major in the order listed in each builder.
"""
import math
import numpy as np

JNT_FREE, JNT_HINGE, JNT_SLIDE = 0, 1, 2
GEOM_PLANE, GEOM_SPHERE, GEOM_CAPSULE, GEOM_BOX = 0, 1, 2, 3
ACT_MOTOR, ACT_PD = 0, 1
DOPRI5, TSIT5 = 0, 1

SOLIMP_DEFAULT = (0.0, 0.95, 0.001, 0.5, 2.0)
SOLIMP_CFD_ON = (0.1, 0.95, 0.001, 0.5, 2.0)
SOLIMP_CFD = (0.0, 0.1, 1.0, 1.0, 4.0)             # PAPER.md:537 (d_c, d_0, w_c, m_c, p_c)
SOLIMP_CFD_SMOOTH = (0.01, 0.0, 1.0, 1.0, 4.0)     # PAPER.md:515 ("d_c=0.01, d_0=0 with w_c=1 m"), pairs with d_o=0


class SplitMix64:
    """Counter-based: draw i depends only on (seed, i)."""
    _G = np.uint64(0x9E3779B97F4A7C15)

    def __init__(self, seed):
        self.seed = np.uint64(seed)
        self.count = 0

    def _bits(self, n):
        idx = np.arange(self.count + 1, self.count + n + 1, dtype=np.uint64)
        self.count += n
        with np.errstate(over="ignore"):
            z = self.seed + idx * self._G
            z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
            z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
            z = z ^ (z >> np.uint64(31))
        return z

    def uniform(self, n, lo=0.0, hi=1.0):
        u = (self._bits(n) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)
        return lo + (hi - lo) * u

    def normal(self, n, sigma=1.0):
        m = (n + 1) // 2
        u = self.uniform(2 * m)
        u1 = 1.0 - u[0::2]          # (0,1]
        u2 = u[1::2]
        r = np.sqrt(-2.0 * np.log(u1))
        z = np.stack([r * np.cos(2 * math.pi * u2), r * np.sin(2 * math.pi * u2)], axis=1).reshape(-1)
        return sigma * z[:n]


class ModelBuilder:
    """Assembles the flat arrays of the model description (SURVEY.md §8(b) dmx_model_desc)."""

    def __init__(self, gravity=(0.0, 0.0, -9.81), newton_iters=4, ls_iters=16):
        self.gravity = tuple(gravity)
        self.newton_iters, self.ls_iters = newton_iters, ls_iters
        self.bodies = [dict(parent=0, pos=(0, 0, 0), quat=(1, 0, 0, 0), mass=0.0, ipos=(0, 0, 0),
                            iquat=(1, 0, 0, 0), inertia_unit=(0, 0, 0))]
        self.joints, self.geoms, self.pairs, self.acts = [], [], [], []
        self.nq = self.nv = 0
        self.qpos0 = []

    def body(self, parent, pos=(0, 0, 0), quat=(1, 0, 0, 0), mass=1.0, ipos=(0, 0, 0), iquat=(1, 0, 0, 0),
             inertia_unit=(1, 1, 1)):
        self.bodies.append(dict(parent=parent, pos=pos, quat=quat, mass=mass, ipos=ipos, iquat=iquat,
                                inertia_unit=inertia_unit))
        return len(self.bodies) - 1

    def joint(self, body, jtype, axis=(0, 0, 1), pos=(0, 0, 0), damping=0.0, armature=0.0, q0=None):
        self.joints.append(dict(type=jtype, body=body, qadr=self.nq, vadr=self.nv, axis=axis, pos=pos,
                                damping=damping, armature=armature))
        if jtype == JNT_FREE:
            b = self.bodies[body]
            self.qpos0 += list(q0 if q0 is not None else tuple(b["pos"]) + tuple(b["quat"]))
            self.nq += 7
            self.nv += 6
        else:
            self.qpos0 += [0.0 if q0 is None else q0]
            self.nq += 1
            self.nv += 1
        return len(self.joints) - 1

    def geom(self, body, gtype, size=(0, 0, 0), pos=(0, 0, 0), quat=(1, 0, 0, 0)):
        size = tuple(size) + (0.0,) * (3 - len(size))
        self.geoms.append(dict(type=gtype, body=body, size=size, pos=pos, quat=quat))
        return len(self.geoms) - 1

    def pair(self, g1, g2, condim=3, friction=1.0, solref=(0.002, 1.0), solimp=SOLIMP_DEFAULT,
             solimp_cfd=SOLIMP_CFD, cfd_beta=None):
        if cfd_beta is None:
            # reading G17: the softplus turns on over the contact's own length scale, the solimp
            # width.  A sharpness tied to w_c instead (10/w_c) offsets a_ref by ln2/beta = 7 cm at w_c = 1 m,
            # which times the impedance slope makes the backward pass of F~ unstable at the forward step sizes.
            cfd_beta = 1.0 / solimp[2]
        self.pairs.append(dict(g1=g1, g2=g2, condim=condim, friction=friction, solref=solref, solimp=solimp,
                               solimp_cfd=solimp_cfd, cfd_beta=cfd_beta))
        return len(self.pairs) - 1

    def actuator(self, joint, atype=ACT_MOTOR, gear=1.0, kp=0.0, kd=0.0):
        self.acts.append(dict(type=atype, jnt=joint, gear=gear, kp=kp, kd=kd))
        return len(self.acts) - 1

    def build(self):
        f8 = lambda key, src: np.ascontiguousarray(np.array([s[key] for s in src], dtype=np.float64).reshape(-1))
        i4 = lambda key, src: np.ascontiguousarray(np.array([s[key] for s in src], dtype=np.int32).reshape(-1))
        B, J, G, P, A = self.bodies, self.joints, self.geoms, self.pairs, self.acts
        return dict(
            nbody=len(B), njnt=len(J), nq=self.nq, nv=self.nv, nu=len(A), ngeom=len(G), npair=len(P),
            body_parent=i4("parent", B), body_pos=f8("pos", B), body_quat=f8("quat", B), body_mass=f8("mass", B),
            body_ipos=f8("ipos", B), body_iquat=f8("iquat", B), body_inertia_unit=f8("inertia_unit", B),
            jnt_type=i4("type", J), jnt_body=i4("body", J), jnt_qadr=i4("qadr", J), jnt_vadr=i4("vadr", J),
            jnt_axis=f8("axis", J), jnt_pos=f8("pos", J), jnt_damping=f8("damping", J), jnt_armature=f8("armature", J),
            geom_type=i4("type", G), geom_body=i4("body", G), geom_size=f8("size", G), geom_pos=f8("pos", G),
            geom_quat=f8("quat", G),
            pair_geom1=i4("g1", P), pair_geom2=i4("g2", P), pair_condim=i4("condim", P),
            pair_friction=f8("friction", P), pair_solref=f8("solref", P), pair_solimp=f8("solimp", P),
            pair_solimp_cfd=f8("solimp_cfd", P), pair_cfd_beta=f8("cfd_beta", P),
            act_type=i4("type", A), act_jnt=i4("jnt", A), act_gear=f8("gear", A), act_kp=f8("kp", A), act_kd=f8("kd", A),
            gravity=np.array(self.gravity, dtype=np.float64), newton_iters=self.newton_iters, ls_iters=self.ls_iters,
            qpos0=np.array(self.qpos0, dtype=np.float64),
        )


# per-unit-mass principal inertias of the primitives (input data, not method arithmetic)
def sphere_inertia(r):
    return (0.4 * r * r,) * 3


def box_inertia(hx, hy, hz):
    return ((hy * hy + hz * hz) / 3.0, (hx * hx + hz * hz) / 3.0, (hx * hx + hy * hy) / 3.0)


def capsule_inertia(r, hl):
    vc, vs = math.pi * r * r * 2 * hl, 4.0 / 3.0 * math.pi * r ** 3
    mc, ms = vc / (vc + vs), vs / (vc + vs)
    ixx = mc * (r * r / 4 + hl * hl / 3) + ms * (0.4 * r * r + hl * hl + 0.75 * r * hl)
    izz = mc * r * r / 2 + ms * 0.4 * r * r
    return (ixx, ixx, izz)


def default_opts(tableau=TSIT5, rtol=1e-6, atol=1e-6, h0=2e-3, max_steps=200000):
    """Solver options: P=0.2, I=0.4, safety .9, fac in [.2,10]."""
    return dict(tableau=tableau, rtol=rtol, atol=atol, h0=h0, pcoeff=0.2, icoeff=0.4, safety=0.9,
                fac_min=0.2, fac_max=10.0, max_steps=max_steps)


def _workload(name, model, x0, ctrl, nknot, knot_dt, horizon, opts, loss_grad, grad_targets, cfd):
    return dict(name=name, model=model, x0=np.ascontiguousarray(x0), ctrl=ctrl, nknot=nknot, knot_dt=knot_dt,
                horizon=horizon, opts=opts, loss_grad=loss_grad, grad_targets=grad_targets, cfd=cfd,
                nenv=x0.shape[0])


def ball_drop(nenv=1024, horizon=1.0, seed=250614186 + 1, gravity=-9.81, solref=(0.002, 1.0),
              solimp=SOLIMP_DEFAULT, rtol=1e-8):
    """C1 (shape of Fig. 20): 1-DoF ball on a slide joint dropped on a plane."""
    mb = ModelBuilder(gravity=(0, 0, gravity))
    b = mb.body(0, mass=1.0, inertia_unit=sphere_inertia(0.1))
    mb.joint(b, JNT_SLIDE, axis=(0, 0, 1))
    gp = mb.geom(0, GEOM_PLANE)
    gs = mb.geom(b, GEOM_SPHERE, size=(0.1,))
    mb.pair(gp, gs, condim=1, friction=0.0, solref=solref, solimp=solimp)
    rng = SplitMix64(seed)
    d = rng.uniform(2 * nenv).reshape(nenv, 2)
    x0 = np.stack([0.2 + 0.8 * d[:, 0], -2.0 + 4.0 * d[:, 1]], axis=1)

    def loss_grad(xT, x0_):
        g = np.zeros_like(xT); g[:, 0] = 1.0
        return xT[:, 0].copy(), g
    return _workload("C1_ball_drop", mb.build(), x0, None, 0, 0.0, horizon,
                     default_opts(DOPRI5, rtol, rtol), loss_grad, ("x0",), False)


_QY90 = (math.cos(math.pi / 4), 0.0, math.sin(math.pi / 4), 0.0)   # local z -> world x


def planar_push(nenv=4096, horizon=0.5, seed=250614186 + 2, cfd_model=True):
    """C2 (shape of Fig. 8): 2-link planar finger pushing a sphere on a frictional plane."""
    mb = ModelBuilder()
    L, rho = 0.3, 0.02
    l1 = mb.body(0, pos=(0, 0, 0.05), mass=0.2, ipos=(L / 2, 0, 0), iquat=_QY90, inertia_unit=capsule_inertia(rho, L / 2))
    j1 = mb.joint(l1, JNT_HINGE, axis=(0, 0, 1), damping=0.05)
    l2 = mb.body(l1, pos=(L, 0, 0), mass=0.2, ipos=(L / 2, 0, 0), iquat=_QY90, inertia_unit=capsule_inertia(rho, L / 2))
    j2 = mb.joint(l2, JNT_HINGE, axis=(0, 0, 1), damping=0.05)
    sp = mb.body(0, pos=(0.7, 0, 0.05), mass=0.1, inertia_unit=sphere_inertia(0.05))
    mb.joint(sp, JNT_FREE)
    gp = mb.geom(0, GEOM_PLANE)
    mb.geom(l1, GEOM_CAPSULE, size=(rho, L / 2), pos=(L / 2, 0, 0), quat=_QY90)
    mb.geom(l2, GEOM_CAPSULE, size=(rho, L / 2), pos=(L / 2, 0, 0), quat=_QY90)
    gt = mb.geom(l2, GEOM_SPHERE, size=(rho,), pos=(L, 0, 0))
    gs = mb.geom(sp, GEOM_SPHERE, size=(0.05,))
    simp = SOLIMP_CFD_ON if cfd_model else SOLIMP_DEFAULT
    mb.pair(gp, gs, condim=3, friction=0.8, solimp=simp)
    mb.pair(gt, gs, condim=3, friction=0.8, solimp=simp)
    mb.actuator(j1); mb.actuator(j2)
    nknot, knot_dt = int(round(horizon / 0.002)), 0.002
    rng = SplitMix64(seed)
    d = rng.uniform(4 * nenv).reshape(nenv, 4)
    th1, th2 = -0.5 + d[:, 0], -0.5 + d[:, 1]
    ahead, lat = 0.08 + 0.12 * d[:, 2], -0.05 + 0.1 * d[:, 3]
    a12 = th1 + th2
    tipx = L * np.cos(th1) + L * np.cos(a12); tipy = L * np.sin(th1) + L * np.sin(a12)
    sx = tipx + ahead * np.cos(a12) - lat * np.sin(a12); sy = tipy + ahead * np.sin(a12) + lat * np.cos(a12)
    x0 = np.zeros((nenv, 9 + 8))
    x0[:, 0], x0[:, 1], x0[:, 2], x0[:, 3], x0[:, 4], x0[:, 5] = th1, th2, sx, sy, 0.05, 1.0
    ctrl = rng.normal(nenv * nknot * 2, 0.5).reshape(nenv, nknot, 2)
    goal = np.array([0.6, 0.0])

    def loss_grad(xT, x0_):
        e = xT[:, 2:4] - goal
        g = np.zeros_like(xT); g[:, 2:4] = 2 * e
        return (e * e).sum(1), g
    return _workload("C2_planar_push", mb.build(), x0, np.ascontiguousarray(ctrl), nknot, knot_dt, horizon,
                     default_opts(TSIT5, 1e-6, 1e-6), loss_grad, ("ctrl",), True)


def cube_toss(nenv=8192, horizon=1.0, seed=250614186 + 3, mu=1.0, rtol=1e-6):
    """C3 (shape of Fig. 3/21; ContactNets cube): free box, 8 corner-plane contacts."""
    mb = ModelBuilder()
    c = mb.body(0, pos=(0, 0, 0.5), mass=0.37, inertia_unit=box_inertia(0.05, 0.05, 0.05))
    mb.joint(c, JNT_FREE)
    gp = mb.geom(0, GEOM_PLANE)
    gb = mb.geom(c, GEOM_BOX, size=(0.05, 0.05, 0.05))
    mb.pair(gp, gb, condim=3, friction=mu, solref=(0.001, 1.0), solimp=SOLIMP_DEFAULT)
    rng = SplitMix64(seed)
    quat = rng.normal(4 * nenv).reshape(nenv, 4)
    quat /= np.linalg.norm(quat, axis=1, keepdims=True)
    u = rng.uniform(6 * nenv).reshape(nenv, 6)
    x0 = np.zeros((nenv, 13))
    x0[:, 2] = 0.5; x0[:, 3:7] = quat
    x0[:, 7:10] = -3.0 + 6.0 * u[:, 0:3]; x0[:, 10:13] = -10.0 + 20.0 * u[:, 3:6]

    def loss_grad(xT, x0_):
        g = np.zeros_like(xT); g[:, 0] = 1.0
        return xT[:, 0].copy(), g                                   # reading G18
    return _workload("C3_cube_toss", mb.build(), x0, None, 0, 0.0, horizon,
                     default_opts(TSIT5, rtol, rtol), loss_grad, ("x0", "mu"), False)


def arm_target(nenv=16384, horizon=2.0, seed=250614186 + 4):
    """C4: 7-DoF hinge arm over a table plane plus a free sphere target; 12 candidate contacts."""
    mb = ModelBuilder()
    lens = [0.30, 0.30, 0.25, 0.25, 0.20, 0.15, 0.10]
    masses = [4, 3.5, 3, 2, 1.5, 1, 0.5]
    axes = [(0, 0, 1), (0, 1, 0)] * 3 + [(0, 0, 1)]
    rho = 0.03
    gp = mb.geom(0, GEOM_PLANE)
    parent, jn, caps = 0, [], []
    for i in range(7):
        pos = (0, 0, 0.35) if i == 0 else (0, 0, lens[i - 1])
        b = mb.body(parent, pos=pos, mass=masses[i], ipos=(0, 0, lens[i] / 2), inertia_unit=capsule_inertia(rho, lens[i] / 2))
        jn.append(mb.joint(b, JNT_HINGE, axis=axes[i], damping=0.1))
        caps.append(mb.geom(b, GEOM_CAPSULE, size=(rho, lens[i] / 2), pos=(0, 0, lens[i] / 2)))
        parent = b
    gtip = mb.geom(parent, GEOM_SPHERE, size=(rho,), pos=(0, 0, lens[6]))
    sp = mb.body(0, pos=(0.45, 0, 0.04), mass=0.2, inertia_unit=sphere_inertia(0.04))
    mb.joint(sp, JNT_FREE)
    gs = mb.geom(sp, GEOM_SPHERE, size=(0.04,))
    # d_o = 0 keeps the contact force continuous at r=0 (with d_o>0 the resting arm chatters
    # across the force jump and exhausts the step budget); CFD continuation d_0=0 -> d_c=0.01
    kw = dict(condim=3, friction=0.8, solimp=SOLIMP_DEFAULT, solimp_cfd=SOLIMP_CFD_SMOOTH)
    for i in range(2, 7):
        mb.pair(gp, caps[i], **kw)
    mb.pair(gtip, gs, **kw)
    mb.pair(gp, gs, **kw)
    for j in jn:
        mb.actuator(j)
    nknot, knot_dt = int(round(horizon / 0.01)), 0.01
    rng = SplitMix64(seed)
    d = rng.uniform(9 * nenv).reshape(nenv, 9)
    x0 = np.zeros((nenv, 14 + 13))
    x0[:, 0:7] = -0.8 + 1.6 * d[:, 0:7]
    x0[:, 7] = 0.3 + 0.3 * d[:, 7]; x0[:, 8] = -0.2 + 0.4 * d[:, 8]; x0[:, 9] = 0.04; x0[:, 10] = 1.0
    ctrl = rng.normal(nenv * nknot * 7, 1.0).reshape(nenv, nknot, 7)
    goal = np.array([0.5, 0.0, 0.04])

    def loss_grad(xT, x0_):
        e = xT[:, 7:10] - goal
        g = np.zeros_like(xT); g[:, 7:10] = 2 * e
        return (e * e).sum(1), g
    return _workload("C4_arm_target", mb.build(), x0, np.ascontiguousarray(ctrl), nknot, knot_dt, horizon,
                     default_opts(TSIT5, 1e-6, 1e-6), loss_grad, ("ctrl", "mass"), True)


def quadruped(nenv=4096, horizon=2.0, seed=250614186 + 5):
    """C5 (shape of Fig. 7): floating base + 12 hinges, 4 sphere feet on a plane."""
    mb = ModelBuilder()
    trunk = mb.body(0, pos=(0, 0, 0.335), mass=6.0, inertia_unit=box_inertia(0.2, 0.1, 0.05))
    mb.joint(trunk, JNT_FREE)
    gp = mb.geom(0, GEOM_PLANE)
    mb.geom(trunk, GEOM_BOX, size=(0.2, 0.1, 0.05))
    jn, feet = [], []
    for sx in (1, -1):
        for sy in (1, -1):
            ab = mb.body(trunk, pos=(0.2 * sx, 0.1 * sy, 0), mass=0.2, inertia_unit=sphere_inertia(0.03))
            jn.append(mb.joint(ab, JNT_HINGE, axis=(1, 0, 0), damping=0.05))
            th = mb.body(ab, mass=0.5, ipos=(0, 0, -0.1), inertia_unit=capsule_inertia(0.02, 0.1))
            jn.append(mb.joint(th, JNT_HINGE, axis=(0, 1, 0), damping=0.05))
            mb.geom(th, GEOM_CAPSULE, size=(0.02, 0.1), pos=(0, 0, -0.1))
            sh = mb.body(th, pos=(0, 0, -0.2), mass=0.3, ipos=(0, 0, -0.1), inertia_unit=capsule_inertia(0.02, 0.1))
            jn.append(mb.joint(sh, JNT_HINGE, axis=(0, 1, 0), damping=0.05))
            mb.geom(sh, GEOM_CAPSULE, size=(0.02, 0.1), pos=(0, 0, -0.1))
            feet.append(mb.geom(sh, GEOM_SPHERE, size=(0.02,), pos=(0, 0, -0.2)))
    for f in feet:
        mb.pair(gp, f, condim=3, friction=1.0, solref=(0.002, 1.0), solimp=SOLIMP_DEFAULT)
    for j in jn:
        mb.actuator(j, ACT_PD, kp=20.0, kd=0.5)
    nknot, knot_dt = int(round(horizon / 0.02)), 0.02
    stance = np.tile(np.array([0.0, 0.7, -1.4]), 4)
    rng = SplitMix64(seed)
    d = rng.uniform(12 * nenv).reshape(nenv, 12)
    x0 = np.zeros((nenv, 19 + 18))
    x0[:, 2] = 0.335; x0[:, 3] = 1.0
    x0[:, 7:19] = stance + (-0.05 + 0.1 * d)
    ctrl = stance + rng.normal(nenv * nknot * 12, 0.3).reshape(nenv, nknot, 12)

    def loss_grad(xT, x0_):
        g = np.zeros_like(xT); g[:, 0] = -1.0
        return -(xT[:, 0] - x0_[:, 0]), g
    return _workload("C5_quadruped", mb.build(), x0, np.ascontiguousarray(ctrl), nknot, knot_dt, horizon,
                     default_opts(TSIT5, 1e-5, 1e-5), loss_grad, ("ctrl",), False)


CONFIGS = dict(C1=ball_drop, C2=planar_push, C3=cube_toss, C4=arm_target, C5=quadruped)


def make(name, **kw):
    return CONFIGS[name](**kw)
