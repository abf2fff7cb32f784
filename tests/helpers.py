"""Small model builders and finite-difference helpers shared by the tests (inputs only)."""
import math
import numpy as np
from paper_2506_14186_b200 import workloads as W


def oscillator(m=1.3, kp=7.0):
    """Slide-joint mass with a PD actuator (kd=0), no gravity: m q'' = kp (u - q)."""
    mb = W.ModelBuilder(gravity=(0, 0, 0))
    b = mb.body(0, mass=m, inertia_unit=(1, 1, 1))
    j = mb.joint(b, W.JNT_SLIDE, axis=(0, 0, 1))
    mb.actuator(j, W.ACT_PD, kp=kp, kd=0.0)
    return mb.build()


def free_box(half=(0.05, 0.08, 0.13), mass=0.7, gravity=(0, 0, 0), with_plane=False, mu=0.6, solref=(0.004, 1.0),
             solimp=W.SOLIMP_DEFAULT):
    mb = W.ModelBuilder(gravity=gravity)
    c = mb.body(0, pos=(0, 0, 0.5), mass=mass, ipos=(0.01, -0.02, 0.005), inertia_unit=W.box_inertia(*half))
    mb.joint(c, W.JNT_FREE)
    if with_plane:
        gp = mb.geom(0, W.GEOM_PLANE)
        gb = mb.geom(c, W.GEOM_BOX, size=half)
        mb.pair(gp, gb, condim=3, friction=mu, solref=solref, solimp=solimp)
    return mb.build()


def arm(n=3, gravity=(0, 0, -9.81), damping=0.0, with_contacts=False, slide_last=False):
    """Serial chain with alternating axes, oblique frames and offset COMs."""
    mb = W.ModelBuilder(gravity=gravity)
    axes = [(0, 0, 1), (0, 1, 0), (1, 0, 0), (0, 0.6, 0.8)]
    parent, gp = 0, None
    caps = []
    for i in range(n):
        quat = np.array([1.0, 0.1 * i, -0.05, 0.07 * i]); quat /= np.linalg.norm(quat)
        b = mb.body(parent, pos=(0.05, 0.02 * i, 0.3 if i else (0.12 if with_contacts else 0.4)), quat=tuple(quat), mass=1.0 + 0.5 * i,
                    ipos=(0.01, 0.02, 0.12), iquat=(math.cos(0.3), 0, math.sin(0.3), 0), inertia_unit=(0.01, 0.02, 0.005))
        jt = W.JNT_SLIDE if (slide_last and i == n - 1) else W.JNT_HINGE
        mb.joint(b, jt, axis=axes[i % 4], pos=(0.0, 0.01, -0.02), damping=damping, armature=0.01 * (i == 1))
        caps.append((b, mb.geom(b, W.GEOM_CAPSULE, size=(0.03, 0.12), pos=(0, 0, 0.12))))
        parent = b
    if with_contacts:
        gp = mb.geom(0, W.GEOM_PLANE)
        for b, g in caps[1:]:
            mb.pair(gp, g, condim=3, friction=0.7, solref=(0.01, 1.0), solimp=(0.1, 0.9, 0.01, 0.5, 2))
    for j in range(n):
        mb.actuator(j)
    return mb.build()


def two_spheres(gravity=(0, 0, 0), solimp=W.SOLIMP_CFD_ON, solref=(0.01, 1.0), mu=0.5):
    """Billiard-like: two free spheres, sphere-sphere pair only."""
    mb = W.ModelBuilder(gravity=gravity)
    a = mb.body(0, pos=(0, 0, 0), mass=0.17, inertia_unit=W.sphere_inertia(0.03))
    mb.joint(a, W.JNT_FREE)
    b = mb.body(0, pos=(0.3, 0, 0), mass=0.17, inertia_unit=W.sphere_inertia(0.03))
    mb.joint(b, W.JNT_FREE)
    ga = mb.geom(a, W.GEOM_SPHERE, size=(0.03,))
    gb = mb.geom(b, W.GEOM_SPHERE, size=(0.03,))
    mb.pair(ga, gb, condim=3, friction=mu, solref=solref, solimp=solimp, solimp_cfd=(0.0, solimp[0], 0.2, 1.0, 4.0))
    return mb.build()


def rand_quat(rng):
    q = rng.normal(size=4)
    return q / np.linalg.norm(q)


def perturb_x(orc, x, d, eps):
    """x (+) eps e_d in tangent coordinates (d < nv: configuration, else velocity)."""
    nq, nv = orc.nq, orc.nv
    y = x.copy()
    if d < nv:
        delta = np.zeros(nv); delta[d] = eps
        y[:nq] = orc.retract(x[:nq], delta)
    else:
        y[nq + d - nv] += eps
    return y
