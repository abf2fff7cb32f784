// ORACLE — test infrastructure only (see oracle/README.md). Not part of the product path.
//
// O1/O2 of SURVEY.md §8(c): kinematics over the flattened tree, joint-space inertia M(q)
// and inverse dynamics ID(q,v,a) (Eq. 1: v' = M^-1 (tau - c + J^T f)).
// Written with plain 3-D rigid-body kinematics (every body carries origin position,
// rotation, angular velocity/acceleration and origin velocity/acceleration) and the
// principle of virtual work with the point Jacobian of SURVEY D3; M is the definition
// sum_b m Jc^T Jc + Jw^T I Jw (the quantity that composite-rigid-body computes).
#pragma once
#include "model.hpp"

namespace orc {

template <class S> struct Frame {
  V3<S> p;    // origin, world
  M3<S> R;    // orientation, world
  V3<S> w;    // angular velocity, world
  V3<S> al;   // angular acceleration, world
  V3<S> vp;   // velocity of the origin
  V3<S> ap;   // acceleration of the origin (inertial; gravity is applied as a force)
};

template <class S> struct Kin {
  std::vector<Frame<S>> fr;          // per body
  std::vector<V3<S>> dof_axis;       // per dof: world axis (hinge/slide), world unit vector
                                     // (free translation) or body axis R[:,k] (free rotation)
  std::vector<V3<S>> dof_anchor;     // per dof: world anchor (hinge) / body origin (free rotation)
  std::vector<V3<S>> com;            // per body: world centre of mass
};

template <class S> inline V3<S> vconst(const double* a) { return mk<S>(S(a[0]), S(a[1]), S(a[2])); }

// velocity / acceleration of a point x rigidly attached to frame f
template <class S> inline V3<S> point_vel(const Frame<S>& f, const V3<S>& x) { return f.vp + cross(f.w, x - f.p); }
template <class S> inline V3<S> point_acc(const Frame<S>& f, const V3<S>& x) {
  V3<S> d = x - f.p;
  return f.ap + cross(f.al, d) + cross(f.w, cross(f.w, d));
}

// Forward kinematics with first and second time derivatives.  q[nq], v[nv], a[nv]
// (a = joint accelerations; pass zeros for the bias force).  SURVEY O1, O2, G1.
template <class S>
void kinematics(const Model& m, const S* q, const S* v, const S* a, Kin<S>& k) {
  k.fr.resize(m.nbody); k.dof_axis.resize(m.nv); k.dof_anchor.resize(m.nv); k.com.resize(m.nbody);
  Frame<S>& w0 = k.fr[0];
  w0.p = mk<S>(S(0.0), S(0.0), S(0.0)); w0.R = eye<S>(); w0.w = w0.p; w0.al = w0.p; w0.vp = w0.p; w0.ap = w0.p;
  k.com[0] = w0.p;
  for (int b = 1; b < m.nbody; ++b) {
    const Frame<S>& par = k.fr[m.body_parent[b]];
    Frame<S> f;
    f.p = par.p + par.R * vconst<S>(&m.body_pos[3 * b]);
    f.R = par.R * quat_to_mat<S>(S(m.body_quat[4 * b]), S(m.body_quat[4 * b + 1]), S(m.body_quat[4 * b + 2]), S(m.body_quat[4 * b + 3]));
    f.w = par.w; f.al = par.al;
    f.vp = point_vel(par, f.p); f.ap = point_acc(par, f.p);
    int j = m.body_jnt[b];
    if (j >= 0) {
      int qa = m.jnt_qadr[j], va = m.jnt_vadr[j];
      if (m.jnt_type[j] == JNT_HINGE) {
        V3<S> ax = f.R * vconst<S>(&m.jnt_axis[3 * j]);
        V3<S> o = f.p + f.R * vconst<S>(&m.jnt_pos[3 * j]);
        V3<S> vo = point_vel(f, o), ao = point_acc(f, o);
        M3<S> Rot = axis_angle(ax, q[qa]);
        Frame<S> g;
        g.R = Rot * f.R;
        g.p = o + Rot * (f.p - o);
        g.w = f.w + ax * v[va];
        g.al = f.al + ax * a[va] + cross(f.w, ax) * v[va];
        V3<S> d = g.p - o;
        g.vp = vo + cross(g.w, d);
        g.ap = ao + cross(g.al, d) + cross(g.w, cross(g.w, d));
        f = g;
        k.dof_axis[va] = ax; k.dof_anchor[va] = o;
      } else if (m.jnt_type[j] == JNT_SLIDE) {
        V3<S> ax = f.R * vconst<S>(&m.jnt_axis[3 * j]);
        V3<S> s = ax * q[qa];
        Frame<S> g = f;
        g.p = f.p + s;
        g.vp = f.vp + cross(f.w, s) + ax * v[va];
        g.ap = f.ap + cross(f.al, s) + cross(f.w, cross(f.w, s)) + cross(f.w, ax) * (S(2.0) * v[va]) + ax * a[va];
        f = g;
        k.dof_axis[va] = ax; k.dof_anchor[va] = g.p;
      } else {  // JNT_FREE: position + unit quaternion; velocity = (world linear, body angular), G1
        f.p = mk<S>(q[qa], q[qa + 1], q[qa + 2]);
        f.R = quat_to_mat<S>(q[qa + 3], q[qa + 4], q[qa + 5], q[qa + 6]);
        f.vp = mk<S>(v[va], v[va + 1], v[va + 2]);
        f.ap = mk<S>(a[va], a[va + 1], a[va + 2]);
        f.w = f.R * mk<S>(v[va + 3], v[va + 4], v[va + 5]);
        f.al = f.R * mk<S>(a[va + 3], a[va + 4], a[va + 5]);  // d/dt(R w_b) = R w_b' + w x w
        for (int c = 0; c < 3; ++c) {
          k.dof_axis[va + c] = mk<S>(S(c == 0 ? 1.0 : 0.0), S(c == 1 ? 1.0 : 0.0), S(c == 2 ? 1.0 : 0.0));
          k.dof_anchor[va + c] = f.p;
          k.dof_axis[va + 3 + c] = col(f.R, c);
          k.dof_anchor[va + 3 + c] = f.p;
        }
      }
    }
    k.fr[b] = f;
    k.com[b] = f.p + f.R * vconst<S>(&m.body_ipos[3 * b]);
  }
}

// velocity of the world point x, fixed to body b, per unit rate of dof j
// (linear part) and the angular velocity of body b per unit rate of dof j.
template <class S>
inline void dof_twist(const Model& m, const Kin<S>& k, int j, int b, const V3<S>& x, V3<S>& lin, V3<S>& ang) {
  V3<S> zero = mk<S>(S(0.0), S(0.0), S(0.0));
  lin = zero; ang = zero;
  if (!m.is_ancestor_or_self(m.dof_body[j], b)) return;
  int jt = m.jnt_type[m.dof_jnt[j]];
  if (jt == JNT_HINGE) { ang = k.dof_axis[j]; lin = cross(k.dof_axis[j], x - k.dof_anchor[j]); }
  else if (jt == JNT_SLIDE) { lin = k.dof_axis[j]; }
  else {
    int c = j - m.jnt_vadr[m.dof_jnt[j]];
    if (c < 3) lin = k.dof_axis[j];
    else { ang = k.dof_axis[j]; lin = cross(k.dof_axis[j], x - k.dof_anchor[j]); }
  }
}

// world inertia tensor about the centre of mass; mass[] are the per-env masses (params)
template <class S>
inline M3<S> world_inertia(const Model& m, const Kin<S>& k, int b, const S& mass) {
  M3<S> Ri = k.fr[b].R * quat_to_mat<S>(S(m.body_iquat[4 * b]), S(m.body_iquat[4 * b + 1]), S(m.body_iquat[4 * b + 2]), S(m.body_iquat[4 * b + 3]));
  M3<S> Dg;
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) Dg.m[i][j] = Ri.m[i][j] * (mass * S(m.body_inertia_unit[3 * b + j]));
  return Dg * transpose(Ri);
}

// Inverse dynamics ID(q,v,a) = M a + c(q,v), gravity included.
template <class S>
void inverse_dynamics(const Model& m, const S* q, const S* v, const S* a, const S* mass, S* out) {
  Kin<S> k; kinematics(m, q, v, a, k);
  V3<S> g = vconst<S>(m.gravity);
  for (int j = 0; j < m.nv; ++j) out[j] = S(m.jnt_armature[m.dof_jnt[j]]) * a[j];
  for (int b = 1; b < m.nbody; ++b) {
    const Frame<S>& f = k.fr[b];
    V3<S> ac = point_acc(f, k.com[b]);
    V3<S> Fb = (ac - g) * mass[b];                         // Newton
    M3<S> I = world_inertia(m, k, b, mass[b]);
    V3<S> Nb = I * f.al + cross(f.w, I * f.w);             // Euler, about the centre of mass
    for (int j = 0; j < m.nv; ++j) {
      V3<S> lin, ang; dof_twist(m, k, j, b, k.com[b], lin, ang);
      out[j] = out[j] + dot(lin, Fb) + dot(ang, Nb);       // virtual work
    }
  }
}

// M(q) = sum_b m Jc^T Jc + Jw^T I Jw + diag(armature); dense row-major nv*nv.
template <class S>
void mass_matrix(const Model& m, const S* q, const S* mass, S* M) {
  std::vector<S> zero(m.nv, S(0.0));
  Kin<S> k; kinematics(m, q, zero.data(), zero.data(), k);
  for (int i = 0; i < m.nv * m.nv; ++i) M[i] = S(0.0);
  for (int j = 0; j < m.nv; ++j) M[j * m.nv + j] = S(m.jnt_armature[m.dof_jnt[j]]);
  std::vector<V3<S>> lin(m.nv), ang(m.nv);
  for (int b = 1; b < m.nbody; ++b) {
    M3<S> I = world_inertia(m, k, b, mass[b]);
    for (int j = 0; j < m.nv; ++j) dof_twist(m, k, j, b, k.com[b], lin[j], ang[j]);
    for (int i = 0; i < m.nv; ++i) for (int j = 0; j < m.nv; ++j)
      M[i * m.nv + j] = M[i * m.nv + j] + mass[b] * dot(lin[i], lin[j]) + dot(ang[i], I * ang[j]);
  }
}

// tau(x,a): actuators (motor: gear*u; PD: kp(u-q_j) - kd v_j) and joint damping.  SURVEY O2/S3.
template <class S>
void applied_force(const Model& m, const S* q, const S* v, const S* u, S* tau) {
  for (int j = 0; j < m.nv; ++j) tau[j] = -(S(m.jnt_damping[m.dof_jnt[j]]) * v[j]);
  for (int i = 0; i < m.nu; ++i) {
    int jn = m.act_jnt[i], va = m.jnt_vadr[jn], qa = m.jnt_qadr[jn];
    if (m.act_type[i] == ACT_MOTOR) tau[va] = tau[va] + S(m.act_gear[i]) * u[i];
    else tau[va] = tau[va] + S(m.act_kp[i]) * (u[i] - q[qa]) - S(m.act_kd[i]) * v[va];
  }
}

}  // namespace orc
