// dmx_field.cuh — the vector field F_theta(t,x) of PAPER.md Eq. (1)/(5) and its CFD variant F~
// as lane-group device code:
//   S1 forward kinematics, S2 mass matrix + Cholesky, S3 bias / applied forces, S4 narrow phase,
//   S5 constraint rows (Eq. 3, impedance, regulariser), S6 fixed-iteration Newton contact solve
//   (Eq. 2), and S11/S12 the vector-Jacobian product by implicit differentiation of the
//   stationarity condition at the final active set (PAPER.md:543 suggests implicit
//   differentiation).
#pragma once
#include "dmx_model.cuh"

namespace dmx {

// ---- inputs of one evaluation -----------------------------------------------------------------
template <class R, int ST> struct InPlain {
  typedef R S;
  Arr<R, ST> qa, va, aa; const R* ua; const R* pa;
  DMX_DI R q(int i) const { return qa[i]; }
  DMX_DI R v(int i) const { return va[i]; }
  DMX_DI R a(int i) const { return aa[i]; }
  DMX_DI R u(int i) const { return ua[i]; }
  DMX_DI R p(int i) const { return pa[i]; }
};
// parameters carrying one tangent direction (index idx; idx < 0: none), for the candidate scalars of the VJP
template <class R, int ST> struct InDual {
  typedef Dual<R> S;
  const R* pa; int kind, idx;
  DMX_DI S p(int i) const { return S(pa[i], (i == idx) ? R(1) : R(0)); }
};

template <class S> struct FrameT { V3<S> p; M3<S> R; V3<S> w, al, vp, ap; };

template <class S> DMX_DI V3<S> point_vel(const FrameT<S>& f, const V3<S>& x) { return f.vp + cross(f.w, x - f.p); }
template <class S> DMX_DI V3<S> point_acc(const FrameT<S>& f, const V3<S>& x) {
  V3<S> d = x - f.p;
  return f.ap + cross(f.al, d) + cross(f.w, cross(f.w, d));
}

// ---- S1: forward kinematics with first and second time derivatives ---------------
// One body: frame from the parent's frame and the body's joint.  ACC: joint accelerations in.a
// enter (inverse dynamics at a given acceleration); otherwise they are zero (bias force).
template <class WS, class R, class IN, bool ACC>
DMX_DI void body_kin(const ModelDev<R>& m, const IN& in, const WS& ws, int b) {
  typedef typename WS::S S;
  int par = m.body_parent[b];
  FrameT<S> P;
  P.p = ld3(ws.fp(), par); P.R = ld9(ws.fR(), par); P.w = ld3(ws.fw(), par); P.al = ld3(ws.fal(), par);
  P.vp = ld3(ws.fvp(), par); P.ap = ld3(ws.fap(), par);
  FrameT<S> f;
  f.p = P.p + P.R * c3<S>(m.body_pos, b);
  f.R = P.R * c9<S>(m.body_rot, b);
  f.w = P.w; f.al = P.al;
  f.vp = point_vel(P, f.p); f.ap = point_acc(P, f.p);
  int j = m.body_jnt[b];
  if (j >= 0) {
    int qa = m.jnt_qadr[j], va = m.jnt_vadr[j], jt = m.jnt_type[j];
    if (jt == JNT_HINGE) {
      V3<S> ax = f.R * c3<S>(m.jnt_axis, j);
      V3<S> o = f.p + f.R * c3<S>(m.jnt_pos, j);
      V3<S> vo = point_vel(f, o), ao = point_acc(f, o);
      M3<S> Rot = axis_angle(ax, in.q(qa));
      S vj = in.v(va);
      FrameT<S> g;
      g.R = Rot * f.R;
      g.p = o + Rot * (f.p - o);
      g.w = f.w + ax * vj;
      g.al = f.al + cross(f.w, ax) * vj;
      if (ACC) g.al = g.al + ax * in.a(va);
      V3<S> d = g.p - o;
      g.vp = vo + cross(g.w, d);
      g.ap = ao + cross(g.al, d) + cross(g.w, cross(g.w, d));
      f = g;
      st3(ws.dax(), va, ax); st3(ws.dan(), va, o);
    } else if (jt == JNT_SLIDE) {
      V3<S> ax = f.R * c3<S>(m.jnt_axis, j);
      V3<S> s = ax * in.q(qa);
      S vj = in.v(va);
      V3<S> np = f.p + s;
      V3<S> nvp = f.vp + cross(f.w, s) + ax * vj;
      V3<S> nap = f.ap + cross(f.al, s) + cross(f.w, cross(f.w, s)) + cross(f.w, ax) * (S(2.0) * vj);
      if (ACC) nap = nap + ax * in.a(va);
      f.p = np; f.vp = nvp; f.ap = nap;
      st3(ws.dax(), va, ax); st3(ws.dan(), va, np);
    } else {  // free joint: world linear velocity, body angular velocity
      f.p = mk3<S>(in.q(qa), in.q(qa + 1), in.q(qa + 2));
      f.R = quat_to_mat<S>(in.q(qa + 3), in.q(qa + 4), in.q(qa + 5), in.q(qa + 6));
      f.vp = mk3<S>(in.v(va), in.v(va + 1), in.v(va + 2));
      f.w = f.R * mk3<S>(in.v(va + 3), in.v(va + 4), in.v(va + 5));
      S z(0.0);
      if (ACC) {
        f.ap = mk3<S>(in.a(va), in.a(va + 1), in.a(va + 2));
        f.al = f.R * mk3<S>(in.a(va + 3), in.a(va + 4), in.a(va + 5));
      } else { f.ap = mk3<S>(z, z, z); f.al = f.ap; }
      S one(1.0);
      st3(ws.dax(), va, mk3<S>(one, z, z)); st3(ws.dax(), va + 1, mk3<S>(z, one, z)); st3(ws.dax(), va + 2, mk3<S>(z, z, one));
#pragma unroll
      for (int c = 0; c < 3; ++c) { st3(ws.dan(), va + c, f.p); st3(ws.dax(), va + 3 + c, colv(f.R, c)); st3(ws.dan(), va + 3 + c, f.p); }
    }
  }
  st3(ws.fp(), b, f.p); st9(ws.fR(), b, f.R); st3(ws.fw(), b, f.w); st3(ws.fal(), b, f.al); st3(ws.fvp(), b, f.vp); st3(ws.fap(), b, f.ap);
  st3(ws.com(), b, f.p + f.R * c3<S>(m.body_ipos, b));
}

// Bodies of one tree level are independent: one lane per body, levels in order.
template <class WS, class R, int G, class IN, bool ACC>
DMX_DN void kinematics(const ModelDev<R>& m, const IN& in, const WS& ws, const Grp<G>& gr) {
  typedef typename WS::S S;
  if (gr.lane == 0) {
    S z(0.0), o(1.0);
    V3<S> z3 = mk3<S>(z, z, z);
    st3(ws.fp(), 0, z3); st3(ws.fw(), 0, z3); st3(ws.fal(), 0, z3); st3(ws.fvp(), 0, z3); st3(ws.fap(), 0, z3); st3(ws.com(), 0, z3);
    M3<S> I; for (int k = 0; k < 9; ++k) I.m[k] = (k % 4 == 0) ? o : z;
    st9(ws.fR(), 0, I);
  }
  gr.sync();
#pragma unroll 1
  for (int lv = 0; lv < m.nlevel; ++lv) {
#pragma unroll 1
    for (int i = m.level_ptr[lv] + gr.lane; i < m.level_ptr[lv + 1]; i += G) body_kin<WS, R, IN, ACC>(m, in, ws, m.level_body[i]);
    gr.sync();
  }
}

// linear velocity of the world point x fixed to a body per unit rate of dof j (j on the body's
// path to the world)
template <class WS> DMX_DI V3<typename WS::S> twist_lin(const WS& ws, int j, int rot, const V3<typename WS::S>& x) {
  typedef typename WS::S S;
  V3<S> ax = ld3(ws.dax(), j);
  if (!rot) return ax;
  return cross(ax, x - ld3(ws.dan(), j));
}

// Newton-Euler wrench of body b about its centre of mass and its world inertia
template <class WS, class R, class IN>
DMX_DI void body_wrench(const ModelDev<R>& m, const IN& in, const WS& ws, int b, V3<typename WS::S>& Fb, V3<typename WS::S>& Nb, M3<typename WS::S>& Iw) {
  typedef typename WS::S S;
  FrameT<S> f;
  f.p = ld3(ws.fp(), b); f.R = ld9(ws.fR(), b); f.w = ld3(ws.fw(), b); f.al = ld3(ws.fal(), b); f.ap = ld3(ws.fap(), b);
  S mass = in.p(b);
  V3<S> ac = point_acc(f, ld3(ws.com(), b));
  Fb = (ac - mk3<S>(S(m.gravity[0]), S(m.gravity[1]), S(m.gravity[2]))) * mass;
  M3<S> Ri = f.R * c9<S>(m.body_irot, b);
  M3<S> Dg;
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) Dg.m[3 * i + j] = Ri.m[3 * i + j] * (mass * S(m.body_iunit[3 * b + j]));
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) Iw.m[3 * i + j] = Dg.m[3 * i] * Ri.m[3 * j] + Dg.m[3 * i + 1] * Ri.m[3 * j + 1] + Dg.m[3 * i + 2] * Ri.m[3 * j + 2];
  Nb = Iw * f.al + cross(f.w, Iw * f.w);
}

// ---- S2/S3: M(q), c(q,v), tau(x,u) ---------------------------------------------
// M = sum_b m Jc^T Jc + Jw^T I Jw + diag(armature): the linear part is summed over the subtree
// below the deeper dof from a (body, ancestor-dof) twist table; the angular part uses the summed
// world inertias of that subtree.  c_j = sum_b lin_jb . F_b + ang_j . N_b (virtual work).
template <class WS, class R, int G, class IN>
DMX_DN void dynamics(const ModelDev<R>& m, const IN& in, const WS& ws, const Grp<G>& gr) {
  const int ld = ws.ld();
  typedef typename WS::S S;
  const int nv = ws.nv(m), nb = m.nbody;
#pragma unroll 1
  for (int b = 1 + gr.lane; b < nb; b += G) {
    V3<S> Fb, Nb; M3<S> Iw;
    body_wrench<WS, R, IN>(m, in, ws, b, Fb, Nb, Iw);
    st3(ws.Fb(), b, Fb); st3(ws.Nb(), b, Nb); st9(ws.Iw(), b, Iw);
  }
#pragma unroll 1
  for (int e = gr.lane; e < m.ntw; e += G) {
    int j = m.tw_dof[e];
    st3(ws.tw(), e, twist_lin(ws, j, m.dof_rot[j], ld3(ws.com(), m.tw_body[e])));
  }
  gr.sync();
#pragma unroll 1
  for (int i = gr.lane; i < 9 * (nb - 1); i += G) {
    int b = 1 + i / 9, k = i % 9;
    S acc(0.0);
#pragma unroll 1
    for (int t = m.sub_ptr[b]; t < m.sub_ptr[b + 1]; ++t) acc = acc + ws.Iw()[9 * m.sub_body[t] + k];
    ws.Isub()[9 * b + k] = acc;
  }
  gr.sync();
#pragma unroll 1
  for (int e = gr.lane; e < m.nmp; e += G) {
    int i = m.mp_i[e], j = m.mp_j[e], deep = m.mp_deep[e];
    S acc(0.0);
    if (deep >= 0) {
#pragma unroll 1
      for (int t = m.sub_ptr[deep]; t < m.sub_ptr[deep + 1]; ++t) {
        int b = m.sub_body[t];
        acc = acc + in.p(b) * dot(ld3(ws.tw(), m.tw_idx[b * nv + i]), ld3(ws.tw(), m.tw_idx[b * nv + j]));
      }
      if (m.dof_rot[i] && m.dof_rot[j]) acc = acc + dot(ld3(ws.dax(), i), ld9(ws.Isub(), deep) * ld3(ws.dax(), j));
      if (i == j) acc = acc + S(m.jnt_armature[m.dof_jnt[i]]);
    }
    ws.M()[i * ld + j] = acc; ws.M()[j * ld + i] = acc;
  }
#pragma unroll 1
  for (int j = gr.lane; j < nv; j += G) {
    int bj = m.dof_body[j], rot = m.dof_rot[j];
    V3<S> ax = ld3(ws.dax(), j);
    S acc(0.0);
#pragma unroll 1
    for (int t = m.sub_ptr[bj]; t < m.sub_ptr[bj + 1]; ++t) {
      int b = m.sub_body[t];
      acc = acc + dot(ld3(ws.tw(), m.tw_idx[b * nv + j]), ld3(ws.Fb(), b));
      if (rot) acc = acc + dot(ax, ld3(ws.Nb(), b));
    }
    ws.c()[j] = acc;
    S tau = -(S(m.jnt_damping[m.dof_jnt[j]]) * in.v(j));
#pragma unroll 1
    for (int i = 0; i < m.nu; ++i) {
      int jn = m.act_jnt[i];
      if (m.jnt_vadr[jn] != j) continue;
      if (m.act_type[i] == ACT_MOTOR) tau = tau + S(m.act_gear[i]) * in.u(i);
      else tau = tau + S(m.act_kp[i]) * (in.u(i) - in.q(m.jnt_qadr[jn])) - S(m.act_kd[i]) * in.v(j);
    }
    ws.tau()[j] = tau;
  }
  gr.sync();
}

// (a, b), b <= a, of the e-th entry of a row-major lower triangle
DMX_DI void tri_index(int e, int& a, int& b) {
  a = (int)((sqrtf(8.0f * (float)e + 1.0f) - 1.0f) * 0.5f);
  if ((a + 1) * (a + 2) / 2 <= e) ++a;
  if (a * (a + 1) / 2 > e) --a;
  b = e - a * (a + 1) / 2;
}

// ---- dense Cholesky on the lower triangle, one column at a time, lanes over rows ---------------
// The factor is stored with the RECIPROCAL of its diagonal (l_jj^-1 = rsqrt of the pivot), so the column scaling
// and both substitutions multiply instead of divide: the dependent chain per column is one rsqrt, not sqrt + div.
// With n <= G lane i owns row i: the pivot travels by shuffle and every lane scales its own entry, so a column costs one
// group barrier instead of three (same operations per entry: bitwise the result of the general version below).
template <class S, int ST, int G> DMX_DN bool cholesky(const Arr<S, ST>& A, int n, int ld, const Grp<G>& gr) {
  if (G > 1 && n <= G) {
    const int i = gr.lane;
#pragma unroll 1
    for (int j = 0; j < n; ++j) {
      const bool act = i >= j && i < n;
      S t(0.0);
      if (act) {
        t = A[i * ld + j];
#pragma unroll 4
        for (int k = 0; k < j; ++k) t = t - A[i * ld + k] * A[j * ld + k];
      }
      S s = gr.from_lane(t, j);
      if (!(val(s) > 0)) return false;       // uniform over the group
      S il = m_rsqrt(s);
      if (act) A[i * ld + j] = (i == j) ? il : t * il;
      gr.sync();
    }
    return true;
  }
#pragma unroll 1
  for (int j = 0; j < n; ++j) {
#pragma unroll 1
    for (int i = j + gr.lane; i < n; i += G) {
      S t = A[i * ld + j];
#pragma unroll 4
      for (int k = 0; k < j; ++k) t = t - A[i * ld + k] * A[j * ld + k];
      A[i * ld + j] = t;
    }
    gr.sync();
    S s = A[j * ld + j];
    if (!(val(s) > 0)) return false;       // uniform over the group
    S il = m_rsqrt(s);
    gr.sync();
#pragma unroll 1
    for (int i = j + gr.lane; i < n; i += G) A[i * ld + j] = (i == j) ? il : A[i * ld + j] * il;
    gr.sync();
  }
  return true;
}
// b <- (L L^T)^-1 b; column-oriented substitutions (diagonal of L holds reciprocals)
// With n <= G the right-hand side lives in registers, one entry per lane, and the pivot entry travels by shuffle: the
// dependent chain per column is shuffle + multiply + fma instead of shared load + multiply + fma + store + group barrier
// (same operations on every entry in the same order, so the result is bitwise that of the shared-memory version).
template <class S, int ST, int G> DMX_DN void chol_solve(const Arr<S, ST>& L, int n, int ld, const Arr<S, ST>& b, const Grp<G>& gr) {
  if (G > 1 && n <= G) {
    const int k = gr.lane;
    const bool in = k < n;
    S bk = in ? b[k] : S(0.0);
#pragma unroll 1
    for (int i = 0; i < n; ++i) {
      S bi = gr.from_lane(bk, i) * L[i * ld + i];
      if (in && k > i) bk = bk - L[k * ld + i] * bi;
      else if (k == i) bk = bi;
    }
#pragma unroll 1
    for (int i = n - 1; i >= 0; --i) {
      S bi = gr.from_lane(bk, i) * L[i * ld + i];
      if (k < i) bk = bk - L[i * ld + k] * bi;
      else if (k == i) bk = bi;
    }
    if (in) b[k] = bk;
    gr.sync();
    return;
  }
#pragma unroll 1
  for (int i = 0; i < n; ++i) {
    S bi = b[i] * L[i * ld + i];
#pragma unroll 1
    for (int k = i + 1 + gr.lane; k < n; k += G) b[k] = b[k] - L[k * ld + i] * bi;
    gr.sync();
  }
#pragma unroll 1
  for (int i = gr.lane; i < n; i += G) b[i] = b[i] * L[i * ld + i];
  gr.sync();
#pragma unroll 1
  for (int i = n - 1; i >= 0; --i) {
    S bi = b[i] * L[i * ld + i];
#pragma unroll 1
    for (int k = gr.lane; k < i; k += G) b[k] = b[k] - L[i * ld + k] * bi;
    gr.sync();
  }
#pragma unroll 1
  for (int i = gr.lane; i < n; i += G) b[i] = b[i] * L[i * ld + i];
  gr.sync();
}

// ---- S5: impedance d(r) from solimp (spline: SURVEY G5) and the CFD continuation --
// general exponent: one out-of-line copy (pow is ~300 instructions; the BASELINE configs use power = 2)
template <class S> __device__ __noinline__ S imp_spline_pow(S x, S mid, S power) {
  S one(1.0);
  if (val(x) <= val(mid)) return m_pow(x, power) / m_pow(mid, power - one);
  return one - m_pow(one - x, power) / m_pow(one - mid, power - one);
}
template <class S> DMX_DI S int_pow(const S& x, int n) { S r = x; for (int k = 1; k < n; ++k) r = r * x; return r; }   // n >= 1
template <class S> DMX_DI S imp_spline(const S& x, const S& mid, const S& power) {
  if (val(x) <= 0) return S(0.0) * x;
  if (val(x) >= 1) return S(1.0) + S(0.0) * x;
  S one(1.0);
  const int n = (int)val(power);
  if (n >= 2 && n <= 8 && val(power) == (double)n && !has_tangent(power)) {   // integer exponent (2: PAPER.md:347, 537; 4: the CFD
    if (val(x) <= val(mid)) return int_pow(x, n) / int_pow(mid, n - 1);       // spline): products instead of pow
    return one - int_pow(one - x, n) / int_pow(one - mid, n - 1);
  }
  return imp_spline_pow<S>(x, mid, power);
}
template <class S> DMX_DI S clamp_imp(S d) {
  if (val(d) < 0) d = S(0.0);
  if (val(d) > 1.0 - 1e-4) d = S(1.0 - 1e-4);
  return d;
}
template <class S> DMX_DI S impedance(const S& r, const S& d_o, const S& d_w, const S& w, const S& mid, const S& power) {
  S ar = val(r) < 0 ? -r : r;
  S x = ar / w;
  if (val(x) > 1) x = S(1.0);
  return clamp_imp(d_o + imp_spline(x, mid, power) * (d_w - d_o));
}
template <class S, class R> DMX_DI S impedance_cfd(const S& r, const R* sc) {   // (d_c, d_0, w_c, m_c, p_c)
  S x = r / S(sc[2]);
  return clamp_imp(S(sc[1]) + imp_spline(x, S(sc[3]), S(sc[4])) * S(sc[0] - sc[1]));
}
template <class S, class R> DMX_DI S softplus(const S& z, R beta) {
  S bz = z * S(beta), one(1.0);
  if (val(bz) > 0) return z + m_log(one + m_exp(-bz)) / S(beta);
  return m_log(one + m_exp(bz)) / S(beta);
}

// ---- S4: narrow phase of one flattened candidate ----------
template <class S> struct GeoT { S r; V3<S> n, pos, t1, t2; };
template <class WS, class R> DMX_DI GeoT<typename WS::S> collide(const ModelDev<R>& m, const WS& ws, int c) {
  typedef typename WS::S S;
  GeoT<S> g;
  int b2 = m.ct_b2[c];
  V3<S> c2 = ld3(ws.fp(), b2) + ld9(ws.fR(), b2) * c3<S>(m.ct_p2, c);
  S rho2(m.ct_rho2[c]);
  if (m.ct_kind[c] == CK_POINT_PLANE) {
    g.n = c3<S>(m.ct_n, c); g.t1 = c3<S>(m.ct_t1, c); g.t2 = c3<S>(m.ct_t2, c);
    g.r = dot(g.n, c2 - c3<S>(m.ct_p1, c)) - rho2;
    g.pos = c2 - g.n * (rho2 + S(0.5) * g.r);
  } else {
    int b1 = m.ct_b1[c];
    V3<S> c1 = ld3(ws.fp(), b1) + ld9(ws.fR(), b1) * c3<S>(m.ct_p1, c);
    V3<S> dl = c2 - c1;
    S dist = m_sqrt(dot(dl, dl)), rho1(m.ct_rho1[c]);
    g.n = dl * (S(1.0) / dist);
    g.r = dist - rho1 - rho2;
    g.pos = c1 + g.n * (rho1 + S(0.5) * g.r);
    typename RealOf<S>::type ax = fabs(val(g.n.x)), ay = fabs(val(g.n.y)), az = fabs(val(g.n.z));
    int e = 0; if (ay < ax) { e = 1; ax = ay; } if (az < ax) e = 2;
    S z(0.0), o(1.0);
    V3<S> ev = mk3<S>(e == 0 ? o : z, e == 1 ? o : z, e == 2 ? o : z);
    V3<S> t = ev - g.n * dot(ev, g.n);
    g.t1 = t * (S(1.0) / m_sqrt(dot(t, t)));
    g.t2 = cross(g.n, g.t1);
  }
  return g;
}

// per-candidate scalars of Eq. 3 and the regulariser: D = d / (A^ (1-d)), position term of a_ref,
// damping coefficient b.  cfd: impedance continued for r>0 and softplus.
template <class S, class R, class IN>
DMX_DI void candidate_terms(const ModelDev<R>& m, const IN& in, int c, const S& r, bool cfd, S& Dw, S& post, S& bdamp, S& mu) {
  int pr = m.ct_pair[c];
  int o = m.p_solimp + 5 * pr;
  S d_o = in.p(o), d_w = in.p(o + 1), wid = in.p(o + 2), mid = in.p(o + 3), pw = in.p(o + 4);
  S tc = in.p(m.p_solref + 2 * pr), phi = in.p(m.p_solref + 2 * pr + 1);
  mu = in.p(m.p_fric + pr);
  S kden = d_w * d_w * tc * tc * phi * phi;
  S d;
  if (cfd) {
    d = val(r) > 0 ? impedance_cfd<S, R>(r, m.pair_solimp_cfd + 5 * pr) : impedance(r, d_o, d_w, wid, mid, pw);
    post = (d / kden) * softplus<S, R>(-r, m.pair_cfd_beta[pr]);
  } else {
    d = impedance(r, d_o, d_w, wid, mid, pw);
    post = -((d / kden) * r);
  }
  bdamp = S(2.0) / (d_w * tc);
  S Ahat(m.pair_invweight[pr]);
  if (m.ct_condim[c] == 3) Ahat = Ahat * (S(1.0) + mu * mu);
  Dw = d / (Ahat * (S(1.0) - d));
}

// one shared copy of the tangent-scalar evaluation of the candidate terms (impedance spline, softplus: large code)
template <class R, class IN>
__device__ __noinline__ void candidate_terms_dual(const ModelDev<R>& m, const IN& in, int c, Dual<R> r, bool cfd, Dual<R>& Dw, Dual<R>& post,
                                                  Dual<R>& bd, Dual<R>& mu) {
  candidate_terms<Dual<R>, R, IN>(m, in, c, r, cfd, Dw, post, bd, mu);
}

// relative velocity of the contact point per unit rate of dof j, body2 minus body1
template <class WS, class R>
DMX_DI V3<typename WS::S> rel_twist(const ModelDev<R>& m, const WS& ws, int j, int b1, int b2, const V3<typename WS::S>& pos) {
  typedef typename WS::S S;
  S z(0.0);
  V3<S> d = mk3<S>(z, z, z);
  int rot = m.dof_rot[j];
  const int nv = ws.nv(m);
  if (m.tw_idx[b2 * nv + j] >= 0) d = twist_lin(ws, j, rot, pos);
  if (m.tw_idx[b1 * nv + j] >= 0) d = d - twist_lin(ws, j, rot, pos);
  return d;
}

// ---- S4+S5: rows of every candidate with r<0 (cfd: r<w_c), compacted in candidate order ----------
template <class WS, class R, int G, class IN>
DMX_DN int build_rows(const ModelDev<R>& m, const IN& in, const WS& ws, bool cfd, const Grp<G>& gr) {
  const int ld = ws.ld();
  typedef typename WS::S S;
  const int nv = ws.nv(m), nc = ws.nc(m);
#pragma unroll 1
  for (int c = gr.lane; c < nc; c += G) {
    GeoT<S> g = collide<WS, R>(m, ws, c);
    ws.cr()[c] = g.r; st3(ws.cn(), c, g.n); st3(ws.cpos(), c, g.pos); st3(ws.ct1(), c, g.t1); st3(ws.ct2(), c, g.t2);
    bool inc = (val(g.r) < 0) || (cfd && val(g.r) < m.pair_solimp_cfd[5 * m.ct_pair[c] + 2]);
    ws.incl()[c] = inc ? (m.ct_condim[c] == 3 ? 4 : 1) : 0;
    if (inc) {
      S Dw, post, bd, mu;
      candidate_terms<S, R, IN>(m, in, c, g.r, cfd, Dw, post, bd, mu);
      ws.cD()[c] = Dw; ws.cpost()[c] = post; ws.cbd()[c] = bd; ws.cmu()[c] = mu;
    }
  }
  gr.sync();
  int nr = 0;
#pragma unroll 1
  for (int c = 0; c < nc; ++c) {
    int n = ws.incl()[c];
    if (gr.lane == 0) { ws.rowstart()[c] = nr; for (int e = 0; e < n; ++e) ws.rowcand()[nr + e] = 4 * c + e; }
    nr += n;
  }
  gr.sync();
  if (nr == 0) return 0;
  // Jacobian entries: one (candidate, dof) item yields that candidate's 1 or 4 row entries
#pragma unroll 1
  for (int it = gr.lane; it < nc * nv; it += G) {
    int c = it / nv, j = it - c * nv;
    int n = ws.incl()[c];
    if (n == 0) continue;
    int r0 = ws.rowstart()[c];
    V3<S> d = rel_twist<WS, R>(m, ws, j, m.ct_b1[c], m.ct_b2[c], ld3(ws.cpos(), c));
    S nd = dot(ld3(ws.cn(), c), d);
    if (n == 1) ws.J()[r0 * ld + j] = nd;
    else {
      S mu = ws.cmu()[c];
      S t1d = mu * dot(ld3(ws.ct1(), c), d), t2d = mu * dot(ld3(ws.ct2(), c), d);
      ws.J()[r0 * ld + j] = nd + t1d; ws.J()[(r0 + 1) * ld + j] = nd - t1d;
      ws.J()[(r0 + 2) * ld + j] = nd + t2d; ws.J()[(r0 + 3) * ld + j] = nd - t2d;
    }
  }
  gr.sync();
#pragma unroll 1
  for (int i = gr.lane; i < nr; i += G) {
    int c = ws.rowcand()[i] >> 2;
    S Jv(0.0);
#pragma unroll 4
    for (int j = 0; j < nv; ++j) Jv = Jv + ws.J()[i * ld + j] * in.v(j);
    ws.aref()[i] = ws.cpost()[c] - ws.cbd()[c] * Jv;
    ws.D()[i] = ws.cD()[c];
  }
  gr.sync();
  return nr;
}


// ---- D1: line search of S6.  phi'(a) = dl^T M (x + a dl - a0) + sum_i D_i p_i min(0, s_i + a p_i) is piecewise linear and
// increasing; bracketed 1-D Newton from a = 1.  The two row sums of an iterate (phi' and phi'') are taken cooperatively
// in the fixed order both sides document (D1/D4, "32-slot order"): row i is added to slot i mod 32 in
// increasing i, then the slots are combined by the butterfly slot[k] += slot[k xor s], s = 1, 2, 4, 8, 16.  A group of
// G lanes holds slots lane, lane + G, ... (32 / G per lane): the steps s < G are shuffles, the others in-lane adds.
// The butterfly leaves the same bits in every lane, so the search stays uniform over the group.
template <class WS, int G>
DMX_DI void ls_row_sums(int nr, const WS& ws, const Grp<G>& gr, const typename WS::S& a, typename WS::S& r1, typename WS::S& r2) {
  typedef typename WS::S S;
  const int NCOMP = 32 / G;
  S p1[NCOMP], p2[NCOMP];
#pragma unroll
  for (int c = 0; c < NCOMP; ++c) {
    p1[c] = S(0.0); p2[c] = S(0.0);
#pragma unroll 1
    for (int i = gr.lane + c * G; i < nr; i += 32) {
      const S pi = ws.pr()[i], si = ws.s()[i] + a * pi;
      if (val(si) < 0) { const S dp = ws.D()[i] * pi; p1[c] = p1[c] + dp * si; p2[c] = p2[c] + dp * pi; }
    }
  }
#pragma unroll
  for (int sft = 1; sft < G; sft <<= 1) {
#pragma unroll
    for (int c = 0; c < NCOMP; ++c) { p1[c] = p1[c] + gr.xor_lane(p1[c], sft); p2[c] = p2[c] + gr.xor_lane(p2[c], sft); }
  }
#pragma unroll
  for (int sft = 1; sft < NCOMP; sft <<= 1) {
#pragma unroll
    for (int c = 0; c < NCOMP; c += 2 * sft) { p1[c] = p1[c] + p1[c + sft]; p2[c] = p2[c] + p2[c + sft]; }
  }
  r1 = p1[0]; r2 = p2[0];
}
template <class WS, int G>
DMX_DN typename WS::S line_search(int nv, int nr, int n_ls, const WS& ws, const Grp<G>& gr) {
  typedef typename WS::S S;
  S dMd(0.0), dMxa(0.0);
#pragma unroll 1
  for (int a = 0; a < nv; ++a) { dMd = dMd + ws.dl()[a] * ws.Md()[a]; dMxa = dMxa + ws.Md()[a] * ws.xa()[a]; }
  S lo(0.0), hi(0.0), a(0.0), d2, d1a, r1, r2; bool hi_inf = true, frozen = false;
  ls_row_sums<WS, G>(nr, ws, gr, a, r1, r2);
  d1a = dMxa + r1; d2 = dMd + r2;
#pragma unroll 1
  for (int ls = 0; ls < n_ls && !frozen; ++ls) {
    S an = (ls == 0) ? S(1.0) : a - d1a / d2;
    if (ls > 0 && val(an) == val(a)) break;      // no representable progress: the root of phi' is reached
    bool inside = (val(an) > val(lo)) && (hi_inf || val(an) < val(hi));
    if (!inside) an = hi_inf ? S(2.0) * (val(a) > 1 ? a : S(1.0)) : S(0.5) * (lo + hi);
    a = an;
    ls_row_sums<WS, G>(nr, ws, gr, a, r1, r2);
    d1a = (dMxa + a * dMd) + r1; d2 = dMd + r2;
    if (val(d1a) < 0) lo = a; else if (val(d1a) > 0) { hi = a; hi_inf = false; } else frozen = true;
  }
  return a;
}

// ---- static sizes (Shape): Cholesky and substitutions with the rows in registers ----------------------------------
// Lane a of the group owns row a of the symmetric matrix (NV <= G).  Right-looking factorisation: once column j is
// known, every lane updates the rest of its own row, h[k] -= L[a][j] L[k][j], with L[k][j] fetched from lane k by
// shuffle; there is no shared-memory round trip and no group barrier inside the factorisation.  Every entry sees the
// operations of the left-looking shared-memory version in the same order (for entry (a,k): subtract L[a][j] L[k][j],
// j = 0, 1, ...), so the factor is bitwise the same.  The factor is stored with the reciprocal of its diagonal.  On
// exit the lower triangle of `dst` holds L row-major (for the backward substitution and for vjp_prepare's reuse) and
// hd the lane's own diagonal entry.
template <int NV, class S, int ST, int G>
DMX_DI bool chol_static(const Arr<S, ST>& src, const Arr<S, ST>& dst, int ld, const Grp<G>& gr, S (&h)[NV], S& hd) {
  const int a = gr.lane, ar = a < NV ? a : NV - 1;
#pragma unroll
  for (int b = 0; b < NV; ++b) h[b] = src[ar * ld + b];
  hd = S(0.0);
#pragma unroll
  for (int j = 0; j < NV; ++j) {
    const S piv = gr.from_lane(h[j], j);
    if (!(val(piv) > 0)) return false;       // uniform over the group
    const S il = m_rsqrt(piv);
    const S lj = (a == j) ? il : h[j] * il;
    h[j] = lj;
    if (a == j) hd = il;
#pragma unroll
    for (int k = j + 1; k < NV; ++k) h[k] = h[k] - lj * gr.from_lane(lj, k);
  }
  if (a < NV) {
#pragma unroll
    for (int b = 0; b < NV; ++b) if (b <= a) dst[a * ld + b] = h[b];
  }
  gr.sync();
  return true;
}
// bk (lane a holds entry a of the right-hand side) <- (L L^T)^-1 b with lane a's row of L in h, its diagonal in hd, and
// L row-major in `Lm` (column a of L for the backward substitution).  Same operations per entry as chol_solve.
template <int NV, class S, int ST, int G>
DMX_DI S solve_static(const Arr<S, ST>& Lm, int ld, const Grp<G>& gr, const S (&h)[NV], const S& hd, S bk) {
  const int a = gr.lane, ac = a < NV ? a : 0;
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    const S bi = gr.from_lane(bk * hd, i);
    if (a > i) bk = bk - h[i] * bi; else if (a == i) bk = bi;
  }
#pragma unroll
  for (int i = NV - 1; i >= 0; --i) {
    const S bi = gr.from_lane(bk * hd, i);
    if (a < i) bk = bk - Lm[i * ld + ac] * bi; else if (a == i) bk = bi;
  }
  return bk;
}
// row a of a factor left in shared memory by chol_static (reuse by the VJP)
template <int NV, class S, int ST, int G>
DMX_DI void load_factor_row(const Arr<S, ST>& Lm, int ld, const Grp<G>& gr, S (&h)[NV], S& hd) {
  const int a = gr.lane, ar = a < NV ? a : NV - 1;
#pragma unroll
  for (int b = 0; b < NV; ++b) h[b] = Lm[ar * ld + b];
  hd = Lm[ar * ld + ar];
}
// One copy per kernel of the unrolled factorisation / substitution code (the instruction cache is the scarce resource:
// the kernels are fetch-bound when every call site carries its own copy).  ok is uniform over the group.
template <class S> struct SolveOut { S x; bool ok; };
template <int NV, class S, int ST, int G>
__device__ __noinline__ SolveOut<S> factor_solve_static(unsigned src, unsigned dst, int ld, S rhs) {   // offsets in the CTA's dynamic shared memory
  const Grp<G> gr = make_group<G>();
  S h[NV], hd;
  SolveOut<S> o; o.x = rhs;
  o.ok = chol_static<NV>(Arr<S, ST>(smem_ptr<S>(src)), Arr<S, ST>(smem_ptr<S>(dst)), ld, gr, h, hd);
  if (o.ok) o.x = solve_static<NV>(Arr<S, ST>(smem_ptr<S>(dst)), ld, gr, h, hd, rhs);
  return o;
}
template <int NV, class S, int ST, int G>
__device__ __noinline__ S resolve_static(unsigned Lm, int ld, S rhs) {
  const Grp<G> gr = make_group<G>();
  S h[NV], hd;
  load_factor_row<NV>(Arr<S, ST>(smem_ptr<S>(Lm)), ld, gr, h, hd);
  return solve_static<NV>(Arr<S, ST>(smem_ptr<S>(Lm)), ld, gr, h, hd, rhs);
}
// H = M + J^T diag(w) J on the lower triangle: lane per entry; the entry -> (a, b) map of a lane is computed once
template <int NV, int G> struct TriMap {
  static const int NT = NV * (NV + 1) / 2, NE = (NT + G - 1) / G;
  int off[NE], ca[NE], cb[NE];
  DMX_DI void init(int lane, int ld) {
#pragma unroll
    for (int q = 0; q < NE; ++q) {
      int e = lane + q * G, a = 0, b = 0;
      if (e < NT) tri_index(e, a, b);
      off[q] = e < NT ? a * ld + b : -1; ca[q] = a; cb[q] = b;
    }
  }
};
template <int NV, int G, class WS>
DMX_DI void build_h_static(const TriMap<NV, G>& tm, int nr, int ld, const WS& ws) {
  typedef typename WS::S S;
#pragma unroll
  for (int q = 0; q < TriMap<NV, G>::NE; ++q) {
    if (tm.off[q] < 0) continue;
    S t = ws.M()[tm.off[q]];
    const int ca = tm.ca[q], cb = tm.cb[q];
#pragma unroll 4
    for (int i = 0; i < nr; ++i) t = t + ws.pr()[i] * ws.J()[i * ld + ca] * ws.J()[i * ld + cb];
    ws.Hc()[tm.off[q]] = t;
  }
}

// ---- S6 with static sizes: the Newton iteration of `newton` below with the vectors x, a0, the step and the rows of the
// factor in registers (lane a owns dof a), the products J x, J dl unrolled over the dofs.  Same operations per entry
// and the same summation orders as the generic version: results are bitwise equal.
template <class WS, int G>
DMX_DN bool newton_static(int nr, int n_it, int n_ls, const WS& ws, const Grp<G>& gr, int& iters) {
  typedef typename WS::S S;
  const int NV = WS::SH::NV, ld = WS::SH::LD;
  const int a = gr.lane, ac = a < NV ? a : NV - 1;
  const bool own = a < NV;
  const S a0a = ws.a0()[ac];
  S xa_ = a0a;                          // x[a]
  if (own) ws.x()[a] = xa_;
  gr.sync();
  iters = 0;
  if (nr == 0) return true;
  TriMap<WS::SH::NV, G> tm; tm.init(a, ld);
  bool conv = false;
#pragma unroll 1
  for (int it = 0; it < n_it; ++it) {
    ++iters;
    {
      S xr[WS::SH::NV];
#pragma unroll
      for (int j = 0; j < NV; ++j) xr[j] = ws.x()[j];
#pragma unroll 1
      for (int i = a; i < nr; i += G) {
        S t(0.0);
#pragma unroll
        for (int j = 0; j < NV; ++j) t = t + ws.J()[i * ld + j] * xr[j];
        const S si = t - ws.aref()[i];
        ws.s()[i] = si;
        ws.active()[i] = val(si) < 0 ? 1 : 0;
        ws.pr()[i] = val(si) < 0 ? ws.D()[i] : S(0.0);
      }
      if (own) ws.xa()[a] = xa_ - a0a;
      gr.sync();
    }
    S dla;
    {
      S t(0.0);
#pragma unroll
      for (int b = 0; b < NV; ++b) t = t + ws.M()[ac * ld + b] * ws.xa()[b];
#pragma unroll 4
      for (int i = 0; i < nr; ++i) t = t + ws.J()[i * ld + ac] * ws.pr()[i] * ws.s()[i];
      if (own) ws.g()[a] = t;
      dla = -t;
    }
    build_h_static<WS::SH::NV, G>(tm, nr, ld, ws);
    gr.sync();
    {
      const SolveOut<S> so = factor_solve_static<WS::SH::NV, S, WS::ST, G>(smem_off(ws.Hc().p), smem_off(ws.Hc().p), ld, dla);
      if (!so.ok) break;
      dla = so.x;
    }
    if (own) ws.dl()[a] = dla;
    gr.sync();
    bool same = true;
    {
      S dr[WS::SH::NV];
#pragma unroll
      for (int j = 0; j < NV; ++j) dr[j] = ws.dl()[j];
#pragma unroll 1
      for (int i = a; i < nr; i += G) {
        S t(0.0);
#pragma unroll
        for (int j = 0; j < NV; ++j) t = t + ws.J()[i * ld + j] * dr[j];
        ws.pr()[i] = t;
        const S si = ws.s()[i];
        if ((val(si) < 0) != (val(si + t) < 0)) same = false;
      }
      same = gr.all(same);
      if (!same && own) {
        S t(0.0);
#pragma unroll
        for (int b = 0; b < NV; ++b) t = t + ws.M()[a * ld + b] * dr[b];
        ws.Md()[a] = t;
      }
      gr.sync();
    }
    S alpha(1.0);
    if (!same) alpha = line_search<WS, G>(NV, nr, n_ls, ws, gr);
    xa_ = xa_ + alpha * dla;
    if (own) ws.x()[a] = xa_;
    gr.sync();
    if (same) { conv = true; break; }
  }
  return conv;
}

// ---- S6: Newton with a fixed iteration budget on the reduced primal problem of Eq. 2 -------------
//   Phi(x) = 1/2 (x-a0)^T M (x-a0) + 1/2 sum_i D_i min(0, J_i x - aref_i)^2
// (iterations / ls_iterations PAPER.md:515, 539).
// Returns true when the last step was a full step inside an unchanged active set.
template <class WS, int G>
DMX_DN bool newton(int nv, int nr, int n_it, int n_ls, const WS& ws, const Grp<G>& gr, int& iters) {
  if constexpr (WS::SH::NV > 0 && G > 1) return newton_static<WS, G>(nr, n_it, n_ls, ws, gr, iters);
  const int ld = ws.ld();
  typedef typename WS::S S;
#pragma unroll 1
  for (int j = gr.lane; j < nv; j += G) ws.x()[j] = ws.a0()[j];
  gr.sync();
  iters = 0;
  if (nr == 0) return true;
  bool conv = false;
#pragma unroll 1
  for (int it = 0; it < n_it; ++it) {
    ++iters;
#pragma unroll 1
    for (int i = gr.lane; i < nr; i += G) {
      S t(0.0);
#pragma unroll 4
      for (int j = 0; j < nv; ++j) t = t + ws.J()[i * ld + j] * ws.x()[j];
      ws.s()[i] = t - ws.aref()[i];
      ws.active()[i] = val(ws.s()[i]) < 0 ? 1 : 0;     // the set the factor left in Hc belongs to (reused by vjp_prepare)
      ws.pr()[i] = val(ws.s()[i]) < 0 ? ws.D()[i] : S(0.0);   // masked weight (pr is free until the step direction is known): branch-free sums below
    }
#pragma unroll 1
    for (int j = gr.lane; j < nv; j += G) ws.xa()[j] = ws.x()[j] - ws.a0()[j];
    gr.sync();
#pragma unroll 1
    for (int a = gr.lane; a < nv; a += G) {
      S t(0.0);
#pragma unroll 4
      for (int b = 0; b < nv; ++b) t = t + ws.M()[a * ld + b] * ws.xa()[b];
#pragma unroll 4
      for (int i = 0; i < nr; ++i) t = t + ws.J()[i * ld + a] * ws.pr()[i] * ws.s()[i];
      ws.g()[a] = t; ws.dl()[a] = -t;
    }
#pragma unroll 1
    for (int e = gr.lane; e < nv * (nv + 1) / 2; e += G) {
      int a, b; tri_index(e, a, b);
      S t = ws.M()[a * ld + b];
#pragma unroll 4
      for (int i = 0; i < nr; ++i) t = t + ws.pr()[i] * ws.J()[i * ld + a] * ws.J()[i * ld + b];
      ws.Hc()[a * ld + b] = t;
    }
    gr.sync();
    if (!cholesky(ws.Hc(), nv, ld, gr)) break;
    chol_solve(ws.Hc(), nv, ld, ws.dl(), gr);
    bool same = true;
#pragma unroll 1
    for (int i = gr.lane; i < nr; i += G) {
      S t(0.0);
#pragma unroll 4
      for (int j = 0; j < nv; ++j) t = t + ws.J()[i * ld + j] * ws.dl()[j];
      ws.pr()[i] = t;
      if ((val(ws.s()[i]) < 0) != (val(ws.s()[i] + t) < 0)) same = false;
    }
    same = gr.all(same);
    gr.sync();
    S alpha(1.0);
    if (!same) {
#pragma unroll 1
      for (int a = gr.lane; a < nv; a += G) {
        S t(0.0);
#pragma unroll 4
        for (int b = 0; b < nv; ++b) t = t + ws.M()[a * ld + b] * ws.dl()[b];
        ws.Md()[a] = t;
      }
      gr.sync();
      alpha = line_search<WS, G>(nv, nr, n_ls, ws, gr);
    }
#pragma unroll 1
    for (int j = gr.lane; j < nv; j += G) ws.x()[j] = ws.x()[j] + alpha * ws.dl()[j];
    gr.sync();
    if (same) { conv = true; break; }
  }
  return conv;
}

// ---- F (cfd=false) or F~ (cfd=true) at one state: result in ws.x, rows and M left in ws ----------
// returns nr >= 0, or -1 when M is not positive definite / the result is not finite.
// xk != nullptr: the solution x* is already known (stage rate read from the tape; element j at xk[j*xst]); the
// unconstrained solve and the Newton iterations are skipped and only M, the rows and x* are set up for the VJP.
template <class WS, class R, int G, class IN>
DMX_DN int vector_field(const ModelDev<R>& m, const IN& in, const WS& ws, bool cfd, bool& conv, int& iters, const Grp<G>& gr,
                        const double* xk = nullptr, int xst = 1) {
  const int ld = ws.ld();
  const int nv = ws.nv(m);
  phase_sync(0);
  DMX_T0;
  kinematics<WS, R, G, IN, false>(m, in, ws, gr);
  DMX_TICK(gr, 0);
  phase_sync(1);
  dynamics<WS, R, G, IN>(m, in, ws, gr);
  DMX_TICK(gr, 1);
  conv = true; iters = 0;
  if (!xk) {
    phase_sync(2);
    if constexpr (WS::SH::NV > 0 && G > 1) {        // factor of M and a0 = M^-1 (tau - c) with the rows in registers
      const int a = gr.lane < nv ? gr.lane : nv - 1;
      const SolveOut<typename WS::S> so = factor_solve_static<WS::SH::NV, typename WS::S, WS::ST, G>(smem_off(ws.M().p), smem_off(ws.Hc().p), ld, ws.tau()[a] - ws.c()[a]);
      if (!so.ok) return -1;
      if (gr.lane < nv) ws.a0()[gr.lane] = so.x;
      gr.sync();
    } else {
      for (int e = gr.lane; e < nv * ld; e += G) ws.Hc()[e] = ws.M()[e];
      for (int j = gr.lane; j < nv; j += G) ws.a0()[j] = ws.tau()[j] - ws.c()[j];
      gr.sync();
      if (!cholesky(ws.Hc(), nv, ld, gr)) return -1;
      chol_solve(ws.Hc(), nv, ld, ws.a0(), gr);
    }
    DMX_TICK(gr, 2);
  }
  phase_sync(3);
  int nr = build_rows<WS, R, G, IN>(m, in, ws, cfd, gr);
  DMX_TICK(gr, 3);
  if (xk) {
    for (int j = gr.lane; j < nv; j += G) ws.x()[j] = (R)xk[j * xst];
    gr.sync();
    return nr;
  }
  phase_sync(4);
  conv = newton<WS, G>(nv, nr, m.newton_iters, m.ls_iters, ws, gr, iters);
  DMX_TICK(gr, 4);
  bool fin = true;
  for (int j = gr.lane; j < nv; j += G) if (!isfinite(val(ws.x()[j]))) fin = false;
  if (!gr.all(fin)) return -1;
  return nr;
}

// ---- S11/S12, cooperative part: final active set A, H = M + J_A^T D_A J_A, w = H^-1 kappa ---------
// ws.kap() holds kappa on entry and w on exit.  Returns false if H is not positive definite.
template <class WS, int G>
DMX_DN bool vjp_prepare(int nv, int nr, bool hc_valid, const WS& ws, const Grp<G>& gr) {
  const int ld = ws.ld();
  typedef typename WS::S S;
  // hc_valid: Hc still holds the Cholesky factor of the last Newton iteration (or of M when there are no rows) and
  // ws.active the set it was built for.  A converged solve ends on an unchanged active set, so that factor IS the
  // factor of H at x*; it is reused unless the recomputed residuals disagree with the set on a sign.
  bool same = hc_valid;
#pragma unroll 1
  for (int i = gr.lane; i < nr; i += G) {
    S t(0.0);
#pragma unroll 4
    for (int j = 0; j < nv; ++j) t = t + ws.J()[i * ld + j] * ws.x()[j];
    t = t - ws.aref()[i];
    ws.s()[i] = t;
    const int act = val(t) < 0 ? 1 : 0;
    if (hc_valid && ws.active()[i] != act) same = false;
    ws.active()[i] = act;
    ws.pr()[i] = act ? ws.D()[i] : S(0.0);               // masked weight for the branch-free H build (pr is rewritten by vjp_velocity)
  }
  const bool reuse = gr.all(same);
  gr.sync();
  if constexpr (WS::SH::NV > 0 && G > 1) {
    const int a = gr.lane < nv ? gr.lane : nv - 1;
    S w;
    if (!reuse) {
      TriMap<WS::SH::NV, G> tm; tm.init(gr.lane, ld);
      build_h_static<WS::SH::NV, G>(tm, nr, ld, ws);
      gr.sync();
      const SolveOut<S> so = factor_solve_static<WS::SH::NV, S, WS::ST, G>(smem_off(ws.Hc().p), smem_off(ws.Hc().p), ld, ws.kap()[a]);
      if (!so.ok) return false;
      w = so.x;
    } else w = resolve_static<WS::SH::NV, S, WS::ST, G>(smem_off(ws.Hc().p), ld, ws.kap()[a]);
    gr.sync();                                     // every lane has read kappa before w overwrites it
    if (gr.lane < nv) ws.kap()[gr.lane] = w;
    gr.sync();
    return true;
  }
  if (!reuse) {
#pragma unroll 1
    for (int e = gr.lane; e < nv * (nv + 1) / 2; e += G) {
      int a, b; tri_index(e, a, b);
      S t = ws.M()[a * ld + b];
#pragma unroll 4
      for (int i = 0; i < nr; ++i) t = t + ws.pr()[i] * ws.J()[i * ld + a] * ws.J()[i * ld + b];
      ws.Hc()[a * ld + b] = t;
    }
    gr.sync();
    if (!cholesky(ws.Hc(), nv, ld, gr)) return false;
  }
  chol_solve(ws.Hc(), nv, ld, ws.kap(), gr);
  return true;
}

// ---- S11/S12: derivative of  S = w^T g(z; x*),  g = ID(q,v,x*) - tau(q,v,u) + sum_{i in A} J_i^T D_i (J_i x* - aref_i)
// (stationarity of Eq. 2 at the final active set A; x*, A and w = H^-1 kappa are constants).  The VJP of the
// vector field is minus the gradient of S.  With the virtual-work identity
//   w^T ID = sum_b velw(com_b).F_b + omegaw(b).N_b            (velw, omegaw: body velocities under joint rates w)
// and  J_i y = dir_i . relvel_y(pos_i)  for y in {x*, v, w}, the gradient splits into
//   u : closed form;   v : one reverse sweep over the tree (geometry fixed) + closed-form row / damping terms;
//   q : one tangent pass per dof over the subtree below that dof;   p : tangent passes without kinematics.

// velocity part, cooperative: vbar = -dS/dv.  Needs in ws: frames (any acceleration), tw, Iw, J, D, cbd, active,
// w in ws.kap.  Uses ws.Fb/ws.Nb for velw/omegaw, ws.Isub for the body adjoints, ws.pr for J_i w.
template <class WS, class R, int G, class IN, class AOUT>
DMX_D void vjp_velocity(const ModelDev<R>& m, const IN& in, const WS& ws, int nr, const AOUT& vbar, const Grp<G>& gr) {
  const int ld = ws.ld();
  typedef typename WS::S S;
  const int nv = ws.nv(m), nb = m.nbody;
  // seeds: cotangents of (omega_b, alpha_b, ap_b) from F_b = m (ac_b - g), N_b = I alpha + omega x I omega
#pragma unroll 1
  for (int b = 1 + gr.lane; b < nb; b += G) {
    S z(0.0);
    V3<S> vw = mk3<S>(z, z, z), ow = vw, comb = ld3(ws.com(), b);
#pragma unroll 1
    for (int e = m.tw_ptr[b]; e < m.tw_ptr[b + 1]; ++e) {
      int j = m.tw_dof[e];
      S wj = ws.kap()[j];
      vw = vw + ld3(ws.tw(), e) * wj;
      if (m.dof_rot[j]) ow = ow + ld3(ws.dax(), j) * wj;
    }
    st3(ws.Fb(), b, vw); st3(ws.Nb(), b, ow);
    V3<S> om = ld3(ws.fw(), b), rc = comb - ld3(ws.fp(), b);
    M3<S> I = ld9(ws.Iw(), b);
    V3<S> acb = vw * in.p(b);
    V3<S> alb = cross(rc, acb) + I * ow;
    V3<S> omb = cross(cross(om, rc), acb) + cross(rc, cross(acb, om)) + cross(I * om, ow) + I * cross(ow, om);
    st3(ws.Isub(), 3 * b, omb); st3(ws.Isub(), 3 * b + 1, alb); st3(ws.Isub(), 3 * b + 2, acb);
  }
#pragma unroll 1
  for (int i = gr.lane; i < nr; i += G) {
    S t(0.0);
    if (ws.active()[i]) for (int j = 0; j < nv; ++j) t = t + ws.J()[i * ld + j] * ws.kap()[j];
    ws.pr()[i] = t;
  }
  gr.sync();
  // leaves to root: every body gathers its children's cotangents through their joints
#pragma unroll 1
  for (int lv = m.nlevel - 1; lv >= 0; --lv) {
#pragma unroll 1
    for (int i = m.level_ptr[lv] + gr.lane; i < m.level_ptr[lv + 1]; i += G) {
      int b = m.level_body[i];
      V3<S> omb = ld3(ws.Isub(), 3 * b), alb = ld3(ws.Isub(), 3 * b + 1), apb = ld3(ws.Isub(), 3 * b + 2);
      V3<S> wp = ld3(ws.fw(), b), pp = ld3(ws.fp(), b);
#pragma unroll 1
      for (int t = m.child_ptr[b]; t < m.child_ptr[b + 1]; ++t) {
        int c = m.child_idx[t], j = m.body_jnt[c];
        V3<S> oc = ld3(ws.Isub(), 3 * c), ac = ld3(ws.Isub(), 3 * c + 1), pc = ld3(ws.Isub(), 3 * c + 2);
        V3<S> E = ld3(ws.fp(), c) - pp;
        if (j >= 0 && m.jnt_type[j] == JNT_HINGE) {
          int va = m.jnt_vadr[j];
          V3<S> ax = ld3(ws.dax(), va), o = ld3(ws.dan(), va), wc = ld3(ws.fw(), c);
          V3<S> d = ld3(ws.fp(), c) - o;
          ac = ac + cross(d, pc);
          oc = oc + cross(cross(wc, d), pc) + cross(d, cross(pc, wc));
          E = o - pp;
          omb = omb + cross(ax, ac) * in.v(va);
        } else if (j >= 0 && m.jnt_type[j] == JNT_SLIDE) {
          int va = m.jnt_vadr[j];
          omb = omb + cross(ld3(ws.dax(), va), pc) * (S(2.0) * in.v(va));
        }
        omb = omb + oc + cross(cross(wp, E), pc) + cross(E, cross(pc, wp));
        alb = alb + ac + cross(E, pc);
        apb = apb + pc;
      }
      st3(ws.Isub(), 3 * b, omb); st3(ws.Isub(), 3 * b + 1, alb); st3(ws.Isub(), 3 * b + 2, apb);
    }
    gr.sync();
  }
  // joint rates: Coriolis part through each body's own joint, damping / PD and the rows' -b J v term
#pragma unroll 1
  for (int j = gr.lane; j < nv; j += G) {
    int jn = m.dof_jnt[j], b = m.dof_body[j], jt = m.jnt_type[jn], par = m.body_parent[b];
    V3<S> omb = ld3(ws.Isub(), 3 * b), alb = ld3(ws.Isub(), 3 * b + 1), apb = ld3(ws.Isub(), 3 * b + 2);
    V3<S> ax = ld3(ws.dax(), j), wp = ld3(ws.fw(), par);
    S g(0.0);
    if (jt == JNT_HINGE) {
      V3<S> d = ld3(ws.fp(), b) - ld3(ws.dan(), j), wc = ld3(ws.fw(), b);
      V3<S> a2 = alb + cross(d, apb);
      V3<S> o2 = omb + cross(cross(wc, d), apb) + cross(d, cross(apb, wc));
      g = dot(o2, ax) + dot(a2, cross(wp, ax));
    } else if (jt == JNT_SLIDE) g = S(2.0) * dot(cross(wp, ax), apb);
    else if (m.dof_rot[j]) g = dot(omb, ax);
    S kd(m.jnt_damping[jn]);
#pragma unroll 1
    for (int i = 0; i < m.nu; ++i) if (m.act_type[i] == ACT_PD && m.jnt_vadr[m.act_jnt[i]] == j) kd = kd + S(m.act_kd[i]);
    g = g + ws.kap()[j] * kd;
#pragma unroll 1
    for (int i = 0; i < nr; ++i) if (ws.active()[i]) g = g + ws.pr()[i] * ws.D()[i] * ws.cbd()[ws.rowcand()[i] >> 2] * ws.J()[i * ld + j];
    vbar[j] = -(double)g;
  }
  gr.sync();
}

// ---- configuration part, bodies: closed-form variation, cooperative over the (body, ancestor-dof) table -----------
// For dof j with axis ax through o carried by the parent frame P of body(j) (free-joint rotation: P = world and the
// anchor moves with the root origin), every material point x and vector of the subtree varies as
//   dx = ax x (x-o),  dR = [ax]x R,  dOm = ax x (Om-Om_P),  dal = adot x (Om-Om_P) + ax x (al-al_P),
//   dV(x) = adot x r + ax x (V(x)-odot),  da(x) = addot x r + 2 adot x (V(x)-odot) + ax x (a(x)-oddot),
// adot = Om_P x ax, addot = al_P x ax + Om_P x adot (the variation commutes with d/dt along theta_j(t)+eps); the
// virtual fields under w follow the first-order rules with the w-twists.  Slide and free-translation dofs shift the
// subtree.  Then dS_b = dvw.F + m vw.da_c + dow.N + ow.dN with dN from the rotated inertia.
// Needs: frames at x* (ACC kinematics), ws.Fb = velw(com), ws.Nb = omegaw (vjp_velocity), ws.Iw.  Uses ws.Isub for
// (F, N, a_com) per body and ws.tw for the per-entry contributions.  Writes qbar[j] = -(dS/dq_j) of the body part and
// the PD term; the rows' part is added by the tangent lanes.
template <class WS, class R, int G, class IN, class AOUT>
DMX_D void vjp_config_bodies(const ModelDev<R>& m, const IN& in, const WS& ws, const AOUT& qbar, const Grp<G>& gr) {
  typedef typename WS::S S;
  const int nv = ws.nv(m), nb = m.nbody;
#pragma unroll 1
  for (int b = 1 + gr.lane; b < nb; b += G) {
    V3<S> Fb, Nb; M3<S> Iw;
    body_wrench<WS, R, IN>(m, in, ws, b, Fb, Nb, Iw);
    FrameT<S> f; f.p = ld3(ws.fp(), b); f.w = ld3(ws.fw(), b); f.al = ld3(ws.fal(), b); f.ap = ld3(ws.fap(), b);
    st3(ws.Isub(), 3 * b, Fb); st3(ws.Isub(), 3 * b + 1, Nb); st3(ws.Isub(), 3 * b + 2, point_acc(f, ld3(ws.com(), b)));
    S z(0.0);
    V3<S> vx = mk3<S>(z, z, z), ox = vx;                // twist of the body under the joint rates x* (for J_i x*)
#pragma unroll 1
    for (int e = m.tw_ptr[b]; e < m.tw_ptr[b + 1]; ++e) {
      int j = m.tw_dof[e];
      S xj = ws.x()[j];
      vx = vx + ld3(ws.tw(), e) * xj;
      if (m.dof_rot[j]) ox = ox + ld3(ws.dax(), j) * xj;
    }
    st3(ws.fvx(), b, vx); st3(ws.fox(), b, ox);
  }
  gr.sync();
#pragma unroll 1
  for (int e = gr.lane; e < m.ntw; e += G) {
    const int b = m.tw_body[e], j = m.tw_dof[e], jn = m.dof_jnt[j], jt = m.jnt_type[jn], bj = m.dof_body[j], par = m.body_parent[bj];
    S z(0.0), contrib(0.0);
    V3<S> z3 = mk3<S>(z, z, z);
    if (!(jt == JNT_FREE && !m.dof_rot[j])) {
      V3<S> ax = ld3(ws.dax(), j);
      V3<S> OmP = z3, alP = z3, OmPw = z3, od = z3, odd = z3, odw = z3, o = ld3(ws.dan(), j);
      if (jt == JNT_FREE) {
        int va = m.jnt_vadr[jn];
        od = ld3(ws.fvp(), bj); odd = ld3(ws.fap(), bj);
        odw = mk3<S>(ws.kap()[va], ws.kap()[va + 1], ws.kap()[va + 2]);
      } else {
        FrameT<S> P; P.p = ld3(ws.fp(), par); P.w = ld3(ws.fw(), par); P.al = ld3(ws.fal(), par); P.vp = ld3(ws.fvp(), par); P.ap = ld3(ws.fap(), par);
        OmP = P.w; alP = P.al;
        od = point_vel(P, o); odd = point_acc(P, o);
        if (par > 0) { OmPw = ld3(ws.Nb(), par); odw = ld3(ws.Fb(), par) + cross(OmPw, o - ld3(ws.com(), par)); }
      }
      V3<S> adot = cross(OmP, ax), adotw = cross(OmPw, ax);
      V3<S> addot = cross(alP, ax) + cross(OmP, adot);
      V3<S> F = ld3(ws.Isub(), 3 * b), N = ld3(ws.Isub(), 3 * b + 1), vw = ld3(ws.Fb(), b), ow = ld3(ws.Nb(), b);
      S mass = in.p(b);
      if (jt == JNT_SLIDE) contrib = dot(adotw, F) + mass * dot(vw, addot);
      else {
        V3<S> c = ld3(ws.com(), b), Om = ld3(ws.fw(), b), al = ld3(ws.fal(), b), ac = ld3(ws.Isub(), 3 * b + 2);
        V3<S> rc = c - o, Vc = ld3(ws.fvp(), b) + cross(Om, c - ld3(ws.fp(), b));
        M3<S> I = ld9(ws.Iw(), b);
        V3<S> d_ow = cross(ax, ow - OmPw);
        V3<S> d_vw = cross(adotw, rc) + cross(ax, vw - odw);
        V3<S> d_ac = cross(addot, rc) + cross(adot, Vc - od) * S(2.0) + cross(ax, ac - odd);
        V3<S> d_Om = cross(ax, Om - OmP);
        V3<S> d_al = cross(adot, Om - OmP) + cross(ax, al - alP);
        V3<S> IOm = I * Om;
        V3<S> dI_al = cross(ax, I * al) - I * cross(ax, al), dI_Om = cross(ax, IOm) - I * cross(ax, Om);
        V3<S> d_N = dI_al + I * d_al + cross(d_Om, IOm) + cross(Om, dI_Om + I * d_Om);
        contrib = dot(d_vw, F) + mass * dot(vw, d_ac) + dot(d_ow, N) + dot(ow, d_N);
      }
    }
    ws.tw()[3 * e] = contrib;
  }
  gr.sync();
#pragma unroll 1
  for (int j = gr.lane; j < nv; j += G) {
    int bj = m.dof_body[j], jn = m.dof_jnt[j];
    S acc(0.0);
#pragma unroll 1
    for (int t = m.sub_ptr[bj]; t < m.sub_ptr[bj + 1]; ++t) acc = acc + ws.tw()[3 * m.tw_idx[m.sub_body[t] * nv + j]];
    if (m.jnt_type[jn] != JNT_FREE)
      for (int i = 0; i < m.nu; ++i) if (m.act_type[i] == ACT_PD && m.act_jnt[i] == jn) acc = acc + ws.kap()[j] * S(m.act_kp[i]);
    qbar[j] = -(double)acc;
  }
  gr.sync();
}

// ---- configuration part, rows: closed-form variation, cooperative over (candidate, ancestor-dof) --------------
// A candidate is a pair of material points c1 (body1; absent for a plane) and c2 (body2), pos on the mid-surface.
// For y in {x*, v, w}: J_e y = dir_e . (V^y_2(pos) - V^y_1(pos)), V^y_b(pos) = V^y_b(c_b) + Om^y_b x (pos - c_b);
// S_c = sum_{e in A} (J_e w) D(r) (J_e x* - post(r) + b J_e v).  Material points and twists of a body below dof j vary
// by the rules above; r, n, the tangent frame and pos follow (sphere-sphere: n = (c2-c1)/|c2-c1|, Gram-Schmidt frame).
// Uses ws.J as the (candidate, dof) contribution buffer.  Needs ws.fox / ws.fvx (x*-twists), ws.Fb / ws.Nb
// (w-twists), ws.active, the frames at x*, and the candidate geometry stored by build_rows.
template <bool PP, class WS, class R, int G, class IN, class AOUT>
DMX_D void vjp_config_rows(const ModelDev<R>& m, const IN& in, const WS& ws, bool cfd, const AOUT& qbar, const Grp<G>& gr) {
  typedef typename WS::S S;
  const int nv = ws.nv(m), nc = ws.nc(m);
#pragma unroll 1
  for (int c = gr.lane; c < nc; c += G) {
    if (ws.incl()[c] == 0 || (m.ct_kind[c] == CK_POINT_POINT) != PP) continue;
    InDual<S, WS::ST> din; din.pa = in.pa; din.kind = -1; din.idx = -1;      // parameters without tangent; r carries the seed
    Dual<S> Dw, post, bd, mu;
    candidate_terms_dual<R, InDual<S, WS::ST> >(m, din, c, Dual<S>(ws.cr()[c], S(1.0)), cfd, Dw, post, bd, mu);
    ws.cdD()[c] = Dw.d; ws.cdpost()[c] = post.d;
  }
  gr.sync();
#pragma unroll 1
  for (int it = gr.lane; it < nc * nv; it += G) {
    const int c = it / nv, j = it - c * nv;
    S contrib(0.0);
    const int n = ws.incl()[c], b1 = m.ct_b1[c], b2 = m.ct_b2[c];
    const bool in1 = b1 > 0 && m.tw_idx[b1 * nv + j] >= 0, in2 = b2 > 0 && m.tw_idx[b2 * nv + j] >= 0;
    bool go = n > 0 && (in1 || in2) && (m.ct_kind[c] == CK_POINT_POINT) == PP;
    int r0 = 0;
    if (go) { r0 = ws.rowstart()[c]; bool any = false; for (int e = 0; e < n; ++e) any = any || ws.active()[r0 + e]; go = any; }
    if (go) {
      const int jn = m.dof_jnt[j], jt = m.jnt_type[jn], bj = m.dof_body[j], par = m.body_parent[bj];
      const bool turn = m.dof_rot[j] != 0, pp = PP;
      S z(0.0);
      V3<S> z3 = mk3<S>(z, z, z), ax = ld3(ws.dax(), j), o = ld3(ws.dan(), j);
      V3<S> OmP[3] = {z3, z3, z3}, od[3] = {z3, z3, z3};      // parent-side data of the dof for the rate fields x*, v, w
      if (jt == JNT_FREE) {
        int va = m.jnt_vadr[jn];
        od[0] = mk3<S>(ws.x()[va], ws.x()[va + 1], ws.x()[va + 2]);
        od[1] = ld3(ws.fvp(), bj);
        od[2] = mk3<S>(ws.kap()[va], ws.kap()[va + 1], ws.kap()[va + 2]);
      } else if (par > 0) {
        V3<S> ro = o - ld3(ws.com(), par);
        OmP[0] = ld3(ws.fox(), par); od[0] = ld3(ws.fvx(), par) + cross(OmP[0], ro);
        OmP[1] = ld3(ws.fw(), par);  od[1] = ld3(ws.fvp(), par) + cross(OmP[1], o - ld3(ws.fp(), par));
        OmP[2] = ld3(ws.Nb(), par);  od[2] = ld3(ws.Fb(), par) + cross(OmP[2], ro);
      }
      // material points and their variations
      V3<S> nrm = ld3(ws.cn(), c), t1 = ld3(ws.ct1(), c), t2 = ld3(ws.ct2(), c), pos = ld3(ws.cpos(), c);
      S r = ws.cr()[c], rho1(m.ct_rho1[c]);
      V3<S> c1 = z3, c2 = ld3(ws.fp(), b2) + ld9(ws.fR(), b2) * c3<S>(m.ct_p2, c);
      if (pp) c1 = ld3(ws.fp(), b1) + ld9(ws.fR(), b1) * c3<S>(m.ct_p1, c);
      V3<S> dc1 = in1 ? (turn ? cross(ax, c1 - o) : ax) : z3, dc2 = in2 ? (turn ? cross(ax, c2 - o) : ax) : z3;
      // geometry: r, n, tangent frame, pos
      S dr; V3<S> dn = z3, dt1 = z3, dt2 = z3, dpos;
      if (!pp) { dr = dot(nrm, dc2); dpos = dc2 - nrm * (S(0.5) * dr); }
      else {
        S dist = r + rho1 + S(m.ct_rho2[c]);
        V3<S> ddl = dc2 - dc1;
        dr = dot(nrm, ddl);
        dn = (ddl - nrm * dr) * (S(1.0) / dist);
        dpos = dc1 + dn * (rho1 + S(0.5) * r) + nrm * (S(0.5) * dr);
        typename RealOf<S>::type axn = fabs(val(nrm.x)), ayn = fabs(val(nrm.y)), azn = fabs(val(nrm.z));
        int ei = 0; if (ayn < axn) { ei = 1; axn = ayn; } if (azn < axn) ei = 2;
        S o1(1.0);
        V3<S> ev = mk3<S>(ei == 0 ? o1 : z, ei == 1 ? o1 : z, ei == 2 ? o1 : z);
        S en = dot(ev, nrm);
        V3<S> t = ev - nrm * en;
        S tl = m_sqrt(dot(t, t));
        V3<S> dt = z3 - dn * en - nrm * dot(ev, dn);
        dt1 = (dt - t1 * dot(t1, dt)) * (S(1.0) / tl);
        dt2 = cross(dn, t1) + cross(nrm, dt1);
      }
      // relative velocities at pos under the three rate fields and their variations
      V3<S> rel[3] = {z3, z3, z3}, drel[3] = {z3, z3, z3};
#pragma unroll 1
      for (int side = PP ? 0 : 1; side < 2; ++side) {
        const int b = side ? b2 : b1;
        if (b == 0) continue;
        const bool ins = side ? in2 : in1;
        V3<S> cs = side ? c2 : c1, dcs = side ? dc2 : dc1;
        V3<S> pb = ld3(ws.fp(), b), cb = ld3(ws.com(), b), pc = pos - cs, dpc = dpos - dcs;
        S sg = side ? S(1.0) : S(-1.0);
#pragma unroll
        for (int y = 0; y < 3; ++y) {
          V3<S> Om = y == 0 ? ld3(ws.fox(), b) : (y == 1 ? ld3(ws.fw(), b) : ld3(ws.Nb(), b));
          V3<S> Vc = y == 0 ? ld3(ws.fvx(), b) + cross(Om, cs - cb) : (y == 1 ? ld3(ws.fvp(), b) + cross(Om, cs - pb) : ld3(ws.Fb(), b) + cross(Om, cs - cb));
          V3<S> dV = z3, dO = z3;
          if (ins) {
            if (turn) { dV = cross(cross(OmP[y], ax), cs - o) + cross(ax, Vc - od[y]); dO = cross(ax, Om - OmP[y]); }
            else dV = cross(OmP[y], ax);
          }
          rel[y] = rel[y] + (Vc + cross(Om, pc)) * sg;
          drel[y] = drel[y] + (dV + cross(dO, pc) + cross(Om, dpc)) * sg;
        }
      }
      S D = ws.cD()[c], post = ws.cpost()[c], bd = ws.cbd()[c], mu = ws.cmu()[c], dD = ws.cdD()[c] * dr, dpost = ws.cdpost()[c] * dr;
#pragma unroll 1
      for (int e = 0; e < n; ++e) {
        if (!ws.active()[r0 + e]) continue;
        V3<S> dir = nrm, ddir = dn;
        if (n == 4) { S sg = (e & 1) ? -mu : mu; dir = nrm + (e < 2 ? t1 : t2) * sg; ddir = dn + (e < 2 ? dt1 : dt2) * sg; }
        S JX = dot(dir, rel[0]), JV = dot(dir, rel[1]), JW = dot(dir, rel[2]);
        S dJX = dot(ddir, rel[0]) + dot(dir, drel[0]), dJV = dot(ddir, rel[1]) + dot(dir, drel[1]), dJW = dot(ddir, rel[2]) + dot(dir, drel[2]);
        S s = JX - post + bd * JV;
        contrib = contrib + dJW * D * s + JW * dD * s + JW * D * (dJX - dpost + bd * dJV);
      }
    }
    ws.J()[it] = contrib;
  }
  gr.sync();
#pragma unroll 1
  for (int j = gr.lane; j < nv; j += G) {
    S acc(0.0);
#pragma unroll 1
    for (int c = 0; c < nc; ++c) acc = acc + ws.J()[c * nv + j];
    qbar[j] = qbar[j] - (double)acc;
  }
  gr.sync();
}

// ---- parameter part, closed form: S is linear in each body mass (dS/dm_b = S_b / m_b) and depends on a pair's
// friction / solref / solimp only through the scalars (D, position term, b, mu) of that pair's candidates; the row
// velocities J_e y come from the bodies' twists at the stored contact points.  One lane per body, then per
// (pair, parameter slot).  Needs what vjp_config_bodies left in ws (F, N in ws.Isub; twists).
template <class WS, class R, int G, class IN, class AOUT>
DMX_D void vjp_params(const ModelDev<R>& m, const IN& in, const WS& ws, bool cfd, const AOUT& pbar, const Grp<G>& gr) {
  typedef typename WS::S S;
  const int nc = ws.nc(m);
#pragma unroll 1
  for (int b = gr.lane; b < m.nbody; b += G) {
    S g(0.0);
    if (b > 0) g = (dot(ld3(ws.Fb(), b), ld3(ws.Isub(), 3 * b)) + dot(ld3(ws.Nb(), b), ld3(ws.Isub(), 3 * b + 1))) / in.p(b);
    pbar[b] = -(double)g;
  }
#pragma unroll 1
  for (int it = gr.lane; it < 8 * m.npair; it += G) {
    const int pr = it >> 3, k = it & 7;
    const int ip = k == 0 ? m.p_fric + pr : (k < 3 ? m.p_solref + 2 * pr + (k - 1) : m.p_solimp + 5 * pr + (k - 3));
    S acc(0.0);
#pragma unroll 1
    for (int c = 0; c < nc; ++c) {
      const int n = ws.incl()[c];
      if (n == 0 || m.ct_pair[c] != pr) continue;
      const int r0 = ws.rowstart()[c];
      bool any = false;
      for (int e = 0; e < n; ++e) any = any || ws.active()[r0 + e];
      if (!any) continue;
      S z(0.0);
      V3<S> pos = ld3(ws.cpos(), c), dX = mk3<S>(z, z, z), dV = dX, dW = dX;
#pragma unroll 1
      for (int side = 0; side < 2; ++side) {
        const int b = side ? m.ct_b2[c] : m.ct_b1[c];
        if (b == 0) continue;
        S sg = side ? S(1.0) : S(-1.0);
        V3<S> rc = pos - ld3(ws.com(), b);
        dX = dX + (ld3(ws.fvx(), b) + cross(ld3(ws.fox(), b), rc)) * sg;
        dV = dV + (ld3(ws.fvp(), b) + cross(ld3(ws.fw(), b), pos - ld3(ws.fp(), b))) * sg;
        dW = dW + (ld3(ws.Fb(), b) + cross(ld3(ws.Nb(), b), rc)) * sg;
      }
      V3<S> nrm = ld3(ws.cn(), c), t1 = ld3(ws.ct1(), c), t2 = ld3(ws.ct2(), c);
      InDual<S, WS::ST> din; din.pa = in.pa; din.kind = 3; din.idx = ip;
      Dual<S> Dw, post, bd, mu;
      candidate_terms_dual<R, InDual<S, WS::ST> >(m, din, c, Dual<S>(ws.cr()[c]), cfd, Dw, post, bd, mu);
      S nX = dot(nrm, dX), nV = dot(nrm, dV), nW = dot(nrm, dW);
      S tX[2] = {dot(t1, dX), dot(t2, dX)}, tV[2] = {dot(t1, dV), dot(t2, dV)}, tW[2] = {dot(t1, dW), dot(t2, dW)};
#pragma unroll 1
      for (int e = 0; e < n; ++e) {
        if (!ws.active()[r0 + e]) continue;
        Dual<S> JX(nX), JV(nV), JW(nW);
        if (n == 4) {
          Dual<S> sg = (e & 1) ? -mu : mu;
          int a = e >> 1;
          JX = JX + sg * Dual<S>(tX[a]); JV = JV + sg * Dual<S>(tV[a]); JW = JW + sg * Dual<S>(tW[a]);
        }
        acc = acc + (JW * (Dw * (JX - (post - bd * JV)))).d;
      }
    }
    pbar[ip] = -(double)acc;
  }
  gr.sync();
}

}  // namespace dmx
