// ORACLE — test infrastructure only (see oracle/README.md). Not part of the product path.
//
// The vector field F_theta(t,x) of PAPER.md Eq. (1)/(5): v' = M^-1 (tau - c + J^T f), with f from
// the contact problem Eq. (2); its CFD variant F~; and the vector-Jacobian
// product of either.  The VJP uses the implicit function theorem on the
// stationarity condition of Eq. (2) at the final active set A (reading G9; the paper itself
// proposes implicit differentiation of the solver):
//     g(z; x) = ID(q,v,x) - tau(q,v,u) + sum_{i in A} J_i^T D_i (J_i x - aref_i) = 0,
//     dx*/dz = -H^-1 dg/dz,  H = M + J_A^T D_A J_A   =>   zbar = -(dg/dz)^T H^-1 kappa.
// dg/dz is obtained by forward-mode tangents (dual.hpp) through the same templated routines
// that evaluate F, with x*, A and w = H^-1 kappa held fixed.
#pragma once
#include "contact.hpp"
#include "solve.hpp"

namespace orc {

struct FieldOut {
  std::vector<double> acc;       // v' (= x*)
  std::vector<double> M, a0;
  Rows<double> rows;
  SolveResult sol;
  bool ok = true;
};

inline FieldOut vector_field(const Model& m, const double* q, const double* v, const double* u,
                             const double* p, bool cfd) {
  FieldOut o;
  int nv = m.nv;
  std::vector<double> zero(nv, 0.0), c(nv), tau(nv);
  Kin<double> k; kinematics(m, q, v, zero.data(), k);
  o.M.assign(nv * nv, 0.0);
  mass_matrix(m, q, p + m.p_mass(), o.M.data());
  inverse_dynamics(m, q, v, zero.data(), p + m.p_mass(), c.data());      // bias force c(q,v)
  applied_force(m, q, v, u, tau.data());
  std::vector<double> L = o.M;
  if (!cholesky(L, nv)) { o.ok = false; o.acc.assign(nv, NAN); return o; }
  o.a0.resize(nv);
  for (int j = 0; j < nv; ++j) o.a0[j] = tau[j] - c[j];
  chol_solve(L, nv, o.a0.data());
  build_rows(m, k, v, p, cfd, o.rows);
  o.sol = contact_solve(nv, o.rows.nr, o.M, o.a0.data(), o.rows.J, o.rows.aref.data(), o.rows.D.data(),
                        m.newton_iters, m.ls_iters);
  o.acc = o.sol.x;
  for (int j = 0; j < nv; ++j) if (!std::isfinite(o.acc[j])) o.ok = false;
  return o;
}

// residual g(z; x*) of the stationarity condition, templated (see header)
template <class S>
void residual(const Model& m, const S* q, const S* v, const S* u, const S* p, const double* xstar,
              const std::vector<char>& active, bool cfd, S* g) {
  int nv = m.nv;
  std::vector<S> xs(nv), tau(nv), zero(nv, S(0.0));
  for (int j = 0; j < nv; ++j) xs[j] = S(xstar[j]);
  inverse_dynamics(m, q, v, xs.data(), p + m.p_mass(), g);
  applied_force(m, q, v, u, tau.data());
  for (int j = 0; j < nv; ++j) g[j] = g[j] - tau[j];
  Kin<S> k; kinematics(m, q, v, zero.data(), k);
  Rows<S> R; build_rows(m, k, v, p, cfd, R);
  for (int i = 0; i < R.nr; ++i) if (active[i]) {
    S s(0.0);
    for (int j = 0; j < nv; ++j) s = s + R.J[i][j] * xs[j];
    s = s - R.aref[i];
    for (int j = 0; j < nv; ++j) g[j] = g[j] + R.J[i][j] * (R.D[i] * s);
  }
}

// tangent direction d of the configuration: q (+) eps e_d  (D2; free-joint rotation in body frame)
inline void q_tangent_dir(const Model& m, const double* q, int d, double* dq) {
  for (int i = 0; i < m.nq; ++i) dq[i] = 0.0;
  int j = m.dof_jnt[d], c = d - m.jnt_vadr[j], qa = m.jnt_qadr[j];
  if (m.jnt_type[j] != JNT_FREE || c < 3) { dq[qa + c] = 1.0; return; }
  const double* w = q + qa + 3;                       // d/de [ w (x) (1, e/2) ]
  double e[3] = {0, 0, 0}; e[c - 3] = 0.5;
  dq[qa + 3] = -w[1] * e[0] - w[2] * e[1] - w[3] * e[2];
  dq[qa + 4] = w[0] * e[0] + w[2] * e[2] - w[3] * e[1];
  dq[qa + 5] = w[0] * e[1] - w[1] * e[2] + w[3] * e[0];
  dq[qa + 6] = w[0] * e[2] + w[1] * e[1] - w[2] * e[0];
}

struct VjpOut { std::vector<double> qbar, vbar, ubar, pbar; FieldOut f; };

// (qbar, vbar, ubar, pbar) = kappa^T dF/d(q,v,u,p) at (q,v,u,p); F~ when cfd.  O11, O12.
inline VjpOut vjp_field(const Model& m, const double* q, const double* v, const double* u, const double* p,
                        const double* kappa, bool cfd, bool want_p) {
  VjpOut o;
  int nv = m.nv, nq = m.nq, nu = m.nu, np = m.np;
  o.f = vector_field(m, q, v, u, p, cfd);
  o.qbar.assign(nv, 0.0); o.vbar.assign(nv, 0.0); o.ubar.assign(nu, 0.0); o.pbar.assign(np, 0.0);
  if (!o.f.ok) return o;
  std::vector<double> H = o.f.M, w(kappa, kappa + nv);
  const Rows<double>& R = o.f.rows;
  for (int i = 0; i < R.nr; ++i) if (o.f.sol.active[i])
    for (int a = 0; a < nv; ++a) for (int b = 0; b < nv; ++b) H[a * nv + b] += R.D[i] * R.J[i][a] * R.J[i][b];
  if (!cholesky(H, nv)) { o.f.ok = false; return o; }
  chol_solve(H, nv, w.data());
  int ndir = 2 * nv + nu + (want_p ? np : 0);
  std::vector<Dual> qd(nq), vd(nv), ud(nu), pd(np), g(nv);
  std::vector<double> dq(nq);
  for (int d0 = 0; d0 < ndir; d0 += ND) {
    for (int i = 0; i < nq; ++i) qd[i] = Dual(q[i]);
    for (int i = 0; i < nv; ++i) vd[i] = Dual(v[i]);
    for (int i = 0; i < nu; ++i) ud[i] = Dual(u[i]);
    for (int i = 0; i < np; ++i) pd[i] = Dual(p[i]);
    for (int l = 0; l < ND && d0 + l < ndir; ++l) {
      int d = d0 + l;
      if (d < nv) { q_tangent_dir(m, q, d, dq.data()); for (int i = 0; i < nq; ++i) qd[i].d[l] = dq[i]; }
      else if (d < 2 * nv) vd[d - nv].d[l] = 1.0;
      else if (d < 2 * nv + nu) ud[d - 2 * nv].d[l] = 1.0;
      else pd[d - 2 * nv - nu].d[l] = 1.0;
    }
    residual<Dual>(m, qd.data(), vd.data(), ud.data(), pd.data(), o.f.acc.data(), o.f.sol.active, cfd, g.data());
    for (int l = 0; l < ND && d0 + l < ndir; ++l) {
      int d = d0 + l;
      double s = 0.0;
      for (int j = 0; j < nv; ++j) s -= w[j] * g[j].d[l];
      if (d < nv) o.qbar[d] = s; else if (d < 2 * nv) o.vbar[d - nv] = s;
      else if (d < 2 * nv + nu) o.ubar[d - 2 * nv] = s; else o.pbar[d - 2 * nv - nu] = s;
    }
  }
  return o;
}

}  // namespace orc
