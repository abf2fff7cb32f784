// ORACLE — test infrastructure only (see oracle/README.md). Not part of the product path.
//
// O8-O10 of SURVEY.md §8(c): embedded Runge-Kutta pair on the configuration manifold
// (PAPER.md:88 adaptive integration; PAPER.md:429 exact quaternion integration; Dopri5 /
// Tsit5), PI step-size controller (P=0.2 I=0.4 D=0;
// formulas: reading G12), and the discrete adjoint through the accepted steps with frozen
// step sizes (discretize-then-optimize; reading G15).
#pragma once
#include "field.hpp"

namespace orc {

struct Tableau { int s; double c[7], a[7][7], b[7], e[7]; /* e = b - bhat */ };

inline Tableau dopri5() {   // Dormand & Prince 1980; reading G11
  Tableau T{}; T.s = 7;
  double c[7] = {0, 1.0 / 5, 3.0 / 10, 4.0 / 5, 8.0 / 9, 1, 1};
  double a[7][7] = {{0},
                    {1.0 / 5},
                    {3.0 / 40, 9.0 / 40},
                    {44.0 / 45, -56.0 / 15, 32.0 / 9},
                    {19372.0 / 6561, -25360.0 / 2187, 64448.0 / 6561, -212.0 / 729},
                    {9017.0 / 3168, -355.0 / 33, 46732.0 / 5247, 49.0 / 176, -5103.0 / 18656},
                    {35.0 / 384, 0, 500.0 / 1113, 125.0 / 192, -2187.0 / 6784, 11.0 / 84}};
  double b[7] = {35.0 / 384, 0, 500.0 / 1113, 125.0 / 192, -2187.0 / 6784, 11.0 / 84, 0};
  double bh[7] = {5179.0 / 57600, 0, 7571.0 / 16695, 393.0 / 640, -92097.0 / 339200, 187.0 / 2100, 1.0 / 40};
  for (int i = 0; i < 7; ++i) { T.c[i] = c[i]; T.b[i] = b[i]; T.e[i] = b[i] - bh[i]; for (int j = 0; j < 7; ++j) T.a[i][j] = a[i][j]; }
  return T;
}
inline Tableau tsit5() {    // Tsitouras 2011, Table 1; reading G11, accepted by pin P9
  Tableau T{}; T.s = 7;
  double c[7] = {0, 0.161, 0.327, 0.9, 0.9800255409045097, 1, 1};
  double a[7][7] = {{0},
                    {0.161},
                    {-0.008480655492356989, 0.335480655492357},
                    {2.8971530571054935, -6.359448489975075, 4.3622954328695815},
                    {5.325864828439257, -11.748883564062828, 7.4955393428898365, -0.09249506636175525},
                    {5.86145544294642, -12.92096931784711, 8.159367898576159, -0.071584973281401, -0.028269050394068383},
                    {0.09646076681806523, 0.01, 0.4798896504144996, 1.379008574103742, -3.290069515436081, 2.324710524099774}};
  double e[7] = {-0.00178001105222577714, -0.0008164344596567469, 0.007880878010261995, -0.1447110071732629,
                 0.5823571654525552, -0.45808210592918697, 0.015151515151515152};
  for (int i = 0; i < 7; ++i) { T.c[i] = c[i]; T.b[i] = a[6][i]; T.e[i] = e[i]; for (int j = 0; j < 7; ++j) T.a[i][j] = a[i][j]; }
  T.b[6] = 0.0;
  return T;
}

// ---- D2: the retraction q (+) delta and its Jacobians --------------------------------------
inline void rotvec_to_quat(const double* d, double* e) {     // exp(delta/2) as (w,x,y,z)
  double th2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2], th = std::sqrt(th2);
  double k = th < 1e-4 ? 0.5 - th2 / 48.0 : std::sin(0.5 * th) / th;
  e[0] = std::cos(0.5 * th); e[1] = k * d[0]; e[2] = k * d[1]; e[3] = k * d[2];
}
inline void quat_mul(const double* a, const double* b, double* r) {
  r[0] = a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3];
  r[1] = a[0] * b[1] + a[1] * b[0] + a[2] * b[3] - a[3] * b[2];
  r[2] = a[0] * b[2] - a[1] * b[3] + a[2] * b[0] + a[3] * b[1];
  r[3] = a[0] * b[3] + a[1] * b[2] - a[2] * b[1] + a[3] * b[0];
}
// qout = q (+) delta ; delta in R^nv
inline void retract(const Model& m, const double* q, const double* delta, double* qout) {
  for (int j = 0; j < m.njnt; ++j) {
    int qa = m.jnt_qadr[j], va = m.jnt_vadr[j];
    if (m.jnt_type[j] != JNT_FREE) { qout[qa] = q[qa] + delta[va]; continue; }
    for (int c = 0; c < 3; ++c) qout[qa + c] = q[qa + c] + delta[va + c];
    double e[4], r[4]; rotvec_to_quat(delta + va + 3, e); quat_mul(q + qa + 3, e, r);
    double n = std::sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2] + r[3] * r[3]);
    for (int c = 0; c < 4; ++c) qout[qa + 3 + c] = r[c] / n;
  }
}
inline void rotvec_to_mat(const double* d, double R[3][3]) {  // R(exp delta), Rodrigues
  double th2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2], th = std::sqrt(th2);
  double A = th < 1e-4 ? 1.0 - th2 / 6.0 : std::sin(th) / th;
  double B = th < 1e-4 ? 0.5 - th2 / 24.0 : (1.0 - std::cos(th)) / th2;
  double K[3][3] = {{0, -d[2], d[1]}, {d[2], 0, -d[0]}, {-d[1], d[0], 0}};
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
    double k2 = 0; for (int l = 0; l < 3; ++l) k2 += K[i][l] * K[l][j];
    R[i][j] = (i == j ? 1.0 : 0.0) + A * K[i][j] + B * k2;
  }
}
inline void right_jacobian(const double* d, double Jr[3][3]) {  // I - (1-cos)/th^2 K + (th-sin)/th^3 K^2
  double th2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2], th = std::sqrt(th2);
  double B = th < 1e-4 ? 0.5 - th2 / 24.0 : (1.0 - std::cos(th)) / th2;
  double C = th < 1e-4 ? 1.0 / 6.0 - th2 / 120.0 : (th - std::sin(th)) / (th2 * th);
  double K[3][3] = {{0, -d[2], d[1]}, {d[2], 0, -d[0]}, {-d[1], d[0], 0}};
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
    double k2 = 0; for (int l = 0; l < 3; ++l) k2 += K[i][l] * K[l][j];
    Jr[i][j] = (i == j ? 1.0 : 0.0) - B * K[i][j] + C * k2;
  }
}
// Pull a cotangent Qbar (tangent coords at q (+) delta) back to the base point and to delta:
//   base += T^T Qbar with T = blockdiag(I, R(exp delta)^T);  dbar += Jr^T Qbar.
inline void retract_pullback(const Model& m, const double* delta, const double* Qbar, double* base, double* dbar) {
  for (int j = 0; j < m.njnt; ++j) {
    int va = m.jnt_vadr[j];
    if (m.jnt_type[j] != JNT_FREE) { base[va] += Qbar[va]; dbar[va] += Qbar[va]; continue; }
    for (int c = 0; c < 3; ++c) { base[va + c] += Qbar[va + c]; dbar[va + c] += Qbar[va + c]; }
    double R[3][3], Jr[3][3]; rotvec_to_mat(delta + va + 3, R); right_jacobian(delta + va + 3, Jr);
    for (int i = 0; i < 3; ++i) for (int l = 0; l < 3; ++l) {
      base[va + 3 + i] += R[i][l] * Qbar[va + 3 + l];          // (R^T)^T = R
      dbar[va + 3 + i] += Jr[l][i] * Qbar[va + 3 + l];         // Jr^T
    }
  }
}

// Chart rate (reading G10): with Q = q_n (+) Theta the rotation vector obeys
// Theta' = dexp^-1_Theta(w_body).  Summing raw body rates of different stages would cap the
// order at 2 for tumbling bodies; the Munthe-Kaas correction truncated after the B_2 term
//   K = w + 1/2 Theta x w + 1/12 Theta x (Theta x w)
// keeps order 5 (B_3 = 0) and stays exact for constant body rate (Theta || w).  Other
// coordinates: K = V.
inline void cross3(const double* a, const double* b, double* r) { r[0] = a[1] * b[2] - a[2] * b[1]; r[1] = a[2] * b[0] - a[0] * b[2]; r[2] = a[0] * b[1] - a[1] * b[0]; }
inline void chart_rate(const Model& m, const double* delta, const double* V, double* K) {
  for (int j = 0; j < m.nv; ++j) K[j] = V[j];
  for (int j = 0; j < m.njnt; ++j) if (m.jnt_type[j] == JNT_FREE) {
    const double* th = delta + m.jnt_vadr[j] + 3; const double* w = V + m.jnt_vadr[j] + 3;
    double a[3], b[3]; cross3(th, w, a); cross3(th, a, b);
    for (int c = 0; c < 3; ++c) K[m.jnt_vadr[j] + 3 + c] = w[c] + 0.5 * a[c] + b[c] / 12.0;
  }
}
// cotangent Kbar of K  ->  Vbar += (dK/dV)^T Kbar,  dbar += (dK/dTheta)^T Kbar
inline void chart_rate_pullback(const Model& m, const double* delta, const double* V, const double* Kbar, double* Vbar, double* dbar) {
  for (int j = 0; j < m.njnt; ++j) {
    int va = m.jnt_vadr[j];
    if (m.jnt_type[j] != JNT_FREE) { Vbar[va] += Kbar[va]; continue; }
    for (int c = 0; c < 3; ++c) Vbar[va + c] += Kbar[va + c];
    const double* th = delta + va + 3; const double* w = V + va + 3; const double* kb = Kbar + va + 3;
    double t1[3], t2[3], tw[3], a[3], b[3], c3[3];
    cross3(th, kb, t1); cross3(th, t1, t2);                 // B^T kb = kb - 1/2 th x kb + 1/12 th x (th x kb)
    for (int c = 0; c < 3; ++c) Vbar[va + 3 + c] += kb[c] - 0.5 * t1[c] + t2[c] / 12.0;
    cross3(w, kb, a); cross3(th, w, tw); cross3(tw, kb, b); cross3(w, t1, c3);
    for (int c = 0; c < 3; ++c) dbar[va + 3 + c] += 0.5 * a[c] + b[c] / 12.0 - c3[c] / 12.0;
  }
}

// ---- O8: one attempted step ---------------------------------------------------------------
struct StepWork {
  std::vector<std::vector<double>> Yq, V, A, K, Dl;   // stage configurations, velocities, accelerations, chart rates, increments
  std::vector<double> qn1, vn1, err;           // proposal and error vector (2 nv)
  int unconverged = 0; bool ok = true;
};

// k1 (V[0]=v, A[0]) must be supplied in W.A[0] when have_k1; stages 2..7 evaluated here.
inline void rk_attempt(const Model& m, const Tableau& T, const double* q, const double* v, const double* u,
                       const double* p, double h, bool have_k1, StepWork& W) {
  int nv = m.nv, nq = m.nq;
  W.Yq.assign(7, std::vector<double>(nq)); W.V.assign(7, std::vector<double>(nv));
  W.K.assign(7, std::vector<double>(nv)); W.Dl.assign(7, std::vector<double>(nv));
  if (!have_k1) W.A.assign(7, std::vector<double>(nv)); else W.A.resize(7, std::vector<double>(nv));
  W.unconverged = 0; W.ok = true;
  std::vector<double> dq(nv), dv(nv);
  for (int i = 0; i < 7; ++i) {
    for (int j = 0; j < nv; ++j) {
      double sq = 0, sv = 0;
      for (int l = 0; l < i; ++l) { sq += T.a[i][l] * W.K[l][j]; sv += T.a[i][l] * W.A[l][j]; }
      dq[j] = h * sq; dv[j] = h * sv;
    }
    retract(m, q, dq.data(), W.Yq[i].data());
    for (int j = 0; j < nv; ++j) W.V[i][j] = v[j] + dv[j];
    W.Dl[i] = dq;
    chart_rate(m, dq.data(), W.V[i].data(), W.K[i].data());
    if (i == 0 && have_k1) continue;
    FieldOut f = vector_field(m, W.Yq[i].data(), W.V[i].data(), u, p, false);
    if (!f.ok) W.ok = false;
    if (f.rows.nr > 0 && !f.sol.converged) W.unconverged++;
    W.A[i] = f.acc;
  }
  // a[6][:] = b, so stage 7 is the proposal (FSAL): y_{n+1} = (Yq[6], V[6]), k7 = (V[6], A[6])
  W.qn1 = W.Yq[6]; W.vn1 = W.V[6];
  W.err.assign(2 * nv, 0.0);
  for (int j = 0; j < nv; ++j) {
    double eq = 0, ev = 0;
    for (int i = 0; i < 7; ++i) { eq += T.e[i] * W.K[i][j]; ev += T.e[i] * W.A[i][j]; }
    W.err[j] = h * eq; W.err[nv + j] = h * ev;
  }
}

// ---- O9: error norm (D4: index order, plain adds) -------------------------------------------
inline double error_norm(const Model& m, const double* q0, const double* v0, const double* q1, const double* v1,
                         const double* err, double rtol, double atol) {
  int nv = m.nv; double acc = 0.0;
  for (int d = 0; d < nv; ++d) {
    int j = m.dof_jnt[d], c = d - m.jnt_vadr[j];
    double mag = 1.0;                                        // rotational tangent coordinates: magnitude 1
    if (m.jnt_type[j] != JNT_FREE || c < 3) { int qi = m.jnt_qadr[j] + c; mag = std::fmax(std::fabs(q0[qi]), std::fabs(q1[qi])); }
    double r = err[d] / (atol + rtol * mag);
    acc = acc + r * r;
  }
  for (int d = 0; d < nv; ++d) {
    double r = err[nv + d] / (atol + rtol * std::fmax(std::fabs(v0[d]), std::fabs(v1[d])));
    acc = acc + r * r;
  }
  return std::sqrt(acc / (2 * nv));
}

struct SolverOpts { int tableau; double rtol, atol, h0, pcoeff, icoeff, safety, fac_min, fac_max; int max_steps; };
struct TapeRec { std::vector<double> q, v; double t, h; int knot; };
struct EnvStats { int n_accept = 0, n_reject = 0, n_feval = 0, n_unconv = 0, status = 0; double h_min = INFINITY, h_max = 0, t_end = 0; };

// Rollout of one environment (O8, O9).  ctrl[nknot*nu] zero-order hold (G2).  h_replay: if
// non-null, take exactly these steps (terminated by n_replay or a zero entry), no error control.
inline void rollout_env(const Model& m, const double* x0, const double* ctrl, int nknot, double knot_dt,
                        const double* p, double horizon, const SolverOpts& so, const double* h_replay, int n_replay,
                        double* xT, EnvStats& st, std::vector<TapeRec>* tape) {
  Tableau T = so.tableau == 0 ? dopri5() : tsit5();
  int nq = m.nq, nv = m.nv, nu = m.nu;
  std::vector<double> q(x0, x0 + nq), v(x0 + nq, x0 + nq + nv), k1(nv);
  double t = 0.0, hprop = so.h0, Eprev = 1.0;
  int knot = 0; bool have_k1 = false, last_nonfinite = false; int attempts = 0, ir = 0;
  std::vector<double> uzero(nu > 0 ? nu : 1, 0.0);
  StepWork W; st = EnvStats();
  while (t < horizon) {
    double tb = (nknot > 0 && nu > 0) ? std::fmin((knot + 1) * knot_dt, horizon) : horizon;
    if (knot + 1 >= nknot) tb = horizon;
    const double* u = (nknot > 0 && nu > 0) ? ctrl + (size_t)knot * nu : uzero.data();
    double rem = tb - t, h; bool hits;
    if (h_replay) {
      if (ir >= n_replay || !(h_replay[ir] > 0.0)) break;
      h = h_replay[ir++]; hits = (h == rem);
    } else {
      if (attempts >= so.max_steps) { st.status = 1; break; }
      if (hprop * (1.0 + 1e-7) >= rem) { h = rem; hits = true; } else { h = hprop; hits = false; }
      if (!hits && h < 1e-14 * std::fmax(1.0, std::fabs(t))) { st.status = last_nonfinite ? 3 : 2; break; }
    }
    attempts++;
    if (have_k1) { W.A.resize(7, std::vector<double>(nv)); W.A[0] = k1; }
    rk_attempt(m, T, q.data(), v.data(), u, p, h, have_k1, W);
    st.n_feval += have_k1 ? 6 : 7; st.n_unconv += W.unconverged;
    k1 = W.A[0]; have_k1 = true;
    bool finite = W.ok;
    for (double e : W.err) if (!std::isfinite(e)) finite = false;
    double E = 0.0; bool accept = true;
    last_nonfinite = !finite;
    if (!h_replay) {
      if (!finite) { E = INFINITY; accept = false; }
      else { E = error_norm(m, q.data(), v.data(), W.qn1.data(), W.vn1.data(), W.err.data(), so.rtol, so.atol); accept = E <= 1.0; }
      double Ec = std::fmax(E, 1e-30);
      double fac = finite ? so.safety * std::exp(-(so.pcoeff + so.icoeff) / 5.0 * std::log(Ec)) * std::exp(so.pcoeff / 5.0 * std::log(Eprev)) : so.fac_min;
      fac = std::fmin(so.fac_max, std::fmax(so.fac_min, fac));
      if (!accept || !hits) hprop = h * fac;               // a clipped accepted step keeps the proposal (G2)
      if (accept) Eprev = Ec;
    } else if (!finite) { st.status = 3; break; }
    if (!accept) { st.n_reject++; continue; }
    if (tape) { TapeRec r; r.q = q; r.v = v; r.t = t; r.h = h; r.knot = knot; tape->push_back(r); }
    q = W.qn1; v = W.vn1; st.n_accept++;
    st.h_min = std::fmin(st.h_min, h); st.h_max = std::fmax(st.h_max, h);
    if (hits) {
      t = tb;
      if (tb < horizon) { knot++; have_k1 = false; }        // control changes: FSAL stage is stale
      else k1 = W.A[6];
    } else { t += h; k1 = W.A[6]; }
  }
  st.t_end = t;
  for (int i = 0; i < nq; ++i) xT[i] = q[i];
  for (int i = 0; i < nv; ++i) xT[nq + i] = v[i];
}

// ambient gradient (nq+nv) at x -> tangent cotangent (2 nv):  E(q)^T g
inline void ambient_to_tangent(const Model& m, const double* x, const double* g, double* lam) {
  std::vector<double> dq(m.nq);
  for (int d = 0; d < m.nv; ++d) {
    q_tangent_dir(m, x, d, dq.data());
    double s = 0; for (int i = 0; i < m.nq; ++i) s += dq[i] * g[i];
    lam[d] = s; lam[m.nv + d] = g[m.nq + d];
  }
}

// O10: reverse sweep over the tape.  lam (2nv) in/out; gctrl[nknot*nu], gp[np] accumulated.
inline bool reverse_sweep(const Model& m, const std::vector<TapeRec>& tape, const double* ctrl, int nknot,
                          const double* p, const SolverOpts& so, bool cfd, double* lam, double* gctrl, double* gp) {
  Tableau T = so.tableau == 0 ? dopri5() : tsit5();
  int nv = m.nv, nu = m.nu, np = m.np;
  std::vector<double> uzero(nu > 0 ? nu : 1, 0.0);
  StepWork W;
  for (int n = (int)tape.size() - 1; n >= 0; --n) {
    const TapeRec& r = tape[n];
    const double* u = (nknot > 0 && nu > 0) ? ctrl + (size_t)r.knot * nu : uzero.data();
    double h = r.h;
    rk_attempt(m, T, r.q.data(), r.v.data(), u, p, h, false, W);     // recompute stages with F
    // cotangents of the stage chart rates K_i, velocities V_i and accelerations A_i
    std::vector<std::vector<double>> Kb(6, std::vector<double>(nv, 0.0)), Ab(6, std::vector<double>(nv, 0.0));
    std::vector<double> qb(nv, 0.0), vb(nv, 0.0), dbar(nv), delta(nv), Vb(nv);
    // y_{n+1} = (q_n (+) h sum b_i K_i, v_n + h sum b_i A_i)
    for (int j = 0; j < nv; ++j) { double s = 0; for (int i = 0; i < 6; ++i) s += T.b[i] * W.K[i][j]; delta[j] = h * s; dbar[j] = 0; }
    retract_pullback(m, delta.data(), lam, qb.data(), dbar.data());
    for (int i = 0; i < 6; ++i) for (int j = 0; j < nv; ++j) { Kb[i][j] += h * T.b[i] * dbar[j]; Ab[i][j] += h * T.b[i] * lam[nv + j]; }
    for (int j = 0; j < nv; ++j) vb[j] += lam[nv + j];
    for (int i = 5; i >= 0; --i) {
      // K_i = chart_rate(delta_i, V_i)
      for (int j = 0; j < nv; ++j) { Vb[j] = 0.0; dbar[j] = 0.0; }
      chart_rate_pullback(m, W.Dl[i].data(), W.V[i].data(), Kb[i].data(), Vb.data(), dbar.data());
      // A_i = F(Y_i) (or F~ for the straight-through estimator, Eq. 4)
      VjpOut vj = vjp_field(m, W.Yq[i].data(), W.V[i].data(), u, p, Ab[i].data(), cfd, gp != nullptr);
      if (!vj.f.ok) return false;
      for (int j = 0; j < nv; ++j) Vb[j] += vj.vbar[j];
      if (gctrl && nknot > 0) for (int a = 0; a < nu; ++a) gctrl[(size_t)r.knot * nu + a] += vj.ubar[a];
      if (gp) for (int a = 0; a < np; ++a) gp[a] += vj.pbar[a];
      // Y_i.q = q_n (+) delta_i,  delta_i = h sum_{l<i} a_il K_l
      retract_pullback(m, W.Dl[i].data(), vj.qbar.data(), qb.data(), dbar.data());
      // V_i = v_n + h sum_{l<i} a_il A_l
      for (int j = 0; j < nv; ++j) vb[j] += Vb[j];
      for (int l = 0; l < i; ++l) for (int j = 0; j < nv; ++j) {
        Kb[l][j] += h * T.a[i][l] * dbar[j];
        Ab[l][j] += h * T.a[i][l] * Vb[j];
      }
    }
    for (int j = 0; j < nv; ++j) { lam[j] = qb[j]; lam[nv + j] = vb[j]; }
  }
  return true;
}

}  // namespace orc
