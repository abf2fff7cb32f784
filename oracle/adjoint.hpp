// ORACLE — test infrastructure only (see oracle/README.md). Not part of the product path.
//
// Optimize-then-discretize (Eq. 6-7; with Contacts From Distance PAPER.md:462-477, Eq. 8-9): the
// gradient of a terminal loss as the solution of the continuous adjoint equations
//     a_x(T) = dL/dx(T),   a_x' = -a_x^T dF/dx (t, x(t)),      a_theta(T) = 0,   a_theta' = -a_x^T dF/dtheta,
// (F~ in place of F when CFD is on) solved BACKWARDS with its own error-controlled steps, so that the step size follows
// the stiffness of the adjoint equation and not that of the forward one (Fig. 19).
//
// Reading G21: the paper delegates this to a library and prints no scheme.  Here
//  - the state x(t) comes from the tape of the forward solve: inside the accepted step [t_n, t_n+1] it is the cubic
//    Hermite interpolant of (Theta, v) in the chart Q = q_n (+) Theta of that step, from the end values and end rates
//    (Theta = 0, Theta' = v_n, v' = A_1 at t_n; Theta_n+1, Theta' = K(Theta_n+1, v_n+1), v' = F(y_n+1) at t_n+1);
//  - the adjoint is carried in the coordinates of the same chart, mu = (mu_Theta, mu_v): at t_n+1 it is the pullback
//    Jr(Theta_n+1)^T of the tangent cotangent lambda_n+1, at t_n (Theta = 0) it IS lambda_n;
//  - in reversed time s = t_n+1 - t the system is  mu' = G^T mu,  with
//        G^T mu = ( dK/dTheta^T mu_Theta + Jr(Theta)^T qbar ,  dK/dV^T mu_Theta + vbar ),
//        (qbar, vbar, ubar, pbar) = VJP of F (or F~) at (q_n (+) Theta, v) with kappa = mu_v,
//    integrated with the same embedded pair and PI controller as the forward solve (error norm over the 2 nv adjoint
//    components), steps clipped to the checkpoint times; the controller's proposal carries across checkpoints;
//  - dL/du[knot] and dL/dp accumulate  hs sum_i b_i ubar_i  and  hs sum_i b_i pbar_i  over the accepted sub-steps.
#pragma once
#include "rk.hpp"

namespace orc {

struct AdjStats { int n_accept = 0, n_reject = 0, status = 0; };

// one evaluation of the reversed-time adjoint right-hand side at tau in [0,1] of the step (q_n, h)
struct AdjStep {
  const Model& m; const double* qn; const double* u; const double* p; bool cfd, want_p; double h;
  std::vector<double> z0, dz0, z1, dz1;     // Hermite data, each 2 nv: (Theta, v) and their rates
  bool ok = true;
  void state(double tau, double* Theta, double* v) const {
    int nv = m.nv;
    double t2 = tau * tau, t3 = t2 * tau;
    double h00 = 2 * t3 - 3 * t2 + 1, h10 = t3 - 2 * t2 + tau, h01 = -2 * t3 + 3 * t2, h11 = t3 - t2;
    for (int j = 0; j < nv; ++j) {
      Theta[j] = h00 * z0[j] + h10 * h * dz0[j] + h01 * z1[j] + h11 * h * dz1[j];
      v[j] = h00 * z0[nv + j] + h10 * h * dz0[nv + j] + h01 * z1[nv + j] + h11 * h * dz1[nv + j];
    }
  }
  // k = G^T mu (2 nv), ubar, pbar
  void rhs(double tau, const double* mu, double* k, double* ubar, double* pbar) {
    int nv = m.nv;
    std::vector<double> Theta(nv), v(nv), Q(m.nq), Vbar(nv, 0.0), dbar(nv, 0.0), base(nv, 0.0);
    state(tau, Theta.data(), v.data());
    retract(m, qn, Theta.data(), Q.data());
    VjpOut vj = vjp_field(m, Q.data(), v.data(), u, p, mu + nv, cfd, want_p);
    if (!vj.f.ok) ok = false;
    chart_rate_pullback(m, Theta.data(), v.data(), mu, Vbar.data(), dbar.data());
    retract_pullback(m, Theta.data(), vj.qbar.data(), base.data(), dbar.data());   // dbar += Jr(Theta)^T qbar
    for (int j = 0; j < nv; ++j) { k[j] = dbar[j]; k[nv + j] = Vbar[j] + vj.vbar[j]; }
    for (int a = 0; a < m.nu; ++a) ubar[a] = vj.ubar[a];
    if (want_p) for (int a = 0; a < m.np; ++a) pbar[a] = vj.pbar[a];
  }
};

// lam (2 nv) in: cotangent at x_T, out: cotangent at x_0.  gctrl[nknot*nu], gp[np] accumulated (may be null).
inline bool reverse_sweep_continuous(const Model& m, const std::vector<TapeRec>& tape, const double* ctrl, int nknot,
                                     const double* p, const SolverOpts& so, const SolverOpts& sa, bool cfd, double* lam,
                                     double* gctrl, double* gp, AdjStats& st, const double* hs_replay = nullptr, int n_replay = 0,
                                     std::vector<double>* hs_out = nullptr) {
  // hs_replay: if non-null, exactly these sub-steps are taken in order (no error control), like h_replay of the forward
  // solve; hs_out collects the accepted sub-steps
  Tableau T = sa.tableau == 0 ? dopri5() : tsit5();
  Tableau Tf = so.tableau == 0 ? dopri5() : tsit5();
  int nv = m.nv, nu = m.nu, np = m.np, n2 = 2 * nv;
  std::vector<double> uzero(nu > 0 ? nu : 1, 0.0);
  StepWork W;
  double hprop = -1.0, Eprev = 1.0; int attempts = 0, ir = 0;
  st = AdjStats();
  std::vector<std::vector<double>> k(7, std::vector<double>(n2)), ub(7, std::vector<double>(nu > 0 ? nu : 1)), pb(7, std::vector<double>(np));
  std::vector<double> mu(n2), mus(n2), munew(n2), err(n2);
  for (int n = (int)tape.size() - 1; n >= 0; --n) {
    const TapeRec& r = tape[n];
    const double* u = (nknot > 0 && nu > 0) ? ctrl + (size_t)r.knot * nu : uzero.data();
    double h = r.h;
    rk_attempt(m, Tf, r.q.data(), r.v.data(), u, p, h, false, W);          // stage rates of the forward step (the tape's content)
    if (!W.ok) return false;
    AdjStep S{m, r.q.data(), u, p, cfd, gp != nullptr, h};
    S.z0.assign(n2, 0.0); S.dz0.resize(n2); S.z1.resize(n2); S.dz1.resize(n2);
    for (int j = 0; j < nv; ++j) {
      S.z0[nv + j] = r.v[j]; S.dz0[j] = r.v[j]; S.dz0[nv + j] = W.A[0][j];
      S.z1[j] = W.Dl[6][j]; S.z1[nv + j] = W.V[6][j]; S.dz1[j] = W.K[6][j]; S.dz1[nv + j] = W.A[6][j];
    }
    // lambda_n+1 (tangent coordinates at y_n+1) -> chart coordinates: mu_Theta = Jr(Theta_n+1)^T lambda_q
    {
      std::vector<double> base(nv, 0.0), dbar(nv, 0.0);
      retract_pullback(m, S.z1.data(), lam, base.data(), dbar.data());
      for (int j = 0; j < nv; ++j) { mu[j] = dbar[j]; mu[nv + j] = lam[nv + j]; }
    }
    if (hprop < 0) hprop = h;
    double s = 0.0; bool have_k1 = false;
    while (s < h) {
      if (attempts >= sa.max_steps) { st.status = 1; return false; }
      double rem = h - s, hs; bool hits;
      if (hs_replay) {
        if (ir >= n_replay || !(hs_replay[ir] > 0.0)) { st.status = 1; return false; }
        hs = hs_replay[ir++]; hits = (hs == rem);
        if (hs > rem) { st.status = 3; return false; }
      } else {
        if (hprop * (1.0 + 1e-7) >= rem) { hs = rem; hits = true; } else { hs = hprop; hits = false; }
        if (!hits && hs < 1e-14 * std::fmax(1.0, h)) { st.status = 2; return false; }
      }
      attempts++;
      for (int i = 0; i < 7; ++i) {
        if (i == 0 && have_k1) continue;
        for (int j = 0; j < n2; ++j) { double a = 0; for (int l = 0; l < i; ++l) a += T.a[i][l] * k[l][j]; mus[j] = mu[j] + hs * a; }
        S.rhs(1.0 - (s + T.c[i] * hs) / h, mus.data(), k[i].data(), ub[i].data(), pb[i].data());
      }
      if (!S.ok) return false;
      have_k1 = true;
      bool finite = true;
      for (int j = 0; j < n2; ++j) {
        double a = 0, e = 0;
        for (int i = 0; i < 6; ++i) a += T.b[i] * k[i][j];
        for (int i = 0; i < 7; ++i) e += T.e[i] * k[i][j];
        munew[j] = mu[j] + hs * a; err[j] = hs * e;
        if (!std::isfinite(err[j]) || !std::isfinite(munew[j])) finite = false;
      }
      double E = INFINITY; bool accept = false;
      if (hs_replay) { if (!finite) return false; accept = true; E = 1.0; }
      else if (finite) {
        double acc = 0.0;
        for (int j = 0; j < n2; ++j) { double q = err[j] / (sa.atol + sa.rtol * std::fmax(std::fabs(mu[j]), std::fabs(munew[j]))); acc = acc + q * q; }
        E = std::sqrt(acc / n2); accept = E <= 1.0;
      }
      double Ec = std::fmax(E, 1e-30);
      double fac = finite ? sa.safety * std::exp(-(sa.pcoeff + sa.icoeff) / 5.0 * std::log(Ec)) * std::exp(sa.pcoeff / 5.0 * std::log(Eprev)) : sa.fac_min;
      fac = std::fmin(sa.fac_max, std::fmax(sa.fac_min, fac));
      if (!accept || !hits) hprop = hs * fac;
      if (!accept) { st.n_reject++; continue; }
      Eprev = Ec; st.n_accept++;
      if (hs_out) hs_out->push_back(hs);
      if (gctrl && nknot > 0) for (int a = 0; a < nu; ++a) { double t = 0; for (int i = 0; i < 6; ++i) t += T.b[i] * ub[i][a]; gctrl[(size_t)r.knot * nu + a] += hs * t; }
      if (gp) for (int a = 0; a < np; ++a) { double t = 0; for (int i = 0; i < 6; ++i) t += T.b[i] * pb[i][a]; gp[a] += hs * t; }
      mu = munew; k[0] = k[6]; ub[0] = ub[6]; pb[0] = pb[6];      // FSAL inside the step
      s = hits ? h : s + hs;
    }
    for (int j = 0; j < n2; ++j) lam[j] = mu[j];                  // Theta = 0 at t_n: chart coordinates = tangent coordinates
  }
  return true;
}

}  // namespace orc
