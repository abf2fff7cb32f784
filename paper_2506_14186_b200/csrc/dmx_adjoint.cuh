// dmx_adjoint.cuh — optimize-then-discretize (Eq. 6-7; with CFD PAPER.md:462-477 Eq. 8-9; DESIGN.md
// reading G21): the continuous adjoint solved backwards with its own error-controlled steps, so that the step size
// follows the stiffness of the adjoint equation and not that of the forward one (Fig. 19).
//
// Inside the accepted forward step [t_n, t_n+1] the state is the cubic Hermite interpolant of (Theta, v) in the step's
// chart Q = q_n (+) Theta, from the taped end values and rates (plus one evaluation F(y_n+1)); the adjoint is carried in
// chart coordinates mu = (mu_Theta, mu_v): Jr(Theta_n+1)^T lambda_n+1 at t_n+1, lambda_n at t_n (Theta = 0).  In
// reversed time s = t_n+1 - t:
//   mu' = ( dK/dTheta^T mu_Theta + Jr(Theta)^T qbar ,  dK/dV^T mu_Theta + vbar ),  (qbar, vbar, ubar, pbar) = VJP of F or F~
// at (q_n (+) Theta, v) with kappa = mu_v, integrated with the embedded pair and PI controller of the forward solve
// (error norm over the 2 nv adjoint components, sub-steps clipped to the checkpoints, proposal carried across them).
#pragma once
#include "dmx_kernels.cuh"

namespace dmx {

template <class R> struct AdjointArgs {
  BackwardArgs<R> b;
  SolverOpts sa;            // options of the backward solve
  const double* replay;     // [nenv][n_replay] or null: take exactly these sub-steps, in order, without error control
  int n_replay;
  int* info;                // [nenv][3] or null: accepted sub-steps, rejected sub-steps, status (0 ok, 1 budget, 2 underflow, 3 failed)
};

// ambient gradient at x_T -> tangent cotangent lam = E(q_T)^T g; same arithmetic as backward_kernel
template <class R, int G, int ST>
DMX_DI void ambient_to_tangent(const ModelDev<R>& m, const R* xT, const R* gT, const Rk<ST>& rk, const Grp<G>& gr) {
  const int nq = m.nq, nv = m.nv;
#pragma unroll 1
  for (int d = gr.lane; d < nv; d += G) {
    int j = m.dof_jnt[d], c = d - m.jnt_vadr[j], qa = m.jnt_qadr[j];
    double s;
    if (m.jnt_type[j] != JNT_FREE || c < 3) s = (double)gT[qa + c];
    else {
      double w0 = xT[qa + 3], w1 = xT[qa + 4], w2 = xT[qa + 5], w3 = xT[qa + 6];
      double e0 = c == 3 ? 0.5 : 0.0, e1 = c == 4 ? 0.5 : 0.0, e2 = c == 5 ? 0.5 : 0.0;
      s = (-w1 * e0 - w2 * e1 - w3 * e2) * (double)gT[qa + 3] + (w0 * e0 + w2 * e2 - w3 * e1) * (double)gT[qa + 4] +
          (w0 * e1 - w1 * e2 + w3 * e0) * (double)gT[qa + 5] + (w0 * e2 + w1 * e1 - w2 * e0) * (double)gT[qa + 6];
    }
    rk.lam()[d] = s; rk.lam()[nv + d] = (double)gT[nq + d];
  }
}

// one evaluation of the reversed-time right-hand side at tau in [0,1] of the step (q_n, h): k_i, ubar_i, pbar_i of
// stage i from the stage adjoint in rk.amus.  Returns false when the field evaluation fails.
template <class R, int G, class SH>
DMX_DN bool adjoint_rhs(const ModelDev<R>& m, const BackwardArgs<R>& a, const R* u, const R* p, double h, double tau, int i,
                        const Rk<StrideOf<G>::value>& rk, const Ws<R, StrideOf<G>::value, SH>& ws, const Arr<R, StrideOf<G>::value>& Yqr,
                        const Arr<R, StrideOf<G>::value>& Vr, const Grp<G>& gr, int* n_unc, unsigned long long* work) {
  const int nq = m.nq, nv = m.nv, nu = m.nu, np = m.np, n2 = 2 * nv;
  const double t2 = tau * tau, t3 = t2 * tau;
  const double h00 = 2 * t3 - 3 * t2 + 1, h10 = t3 - 2 * t2 + tau, h01 = -2 * t3 + 3 * t2, h11 = t3 - t2;
#pragma unroll 1
  for (int j = gr.lane; j < nv; j += G) {       // Hermite state: z0 = (0, v_n), z0' = (v_n, A_1); z1, z1' in az1, adz1
    rk.Dl()[j] = h10 * h * rk.v()[j] + h01 * rk.az1()[j] + h11 * h * rk.adz1()[j];
    rk.V()[j] = h00 * rk.v()[j] + h10 * h * rk.A()[j] + h01 * rk.az1()[nv + j] + h11 * h * rk.adz1()[nv + j];
    rk.Vb()[j] = 0; rk.dbar()[j] = 0; rk.qb()[j] = 0;
  }
  gr.sync();
#pragma unroll 1
  for (int jn = gr.lane; jn < m.njnt; jn += G) {
    retract_joint(m, jn, rk.q(), rk.Dl(), rk.V(), rk.Yq(), rk.err());        // err: scratch for the chart rate
    chart_pullback_joint(m, jn, rk.Dl(), rk.V(), rk.amus(), rk.Vb(), rk.dbar());
  }
  gr.sync();
#pragma unroll 1
  for (int j = gr.lane; j < nq; j += G) Yqr[j] = (R)rk.Yq()[j];
#pragma unroll 1
  for (int j = gr.lane; j < nv; j += G) Vr[j] = (R)rk.V()[j];
  gr.sync();
  if (!vjp_stage<R, G, SH>(m, Yqr, Vr, u, p, rk.amus().at(nv), a.cfd != 0, a.want_p != 0, ws, rk, gr, a.dbg, nullptr, n_unc, work)) return false;
#pragma unroll 1
  for (int jn = gr.lane; jn < m.njnt; jn += G) retract_pullback_joint(m, jn, rk.Dl(), rk.qbar(), rk.qb(), rk.dbar());   // dbar += Jr(Theta)^T qbar
  gr.sync();
#pragma unroll 1
  for (int j = gr.lane; j < nv; j += G) { rk.ak()[i * n2 + j] = rk.dbar()[j]; rk.ak()[i * n2 + nv + j] = rk.Vb()[j] + rk.vbar()[j]; }
#pragma unroll 1
  for (int c = gr.lane; c < nu; c += G) rk.aub()[i * nu + c] = rk.ubar()[c];
  if (a.want_p) for (int c = gr.lane; c < np; c += G) rk.apb()[i * np + c] = rk.pbar()[c];
  gr.sync();
  return true;
}

template <class R, int G, class SH>
__global__ void __launch_bounds__(256) adjoint_kernel(const __grid_constant__ ModelDev<R> m_, const __grid_constant__ AdjointArgs<R> aa) {
  const BackwardArgs<R>& a = aa.b;
  unsigned char* smem = dyn_smem;
  CtaConst<R>& cc = cta_const<R>();
  if (threadIdx.x == 0) g_lockstep = a.lockstep;
  load_cta_const<R>(cc, m_, a.wl, a.wl, a.rl, 0);
  const ModelDev<R>& m = cc.m;
  const int ST = StrideOf<G>::value;
  const Grp<G> gr = make_group<G>();
  Rk<ST> rk; Ws<R, ST, SH> ws; Arr<R, ST> Yqr, Vr;
  bind_shared<R, G, SH>(smem, 0, a.wl.size + a.rl.rsize, a.wl.isize, rk, ws, Yqr, Vr, &cc.rl, &cc.wl);
  if (G == 1) rk.b = a.rk_scratch + ((size_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5)) * 32 * (size_t)a.rl.size_adj + (threadIdx.x & 31);
  else rk.b = a.rk_scratch + ((size_t)blockIdx.x * (blockDim.x / G) + threadIdx.x / G) * (size_t)a.rl.size_adj;
  const int nq = m.nq, nv = m.nv, nu = m.nu, np = m.np, nx = nq + nv, n2 = 2 * nv, tabf = a.so.tableau, tab = aa.sa.tableau, rec = a.tp.rec;
  const bool has_ctrl = a.ctrl != nullptr && a.nknot > 0 && nu > 0;
  const int nknot = has_ctrl ? a.nknot : 0;
  const SolverOpts& sa = aa.sa;
  const bool tape_ok = a.tp.meta[0] == TAPE_MAGIC && a.tp.meta[1] == a.nenv && a.tp.meta[2] == rec && a.tp.meta[3] == a.tp.o_A &&
                       a.tp.meta[4] == (a.pl.offset ? 1 : 0) && a.tp.meta[5] == 1 && a.tp.stride == 1;
  bool first_env = true;
#pragma unroll 1
  for (;;) {
    int e = 0;
    if (gr.lane == 0) e = next_env<G>(a.queue, a.pl.order, a.nenv, -1, first_env);
    e = gr.bcast_int(e);
    if (e >= a.nenv) break;
    const R* p = a.params ? a.params + (size_t)e * np : m.p_default;
    const int N = a.tp.hdr[2 * e];
    int knot = a.tp.hdr[2 * e + 1], n_unc = 0, n_acc = 0, n_rej = 0, status = 0, attempts = 0, ir = 0;
    unsigned long long work[3] = {0, 0, 0};
    long long first; int tape_cap;
    tape_slot(a.tp, a.pl, e, first, tape_cap);
    bool good = tape_ok && knot >= 0 && N <= tape_cap && (!a.status || a.status[e] == 0);
    if (good) {
      ambient_to_tangent<R, G, ST>(m, a.xT + (size_t)e * nx, a.dLdxT + (size_t)e * nx, rk, gr);
#pragma unroll 1
      for (int i = gr.lane; i < np; i += G) rk.gp()[i] = 0.0;
      gr.sync();
    }
    double hprop = -1.0, Eprev = 1.0;
    const double* rep = aa.replay ? aa.replay + (size_t)e * aa.n_replay : nullptr;
#pragma unroll 1
    for (int n = N - 1; n >= 0 && good; --n) {
      const R* r = a.tp.data + ((size_t)first + n) * rec;
#pragma unroll 1
      for (int j = gr.lane; j < nq; j += G) rk.q()[j] = (double)r[j];
#pragma unroll 1
      for (int j = gr.lane; j < nv; j += G) rk.v()[j] = (double)r[nq + j];
      double tn, hsgn; tape_load_th(r, a.tp.o_th, tn, hsgn);
      const double h = fabs(hsgn);
      if (hsgn < 0) knot--;
      const R* u = has_ctrl ? a.ctrl + ((size_t)e * nknot + knot) * nu : a.zero_u;
      if (a.tape_stages) for (int j = gr.lane; j < 6 * nv; j += G) rk.A()[j] = (double)r[a.tp.o_A + j];
      gr.sync();
      bool ok; int unc;
      rk_attempt<R, G, SH, true>(m, tabf, rk, Yqr, Vr, u, p, h, false, ws, ok, unc, gr, a.tape_stages != 0, work);
      if (!ok) { good = false; status = 3; break; }
      // end of the step: Theta_n+1 = h sum b_i K_i, v_n+1 = v_n + h sum b_i A_i; rates K(Theta_n+1, v_n+1) and F(y_n+1)
#pragma unroll 1
      for (int j = gr.lane; j < nv; j += G) {
        double sk = 0, sv = 0;
#pragma unroll 1
        for (int i = 0; i < 6; ++i) { sk += TAB_A[tabf][6][i] * rk.K()[i * nv + j]; sv += TAB_A[tabf][6][i] * rk.A()[i * nv + j]; }
        rk.az1()[j] = h * sk; rk.az1()[nv + j] = rk.v()[j] + h * sv;
        rk.Dl()[j] = h * sk; rk.V()[j] = rk.v()[j] + h * sv;
        rk.dbar()[j] = 0; rk.qb()[j] = 0;
      }
      gr.sync();
#pragma unroll 1
      for (int jn = gr.lane; jn < m.njnt; jn += G) {
        retract_joint(m, jn, rk.q(), rk.Dl(), rk.V(), rk.Yq(), rk.adz1());          // adz1[0..nv) = K(Theta_n+1, v_n+1)
        retract_pullback_joint(m, jn, rk.az1(), rk.lam(), rk.qb(), rk.dbar());       // dbar = Jr(Theta_n+1)^T lambda_q
      }
      gr.sync();
#pragma unroll 1
      for (int j = gr.lane; j < nq; j += G) Yqr[j] = (R)rk.Yq()[j];
#pragma unroll 1
      for (int j = gr.lane; j < nv; j += G) { Vr[j] = (R)rk.V()[j]; rk.amu()[j] = rk.dbar()[j]; rk.amu()[nv + j] = rk.lam()[nv + j]; }
      gr.sync();
      {
        int conv;
        int nr = field_eval<R, G, SH>(u, p, 0, &conv);
        if (nr < 0) { good = false; status = 3; break; }
#pragma unroll 1
        for (int j = gr.lane; j < nv; j += G) rk.adz1()[nv + j] = (double)ws.x()[j];
        gr.sync();
      }
      if (hprop < 0) hprop = h;
      double s = 0.0; bool have_k1 = false;
#pragma unroll 1
      while (s < h && good) {
        if (attempts >= sa.max_steps) { good = false; status = 1; break; }
        const double rem = h - s;
        bool hits; double hs;
        if (rep) {
          if (ir >= aa.n_replay || !(rep[ir] > 0.0)) { good = false; status = 1; break; }
          hs = rep[ir++]; hits = (hs == rem);
          if (hs > rem) { good = false; status = 3; break; }
        } else {
          hits = hprop * (1.0 + 1e-7) >= rem; hs = hits ? rem : hprop;
          if (!hits && hs < 1e-14 * fmax(1.0, h)) { good = false; status = 2; break; }
        }
        attempts++;
#pragma unroll 1
        for (int i = 0; i < 7 && good; ++i) {
          if (i == 0 && have_k1) continue;
          double ci = 0;
#pragma unroll 1
          for (int l = 0; l < i; ++l) ci += TAB_A[tab][i][l];
#pragma unroll 1
          for (int j = gr.lane; j < n2; j += G) {
            double acc = 0;
#pragma unroll 1
            for (int l = 0; l < i; ++l) acc += TAB_A[tab][i][l] * rk.ak()[l * n2 + j];
            rk.amus()[j] = rk.amu()[j] + hs * acc;
          }
          gr.sync();
          if (!adjoint_rhs<R, G, SH>(m, a, u, p, h, 1.0 - (s + ci * hs) / h, i, rk, ws, Yqr, Vr, gr, &n_unc, work)) { good = false; status = 3; }
        }
        if (!good) break;
        have_k1 = true;
#pragma unroll 1
        for (int j = gr.lane; j < n2; j += G) {
          double sb = 0, se = 0;
#pragma unroll 1
          for (int i = 0; i < 6; ++i) sb += TAB_A[tab][6][i] * rk.ak()[i * n2 + j];
#pragma unroll 1
          for (int i = 0; i < 7; ++i) se += TAB_E[tab][i] * rk.ak()[i * n2 + j];
          rk.amunew()[j] = rk.amu()[j] + hs * sb; rk.amus()[j] = hs * se;          // amus: error vector from here on
        }
        gr.sync();
        bool finite = true; double accn = 0.0;
#pragma unroll 1
        for (int j = 0; j < n2; ++j) {                   // every lane: index order, plain adds
          const double ej = rk.amus()[j], mn = rk.amunew()[j];
          if (!isfinite(ej) || !isfinite(mn)) finite = false;
          const double q = __ddiv_rn(ej, __dadd_rn(sa.atol, __dmul_rn(sa.rtol, fmax(fabs(rk.amu()[j]), fabs(mn)))));
          accn = __dadd_rn(accn, __dmul_rn(q, q));
        }
        double E = INFINITY; bool accept = false;
        if (rep) { if (!finite) { good = false; status = 3; break; } accept = true; E = 1.0; }
        else if (finite) { E = sqrt(accn / n2); accept = E <= 1.0; }
        const double Ec = fmax(E, 1e-30);
        double fac = finite ? sa.safety * exp(-(sa.pcoeff + sa.icoeff) / 5.0 * log(Ec)) * exp(sa.pcoeff / 5.0 * log(Eprev)) : sa.fac_min;
        fac = fmin(sa.fac_max, fmax(sa.fac_min, fac));
        if (!accept || !hits) hprop = hs * fac;
        gr.sync();
        if (!accept) { n_rej++; continue; }
        Eprev = Ec; n_acc++;
        if (a.dLdctrl && has_ctrl) for (int c = gr.lane; c < nu; c += G) {
          double t = 0;
#pragma unroll 1
          for (int i = 0; i < 6; ++i) t += TAB_A[tab][6][i] * rk.aub()[i * nu + c];
          a.dLdctrl[((size_t)e * nknot + knot) * nu + c] += (R)(hs * t);
        }
        if (a.want_p) for (int c = gr.lane; c < np; c += G) {
          double t = 0;
#pragma unroll 1
          for (int i = 0; i < 6; ++i) t += TAB_A[tab][6][i] * rk.apb()[i * np + c];
          rk.gp()[c] += hs * t;
        }
#pragma unroll 1
        for (int j = gr.lane; j < n2; j += G) { rk.amu()[j] = rk.amunew()[j]; rk.ak()[j] = rk.ak()[6 * n2 + j]; }     // FSAL inside the step
#pragma unroll 1
        for (int c = gr.lane; c < nu; c += G) rk.aub()[c] = rk.aub()[6 * nu + c];
        if (a.want_p) for (int c = gr.lane; c < np; c += G) rk.apb()[c] = rk.apb()[6 * np + c];
        gr.sync();
        s = hits ? h : s + hs;
      }
      if (!good) break;
#pragma unroll 1
      for (int j = gr.lane; j < n2; j += G) rk.lam()[j] = rk.amu()[j];        // Theta = 0 at t_n: chart = tangent coordinates
      gr.sync();
    }
    R* g0 = a.dLdx0 + (size_t)e * 2 * nv;
#pragma unroll 1
    for (int j = gr.lane; j < 2 * nv; j += G) g0[j] = good ? (R)rk.lam()[j] : R(0);
    if (a.dLdparams) for (int c = gr.lane; c < np; c += G) a.dLdparams[(size_t)e * np + c] = good ? (R)rk.gp()[c] : R(0);
    if (!good && a.dLdctrl && has_ctrl) for (int c = gr.lane; c < nknot * nu; c += G) a.dLdctrl[(size_t)e * nknot * nu + c] = R(0);
    if (gr.lane == 0) {
      if (a.n_unconv) a.n_unconv[e] = n_unc;
      if (a.work) { a.work[6 * (size_t)e + 3] = work[0]; a.work[6 * (size_t)e + 4] = work[1]; a.work[6 * (size_t)e + 5] = work[2]; }
      if (aa.info) { aa.info[3 * e] = n_acc; aa.info[3 * e + 1] = n_rej; aa.info[3 * e + 2] = good ? 0 : (status ? status : 3); }
    }
    gr.sync();
  }
  phase_drain();
}

template <class R, int G, class SH> cudaError_t launch_adjoint(const ModelDev<R>& m, const AdjointArgs<R>& a, LaunchCfg c, cudaStream_t s);

}  // namespace dmx
