// dmx_kernels.cuh — reverse sweep (S10-S12), the building-block kernels behind dmx_vector_field /
// dmx_vjp_field, the model-create kernel for the diagonal approximation A^
// and the host launchers, instantiated once per (real type, lanes per environment).
#pragma once
#include "dmx_rk.cuh"

namespace dmx {

// ---- S11/S12: (qbar,vbar,ubar,pbar) = kappa^T dF/d(q,v,u,p), F~ when cfd (Eq. 4) ----------
// Cooperative solve for x*, the active set and w = H^-1 kappa; then the closed-form gradient of S (dmx_field.cuh).
template <class R, int G, class SH>
DMX_DN bool vjp_stage(const ModelDev<R>& m, const Arr<R, StrideOf<G>::value>& Yqr, const Arr<R, StrideOf<G>::value>& Vr, const R* u, const R* p,
                      const Arr<double, StrideOf<G>::value>& kappa, bool cfd, bool want_p, const Ws<R, StrideOf<G>::value, SH>& ws,
                      const Rk<StrideOf<G>::value>& rk, const Grp<G>& gr, int dbg = 0, const double* xk = nullptr, int* unconv = nullptr,
                      unsigned long long* work = nullptr) {
  const int ST = StrideOf<G>::value;
  const int nv = m.nv;
  if (dbg & 4) return true;
  DMX_T0;
  InPlain<R, ST> in; in.qa = Yqr; in.va = Vr; in.aa = Vr; in.ua = u; in.pa = p;
  int conv;
  int nr = field_eval<R, G, SH>(u, p, cfd ? 1 : 0, &conv, xk);
  if (nr < 0) return false;
  if (unconv && !xk && nr > 0 && !(conv & 1)) ++*unconv;     // the implicit-function gradient is taken at a non-stationary point
  if (work) { work[0] += (unsigned)(conv >> 8); work[1] += (unsigned long long)(conv >> 8) * nr; work[2] += (unsigned)nr; }
  DMX_TICK(gr, 8);
  phase_sync(5);
#pragma unroll 1
  for (int j = gr.lane; j < nv; j += G) ws.kap()[j] = (R)kappa[j];
  gr.sync();
  if (!vjp_prepare<Ws<R, ST, SH>, G>(nv, nr, xk == nullptr && (conv & 1) != 0 && !(dbg & 8), ws, gr)) return false;
  DMX_TICK(gr, 9);
  phase_sync(6);
  // u: closed form; v: reverse sweep over the tree; then the frames at acceleration x* for the tangent passes
#pragma unroll 1
  for (int i = gr.lane; i < m.nu; i += G)
    rk.ubar()[i] = (double)(ws.kap()[m.jnt_vadr[m.act_jnt[i]]] * (m.act_type[i] == ACT_MOTOR ? m.act_gear[i] : m.act_kp[i]));
  if (!(dbg & 2)) vjp_velocity<Ws<R, ST, SH>, R, G, InPlain<R, ST> >(m, in, ws, nr, rk.vbar(), gr);
  DMX_TICK(gr, 10);
  phase_sync(7);
  in.aa = ws.x();
  kinematics<Ws<R, ST, SH>, R, G, InPlain<R, ST>, true>(m, in, ws, gr);
  DMX_TICK(gr, 11);
  phase_sync(8);
  // q: bodies in closed form (cooperative), then the rows' part and the parameters by one tangent lane per direction
  vjp_config_bodies<Ws<R, ST, SH>, R, G, InPlain<R, ST> >(m, in, ws, rk.qbar(), gr);
  vjp_config_rows<false, Ws<R, ST, SH>, R, G, InPlain<R, ST> >(m, in, ws, cfd, rk.qbar(), gr);                 // point-plane rows
  if (m.npp > 0) vjp_config_rows<true, Ws<R, ST, SH>, R, G, InPlain<R, ST> >(m, in, ws, cfd, rk.qbar(), gr);   // sphere-sphere rows
  if (want_p) vjp_params<Ws<R, ST, SH>, R, G, InPlain<R, ST> >(m, in, ws, cfd, rk.pbar(), gr);
  gr.sync();
  DMX_TICK(gr, 12);
  return true;
}

template <class R> struct BackwardArgs {
  int nenv, nknot, want_p, cfd, dbg, lockstep, tape_stages, n_light;   // n_light: see next_env (dmx_rk.cuh)
  const R *ctrl, *params, *zero_u, *xT, *dLdxT;
  const int* status;
  int* n_unconv;            // [nenv] or null: contact solves of the reverse sweep that did not converge
  unsigned long long* work; // [nenv][6] or null (slots 3..5: Newton iterations, row-iterations and rows of the reverse sweep)
  SolverOpts so;
  R *dLdx0, *dLdctrl, *dLdparams;
  TapeView<R> tp; PlanView pl;
  int* queue;
  double* rk_scratch;       // integrator / adjoint arrays of every resident group (global memory: touched once per stage)
  R* seg_scratch;           // checkpoint stride > 1: [resident groups][stride][seg_rec] segment buffers
  WsLayout wl; RkLayout rl;
};

// ---- S10: reverse sweep over the tape, frozen step sizes ---------------------------
// CKPT: the tape holds a checkpoint every a.tp.stride steps and the step schedule (TapeView); the sweep re-runs each
// segment forward from its checkpoint (same stages, same FSAL rule as rollout_kernel, step sizes from the schedule)
// into this group's buffer of `stride` full records, then sweeps the buffer exactly as it would sweep a full tape.
template <class R, int G, class SH, bool CKPT = false>
__global__ void __launch_bounds__(256) backward_kernel(const __grid_constant__ ModelDev<R> m_, const __grid_constant__ BackwardArgs<R> a) {
  unsigned char* smem = dyn_smem;
  CtaConst<R>& cc = cta_const<R>();
  if (threadIdx.x == 0) g_lockstep = a.lockstep;
  load_cta_const<R>(cc, m_, a.wl, a.wl, a.rl, 0);
  const ModelDev<R>& m = cc.m;
  const int ST = StrideOf<G>::value;
  const Grp<G> gr = make_group<G>();
  Rk<ST> rk; Ws<R, ST, SH> ws; Arr<R, ST> Yqr, Vr;
  bind_shared<R, G, SH>(smem, 0, a.wl.size + a.rl.rsize, a.wl.isize, rk, ws, Yqr, Vr, &cc.rl, &cc.wl);
  if (G == 1) rk.b = a.rk_scratch + ((size_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5)) * 32 * (size_t)a.rl.size_bwd + (threadIdx.x & 31);
  else rk.b = a.rk_scratch + ((size_t)blockIdx.x * (blockDim.x / G) + threadIdx.x / G) * (size_t)a.rl.size_bwd;
  const int nq = m.nq, nv = m.nv, nu = m.nu, np = m.np, nx = nq + nv, tab = a.so.tableau, rec = a.tp.rec;
  const bool has_ctrl = a.ctrl != nullptr && a.nknot > 0 && nu > 0;
  const int nknot = has_ctrl ? a.nknot : 0;
  // the tape must be the one a rollout of this model wrote for this batch, record layout and plan
  const bool tape_ok = a.tp.meta[0] == TAPE_MAGIC && a.tp.meta[1] == a.nenv && a.tp.meta[2] == rec && a.tp.meta[3] == a.tp.o_A &&
                       a.tp.meta[4] == (a.pl.offset ? 1 : 0) && a.tp.meta[5] == a.tp.stride && (CKPT == (a.tp.stride > 1));
  const int stride = CKPT ? a.tp.stride : 1, srec = CKPT ? a.tp.seg_rec : rec, o_A = CKPT ? a.tp.seg_oA : a.tp.o_A;
  R* segbuf = nullptr;
  if (CKPT) segbuf = a.seg_scratch + ((size_t)blockIdx.x * (G == 1 ? blockDim.x : blockDim.x / G) + (G == 1 ? threadIdx.x : threadIdx.x / G)) * (size_t)stride * srec;
  const bool restore = CKPT || a.tape_stages != 0;
  // One pass of the loop = one segment of one environment (the whole tape when !CKPT).  With CKPT and lockstep on, the
  // CTA alternates between two modes, all groups re-running their next segment, then all groups sweeping it, separated
  // by mode_sync: otherwise groups in the forward code and groups in the VJP code would meet at every phase barrier and
  // each interval would last as long as the longest phase of either (measured 3-4.6x on the whole sweep).
  int e = 0, N = 0, knot = 0, n = -1, n_unc = 0, tape_cap = 0;
  long long first = 0;
  bool good = false, active = false, fresh = false, first_env = true;
  const R* p = nullptr;
  unsigned long long work[3] = {0, 0, 0};
#pragma unroll 1
  for (;;) {
    if (!active) {
      if (gr.lane == 0) e = next_env<G>(a.queue, a.pl.order, a.nenv, a.n_light, first_env);
      e = gr.bcast_int(e);
      if (e >= a.nenv) break;
      p = a.params ? a.params + (size_t)e * np : m.p_default;
      N = a.tp.hdr[2 * e];
      knot = a.tp.hdr[2 * e + 1]; n_unc = 0;
      work[0] = work[1] = work[2] = 0;
      tape_slot(a.tp, a.pl, e, first, tape_cap);
      good = tape_ok && knot >= 0 && N <= tape_cap && (!a.status || a.status[e] == 0);
      n = N - 1; active = true; fresh = true;
    }
    if (good && fresh) {
      fresh = false;
      // ambient gradient at x_T -> tangent cotangent: lam = E(q_T)^T g
      const R* xT = a.xT + (size_t)e * nx; const R* gT = a.dLdxT + (size_t)e * nx;
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
#pragma unroll 1
      for (int i = gr.lane; i < np; i += G) rk.gp()[i] = 0.0;
      gr.sync();
    }
    const int s0 = (CKPT && n >= 0) ? (n / stride) * stride : 0;
    if (CKPT) {
      if (good && n >= 0) {                                       // re-run segment n / stride forward from its checkpoint
        const double* sch = a.tp.sched + first;
        int kj = knot;                                            // knot in effect after step n; minus the intervals ended inside
#pragma unroll 1
        for (int j = s0; j <= n; ++j) if (sch[j] < 0) --kj;
        const R* c = a.tp.data + ((size_t)(first / stride + e) + n / stride) * rec;
#pragma unroll 1
        for (int j = gr.lane; j < nq; j += G) rk.q()[j] = (double)c[j];
#pragma unroll 1
        for (int j = gr.lane; j < nv; j += G) rk.v()[j] = (double)c[nq + j];
        // the forward pass reused the previous step's last stage as A_1 here (FSAL) unless that step ended a control
        // interval (or this is the first step): take the taped A_1 in the first case, evaluate afresh in the second
        bool have_k1 = s0 > 0 && !(sch[s0 - 1] < 0);
        if (have_k1) for (int j = gr.lane; j < nv; j += G) rk.A()[j] = (double)c[a.tp.o_A + j];
        gr.sync();
#pragma unroll 1
        for (int j = s0; j <= n && good; ++j) {
          const double hsj = sch[j];
          const R* uj = has_ctrl ? a.ctrl + ((size_t)e * nknot + kj) * nu : a.zero_u;
          bool okf; int uncf;
          rk_attempt<R, G, SH, false>(m, tab, rk, Yqr, Vr, uj, p, fabs(hsj), have_k1, ws, okf, uncf, gr);
          if (!okf) { good = false; break; }                      // cannot happen on a tape this model wrote
          R* w = segbuf + (size_t)(j - s0) * srec;
          const int nchunk = srec * (int)sizeof(R) / 16;
#pragma unroll 1
          for (int ch = gr.lane; ch < nchunk; ch += G) tape_store_chunk(w, ch, rk, nq, nx, a.tp.o_th, o_A, 6 * nv, 0.0, hsj);
          gr.sync();
#pragma unroll 1
          for (int i = gr.lane; i < nq; i += G) rk.q()[i] = rk.Yq()[i];
#pragma unroll 1
          for (int i = gr.lane; i < nv; i += G) rk.v()[i] = rk.V()[i];
          if (hsj < 0) { ++kj; have_k1 = false; }                 // the step ended a control interval: the FSAL stage is stale
          else { have_k1 = true; for (int i = gr.lane; i < nv; i += G) rk.A()[i] = rk.A()[6 * nv + i]; }
          gr.sync();
        }
      }
      mode_sync(false);
    }
#pragma unroll 1
    for (; n >= s0 && good; --n) {
      const R* r = CKPT ? segbuf + (size_t)(n % stride) * srec : a.tp.data + ((size_t)first + n) * rec;
#pragma unroll 1
      for (int j = gr.lane; j < nq; j += G) rk.q()[j] = (double)r[j];
#pragma unroll 1
      for (int j = gr.lane; j < nv; j += G) rk.v()[j] = (double)r[nq + j];
      double tn, hs; tape_load_th(r, a.tp.o_th, tn, hs);      // t_n, h_n are fp64 on the tape in both precisions (G14)
      const double h = fabs(hs);
      if (hs < 0) knot--;
      const R* u = has_ctrl ? a.ctrl + ((size_t)e * nknot + knot) * nu : a.zero_u;
      if (restore) for (int j = gr.lane; j < 6 * nv; j += G) rk.A()[j] = (double)r[o_A + j];
      gr.sync();
      bool ok; int unc;
      // stage states: recomputed with F from the checkpoint, or rebuilt from the taped stage rates
      rk_attempt<R, G, SH, true>(m, tab, rk, Yqr, Vr, u, p, h, false, ws, ok, unc, gr, restore, work);
      // y_{n+1} = (q_n (+) h sum b_i K_i, v_n + h sum b_i A_i), b = row 6 of a
#pragma unroll 1
      for (int j = gr.lane; j < nv; j += G) {
        double s = 0; for (int i = 0; i < 6; ++i) s += TAB_A[tab][6][i] * rk.K()[i * nv + j];
        rk.delta()[j] = h * s; rk.dbar()[j] = 0; rk.qb()[j] = 0; rk.vb()[j] = rk.lam()[nv + j];
      }
      gr.sync();
#pragma unroll 1
      for (int jn = gr.lane; jn < m.njnt; jn += G) retract_pullback_joint(m, jn, rk.delta(), rk.lam(), rk.qb(), rk.dbar());
      gr.sync();
#pragma unroll 1
      for (int j = gr.lane; j < nv; j += G)
#pragma unroll 1
        for (int i = 0; i < 6; ++i) { rk.Kb()[i * nv + j] = h * TAB_A[tab][6][i] * rk.dbar()[j]; rk.Ab()[i * nv + j] = h * TAB_A[tab][6][i] * rk.lam()[nv + j]; }
      gr.sync();
#pragma unroll 1
      for (int i = 5; i >= 0 && good; --i) {
#pragma unroll 1
        for (int j = gr.lane; j < nv; j += G) { rk.Vb()[j] = 0; rk.dbar()[j] = 0; }
        gr.sync();
#pragma unroll 1
        for (int jn = gr.lane; jn < m.njnt; jn += G) chart_pullback_joint(m, jn, rk.sDl().at(i * nv), rk.sV().at(i * nv), rk.Kb().at(i * nv), rk.Vb(), rk.dbar());
#pragma unroll 1
        for (int j = gr.lane; j < nq; j += G) Yqr[j] = (R)rk.sYq()[i * nq + j];
#pragma unroll 1
        for (int j = gr.lane; j < nv; j += G) Vr[j] = (R)rk.sV()[i * nv + j];
        gr.sync();
        // A_i = F(Y_i), or F~ for the straight-through estimator (Eq. 4)
        if (!vjp_stage<R, G, SH>(m, Yqr, Vr, u, p, rk.Ab().at(i * nv), a.cfd != 0, a.want_p != 0, ws, rk, gr, a.dbg,
                              (restore && !a.cfd) ? rk.A().at(i * nv).p : nullptr, &n_unc, work)) { good = false; break; }   // F: x* = taped A_i
#pragma unroll 1
        for (int j = gr.lane; j < nv; j += G) rk.Vb()[j] += rk.vbar()[j];
        if (a.dLdctrl && has_ctrl) for (int c = gr.lane; c < nu; c += G) a.dLdctrl[((size_t)e * nknot + knot) * nu + c] += (R)rk.ubar()[c];
        if (a.want_p) for (int c = gr.lane; c < np; c += G) rk.gp()[c] += rk.pbar()[c];
        gr.sync();
#pragma unroll 1
        for (int jn = gr.lane; jn < m.njnt; jn += G) retract_pullback_joint(m, jn, rk.sDl().at(i * nv), rk.qbar(), rk.qb(), rk.dbar());
        gr.sync();
#pragma unroll 1
        for (int j = gr.lane; j < nv; j += G) {
          rk.vb()[j] += rk.Vb()[j];
#pragma unroll 1
          for (int l = 0; l < i; ++l) { rk.Kb()[l * nv + j] += h * TAB_A[tab][i][l] * rk.dbar()[j]; rk.Ab()[l * nv + j] += h * TAB_A[tab][i][l] * rk.Vb()[j]; }
        }
        gr.sync();
      }
#pragma unroll 1
      for (int j = gr.lane; j < nv; j += G) { rk.lam()[j] = rk.qb()[j]; rk.lam()[nv + j] = rk.vb()[j]; }
      gr.sync();
    }
    if (n < 0 || !good) {                                         // the environment is finished
      R* g0 = a.dLdx0 + (size_t)e * 2 * nv;
#pragma unroll 1
      for (int j = gr.lane; j < 2 * nv; j += G) g0[j] = good ? (R)rk.lam()[j] : R(0);
      if (a.dLdparams) for (int c = gr.lane; c < np; c += G) a.dLdparams[(size_t)e * np + c] = good ? (R)rk.gp()[c] : R(0);
      if (!good && a.dLdctrl && has_ctrl) for (int c = gr.lane; c < nknot * nu; c += G) a.dLdctrl[(size_t)e * nknot * nu + c] = R(0);
      if (a.n_unconv && gr.lane == 0) a.n_unconv[e] = n_unc;
      if (a.work && gr.lane == 0) { a.work[6 * (size_t)e + 3] = work[0]; a.work[6 * (size_t)e + 4] = work[1]; a.work[6 * (size_t)e + 5] = work[2]; }
      gr.sync();
      active = false;
    }
    if (CKPT) mode_sync(false);
  }
  if (CKPT) { while (!mode_sync(true)) {} return; }
  phase_drain();
}

// ---- building blocks for parity tests: one lane group per state --------------------------------------
template <class R> struct FieldArgs {
  int n, cfd, want_p;
  const R *x, *u, *params, *zero_u, *kappa;
  R *acc, *qbar, *vbar, *ubar, *pbar; int* nrow;
  WsLayout wl; RkLayout rl;
};
template <class R, int G, class SH>
__global__ void __launch_bounds__(128) field_kernel(const __grid_constant__ ModelDev<R> m_, const __grid_constant__ FieldArgs<R> a) {
  unsigned char* smem = dyn_smem;
  CtaConst<R>& cc = cta_const<R>();
  if (threadIdx.x == 0) g_lockstep = 0;
  load_cta_const<R>(cc, m_, a.wl, a.wl, a.rl, a.rl.size_bwd);
  const ModelDev<R>& m = cc.m;
  const int ST = StrideOf<G>::value;
  const Grp<G> gr = make_group<G>();
  Rk<ST> rk; Ws<R, ST, SH> ws; Arr<R, ST> Yqr, Vr;
  bind_shared<R, G, SH>(smem, a.rl.size_bwd, a.wl.size + a.rl.rsize, a.wl.isize, rk, ws, Yqr, Vr, &cc.rl, &cc.wl);
  const int nq = m.nq, nv = m.nv, nx = nq + nv;
  const int ngr = (gridDim.x * blockDim.x) / G;
#pragma unroll 1
  for (int e = (blockIdx.x * blockDim.x + threadIdx.x) / G; e < a.n; e += ngr) {
    const R* x = a.x + (size_t)e * nx;
    const R* u = (a.u && m.nu > 0) ? a.u + (size_t)e * m.nu : a.zero_u;
    const R* p = a.params ? a.params + (size_t)e * m.np : m.p_default;
#pragma unroll 1
    for (int j = gr.lane; j < nq; j += G) Yqr[j] = x[j];
#pragma unroll 1
    for (int j = gr.lane; j < nv; j += G) Vr[j] = x[nq + j];
    gr.sync();
    if (!a.kappa) {
      int conv;
      int nr = field_eval<R, G, SH>(u, p, a.cfd, &conv);
#pragma unroll 1
      for (int j = gr.lane; j < nv; j += G) a.acc[(size_t)e * nv + j] = nr < 0 ? R(nan("")) : ws.x()[j];
      if (gr.lane == 0 && a.nrow) a.nrow[e] = nr;
    } else {
#pragma unroll 1
      for (int j = gr.lane; j < nv; j += G) rk.lam()[j] = (double)a.kappa[(size_t)e * nv + j];
      gr.sync();
      bool ok = vjp_stage<R, G, SH>(m, Yqr, Vr, u, p, rk.lam(), a.cfd != 0, a.want_p != 0, ws, rk, gr);
      R bad = R(nan(""));
#pragma unroll 1
      for (int j = gr.lane; j < nv; j += G) { a.qbar[(size_t)e * nv + j] = ok ? (R)rk.qbar()[j] : bad; a.vbar[(size_t)e * nv + j] = ok ? (R)rk.vbar()[j] : bad; }
#pragma unroll 1
      for (int j = gr.lane; j < m.nu; j += G) a.ubar[(size_t)e * m.nu + j] = ok ? (R)rk.ubar()[j] : bad;
      if (a.want_p) for (int j = gr.lane; j < m.np; j += G) a.pbar[(size_t)e * m.np + j] = ok ? (R)rk.pbar()[j] : bad;
    }
    gr.sync();
  }
}

// ---- A^: w(b) = mean diagonal of the translational block of Jc_b M(qpos0)^-1 Jc_b^T -------
template <class R, int G, class SH>
__global__ void __launch_bounds__(128) invweight_kernel(const __grid_constant__ ModelDev<R> m_, const R* qpos0, const R* zero_v, R* body_w,
                                                        const __grid_constant__ WsLayout wl, const __grid_constant__ RkLayout rl) {
  unsigned char* smem = dyn_smem;
  CtaConst<R>& cc = cta_const<R>();
  if (threadIdx.x == 0) g_lockstep = 0;
  load_cta_const<R>(cc, m_, wl, wl, rl, rl.size_bwd);
  const ModelDev<R>& m = cc.m;
  const int ST = StrideOf<G>::value;
  const Grp<G> gr = make_group<G>();
  Rk<ST> rk; Ws<R, ST, SH> ws; Arr<R, ST> Yqr, Vr;
  bind_shared<R, G, SH>(smem, rl.size_bwd, wl.size + rl.rsize, wl.isize, rk, ws, Yqr, Vr, &cc.rl, &cc.wl);
  if (blockIdx.x != 0 || threadIdx.x >= G) return;
  const int nv = m.nv;
#pragma unroll 1
  for (int j = gr.lane; j < m.nq; j += G) Yqr[j] = qpos0[j];
#pragma unroll 1
  for (int j = gr.lane; j < nv; j += G) Vr[j] = R(0);
  gr.sync();
  InPlain<R, ST> in; in.qa = Yqr; in.va = Vr; in.aa = Vr; in.ua = zero_v; in.pa = m.p_default;
  kinematics<Ws<R, ST, SH>, R, G, InPlain<R, ST>, false>(m, in, ws, gr);
  dynamics<Ws<R, ST, SH>, R, G, InPlain<R, ST> >(m, in, ws, gr);
  const int ld = ws.L->ld;
#pragma unroll 1
  for (int e = gr.lane; e < nv * ld; e += G) ws.Hc()[e] = ws.M()[e];
  gr.sync();
  bool pd = cholesky(ws.Hc(), nv, ld, gr);
#pragma unroll 1
  for (int b = 0; b < m.nbody; ++b) {
    R tr = R(0);
#pragma unroll 1
    for (int c = 0; c < 3 && pd && b > 0; ++c) {
#pragma unroll 1
      for (int j = gr.lane; j < nv; j += G) {
        int e = m.tw_idx[b * nv + j];
        R val_ = R(0);
        if (e >= 0) { V3<R> l = ld3(ws.tw(), e); val_ = c == 0 ? l.x : (c == 1 ? l.y : l.z); }
        ws.g()[j] = val_; ws.dl()[j] = val_;
      }
      gr.sync();
      chol_solve(ws.Hc(), nv, ld, ws.dl(), gr);
#pragma unroll 1
      for (int j = 0; j < nv; ++j) tr += ws.g()[j] * ws.dl()[j];
      gr.sync();
    }
    if (gr.lane == 0) body_w[b] = pd ? tr / R(3) : R(nan(""));
  }
}

template <class R, int G, class SH> __global__ void prof_dump_kernel(unsigned long long* out) {
  if (threadIdx.x < 32) { out[threadIdx.x] = g_prof[threadIdx.x]; g_prof[threadIdx.x] = 0; }
}

// ---- host launchers (defined per instantiation in dmx_inst.cuh) -----------------------------------------
struct LaunchCfg { int block, grid; size_t smem; };

template <class R, int G, class SH> cudaError_t launch_rollout(const ModelDev<R>& m, const RolloutArgs<R>& a, LaunchCfg c, cudaStream_t s);
template <class R, int G, class SH> cudaError_t launch_backward(const ModelDev<R>& m, const BackwardArgs<R>& a, LaunchCfg c, cudaStream_t s);
template <class R, int G, class SH> cudaError_t launch_backward_ckpt(const ModelDev<R>& m, const BackwardArgs<R>& a, LaunchCfg c, cudaStream_t s);
template <class R, int G, class SH> cudaError_t launch_field(const ModelDev<R>& m, const FieldArgs<R>& a, LaunchCfg c, cudaStream_t s);
template <class R, int G, class SH> cudaError_t launch_invweight(const ModelDev<R>& m, const R* qpos0, const R* zero_v, R* body_w, const WsLayout& wl,
                                                                 const RkLayout& rl, LaunchCfg c, cudaStream_t s);
template <class R, int G, class SH> cudaError_t launch_prof_dump(unsigned long long* out, cudaStream_t s);
template <class R, int G, class SH> cudaError_t kernel_occupancy(int block, size_t smem_fwd, size_t smem_bwd, size_t smem_field, int* occ_fwd, int* occ_bwd, int* occ_field);

}  // namespace dmx
