// dmx_rk.cuh — embedded Runge-Kutta pair on the configuration manifold, PI step-size control and
// the discrete adjoint through the accepted steps (PAPER.md:88 adaptive integration; :429 exact
// quaternion integration; :347 Tsit5/Dopri5 and the PID controller; :431, 456
// discretize-then-optimize).  Time, step size, the stage combinations, the error norm and the
// controller are always fp64; the vector field runs in the model's real type R.
#pragma once
#include "dmx_field.cuh"

namespace dmx {

// ---- Butcher tableaus: index 0 Dopri5 (Dormand & Prince 1980), 1 Tsit5 (Tsitouras 2011)
static __constant__ double TAB_A[2][7][7] = {
    {{0},
     {1.0 / 5},
     {3.0 / 40, 9.0 / 40},
     {44.0 / 45, -56.0 / 15, 32.0 / 9},
     {19372.0 / 6561, -25360.0 / 2187, 64448.0 / 6561, -212.0 / 729},
     {9017.0 / 3168, -355.0 / 33, 46732.0 / 5247, 49.0 / 176, -5103.0 / 18656},
     {35.0 / 384, 0, 500.0 / 1113, 125.0 / 192, -2187.0 / 6784, 11.0 / 84}},
    {{0},
     {0.161},
     {-0.008480655492356989, 0.335480655492357},
     {2.8971530571054935, -6.359448489975075, 4.3622954328695815},
     {5.325864828439257, -11.748883564062828, 7.4955393428898365, -0.09249506636175525},
     {5.86145544294642, -12.92096931784711, 8.159367898576159, -0.071584973281401, -0.028269050394068383},
     {0.09646076681806523, 0.01, 0.4798896504144996, 1.379008574103742, -3.290069515436081, 2.324710524099774}}};
// e = b - bhat; b is row 6 of a (FSAL)
static __constant__ double TAB_E[2][7] = {
    {35.0 / 384 - 5179.0 / 57600, 0.0, 500.0 / 1113 - 7571.0 / 16695, 125.0 / 192 - 393.0 / 640,
     -2187.0 / 6784 - (-92097.0 / 339200), 11.0 / 84 - 187.0 / 2100, 0.0 - 1.0 / 40},
    {-0.00178001105222577714, -0.0008164344596567469, 0.007880878010261995, -0.1447110071732629,
     0.5823571654525552, -0.45808210592918697, 0.015151515151515152}};

struct SolverOpts { int tableau; double rtol, atol, h0, pcoeff, icoeff, safety, fac_min, fac_max; int max_steps; };

// ---- the retraction q (+) delta, the chart rate and their pullbacks (reading G10) ------
DMX_DI void rotvec_to_quat(const double* d, double* e) {
  double th2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2], th = sqrt(th2);
  double s, c; sincos(0.5 * th, &s, &c);
  double k = th < 1e-4 ? 0.5 - th2 / 48.0 : s / th;
  e[0] = c; e[1] = k * d[0]; e[2] = k * d[1]; e[3] = k * d[2];
}
DMX_DI void cross3(const double* a, const double* b, double* r) {
  r[0] = a[1] * b[2] - a[2] * b[1]; r[1] = a[2] * b[0] - a[0] * b[2]; r[2] = a[0] * b[1] - a[1] * b[0];
}
// joint jn of: qout = q (+) delta and K = chart_rate(delta, V)
template <class R, class AD>
DMX_DI void retract_joint(const ModelDev<R>& m, int jn, const AD& q, const AD& delta, const AD& V, const AD& qout, const AD& K) {
  int qa = m.jnt_qadr[jn], va = m.jnt_vadr[jn];
  if (m.jnt_type[jn] != JNT_FREE) { qout[qa] = q[qa] + delta[va]; K[va] = V[va]; return; }
  double d[3], w[3], e[4], a[4], r[4], ql[3], dl[3], vl[3];     // reads first, writes last (see retract_pullback_joint)
#pragma unroll
  for (int c = 0; c < 3; ++c) { ql[c] = q[qa + c]; dl[c] = delta[va + c]; vl[c] = V[va + c]; d[c] = delta[va + 3 + c]; w[c] = V[va + 3 + c]; }
#pragma unroll
  for (int c = 0; c < 4; ++c) a[c] = q[qa + 3 + c];
#pragma unroll
  for (int c = 0; c < 3; ++c) { qout[qa + c] = ql[c] + dl[c]; K[va + c] = vl[c]; }
  rotvec_to_quat(d, e);
  r[0] = a[0] * e[0] - a[1] * e[1] - a[2] * e[2] - a[3] * e[3];
  r[1] = a[0] * e[1] + a[1] * e[0] + a[2] * e[3] - a[3] * e[2];
  r[2] = a[0] * e[2] - a[1] * e[3] + a[2] * e[0] + a[3] * e[1];
  r[3] = a[0] * e[3] + a[1] * e[2] - a[2] * e[1] + a[3] * e[0];
  double n = sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2] + r[3] * r[3]);
#pragma unroll 1
  for (int c = 0; c < 4; ++c) qout[qa + 3 + c] = r[c] / n;
  // Theta' = dexp^-1_Theta(w) truncated after the B_2 term: w + 1/2 Theta x w + 1/12 Theta x (Theta x w)
  double t1[3], t2[3]; cross3(d, w, t1); cross3(d, t1, t2);
#pragma unroll 1
  for (int c = 0; c < 3; ++c) K[va + 3 + c] = w[c] + 0.5 * t1[c] + t2[c] / 12.0;
}
DMX_DI void rot_AB(const double* d, double& A, double& B, double& C) {
  double th2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2], th = sqrt(th2);
  double s, c; sincos(th, &s, &c);
  bool sm = th < 1e-4;
  A = sm ? 1.0 - th2 / 6.0 : s / th;
  B = sm ? 0.5 - th2 / 24.0 : (1.0 - c) / th2;
  C = sm ? 1.0 / 6.0 - th2 / 120.0 : (th - s) / (th2 * th);
}
// joint jn of: base += T^T Qbar (T = blockdiag(I, R(exp delta)^T)), dbar += Jr(delta)^T Qbar
template <class R, class AD>
DMX_DI void retract_pullback_joint(const ModelDev<R>& m, int jn, const AD& delta, const AD& Qbar, const AD& base, const AD& dbar) {
  int va = m.jnt_vadr[jn];
  if (m.jnt_type[jn] != JNT_FREE) { base[va] += Qbar[va]; dbar[va] += Qbar[va]; return; }
  // all operands are read before anything is written: in the reverse sweep they live in global memory, and loads issued
  // back to back overlap their latencies (one round trip instead of one per component)
  double d[3], qb[3], ql[3], bs[6], db[6];
#pragma unroll
  for (int c = 0; c < 3; ++c) { ql[c] = Qbar[va + c]; qb[c] = Qbar[va + 3 + c]; d[c] = delta[va + 3 + c]; }
#pragma unroll
  for (int c = 0; c < 6; ++c) { bs[c] = base[va + c]; db[c] = dbar[va + c]; }
  double A, B, C; rot_AB(d, A, B, C);
  // R qb = qb + A d x qb + B d x (d x qb);  Jr^T qb = qb + B d x qb + C d x (d x qb)   (K^T = -K)
  double k1[3], k2[3]; cross3(d, qb, k1); cross3(d, k1, k2);
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    base[va + c] = bs[c] + ql[c]; dbar[va + c] = db[c] + ql[c];
    base[va + 3 + c] = bs[3 + c] + (qb[c] + A * k1[c] + B * k2[c]); dbar[va + 3 + c] = db[3 + c] + (qb[c] + B * k1[c] + C * k2[c]);
  }
}
// joint jn of: Vbar += (dK/dV)^T Kbar, dbar += (dK/dTheta)^T Kbar
template <class R, class AD>
DMX_DI void chart_pullback_joint(const ModelDev<R>& m, int jn, const AD& delta, const AD& V, const AD& Kbar, const AD& Vbar, const AD& dbar) {
  int va = m.jnt_vadr[jn];
  if (m.jnt_type[jn] != JNT_FREE) { Vbar[va] += Kbar[va]; return; }
  double th[3], w[3], kb[3], kl[3], vb[6], db[3];            // reads first, writes last (see retract_pullback_joint)
#pragma unroll
  for (int c = 0; c < 3; ++c) { kl[c] = Kbar[va + c]; kb[c] = Kbar[va + 3 + c]; th[c] = delta[va + 3 + c]; w[c] = V[va + 3 + c]; db[c] = dbar[va + 3 + c]; }
#pragma unroll
  for (int c = 0; c < 6; ++c) vb[c] = Vbar[va + c];
  double t1[3], t2[3], tw[3], a[3], b[3], c3v[3];
  cross3(th, kb, t1); cross3(th, t1, t2);
  cross3(w, kb, a); cross3(th, w, tw); cross3(tw, kb, b); cross3(w, t1, c3v);
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    Vbar[va + c] = vb[c] + kl[c];
    Vbar[va + 3 + c] = vb[3 + c] + (kb[c] - 0.5 * t1[c] + t2[c] / 12.0);
    dbar[va + 3 + c] = db[c] + (0.5 * a[c] + b[c] / 12.0 - c3v[c] / 12.0);
  }
}

// ---- per-environment fp64 integrator state in the group's workspace ---------------------------------
struct RkLayout {
  int q, v, Yq, V, Dl, K, A, err;            // forward (Yq, V, Dl: one stage; K, A: 7 stages)
  int sYq, sV, sDl;                          // backward: 6 stages each
  int Kb, Ab, qb, vb, dbar, Vb, lam, delta, qbar, vbar, ubar, pbar, gp;
  int size_fwd, size_bwd;
  int Yqr, Vr, rsize;                        // stage inputs in the real type R
  // continuous adjoint (adjoint_kernel): stage rates of the backward solve k[7][2nv], their control / parameter parts,
  // the adjoint in chart coordinates (current, stage, proposal) and the Hermite end data of the forward step
  int ak, aub, apb, amu, amus, amunew, az1, adz1, size_adj;
};
#define DMX_RK_ARR(name) DMX_DI Arr<double, ST> name() const { return Arr<double, ST>(b + L->name * ST); }
template <int ST_> struct Rk {
  static const int ST = ST_;
  double* b; const RkLayout* L;
  DMX_RK_ARR(q) DMX_RK_ARR(v) DMX_RK_ARR(Yq) DMX_RK_ARR(V) DMX_RK_ARR(Dl) DMX_RK_ARR(K) DMX_RK_ARR(A) DMX_RK_ARR(err)
  DMX_RK_ARR(sYq) DMX_RK_ARR(sV) DMX_RK_ARR(sDl) DMX_RK_ARR(Kb) DMX_RK_ARR(Ab) DMX_RK_ARR(qb) DMX_RK_ARR(vb) DMX_RK_ARR(dbar)
  DMX_RK_ARR(Vb) DMX_RK_ARR(lam) DMX_RK_ARR(delta) DMX_RK_ARR(qbar) DMX_RK_ARR(vbar) DMX_RK_ARR(ubar) DMX_RK_ARR(pbar) DMX_RK_ARR(gp)
  DMX_RK_ARR(ak) DMX_RK_ARR(aub) DMX_RK_ARR(apb) DMX_RK_ARR(amu) DMX_RK_ARR(amus) DMX_RK_ARR(amunew) DMX_RK_ARR(az1) DMX_RK_ARR(adz1)
};
// stride of the cooperative workspaces: contiguous per group, warp-interleaved for one-lane groups
template <int G> struct StrideOf { static const int value = (G == 1) ? 32 : 1; };

template <class R, int G, class SH> __device__ __noinline__ int field_eval(const R* u, const R* p, int cfd, int* conv_out, const double* xk = nullptr);

// ---- S7: one attempted step: stages 1..7 (stage 1 reused when have_k1), proposal, error vector -----
// KEEP: also store every stage's (Yq, V, Dl) for the reverse sweep.
template <class R, int G, class SH, bool KEEP>
DMX_DN void rk_attempt(const ModelDev<R>& m, int tab, const Rk<StrideOf<G>::value>& rk, const Arr<R, StrideOf<G>::value>& Yqr,
                       const Arr<R, StrideOf<G>::value>& Vr, const R* u, const R* p, double h, bool have_k1,
                       const Ws<R, StrideOf<G>::value, SH>& ws, bool& ok, int& unconverged, const Grp<G>& gr, bool restore = false,
                       unsigned long long* work = nullptr) {
  const int ST = StrideOf<G>::value;
  const int nv = m.nv, nq = m.nq;
  ok = true; unconverged = 0;
  const int ns = KEEP ? 6 : 7;     // the reverse sweep needs stages 1..6 only
#pragma unroll 1
  for (int i = 0; i < ns; ++i) {
#pragma unroll 1
    for (int j = gr.lane; j < nv; j += G) {
      double sq = 0, sv = 0;
#pragma unroll 1
      for (int l = 0; l < i; ++l) { sq += TAB_A[tab][i][l] * rk.K()[l * nv + j]; sv += TAB_A[tab][i][l] * rk.A()[l * nv + j]; }
      rk.Dl()[j] = h * sq; rk.V()[j] = rk.v()[j] + h * sv;
    }
    gr.sync();
#pragma unroll 1
    for (int jn = gr.lane; jn < m.njnt; jn += G) retract_joint(m, jn, rk.q(), rk.Dl(), rk.V(), rk.Yq(), rk.K().at(i * nv));
    gr.sync();
#pragma unroll 1
    for (int j = gr.lane; j < nq; j += G) { Yqr[j] = (R)rk.Yq()[j]; if (KEEP && i < 6) rk.sYq()[i * nq + j] = rk.Yq()[j]; }
#pragma unroll 1
    for (int j = gr.lane; j < nv; j += G) {
      Vr[j] = (R)rk.V()[j];
      if (KEEP && i < 6) { rk.sV()[i * nv + j] = rk.V()[j]; rk.sDl()[i * nv + j] = rk.Dl()[j]; }
    }
    gr.sync();
    if (restore) continue;       // stage rates A_i come from the tape: stage states only
    if (i == 0 && have_k1) { for (int k = 0; k < 5; ++k) phase_sync(k); continue; }   // keep the CTA's phases aligned
    int conv;
    int nr = field_eval<R, G, SH>(u, p, 0, &conv);
    if (nr < 0) { ok = false; for (int j = gr.lane; j < nv; j += G) rk.A()[i * nv + j] = nan(""); }
    else {
      for (int j = gr.lane; j < nv; j += G) rk.A()[i * nv + j] = (double)ws.x()[j];
      if (nr > 0 && !(conv & 1)) unconverged++;
      if (work) { work[0] += (unsigned)(conv >> 8); work[1] += (unsigned long long)(conv >> 8) * nr; work[2] += (unsigned)nr; }
    }
    gr.sync();
  }
  if (!KEEP) {
    // row 6 of a is b: stage 7 is the proposal y_{n+1} = (Yq, V) and k7 = (V, A[6]) (FSAL)
#pragma unroll 1
    for (int j = gr.lane; j < nv; j += G) {
      double eq = 0, ev = 0;
#pragma unroll 1
      for (int i = 0; i < 7; ++i) { eq += TAB_E[tab][i] * rk.K()[i * nv + j]; ev += TAB_E[tab][i] * rk.A()[i * nv + j]; }
      rk.err()[j] = h * eq; rk.err()[nv + j] = h * ev;
    }
    gr.sync();
  }
}

// ---- S8: scaled RMS error in index order with plain adds; every lane computes it -------
template <class R, int ST>
DMX_DN double error_norm(const ModelDev<R>& m, const Rk<ST>& rk, double rtol, double atol, bool& finite) {
  const int nv = m.nv;
  double acc = 0.0;
#pragma unroll 1
  for (int d = 0; d < nv; ++d) {
    int j = m.dof_jnt[d], c = d - m.jnt_vadr[j];
    double mag = 1.0;
    if (m.jnt_type[j] != JNT_FREE || c < 3) { int qi = m.jnt_qadr[j] + c; mag = fmax(fabs(rk.q()[qi]), fabs(rk.Yq()[qi])); }
    double e = rk.err()[d];
    if (!isfinite(e)) finite = false;
    double r = __ddiv_rn(e, __dadd_rn(atol, __dmul_rn(rtol, mag)));
    acc = __dadd_rn(acc, __dmul_rn(r, r));
  }
#pragma unroll 1
  for (int d = 0; d < nv; ++d) {
    double e = rk.err()[nv + d];
    if (!isfinite(e)) finite = false;
    double r = __ddiv_rn(e, __dadd_rn(atol, __dmul_rn(rtol, fmax(fabs(rk.v()[d]), fabs(rk.V()[d])))));
    acc = __dadd_rn(acc, __dmul_rn(r, r));
  }
  return sqrt(acc / (2 * nv));
}

// ---- kernel arguments ------------------------------------------------------------------------------
// ---- S9: the tape in HBM ------------------------------------------------------
// [meta 256 B | (n_acc, final knot)[nenv] | records].  A record is `rec` reals, a multiple of 16 bytes, written with
// 16-byte stores: [q(nq) v(nv) | pad | t_n, h_n as two DOUBLES | A_1..A_6 (6 nv, when the stage rates are taped) | pad].
// Environment e owns records [offset(e), offset(e) + cap(e)): uniform (e * cap) or, with a plan (dmx_tape_plan), the
// prefix sum of per-environment capacities sized from a previous pass, so that one long environment does not size
// every slot ("memory = number of checkpoints x state size").
// Checkpoint stride k > 1 (dmx_model_set_checkpoint_stride; PAPER.md:371-375 "number of checkpoints", :431): a full
// record is kept only for the accepted steps n = 0, k, 2k, ... (record ckpt(e, n/k): y_n, t_n, h_n and the first-stage rate
// A_1, which is the FSAL value the forward pass used there unless the previous step ended a control interval) and every step
// keeps its signed step size in the schedule sched[first + n] (8 bytes); the reverse sweep re-runs a segment forward from
// its checkpoint into a per-group buffer of k full records and then sweeps it.  Checkpoint records of environment e start
// at record floor(first / k) + e, which leaves every environment ceil(cap / k) records.
enum { TAPE_MAGIC = 0x646d7832, TAPE_META_INTS = 64 };
template <class R> struct TapeView {
  int rec, o_th, o_A;          // reals per record; offsets of (t, h) and of the stage rates (o_A < 0: not taped)
  int uniform_cap;             // records per environment without a plan
  int stride;                  // 1: a record per accepted step; k > 1: a checkpoint every k steps + the schedule
  int seg_rec, seg_oA;         // stride > 1: geometry of the records (with stage rates) of the sweep's segment buffer
  double* sched;               // stride > 1: [capacity] signed step sizes
  long long capacity;          // accepted steps the buffer holds
  int* meta;                   // [TAPE_META_INTS]: magic, nenv, rec, o_A, planned, stride
  int* hdr;                    // [nenv*2]: accepted steps on tape, final knot (-1-knot: failed)
  R* data;
};
// Plan of a launch (dmx_tape_plan): hand-out order of the work queue (longest environment first, so that the launch
// does not end on a lone long chain) and per-environment tape slots.  All null: identity / uniform.
struct PlanView { const int* order; const int* cap; const long long* offset; };

template <class R> struct RolloutArgs {
  int nenv, nknot, n_replay, want_tape, lockstep, n_light;   // n_light: see next_env
  const R *x0, *ctrl, *params, *zero_u;
  const double* h_replay;
  double knot_dt, horizon;
  SolverOpts so;
  R* xT;
  int *n_accept, *n_reject, *n_feval, *n_unconv, *status;
  double *h_min, *h_max, *t_end;
  unsigned long long* work;     // [nenv][6] or null: Newton iterations, row-iterations and rows, forward [0..2] / reverse sweep [3..5]
  TapeView<R> tp; PlanView pl;
  int* queue;
  double* rk_scratch;           // null: integrator arrays in shared memory; else [resident groups][size_fwd] in global memory
  WsLayout wl; RkLayout rl;
};

// slot of environment e: first record and capacity (0 when the plan does not fit the buffer)
template <class R> DMX_DI void tape_slot(const TapeView<R>& tp, const PlanView& pl, int e, long long& first, int& cap) {
  if (pl.offset) { first = pl.offset[e]; cap = pl.cap[e]; if (first + cap > tp.capacity) cap = 0; }
  else { first = (long long)e * tp.uniform_cap; cap = tp.uniform_cap; }
}
// 16-byte chunk c of the record of the step (q_n, v_n, t_n, hs, A_1..6) held in the integrator arrays
template <int ST> DMX_DI double tape_elem(const Rk<ST>& rk, int i, int nq, int nx, int o_A, int nA) {
  if (i < nq) return rk.q()[i];
  if (i < nx) return rk.v()[i - nq];
  if (o_A >= 0 && i >= o_A && i < o_A + nA) return rk.A()[i - o_A];
  return 0.0;
}
template <int ST> DMX_DI void tape_store_chunk(double* r, int c, const Rk<ST>& rk, int nq, int nx, int o_th, int o_A, int nA, double t, double hs) {
  const int i = 2 * c;
  double2 v;
  if (i == o_th) { v.x = t; v.y = hs; }
  else { v.x = tape_elem(rk, i, nq, nx, o_A, nA); v.y = tape_elem(rk, i + 1, nq, nx, o_A, nA); }
  reinterpret_cast<double2*>(r)[c] = v;
}
template <int ST> DMX_DI void tape_store_chunk(float* r, int c, const Rk<ST>& rk, int nq, int nx, int o_th, int o_A, int nA, double t, double hs) {
  const int i = 4 * c;
  float4 v;
  if (i == o_th) { double2 d; d.x = t; d.y = hs; v = *reinterpret_cast<float4*>(&d); }
  else { v.x = (float)tape_elem(rk, i, nq, nx, o_A, nA); v.y = (float)tape_elem(rk, i + 1, nq, nx, o_A, nA);
         v.z = (float)tape_elem(rk, i + 2, nq, nx, o_A, nA); v.w = (float)tape_elem(rk, i + 3, nq, nx, o_A, nA); }
  reinterpret_cast<float4*>(r)[c] = v;
}
// Next environment of a lane group (lane 0's value; the caller broadcasts it).  n_light < 0: the work queue, in launch
// order.  n_light >= 0: a single wave with one CTA per SM and no queue - the first n_light CTAs are half filled with the head
// of the launch order (the longest environments under a plan), the others are full: a launch lasts as long as its
// slowest SM, an SM with half the groups steps its environments ~8-14 % faster, so the spare group slots of a batch that
// does not fill the chip go next to the longest chains.  Which group runs an environment never
// changes its result (batch independence is tested).
template <int G> DMX_DI int next_env(int* queue, const int* order, int nenv, int n_light, bool& first) {
  int e;
  if (n_light < 0) e = atomicAdd(queue, 1);
  else if (first) {
    const int gpb = G == 1 ? blockDim.x : blockDim.x / G, gi = G == 1 ? threadIdx.x : threadIdx.x / G, half = gpb / 2, b = blockIdx.x;
    if (b < n_light) e = gi < half ? b * half + gi : nenv;
    else e = n_light * half + (b - n_light) * gpb + gi;
  } else e = nenv;
  first = false;
  if (e < nenv && order) e = order[e];
  return e;
}
template <class R> DMX_DI void tape_load_th(const R* r, int o_th, double& t, double& hs) {
  const double* d = reinterpret_cast<const double*>(r + o_th);
  t = d[0]; hs = d[1];
}

// Shared-memory copies of the model header and the layouts (one per CTA), so that the non-inlined device
// functions read them with plain shared loads.
template <class R> struct CtaConst { ModelDev<R> m; WsLayout wl, rwl; RkLayout rl; int nd; };
static __shared__ CtaConst<double> g_cc64;
static __shared__ CtaConst<float> g_cc32;
template <class R> DMX_DI CtaConst<R>& cta_const();
template <> DMX_DI CtaConst<double>& cta_const<double>() { return g_cc64; }
template <> DMX_DI CtaConst<float>& cta_const<float>() { return g_cc32; }
template <class R>
DMX_DI void load_cta_const(CtaConst<R>& c, const ModelDev<R>& m, const WsLayout& wl, const WsLayout& rwl, const RkLayout& rl, int nd) {
  if (threadIdx.x == 0) c.nd = nd;
  const int* src[4] = {reinterpret_cast<const int*>(&m), reinterpret_cast<const int*>(&wl), reinterpret_cast<const int*>(&rwl), reinterpret_cast<const int*>(&rl)};
  int* dst[4] = {reinterpret_cast<int*>(&c.m), reinterpret_cast<int*>(&c.wl), reinterpret_cast<int*>(&c.rwl), reinterpret_cast<int*>(&c.rl)};
  const int n[4] = {(int)(sizeof(ModelDev<R>) / 4), (int)(sizeof(WsLayout) / 4), (int)(sizeof(WsLayout) / 4), (int)(sizeof(RkLayout) / 4)};
#pragma unroll 1
  for (int k = 0; k < 4; ++k) for (int i = threadIdx.x; i < n[k]; i += blockDim.x) dst[k][i] = src[k][i];
  if (m.arena_smem) {
    // the constant arena goes to the last arena_bytes (a multiple of 16) of the CTA's dynamic shared memory
    unsigned dyn_bytes;
    asm volatile("mov.u32 %0, %%dynamic_smem_size;" : "=r"(dyn_bytes));
    unsigned char* sa = dyn_smem + (dyn_bytes - (unsigned)m.arena_bytes);
    const int4* g4 = reinterpret_cast<const int4*>(m.arena);
    int4* s4 = reinterpret_cast<int4*>(sa);
#pragma unroll 1
    for (int i = threadIdx.x; i < m.arena_bytes / 16; i += blockDim.x) s4[i] = g4[i];
    __syncthreads();
    const unsigned char** ptr = reinterpret_cast<const unsigned char**>(&c.m.body_parent);
#pragma unroll 1
    for (int i = threadIdx.x; i < N_ARENA_PTR; i += blockDim.x) ptr[i] = sa + (ptr[i] - m.arena);
  }
  __syncthreads();
}

// workspace bases of this thread's lane group inside the CTA's dynamic shared memory:
// [doubles | reals | ints], each region holding all groups of the CTA
template <class R, int G, class SH>
DMX_DI void bind_shared(unsigned char* smem, int nd, int nr_, int ni, Rk<StrideOf<G>::value>& rk, Ws<R, StrideOf<G>::value, SH>& ws,
                        Arr<R, StrideOf<G>::value>& Yqr, Arr<R, StrideOf<G>::value>& Vr, const RkLayout* rl, const WsLayout* wl) {
  const int ST = StrideOf<G>::value;
  const int ngr = (G == 1) ? blockDim.x : blockDim.x / G;
  double* dreg = reinterpret_cast<double*>(smem);
  R* rreg = reinterpret_cast<R*>(smem + (size_t)ngr * nd * sizeof(double));
  int* ireg = reinterpret_cast<int*>(smem + (size_t)ngr * nd * sizeof(double) + (size_t)ngr * nr_ * sizeof(R));
  if (G == 1) { int w = threadIdx.x >> 5, l = threadIdx.x & 31; dreg += (size_t)w * 32 * nd + l; rreg += (size_t)w * 32 * nr_ + l; ireg += (size_t)w * 32 * ni + l; }
  else { size_t gi = threadIdx.x / G; dreg += gi * nd; rreg += gi * nr_; ireg += gi * ni; }
  rk.b = dreg; rk.L = rl;
  ws.b = rreg; ws.ib = ireg; ws.L = wl;
  Yqr = Arr<R, ST>(rreg + rl->Yqr * ST); Vr = Arr<R, ST>(rreg + rl->Vr * ST);
}

// F or F~ at the stage state held in this group's (Yqr, Vr); one copy per kernel, shared by the stage recomputation
// and the VJP.  All pointers are re-derived from the CTA's shared memory, so the accesses stay shared-space loads.
template <class R, int G, class SH>
__device__ __noinline__ int field_eval(const R* u, const R* p, int cfd, int* conv_out, const double* xk) {
  const int ST = StrideOf<G>::value;
  CtaConst<R>& cc = cta_const<R>();
  const Grp<G> gr = make_group<G>();
  Rk<ST> rk; Ws<R, ST, SH> ws; Arr<R, ST> Yqr, Vr;
  bind_shared<R, G, SH>(dyn_smem, cc.nd, cc.wl.size + cc.rl.rsize, cc.wl.isize, rk, ws, Yqr, Vr, &cc.rl, &cc.wl);
  InPlain<R, ST> in; in.qa = Yqr; in.va = Vr; in.aa = Vr; in.ua = u; in.pa = p;
  bool conv; int iters;
  int nr = vector_field<Ws<R, ST, SH>, R, G, InPlain<R, ST> >(cc.m, in, ws, cfd != 0, conv, iters, gr, xk, ST);
  *conv_out = (conv ? 1 : 0) | (iters << 8);       // bit 0: converged; bits 8..: Newton iterations taken
  return nr;
}

// ---- forward rollout: persistent lane groups pulling environments from a global queue --------------
// register cap: three CTAs per SM where shared memory allows three (16 and 32 lanes: 168 registers); with 1 or 8 lanes
// shared memory allows two at most, and the cap of 255 removes the spills (C2 forward 49.5 -> 48 ms) and admits one CTA
// of 256 threads per SM (the single-wave launch of next_env)
template <class R, int G, class SH>
__global__ void __launch_bounds__((G <= 8 ? 256 : 128), (G <= 8 ? 1 : 3)) rollout_kernel(const __grid_constant__ ModelDev<R> m_, const __grid_constant__ RolloutArgs<R> a) {
  unsigned char* smem = dyn_smem;
  CtaConst<R>& cc = cta_const<R>();
  if (threadIdx.x == 0) g_lockstep = a.lockstep;
  const int nd_smem = a.rk_scratch ? 0 : a.rl.size_fwd;
  load_cta_const<R>(cc, m_, a.wl, a.wl, a.rl, nd_smem);
  const ModelDev<R>& m = cc.m;
  const int ST = StrideOf<G>::value;
  const Grp<G> gr = make_group<G>();
  Rk<ST> rk; Ws<R, ST, SH> ws; Arr<R, ST> Yqr, Vr;
  bind_shared<R, G, SH>(smem, nd_smem, a.wl.size + a.rl.rsize, a.wl.isize, rk, ws, Yqr, Vr, &cc.rl, &cc.wl);
  if (a.rk_scratch) {
    if (G == 1) rk.b = a.rk_scratch + ((size_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5)) * 32 * (size_t)a.rl.size_fwd + (threadIdx.x & 31);
    else rk.b = a.rk_scratch + ((size_t)blockIdx.x * (blockDim.x / G) + threadIdx.x / G) * (size_t)a.rl.size_fwd;
  }
  const int nq = m.nq, nv = m.nv, nu = m.nu, nx = nq + nv, tab = a.so.tableau, rec = a.tp.rec;
  const bool has_ctrl = a.ctrl != nullptr && a.nknot > 0 && nu > 0;
  const int nknot = has_ctrl ? a.nknot : 0;
  if (a.want_tape && blockIdx.x == 0 && threadIdx.x == 0) {   // what this tape holds; checked by the reverse sweep
    a.tp.meta[0] = TAPE_MAGIC; a.tp.meta[1] = a.nenv; a.tp.meta[2] = rec; a.tp.meta[3] = a.tp.o_A; a.tp.meta[4] = a.pl.offset ? 1 : 0;
    a.tp.meta[5] = a.tp.stride;
  }
  bool first_env = true;
#pragma unroll 1
  for (;;) {
    int e = 0;
    if (gr.lane == 0) e = next_env<G>(a.queue, a.pl.order, a.nenv, a.n_light, first_env);
    e = gr.bcast_int(e);
    if (e >= a.nenv) break;
    const R* x0 = a.x0 + (size_t)e * nx;
    const R* p = a.params ? a.params + (size_t)e * m.np : m.p_default;
#pragma unroll 1
    for (int j = gr.lane; j < nq; j += G) rk.q()[j] = (double)x0[j];
#pragma unroll 1
    for (int j = gr.lane; j < nv; j += G) rk.v()[j] = (double)x0[nq + j];
    gr.sync();
    double t = 0.0, hprop = a.so.h0, Eprev = 1.0, hmin = INFINITY, hmax = 0.0;
    int knot = 0, attempts = 0, ir = 0, status = 0, n_acc = 0, n_rej = 0, n_feval = 0, n_unc = 0;
    unsigned long long work[3] = {0, 0, 0};
    bool have_k1 = false, last_nonfinite = false;
    const double* hr = a.h_replay ? a.h_replay + (size_t)e * a.n_replay : nullptr;
    R* tape = nullptr; int tape_cap = 0; double* sched = nullptr;
    if (a.want_tape) {
      long long first; tape_slot(a.tp, a.pl, e, first, tape_cap);
      if (a.tp.stride > 1) { tape = a.tp.data + (size_t)(first / a.tp.stride + e) * rec; sched = a.tp.sched + first; }
      else tape = a.tp.data + (size_t)first * rec;
    }
    while (t < a.horizon) {
      double tb = has_ctrl ? fmin((knot + 1) * a.knot_dt, a.horizon) : a.horizon;
      if (knot + 1 >= nknot) tb = a.horizon;
      const R* u = has_ctrl ? a.ctrl + ((size_t)e * nknot + knot) * nu : a.zero_u;
      double rem = tb - t, h; bool hits;
      if (hr) {
        if (ir >= a.n_replay || !(hr[ir] > 0.0)) break;
        h = hr[ir++]; hits = (h == rem);
      } else {
        if (attempts >= a.so.max_steps) { status = 1; break; }
        if (hprop * (1.0 + 1e-7) >= rem) { h = rem; hits = true; } else { h = hprop; hits = false; }
        if (!hits && h < 1e-14 * fmax(1.0, fabs(t))) { status = last_nonfinite ? 3 : 2; break; }
      }
      if (tape && n_acc >= tape_cap) { status = 4; break; }
      attempts++;
      bool ok; int unc;
      rk_attempt<R, G, SH, false>(m, tab, rk, Yqr, Vr, u, p, h, have_k1, ws, ok, unc, gr, false, work);
      n_feval += have_k1 ? 6 : 7; n_unc += unc;
      have_k1 = true;
      bool finite = ok;
      double E = error_norm<R, ST>(m, rk, a.so.rtol, a.so.atol, finite);
      bool accept = true;
      last_nonfinite = !finite;
      if (!hr) {
        if (!finite) { E = INFINITY; accept = false; } else accept = E <= 1.0;
        double Ec = fmax(E, 1e-30);
        double fac = finite ? a.so.safety * exp(-(a.so.pcoeff + a.so.icoeff) / 5.0 * log(Ec)) * exp(a.so.pcoeff / 5.0 * log(Eprev)) : a.so.fac_min;
        fac = fmin(a.so.fac_max, fmax(a.so.fac_min, fac));
        if (!accept || !hits) hprop = h * fac;
        if (accept) Eprev = Ec;
      } else if (!finite) { status = 3; break; }
      if (!accept) { n_rej++; continue; }
      bool knot_up = hits && tb < a.horizon;
      if (tape && (!sched || n_acc % a.tp.stride == 0)) {   // S9: checkpoint record (y_n, t_n, +-h_n); a negative h marks a step that ends a control interval
        R* r = tape + (size_t)(sched ? n_acc / a.tp.stride : n_acc) * rec;
        const int nchunk = rec * (int)sizeof(R) / 16;
#pragma unroll 1
        for (int c = gr.lane; c < nchunk; c += G) tape_store_chunk(r, c, rk, nq, nx, a.tp.o_th, a.tp.o_A, sched ? nv : 6 * nv, t, knot_up ? -h : h);
      }
      if (sched && gr.lane == 0) sched[n_acc] = knot_up ? -h : h;
      gr.sync();
#pragma unroll 1
      for (int j = gr.lane; j < nq; j += G) rk.q()[j] = rk.Yq()[j];
#pragma unroll 1
      for (int j = gr.lane; j < nv; j += G) rk.v()[j] = rk.V()[j];
      n_acc++; hmin = fmin(hmin, h); hmax = fmax(hmax, h);
      if (hits) {
        t = tb;
        if (knot_up) { knot++; have_k1 = false; }
      } else t += h;
      if (have_k1) for (int j = gr.lane; j < nv; j += G) rk.A()[j] = rk.A()[6 * nv + j];
      gr.sync();
    }
    R* xT = a.xT + (size_t)e * nx;
#pragma unroll 1
    for (int j = gr.lane; j < nq; j += G) xT[j] = (R)rk.q()[j];
#pragma unroll 1
    for (int j = gr.lane; j < nv; j += G) xT[nq + j] = (R)rk.v()[j];
    if (gr.lane == 0) {
      if (a.n_accept) a.n_accept[e] = n_acc;
      if (a.n_reject) a.n_reject[e] = n_rej;
      if (a.n_feval) a.n_feval[e] = n_feval;
      if (a.n_unconv) a.n_unconv[e] = n_unc;
      if (a.status) a.status[e] = status;
      if (a.h_min) a.h_min[e] = hmin;
      if (a.h_max) a.h_max[e] = hmax;
      if (a.t_end) a.t_end[e] = t;
      if (a.work) { a.work[6 * (size_t)e] = work[0]; a.work[6 * (size_t)e + 1] = work[1]; a.work[6 * (size_t)e + 2] = work[2]; }
      if (a.want_tape) { a.tp.hdr[2 * e] = n_acc; a.tp.hdr[2 * e + 1] = (status == 0) ? knot : -1 - knot; }
    }
    gr.sync();
  }
  phase_drain();
}

}  // namespace dmx
