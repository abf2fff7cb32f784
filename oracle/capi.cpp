// ORACLE — test infrastructure only (see oracle/README.md). Not part of the product path.
//
// Flat C entry points for oracle/oracle.py (ctypes).  Single-threaded, fp64, plain loops.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
// may load this library.
#include <cstring>
#include <cstdio>
#include "rk.hpp"
#include "adjoint.hpp"

using namespace orc;

template <class T> static std::vector<T> cp(const T* p, size_t n) { return p ? std::vector<T>(p, p + n) : std::vector<T>(n, T(0)); }

extern "C" {

struct orc_desc {
  int nbody, njnt, nq, nv, nu, ngeom, npair;
  const int* body_parent; const double *body_pos, *body_quat, *body_mass, *body_ipos, *body_iquat, *body_inertia_unit;
  const int *jnt_type, *jnt_body, *jnt_qadr, *jnt_vadr; const double *jnt_axis, *jnt_pos, *jnt_damping, *jnt_armature;
  const int *geom_type, *geom_body; const double *geom_size, *geom_pos, *geom_quat;
  const int *pair_geom1, *pair_geom2, *pair_condim;
  const double *pair_friction, *pair_solref, *pair_solimp, *pair_solimp_cfd, *pair_cfd_beta;
  const int *act_type, *act_jnt; const double *act_gear, *act_kp, *act_kd;
  double gravity[3]; int newton_iters, ls_iters;
  const double* qpos0;
};

static char g_err[512] = "";
const char* orc_last_error() { return g_err; }


static void flatten_contacts(Model& m) {
  for (int pi = 0; pi < m.npair; ++pi) {
    int g1 = m.pair_geom1[pi], g2 = m.pair_geom2[pi];
    int t1 = m.geom_type[g1], t2 = m.geom_type[g2];
    Contact c; std::memset(&c, 0, sizeof(c));
    c.pair = pi; c.body1 = m.geom_body[g1]; c.body2 = m.geom_body[g2]; c.condim = m.pair_condim[pi];
    M3<double> R2 = quat_to_mat<double>(m.geom_quat[4 * g2], m.geom_quat[4 * g2 + 1], m.geom_quat[4 * g2 + 2], m.geom_quat[4 * g2 + 3]);
    V3<double> o2 = vconst<double>(&m.geom_pos[3 * g2]);
    auto setp2 = [&](const V3<double>& x) { c.p2[0] = x.x; c.p2[1] = x.y; c.p2[2] = x.z; };
    if (t1 == GEOM_PLANE) {
      if (c.body1 != 0) throw std::runtime_error("plane geoms must be attached to the world body");
      c.kind = CK_POINT_PLANE;
      M3<double> Rp = quat_to_mat<double>(m.geom_quat[4 * g1], m.geom_quat[4 * g1 + 1], m.geom_quat[4 * g1 + 2], m.geom_quat[4 * g1 + 3]);
      for (int k = 0; k < 3; ++k) { c.p1[k] = m.geom_pos[3 * g1 + k]; c.t1[k] = Rp.m[k][0]; c.t2[k] = Rp.m[k][1]; c.n[k] = Rp.m[k][2]; }
      const double* sz = &m.geom_size[3 * g2];
      if (t2 == GEOM_SPHERE) { c.rho2 = sz[0]; setp2(o2); m.contacts.push_back(c); }
      else if (t2 == GEOM_CAPSULE) {
        c.rho2 = sz[0];
        for (int s = -1; s <= 1; s += 2) { setp2(o2 + R2 * mk<double>(0.0, 0.0, s * sz[1])); m.contacts.push_back(c); }
      } else if (t2 == GEOM_BOX) {
        c.rho2 = 0.0;
        for (int k = 0; k < 8; ++k) {
          setp2(o2 + R2 * mk<double>((k & 1 ? 1 : -1) * sz[0], (k & 2 ? 1 : -1) * sz[1], (k & 4 ? 1 : -1) * sz[2]));
          m.contacts.push_back(c);
        }
      } else throw std::runtime_error("unsupported geom pair");
    } else if (t1 == GEOM_SPHERE && t2 == GEOM_SPHERE) {
      c.kind = CK_POINT_POINT; c.rho1 = m.geom_size[3 * g1]; c.rho2 = m.geom_size[3 * g2];
      for (int k = 0; k < 3; ++k) c.p1[k] = m.geom_pos[3 * g1 + k];
      setp2(o2); m.contacts.push_back(c);
    } else throw std::runtime_error("unsupported geom pair (plane must be geom1)");
  }
  m.nc = (int)m.contacts.size();
}

// G7: w(b) = mean diagonal of the translational block of Jc_b M(qpos0)^-1 Jc_b^T at the body's COM
static void inv_weights(Model& m) {
  int nv = m.nv;
  std::vector<double> M(nv * nv), zero(nv, 0.0);
  mass_matrix<double>(m, m.qpos0.data(), m.body_mass.data(), M.data());
  if (!cholesky(M, nv)) throw std::runtime_error("mass matrix at qpos0 is not positive definite");
  Kin<double> k; kinematics<double>(m, m.qpos0.data(), zero.data(), zero.data(), k);
  m.body_invweight.assign(m.nbody, 0.0);
  for (int b = 1; b < m.nbody; ++b) {
    double tr = 0.0;
    for (int c = 0; c < 3; ++c) {
      std::vector<double> row(nv);
      for (int j = 0; j < nv; ++j) { V3<double> lin, ang; dof_twist(m, k, j, b, k.com[b], lin, ang); row[j] = comp(lin, c); }
      std::vector<double> y = row; chol_solve(M, nv, y.data());
      for (int j = 0; j < nv; ++j) tr += row[j] * y[j];
    }
    m.body_invweight[b] = tr / 3.0;
  }
  m.pair_invweight.assign(m.npair, 0.0);
  for (int pi = 0; pi < m.npair; ++pi)
    m.pair_invweight[pi] = m.body_invweight[m.geom_body[m.pair_geom1[pi]]] + m.body_invweight[m.geom_body[m.pair_geom2[pi]]];
}

void* orc_model_create(const orc_desc* d) {
  try {
    Model* mp = new Model(); Model& m = *mp;
    m.nbody = d->nbody; m.njnt = d->njnt; m.nq = d->nq; m.nv = d->nv; m.nu = d->nu; m.ngeom = d->ngeom; m.npair = d->npair;
    m.np = m.nbody + 8 * m.npair;
    m.body_parent = cp(d->body_parent, m.nbody); m.body_pos = cp(d->body_pos, 3 * m.nbody); m.body_quat = cp(d->body_quat, 4 * m.nbody);
    m.body_mass = cp(d->body_mass, m.nbody); m.body_ipos = cp(d->body_ipos, 3 * m.nbody); m.body_iquat = cp(d->body_iquat, 4 * m.nbody);
    m.body_inertia_unit = cp(d->body_inertia_unit, 3 * m.nbody);
    m.jnt_type = cp(d->jnt_type, m.njnt); m.jnt_body = cp(d->jnt_body, m.njnt); m.jnt_qadr = cp(d->jnt_qadr, m.njnt); m.jnt_vadr = cp(d->jnt_vadr, m.njnt);
    m.jnt_axis = cp(d->jnt_axis, 3 * m.njnt); m.jnt_pos = cp(d->jnt_pos, 3 * m.njnt); m.jnt_damping = cp(d->jnt_damping, m.njnt); m.jnt_armature = cp(d->jnt_armature, m.njnt);
    m.geom_type = cp(d->geom_type, m.ngeom); m.geom_body = cp(d->geom_body, m.ngeom); m.geom_size = cp(d->geom_size, 3 * m.ngeom);
    m.geom_pos = cp(d->geom_pos, 3 * m.ngeom); m.geom_quat = cp(d->geom_quat, 4 * m.ngeom);
    m.pair_geom1 = cp(d->pair_geom1, m.npair); m.pair_geom2 = cp(d->pair_geom2, m.npair); m.pair_condim = cp(d->pair_condim, m.npair);
    m.pair_friction = cp(d->pair_friction, m.npair); m.pair_solref = cp(d->pair_solref, 2 * m.npair); m.pair_solimp = cp(d->pair_solimp, 5 * m.npair);
    m.pair_solimp_cfd = cp(d->pair_solimp_cfd, 5 * m.npair); m.pair_cfd_beta = cp(d->pair_cfd_beta, m.npair);
    m.act_type = cp(d->act_type, m.nu); m.act_jnt = cp(d->act_jnt, m.nu); m.act_gear = cp(d->act_gear, m.nu); m.act_kp = cp(d->act_kp, m.nu); m.act_kd = cp(d->act_kd, m.nu);
    for (int k = 0; k < 3; ++k) m.gravity[k] = d->gravity[k];
    m.newton_iters = d->newton_iters; m.ls_iters = d->ls_iters; m.qpos0 = cp(d->qpos0, m.nq);
    m.body_jnt.assign(m.nbody, -1); m.dof_jnt.assign(m.nv, -1); m.dof_body.assign(m.nv, -1);
    for (int j = 0; j < m.njnt; ++j) {
      int b = m.jnt_body[j];
      if (b <= 0 || b >= m.nbody || m.body_jnt[b] >= 0) throw std::runtime_error("each body carries at most one joint");
      if (m.jnt_type[j] == JNT_FREE && m.body_parent[b] != 0) throw std::runtime_error("free joints only on children of the world");
      m.body_jnt[b] = j;
      int nd = m.jnt_type[j] == JNT_FREE ? 6 : 1;
      for (int c = 0; c < nd; ++c) { m.dof_jnt[m.jnt_vadr[j] + c] = j; m.dof_body[m.jnt_vadr[j] + c] = b; }
    }
    for (int b = 1; b < m.nbody; ++b) if (m.body_parent[b] < 0 || m.body_parent[b] >= b) throw std::runtime_error("body_parent must precede the child");
    flatten_contacts(m);
    inv_weights(m);
    m.p_default.assign(m.np, 0.0);
    for (int b = 0; b < m.nbody; ++b) m.p_default[b] = m.body_mass[b];
    for (int i = 0; i < m.npair; ++i) m.p_default[m.p_fric() + i] = m.pair_friction[i];
    for (int i = 0; i < 2 * m.npair; ++i) m.p_default[m.p_solref() + i] = m.pair_solref[i];
    for (int i = 0; i < 5 * m.npair; ++i) m.p_default[m.p_solimp() + i] = m.pair_solimp[i];
    return mp;
  } catch (std::exception& e) { std::snprintf(g_err, sizeof(g_err), "%s", e.what()); return nullptr; }
}
void orc_model_destroy(void* h) { delete (Model*)h; }
int orc_np(void* h) { return ((Model*)h)->np; }
int orc_nc(void* h) { return ((Model*)h)->nc; }
void orc_default_params(void* h, double* p) { Model& m = *(Model*)h; for (int i = 0; i < m.np; ++i) p[i] = m.p_default[i]; }
void orc_invweight(void* h, double* body_w, double* pair_w) {
  Model& m = *(Model*)h;
  for (int i = 0; i < m.nbody; ++i) body_w[i] = m.body_invweight[i];
  for (int i = 0; i < m.npair; ++i) pair_w[i] = m.pair_invweight[i];
}

// ---- fine-grained entry points used by the pins --------------------------------------------
void orc_mass_matrix(void* h, const double* q, const double* p, double* M) { Model& m = *(Model*)h; mass_matrix<double>(m, q, p ? p : m.p_default.data(), M); }
void orc_inverse_dynamics(void* h, const double* q, const double* v, const double* a, const double* p, double* out) {
  Model& m = *(Model*)h; inverse_dynamics<double>(m, q, v, a, p ? p : m.p_default.data(), out);
}
// body frames: pos[nbody*3], mat[nbody*9], com[nbody*3], angular velocity [nbody*3], com velocity [nbody*3]
void orc_kinematics(void* h, const double* q, const double* v, double* pos, double* mat, double* com, double* angvel, double* comvel) {
  Model& m = *(Model*)h; std::vector<double> zero(m.nv, 0.0); Kin<double> k; kinematics<double>(m, q, v, zero.data(), k);
  for (int b = 0; b < m.nbody; ++b) {
    V3<double> cv = point_vel(k.fr[b], k.com[b]);
    for (int c = 0; c < 3; ++c) {
      pos[3 * b + c] = comp(k.fr[b].p, c); com[3 * b + c] = comp(k.com[b], c);
      angvel[3 * b + c] = comp(k.fr[b].w, c); comvel[3 * b + c] = comp(cv, c);
      for (int e = 0; e < 3; ++e) mat[9 * b + 3 * c + e] = k.fr[b].R.m[c][e];
    }
  }
}
// world inertia about the COM per body [nbody*9] (for momentum / energy invariants)
void orc_world_inertia(void* h, const double* q, const double* p, double* I) {
  Model& m = *(Model*)h; std::vector<double> zero(m.nv, 0.0); Kin<double> k; kinematics<double>(m, q, zero.data(), zero.data(), k);
  const double* pp = p ? p : m.p_default.data();
  for (int b = 0; b < m.nbody; ++b) { M3<double> W = world_inertia<double>(m, k, b, pp[b]); for (int c = 0; c < 3; ++c) for (int e = 0; e < 3; ++e) I[9 * b + 3 * c + e] = W.m[c][e]; }
}
// narrow phase for all candidates: r[nc], n[nc*3], pos[nc*3], t1[nc*3], t2[nc*3]
void orc_collide(void* h, const double* q, double* r, double* n, double* pos, double* t1, double* t2) {
  Model& m = *(Model*)h; std::vector<double> zero(m.nv, 0.0); Kin<double> k; kinematics<double>(m, q, zero.data(), zero.data(), k);
  for (int i = 0; i < m.nc; ++i) {
    Geo<double> g = collide<double>(m, k, m.contacts[i]); r[i] = g.r;
    for (int c = 0; c < 3; ++c) { n[3 * i + c] = comp(g.n, c); pos[3 * i + c] = comp(g.pos, c); t1[3 * i + c] = comp(g.t1, c); t2[3 * i + c] = comp(g.t2, c); }
  }
}
double orc_impedance(const double* solimp, double r) { return impedance<double>(r, solimp); }
double orc_impedance_cfd(const double* solimp_cfd, double r) { return impedance_cfd<double>(r, solimp_cfd); }
double orc_softplus(double z, double beta) { return softplus<double>(z, beta); }
// constraint rows at (q,v): returns nr; J[nr*nv], aref[nr], D[nr], r[nr] (buffers sized 4*nc rows)
int orc_rows(void* h, const double* q, const double* v, const double* p, int cfd, double* J, double* aref, double* D, double* r) {
  Model& m = *(Model*)h; std::vector<double> zero(m.nv, 0.0); Kin<double> k; kinematics<double>(m, q, v, zero.data(), k);
  Rows<double> R; build_rows<double>(m, k, v, p ? p : m.p_default.data(), cfd != 0, R);
  for (int i = 0; i < R.nr; ++i) { for (int j = 0; j < m.nv; ++j) J[i * m.nv + j] = R.J[i][j]; aref[i] = R.aref[i]; D[i] = R.D[i]; r[i] = R.r[i]; }
  return R.nr;
}
// generic contact solve on caller-supplied data (pins P5, P6)
int orc_contact_solve(int nv, int nr, const double* M, const double* a0, const double* J, const double* aref, const double* D,
                      int n_it, int n_ls, double* x, double* f, int* active) {
  std::vector<double> Mv(M, M + nv * nv); std::vector<std::vector<double>> Jv(nr, std::vector<double>(nv));
  for (int i = 0; i < nr; ++i) for (int j = 0; j < nv; ++j) Jv[i][j] = J[i * nv + j];
  SolveResult R = contact_solve(nv, nr, Mv, a0, Jv, aref, D, n_it, n_ls);
  for (int j = 0; j < nv; ++j) x[j] = R.x[j];
  for (int i = 0; i < nr; ++i) { f[i] = R.f[i]; active[i] = R.active[i]; }
  return R.converged ? R.iters : -R.iters;
}
// vector field: acc[nv]; returns rows in the solve, or -1 on failure; conv = solver converged flag
int orc_vector_field(void* h, const double* q, const double* v, const double* u, const double* p, int cfd, double* acc, int* conv) {
  Model& m = *(Model*)h; FieldOut f = vector_field(m, q, v, u, p ? p : m.p_default.data(), cfd != 0);
  for (int j = 0; j < m.nv; ++j) acc[j] = f.acc[j];
  if (conv) *conv = f.sol.converged;
  return f.ok ? f.rows.nr : -1;
}
int orc_vjp_field(void* h, const double* q, const double* v, const double* u, const double* p, const double* kappa, int cfd,
                  double* qbar, double* vbar, double* ubar, double* pbar) {
  Model& m = *(Model*)h; VjpOut o = vjp_field(m, q, v, u, p ? p : m.p_default.data(), kappa, cfd != 0, pbar != nullptr);
  for (int j = 0; j < m.nv; ++j) { qbar[j] = o.qbar[j]; vbar[j] = o.vbar[j]; }
  for (int j = 0; j < m.nu; ++j) ubar[j] = o.ubar[j];
  if (pbar) for (int j = 0; j < m.np; ++j) pbar[j] = o.pbar[j];
  return o.f.ok ? 0 : -1;
}
void orc_tableau(int which, double* c, double* a, double* b, double* e) {
  Tableau T = which == 0 ? dopri5() : tsit5();
  for (int i = 0; i < 7; ++i) { c[i] = T.c[i]; b[i] = T.b[i]; e[i] = T.e[i]; for (int j = 0; j < 7; ++j) a[7 * i + j] = T.a[i][j]; }
}
void orc_retract(void* h, const double* q, const double* delta, double* qout) { retract(*(Model*)h, q, delta, qout); }
void orc_ambient_to_tangent(void* h, const double* x, const double* g, double* lam) { ambient_to_tangent(*(Model*)h, x, g, lam); }

// ---- batched rollouts (SURVEY §8(b) shapes; env-major, row-contiguous) ----------------------
struct orc_opts { int tableau; double rtol, atol, h0, pcoeff, icoeff, safety, fac_min, fac_max; int max_steps; };

static SolverOpts so_of(const orc_opts* o) { SolverOpts s; s.tableau = o->tableau; s.rtol = o->rtol; s.atol = o->atol; s.h0 = o->h0; s.pcoeff = o->pcoeff; s.icoeff = o->icoeff; s.safety = o->safety; s.fac_min = o->fac_min; s.fac_max = o->fac_max; s.max_steps = o->max_steps; return s; }

// stats: int [nenv*5] (accept, reject, feval, unconverged, status), double [nenv*3] (h_min, h_max, t_end).
// h_out (optional): [nenv*n_hout] accepted step sizes, zero padded.  env range [e0,e1).
int orc_rollout(void* h, int e0, int e1, const double* x0, const double* ctrl, int nknot, double knot_dt, const double* params,
                double horizon, const orc_opts* opts, const double* h_replay, int n_replay,
                double* xT, int* istats, double* dstats, double* h_out, int n_hout) {
  Model& m = *(Model*)h; SolverOpts so = so_of(opts); int nx = m.nq + m.nv;
  for (int e = e0; e < e1; ++e) {
    EnvStats st; std::vector<TapeRec> tape;
    rollout_env(m, x0 + (size_t)e * nx, ctrl ? ctrl + (size_t)e * nknot * m.nu : nullptr, ctrl ? nknot : 0, knot_dt,
                params ? params + (size_t)e * m.np : m.p_default.data(), horizon, so,
                h_replay ? h_replay + (size_t)e * n_replay : nullptr, n_replay, xT + (size_t)e * nx, st, h_out ? &tape : nullptr);
    istats[5 * e] = st.n_accept; istats[5 * e + 1] = st.n_reject; istats[5 * e + 2] = st.n_feval; istats[5 * e + 3] = st.n_unconv; istats[5 * e + 4] = st.status;
    dstats[3 * e] = st.h_min; dstats[3 * e + 1] = st.h_max; dstats[3 * e + 2] = st.t_end;
    if (h_out) for (int i = 0; i < n_hout; ++i) h_out[(size_t)e * n_hout + i] = i < (int)tape.size() ? tape[i].h : 0.0;
  }
  return 0;
}
// forward with tape + reverse sweep.  dLdxT ambient [nenv, nq+nv]; outputs dLdx0 [nenv,2nv] tangent,
// dLdctrl [nenv,nknot,nu], dLdparams [nenv,np] (may be null).
int orc_rollout_grad(void* h, int e0, int e1, const double* x0, const double* ctrl, int nknot, double knot_dt, const double* params,
                     double horizon, const orc_opts* opts, const double* h_replay, int n_replay, const double* dLdxT, int cfd_on,
                     double* xT, int* istats, double* dstats, double* dLdx0, double* dLdctrl, double* dLdparams) {
  Model& m = *(Model*)h; SolverOpts so = so_of(opts); int nx = m.nq + m.nv, nv = m.nv;
  for (int e = e0; e < e1; ++e) {
    EnvStats st; std::vector<TapeRec> tape;
    const double* ce = ctrl ? ctrl + (size_t)e * nknot * m.nu : nullptr;
    const double* pe = params ? params + (size_t)e * m.np : m.p_default.data();
    rollout_env(m, x0 + (size_t)e * nx, ce, ctrl ? nknot : 0, knot_dt, pe, horizon, so,
                h_replay ? h_replay + (size_t)e * n_replay : nullptr, n_replay, xT + (size_t)e * nx, st, &tape);
    istats[5 * e] = st.n_accept; istats[5 * e + 1] = st.n_reject; istats[5 * e + 2] = st.n_feval; istats[5 * e + 3] = st.n_unconv; istats[5 * e + 4] = st.status;
    dstats[3 * e] = st.h_min; dstats[3 * e + 1] = st.h_max; dstats[3 * e + 2] = st.t_end;
    std::vector<double> lam(2 * nv, 0.0);
    double* gc = dLdctrl ? dLdctrl + (size_t)e * nknot * m.nu : nullptr;
    double* gp = dLdparams ? dLdparams + (size_t)e * m.np : nullptr;
    if (gc) for (int i = 0; i < nknot * m.nu; ++i) gc[i] = 0.0;
    if (gp) for (int i = 0; i < m.np; ++i) gp[i] = 0.0;
    bool ok = st.status == 0;
    if (ok) {
      ambient_to_tangent(m, xT + (size_t)e * nx, dLdxT + (size_t)e * nx, lam.data());
      ok = reverse_sweep(m, tape, ce, ctrl ? nknot : 0, pe, so, cfd_on != 0, lam.data(), gc, gp);
    }
    if (!ok) {   // failed env: zero gradients (SURVEY §8(b) Errors)
      for (auto& l : lam) l = 0.0;
      if (gc) for (int i = 0; i < nknot * m.nu; ++i) gc[i] = 0.0;
      if (gp) for (int i = 0; i < m.np; ++i) gp[i] = 0.0;
    }
    for (int i = 0; i < 2 * nv; ++i) dLdx0[(size_t)e * 2 * nv + i] = lam[i];
  }
  return 0;
}

// forward with tape, then the continuous adjoint solved backwards with its own steps (adjoint.hpp; PAPER.md:435-448,
// 462-477).  adj: solver options of the backward solve.  asub [nenv,3]: accepted / rejected sub-steps, status.
int orc_rollout_grad_adjoint(void* h, int e0, int e1, const double* x0, const double* ctrl, int nknot, double knot_dt, const double* params,
                             double horizon, const orc_opts* opts, const orc_opts* adj, const double* h_replay, int n_replay, const double* dLdxT,
                             int cfd_on, double* xT, int* istats, double* dstats, int* asub, double* dLdx0, double* dLdctrl, double* dLdparams,
                             const double* adj_replay, int n_adj_replay, double* adj_hout, int n_adj_hout) {
  Model& m = *(Model*)h; SolverOpts so = so_of(opts), sa = so_of(adj); int nx = m.nq + m.nv, nv = m.nv;
  for (int e = e0; e < e1; ++e) {
    EnvStats st; std::vector<TapeRec> tape;
    const double* ce = ctrl ? ctrl + (size_t)e * nknot * m.nu : nullptr;
    const double* pe = params ? params + (size_t)e * m.np : m.p_default.data();
    rollout_env(m, x0 + (size_t)e * nx, ce, ctrl ? nknot : 0, knot_dt, pe, horizon, so,
                h_replay ? h_replay + (size_t)e * n_replay : nullptr, n_replay, xT + (size_t)e * nx, st, &tape);
    istats[5 * e] = st.n_accept; istats[5 * e + 1] = st.n_reject; istats[5 * e + 2] = st.n_feval; istats[5 * e + 3] = st.n_unconv; istats[5 * e + 4] = st.status;
    dstats[3 * e] = st.h_min; dstats[3 * e + 1] = st.h_max; dstats[3 * e + 2] = st.t_end;
    std::vector<double> lam(2 * nv, 0.0);
    double* gc = dLdctrl ? dLdctrl + (size_t)e * nknot * m.nu : nullptr;
    double* gp = dLdparams ? dLdparams + (size_t)e * m.np : nullptr;
    if (gc) for (int i = 0; i < nknot * m.nu; ++i) gc[i] = 0.0;
    if (gp) for (int i = 0; i < m.np; ++i) gp[i] = 0.0;
    bool ok = st.status == 0;
    AdjStats as; std::vector<double> hsub;
    if (ok) {
      ambient_to_tangent(m, xT + (size_t)e * nx, dLdxT + (size_t)e * nx, lam.data());
      ok = reverse_sweep_continuous(m, tape, ce, ctrl ? nknot : 0, pe, so, sa, cfd_on != 0, lam.data(), gc, gp, as,
                                    adj_replay ? adj_replay + (size_t)e * n_adj_replay : nullptr, n_adj_replay, adj_hout ? &hsub : nullptr);
    }
    if (adj_hout) for (int i = 0; i < n_adj_hout; ++i) adj_hout[(size_t)e * n_adj_hout + i] = i < (int)hsub.size() ? hsub[i] : 0.0;
    if (!ok) {
      for (auto& l : lam) l = 0.0;
      if (gc) for (int i = 0; i < nknot * m.nu; ++i) gc[i] = 0.0;
      if (gp) for (int i = 0; i < m.np; ++i) gp[i] = 0.0;
    }
    if (asub) { asub[3 * e] = as.n_accept; asub[3 * e + 1] = as.n_reject; asub[3 * e + 2] = ok ? 0 : (as.status ? as.status : 3); }
    for (int i = 0; i < 2 * nv; ++i) dLdx0[(size_t)e * 2 * nv + i] = lam[i];
  }
  return 0;
}

}  // extern "C"
