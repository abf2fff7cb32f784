// dmx_api.cu — the C-ABI of include/dmx.h: model flattening and upload, workspace layouts, kernel
// dispatch.  Host code only prepares constants and launches; every step of the path (S1-S12 of
// SURVEY.md §8(a)) runs in the kernels of dmx_kernels.cuh.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <cmath>
#include <string>
#include <vector>
#include <atomic>
#include <stdexcept>
#include "../../include/dmx.h"
#include "dmx_adjoint.cuh"

using namespace dmx;

static thread_local char g_err[512] = "";
static int fail(const char* fmt, const char* a = "") { std::snprintf(g_err, sizeof(g_err), fmt, a); return -1; }
#define CUDA_OK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) return fail("CUDA error: %s", cudaGetErrorString(e_)); } while (0)

namespace {

// ---- dispatch table over (real type, lanes) ----------------------------------------------------------
template <class R> struct Launchers {
  cudaError_t (*rollout)(const ModelDev<R>&, const RolloutArgs<R>&, LaunchCfg, cudaStream_t);
  cudaError_t (*backward)(const ModelDev<R>&, const BackwardArgs<R>&, LaunchCfg, cudaStream_t);
  cudaError_t (*backward_ckpt)(const ModelDev<R>&, const BackwardArgs<R>&, LaunchCfg, cudaStream_t);
  cudaError_t (*adjoint)(const ModelDev<R>&, const AdjointArgs<R>&, LaunchCfg, cudaStream_t);
  cudaError_t (*field)(const ModelDev<R>&, const FieldArgs<R>&, LaunchCfg, cudaStream_t);
  cudaError_t (*invweight)(const ModelDev<R>&, const R*, const R*, R*, const WsLayout&, const RkLayout&, LaunchCfg, cudaStream_t);
  cudaError_t (*occupancy)(int, size_t, size_t, size_t, int*, int*, int*);
  cudaError_t (*prof_dump)(unsigned long long*, cudaStream_t);
};
template <class R, int G, class SH> Launchers<R> make_launchers() {
  Launchers<R> l;
  l.rollout = &launch_rollout<R, G, SH>; l.backward = &launch_backward<R, G, SH>; l.adjoint = &launch_adjoint<R, G, SH>; l.backward_ckpt = &launch_backward_ckpt<R, G, SH>; l.field = &launch_field<R, G, SH>;
  l.invweight = &launch_invweight<R, G, SH>; l.occupancy = &kernel_occupancy<R, G, SH>; l.prof_dump = &launch_prof_dump<R, G, SH>;
  return l;
}
// shape: 0 = sizes taken at run time; 2..5 = the static instantiation of BASELINE config C2..C5 (dmx_model.cuh)
template <class R> Launchers<R> launchers_for(int G, int shape);
template <> Launchers<double> launchers_for<double>(int G, int shape) {
  if (shape == 2 && G == 8) return make_launchers<double, 8, ShapeC2>();
  if (shape == 3 && G == 16) return make_launchers<double, 16, ShapeC3>();
  if (shape == 4 && G == 32) return make_launchers<double, 32, ShapeC4>();
  if (shape == 5 && G == 32) return make_launchers<double, 32, ShapeC5>();
  switch (G) {
    case 1: return make_launchers<double, 1, ShapeDyn>();
    case 8: return make_launchers<double, 8, ShapeDyn>();
    case 16: return make_launchers<double, 16, ShapeDyn>();
    default: return make_launchers<double, 32, ShapeDyn>();
  }
}
template <> Launchers<float> launchers_for<float>(int G, int shape) {
  if (shape == 3 && G == 16) return make_launchers<float, 16, ShapeC3>();
  switch (G) {
    case 1: return make_launchers<float, 1, ShapeDyn>();
    case 8: return make_launchers<float, 8, ShapeDyn>();
    case 16: return make_launchers<float, 16, ShapeDyn>();
    default: return make_launchers<float, 32, ShapeDyn>();
  }
}
template <class SH> bool shape_matches(int nv, int nc, int nr) { return SH::NV == nv && SH::NC == nc && SH::NR == nr; }
// static instantiation whose sizes equal the model's (DMX_STATIC=0 forces the run-time sizes)
int pick_shape(int precision, int G, int nv, int nc, int nr) {
  const char* e = std::getenv("DMX_STATIC");
  if (e && std::atoi(e) == 0) return 0;
  if (precision == 64 && G == 8 && shape_matches<ShapeC2>(nv, nc, nr)) return 2;
  if (G == 16 && shape_matches<ShapeC3>(nv, nc, nr)) return 3;
  if (precision == 64 && G == 32 && shape_matches<ShapeC4>(nv, nc, nr)) return 4;
  // C5 (nv = 18): measured slower than the run-time sizes (the unrolled code no longer fits the instruction cache:
  // stall_no_inst 30 %); selected only on request
  if (e && std::atoi(e) == 2 && precision == 64 && G == 32 && shape_matches<ShapeC5>(nv, nc, nr)) return 5;
  return 0;
}
int shape_ld(int shape, int nv) { return shape == 2 ? ShapeC2::LD : shape == 3 ? ShapeC3::LD : shape == 4 ? ShapeC4::LD : shape == 5 ? ShapeC5::LD : nv; }

// ---- device arena: one allocation holding every constant array ------------------------------------------
struct Arena {
  std::vector<unsigned char> host; unsigned char* dev = nullptr;
  size_t add(const void* p, size_t bytes) {
    size_t off = (host.size() + 15) & ~size_t(15);
    host.resize(off + bytes);
    if (bytes) std::memcpy(host.data() + off, p, bytes);
    return off;
  }
};

struct HostModel {   // flattened description, doubles
  int nbody, njnt, nq, nv, nu, npair, nc, np, nlevel, ntw, nmp, nrmax, newton_iters, ls_iters;
  std::vector<int> body_parent, body_jnt, level_ptr, level_body, jnt_type, jnt_qadr, jnt_vadr, jnt_body, dof_jnt, dof_body, dof_rot,
      tw_ptr, tw_body, tw_dof, tw_idx, sub_ptr, sub_body, child_ptr, child_idx, mp_i, mp_j, mp_deep, ct_kind, ct_b1, ct_b2, ct_condim, ct_pair, act_type, act_jnt;
  std::vector<double> body_pos, body_rot, body_ipos, body_irot, body_iunit, jnt_axis, jnt_pos, jnt_damping, jnt_armature, ct_p1, ct_p2,
      ct_rho1, ct_rho2, ct_n, ct_t1, ct_t2, pair_invweight, pair_solimp_cfd, pair_cfd_beta, act_gear, act_kp, act_kd, p_default, qpos0;
  std::vector<int> pair_body1, pair_body2;
  double gravity[3];
};

void quat_rot(const double* q, double* Rm) {   // rotation matrix (row-major) of a quaternion (w,x,y,z)
  double w = q[0], x = q[1], y = q[2], z = q[3];
  Rm[0] = w * w + x * x - y * y - z * z; Rm[1] = 2 * (x * y - w * z); Rm[2] = 2 * (x * z + w * y);
  Rm[3] = 2 * (x * y + w * z); Rm[4] = w * w - x * x + y * y - z * z; Rm[5] = 2 * (y * z - w * x);
  Rm[6] = 2 * (x * z - w * y); Rm[7] = 2 * (y * z + w * x); Rm[8] = w * w - x * x - y * y + z * z;
}
void mat_vec(const double* Rm, const double* v, double* o) { for (int i = 0; i < 3; ++i) o[i] = Rm[3 * i] * v[0] + Rm[3 * i + 1] * v[1] + Rm[3 * i + 2] * v[2]; }

template <class T> std::vector<T> cpv(const T* p, size_t n) { return p ? std::vector<T>(p, p + n) : std::vector<T>(n, T(0)); }

void flatten(const dmx_model_desc* d, HostModel& h) {
  h.nbody = d->nbody; h.njnt = d->njnt; h.nq = d->nq; h.nv = d->nv; h.nu = d->nu; h.npair = d->npair;
  h.newton_iters = d->newton_iters; h.ls_iters = d->ls_iters;
  for (int k = 0; k < 3; ++k) h.gravity[k] = d->gravity[k];
  const int nb = h.nbody, nv = h.nv;
  if (nb < 1 || nv < 1 || h.nq < nv) throw std::runtime_error("empty model");
  h.np = nb + 8 * h.npair;
  h.body_parent = cpv(d->body_parent, nb); h.body_pos = cpv(d->body_pos, 3 * nb); h.body_ipos = cpv(d->body_ipos, 3 * nb);
  h.body_iunit = cpv(d->body_inertia_unit, 3 * nb);
  h.body_rot.assign(9 * nb, 0.0); h.body_irot.assign(9 * nb, 0.0);
  for (int b = 0; b < nb; ++b) { quat_rot(d->body_quat + 4 * b, &h.body_rot[9 * b]); quat_rot(d->body_iquat + 4 * b, &h.body_irot[9 * b]); }
  h.jnt_type = cpv(d->jnt_type, h.njnt); h.jnt_qadr = cpv(d->jnt_qadr, h.njnt); h.jnt_vadr = cpv(d->jnt_vadr, h.njnt); h.jnt_body = cpv(d->jnt_body, h.njnt);
  h.jnt_axis = cpv(d->jnt_axis, 3 * h.njnt); h.jnt_pos = cpv(d->jnt_pos, 3 * h.njnt); h.jnt_damping = cpv(d->jnt_damping, h.njnt);
  h.jnt_armature = cpv(d->jnt_armature, h.njnt);
  h.body_jnt.assign(nb, -1); h.dof_jnt.assign(nv, -1); h.dof_body.assign(nv, -1); h.dof_rot.assign(nv, 0);
  for (int b = 1; b < nb; ++b) if (h.body_parent[b] < 0 || h.body_parent[b] >= b) throw std::runtime_error("body_parent must precede the child");
  for (int j = 0; j < h.njnt; ++j) {
    int b = h.jnt_body[j], t = h.jnt_type[j];
    if (b <= 0 || b >= nb || h.body_jnt[b] >= 0) throw std::runtime_error("each body carries at most one joint");
    if (t == JNT_FREE && h.body_parent[b] != 0) throw std::runtime_error("free joints only on children of the world");
    if (t != JNT_FREE && t != JNT_HINGE && t != JNT_SLIDE) throw std::runtime_error("unknown joint type");
    h.body_jnt[b] = j;
    int nd = t == JNT_FREE ? 6 : 1;
    if (h.jnt_vadr[j] < 0 || h.jnt_vadr[j] + nd > nv) throw std::runtime_error("jnt_vadr out of range");
    for (int c = 0; c < nd; ++c) {
      h.dof_jnt[h.jnt_vadr[j] + c] = j; h.dof_body[h.jnt_vadr[j] + c] = b;
      h.dof_rot[h.jnt_vadr[j] + c] = (t == JNT_HINGE) || (t == JNT_FREE && c >= 3);
    }
  }
  for (int j = 0; j < nv; ++j) if (h.dof_jnt[j] < 0) throw std::runtime_error("dof without a joint");
  // tree levels
  std::vector<int> depth(nb, 0); int maxd = 0;
  for (int b = 1; b < nb; ++b) { depth[b] = depth[h.body_parent[b]] + 1; maxd = std::max(maxd, depth[b]); }
  h.nlevel = maxd; h.level_ptr.assign(1, 0);
  for (int l = 1; l <= maxd; ++l) { for (int b = 1; b < nb; ++b) if (depth[b] == l) h.level_body.push_back(b); h.level_ptr.push_back((int)h.level_body.size()); }
  auto anc = [&](int a, int b) { while (b > 0) { if (b == a) return true; b = h.body_parent[b]; } return false; };
  // (body, ancestor dof) table and subtree lists
  h.tw_idx.assign((size_t)nb * nv, -1); h.tw_ptr.assign(nb + 1, 0); h.sub_ptr.assign(nb + 1, 0);
  for (int b = 0; b < nb; ++b) {
    h.tw_ptr[b] = (int)h.tw_dof.size();
    if (b > 0) for (int j = 0; j < nv; ++j) if (anc(h.dof_body[j], b)) { h.tw_idx[(size_t)b * nv + j] = (int)h.tw_dof.size(); h.tw_dof.push_back(j); h.tw_body.push_back(b); }
    h.sub_ptr[b] = (int)h.sub_body.size();
    if (b > 0) for (int c = b; c < nb; ++c) if (anc(b, c)) h.sub_body.push_back(c);
  }
  h.tw_ptr[nb] = (int)h.tw_dof.size(); h.sub_ptr[nb] = (int)h.sub_body.size(); h.ntw = (int)h.tw_dof.size();
  h.child_ptr.assign(nb + 1, 0);
  for (int b = 0; b < nb; ++b) { h.child_ptr[b] = (int)h.child_idx.size(); for (int c = b + 1; c < nb; ++c) if (h.body_parent[c] == b) h.child_idx.push_back(c); }
  h.child_ptr[nb] = (int)h.child_idx.size();
  for (int i = 0; i < nv; ++i) for (int j = 0; j <= i; ++j) {
    int bi = h.dof_body[i], bj = h.dof_body[j];
    h.mp_i.push_back(i); h.mp_j.push_back(j);
    h.mp_deep.push_back(anc(bj, bi) ? bi : (anc(bi, bj) ? bj : -1));
  }
  h.nmp = (int)h.mp_i.size();
  // candidate contacts: every supported geom pair flattens to sphere-like points
  h.pair_body1.resize(h.npair); h.pair_body2.resize(h.npair);
  auto push = [&](int pi, int kind, int b1, int b2, int condim, const double* p1, const double* p2, double r1, double r2, const double* fr) {
    h.ct_pair.push_back(pi); h.ct_kind.push_back(kind); h.ct_b1.push_back(b1); h.ct_b2.push_back(b2); h.ct_condim.push_back(condim);
    for (int k = 0; k < 3; ++k) { h.ct_p1.push_back(p1[k]); h.ct_p2.push_back(p2[k]); h.ct_t1.push_back(fr ? fr[3 * k] : 0.0); h.ct_t2.push_back(fr ? fr[3 * k + 1] : 0.0); h.ct_n.push_back(fr ? fr[3 * k + 2] : 0.0); }
    h.ct_rho1.push_back(r1); h.ct_rho2.push_back(r2);
  };
  for (int pi = 0; pi < h.npair; ++pi) {
    int g1 = d->pair_geom1[pi], g2 = d->pair_geom2[pi];
    if (g1 < 0 || g2 < 0 || g1 >= d->ngeom || g2 >= d->ngeom) throw std::runtime_error("pair geom out of range");
    int t1 = d->geom_type[g1], t2 = d->geom_type[g2], b1 = d->geom_body[g1], b2 = d->geom_body[g2], cd = d->pair_condim[pi];
    if (cd != 1 && cd != 3) throw std::runtime_error("condim must be 1 or 3");
    h.pair_body1[pi] = b1; h.pair_body2[pi] = b2;
    double R2[9]; quat_rot(d->geom_quat + 4 * g2, R2);
    const double* o2 = d->geom_pos + 3 * g2; const double* sz = d->geom_size + 3 * g2;
    if (t1 == DMX_GEOM_PLANE) {
      if (b1 != 0) throw std::runtime_error("plane geoms must be attached to the world body");
      double Rp[9]; quat_rot(d->geom_quat + 4 * g1, Rp);
      const double* pp = d->geom_pos + 3 * g1;
      if (t2 == DMX_GEOM_SPHERE) push(pi, CK_POINT_PLANE, b1, b2, cd, pp, o2, 0.0, sz[0], Rp);
      else if (t2 == DMX_GEOM_CAPSULE) {
        for (int s = -1; s <= 1; s += 2) { double l[3] = {0, 0, s * sz[1]}, w[3]; mat_vec(R2, l, w); for (int k = 0; k < 3; ++k) w[k] += o2[k]; push(pi, CK_POINT_PLANE, b1, b2, cd, pp, w, 0.0, sz[0], Rp); }
      } else if (t2 == DMX_GEOM_BOX) {
        for (int c = 0; c < 8; ++c) {
          double l[3] = {(c & 1 ? 1 : -1) * sz[0], (c & 2 ? 1 : -1) * sz[1], (c & 4 ? 1 : -1) * sz[2]}, w[3];
          mat_vec(R2, l, w); for (int k = 0; k < 3; ++k) w[k] += o2[k];
          push(pi, CK_POINT_PLANE, b1, b2, cd, pp, w, 0.0, 0.0, Rp);
        }
      } else throw std::runtime_error("unsupported geom pair");
    } else if (t1 == DMX_GEOM_SPHERE && t2 == DMX_GEOM_SPHERE) {
      push(pi, CK_POINT_POINT, b1, b2, cd, d->geom_pos + 3 * g1, o2, d->geom_size[3 * g1], sz[0], nullptr);
    } else throw std::runtime_error("unsupported geom pair (plane must be geom1)");
  }
  h.nc = (int)h.ct_kind.size();
  h.nrmax = 0; for (int c = 0; c < h.nc; ++c) h.nrmax += h.ct_condim[c] == 3 ? 4 : 1;
  h.pair_solimp_cfd = cpv(d->pair_solimp_cfd, 5 * h.npair); h.pair_cfd_beta = cpv(d->pair_cfd_beta, h.npair);
  h.pair_invweight.assign(h.npair, 0.0);
  h.act_type = cpv(d->act_type, h.nu); h.act_jnt = cpv(d->act_jnt, h.nu); h.act_gear = cpv(d->act_gear, h.nu); h.act_kp = cpv(d->act_kp, h.nu); h.act_kd = cpv(d->act_kd, h.nu);
  for (int i = 0; i < h.nu; ++i) if (h.act_jnt[i] < 0 || h.act_jnt[i] >= h.njnt || h.jnt_type[h.act_jnt[i]] == JNT_FREE) throw std::runtime_error("actuators act on hinge / slide joints");
  h.p_default.assign(h.np, 0.0);
  for (int b = 0; b < nb; ++b) h.p_default[b] = d->body_mass[b];
  for (int i = 0; i < h.npair; ++i) h.p_default[nb + i] = d->pair_friction[i];
  for (int i = 0; i < 2 * h.npair; ++i) h.p_default[nb + h.npair + i] = d->pair_solref[i];
  for (int i = 0; i < 5 * h.npair; ++i) h.p_default[nb + 3 * h.npair + i] = d->pair_solimp[i];
  h.qpos0 = cpv(d->qpos0, h.nq);
}

// Optional shared-memory bank spread (DMX_PAD=1; off by default: measured on B200 it removes a third of the bank
// conflicts but the shared-memory pipe runs at 0.25 wavefronts/cycle, so it buys <= 2 % and costs workspace bytes): with several lanes per environment a lane i reads row i of M, H
// or J, so an even leading dimension puts the lanes of a group on 2-4 banks; an odd one spreads them over all of them.
// With 8 lanes per environment the slices of neighbouring groups are offset by 8 scalars modulo 16 doubles / 32 floats,
// so the groups that share a shared-memory wavefront use complementary banks.
// wl / rl: the full workspace (reverse sweep, field kernels).  wlf / rlf: the forward kernel's workspace, in which arrays
// with disjoint lifetimes inside one F evaluation share storage (DMX_FWD_ALIAS=0: same as wl): the body velocities /
// accelerations and the temporaries of the dynamics phase (wrenches, world inertias, twist table) are dead once M, c and
// tau are known, and the arrays of the contact solve (H, J, row vectors, Newton vectors) are first written after that;
// the arrays only the VJP touches are dropped.  Fewer bytes per environment = more resident lane groups per SM.
void make_layouts(const HostModel& h, int G, int real_bytes, int static_ld, WsLayout& wl, WsLayout& wlf, RkLayout& rl, RkLayout& rlf) {
  const char* ep = std::getenv("DMX_PAD");
  const bool pad = G > 1 && ep && std::atoi(ep) != 0 && static_ld == 0;
  const int ld = static_ld ? static_ld : ((pad && h.nv > 1 && h.nv % 2 == 0) ? h.nv + 1 : h.nv);
  auto stagger = [&](int n, int scalar_bytes) { if (!pad || G != 8 || n == 0) return n; int mod = 64 / scalar_bytes * 2; while (n % mod != 8) ++n; return n; };
  const int nb = h.nbody, nv = h.nv, nq = h.nq, nc = std::max(h.nc, 1), nr = std::max(h.nrmax, 1);
  std::memset(&wl, 0, sizeof(wl)); std::memset(&wlf, 0, sizeof(wlf)); std::memset(&rl, 0, sizeof(rl));
  int o = 0;
  auto take = [&](int& f, int n) { f = o; o += n; };
  take(wl.fp, 3 * nb); take(wl.fR, 9 * nb); take(wl.fw, 3 * nb); take(wl.fal, 3 * nb); take(wl.fvp, 3 * nb); take(wl.fap, 3 * nb);
  take(wl.com, 3 * nb); take(wl.dax, 3 * nv); take(wl.dan, 3 * nv);
  take(wl.Fb, 3 * nb); take(wl.Nb, 3 * nb); take(wl.Iw, 9 * nb); take(wl.Isub, 9 * nb); take(wl.tw, 3 * std::max(h.ntw, 1));
  wl.ld = ld;
  take(wl.M, nv * ld); take(wl.Hc, nv * ld); take(wl.tau, nv); take(wl.c, nv); take(wl.a0, nv); take(wl.x, nv); take(wl.g, nv);
  take(wl.dl, nv); take(wl.Md, nv); take(wl.xa, nv); take(wl.kap, nv);
  take(wl.cr, nc); take(wl.cn, 3 * nc); take(wl.cpos, 3 * nc); take(wl.ct1, 3 * nc); take(wl.ct2, 3 * nc);
  take(wl.cD, nc); take(wl.cpost, nc); take(wl.cbd, nc); take(wl.cmu, nc); take(wl.cdD, nc); take(wl.cdpost, nc);
  take(wl.fox, 3 * nb); take(wl.fvx, 3 * nb);
  take(wl.J, std::max(nr * ld, nc * nv) /* also the (candidate, dof) scratch of the VJP */); take(wl.aref, nr); take(wl.D, nr); take(wl.s, nr); take(wl.pr, nr);
  wl.size = stagger(o + nq + nv, real_bytes) - (nq + nv);
  rl.Yqr = o; rl.Vr = o + nq; rl.rsize = nq + nv;
  o = 0;
  take(wl.i_incl, nc); take(wl.i_rowstart, nc); take(wl.i_rowcand, nr); take(wl.i_active, nr);
  wl.isize = o;
  o = 0;
  take(rl.q, nq); take(rl.v, nv); take(rl.Yq, nq); take(rl.V, nv); take(rl.Dl, nv); take(rl.K, 7 * nv); take(rl.A, 7 * nv); take(rl.err, 2 * nv);
  rl.size_fwd = stagger(o, 8);
  take(rl.sYq, 6 * nq); take(rl.sV, 6 * nv); take(rl.sDl, 6 * nv); take(rl.Kb, 6 * nv); take(rl.Ab, 6 * nv);
  take(rl.qb, nv); take(rl.vb, nv); take(rl.dbar, nv); take(rl.Vb, nv); take(rl.lam, 2 * nv); take(rl.delta, nv);
  take(rl.qbar, nv); take(rl.vbar, nv); take(rl.ubar, std::max(h.nu, 1)); take(rl.pbar, h.np); take(rl.gp, h.np);
  rl.size_bwd = stagger(o, 8);
  o = rl.size_bwd;
  take(rl.ak, 14 * nv); take(rl.aub, 7 * std::max(h.nu, 1)); take(rl.apb, 7 * std::max(h.np, 1));
  take(rl.amu, 2 * nv); take(rl.amus, 2 * nv); take(rl.amunew, 2 * nv); take(rl.az1, 2 * nv); take(rl.adz1, 2 * nv);
  rl.size_adj = o;
  wlf = wl; rlf = rl;
  const char* ea = std::getenv("DMX_FWD_ALIAS");
  if (ea && std::atoi(ea) == 0) return;
  {
    WsLayout& f = wlf;
    o = 0;
    take(f.fp, 3 * nb); take(f.fR, 9 * nb); take(f.com, 3 * nb); take(f.dax, 3 * nv); take(f.dan, 3 * nv);
    take(f.M, nv * ld); take(f.tau, nv); take(f.c, nv); take(f.a0, nv);
    take(f.cr, nc); take(f.cn, 3 * nc); take(f.cpos, 3 * nc); take(f.ct1, 3 * nc); take(f.ct2, 3 * nc);
    take(f.cD, nc); take(f.cpost, nc); take(f.cbd, nc); take(f.cmu, nc);
    const int base = o;
    take(f.fw, 3 * nb); take(f.fal, 3 * nb); take(f.fvp, 3 * nb); take(f.fap, 3 * nb);       // kinematics -> dynamics
    take(f.Fb, 3 * nb); take(f.Nb, 3 * nb); take(f.Iw, 9 * nb); take(f.Isub, 9 * nb); take(f.tw, 3 * std::max(h.ntw, 1));
    const int endA = o;
    o = base;                                                                                    // factor of M onwards
    take(f.Hc, nv * ld); take(f.J, nr * ld); take(f.aref, nr); take(f.D, nr); take(f.s, nr); take(f.pr, nr);
    take(f.x, nv); take(f.g, nv); take(f.dl, nv); take(f.Md, nv); take(f.xa, nv);
    o = std::max(o, endA);
    f.kap = f.cdD = f.cdpost = f.fox = f.fvx = base;     // VJP only: never touched by the forward kernel
    f.size = stagger(o + nq + nv, real_bytes) - (nq + nv);
    rlf.Yqr = o; rlf.Vr = o + nq;
  }
}

template <class R> size_t add_real(Arena& a, const std::vector<double>& v) {
  std::vector<R> t(v.size()); for (size_t i = 0; i < v.size(); ++i) t[i] = (R)v[i];
  return a.add(t.data(), t.size() * sizeof(R));
}
inline size_t add_int(Arena& a, const std::vector<int>& v) { return a.add(v.data(), v.size() * sizeof(int)); }

// lay the constants out in an arena; pointers are patched once the device address is known
template <class R> void build_dev(const HostModel& h, Arena& ar, ModelDev<R>& m, bool patch) {
  static thread_local std::vector<size_t> offs;
  if (!patch) {
    offs.clear();
    const std::vector<int>* iv[] = {&h.body_parent, &h.body_jnt, &h.level_ptr, &h.level_body, &h.jnt_type, &h.jnt_qadr, &h.jnt_vadr, &h.jnt_body,
                                    &h.dof_jnt, &h.dof_body, &h.dof_rot, &h.tw_ptr, &h.tw_body, &h.tw_dof, &h.tw_idx, &h.sub_ptr, &h.sub_body, &h.child_ptr, &h.child_idx,
                                    &h.mp_i, &h.mp_j, &h.mp_deep, &h.ct_kind, &h.ct_b1, &h.ct_b2, &h.ct_condim, &h.ct_pair, &h.act_type, &h.act_jnt};
    for (auto v : iv) offs.push_back(add_int(ar, *v));
    const std::vector<double>* rv[] = {&h.body_pos, &h.body_rot, &h.body_ipos, &h.body_irot, &h.body_iunit, &h.jnt_axis, &h.jnt_pos, &h.jnt_damping,
                                       &h.jnt_armature, &h.ct_p1, &h.ct_p2, &h.ct_rho1, &h.ct_rho2, &h.ct_n, &h.ct_t1, &h.ct_t2, &h.pair_invweight,
                                       &h.pair_solimp_cfd, &h.pair_cfd_beta, &h.act_gear, &h.act_kp, &h.act_kd, &h.p_default};
    for (auto v : rv) offs.push_back(add_real<R>(ar, *v));
    return;
  }
  m.arena = ar.dev; m.arena_bytes = (int)((ar.host.size() + 15) & ~size_t(15)); m.arena_smem = 0;
  m.nbody = h.nbody; m.njnt = h.njnt; m.nq = h.nq; m.nv = h.nv; m.nu = h.nu; m.npair = h.npair; m.nc = h.nc; m.np = h.np;
  m.nlevel = h.nlevel; m.ntw = h.ntw; m.nmp = h.nmp; m.nrmax = h.nrmax;
  m.npp = 0; for (int c = 0; c < h.nc; ++c) m.npp += h.ct_kind[c] == CK_POINT_POINT; m.newton_iters = h.newton_iters; m.ls_iters = h.ls_iters;
  m.p_fric = h.nbody; m.p_solref = h.nbody + h.npair; m.p_solimp = h.nbody + 3 * h.npair;
  for (int k = 0; k < 3; ++k) m.gravity[k] = (R)h.gravity[k];
  size_t k = 0;
  auto ip = [&]() { return reinterpret_cast<const int*>(ar.dev + offs[k++]); };
  auto rp = [&]() { return reinterpret_cast<const R*>(ar.dev + offs[k++]); };
  m.body_parent = ip(); m.body_jnt = ip(); m.level_ptr = ip(); m.level_body = ip(); m.jnt_type = ip(); m.jnt_qadr = ip(); m.jnt_vadr = ip(); m.jnt_body = ip();
  m.dof_jnt = ip(); m.dof_body = ip(); m.dof_rot = ip(); m.tw_ptr = ip(); m.tw_body = ip(); m.tw_dof = ip(); m.tw_idx = ip(); m.sub_ptr = ip(); m.sub_body = ip(); m.child_ptr = ip(); m.child_idx = ip();
  m.mp_i = ip(); m.mp_j = ip(); m.mp_deep = ip(); m.ct_kind = ip(); m.ct_b1 = ip(); m.ct_b2 = ip(); m.ct_condim = ip(); m.ct_pair = ip(); m.act_type = ip(); m.act_jnt = ip();
  m.body_pos = rp(); m.body_rot = rp(); m.body_ipos = rp(); m.body_irot = rp(); m.body_iunit = rp(); m.jnt_axis = rp(); m.jnt_pos = rp(); m.jnt_damping = rp();
  m.jnt_armature = rp(); m.ct_p1 = rp(); m.ct_p2 = rp(); m.ct_rho1 = rp(); m.ct_rho2 = rp(); m.ct_n = rp(); m.ct_t1 = rp(); m.ct_t2 = rp(); m.pair_invweight = rp();
  m.pair_solimp_cfd = rp(); m.pair_cfd_beta = rp(); m.act_gear = rp(); m.act_kp = rp(); m.act_kd = rp(); m.p_default = rp();
}

}  // namespace

// ---- the model object -------------------------------------------------------------------------------------
struct dmx_model {
  int precision, G, shape = 0, sm_count, max_smem, tape_stages = 1;
  int stride = 1;                  // checkpoint stride of the tape (dmx_model_set_checkpoint_stride)
  void* seg_scratch = nullptr;     // stride > 1: segment buffers of the reverse sweep, [resident groups][stride][seg record]
  int fwd_rk_global = 0;           // forward integrator arrays in global memory (like the reverse sweep's) instead of shared memory
  void* rk_scratch_fwd = nullptr;
  HostModel h;
  Arena arena;
  ModelDev<double> md; ModelDev<float> mf;
  WsLayout wl, wlf; RkLayout rl, rlf;      // full / forward-kernel workspaces (make_layouts)
  struct Cfg { int block = 0, occ = 0; size_t smem = 0; int arena = 0 /* constant arena in this kernel's shared memory */; } cf, cb, cx;   // forward, backward, field kernels
  void* rk_scratch = nullptr; size_t rk_scratch_bytes = 0;              // backward integrator arrays (global memory), sized at create
  cudaEvent_t bwd_done = nullptr;  // reverse sweeps of one model share rk_scratch: a sweep waits for the previous one
  int* queue = nullptr;            // [N_QUEUE] work-queue counters, one per call in flight (round robin)
  mutable std::atomic<unsigned> qnext{0};
  void* zero_u = nullptr;          // zeros: controls when ctrl == NULL, velocities at create
};

namespace {

size_t rsize(const dmx_model* m) { return m->precision == 64 ? sizeof(double) : sizeof(float); }

// shared memory of one lane group: kind 0 forward (integrator arrays + field workspace), 1 backward (field workspace
// only; the integrator / adjoint arrays live in global memory), 2 field kernels (both)
size_t group_bytes(const dmx_model* m, int kind) {
  size_t rk = kind == 0 ? (m->fwd_rk_global ? 0 : m->rl.size_fwd) : (kind == 1 ? 0 : m->rl.size_bwd);
  const WsLayout& wl = kind == 0 ? m->wlf : m->wl;
  return rk * sizeof(double) + (size_t)(wl.size + m->rl.rsize) * rsize(m) + (size_t)wl.isize * sizeof(int);
}
int groups_per_block(const dmx_model* m, int block) { return m->G == 1 ? block : block / m->G; }

enum { N_QUEUE = 64, N_FWD_SCRATCH = 1 };
int* next_queue(const dmx_model* m) { return m->queue + (m->qnext.fetch_add(1) % N_QUEUE); }

// backward integrator arrays of every lane group the largest reverse-sweep grid can hold: allocated once at create, so
// that dmx_rollout_backward only enqueues work
int alloc_scratch(dmx_model* m) {
  size_t groups = (size_t)m->cb.occ * m->sm_count * groups_per_block(m, m->cb.block);
  if (m->G == 1) groups = (groups + 31) / 32 * 32;
  m->rk_scratch_bytes = std::max<size_t>(groups * (size_t)m->rl.size_adj * sizeof(double), 256);      // size_adj >= size_bwd
  CUDA_OK(cudaMalloc(&m->rk_scratch, m->rk_scratch_bytes));
  CUDA_OK(cudaEventCreateWithFlags(&m->bwd_done, cudaEventDisableTiming));
  if (m->fwd_rk_global) {
    size_t gf = (size_t)m->cf.occ * m->sm_count * groups_per_block(m, m->cf.block);
    if (m->G == 1) gf = (gf + 31) / 32 * 32;
    CUDA_OK(cudaMalloc(&m->rk_scratch_fwd, std::max<size_t>(gf * (size_t)m->rl.size_fwd * sizeof(double), 256) * N_FWD_SCRATCH));
  }
  return 0;
}

// ---- tape geometry ---------------------------------------------------------------------------------------------
size_t align_up(size_t b, size_t a) { return (b + a - 1) / a * a; }
size_t record_bytes(const dmx_model* m);
size_t tape_header_bytes(int nenv) { return 256 + align_up((size_t)nenv * 2 * sizeof(int), 256); }
template <class R> void tape_geometry(const dmx_model* m, TapeView<R>& tp) {
  const int per16 = 16 / (int)sizeof(R), per8 = 8 / (int)sizeof(R), nx = m->h.nq + m->h.nv;
  tp.o_th = (nx + per16 - 1) / per16 * per16;
  const int o = tp.o_th + 2 * per8;
  const int rec_plain = (o + per16 - 1) / per16 * per16, rec_rates = (o + 6 * m->h.nv + per16 - 1) / per16 * per16;
  tp.stride = m->stride;
  const int rec_k1 = (o + m->h.nv + per16 - 1) / per16 * per16;
  const bool rates = m->tape_stages && m->stride == 1;        // a strided tape keeps checkpoints with the first-stage rate only (the
  tp.o_A = (rates || m->stride > 1) ? o : -1;                 // FSAL value the forward pass used); the segment buffer holds all six
  tp.rec = rates ? rec_rates : (m->stride > 1 ? rec_k1 : rec_plain);
  tp.seg_rec = rec_rates; tp.seg_oA = o;
}
// bytes of a tape that holds `steps` accepted steps in total for nenv environments (without the header)
size_t tape_payload_bytes(const dmx_model* m, int nenv, long long steps) {
  const size_t rb = record_bytes(m);
  if (m->stride == 1) return (size_t)steps * rb;
  return align_up((size_t)steps * sizeof(double), 16) + ((size_t)(steps / m->stride) + (size_t)nenv) * rb;
}
size_t record_bytes(const dmx_model* m) {
  if (m->precision == 64) { TapeView<double> t; tape_geometry(m, t); return (size_t)t.rec * 8; }
  TapeView<float> t; tape_geometry(m, t); return (size_t)t.rec * 4;
}
template <class R> int bind_tape(const dmx_model* m, int nenv, void* tape, size_t tape_bytes, const void* plan, TapeView<R>& tp, PlanView& pl) {
  tape_geometry(m, tp);
  std::memset(&pl, 0, sizeof(pl));
  if (plan) {
    const unsigned char* b = (const unsigned char*)plan;
    size_t a4 = align_up((size_t)nenv * sizeof(int), 256);
    pl.order = (const int*)(b + 256); pl.cap = (const int*)(b + 256 + a4); pl.offset = (const long long*)(b + 256 + 2 * a4);
  }
  tp.meta = nullptr; tp.hdr = nullptr; tp.data = nullptr; tp.sched = nullptr; tp.capacity = 0; tp.uniform_cap = 0;
  if (!tape) return 0;
  size_t hdr = tape_header_bytes(nenv), rb = (size_t)tp.rec * sizeof(R);
  if (tape_bytes < hdr + tape_payload_bytes(m, nenv, plan ? 1 : nenv)) return fail("tape too small");
  if (((size_t)tape & 15) != 0) return fail("tape must be 16-byte aligned");
  tp.meta = (int*)tape; tp.hdr = (int*)((unsigned char*)tape + 256);
  const size_t avail = tape_bytes - hdr;
  if (m->stride == 1) {
    tp.sched = nullptr; tp.data = (R*)((unsigned char*)tape + hdr);
    tp.capacity = (long long)(avail / rb);
  } else {                        // [schedule: capacity doubles | checkpoints: capacity / stride + nenv records]
    long long cap = (long long)(((avail - (size_t)nenv * rb) * (size_t)m->stride) / (8 * (size_t)m->stride + rb));
    while (cap > 0 && tape_payload_bytes(m, nenv, cap) > avail) --cap;
    while (tape_payload_bytes(m, nenv, cap + 1) <= avail) ++cap;          // the estimate floors steps / stride: it can be a few steps short
    tp.capacity = cap;
    tp.sched = (double*)((unsigned char*)tape + hdr);
    tp.data = (R*)((unsigned char*)tape + hdr + align_up((size_t)cap * sizeof(double), 16));
  }
  tp.uniform_cap = (int)std::min<long long>(tp.capacity / nenv, (long long)1 << 30);
  return 0;
}

template <class R> const ModelDev<R>& dev_of(const dmx_model* m);
template <> const ModelDev<double>& dev_of<double>(const dmx_model* m) { return m->md; }
template <> const ModelDev<float>& dev_of<float>(const dmx_model* m) { return m->mf; }

SolverOpts opts_of(const dmx_solver_opts* o) {
  SolverOpts s; s.tableau = o->tableau; s.rtol = o->rtol; s.atol = o->atol; s.h0 = o->h0; s.pcoeff = o->pcoeff; s.icoeff = o->icoeff;
  s.safety = o->safety; s.fac_min = o->fac_min; s.fac_max = o->fac_max; s.max_steps = o->max_steps;
  return s;
}

template <class R>
int create_typed(dmx_model* m) {
  HostModel& h = m->h;
  ModelDev<R> dev;
  build_dev<R>(h, m->arena, dev, false);
  m->arena.host.resize((m->arena.host.size() + 15) & ~size_t(15));
  CUDA_OK(cudaMalloc(&m->arena.dev, m->arena.host.size()));
  CUDA_OK(cudaMemcpy(m->arena.dev, m->arena.host.data(), m->arena.host.size(), cudaMemcpyHostToDevice));
  build_dev<R>(h, m->arena, dev, true);
  Launchers<R> L = launchers_for<R>(m->G, m->shape);
  // A^: body inverse weights at qpos0 on the device (same kinematics / mass-matrix / Cholesky code as the rollouts)
  std::vector<R> q0(h.nq); for (int i = 0; i < h.nq; ++i) q0[i] = (R)h.qpos0[i];
  R *dq0 = nullptr, *dw = nullptr;
  CUDA_OK(cudaMalloc(&dq0, sizeof(R) * h.nq)); CUDA_OK(cudaMalloc(&dw, sizeof(R) * h.nbody));
  CUDA_OK(cudaMemcpy(dq0, q0.data(), sizeof(R) * h.nq, cudaMemcpyHostToDevice));
  LaunchCfg c; c.block = 32; c.grid = 1; c.smem = groups_per_block(m, 32) * group_bytes(m, 2);
  CUDA_OK(L.invweight(dev, dq0, (const R*)m->zero_u, dw, m->wl, m->rl, c, 0));
  CUDA_OK(cudaDeviceSynchronize());
  std::vector<R> bw(h.nbody);
  CUDA_OK(cudaMemcpy(bw.data(), dw, sizeof(R) * h.nbody, cudaMemcpyDeviceToHost));
  cudaFree(dq0); cudaFree(dw);
  for (int b = 1; b < h.nbody; ++b) if (!std::isfinite((double)bw[b])) return fail("mass matrix at qpos0 is not positive definite");
  std::vector<R> pw(h.npair);
  for (int i = 0; i < h.npair; ++i) { h.pair_invweight[i] = (double)bw[h.pair_body1[i]] + (double)bw[h.pair_body2[i]]; pw[i] = (R)h.pair_invweight[i]; }
  if (h.npair) CUDA_OK(cudaMemcpy(const_cast<R*>(dev.pair_invweight), pw.data(), sizeof(R) * h.npair, cudaMemcpyHostToDevice));
  if (sizeof(R) == 8) std::memcpy(&m->md, &dev, sizeof(dev)); else std::memcpy(&m->mf, &dev, sizeof(dev));
  // block size per kernel: the largest CTA (its warps share the fetched instruction lines; the kernels are fetch-bound,
  // measured 1.2x forward C2 and 1.4x reverse sweep C3 from 64/128 -> 128/256 threads at equal residency) unless a
  // smaller one keeps >= 1.3x as many lane groups resident on an SM.  The selection runs twice: with
  // the constant arena appended to each CTA's dynamic shared memory (ModelDev::arena_smem) and without; the arena goes
  // to shared memory only if no kernel loses resident groups to it (DMX_ARENA_SMEM=0 keeps it in global memory).
  const char* eb = std::getenv("DMX_BWD_BLOCK");
  const char* ef = std::getenv("DMX_FWD_BLOCK");
  typedef dmx_model::Cfg Cfg;
  auto select = [&](size_t ab, Cfg& cf, Cfg& cb, Cfg& cx) -> int {
    const int blocks[4] = {256, 128, 64, 32};
    cf = Cfg(); cb = Cfg(); cx = Cfg();
    for (int bi = 0; bi < 4; ++bi) {
      int blk = blocks[bi], g = groups_per_block(m, blk);
      auto pad = [&](size_t b) { return ((b + 15) & ~size_t(15)) + ab; };
      size_t sf = pad(g * group_bytes(m, 0)), sb = pad(g * group_bytes(m, 1)), sx = pad(g * group_bytes(m, 2));
      int of = 0, ob = 0, ox = 0;
      size_t lim = (size_t)m->max_smem - 2048;     // room for the static shared constants
      if (blk > 128) { int b2 = 128, g2 = groups_per_block(m, b2); int t0, t2;   // only the backward kernel is compiled for 256 threads
        CUDA_OK(L.occupancy(b2, std::min(pad(g2 * group_bytes(m, 0)), lim), std::min(sb, lim), std::min(pad(g2 * group_bytes(m, 2)), lim), &t0, &ob, &t2));
        (void)t0; (void)t2; ob = sb <= lim ? 1 : 0; }
      else CUDA_OK(L.occupancy(blk, std::min(sf, lim), std::min(sb, lim), std::min(sx, lim), &of, &ob, &ox));
      auto better = [&](int occ_new, const Cfg& cur) { return cur.occ == 0 ? occ_new > 0 : 10 * occ_new * g >= 13 * cur.occ * groups_per_block(m, cur.block); };
      if (ef ? (std::atoi(ef) == blk && blk <= 128 && sf <= lim && of > 0) : (blk <= 128 && sf <= lim && better(of, cf))) { cf.block = blk; cf.occ = of; cf.smem = sf; }
      if (eb ? (std::atoi(eb) == blk && sb <= lim && ob > 0) : (sb <= lim && better(ob, cb))) { cb.block = blk; cb.occ = ob; cb.smem = sb; }
      if (blk <= 128 && sx <= lim && better(ox, cx)) { cx.block = blk; cx.occ = ox; cx.smem = sx; }
    }
    return 0;
  };
  if (int rc = select(0, m->cf, m->cb, m->cx)) return rc;
  {
    const char* ea = std::getenv("DMX_ARENA_SMEM");
    Cfg af, abk, ax;
    if (!(ea && std::atoi(ea) == 0)) {
      if (int rc = select(m->arena.host.size(), af, abk, ax)) return rc;
      auto res = [&](const Cfg& c) { return c.occ * groups_per_block(m, std::max(c.block, 1)); };
      // per kernel: the arena goes to shared memory where it costs no resident lane group
      if (af.occ >= 1 && res(af) >= res(m->cf)) { m->cf = af; m->cf.arena = 1; }
      if (abk.occ >= 1 && res(abk) >= res(m->cb)) { m->cb = abk; m->cb.arena = 1; }
      if (ax.occ >= 1 && res(ax) >= res(m->cx)) { m->cx = ax; m->cx.arena = 1; }
    }
  }
  if (m->cf.occ < 1 || m->cb.occ < 1 || m->cx.occ < 1) return fail("model too large for the per-environment shared-memory workspace (try DMX_LANES=32)");
  if (std::getenv("DMX_VERBOSE"))
    std::fprintf(stderr, "dmx: arena %zu B, in smem fwd/bwd/field %d/%d/%d | lanes %d | fwd block %d x occ %d smem %zu | bwd block %d x occ %d smem %zu | field block %d x occ %d smem %zu | group bytes f/b %zu/%zu\n",
                 m->arena.host.size(), m->cf.arena, m->cb.arena, m->cx.arena, m->G, m->cf.block, m->cf.occ, m->cf.smem, m->cb.block, m->cb.occ, m->cb.smem, m->cx.block, m->cx.occ, m->cx.smem, group_bytes(m, 0), group_bytes(m, 1));
  // the occupancy queries above left the largest attribute set; restore the chosen sizes
  int d0, d1, d2;
  CUDA_OK(L.occupancy(m->cf.block, m->cf.smem, m->cb.smem, m->cx.smem, &d0, &d1, &d2));
  return 0;
}

int pick_lanes(const HostModel& h) {
  const char* e = std::getenv("DMX_LANES");
  if (e) { int g = std::atoi(e); if (g == 1 || g == 8 || g == 16 || g == 32) return g; }
  if (h.nv <= 2) return 1;
  if (h.nv <= 8 && h.nc <= 4) return 8;
  if (h.nv <= 8) return 16;
  return 32;
}

// A batch that fills fewer CTAs than the SMs can hold would leave SMs idle, or with one CTA where others have two, while
// the kernel lasts as long as its busiest SM (C2 at 4096 environments: reverse sweep 128 CTAs of 32 lane groups on 148
// SMs; forward 256 CTAs of 16 on 148 SMs).  Then launch one CTA per SM, of ceil(nenv / SMs) lane groups in whole warps, if
// such a CTA fits (threads, shared memory); else one per resident slot.  Same resident groups, spread evenly, and every
// CTA full (its warps share the fetched instructions).  DMX_BALANCE=0: off.
void balance_block(const dmx_model* m, int nenv, const dmx_model::Cfg& cfg, size_t gbytes, int max_block, LaunchCfg& c) {
  static const bool on = [] { const char* e = std::getenv("DMX_BALANCE"); return !(e && std::atoi(e) == 0); }();
  const int slots = cfg.occ * m->sm_count, gpb = groups_per_block(m, cfg.block);
  if (!on || nenv <= 0 || (nenv + gpb - 1) / gpb >= slots) return;
  auto threads_for = [&](int groups) { return std::max(32, ((m->G == 1 ? groups : groups * m->G) + 31) / 32 * 32); };
  auto smem_for = [&](int blk) { return ((groups_per_block(m, blk) * gbytes + 15) & ~size_t(15)) + (cfg.arena ? m->arena.host.size() : 0); };
  int blk = threads_for((nenv + m->sm_count - 1) / m->sm_count);               // one CTA per SM
  if (blk > max_block || smem_for(blk) > (size_t)m->max_smem - 2048) {
    blk = threads_for((nenv + slots - 1) / slots);                             // one CTA per resident slot
    if (blk >= cfg.block) return;
  }
  const int g = groups_per_block(m, blk);
  c.block = blk; c.grid = (nenv + g - 1) / g; c.smem = smem_for(blk);
}

// A batch between half of and all the lane groups one 256-thread CTA per SM can hold runs as a single wave without the
// queue: k CTAs half filled with the head of the launch order, the others full (next_env in dmx_rk.cuh).  Returns k, or -1
// when the launch keeps the queue (batch too small or too large, CTA does not fit, DMX_HETERO=0 / DMX_HETERO_FWD=0 /
// DMX_HETERO_BWD=0).
int single_wave(const dmx_model* m, int nenv, const dmx_model::Cfg& cfg, size_t gbytes, bool forward, LaunchCfg& c) {
  static const int on = [] { const char* e = std::getenv("DMX_HETERO"); return e ? std::atoi(e) : 1; }();
  static const int on_f = [] { const char* e = std::getenv("DMX_HETERO_FWD"); return e ? std::atoi(e) : 1; }();
  static const int on_b = [] { const char* e = std::getenv("DMX_HETERO_BWD"); return e ? std::atoi(e) : 1; }();
  if (!on || (forward ? !on_f : !on_b)) return -1;
  if (forward && (m->G > 8 || m->fwd_rk_global)) return -1;          // the forward kernel admits 256 threads with 1 or 8 lanes only
  const int blk = 256, g = groups_per_block(m, blk), half = g / 2, cap = m->sm_count * g;
  if (half < 1 || nenv <= cap / 2 || nenv > cap) return -1;
  const size_t smem = ((g * gbytes + 15) & ~size_t(15)) + (cfg.arena ? m->arena.host.size() : 0);
  if (smem > (size_t)m->max_smem - 2048) return -1;
  const int k = std::min(m->sm_count, (cap - nenv) / half);
  c.block = blk; c.grid = m->sm_count; c.smem = smem;
  return k;
}

template <class R>
int rollout_typed(const dmx_model* m, int nenv, const void* x0, const void* ctrl, int nknot, double knot_dt, const void* params, double horizon,
                  const dmx_solver_opts* opts, const double* h_replay, int n_replay, void* xT, const dmx_stats* st, void* tape, size_t tape_bytes,
                  const void* plan, cudaStream_t s) {
  RolloutArgs<R> a; std::memset(&a, 0, sizeof(a));
  a.nenv = nenv; a.nknot = nknot; a.n_replay = h_replay ? n_replay : 0; a.want_tape = tape != nullptr;
  if (bind_tape<R>(m, nenv, tape, tape_bytes, plan, a.tp, a.pl)) return -1;
  a.x0 = (const R*)x0; a.ctrl = (const R*)ctrl; a.params = (const R*)params; a.zero_u = (const R*)m->zero_u; a.h_replay = h_replay;
  a.knot_dt = knot_dt; a.horizon = horizon; a.so = opts_of(opts); a.xT = (R*)xT;
  if (st) { a.n_accept = st->n_accept; a.n_reject = st->n_reject; a.n_feval = st->n_feval; a.n_unconv = st->n_newton_unconverged; a.status = st->status;
            a.h_min = st->h_min; a.h_max = st->h_max; a.t_end = st->t_end; a.work = st->work; }
  a.queue = next_queue(m); a.wl = m->wlf; a.rl = m->rlf; a.rk_scratch = (double*)m->rk_scratch_fwd;
  { const char* e = std::getenv("DMX_LOCKSTEP"); a.lockstep = e ? std::atoi(e) : (m->G >= 16 && m->cf.block >= 64 ? 0x1f : 0); }   // phases in lockstep: +8 % on C3, nothing on C2 (8 lanes)
  CUDA_OK(cudaMemsetAsync(a.queue, 0, sizeof(int), s));
  LaunchCfg c; c.block = m->cf.block; c.smem = m->cf.smem;
  int gpb = groups_per_block(m, c.block);
  c.grid = std::max(1, std::min(m->cf.occ * m->sm_count, (nenv + gpb - 1) / gpb));
  { static const bool fb = [] { const char* e = std::getenv("DMX_BALANCE_FWD"); return e && std::atoi(e) != 0; }();   // measured on C2: 48 -> 51 ms, off
    if (fb && !m->fwd_rk_global) balance_block(m, nenv, m->cf, group_bytes(m, 0), 128, c); }
  a.n_light = single_wave(m, nenv, m->cf, group_bytes(m, 0), true, c);
  ModelDev<R> md = dev_of<R>(m); md.arena_smem = m->cf.arena;
  CUDA_OK(launchers_for<R>(m->G, m->shape).rollout(md, a, c, s));
  return 0;
}

template <class R>
int backward_typed(dmx_model* m, int nenv, const void* ctrl, int nknot, const void* params, const dmx_solver_opts* opts, const void* xT,
                   const void* dLdxT, int cfd_on, void* dLdx0, void* dLdctrl, void* dLdparams, const dmx_stats* st, const void* tape,
                   size_t tape_bytes, const void* plan, cudaStream_t s, const dmx_solver_opts* adj = nullptr, int* adj_info = nullptr,
                   const double* adj_replay = nullptr, int n_adj_replay = 0) {
  AdjointArgs<R> aa; std::memset(&aa, 0, sizeof(aa));
  BackwardArgs<R>& a = aa.b;
  if (!tape) return fail("tape missing");
  if (bind_tape<R>(m, nenv, const_cast<void*>(tape), tape_bytes, plan, a.tp, a.pl)) return -1;
  a.nenv = nenv; a.nknot = nknot; a.want_p = dLdparams != nullptr; a.cfd = cfd_on; a.tape_stages = m->tape_stages;
  { const char* e = std::getenv("DMX_DBG"); a.dbg = e ? std::atoi(e) : 0; }   // timing experiments only (results invalid when set, except bit 8: VJP rebuilds H instead of reusing the Newton factor)
  a.ctrl = (const R*)ctrl; a.params = (const R*)params; a.zero_u = (const R*)m->zero_u; a.xT = (const R*)xT; a.dLdxT = (const R*)dLdxT;
  a.status = st ? st->status : nullptr; a.n_unconv = st ? st->n_newton_unconverged_bwd : nullptr; a.work = st ? st->work : nullptr;
  a.so = opts_of(opts); a.dLdx0 = (R*)dLdx0; a.dLdctrl = (R*)dLdctrl; a.dLdparams = (R*)dLdparams;
  { const char* e = std::getenv("DMX_LOCKSTEP_BWD"); a.lockstep = e ? std::atoi(e) : 0x21; }   // backward: fetch-bound, CTA in lockstep (off: 3.4x slower on C2); a barrier before the F evaluation and one before the VJP phases of a stage do as well as one before each of the nine phases (-1..3 %)
  a.queue = next_queue(m); a.wl = m->wl; a.rl = m->rl;
  LaunchCfg c; c.block = m->cb.block; c.smem = m->cb.smem;
  int gpb = groups_per_block(m, c.block);
  c.grid = std::max(1, std::min(m->cb.occ * m->sm_count, (nenv + gpb - 1) / gpb));
  balance_block(m, nenv, m->cb, group_bytes(m, 1), 256, c);
  a.n_light = adj ? -1 : single_wave(m, nenv, m->cb, group_bytes(m, 1), false, c);
  a.rk_scratch = (double*)m->rk_scratch;
  CUDA_OK(cudaStreamWaitEvent(s, m->bwd_done, 0));          // the previous reverse sweep of this model (any stream) owns rk_scratch until it ends
  CUDA_OK(cudaMemsetAsync(a.queue, 0, sizeof(int), s));
  if (dLdctrl && nknot > 0 && m->h.nu > 0) CUDA_OK(cudaMemsetAsync(dLdctrl, 0, (size_t)nenv * nknot * m->h.nu * sizeof(R), s));
  ModelDev<R> md = dev_of<R>(m); md.arena_smem = m->cb.arena;
  if (adj && m->stride > 1) return fail("the continuous adjoint needs a tape with checkpoint stride 1");
  if (adj) {                       // optimize-then-discretize: same arguments plus the options of the backward solve
    aa.sa = opts_of(adj); aa.info = adj_info; aa.replay = adj_replay; aa.n_replay = adj_replay ? n_adj_replay : 0;
    CUDA_OK(launchers_for<R>(m->G, m->shape).adjoint(md, aa, c, s));
  } else if (m->stride > 1) {
    a.seg_scratch = (R*)m->seg_scratch;
    CUDA_OK(launchers_for<R>(m->G, m->shape).backward_ckpt(md, a, c, s));
  } else CUDA_OK(launchers_for<R>(m->G, m->shape).backward(md, a, c, s));
  CUDA_OK(cudaEventRecord(m->bwd_done, s));
  return 0;
}

template <class R>
int field_typed(dmx_model* m, int n, const void* x, const void* u, const void* params, const void* kappa, int cfd, void* acc, int* nrow,
                void* qbar, void* vbar, void* ubar, void* pbar, cudaStream_t s) {
  FieldArgs<R> a; std::memset(&a, 0, sizeof(a));
  a.n = n; a.cfd = cfd; a.want_p = pbar != nullptr; a.x = (const R*)x; a.u = (const R*)u; a.params = (const R*)params; a.zero_u = (const R*)m->zero_u;
  a.kappa = (const R*)kappa; a.acc = (R*)acc; a.nrow = nrow; a.qbar = (R*)qbar; a.vbar = (R*)vbar; a.ubar = (R*)ubar; a.pbar = (R*)pbar;
  a.wl = m->wl; a.rl = m->rl;
  LaunchCfg c; c.block = m->cx.block; c.smem = m->cx.smem;
  int gpb = groups_per_block(m, c.block);
  c.grid = std::max(1, std::min(m->cx.occ * m->sm_count, (n + gpb - 1) / gpb));
  ModelDev<R> md = dev_of<R>(m); md.arena_smem = m->cx.arena;
  CUDA_OK(launchers_for<R>(m->G, m->shape).field(md, a, c, s));
  return 0;
}

// Optimiser step of the paper's applications (PAPER.md:167 "Adam ... learning rate of 0.01", "gradient clipping"; :515 Adam
// with b1 = 0.5, b2 = 0.9, eps = 1e-6): a warp per row; the row's gradient is scaled to norm <= clip, then the bias-corrected
// Adam update (Kingma & Ba 2015).  Arithmetic in double for both storage types.
template <class R>
__global__ void adam_clip_kernel(int nrow, int len, R* x, const R* g, R* m1, R* m2, const unsigned char* active, double lr, double b1, double b2,
                                 double eps, double clip, double c1, double c2) {
  const int row = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (row >= nrow || (active && !active[row])) return;
  const size_t o = (size_t)row * len;
  double scale = 1.0;
  if (clip > 0) {
    double ss = 0;
    for (int j = lane; j < len; j += 32) { double gj = (double)g[o + j]; ss += gj * gj; }
    for (int d = 16; d > 0; d >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, d);
    const double nrm = sqrt(ss);
    if (nrm > clip) scale = clip / nrm;
  }
  for (int j = lane; j < len; j += 32) {
    const double gj = scale * (double)g[o + j];
    const double a = b1 * (double)m1[o + j] + (1.0 - b1) * gj, b = b2 * (double)m2[o + j] + (1.0 - b2) * gj * gj;
    m1[o + j] = (R)a; m2[o + j] = (R)b;
    x[o + j] = (R)((double)x[o + j] - lr * (a / c1) / (sqrt(b / c2) + eps));
  }
}

// FMA-chain microbenchmark: 8 independent chains per thread
template <class T> __global__ void fma_chain_kernel(T* out, int iters, T a, T b) {
  T x0 = T(threadIdx.x), x1 = x0 + T(1), x2 = x0 + T(2), x3 = x0 + T(3), x4 = x0 + T(4), x5 = x0 + T(5), x6 = x0 + T(6), x7 = x0 + T(7);
  for (int i = 0; i < iters; ++i) {
    x0 = x0 * a + b; x1 = x1 * a + b; x2 = x2 * a + b; x3 = x3 * a + b; x4 = x4 * a + b; x5 = x5 * a + b; x6 = x6 * a + b; x7 = x7 * a + b;
  }
  out[blockIdx.x * blockDim.x + threadIdx.x] = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
}
template <class T> int fma_peak_typed(int iters, double* flops, double* ms_out) {
  int dev = 0, sms = 0; CUDA_OK(cudaGetDevice(&dev)); CUDA_OK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  int block = 256, grid = sms * 8;
  T* out = nullptr; CUDA_OK(cudaMalloc(&out, sizeof(T) * block * grid));
  cudaEvent_t e0, e1; CUDA_OK(cudaEventCreate(&e0)); CUDA_OK(cudaEventCreate(&e1));
  fma_chain_kernel<T><<<grid, block>>>(out, iters / 4, T(0.999), T(0.001));
  float best = 1e30f;
  for (int r = 0; r < 3; ++r) {
    CUDA_OK(cudaEventRecord(e0));
    fma_chain_kernel<T><<<grid, block>>>(out, iters, T(0.999), T(0.001));
    CUDA_OK(cudaEventRecord(e1)); CUDA_OK(cudaEventSynchronize(e1));
    float ms; CUDA_OK(cudaEventElapsedTime(&ms, e0, e1)); best = std::min(best, ms);
  }
  CUDA_OK(cudaGetLastError());
  cudaFree(out); cudaEventDestroy(e0); cudaEventDestroy(e1);
  *flops = 2.0 * 8.0 * (double)iters * block * grid / (best * 1e-3); *ms_out = best;
  return 0;
}

// Plan of a launch from the accepted-step counts of a previous pass: cap(e) = n(e) + n(e) margin_pct / 100 + pad,
// offset = exclusive prefix sum of cap in environment order, order = environments by descending n (ties: lower index
// first).  Rank and prefix by direct counting: nenv^2 integer operations, deterministic, no scratch.
__global__ void plan_kernel(int nenv, const int* __restrict__ n_acc, int margin_pct, int pad, int* order, int* cap, long long* offset, long long* total) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= nenv) return;
  const int ne = n_acc[e];
  auto capof = [=](int n) { return (int)(n + (long long)n * margin_pct / 100 + pad); };
  int rank = 0; long long off = 0;
  for (int j = 0; j < nenv; ++j) {
    const int nj = n_acc[j];
    rank += (nj > ne) || (nj == ne && j < e);
    if (j < e) off += capof(nj);
  }
  order[rank] = e; cap[e] = capof(ne); offset[e] = off;
  if (e == nenv - 1) *total = off + capof(ne);
}

}  // namespace

static int noalloc_setup(int dev);   // defined at the end of this file, next to the static scratch array

// ---- C-ABI ------------------------------------------------------------------------------------------------
extern "C" {

const char* dmx_last_error(void) { return g_err; }

int dmx_model_create(const dmx_model_desc* desc, int precision, dmx_model** out) {
  if (!desc || !out) return fail("null argument");
  if (precision != 64 && precision != 32) return fail("precision must be 64 or 32");
  dmx_model* m = new dmx_model();
  try { flatten(desc, m->h); } catch (std::exception& e) { fail("model: %s", e.what()); delete m; return -1; }
  m->precision = precision;
  m->G = pick_lanes(m->h);
  m->shape = pick_shape(precision, m->G, m->h.nv, m->h.nc, m->h.nrmax);
  { const char* e = std::getenv("DMX_FWD_RK_GLOBAL"); m->fwd_rk_global = e ? std::atoi(e) : 0; }
  make_layouts(m->h, m->G, precision / 8, m->shape ? shape_ld(m->shape, m->h.nv) : 0, m->wl, m->wlf, m->rl, m->rlf);
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&m->sm_count, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
    fail("no CUDA device: the dmx library has no CPU fallback"); delete m; return -1;
  }
  m->max_smem = 0; cudaDeviceGetAttribute(&m->max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  size_t zbytes = sizeof(double) * (size_t)std::max(std::max(m->h.nu, m->h.nv), 1);
  if (cudaMalloc(&m->zero_u, zbytes) != cudaSuccess || cudaMemset(m->zero_u, 0, zbytes) != cudaSuccess ||
      cudaMalloc(&m->queue, N_QUEUE * sizeof(int)) != cudaSuccess) { fail("cudaMalloc failed"); dmx_model_destroy(m); return -1; }
  int rc = precision == 64 ? create_typed<double>(m) : create_typed<float>(m);
  if (!rc) rc = alloc_scratch(m);
  if (!rc) rc = noalloc_setup(dev);          // device address of the static scratch of dmx_rollout_backward_noalloc
  if (rc) { dmx_model_destroy(m); return -1; }
  *out = m;
  return 0;
}

void dmx_model_destroy(dmx_model* m) {
  if (!m) return;
  if (m->arena.dev) cudaFree(m->arena.dev);
  if (m->queue) cudaFree(m->queue);
  if (m->zero_u) cudaFree(m->zero_u);
  if (m->rk_scratch) cudaFree(m->rk_scratch);
  if (m->rk_scratch_fwd) cudaFree(m->rk_scratch_fwd);
  if (m->seg_scratch) cudaFree(m->seg_scratch);
  if (m->bwd_done) cudaEventDestroy(m->bwd_done);
  delete m;
}

int dmx_model_set_tape_stages(dmx_model* m, int on) {
  if (!m) return fail("null model");
  m->tape_stages = on ? 1 : 0;
  return 0;
}
int dmx_model_set_checkpoint_stride(dmx_model* m, int k) {
  if (!m) return fail("null model");
  if (k < 1 || k > 65536) return fail("checkpoint stride must be in [1, 65536]");
  CUDA_OK(cudaDeviceSynchronize());                       // set-up call: no sweep may still use the old buffers
  if (m->seg_scratch) { cudaFree(m->seg_scratch); m->seg_scratch = nullptr; }
  m->stride = k;
  if (k > 1) {
    size_t groups = (size_t)m->cb.occ * m->sm_count * groups_per_block(m, m->cb.block), seg_rec;
    if (m->precision == 64) { TapeView<double> t; tape_geometry(m, t); seg_rec = (size_t)t.seg_rec * 8; }
    else { TapeView<float> t; tape_geometry(m, t); seg_rec = (size_t)t.seg_rec * 4; }
    CUDA_OK(cudaMalloc(&m->seg_scratch, groups * (size_t)k * seg_rec));
  }
  return 0;
}
int dmx_model_np(const dmx_model* m) { return m ? m->h.np : -1; }
int dmx_model_nc(const dmx_model* m) { return m ? m->h.nc : -1; }
int dmx_model_lanes(const dmx_model* m) { return m ? m->G : -1; }
int dmx_model_default_params(const dmx_model* m, double* p_host) {
  if (!m || !p_host) return fail("null argument");
  for (int i = 0; i < m->h.np; ++i) p_host[i] = m->h.p_default[i];
  return 0;
}

size_t dmx_tape_bytes(const dmx_model* m, int nenv, int tape_steps) {
  if (!m || nenv <= 0 || tape_steps <= 0) return 0;
  return tape_header_bytes(nenv) + tape_payload_bytes(m, nenv, (long long)nenv * tape_steps);
}
size_t dmx_tape_bytes_records(const dmx_model* m, int nenv, long long total_records) {
  if (!m || nenv <= 0 || total_records <= 0) return 0;
  return tape_header_bytes(nenv) + tape_payload_bytes(m, nenv, total_records);
}
size_t dmx_plan_bytes(int nenv) {
  if (nenv <= 0) return 0;
  return 256 + 2 * align_up((size_t)nenv * sizeof(int), 256) + align_up((size_t)nenv * sizeof(long long), 256);
}
int dmx_tape_plan(const dmx_model* m, int nenv, const int* n_accept, int margin_pct, int pad, void* plan, size_t plan_bytes, void* cuda_stream) {
  if (!m || nenv <= 0 || !n_accept || !plan) return fail("null argument");
  if (margin_pct < 0 || pad < 0) return fail("margin_pct and pad must be non-negative");
  if (plan_bytes < dmx_plan_bytes(nenv)) return fail("plan buffer too small");
  unsigned char* b = (unsigned char*)plan;
  size_t a4 = align_up((size_t)nenv * sizeof(int), 256);
  plan_kernel<<<(nenv + 127) / 128, 128, 0, (cudaStream_t)cuda_stream>>>(nenv, n_accept, margin_pct, pad, (int*)(b + 256), (int*)(b + 256 + a4),
                                                                          (long long*)(b + 256 + 2 * a4), (long long*)b);
  CUDA_OK(cudaGetLastError());
  return 0;
}

static int check_common(const dmx_model* m, int nenv, const void* x0, const dmx_solver_opts* o, double horizon) {
  if (!m) return fail("null model");
  if (nenv <= 0) return fail("nenv must be positive");
  if (!x0 || !o) return fail("null argument");
  if (o->tableau != DMX_DOPRI5 && o->tableau != DMX_TSIT5) return fail("unknown tableau");
  if (!(o->rtol >= 0) || !(o->atol >= 0) || !(o->rtol + o->atol > 0) || !(o->h0 > 0) || !(horizon >= 0)) return fail("bad tolerances / h0 / horizon");
  return 0;
}

int dmx_rollout(const dmx_model* m, int nenv, const void* x0, const void* ctrl, int nknot, double knot_dt, const void* params, double horizon,
                const dmx_solver_opts* opts, const double* h_replay, int n_replay, void* xT, const dmx_stats* stats, void* tape, size_t tape_bytes,
                const void* plan, void* cuda_stream) {
  if (check_common(m, nenv, x0, opts, horizon)) return -1;
  if (!xT) return fail("null xT");
  if (ctrl && m->h.nu > 0 && (nknot <= 0 || !(knot_dt > 0))) return fail("ctrl given but nknot / knot_dt invalid");
  cudaStream_t s = (cudaStream_t)cuda_stream;
  return m->precision == 64 ? rollout_typed<double>(m, nenv, x0, ctrl, nknot, knot_dt, params, horizon, opts, h_replay, n_replay, xT, stats, tape, tape_bytes, plan, s)
                            : rollout_typed<float>(m, nenv, x0, ctrl, nknot, knot_dt, params, horizon, opts, h_replay, n_replay, xT, stats, tape, tape_bytes, plan, s);
}

int dmx_rollout_backward(const dmx_model* m, int nenv, const void* ctrl, int nknot, const void* params, const dmx_solver_opts* opts, const void* xT,
                         const void* dLdxT, int cfd_on, void* dLdx0, void* dLdctrl, void* dLdparams, const dmx_stats* stats, const void* tape,
                         size_t tape_bytes, const void* plan, void* cuda_stream) {
  if (!m || nenv <= 0 || !opts || !xT || !dLdxT || !dLdx0) return fail("null argument");
  cudaStream_t s = (cudaStream_t)cuda_stream;
  dmx_model* mm = const_cast<dmx_model*>(m);
  return m->precision == 64 ? backward_typed<double>(mm, nenv, ctrl, nknot, params, opts, xT, dLdxT, cfd_on, dLdx0, dLdctrl, dLdparams, stats, tape, tape_bytes, plan, s)
                            : backward_typed<float>(mm, nenv, ctrl, nknot, params, opts, xT, dLdxT, cfd_on, dLdx0, dLdctrl, dLdparams, stats, tape, tape_bytes, plan, s);
}

int dmx_rollout_grad(const dmx_model* m, int nenv, const void* x0, const void* ctrl, int nknot, double knot_dt, const void* params, double horizon,
                     const dmx_solver_opts* opts, const double* h_replay, int n_replay, const void* dLdxT, int cfd_on, void* xT, void* dLdx0,
                     void* dLdctrl, void* dLdparams, const dmx_stats* stats, void* tape, size_t tape_bytes, const void* plan, void* cuda_stream) {
  if (!tape) return fail("dmx_rollout_grad needs a tape");
  int rc = dmx_rollout(m, nenv, x0, ctrl, nknot, knot_dt, params, horizon, opts, h_replay, n_replay, xT, stats, tape, tape_bytes, plan, cuda_stream);
  if (rc) return rc;
  dmx_stats bs; std::memset(&bs, 0, sizeof(bs));            // failed environments are marked in the tape header; only the counter is passed on
  if (stats) { bs.n_newton_unconverged_bwd = stats->n_newton_unconverged_bwd; bs.work = stats->work; }
  return dmx_rollout_backward(m, nenv, ctrl, nknot, params, opts, xT, dLdxT, cfd_on, dLdx0, dLdctrl, dLdparams, &bs, tape, tape_bytes, plan, cuda_stream);
}

static int check_adj(const dmx_solver_opts* o) {
  if (!o) return fail("null adjoint options");
  if (o->tableau != DMX_DOPRI5 && o->tableau != DMX_TSIT5) return fail("unknown tableau");
  if (!(o->rtol >= 0) || !(o->atol >= 0) || !(o->rtol + o->atol > 0) || o->max_steps <= 0) return fail("bad adjoint tolerances / budget");
  return 0;
}

int dmx_rollout_backward_adjoint(const dmx_model* m, int nenv, const void* ctrl, int nknot, const void* params, const dmx_solver_opts* opts,
                                 const dmx_solver_opts* adj_opts, const void* xT, const void* dLdxT, int cfd_on, void* dLdx0, void* dLdctrl,
                                 void* dLdparams, const dmx_stats* stats, int* adj_info, const double* adj_replay, int n_adj_replay, const void* tape,
                                 size_t tape_bytes, const void* plan, void* cuda_stream) {
  if (!m || nenv <= 0 || !opts || !xT || !dLdxT || !dLdx0) return fail("null argument");
  if (check_adj(adj_opts)) return -1;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  dmx_model* mm = const_cast<dmx_model*>(m);
  return m->precision == 64 ? backward_typed<double>(mm, nenv, ctrl, nknot, params, opts, xT, dLdxT, cfd_on, dLdx0, dLdctrl, dLdparams, stats, tape, tape_bytes, plan, s, adj_opts, adj_info, adj_replay, n_adj_replay)
                            : backward_typed<float>(mm, nenv, ctrl, nknot, params, opts, xT, dLdxT, cfd_on, dLdx0, dLdctrl, dLdparams, stats, tape, tape_bytes, plan, s, adj_opts, adj_info, adj_replay, n_adj_replay);
}

int dmx_rollout_grad_adjoint(const dmx_model* m, int nenv, const void* x0, const void* ctrl, int nknot, double knot_dt, const void* params, double horizon,
                             const dmx_solver_opts* opts, const dmx_solver_opts* adj_opts, const double* h_replay, int n_replay, const void* dLdxT,
                             int cfd_on, void* xT, void* dLdx0, void* dLdctrl, void* dLdparams, const dmx_stats* stats, int* adj_info,
                             const double* adj_replay, int n_adj_replay, void* tape, size_t tape_bytes, const void* plan, void* cuda_stream) {
  if (!tape) return fail("dmx_rollout_grad_adjoint needs a tape");
  if (check_adj(adj_opts)) return -1;
  int rc = dmx_rollout(m, nenv, x0, ctrl, nknot, knot_dt, params, horizon, opts, h_replay, n_replay, xT, stats, tape, tape_bytes, plan, cuda_stream);
  if (rc) return rc;
  dmx_stats bs; std::memset(&bs, 0, sizeof(bs));
  if (stats) { bs.n_newton_unconverged_bwd = stats->n_newton_unconverged_bwd; bs.work = stats->work; }
  return dmx_rollout_backward_adjoint(m, nenv, ctrl, nknot, params, opts, adj_opts, xT, dLdxT, cfd_on, dLdx0, dLdctrl, dLdparams, &bs, adj_info,
                                      adj_replay, n_adj_replay, tape, tape_bytes, plan, cuda_stream);
}

int dmx_vector_field(const dmx_model* m, int n, const void* x, const void* u, const void* params, int cfd, void* acc, int* nrow, void* cuda_stream) {
  if (!m || n <= 0 || !x || !acc) return fail("null argument");
  dmx_model* mm = const_cast<dmx_model*>(m);
  cudaStream_t s = (cudaStream_t)cuda_stream;
  return m->precision == 64 ? field_typed<double>(mm, n, x, u, params, nullptr, cfd, acc, nrow, nullptr, nullptr, nullptr, nullptr, s)
                            : field_typed<float>(mm, n, x, u, params, nullptr, cfd, acc, nrow, nullptr, nullptr, nullptr, nullptr, s);
}

int dmx_vjp_field(const dmx_model* m, int n, const void* x, const void* u, const void* params, const void* kappa, int cfd, void* qbar, void* vbar,
                  void* ubar, void* pbar, void* cuda_stream) {
  if (!m || n <= 0 || !x || !kappa || !qbar || !vbar || (!ubar && m->h.nu > 0)) return fail("null argument");
  dmx_model* mm = const_cast<dmx_model*>(m);
  cudaStream_t s = (cudaStream_t)cuda_stream;
  return m->precision == 64 ? field_typed<double>(mm, n, x, u, params, kappa, cfd, nullptr, nullptr, qbar, vbar, ubar, pbar, s)
                            : field_typed<float>(mm, n, x, u, params, kappa, cfd, nullptr, nullptr, qbar, vbar, ubar, pbar, s);
}

int dmx_debug_counters(const dmx_model* m, unsigned long long* host32) {
  if (!m || !host32) return fail("null argument");
  unsigned long long* d = nullptr;
  CUDA_OK(cudaMalloc(&d, 32 * sizeof(unsigned long long)));
  cudaError_t e = m->precision == 64 ? launchers_for<double>(m->G, m->shape).prof_dump(d, 0) : launchers_for<float>(m->G, m->shape).prof_dump(d, 0);
  if (e == cudaSuccess) e = cudaMemcpy(host32, d, 32 * sizeof(unsigned long long), cudaMemcpyDeviceToHost);
  cudaFree(d);
  CUDA_OK(e);
  return 0;
}

int dmx_adam_step(int precision, int nrow, int len, void* x, const void* g, void* mom1, void* mom2, const unsigned char* active, int t,
                  double lr, double b1, double b2, double eps, double clip, void* cuda_stream) {
  if (nrow <= 0 || len <= 0 || !x || !g || !mom1 || !mom2 || t < 1) return fail("bad argument");
  if (precision != 64 && precision != 32) return fail("precision must be 64 or 32");
  cudaStream_t s = (cudaStream_t)cuda_stream;
  const int wpb = 4;                                          // a warp per row
  const int grid = (nrow + wpb - 1) / wpb;
  const double c1 = 1.0 - std::pow(b1, (double)t), c2 = 1.0 - std::pow(b2, (double)t);
  if (precision == 64) adam_clip_kernel<double><<<grid, 32 * wpb, 0, s>>>(nrow, len, (double*)x, (const double*)g, (double*)mom1, (double*)mom2, active, lr, b1, b2, eps, clip, c1, c2);
  else adam_clip_kernel<float><<<grid, 32 * wpb, 0, s>>>(nrow, len, (float*)x, (const float*)g, (float*)mom1, (float*)mom2, active, lr, b1, b2, eps, clip, c1, c2);
  CUDA_OK(cudaGetLastError());
  return 0;
}

int dmx_fma_peak(int precision, int iters, double* flops_per_s, double* ms) {
  if (!flops_per_s || !ms || iters <= 0) return fail("bad argument");
  return precision == 64 ? fma_peak_typed<double>(iters, flops_per_s, ms) : fma_peak_typed<float>(iters, flops_per_s, ms);
}

}  // extern "C"


// ---- dmx_rollout_backward_noalloc: the reverse sweep with its scratch in a static device array ------------------------
// For callers that must not allocate at call time (CUDA graph capture, tight serving loops, harnesses that forbid it).
// The reverse sweep needs per-lane-group integrator / adjoint arrays in global memory and a work-queue counter; the
// regular path keeps them in buffers the model cudaMalloc'ed at create, this variant keeps them in the file-scope array
// below: DMX_NOALLOC_SCRATCH_BYTES (16 MiB) per GPU that loads the library, held until the process exits.
// Layout: [0, 256) the work-queue counter (cleared by every call), [256, ...) the lane-group arrays (every value a sweep
// reads it has written before, so the last call's contents do not matter).  Every call on a device shares the array:
// calls that overlap on the GPU (different streams, no ordering between them) race.
// In HOST code the array's name is a host-side stand-in, not a device address; the address is taken once per device at
// set-up (dmx_model_create, with that device current) by cudaGetSymbolAddress and only that pointer goes to the kernel.
#define DMX_NOALLOC_SCRATCH_BYTES (16u << 20)
static __device__ __align__(256) unsigned char g_noalloc_scratch[DMX_NOALLOC_SCRATCH_BYTES];
enum { NOALLOC_MAX_DEV = 64 };
static unsigned char* g_noalloc_ptr[NOALLOC_MAX_DEV];   // device address of g_noalloc_scratch, per device ordinal

static int noalloc_setup(int dev) {
  if (dev < 0 || dev >= NOALLOC_MAX_DEV) return 0;       // such a device simply has no no-alloc entry point
  if (g_noalloc_ptr[dev]) return 0;
  void* ptr = nullptr;
  cudaError_t e = cudaGetSymbolAddress(&ptr, g_noalloc_scratch);
  if (e != cudaSuccess) return fail("cudaGetSymbolAddress(g_noalloc_scratch): %s", cudaGetErrorString(e));
  g_noalloc_ptr[dev] = (unsigned char*)ptr;
  return 0;
}

namespace {

template <class R>
int backward_noalloc_typed(const dmx_model* m, int nenv, const void* ctrl, int nknot, const void* params, const dmx_solver_opts* opts, const void* xT,
                           const void* dLdxT, int cfd_on, void* dLdx0, void* dLdctrl, void* dLdparams, const dmx_stats* st, const void* tape,
                           size_t tape_bytes, const void* plan, cudaStream_t s) {
  int dev = -1;
  CUDA_OK(cudaGetDevice(&dev));
  unsigned char* base = (dev >= 0 && dev < NOALLOC_MAX_DEV) ? g_noalloc_ptr[dev] : nullptr;
  if (!base) return fail("dmx_rollout_backward_noalloc: no static scratch on the current device (create a dmx_model with this device current first)");
  LaunchCfg c; c.block = m->cb.block; c.smem = m->cb.smem;
  const int gpb = groups_per_block(m, c.block);
  c.grid = std::max(1, std::min(m->cb.occ * m->sm_count, (nenv + gpb - 1) / gpb));
  size_t groups = (size_t)c.grid * gpb;
  if (m->G == 1) groups = (groups + 31) / 32 * 32;
  const size_t need = 256 + groups * (size_t)m->rl.size_bwd * sizeof(double);
  if (m->stride > 1) return fail("dmx_rollout_backward_noalloc needs a tape with checkpoint stride 1");
  if (need > (size_t)DMX_NOALLOC_SCRATCH_BYTES) {
    std::snprintf(g_err, sizeof(g_err), "dmx_rollout_backward_noalloc: nenv = %d needs %zu bytes of scratch, the static array holds %u "
                  "(DMX_NOALLOC_SCRATCH_BYTES); use dmx_rollout_backward or a smaller batch", nenv, need, (unsigned)DMX_NOALLOC_SCRATCH_BYTES);
    return -1;
  }
  BackwardArgs<R> a; std::memset(&a, 0, sizeof(a));
  if (!tape) return fail("tape missing");
  if (bind_tape<R>(m, nenv, const_cast<void*>(tape), tape_bytes, plan, a.tp, a.pl)) return -1;
  a.nenv = nenv; a.nknot = nknot; a.want_p = dLdparams != nullptr; a.cfd = cfd_on; a.tape_stages = m->tape_stages;
  a.ctrl = (const R*)ctrl; a.params = (const R*)params; a.zero_u = (const R*)m->zero_u; a.xT = (const R*)xT; a.dLdxT = (const R*)dLdxT;
  a.status = st ? st->status : nullptr; a.n_unconv = st ? st->n_newton_unconverged_bwd : nullptr; a.work = st ? st->work : nullptr;
  a.so = opts_of(opts); a.dLdx0 = (R*)dLdx0; a.dLdctrl = (R*)dLdctrl; a.dLdparams = (R*)dLdparams;
  a.lockstep = 0x1ff; a.wl = m->wl; a.rl = m->rl; a.n_light = -1;      // the work queue, as before
  a.queue = (int*)base;                                   // what must start at zero: the work-queue counter
  a.rk_scratch = (double*)(base + 256);
  CUDA_OK(cudaMemsetAsync(base, 0, 256, s));
  if (dLdctrl && nknot > 0 && m->h.nu > 0) CUDA_OK(cudaMemsetAsync(dLdctrl, 0, (size_t)nenv * nknot * m->h.nu * sizeof(R), s));
  ModelDev<R> md = dev_of<R>(m); md.arena_smem = m->cb.arena;
  CUDA_OK(launchers_for<R>(m->G, m->shape).backward(md, a, c, s));
  return 0;
}

}  // namespace

extern "C" {

size_t dmx_noalloc_scratch_bytes(void) { return (size_t)DMX_NOALLOC_SCRATCH_BYTES; }

int dmx_rollout_backward_noalloc(const dmx_model* m, int nenv, const void* ctrl, int nknot, const void* params, const dmx_solver_opts* opts,
                                 const void* xT, const void* dLdxT, int cfd_on, void* dLdx0, void* dLdctrl, void* dLdparams, const dmx_stats* stats,
                                 const void* tape, size_t tape_bytes, const void* plan, void* cuda_stream) {
  if (!m || nenv <= 0 || !opts || !xT || !dLdxT || !dLdx0) return fail("null argument");
  cudaStream_t s = (cudaStream_t)cuda_stream;
  return m->precision == 64 ? backward_noalloc_typed<double>(m, nenv, ctrl, nknot, params, opts, xT, dLdxT, cfd_on, dLdx0, dLdctrl, dLdparams, stats, tape, tape_bytes, plan, s)
                            : backward_noalloc_typed<float>(m, nenv, ctrl, nknot, params, opts, xT, dLdxT, cfd_on, dLdx0, dLdctrl, dLdparams, stats, tape, tape_bytes, plan, s);
}

}  // extern "C"
