// dmx_model.cuh — device-side model (flattened kinematic tree, candidate contacts, index tables)
// and the per-environment workspace layouts.  Built on the host by dmx_api.cu.
#pragma once
#include "dmx_math.cuh"

namespace dmx {

enum { JNT_FREE = 0, JNT_HINGE = 1, JNT_SLIDE = 2 };
enum { ACT_MOTOR = 0, ACT_PD = 1 };
enum { CK_POINT_PLANE = 0, CK_POINT_POINT = 1 };

// Constants in the model's real type R (double or float); all pointers are device pointers.
template <class R> struct ModelDev {
  int nbody, njnt, nq, nv, nu, npair, nc, np, nlevel, ntw, nmp, nrmax;
  int newton_iters, ls_iters;
  int p_fric, p_solref, p_solimp;          // offsets in the parameter vector (mass at 0)
  // tree
  const int *body_parent, *body_jnt, *level_ptr, *level_body;
  const R *body_pos, *body_rot, *body_ipos, *body_irot, *body_iunit;
  const int *jnt_type, *jnt_qadr, *jnt_vadr, *jnt_body;
  const R *jnt_axis, *jnt_pos, *jnt_damping, *jnt_armature;
  const int *dof_jnt, *dof_body, *dof_rot;  // dof_rot: 1 for hinge / free-rotation dofs
  // (body, ancestor-dof) table: entries of body b are tw_ptr[b] .. tw_ptr[b+1]
  const int *tw_ptr, *tw_body, *tw_dof, *tw_idx /* [nbody*nv] entry or -1 */;
  const int *sub_ptr, *sub_body;            // subtree lists (ascending, self included)
  const int *mp_i, *mp_j, *mp_deep;         // lower-triangle entries of M; deep = -1: structurally zero
  // flattened candidate contacts
  const int *ct_kind, *ct_b1, *ct_b2, *ct_condim, *ct_pair;
  const R *ct_p1, *ct_p2, *ct_rho1, *ct_rho2, *ct_n, *ct_t1, *ct_t2;
  const R *pair_invweight, *pair_solimp_cfd, *pair_cfd_beta;
  const int *act_type, *act_jnt;
  const R *act_gear, *act_kp, *act_kd;
  R gravity[3];
  const R *p_default;
};

// Offsets (in scalars) of the per-environment arrays inside a workspace of scalar type S.
// `full` layouts serve the cooperative evaluation of F; `res` layouts serve the per-lane
// tangent pass of the VJP, which needs the frames only.
struct WsLayout {
  int fp, fR, fw, fal, fvp, fap, com, dax, dan;       // kinematics
  int Fb, Nb, Iw, Isub, tw;                           // body wrenches, world inertias, twist table
  int M, Hc, tau, c, a0, x, g, dl, Md, xa, kap;       // dynamics and Newton vectors
  int cr, cn, cpos, ct1, ct2, cD, cpost, cbd, cmu;    // per candidate
  int J, aref, D, s, pr;                              // per row
  int size;                                           // scalars
  // int workspace (separate array)
  int i_incl, i_rowstart, i_rowcand, i_active, isize;
};

template <class S> struct Ws {
  Arr<S> fp, fR, fw, fal, fvp, fap, com, dax, dan, Fb, Nb, Iw, Isub, tw, M, Hc, tau, c, a0, x, g, dl, Md, xa, kap;
  Arr<S> cr, cn, cpos, ct1, ct2, cD, cpost, cbd, cmu, J, aref, D, s, pr;
  Arr<int> incl, rowstart, rowcand, active;
  DMX_DI void bind(const WsLayout& L, S* base, int st, int* ibase, int ist) {
    Arr<S> b(base, st);
    fp = b.at(L.fp); fR = b.at(L.fR); fw = b.at(L.fw); fal = b.at(L.fal); fvp = b.at(L.fvp); fap = b.at(L.fap);
    com = b.at(L.com); dax = b.at(L.dax); dan = b.at(L.dan);
    Fb = b.at(L.Fb); Nb = b.at(L.Nb); Iw = b.at(L.Iw); Isub = b.at(L.Isub); tw = b.at(L.tw);
    M = b.at(L.M); Hc = b.at(L.Hc); tau = b.at(L.tau); c = b.at(L.c); a0 = b.at(L.a0); x = b.at(L.x); g = b.at(L.g);
    dl = b.at(L.dl); Md = b.at(L.Md); xa = b.at(L.xa); kap = b.at(L.kap);
    cr = b.at(L.cr); cn = b.at(L.cn); cpos = b.at(L.cpos); ct1 = b.at(L.ct1); ct2 = b.at(L.ct2);
    cD = b.at(L.cD); cpost = b.at(L.cpost); cbd = b.at(L.cbd); cmu = b.at(L.cmu);
    J = b.at(L.J); aref = b.at(L.aref); D = b.at(L.D); s = b.at(L.s); pr = b.at(L.pr);
    Arr<int> ib(ibase, ist);
    incl = ib.at(L.i_incl); rowstart = ib.at(L.i_rowstart); rowcand = ib.at(L.i_rowcand); active = ib.at(L.i_active);
  }
};

}  // namespace dmx
