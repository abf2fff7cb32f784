// dmx_model.cuh — device-side model (flattened kinematic tree, candidate contacts, index tables)
// and the per-environment workspace layouts.  Built on the host by dmx_api.cu.
#pragma once
#include <cstddef>
#include "dmx_math.cuh"

namespace dmx {

enum { JNT_FREE = 0, JNT_HINGE = 1, JNT_SLIDE = 2 };
enum { ACT_MOTOR = 0, ACT_PD = 1 };
enum { CK_POINT_PLANE = 0, CK_POINT_POINT = 1 };

// Constants in the model's real type R (double or float); all pointers are device pointers.
template <class R> struct ModelDev {
  int nbody, njnt, nq, nv, nu, npair, nc, np, nlevel, ntw, nmp, nrmax, npp /* point-point candidates */;
  int newton_iters, ls_iters;
  int p_fric, p_solref, p_solimp;          // offsets in the parameter vector (mass at 0)
  // The constant arrays below live in one device allocation [arena, arena + arena_bytes).  arena_smem != 0: every CTA
  // copies the arena to the end of its dynamic shared memory and rebases the pointers (load_cta_const), so the index
  // tables are read with shared-memory latency instead of L1/L2 latency (the workspaces leave L1 only a few KB).
  int arena_bytes, arena_smem;
  R gravity[3];
  const unsigned char* arena;
  // ---- pointers into the arena: one contiguous block, body_parent first, p_default last (see N_ARENA_PTR) ----
  // tree
  const int *body_parent, *body_jnt, *level_ptr, *level_body;
  const R *body_pos, *body_rot, *body_ipos, *body_irot, *body_iunit;
  const int *jnt_type, *jnt_qadr, *jnt_vadr, *jnt_body;
  const R *jnt_axis, *jnt_pos, *jnt_damping, *jnt_armature;
  const int *dof_jnt, *dof_body, *dof_rot;  // dof_rot: 1 for hinge / free-rotation dofs
  // (body, ancestor-dof) table: entries of body b are tw_ptr[b] .. tw_ptr[b+1]
  const int *tw_ptr, *tw_body, *tw_dof, *tw_idx /* [nbody*nv] entry or -1 */;
  const int *sub_ptr, *sub_body;            // subtree lists (ascending, self included)
  const int *child_ptr, *child_idx;         // children lists
  const int *mp_i, *mp_j, *mp_deep;         // lower-triangle entries of M; deep = -1: structurally zero
  // flattened candidate contacts
  const int *ct_kind, *ct_b1, *ct_b2, *ct_condim, *ct_pair;
  const R *ct_p1, *ct_p2, *ct_rho1, *ct_rho2, *ct_n, *ct_t1, *ct_t2;
  const R *pair_invweight, *pair_solimp_cfd, *pair_cfd_beta;
  const int *act_type, *act_jnt;
  const R *act_gear, *act_kp, *act_kd;
  const R *p_default;
};
enum { N_ARENA_PTR = 52 };
static_assert(offsetof(ModelDev<double>, p_default) - offsetof(ModelDev<double>, body_parent) == (N_ARENA_PTR - 1) * sizeof(void*),
              "ModelDev: the arena pointers must form one contiguous block");
static_assert(offsetof(ModelDev<float>, p_default) - offsetof(ModelDev<float>, body_parent) == (N_ARENA_PTR - 1) * sizeof(void*),
              "ModelDev: the arena pointers must form one contiguous block");

// Offsets (in scalars) of the per-environment arrays inside a workspace of scalar type S.
// `full` layouts serve the cooperative evaluation of F; `res` layouts serve the per-lane
// tangent pass of the VJP, which needs the frames only.
struct WsLayout {
  int fp, fR, fw, fal, fvp, fap, com, dax, dan;       // kinematics
  int Fb, Nb, Iw, Isub, tw;                           // body wrenches, world inertias, twist table
  int M, Hc, tau, c, a0, x, g, dl, Md, xa, kap;       // dynamics and Newton vectors
  int cr, cn, cpos, ct1, ct2, cD, cpost, cbd, cmu;    // per candidate
  int cdD, cdpost;                                    // per candidate: dD/dr, d(position term)/dr (VJP)
  int fox, fvx;                                       // per body: twist under the joint rates x* (angular, velocity of the COM)
  int J, aref, D, s, pr;                              // per row
  int size;                                           // scalars
  int ld;                                             // leading dimension of M, Hc and J (odd when lanes share a warp: bank spread)
  // int workspace (separate array)
  int i_incl, i_rowstart, i_rowcand, i_active, isize;
};

// Compile-time sizes of a model (0: taken from the model at run time).  The kernels are instantiated once with
// ShapeDyn for any model and once per BASELINE configuration with its sizes, so that the loops over dofs unroll, the
// offsets i*ld+j fold into the instructions and the rows of M / H / L live in registers.  The tree,
// joint and candidate tables stay run-time data: any model with these sizes takes the static instantiation.
template <int NV_, int LD_, int NC_, int NR_> struct Shape { static const int NV = NV_, LD = LD_, NC = NC_, NR = NR_; };
typedef Shape<0, 0, 0, 0> ShapeDyn;
typedef Shape<8, 9, 2, 8> ShapeC2;        // planar push: 2 hinges + free sphere, 2 candidates x 4 rows
typedef Shape<6, 7, 8, 32> ShapeC3;       // cube toss: free box, 8 corners x 4 rows
typedef Shape<13, 13, 12, 48> ShapeC4;    // 7-hinge arm + free sphere, 12 candidates x 4 rows
typedef Shape<18, 19, 4, 16> ShapeC5;     // quadruped: free trunk + 12 hinges, 4 feet x 4 rows

// View of one workspace: base pointer + layout (kept in shared memory); arrays are resolved on use.
#define DMX_WS_ARR(name) DMX_DI Arr<S, ST> name() const { return Arr<S, ST>(b + L->name * ST); }
#define DMX_WS_INT(name) DMX_DI Arr<int, ST> name() const { return Arr<int, ST>(ib + L->i_##name * ST); }
template <class S_, int ST_, class SH_ = ShapeDyn> struct Ws {
  typedef S_ S;
  typedef SH_ SH;
  static const int ST = ST_;
  S* b; int* ib; const WsLayout* L;
  DMX_DI int ld() const { return SH::NV ? SH::LD : L->ld; }
  template <class M> DMX_DI int nv(const M& m) const { return SH::NV ? SH::NV : m.nv; }
  template <class M> DMX_DI int nc(const M& m) const { return SH::NV ? SH::NC : m.nc; }
  DMX_WS_ARR(fp) DMX_WS_ARR(fR) DMX_WS_ARR(fw) DMX_WS_ARR(fal) DMX_WS_ARR(fvp) DMX_WS_ARR(fap) DMX_WS_ARR(com) DMX_WS_ARR(dax) DMX_WS_ARR(dan)
  DMX_WS_ARR(Fb) DMX_WS_ARR(Nb) DMX_WS_ARR(Iw) DMX_WS_ARR(Isub) DMX_WS_ARR(tw)
  DMX_WS_ARR(M) DMX_WS_ARR(Hc) DMX_WS_ARR(tau) DMX_WS_ARR(c) DMX_WS_ARR(a0) DMX_WS_ARR(x) DMX_WS_ARR(g) DMX_WS_ARR(dl) DMX_WS_ARR(Md) DMX_WS_ARR(xa) DMX_WS_ARR(kap)
  DMX_WS_ARR(cr) DMX_WS_ARR(cn) DMX_WS_ARR(cpos) DMX_WS_ARR(ct1) DMX_WS_ARR(ct2) DMX_WS_ARR(cD) DMX_WS_ARR(cpost) DMX_WS_ARR(cbd) DMX_WS_ARR(cmu) DMX_WS_ARR(cdD) DMX_WS_ARR(cdpost) DMX_WS_ARR(fox) DMX_WS_ARR(fvx)
  DMX_WS_ARR(J) DMX_WS_ARR(aref) DMX_WS_ARR(D) DMX_WS_ARR(s) DMX_WS_ARR(pr)
  DMX_WS_INT(incl) DMX_WS_INT(rowstart) DMX_WS_INT(rowcand) DMX_WS_INT(active)
};

}  // namespace dmx
