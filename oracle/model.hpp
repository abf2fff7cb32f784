// ORACLE — test infrastructure only (see oracle/README.md). Not part of the product path.
//
// Model container and small 3-D algebra, templated on the scalar so that the same
// routines run on double and on the forward-mode tangent scalar of dual.hpp.
// Model fields follow SURVEY.md §8(b) (flattened kinematic tree, geoms, solref/solimp,
// friction); PAPER.md:41-45 (state x=[q,v]), PAPER.md:51 (collision).
#pragma once
#include <vector>
#include <string>
#include <stdexcept>
#include "dual.hpp"

namespace orc {

enum { JNT_FREE = 0, JNT_HINGE = 1, JNT_SLIDE = 2 };
enum { GEOM_PLANE = 0, GEOM_SPHERE = 1, GEOM_CAPSULE = 2, GEOM_BOX = 3 };
enum { ACT_MOTOR = 0, ACT_PD = 1 };
enum { CK_POINT_PLANE = 0, CK_POINT_POINT = 1 };

template <class S> struct V3 { S x, y, z; };
template <class S> inline V3<S> mk(S x, S y, S z) { V3<S> r; r.x = x; r.y = y; r.z = z; return r; }
template <class S> inline V3<S> operator+(const V3<S>& a, const V3<S>& b) { return mk<S>(a.x + b.x, a.y + b.y, a.z + b.z); }
template <class S> inline V3<S> operator-(const V3<S>& a, const V3<S>& b) { return mk<S>(a.x - b.x, a.y - b.y, a.z - b.z); }
template <class S> inline V3<S> operator*(const V3<S>& a, const S& s) { return mk<S>(a.x * s, a.y * s, a.z * s); }
template <class S> inline S dot(const V3<S>& a, const V3<S>& b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
template <class S> inline V3<S> cross(const V3<S>& a, const V3<S>& b) {
  return mk<S>(a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x);
}
template <class S> inline S comp(const V3<S>& a, int k) { return k == 0 ? a.x : (k == 1 ? a.y : a.z); }

template <class S> struct M3 { S m[3][3]; };
template <class S> inline V3<S> operator*(const M3<S>& A, const V3<S>& b) {
  return mk<S>(A.m[0][0] * b.x + A.m[0][1] * b.y + A.m[0][2] * b.z,
               A.m[1][0] * b.x + A.m[1][1] * b.y + A.m[1][2] * b.z,
               A.m[2][0] * b.x + A.m[2][1] * b.y + A.m[2][2] * b.z);
}
template <class S> inline M3<S> operator*(const M3<S>& A, const M3<S>& B) {
  M3<S> C;
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
    S s = A.m[i][0] * B.m[0][j];
    s = s + A.m[i][1] * B.m[1][j];
    s = s + A.m[i][2] * B.m[2][j];
    C.m[i][j] = s;
  }
  return C;
}
template <class S> inline M3<S> transpose(const M3<S>& A) {
  M3<S> C; for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) C.m[i][j] = A.m[j][i]; return C;
}
template <class S> inline V3<S> col(const M3<S>& A, int k) { return mk<S>(A.m[0][k], A.m[1][k], A.m[2][k]); }
template <class S> inline M3<S> eye() {
  M3<S> C; for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) C.m[i][j] = S(i == j ? 1.0 : 0.0); return C;
}

// Rotation matrix of a (not necessarily exactly unit) quaternion (w,x,y,z), SURVEY G1.
template <class S> inline M3<S> quat_to_mat(const S& w, const S& x, const S& y, const S& z) {
  M3<S> R; S two(2.0);
  R.m[0][0] = w * w + x * x - y * y - z * z; R.m[0][1] = two * (x * y - w * z); R.m[0][2] = two * (x * z + w * y);
  R.m[1][0] = two * (x * y + w * z); R.m[1][1] = w * w - x * x + y * y - z * z; R.m[1][2] = two * (y * z - w * x);
  R.m[2][0] = two * (x * z - w * y); R.m[2][1] = two * (y * z + w * x); R.m[2][2] = w * w - x * x - y * y + z * z;
  return R;
}
// Rodrigues rotation about a unit axis a by angle th.
template <class S> inline M3<S> axis_angle(const V3<S>& a, const S& th) {
  S c = cos(th), s = sin(th), one(1.0); S t = one - c; M3<S> R;
  R.m[0][0] = c + t * a.x * a.x;       R.m[0][1] = t * a.x * a.y - s * a.z; R.m[0][2] = t * a.x * a.z + s * a.y;
  R.m[1][0] = t * a.x * a.y + s * a.z; R.m[1][1] = c + t * a.y * a.y;       R.m[1][2] = t * a.y * a.z - s * a.x;
  R.m[2][0] = t * a.x * a.z - s * a.y; R.m[2][1] = t * a.y * a.z + s * a.x; R.m[2][2] = c + t * a.z * a.z;
  return R;
}

// One candidate contact: every supported geom pair flattens to sphere-like points.
struct Contact {
  int pair, kind, body1, body2, condim;
  double p1[3];   // POINT_POINT: centre in body1 frame. POINT_PLANE: plane point (world; plane on body 0)
  double p2[3];   // centre of the sphere-like point in body2 frame
  double rho1, rho2;
  double n[3], t1[3], t2[3];  // POINT_PLANE only: plane normal (local z) and its own x, y axes (G3)
};

struct Model {
  int nbody = 0, njnt = 0, nq = 0, nv = 0, nu = 0, ngeom = 0, npair = 0, np = 0, nc = 0;
  std::vector<int> body_parent, body_jnt;          // body_jnt: index of the body's joint or -1
  std::vector<double> body_pos, body_quat, body_mass, body_ipos, body_iquat, body_inertia_unit;
  std::vector<int> jnt_type, jnt_body, jnt_qadr, jnt_vadr;
  std::vector<double> jnt_axis, jnt_pos, jnt_damping, jnt_armature;
  std::vector<int> geom_type, geom_body;
  std::vector<double> geom_size, geom_pos, geom_quat;
  std::vector<int> pair_geom1, pair_geom2, pair_condim;
  std::vector<double> pair_friction, pair_solref, pair_solimp, pair_solimp_cfd, pair_cfd_beta;
  std::vector<int> act_type, act_jnt;
  std::vector<double> act_gear, act_kp, act_kd;
  double gravity[3] = {0, 0, -9.81};
  int newton_iters = 4, ls_iters = 16;
  std::vector<double> qpos0;
  // derived
  std::vector<int> dof_jnt, dof_body;   // per dof: owning joint / body
  std::vector<Contact> contacts;        // flattened static candidate list
  std::vector<double> body_invweight;   // w(b), SURVEY G7
  std::vector<double> pair_invweight;   // w_pair = w(body1)+w(body2)
  std::vector<double> p_default;        // default parameter vector [mass | friction | solref | solimp]
  // parameter vector offsets
  int p_mass() const { return 0; }
  int p_fric() const { return nbody; }
  int p_solref() const { return nbody + npair; }
  int p_solimp() const { return nbody + 3 * npair; }
  bool is_ancestor_or_self(int a, int b) const {  // a on the path from b to the world
    while (b > 0) { if (b == a) return true; b = body_parent[b]; }
    return false;
  }
};

}  // namespace orc
