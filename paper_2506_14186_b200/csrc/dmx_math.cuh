// dmx_math.cuh — scalar, 3-D algebra and lane-group primitives of the CUDA path.
//
// The device code is written once, generic in
//   S : the scalar (double or float; the one-direction tangent scalar Dual<R> serves the candidate
//       scalars D(r), position term, b, mu inside the VJP, Eq. 4 / SURVEY O11), and
//   G : the number of lanes that cooperate on one environment (1, 8, 16 or 32; a "lane group",
//       BASELINE.json north_star subsystem 4).
// Loops over independent items are strided over the group's lanes; the group re-converges
// with a masked __syncwarp.  G == 1 turns every such loop into plain serial code.
#pragma once
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

namespace dmx {

#define DMX_DI __device__ __forceinline__
#define DMX_D __device__
#ifdef DMX_NOINLINE
#define DMX_DN __device__ __noinline__
#else
#define DMX_DN __device__
#endif

// ---- optional phase counters (compile with -DDMX_PROF; read back with dmx_debug_counters) ----------
static __device__ unsigned long long g_prof[32];
#ifdef DMX_PROF
#define DMX_T0 long long t0_ = clock64()
#define DMX_TICK(gr, id) do { long long t1_ = clock64(); if ((gr).lane == 0) atomicAdd(&g_prof[id], (unsigned long long)(t1_ - t0_)); t0_ = clock64(); } while (0)
#else
#define DMX_T0 do {} while (0)
#define DMX_TICK(gr, id) do {} while (0)
#endif

// ---- phase synchronisation of a CTA's lane groups ---------------------------------------------------
// With lockstep on, every lane group arrives at a CTA-wide barrier before each phase of the vector field and of
// the VJP, so that the warps of a CTA run the same (small) piece of code at the same time and share the fetched
// instruction lines.  The barrier is the non-aligned form: groups of one warp arrive from different code
// locations.  A group that has run out of environments keeps arriving (with done = 1) until all groups are done.
static __shared__ int g_lockstep;
DMX_DI int cta_barrier_and(int p) {
  int r;
  asm volatile("{\n\t.reg .pred q, o;\n\tsetp.ne.b32 q, %1, 0;\n\tbarrier.cta.red.and.pred o, 1, q;\n\tselp.b32 %0, 1, 0, o;\n\t}" : "=r"(r) : "r"(p) : "memory");
  return r;
}
DMX_DI void phase_sync(int id) { if (g_lockstep & (1 << id)) cta_barrier_and(0); }   // g_lockstep: mask of synchronised phases
DMX_DI void phase_drain() { if (g_lockstep) while (!cta_barrier_and(1)) {} }
// A barrier between two modes of a CTA whose groups reach it after different numbers of phases: round one ends when every
// group is waiting here (or is finished), round two tells whether all of them are finished.  A finished group keeps
// calling mode_sync(true) until it returns true.
DMX_DI bool mode_sync(bool finished) {
  if (!g_lockstep) return true;
  while (!cta_barrier_and(1)) {}
  return cta_barrier_and(finished ? 1 : 0) != 0;
}

// the CTA's dynamic shared memory: per-group workspaces (and, optionally, the constant arena at its end)
extern __shared__ __align__(16) unsigned char dyn_smem[];
template <class T> DMX_DI unsigned smem_off(const T* p) { return (unsigned)(reinterpret_cast<const unsigned char*>(p) - dyn_smem); }
template <class T> DMX_DI T* smem_ptr(unsigned off) { return reinterpret_cast<T*>(dyn_smem + off); }

// ---- tangent scalar: value and one directional derivative -------------------------------
template <class T> struct Dual {
  T v, d;
  DMX_DI Dual() {}
  DMX_DI Dual(T a) : v(a), d(T(0)) {}
  DMX_DI Dual(T a, T b) : v(a), d(b) {}
};
template <class T> DMX_DI Dual<T> operator+(const Dual<T>& a, const Dual<T>& b) { return Dual<T>(a.v + b.v, a.d + b.d); }
template <class T> DMX_DI Dual<T> operator-(const Dual<T>& a, const Dual<T>& b) { return Dual<T>(a.v - b.v, a.d - b.d); }
template <class T> DMX_DI Dual<T> operator-(const Dual<T>& a) { return Dual<T>(-a.v, -a.d); }
template <class T> DMX_DI Dual<T> operator*(const Dual<T>& a, const Dual<T>& b) { return Dual<T>(a.v * b.v, a.d * b.v + a.v * b.d); }
template <class T> DMX_DI Dual<T> operator/(const Dual<T>& a, const Dual<T>& b) {
  T iv = T(1) / b.v, q = a.v * iv;
  return Dual<T>(q, (a.d - q * b.d) * iv);
}
template <class T> DMX_DI Dual<T>& operator+=(Dual<T>& a, const Dual<T>& b) { a.v += b.v; a.d += b.d; return a; }
template <class T> DMX_DI Dual<T>& operator-=(Dual<T>& a, const Dual<T>& b) { a.v -= b.v; a.d -= b.d; return a; }

DMX_DI double val(double a) { return a; }
DMX_DI float val(float a) { return a; }
template <class T> DMX_DI T val(const Dual<T>& a) { return a.v; }

DMX_DI bool has_tangent(double) { return false; }
DMX_DI bool has_tangent(float) { return false; }
template <class T> DMX_DI bool has_tangent(const Dual<T>& a) { return a.d != T(0); }

template <class S> struct RealOf { typedef S type; };
template <class T> struct RealOf<Dual<T> > { typedef T type; };

DMX_DI double m_sqrt(double a) { return sqrt(a); }
DMX_DI float m_sqrt(float a) { return sqrtf(a); }
DMX_DI double m_rsqrt(double a) { return rsqrt(a); }
DMX_DI float m_rsqrt(float a) { return rsqrtf(a); }
DMX_DI double m_exp(double a) { return exp(a); }
DMX_DI float m_exp(float a) { return expf(a); }
DMX_DI double m_log(double a) { return log(a); }
DMX_DI float m_log(float a) { return logf(a); }
DMX_DI double m_pow(double a, double b) { return pow(a, b); }
DMX_DI float m_pow(float a, float b) { return powf(a, b); }
DMX_DI void m_sincos(double a, double& s, double& c) { sincos(a, &s, &c); }
DMX_DI void m_sincos(float a, float& s, float& c) { sincosf(a, &s, &c); }
template <class T> DMX_DI Dual<T> m_sqrt(const Dual<T>& a) { T s = m_sqrt(a.v); return Dual<T>(s, a.d * (T(0.5) / s)); }
template <class T> DMX_DI Dual<T> m_rsqrt(const Dual<T>& a) { T r = m_rsqrt(a.v); return Dual<T>(r, a.d * (T(-0.5) * r / a.v)); }
template <class T> DMX_DI Dual<T> m_exp(const Dual<T>& a) { T e = m_exp(a.v); return Dual<T>(e, e * a.d); }
template <class T> DMX_DI Dual<T> m_log(const Dual<T>& a) { return Dual<T>(m_log(a.v), a.d / a.v); }
template <class T> DMX_DI void m_sincos(const Dual<T>& a, Dual<T>& s, Dual<T>& c) {
  T sv, cv; m_sincos(a.v, sv, cv);
  s = Dual<T>(sv, cv * a.d); c = Dual<T>(cv, -sv * a.d);
}
// a^b for a > 0; both may carry tangents
template <class T> DMX_DI Dual<T> m_pow(const Dual<T>& a, const Dual<T>& b) {
  T f = m_pow(a.v, b.v);
  return Dual<T>(f, b.v * m_pow(a.v, b.v - T(1)) * a.d + f * m_log(a.v) * b.d);
}

// ---- strided array view: element i lives at p[i*ST] ----------------------------------------
// ST == 1: contiguous per-group workspace in shared memory; ST == 32: per-lane workspaces of a
// warp interleaved so that lanes touching the same index coalesce (G == 1 instantiations).  The stride is a compile-time constant.
template <class S, int ST> struct Arr {
  S* p;
  DMX_DI Arr() {}
  DMX_DI explicit Arr(S* p_) : p(p_) {}
  DMX_DI S& operator[](int i) const { return p[i * ST]; }
  DMX_DI Arr<S, ST> at(int o) const { return Arr<S, ST>(p + o * ST); }
};

// ---- lane group ----------------------------------------------------------------------------
template <int G> struct Grp {
  int lane; unsigned mask_;
  // A 32-lane group is the whole warp: the literal mask lets the compiler emit plain SHFL / WARPSYNC instead of the
  // WARPSYNC.COLLECTIVE ... ENDCOLLECTIVE sequence it needs around a shuffle whose mask is a run-time value.
  DMX_DI unsigned mask() const { return G == 32 ? 0xffffffffu : mask_; }
  DMX_DI void sync() const { if (G > 1) __syncwarp(mask()); }
  DMX_DI bool all(bool pred) const {
    if (G == 1) return pred;
    unsigned b = __ballot_sync(mask(), pred);
    return (b & mask()) == mask();
  }
  template <class T> DMX_DI T from_lane(T x, int src) const {   // value held by the group's lane `src` (uniform over the group)
    if (G == 1) return x;
    if (G == 32) return __shfl_sync(0xffffffffu, x, src);
    return __shfl_sync(mask_, x, ((threadIdx.x & 31) & ~(G - 1)) + src);
  }
  template <class T> DMX_DI T xor_lane(T x, int s) const {       // value held by the group's lane (lane xor s), s < G
    if (G == 1) return x;
    return __shfl_xor_sync(mask(), x, s);
  }
  DMX_DI int bcast_int(int x) const {            // value of the group's lane 0
    if (G == 1) return x;
    if (G == 32) return __shfl_sync(0xffffffffu, x, 0);
    return __shfl_sync(mask_, x, (threadIdx.x & 31) & ~(G - 1));
  }
};
template <int G> DMX_DI Grp<G> make_group() {
  Grp<G> g;
  int wl = threadIdx.x & 31;
  g.lane = wl & (G - 1);
  g.mask_ = (G == 32) ? 0xffffffffu : (((1u << G) - 1u) << (wl & ~(G - 1)));
  return g;
}

// ---- 3-D algebra ---------------------------------------------------------------------------
template <class S> struct V3 { S x, y, z; };
template <class S> DMX_DI V3<S> mk3(const S& x, const S& y, const S& z) { V3<S> r; r.x = x; r.y = y; r.z = z; return r; }
template <class S> DMX_DI V3<S> operator+(const V3<S>& a, const V3<S>& b) { return mk3<S>(a.x + b.x, a.y + b.y, a.z + b.z); }
template <class S> DMX_DI V3<S> operator-(const V3<S>& a, const V3<S>& b) { return mk3<S>(a.x - b.x, a.y - b.y, a.z - b.z); }
template <class S> DMX_DI V3<S> operator*(const V3<S>& a, const S& s) { return mk3<S>(a.x * s, a.y * s, a.z * s); }
template <class S> DMX_DI S dot(const V3<S>& a, const V3<S>& b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
template <class S> DMX_DI V3<S> cross(const V3<S>& a, const V3<S>& b) {
  return mk3<S>(a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x);
}
template <class S> struct M3 { S m[9]; };   // row-major
template <class S> DMX_DI V3<S> operator*(const M3<S>& A, const V3<S>& b) {
  return mk3<S>(A.m[0] * b.x + A.m[1] * b.y + A.m[2] * b.z, A.m[3] * b.x + A.m[4] * b.y + A.m[5] * b.z,
                A.m[6] * b.x + A.m[7] * b.y + A.m[8] * b.z);
}
template <class S> DMX_DI M3<S> operator*(const M3<S>& A, const M3<S>& B) {
  M3<S> C;
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) C.m[3 * i + j] = A.m[3 * i] * B.m[j] + A.m[3 * i + 1] * B.m[3 + j] + A.m[3 * i + 2] * B.m[6 + j];
  return C;
}
template <class S> DMX_DI V3<S> colv(const M3<S>& A, int k) { return mk3<S>(A.m[k], A.m[3 + k], A.m[6 + k]); }

template <class S, int ST> DMX_DI V3<S> ld3(const Arr<S, ST>& a, int i) { return mk3<S>(a[3 * i], a[3 * i + 1], a[3 * i + 2]); }
template <class S, int ST> DMX_DI void st3(const Arr<S, ST>& a, int i, const V3<S>& v) { a[3 * i] = v.x; a[3 * i + 1] = v.y; a[3 * i + 2] = v.z; }
template <class S, int ST> DMX_DI M3<S> ld9(const Arr<S, ST>& a, int i) { M3<S> A;
#pragma unroll
  for (int k = 0; k < 9; ++k) A.m[k] = a[9 * i + k];
  return A; }
template <class S, int ST> DMX_DI void st9(const Arr<S, ST>& a, int i, const M3<S>& A) {
#pragma unroll
  for (int k = 0; k < 9; ++k) a[9 * i + k] = A.m[k]; }
// constants of the model (real type R) lifted to the scalar S
template <class S, class R> DMX_DI V3<S> c3(const R* a, int i) { return mk3<S>(S(a[3 * i]), S(a[3 * i + 1]), S(a[3 * i + 2])); }
template <class S, class R> DMX_DI M3<S> c9(const R* a, int i) { M3<S> A;
#pragma unroll
  for (int k = 0; k < 9; ++k) A.m[k] = S(a[9 * i + k]);
  return A; }

// rotation matrix of a quaternion (w,x,y,z), not necessarily exactly unit
template <class S> DMX_DI M3<S> quat_to_mat(const S& w, const S& x, const S& y, const S& z) {
  M3<S> R; S two(2.0);
  R.m[0] = w * w + x * x - y * y - z * z; R.m[1] = two * (x * y - w * z); R.m[2] = two * (x * z + w * y);
  R.m[3] = two * (x * y + w * z); R.m[4] = w * w - x * x + y * y - z * z; R.m[5] = two * (y * z - w * x);
  R.m[6] = two * (x * z - w * y); R.m[7] = two * (y * z + w * x); R.m[8] = w * w - x * x - y * y + z * z;
  return R;
}
// Rodrigues rotation about the unit axis a by angle th
template <class S> DMX_DI M3<S> axis_angle(const V3<S>& a, const S& th) {
  S s, c; m_sincos(th, s, c);
  S t = S(1.0) - c; M3<S> R;
  R.m[0] = c + t * a.x * a.x;       R.m[1] = t * a.x * a.y - s * a.z; R.m[2] = t * a.x * a.z + s * a.y;
  R.m[3] = t * a.x * a.y + s * a.z; R.m[4] = c + t * a.y * a.y;       R.m[5] = t * a.y * a.z - s * a.x;
  R.m[6] = t * a.x * a.z - s * a.y; R.m[7] = t * a.y * a.z + s * a.x; R.m[8] = c + t * a.z * a.z;
  return R;
}

}  // namespace dmx
