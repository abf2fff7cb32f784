// ORACLE — test infrastructure only (see oracle/README.md). Not part of the product path.
//
// O3-O6 and O12 of SURVEY.md §8(c): narrow phase (signed distance r, normal n, mid-surface
// point), pyramidal rows, impedance d(r) from solimp
// (spline: reading G5), reference acceleration (Eq. 3), the
// regulariser R = A^(1-d)/d and the CFD continuation for r>0 with softplus
// (readings G16, G17 — parity unpinned, no formula in the paper).
#pragma once
#include "kin.hpp"

namespace orc {

// spline y(x; mid, power) on x in [0,1] (reading G5)
template <class S> inline S imp_spline(const S& x, const S& mid, const S& power) {
  if (val(x) <= 0.0) return S(0.0) * x;
  if (val(x) >= 1.0) return S(1.0) + S(0.0) * x;
  if (val(x) <= val(mid)) return pow(x, power) / pow(mid, power - S(1.0));
  S one(1.0);
  return one - pow(one - x, power) / pow(one - mid, power - S(1.0));
}

// impedance d(r) for r<=0 from solimp (d_o, d_w, w, mid, power); O5
template <class S> inline S impedance(const S& r, const S* si) {
  S ar = val(r) < 0.0 ? -r : r;
  S x = ar / si[2];
  if (val(x) > 1.0) x = S(1.0);
  S y = imp_spline(x, si[3], si[4]);
  S d = si[0] + y * (si[1] - si[0]);
  if (val(d) < 0.0) d = S(0.0);
  if (val(d) > 1.0 - 1e-4) d = S(1.0 - 1e-4);
  return d;
}
// CFD continuation for 0<r<w_c from solimp-CFD (d_c, d_0, w_c, m_c, p_c); O12(ii)
template <class S> inline S impedance_cfd(const S& r, const double* sc) {
  S x = r / S(sc[2]);
  S y = imp_spline(x, S(sc[3]), S(sc[4]));
  S d = S(sc[1]) + y * S(sc[0] - sc[1]);
  if (val(d) < 0.0) d = S(0.0);
  if (val(d) > 1.0 - 1e-4) d = S(1.0 - 1e-4);
  return d;
}
template <class S> inline S softplus(const S& z, double beta) {  // log(1+exp(beta z))/beta
  S bz = z * S(beta);
  if (val(bz) > 0.0) return z + log(S(1.0) + exp(-bz)) / S(beta);
  return log(S(1.0) + exp(bz)) / S(beta);
}

template <class S> struct Geo { S r; V3<S> n, pos, t1, t2; };

// Narrow phase for one flattened candidate (O3).  Normal points from geom1 to geom2.
template <class S> Geo<S> collide(const Model&, const Kin<S>& k, const Contact& c) {
  Geo<S> g;
  V3<S> c2 = k.fr[c.body2].p + k.fr[c.body2].R * vconst<S>(c.p2);
  if (c.kind == CK_POINT_PLANE) {
    g.n = vconst<S>(c.n); g.t1 = vconst<S>(c.t1); g.t2 = vconst<S>(c.t2);
    g.r = dot(g.n, c2 - vconst<S>(c.p1)) - S(c.rho2);
    g.pos = c2 - g.n * (S(c.rho2) + S(0.5) * g.r);          // surface point - r n / 2
  } else {
    V3<S> c1 = k.fr[c.body1].p + k.fr[c.body1].R * vconst<S>(c.p1);
    V3<S> dl = c2 - c1;
    S dist = sqrt(dot(dl, dl));
    g.n = dl * (S(1.0) / dist);
    g.r = dist - S(c.rho1) - S(c.rho2);
    g.pos = c1 + g.n * (S(c.rho1) + S(0.5) * g.r);
    double an[3] = {std::fabs(val(g.n.x)), std::fabs(val(g.n.y)), std::fabs(val(g.n.z))};
    int e = 0; if (an[1] < an[e]) e = 1; if (an[2] < an[e]) e = 2;   // G3: smallest |n.e|, ties -> lowest
    V3<S> ev = mk<S>(S(e == 0 ? 1.0 : 0.0), S(e == 1 ? 1.0 : 0.0), S(e == 2 ? 1.0 : 0.0));
    V3<S> t = ev - g.n * dot(ev, g.n);
    g.t1 = t * (S(1.0) / sqrt(dot(t, t)));
    g.t2 = cross(g.n, g.t1);
  }
  return g;
}

template <class S> struct Rows {
  int nr = 0;
  std::vector<int> contact;            // candidate index of each row
  std::vector<std::vector<S>> J;       // nr x nv
  std::vector<S> aref, D, r;           // per row
};

// O4-O6 (and O12 when cfd): rows of every candidate with r<0 (cfd: r<w_c).
// p = parameter vector [mass | friction | solref | solimp]; v = joint velocities.
template <class S>
void build_rows(const Model& m, const Kin<S>& k, const S* v, const S* p, bool cfd, Rows<S>& R) {
  R = Rows<S>();
  for (size_t ci = 0; ci < m.contacts.size(); ++ci) {
    const Contact& c = m.contacts[ci];
    Geo<S> g = collide(m, k, c);
    const double* sc = &m.pair_solimp_cfd[5 * c.pair];
    double rv = val(g.r);
    if (!(rv < 0.0) && !(cfd && rv < sc[2])) continue;
    const S* si = p + m.p_solimp() + 5 * c.pair;
    S tc = p[m.p_solref() + 2 * c.pair], phi = p[m.p_solref() + 2 * c.pair + 1];
    S mu = p[m.p_fric() + c.pair];
    S dw = si[1];
    S d, posterm;
    S kden = dw * dw * tc * tc * phi * phi;
    if (cfd) {
      d = rv > 0.0 ? impedance_cfd(g.r, sc) : impedance(g.r, si);
      posterm = (d / kden) * softplus(-g.r, m.pair_cfd_beta[c.pair]);   // +k~ softplus(-r), O12(iii)
    } else {
      d = impedance(g.r, si);
      posterm = -((d / kden) * g.r);                                    // -k r, Eq. 3
    }
    S bdamp = S(2.0) / (dw * tc);
    S Ahat = S(m.pair_invweight[c.pair]);
    if (c.condim == 3) Ahat = Ahat * (S(1.0) + mu * mu);                 // G7
    S Dw = d / (Ahat * (S(1.0) - d));                                   // D = 1/R
    int nrow = c.condim == 3 ? 4 : 1;
    for (int e = 0; e < nrow; ++e) {
      V3<S> dir = g.n;
      if (c.condim == 3) {
        const V3<S>& t = e < 2 ? g.t1 : g.t2;
        dir = (e % 2 == 0) ? g.n + t * mu : g.n - t * mu;
      }
      std::vector<S> row(m.nv);
      S Jv(0.0);
      for (int j = 0; j < m.nv; ++j) {
        V3<S> l2, a2, l1, a1;
        dof_twist(m, k, j, c.body2, g.pos, l2, a2);
        dof_twist(m, k, j, c.body1, g.pos, l1, a1);
        row[j] = dot(dir, l2 - l1);
        Jv = Jv + row[j] * v[j];
      }
      R.J.push_back(row);
      R.aref.push_back(posterm - bdamp * Jv);
      R.D.push_back(Dw);
      R.r.push_back(g.r);
      R.contact.push_back((int)ci);
      R.nr++;
    }
  }
}

}  // namespace orc
