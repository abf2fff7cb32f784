// ORACLE — test infrastructure only (see oracle/README.md). Not part of the product path.
//
// O7 + D1 of SURVEY.md §8(c): minimiser of the reduced primal problem PAPER.md Eq. (2)
//   Phi(x) = 1/2 (x-a0)^T M (x-a0) + 1/2 sum_i D_i min(0, J_i x - aref_i)^2
// by Newton's method with a fixed iteration budget ("exact Newton method";
// iterations 4 / 2, ls_iterations 10 / 16; reading G9) and the bracketed
// one-dimensional Newton line search of D1.  Plain dense Cholesky, doubles only.
#pragma once
#include <vector>
#include <cmath>

namespace orc {

// in-place lower Cholesky of a dense SPD n x n (row-major); returns false if not PD
inline bool cholesky(std::vector<double>& A, int n) {
  for (int j = 0; j < n; ++j) {
    double s = A[j * n + j];
    for (int k = 0; k < j; ++k) s -= A[j * n + k] * A[j * n + k];
    if (!(s > 0.0)) return false;
    double l = std::sqrt(s);
    A[j * n + j] = l;
    for (int i = j + 1; i < n; ++i) {
      double t = A[i * n + j];
      for (int k = 0; k < j; ++k) t -= A[i * n + k] * A[j * n + k];
      A[i * n + j] = t / l;
    }
  }
  return true;
}
inline void chol_solve(const std::vector<double>& L, int n, double* b) {
  for (int i = 0; i < n; ++i) { double s = b[i]; for (int k = 0; k < i; ++k) s -= L[i * n + k] * b[k]; b[i] = s / L[i * n + i]; }
  for (int i = n - 1; i >= 0; --i) { double s = b[i]; for (int k = i + 1; k < n; ++k) s -= L[k * n + i] * b[k]; b[i] = s / L[i * n + i]; }
}

struct SolveResult {
  std::vector<double> x;        // v' = x*
  std::vector<char> active;     // final active set {i : J_i x* - aref_i < 0}
  std::vector<double> f;        // f_i = D_i max(0, aref_i - J_i x*) >= 0
  bool converged = true;        // last Newton step was a full step inside an unchanged active set
  int iters = 0;
};

// M: nv x nv (row-major, SPD), a0[nv], J: nr rows of nv, aref[nr], D[nr]
inline SolveResult contact_solve(int nv, int nr, const std::vector<double>& M, const double* a0,
                                 const std::vector<std::vector<double>>& J, const double* aref, const double* D,
                                 int n_it, int n_ls) {
  SolveResult R; R.x.assign(a0, a0 + nv); R.active.assign(nr, 0); R.f.assign(nr, 0.0);
  if (nr == 0) return R;
  std::vector<double> s(nr), p(nr), g(nv), dl(nv), H(nv * nv), Md(nv), xa(nv);
  R.converged = false;
  for (int it = 0; it < n_it; ++it) {
    R.iters = it + 1;
    for (int i = 0; i < nr; ++i) { double t = 0; for (int j = 0; j < nv; ++j) t += J[i][j] * R.x[j]; s[i] = t - aref[i]; }
    for (int j = 0; j < nv; ++j) xa[j] = R.x[j] - a0[j];
    for (int a = 0; a < nv; ++a) { double t = 0; for (int b = 0; b < nv; ++b) t += M[a * nv + b] * xa[b]; g[a] = t; }
    H = M;
    for (int i = 0; i < nr; ++i) if (s[i] < 0.0) {
      for (int a = 0; a < nv; ++a) {
        g[a] += J[i][a] * D[i] * s[i];
        for (int b = 0; b < nv; ++b) H[a * nv + b] += D[i] * J[i][a] * J[i][b];
      }
    }
    if (!cholesky(H, nv)) break;
    for (int a = 0; a < nv; ++a) dl[a] = -g[a];
    chol_solve(H, nv, dl.data());
    for (int i = 0; i < nr; ++i) { double t = 0; for (int j = 0; j < nv; ++j) t += J[i][j] * dl[j]; p[i] = t; }
    // full step inside the same active set: exact minimiser of the current quadratic -> done
    bool same = true;
    for (int i = 0; i < nr; ++i) if ((s[i] < 0.0) != (s[i] + p[i] < 0.0)) { same = false; break; }
    double alpha = 1.0;
    if (!same) {
      // D1: phi'(a) = dl^T M (x + a dl - a0) + sum_i D_i p_i min(0, s_i + a p_i)
      for (int a = 0; a < nv; ++a) { double t = 0; for (int b = 0; b < nv; ++b) t += M[a * nv + b] * dl[b]; Md[a] = t; }
      double dMd = 0, dMxa = 0;
      for (int a = 0; a < nv; ++a) { dMd += dl[a] * Md[a]; dMxa += Md[a] * xa[a]; }
      // Row sums in the fixed "32-slot" order that both sides document (D1/D4; SURVEY D4 allows any fixed
      // shared order): row i goes to slot i mod 32 in increasing i, the slots are then combined pairwise,
      // slot[k] += slot[k xor s] for s = 1, 2, 4, 8, 16.
      auto d1 = [&](double a, double& d2) {
        double s1[32], s2[32];
        for (int k = 0; k < 32; ++k) { s1[k] = 0.0; s2[k] = 0.0; }
        for (int i = 0; i < nr; ++i) { double si = s[i] + a * p[i]; if (si < 0.0) { s1[i % 32] += D[i] * p[i] * si; s2[i % 32] += D[i] * p[i] * p[i]; } }
        for (int sft = 1; sft < 32; sft <<= 1)
          for (int k = 0; k < 32; ++k) if (!(k & sft)) { s1[k] = s1[k] + s1[k ^ sft]; s2[k] = s2[k] + s2[k ^ sft]; }
        d2 = dMd + s2[0];
        return (dMxa + a * dMd) + s1[0];
      };
      double lo = 0.0, hi = INFINITY, a = 0.0, d2; double d1a = d1(0.0, d2);
      bool frozen = false;
      for (int ls = 0; ls < n_ls && !frozen; ++ls) {
        double an = (ls == 0) ? 1.0 : a - d1a / d2;          // first iterate is exactly alpha = 1
        if (ls > 0 && an == a) break;                        // D1 (amended): no representable progress -> root reached
        if (!(an > lo && an < hi)) an = std::isfinite(hi) ? 0.5 * (lo + hi) : 2.0 * std::fmax(a, 1.0);
        a = an; d1a = d1(a, d2);
        if (d1a < 0.0) lo = a; else if (d1a > 0.0) hi = a; else frozen = true;
      }
      alpha = a;
    }
    for (int a = 0; a < nv; ++a) R.x[a] += alpha * dl[a];
    if (same) { R.converged = true; break; }
  }
  for (int i = 0; i < nr; ++i) {
    double t = 0; for (int j = 0; j < nv; ++j) t += J[i][j] * R.x[j];
    double si = t - aref[i];
    R.active[i] = si < 0.0; R.f[i] = si < 0.0 ? -D[i] * si : 0.0;
  }
  return R;
}

}  // namespace orc
