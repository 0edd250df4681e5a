// ORACLE — TEST INFRASTRUCTURE ONLY.  Not part of the product path; shares no code with the CUDA library.
//
// Minimal tape-based reverse-mode scalar (`orc::AD`).  The oracle's step (rod_step.hpp) is a template on
// its scalar type; instantiating it with `AD` records every arithmetic operation of ONE env-step on a tape,
// and `Tape::reverse` then applies the chain rule backwards.  This gives the exact derivative of the
// discrete map of SURVEY.md Appendix A, piecewise where the map branches (comparisons look only at
// values, so every branch is frozen at its forward outcome -- SURVEY.md App. B-22), which is what the
// paper obtains from Taichi's autodiff (Sec. 3.3).  It is independent of the CUDA path's
// hand-derived adjoint and is itself pinned by central finite differences (tests/test_oracle_adjoint.py).
#pragma once
#include <cmath>
#include <vector>

namespace orc {

struct Tape {
  // node i = f(parent ia[i], parent ib[i]); pa/pb are the partial derivatives wrt the parents.
  std::vector<int> ia, ib;
  std::vector<double> pa, pb;
  int node(int a, double da, int b, double db) {
    ia.push_back(a); ib.push_back(b); pa.push_back(da); pb.push_back(db);
    return (int)ia.size() - 1;
  }
  int input() { return node(-1, 0.0, -1, 0.0); }
  size_t size() const { return ia.size(); }
  void clear() { ia.clear(); ib.clear(); pa.clear(); pb.clear(); }
  // adj has size() entries; on entry the output seeds, on exit the adjoint of every node.
  void reverse(std::vector<double>& adj) const {
    for (int i = (int)ia.size() - 1; i >= 0; --i) {
      const double g = adj[i];
      if (g == 0.0) continue;
      if (ia[i] >= 0) adj[ia[i]] += pa[i] * g;
      if (ib[i] >= 0) adj[ib[i]] += pb[i] * g;
    }
  }
};

inline Tape*& current_tape() { static thread_local Tape* t = nullptr; return t; }

struct AD {
  double v; int i;            // value, tape index (-1 = constant)
  AD() : v(0.0), i(-1) {}
  AD(double c) : v(c), i(-1) {}
  AD(double c, int idx) : v(c), i(idx) {}
  static AD variable(double c) { return AD(c, current_tape()->input()); }
};

inline AD mk(double v, int a, double da, int b, double db) {
  if (a < 0 && b < 0) return AD(v);
  return AD(v, current_tape()->node(a, da, b, db));
}

inline double val(double a) { return a; }
inline double val(const AD& a) { return a.v; }

inline AD operator+(const AD& a, const AD& b) { return mk(a.v + b.v, a.i, 1.0, b.i, 1.0); }
inline AD operator-(const AD& a, const AD& b) { return mk(a.v - b.v, a.i, 1.0, b.i, -1.0); }
inline AD operator*(const AD& a, const AD& b) { return mk(a.v * b.v, a.i, b.v, b.i, a.v); }
inline AD operator/(const AD& a, const AD& b) { return mk(a.v / b.v, a.i, 1.0 / b.v, b.i, -a.v / (b.v * b.v)); }
inline AD operator-(const AD& a) { return mk(-a.v, a.i, -1.0, -1, 0.0); }
inline AD operator+(const AD& a, double b) { return mk(a.v + b, a.i, 1.0, -1, 0.0); }
inline AD operator+(double a, const AD& b) { return mk(a + b.v, b.i, 1.0, -1, 0.0); }
inline AD operator-(const AD& a, double b) { return mk(a.v - b, a.i, 1.0, -1, 0.0); }
inline AD operator-(double a, const AD& b) { return mk(a - b.v, b.i, -1.0, -1, 0.0); }
inline AD operator*(const AD& a, double b) { return mk(a.v * b, a.i, b, -1, 0.0); }
inline AD operator*(double a, const AD& b) { return mk(a * b.v, b.i, a, -1, 0.0); }
inline AD operator/(const AD& a, double b) { return mk(a.v / b, a.i, 1.0 / b, -1, 0.0); }
inline AD operator/(double a, const AD& b) { return mk(a / b.v, b.i, -a / (b.v * b.v), -1, 0.0); }
inline AD& operator+=(AD& a, const AD& b) { a = a + b; return a; }
inline AD& operator-=(AD& a, const AD& b) { a = a - b; return a; }
inline AD& operator*=(AD& a, const AD& b) { a = a * b; return a; }
inline AD& operator+=(AD& a, double b) { a = a + b; return a; }
inline AD& operator-=(AD& a, double b) { a = a - b; return a; }
inline AD& operator*=(AD& a, double b) { a = a * b; return a; }

inline AD sqrt(const AD& a) { const double s = std::sqrt(a.v); return mk(s, a.i, 0.5 / s, -1, 0.0); }
inline AD exp(const AD& a) { const double e = std::exp(a.v); return mk(e, a.i, e, -1, 0.0); }
inline AD sin(const AD& a) { return mk(std::sin(a.v), a.i, std::cos(a.v), -1, 0.0); }
inline AD cos(const AD& a) { return mk(std::cos(a.v), a.i, -std::sin(a.v), -1, 0.0); }

// comparisons act on values only (branches are frozen at their forward outcome)
inline bool operator<(const AD& a, const AD& b) { return a.v < b.v; }
inline bool operator>(const AD& a, const AD& b) { return a.v > b.v; }
inline bool operator<=(const AD& a, const AD& b) { return a.v <= b.v; }
inline bool operator>=(const AD& a, const AD& b) { return a.v >= b.v; }
inline bool operator<(const AD& a, double b) { return a.v < b; }
inline bool operator>(const AD& a, double b) { return a.v > b; }
inline bool operator<=(const AD& a, double b) { return a.v <= b; }
inline bool operator>=(const AD& a, double b) { return a.v >= b; }
inline bool operator<(double a, const AD& b) { return a < b.v; }
inline bool operator>(double a, const AD& b) { return a > b.v; }

}  // namespace orc
