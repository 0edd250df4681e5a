// rod_adj.cuh — hand-written reverse-mode (adjoint) of every per-element operator in rod_ops.cuh.
//
// Convention: for a forward operator  out = F(in)  the adjoint takes the forward inputs (values are recomputed,
// nothing is read from a tape here) plus the adjoints of the outputs ("bar" = dL/d.) and ACCUMULATES (+=) into
// the adjoints of the inputs.  Branches (clamps, yield, contact regions) are frozen at their forward outcome,
// i.e. this is the exact derivative of the discrete map piecewise (gradients of the simulation
// step; R-22).  `T`-generic and host/device like rod_ops.cuh: tests/host/ checks each function
// against central differences in double on the CPU.
#pragma once
#include "rod_ops.cuh"

namespace dlo {

// c = a x b
template <class T> DLO_HD void cross_adj(const V3<T>& a, const V3<T>& b, const V3<T>& cbar, V3<T>& abar, V3<T>& bbar) {
  abar += cross(b, cbar);
  bbar += cross(cbar, a);
}

// t = e / |e|, iL = 1/|e|  ->  ebar
template <class T> DLO_HD V3<T> normalize_adj(const V3<T>& t, T iL, const V3<T>& tbar, T iLbar) {
  // dt = iL (I - t t^T) de ; d(iL) = -iL^2 t . de
  return iL * (tbar - dot(tbar, t) * t) - (iLbar * iL * iL) * t;
}

// shared tail of the curvature computations: given adjoints of kb (vector), m1, m2 and of ichi = 1/(1+ta.tb),
// push them to the tangents and directors.  kb = 2 ichi (ta x tb), m1 = (d1a+d1b)/2, m2 = (ta x d1a + tb x d1b)/2
template <class T> DLO_HD void curvature_tail_adj(const V3<T>& ta, const V3<T>& tb, const V3<T>& d1a, const V3<T>& d1b, T ichi,
                                                  const V3<T>& kbbar, const V3<T>& m1bar, const V3<T>& m2bar, T ichibar,
                                                  V3<T>& tabar, V3<T>& tbbar, V3<T>& d1abar, V3<T>& d1bbar) {
  d1abar += T(0.5) * m1bar;
  d1bbar += T(0.5) * m1bar;
  const V3<T> cbar = T(0.5) * m2bar;
  cross_adj(ta, d1a, cbar, tabar, d1abar);
  cross_adj(tb, d1b, cbar, tbbar, d1bbar);
  const V3<T> X = cross(ta, tb);
  ichibar += T(2) * dot(kbbar, X);
  const V3<T> Xbar = (T(2) * ichi) * kbbar;
  cross_adj(ta, tb, Xbar, tabar, tbbar);
  const T cbar_s = -ichi * ichi * ichibar;
  tabar += cbar_s * tb;
  tbbar += cbar_s * ta;
}

// Eq.4-5 adjoint: (k1, k2) = material_curvature(ta, tb, d1a, d1b)
template <class T> DLO_HD void material_curvature_adj(const V3<T>& ta, const V3<T>& tb, const V3<T>& d1a, const V3<T>& d1b, T k1bar,
                                                      T k2bar, V3<T>& tabar, V3<T>& tbbar, V3<T>& d1abar, V3<T>& d1bbar) {
  const T ichi = T(1) / (T(1) + dot(ta, tb));
  const V3<T> kb = (T(2) * ichi) * cross(ta, tb);
  const V3<T> m1 = T(0.5) * (d1a + d1b), m2 = T(0.5) * (cross(ta, d1a) + cross(tb, d1b));
  const V3<T> kbbar = k1bar * m2 + k2bar * m1;
  curvature_tail_adj(ta, tb, d1a, d1b, ichi, kbbar, k2bar * kb, k1bar * kb, T(0), tabar, tbbar, d1abar, d1bbar);
}

// adjoint of bend_element: (Ga, Gb) = F(ta, tb, iLa, iLb, d1a, d1b, k1b, k2b, s)
template <class T>
DLO_HD void bend_element_adj(const V3<T>& ta, const V3<T>& tb, T iLa, T iLb, const V3<T>& d1a, const V3<T>& d1b, T k1b, T k2b, T s,
                             const V3<T>& Gabar, const V3<T>& Gbbar, V3<T>& tabar, V3<T>& tbbar, T& iLabar, T& iLbbar,
                             V3<T>& d1abar, V3<T>& d1bbar, T& k1bbar, T& k2bbar, T& sbar) {
  // forward values
  const T ichi = T(1) / (T(1) + dot(ta, tb));
  const V3<T> kb = (T(2) * ichi) * cross(ta, tb);
  const V3<T> m1 = T(0.5) * (d1a + d1b), m2 = T(0.5) * (cross(ta, d1a) + cross(tb, d1b));
  const T dk1 = dot(kb, m2) - k1b, dk2 = dot(kb, m1) - k2b;
  const V3<T> q = dk1 * m2 + dk2 * m1;
  const T qkb = dot(q, kb);
  const V3<T> Za = T(2) * cross(tb, q) - qkb * tb, Zb = T(2) * cross(q, ta) - qkb * ta;
  const V3<T> Aa = ichi * Za, Ab = ichi * Zb;
  const T pa = dot(Aa, ta), pb = dot(Ab, tb);
  const V3<T> Ua = Aa - pa * ta, Ub = Ab - pb * tb;
  // reverse
  const T ga = dot(Gabar, Ua), gb = dot(Gbbar, Ub);
  sbar += ga * iLa + gb * iLb;
  iLabar += s * ga;
  iLbbar += s * gb;
  const V3<T> Uabar = (s * iLa) * Gabar, Ubbar = (s * iLb) * Gbbar;
  const T pabar = -dot(Uabar, ta), pbbar = -dot(Ubbar, tb);
  tabar += (-pa) * Uabar + pabar * Aa;
  tbbar += (-pb) * Ubbar + pbbar * Ab;
  const V3<T> Aabar = Uabar + pabar * ta, Abbar = Ubbar + pbbar * tb;
  T ichibar = dot(Aabar, Za) + dot(Abbar, Zb);
  const V3<T> Zabar = ichi * Aabar, Zbbar = ichi * Abbar;
  const T qkbbar = -dot(Zabar, tb) - dot(Zbbar, ta);
  tbbar += (-qkb) * Zabar;
  tabar += (-qkb) * Zbbar;
  V3<T> qbar = qkbbar * kb;
  V3<T> kbbar = qkbbar * q;
  cross_adj(tb, q, T(2) * Zabar, tbbar, qbar);   // Ya = tb x q
  cross_adj(q, ta, T(2) * Zbbar, qbar, tabar);   // Yb = q x ta
  const T dk1bar = dot(qbar, m2), dk2bar = dot(qbar, m1);
  V3<T> m2bar = dk1 * qbar + dk1bar * kb, m1bar = dk2 * qbar + dk2bar * kb;
  kbbar += dk1bar * m2 + dk2bar * m1;
  k1bbar -= dk1bar;
  k2bbar -= dk2bar;
  curvature_tail_adj(ta, tb, d1a, d1b, ichi, kbbar, m1bar, m2bar, ichibar, tabar, tbbar, d1abar, d1bbar);
}

// adjoint of r = ptransport(a, b, u)
template <class T> DLO_HD void ptransport_adj(const V3<T>& a, const V3<T>& b, const V3<T>& u, const V3<T>& rbar, V3<T>& abar,
                                              V3<T>& bbar, V3<T>& ubar) {
  const V3<T> w = cross(a, b);
  const T k = T(1) / (T(1) + dot(a, b));
  const V3<T> wu = cross(w, u), wwu = cross(w, wu);
  ubar += rbar;
  V3<T> wubar = rbar, wbar = zero3<T>();
  const T kbar = dot(rbar, wwu);
  cross_adj(w, wu, k * rbar, wbar, wubar);
  cross_adj(w, u, wubar, wbar, ubar);
  const T cbar = -k * k * kbar;
  abar += cbar * b;
  bbar += cbar * a;
  cross_adj(a, b, wbar, abar, bbar);
}

// A9 frame update of one edge: d1n = normalize(P(to->tn) d1o - ((.) . tn) tn); adjoint given d1nbar
template <class T> DLO_HD void frame_update_adj(const V3<T>& to, const V3<T>& tn, const V3<T>& d1o, const V3<T>& d1nbar, V3<T>& tobar,
                                                V3<T>& tnbar, V3<T>& d1obar) {
  const V3<T> d = ptransport(to, tn, d1o);
  const T p = dot(d, tn);
  const V3<T> dp = d - p * tn;
  const T inrm = rsqrt_(dot(dp, dp));
  const V3<T> d1n = inrm * dp;
  const V3<T> dpbar = inrm * (d1nbar - dot(d1nbar, d1n) * d1n);
  const T pbar = -dot(dpbar, tn);
  tnbar += (-p) * dpbar + pbar * d;
  const V3<T> dbar = dpbar + pbar * tn;
  ptransport_adj(to, tn, d1o, dbar, tobar, tnbar, d1obar);
}

// Eq.11 adjoint.  (k1,k2) current curvature, (k1b,k2b) rest curvature BEFORE the update, g1,g2 = adjoint of the
// updated rest curvature.  Outputs: adjoint of the old rest curvature (returned in g1,g2), of kappa, Y and r_c.
template <class T> DLO_HD void plasticity_adj(T k1, T k2, T k1b, T k2b, T Y, T r_c, T& g1, T& g2, T& k1bar, T& k2bar, T& Ybar, T& rcbar) {
  const T e1 = k1 - k1b, e2 = k2 - k2b;
  const T n2 = e1 * e1 + e2 * e2;
  if (!(n2 > Y * Y)) return;
  const T n = sqrt_(n2), s = r_c * (n - Y) / n;
  const T sbar = g1 * e1 + g2 * e2;
  const T nbar = sbar * r_c * Y / n2;
  rcbar += sbar * (n - Y) / n;
  Ybar -= sbar * r_c / n;
  const T eb1 = s * g1 + nbar * e1 / n, eb2 = s * g2 + nbar * e2 / n;
  k1bar += eb1; k2bar += eb2;
  g1 -= eb1; g2 -= eb2;
}

// Eq.10 adjoint on one edge.  Forward (pre-update values): e, S;  lam, t from project_edge;  then
// S' = S + lam, dxj' = dxj + lam wj t, dxn' = dxn - lam wn t.  In: gj, gn = adjoints of dxj', dxn'; Sbar' .
// Out: ebar (adjoint of the edge vector: += to x^p/dx of the next vertex, -= to those of vertex j), the new
// Sbar (adjoint of S before the update), atilbar +=.
template <class T> DLO_HD void project_edge_adj(const V3<T>& t, T iL, T lam, T Spost, T wj, T wn, T atil, const V3<T>& gj, const V3<T>& gn,
                                                T& Sbar, T& atilbar, V3<T>& ebar) {
  const V3<T> g = wj * gj - wn * gn;
  const T lambar = dot(g, t) + Sbar;
  const T numbar = lambar / (wj + wn + atil);
  atilbar -= numbar * Spost;
  Sbar -= atil * numbar;
  const V3<T> tbar = lam * g;
  ebar = numbar * t + iL * (tbar - dot(tbar, t) * t);
}

// closest_points adjoint: adjoints tbar, ubar of the outputs -> adjoints of the four end points
template <class T> DLO_HD void closest_points_adj(const V3<T>& p1, const V3<T>& q1, const V3<T>& p2, const V3<T>& q2, T tbar, T ubar,
                                                  V3<T>& p1bar, V3<T>& q1bar, V3<T>& p2bar, V3<T>& q2bar) {
  const V3<T> d1 = q1 - p1, d2 = q2 - p2, r = p1 - p2;
  const T a = dot(d1, d1), e = dot(d2, d2), b = dot(d1, d2), c = dot(d1, r), f = dot(d2, r);
  const T den = a * e - b * b;
  const bool den_ok = den > T(1e-12) * a * e;
  T t0 = T(0);
  bool t0_free = false;
  if (den_ok) { T raw = (b * f - c * e) / den; t0 = clamp01(raw); t0_free = raw > T(0) && raw < T(1); }
  const T u0 = (b * t0 + f) / e;
  T abar = T(0), ebar_ = T(0), bbar = T(0), cbar = T(0), fbar = T(0);
  if (u0 < T(0)) {
    const T raw = -c / a;
    if (raw > T(0) && raw < T(1)) { cbar -= tbar / a; abar -= tbar * raw / a; }
  } else if (u0 > T(1)) {
    const T raw = (b - c) / a;
    if (raw > T(0) && raw < T(1)) { bbar += tbar / a; cbar -= tbar / a; abar -= tbar * raw / a; }
  } else {
    bbar += ubar * t0 / e; fbar += ubar / e; ebar_ -= ubar * u0 / e;
    const T t0bar = tbar + ubar * b / e;
    if (t0_free) {
      const T nbar = t0bar / den, denbar = -t0bar * t0 / den;
      bbar += nbar * f - T(2) * denbar * b; fbar += nbar * b; cbar -= nbar * e; ebar_ += -nbar * c + denbar * a; abar += denbar * e;
    }
  }
  const V3<T> d1bar = (T(2) * abar) * d1 + bbar * d2 + cbar * r;
  const V3<T> d2bar = (T(2) * ebar_) * d2 + bbar * d1 + fbar * r;
  const V3<T> rbar = cbar * d1 + fbar * d2;
  p1bar += rbar - d1bar; q1bar += d1bar; p2bar += -rbar - d2bar; q2bar += d2bar;
}

}  // namespace dlo
#include "rod_adj2.cuh"
