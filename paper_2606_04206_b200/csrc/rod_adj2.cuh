// rod_adj2.cuh — adjoints of the contact / coupling operators (second half of rod_adj.cuh; same conventions).
#pragma once

namespace dlo {

// common tail of the two self-contact adjoints: given adjoints of the unit normal n = dv/|dv| (nbar), of
// del = |dv| (delbar), of the barycentric weights a0 = 1-t, t, b0 = 1-u, u, push everything to the four vertices
template <class T>
DLO_HD void contact_geometry_adj(const V3<T> x[4], T t, T u, const V3<T>& n, T del, const V3<T>& nbar, T delbar, T a0bar, T tbar,
                                 T b0bar, T ubar, V3<T> xbar[4]) {
  const V3<T> dvbar = (T(1) / del) * (nbar - dot(nbar, n) * n) + delbar * n;
  // ca = x0 + t (x1 - x0), cb = x2 + u (x3 - x2), dv = ca - cb
  xbar[0] += (T(1) - t) * dvbar; xbar[1] += t * dvbar; xbar[2] -= (T(1) - u) * dvbar; xbar[3] -= u * dvbar;
  const T tb = tbar - a0bar + dot(dvbar, x[1] - x[0]);
  const T ub = ubar - b0bar - dot(dvbar, x[3] - x[2]);
  closest_points_adj(x[0], x[1], x[2], x[3], tb, ub, xbar[0], xbar[1], xbar[2], xbar[3]);
}

// Eq.13 adjoint for one penetrating candidate: outbar[k] = adjoint of the correction of vertex k (= adjoint of
// dx after the pass), dbar_in = adjoint of D_p.  Accumulates into xbar[4] (adjoint of y of the four vertices).
// Returns false (nothing done) if the forward evaluation does not penetrate.
template <class T>
DLO_HD bool contact_adj(const V3<T> x[4], const T w[4], T rsum, const V3<T> outbar[4], T dbar_in, V3<T> xbar[4]) {
  T d, t, u, W;
  V3<T> n;
  if (!contact_eval(x, w, rsum, d, t, u, n, W)) return false;
  const T a0 = T(1) - t, b0 = T(1) - u, s = d / W;
  const T beta[4] = {w[0] * a0, w[1] * t, -w[2] * b0, -w[3] * u};
  V3<T> nbar = zero3<T>();
  T sbar = T(0), cb[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) { nbar += (s * beta[k]) * outbar[k]; cb[k] = dot(outbar[k], n); sbar += cb[k] * beta[k]; }
  T a0bar = cb[0] * s * w[0], tbar = cb[1] * s * w[1], b0bar = -cb[2] * s * w[2], ubar = -cb[3] * s * w[3];
  const T dbar = sbar / W + dbar_in, Wbar = -sbar * s / W;
  a0bar += Wbar * T(2) * w[0] * a0; tbar += Wbar * T(2) * w[1] * t; b0bar += Wbar * T(2) * w[2] * b0; ubar += Wbar * T(2) * w[3] * u;
  const T del = rsum - d;
  contact_geometry_adj(x, t, u, n, del, nbar, -dbar, a0bar, tbar, b0bar, ubar, xbar);
  return true;
}

// L410 friction adjoint for one candidate with D_p > 0 (forward: friction_pass in rod_substep.cuh).
// x: positions y, v: velocities v^2 of the four vertices; outbar[k] = adjoint of the velocity increment of vertex k.
// Accumulates xbar (positions), vbar (velocities v^2, the part through v_rel only), Dpbar.
template <class T>
DLO_HD bool friction_adj(const V3<T> x[4], const V3<T> v[4], const T w[4], T Dp, T mu_s, T inv_h, const V3<T> outbar[4],
                         V3<T> xbar[4], V3<T> vbar[4], T& Dpbar) {
  T t, u;
  closest_points(x[0], x[1], x[2], x[3], t, u);
  const V3<T> dv = axpy(x[0], t, x[1] - x[0]) - axpy(x[2], u, x[3] - x[2]);
  const T del = sqrt_(dot(dv, dv));
  const T a0 = T(1) - t, b0 = T(1) - u;
  const T W = w[0] * a0 * a0 + w[1] * t * t + w[2] * b0 * b0 + w[3] * u * u;
  if (!(del > T(1e-12)) || !(W > T(0))) return false;
  const V3<T> n = (T(1) / del) * dv;
  const V3<T> vrel = (a0 * v[0] + t * v[1]) - (b0 * v[2] + u * v[3]);
  const T vn = dot(vrel, n);
  const V3<T> vt = vrel - vn * n;
  const T vtn = sqrt_(dot(vt, vt));
  if (!(vtn > T(1e-12))) return false;
  const T cap = mu_s * Dp * inv_h;
  const bool capped = cap < vtn;
  const V3<T> that = (T(1) / vtn) * vt;
  const V3<T> D = capped ? (-cap) * that : -vt;
  const T iW = T(1) / W;
  const T coef[4] = {w[0] * a0 * iW, w[1] * t * iW, -w[2] * b0 * iW, -w[3] * u * iW};
  V3<T> Dbar = zero3<T>();
  T cb[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) { Dbar += coef[k] * outbar[k]; cb[k] = dot(outbar[k], D); }
  V3<T> vtbar;
  if (capped) {
    Dpbar += -dot(Dbar, that) * mu_s * inv_h;
    vtbar = (-cap / vtn) * (Dbar - dot(Dbar, that) * that);
  } else vtbar = -Dbar;
  const T vnbar = -dot(vtbar, n);
  V3<T> nbar = (-vn) * vtbar + vnbar * vrel;
  const V3<T> vrelbar = vtbar + vnbar * n;
  vbar[0] += a0 * vrelbar; vbar[1] += t * vrelbar; vbar[2] -= b0 * vrelbar; vbar[3] -= u * vrelbar;
  T a0bar = dot(vrelbar, v[0]) + cb[0] * w[0] * iW, tbar = dot(vrelbar, v[1]) + cb[1] * w[1] * iW;
  T b0bar = -dot(vrelbar, v[2]) - cb[2] * w[2] * iW, ubar = -dot(vrelbar, v[3]) - cb[3] * w[3] * iW;
  const T iWbar = cb[0] * w[0] * a0 + cb[1] * w[1] * t - cb[2] * w[2] * b0 - cb[3] * w[3] * u;
  const T Wbar = -iWbar * iW * iW;
  a0bar += Wbar * T(2) * w[0] * a0; tbar += Wbar * T(2) * w[1] * t; b0bar += Wbar * T(2) * w[2] * b0; ubar += Wbar * T(2) * w[3] * u;
  contact_geometry_adj(x, t, u, n, del, nbar, T(0), a0bar, tbar, b0bar, ubar, xbar);
  return true;
}

// L103 adjoint of rigid_response: v' = F(v, vb, n, d).  Given vpbar (adjoint of v'), accumulates vbar, vbbar,
// nbar and returns dbar.  Only call when the forward response was applied (it re-evaluates the same branches).
template <class T>
DLO_HD T rigid_response_adj(const V3<T>& v, const V3<T>& vb, const V3<T>& n, T d, T inv_eps, T e_rest, T mu, const V3<T>& vpbar,
                            V3<T>& vbar, V3<T>& vbbar, V3<T>& nbar) {
  T f = exp_(d * inv_eps);
  const bool sat = f > T(1);
  if (sat) f = T(1);
  const V3<T> u = v - vb;
  const T un = dot(u, n);
  const V3<T> ut = u - un * n;
  const T J = (T(1) + e_rest) * (-un);
  const T utn = sqrt_(dot(ut, ut));
  T k = T(0);
  bool slide = false;
  if (utn > T(1e-12)) { k = T(1) - mu * J / utn; slide = k > T(0); }
  const V3<T> utp = slide ? k * ut : zero3<T>();
  const V3<T> up = (-e_rest * un) * n + utp;
  // reverse
  vbar += vpbar;
  const T fbar = dot(vpbar, up - u);
  const V3<T> upbar = f * vpbar;
  V3<T> ubar = (-f) * vpbar;
  T unbar = -e_rest * dot(upbar, n);
  nbar += (-e_rest * un) * upbar;
  if (slide) {
    const T kbar = dot(upbar, ut);
    V3<T> utbar = k * upbar;
    const T Jbar = -kbar * mu / utn;
    const T utnbar = kbar * mu * J / (utn * utn);
    utbar += (utnbar / utn) * ut;
    unbar += -(T(1) + e_rest) * Jbar;
    ubar += utbar;
    unbar -= dot(utbar, n);
    nbar += (-un) * utbar;
  }
  ubar += unbar * n;
  nbar += unbar * u;
  vbar += ubar;
  vbbar -= ubar;
  return sat ? T(0) : fbar * f * inv_eps;
}

// capsule SDF adjoint: phi, n = sdf(a, b, R; y).  Given phibar, nbar: accumulates ybar, abar, bbar.
template <class T>
DLO_HD void sdf_capsule_adj(const V3<T>& a, const V3<T>& b, const V3<T>& y, T phibar, const V3<T>& nbar, V3<T>& ybar, V3<T>& abar,
                            V3<T>& bbar) {
  const V3<T> ab = b - a;
  const T den = dot(ab, ab), raw = dot(y - a, ab) / den, s = clamp01(raw);
  const V3<T> dv = y - axpy(a, s, ab);
  const T dist = sqrt_(dot(dv, dv));
  const V3<T> n = (T(1) / dist) * dv;
  const V3<T> dvbar = phibar * n + (T(1) / dist) * (nbar - dot(nbar, n) * n);
  ybar += dvbar;
  abar -= dvbar;
  V3<T> abbar = (-s) * dvbar;
  if (raw > T(0) && raw < T(1)) {
    const T sbar = -dot(dvbar, ab);
    const T numbar = sbar / den, denbar = -sbar * s / den;
    ybar += numbar * ab;
    abar -= numbar * ab;
    abbar += numbar * (y - a) + (T(2) * denbar) * ab;
  }
  bbar += abbar;
  abar -= abbar;
}

// adjoint w.r.t. y of the fixed primitives (plane, capsule, cylinder, box with pre-expanded rotation)
template <class T> DLO_HD void sdf_pre_adj(int type, const T* P, const V3<T>& y, T phibar, const V3<T>& nbar, V3<T>& ybar) {
  if (type == 0) { ybar += phibar * mk3<T>(P[0], P[1], P[2]); return; }
  if (type == 1) {
    V3<T> ab = zero3<T>(), bb = zero3<T>();
    sdf_capsule_adj(mk3<T>(P[0], P[1], P[2]), mk3<T>(P[3], P[4], P[5]), y, phibar, nbar, ybar, ab, bb);
    return;
  }
  if (type == 2) {
    const V3<T> ax = mk3<T>(P[3], P[4], P[5]), p = y - mk3<T>(P[0], P[1], P[2]);
    const T a = dot(p, ax);
    const V3<T> rv = p - a * ax;
    const T rho = sqrt_(dot(rv, rv));
    const T sgn = (a < T(0)) ? T(-1) : T(1);
    const T dr = rho - P[6], da = sgn * a - P[7];
    const bool radial_ok = rho > T(1e-12);
    const V3<T> er = radial_ok ? (T(1) / rho) * rv : zero3<T>();
    T drbar = T(0), dabar = T(0);
    V3<T> erbar = zero3<T>();
    const bool side = (dr <= T(0) && da <= T(0)) ? (dr > da) : (da <= T(0));
    const bool cap = (dr <= T(0) && da <= T(0)) ? !(dr > da) : (da > T(0) && dr <= T(0));
    if (side) { drbar = phibar; erbar = nbar; }
    else if (cap) { dabar = phibar; }
    else {   // rim
      const T phi = sqrt_(dr * dr + da * da);
      const T crbar = dot(nbar, er), czbar = sgn * dot(nbar, ax);
      erbar = (dr / phi) * nbar;
      const T phit = phibar - (crbar * dr + czbar * da) / (phi * phi);
      drbar = crbar / phi + phit * dr / phi;
      dabar = czbar / phi + phit * da / phi;
    }
    V3<T> rvbar = drbar * er;
    if (radial_ok) rvbar += (T(1) / rho) * (erbar - dot(erbar, er) * er);
    const T abar = sgn * dabar - dot(rvbar, ax);
    ybar += rvbar + abar * ax;
    return;
  }
  if (type == 3) {
    M3<T> R;
#pragma unroll
    for (int k = 0; k < 9; ++k) R.m[k] = P[6 + k];
    const V3<T> p = mulT(R, y - mk3<T>(P[0], P[1], P[2]));
    const T pc[3] = {p.x, p.y, p.z};
    T sg[3], q[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) { sg[k] = (pc[k] < T(0)) ? T(-1) : T(1); q[k] = sg[k] * pc[k] - P[3 + k]; }
    const V3<T> nlbar = mulT(R, nbar);
    const T nb[3] = {nlbar.x, nlbar.y, nlbar.z};
    T pb[3] = {T(0), T(0), T(0)};
    if (q[0] > T(0) || q[1] > T(0) || q[2] > T(0)) {
      T o[3], phi2 = T(0);
#pragma unroll
      for (int k = 0; k < 3; ++k) { o[k] = q[k] > T(0) ? q[k] : T(0); phi2 += o[k] * o[k]; }
      const T phi = sqrt_(phi2);
      T ub[3], udot = T(0);
#pragma unroll
      for (int k = 0; k < 3; ++k) { ub[k] = nb[k] * sg[k]; udot += ub[k] * o[k] / phi; }
#pragma unroll
      for (int k = 0; k < 3; ++k) if (q[k] > T(0)) pb[k] = sg[k] * (phibar * o[k] / phi + (ub[k] - udot * o[k] / phi) / phi);
    } else {
      int k = 0;
      T qk = q[0];
      if (q[1] > qk) { k = 1; qk = q[1]; }
      if (q[2] > qk) { k = 2; qk = q[2]; }
#pragma unroll
      for (int j = 0; j < 3; ++j) if (j == k) pb[j] = sg[j] * phibar;
    }
    ybar += mul(R, mk3<T>(pb[0], pb[1], pb[2]));
  }
}

// pose adjoint accumulator: adjoints of p (3) and of the rotation matrix R (9, row-major)
template <class T> struct PoseBar { V3<T> p; T R[9]; };
template <class T> DLO_HD void pose_bar_zero(PoseBar<T>& g) { g.p = zero3<T>(); for (int k = 0; k < 9; ++k) g.R[k] = T(0); }
// y = p + R q  ->  pbar += ybar, Rbar += ybar q^T
template <class T> DLO_HD void rigid_point_adj(const V3<T>& q, const V3<T>& ybar, PoseBar<T>& g) {
  g.p += ybar;
  g.R[0] += ybar.x * q.x; g.R[1] += ybar.x * q.y; g.R[2] += ybar.x * q.z;
  g.R[3] += ybar.y * q.x; g.R[4] += ybar.y * q.y; g.R[5] += ybar.y * q.z;
  g.R[6] += ybar.z * q.x; g.R[7] += ybar.z * q.y; g.R[8] += ybar.z * q.z;
}
// vb = inv_h (c - (p0 + R0 R1^T (c - p1)));  given vbbar: accumulates cbar and the two pose adjoints
template <class T>
DLO_HD void body_point_velocity_adj(const Pose<T>& g0, const Pose<T>& g1, const V3<T>& c, T inv_h, const V3<T>& vbbar, V3<T>& cbar,
                                    PoseBar<T>& b0, PoseBar<T>& b1) {
  const V3<T> rel = c - g1.p, local = mulT(g1.R, rel);
  cbar += inv_h * vbbar;
  const V3<T> beforebar = (-inv_h) * vbbar;
  rigid_point_adj(local, beforebar, b0);
  const V3<T> localbar = mulT(g0.R, beforebar);
  // local_j = sum_i R1[i][j] rel_i
  b1.R[0] += rel.x * localbar.x; b1.R[1] += rel.x * localbar.y; b1.R[2] += rel.x * localbar.z;
  b1.R[3] += rel.y * localbar.x; b1.R[4] += rel.y * localbar.y; b1.R[5] += rel.y * localbar.z;
  b1.R[6] += rel.z * localbar.x; b1.R[7] += rel.z * localbar.y; b1.R[8] += rel.z * localbar.z;
  const V3<T> relbar = mul(g1.R, localbar);
  cbar += relbar;
  b1.p -= relbar;
}

// Rodrigues adjoint: R = rodrigues(rho); given Rbar (9) returns rhobar
template <class T> DLO_HD V3<T> rodrigues_adj(const V3<T>& rho, const T* Rb) {
  const T th2 = dot(rho, rho);
  T A, B, dA, dB;
  if (th2 < T(1e-8)) { A = T(1) - th2 / T(6); B = T(0.5) - th2 / T(24); dA = T(-1) / T(6); dB = T(-1) / T(24); }
  else {
    const T th = sqrt_(th2);
    T s, c;
    sincos_(th, &s, &c);
    A = s / th; B = (T(1) - c) / th2;
    dA = (c - A) / (T(2) * th2); dB = (T(0.5) * A - B) / th2;
  }
  const T kx = rho.x, ky = rho.y, kz = rho.z;
  const T Abar = -kz * Rb[1] + ky * Rb[2] + kz * Rb[3] - kx * Rb[5] - ky * Rb[6] + kx * Rb[7];
  const T tr = Rb[0] + Rb[4] + Rb[8];
  const T Bbar = kx * kx * Rb[0] + ky * ky * Rb[4] + kz * kz * Rb[8] + kx * ky * (Rb[1] + Rb[3]) + kx * kz * (Rb[2] + Rb[6]) +
                 ky * kz * (Rb[5] + Rb[7]) - th2 * tr;
  V3<T> rb = A * mk3<T>(Rb[7] - Rb[5], Rb[2] - Rb[6], Rb[3] - Rb[1]);
  // through rho rho^T: B (Rb + Rb^T) rho
  rb += B * mk3<T>(T(2) * Rb[0] * kx + (Rb[1] + Rb[3]) * ky + (Rb[2] + Rb[6]) * kz,
                   (Rb[1] + Rb[3]) * kx + T(2) * Rb[4] * ky + (Rb[5] + Rb[7]) * kz,
                   (Rb[2] + Rb[6]) * kx + (Rb[5] + Rb[7]) * ky + T(2) * Rb[8] * kz);
  const T th2bar = Abar * dA + Bbar * dB - B * tr;
  rb += (T(2) * th2bar) * rho;
  return rb;
}

// pose = make_pose(a_prev, a_cur, tau): adjoint of (p, R) -> a_prev, a_cur
template <class T> DLO_HD void make_pose_adj(const T* a_prev, const T* a_cur, T tau, const PoseBar<T>& g, T* apbar, T* acbar) {
  T xi[6];
#pragma unroll
  for (int k = 0; k < 6; ++k) xi[k] = (T(1) - tau) * a_prev[k] + tau * a_cur[k];
  const V3<T> rb = rodrigues_adj(mk3<T>(xi[3], xi[4], xi[5]), g.R);
  const T xb[6] = {g.p.x, g.p.y, g.p.z, rb.x, rb.y, rb.z};
#pragma unroll
  for (int k = 0; k < 6; ++k) { apbar[k] += (T(1) - tau) * xb[k]; acbar[k] += tau * xb[k]; }
}

}  // namespace dlo
