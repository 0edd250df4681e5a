// ORACLE — TEST INFRASTRUCTURE ONLY.  Not part of the product path; shares no code with the CUDA library.
//
// Plain, slow, scalar implementation of ONE substep of the DLO-Lab rod time-step, written from PAPER.md
// (P:L<line>) in the order and notation of SURVEY.md Appendix A, which fixes the readings where the paper is
// silent (register: DESIGN.md section 3 / SURVEY.md Appendix B).  No blocking, fusion or reordering: one
// function per paper equation, called in the order of the substep.  `T` is `double` for values and `orc::AD`
// (tape.hpp) for derivatives; nothing else differs between the two instantiations.
//
//   Eq.1   state: vertices x_i, adapted frames (d1,d2,d3=t) per edge
//   Eq.2-3 stretching strain / energy (stretch mode 0)
//   Eq.4   curvature binormal
//   Eq.5   material curvature (component order as printed)
//   Eq.6-7 bending energy, isotropic B = alpha*I
//   Eq.10  inextensibility projection (+ XPBD compliance, reading B-8)
//   Eq.11  bending plasticity
//   Eq.12  loop holonomy / frame correction
//   Eq.13  segment-segment self-contact projection + Coulomb friction
//   rigid soft coupling f=min(exp(d/eps_s),1), threshold, restitution+friction
//   symplectic Euler, 5 substeps per frame
#pragma once
#include <cmath>
#include <cstdint>
#include <utility>
#include <vector>
#include "tape.hpp"

namespace orc {

using std::sqrt; using std::exp; using std::sin; using std::cos;

// ---------------------------------------------------------------------------------------------------------
// small vector algebra
template <class T> struct Vec3 { T x, y, z; };
template <class T> inline Vec3<T> mkv(const T& a, const T& b, const T& c) { Vec3<T> r; r.x = a; r.y = b; r.z = c; return r; }
template <class T> inline Vec3<T> operator+(const Vec3<T>& a, const Vec3<T>& b) { return mkv<T>(a.x + b.x, a.y + b.y, a.z + b.z); }
template <class T> inline Vec3<T> operator-(const Vec3<T>& a, const Vec3<T>& b) { return mkv<T>(a.x - b.x, a.y - b.y, a.z - b.z); }
template <class T> inline Vec3<T> operator-(const Vec3<T>& a) { return mkv<T>(-a.x, -a.y, -a.z); }
template <class T> inline Vec3<T> operator*(const T& s, const Vec3<T>& a) { return mkv<T>(s * a.x, s * a.y, s * a.z); }
template <class T> inline Vec3<T> operator*(const Vec3<T>& a, const T& s) { return mkv<T>(s * a.x, s * a.y, s * a.z); }
template <class T> inline T dot(const Vec3<T>& a, const Vec3<T>& b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
template <class T> inline Vec3<T> cross(const Vec3<T>& a, const Vec3<T>& b) {
  return mkv<T>(a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x);
}
template <class T> inline T norm(const Vec3<T>& a) { return sqrt(dot(a, a)); }
template <class T> inline Vec3<T> cst(const Vec3<double>& a) { return mkv<T>(T(a.x), T(a.y), T(a.z)); }
template <class T> inline Vec3<double> vval(const Vec3<T>& a) { return mkv<double>(val(a.x), val(a.y), val(a.z)); }
template <class T> inline Vec3<T> zero3() { return mkv<T>(T(0.0), T(0.0), T(0.0)); }
template <class T> struct Mat3 { T m[3][3]; };
template <class T> inline Vec3<T> mul(const Mat3<T>& R, const Vec3<T>& a) {
  return mkv<T>(R.m[0][0] * a.x + R.m[0][1] * a.y + R.m[0][2] * a.z,
                R.m[1][0] * a.x + R.m[1][1] * a.y + R.m[1][2] * a.z,
                R.m[2][0] * a.x + R.m[2][1] * a.y + R.m[2][2] * a.z);
}
template <class T> inline Vec3<T> mulT(const Mat3<T>& R, const Vec3<T>& a) {   // R^T a
  return mkv<T>(R.m[0][0] * a.x + R.m[1][0] * a.y + R.m[2][0] * a.z,
                R.m[0][1] * a.x + R.m[1][1] * a.y + R.m[2][1] * a.z,
                R.m[0][2] * a.x + R.m[1][2] * a.y + R.m[2][2] * a.z);
}

// ---------------------------------------------------------------------------------------------------------
// problem description
enum { TOPO_OPEN = 0, TOPO_RING = 1 };
enum { STRETCH_ENERGY = 0, STRETCH_PROJECT = 1 };
enum { PRIM_PLANE = 0, PRIM_CAPSULE = 1, PRIM_CYLINDER = 2, PRIM_BOX = 3 };
enum { KIN_FREE = 0, KIN_PINNED = 1, KIN_GRASPED = 2 };
static const int PRIM_NPARAM = 10;

struct Config {
  int N, topology, n_sub, N_C, stretch_mode, plasticity, self_contact, self_skip, G, n_grasp_max, K;
  int kappa_bar_from_x0;
  double dt, g[3], r, eps_s, f_thresh, e_rest;
  // Several DLOs in one env (P:L145 Separation, P:L155 Letter Art: Eq.13 acts between different ropes): the ropes
  // are laid back to back in the vertex array of an OPEN topology and cut[j] != 0 says that edge j (j, j+1) does not
  // exist.  Borrowed, [N], or null = one rope.  An absent edge carries no stretch / Eq.10 constraint, no frame and is no
  // self-contact segment; a vertex next to it is a rope END (no bending, no rest curvature).
  const uint8_t* cut;
  int E() const { return topology == TOPO_RING ? N : N - 1; }
};
inline bool edge_exists(const Config& c, int j) { return !(c.cut && c.cut[j]); }

// constants of one environment (never differentiated)
struct Scene {
  double m, l0, mu_r, mu_s;
  std::vector<int> kin;             // [N] KIN_*
  std::vector<int> grasp_g, grasp_k;// [N] gripper / slot of a grasped vertex
  std::vector<int> prim_type;       // [K]
  std::vector<double> prim_param;   // [K][10]
  std::vector<double> finger_geom;  // [G][4]: gap, length, radius, pad
  std::vector<int> grasp_vert;      // [G][n_grasp_max], -1 = none
  std::vector<Vec3<double>> q;      // [G][n_grasp_max] grasp-local coordinates (A0)
  std::vector<double> pose0;        // [G][6] a_{-1}: gripper pose before the first action
};

// the five differentiable material parameters (g_material order)
template <class T> struct Params { T stretch, alpha, gamma, sigma_y, r_c; };

template <class T> struct State {
  std::vector<Vec3<T>> x, v;   // [N]
  std::vector<Vec3<T>> d1;     // [E]
  std::vector<T> k1, k2;       // [N] rest curvature kappa_bar (used at interior vertices only)
};

// vertex/edge index helpers (open: edge j joins j,j+1; ring: j,(j+1) mod N)
inline int vnext(const Config& c, int i) { return (c.topology == TOPO_RING) ? (i + 1) % c.N : i + 1; }
inline int vprev(const Config& c, int i) { return (c.topology == TOPO_RING) ? (i + c.N - 1) % c.N : i - 1; }
inline bool interior(const Config& c, int i) {
  if (c.topology == TOPO_RING) return true;
  return i >= 1 && i <= c.N - 2 && edge_exists(c, i - 1) && edge_exists(c, i);
}

// ---------------------------------------------------------------------------------------------------------
// Rodrigues: R = exp([rho]x) (App. A step 1; series for |rho| < 1e-4)
template <class T> inline Mat3<T> rodrigues(const Vec3<T>& rho) {
  T th2 = dot(rho, rho);
  T A, B;
  if (val(th2) < 1e-8) { A = 1.0 - th2 / 6.0; B = 0.5 - th2 / 24.0; }
  else { T th = sqrt(th2); A = sin(th) / th; B = (1.0 - cos(th)) / th2; }
  Mat3<T> R;
  // K = [rho]x ; K^2 = rho rho^T - th2 I
  const T kx = rho.x, ky = rho.y, kz = rho.z;
  R.m[0][0] = 1.0 + B * (kx * kx - th2); R.m[0][1] = -A * kz + B * kx * ky;      R.m[0][2] = A * ky + B * kx * kz;
  R.m[1][0] = A * kz + B * kx * ky;      R.m[1][1] = 1.0 + B * (ky * ky - th2);  R.m[1][2] = -A * kx + B * ky * kz;
  R.m[2][0] = -A * ky + B * kx * kz;     R.m[2][1] = A * kx + B * ky * kz;       R.m[2][2] = 1.0 + B * (kz * kz - th2);
  return R;
}

// parallel transport of u from unit tangent a to unit tangent b (rotation-minimising; App. A0)
template <class T> inline Vec3<T> ptransport(const Vec3<T>& a, const Vec3<T>& b, const Vec3<T>& u) {
  Vec3<T> w = cross(a, b);
  T c = dot(a, b);
  return u + cross(w, u) + (T(1.0) / (1.0 + c)) * cross(w, cross(w, u));
}

// Eq.4: curvature binormal from the two unit tangents at an interior vertex
template <class T> inline Vec3<T> curvature_binormal(const Vec3<T>& ta, const Vec3<T>& tb) {
  T chi = 1.0 + dot(ta, tb);
  return (T(2.0) / chi) * cross(ta, tb);
}

// Eq.5 as printed: kappa_i = 1/2 sum_{j=i-1..i} ( kb.d2^j , kb.d1^j )
template <class T> inline void material_curvature(const Vec3<T>& ta, const Vec3<T>& tb, const Vec3<T>& d1a,
                                                  const Vec3<T>& d1b, T& k1, T& k2) {
  Vec3<T> kb = curvature_binormal(ta, tb);
  Vec3<T> d2a = cross(ta, d1a), d2b = cross(tb, d1b);
  Vec3<T> m1 = T(0.5) * (d1a + d1b), m2 = T(0.5) * (d2a + d2b);
  k1 = dot(kb, m2);
  k2 = dot(kb, m1);
}

// ---------------------------------------------------------------------------------------------------------
// A0 frame initialisation (space-parallel transport from edge 0; ring: Eq.12 holonomy correction)
inline void frames_init(const Config& c, const std::vector<Vec3<double>>& x, std::vector<Vec3<double>>& d1,
                        double* psiH_out) {
  const int E = c.E();
  std::vector<Vec3<double>> t(E);
  for (int j = 0; j < E; ++j) { Vec3<double> e = x[vnext(c, j)] - x[j]; t[j] = (1.0 / norm(e)) * e; }
  d1.assign(E, zero3<double>());
  Vec3<double> zhat = mkv(0.0, 0.0, 1.0), yhat = mkv(0.0, 1.0, 0.0);
  bool first = true;                                  // the first edge of every rope starts a chain of its own
  for (int j = 0; j < E; ++j) {
    if (!edge_exists(c, j)) { first = true; continue; }   // absent edge: no frame (left at zero)
    if (first) {
      Vec3<double> ref = (norm(cross(t[j], zhat)) < 1e-6) ? yhat : zhat;
      Vec3<double> u = ref - dot(ref, t[j]) * t[j];
      d1[j] = (1.0 / norm(u)) * u;
      first = false;
    } else d1[j] = ptransport(t[j - 1], t[j], d1[j - 1]);
  }
  double psiH = 0.0;
  if (c.topology == TOPO_RING) {
    Vec3<double> uu = ptransport(t[E - 1], t[0], d1[E - 1]);     // transported once around the loop
    psiH = std::atan2(dot(cross(d1[0], uu), t[0]), dot(d1[0], uu));
    for (int j = 0; j < E; ++j) {                                  // Eq.12 with phi^j = -psiH * j / E (0-based)
      double phi = -psiH * double(j) / double(E);
      Vec3<double> d2 = cross(t[j], d1[j]);
      d1[j] = std::cos(phi) * d1[j] + std::sin(phi) * d2;
    }
  }
  if (psiH_out) *psiH_out = psiH;
}

// ---------------------------------------------------------------------------------------------------------
// Eq.6-7 bending energy (isotropic B_i = alpha I), l_bar = Voronoi length (uniform l0 here)
template <class T>
T bend_energy(const Config& c, const std::vector<Vec3<T>>& x, const std::vector<Vec3<T>>& d1,
              const std::vector<T>& k1b, const std::vector<T>& k2b, const T& alpha, double lbar) {
  T U = T(0.0);
  for (int i = 0; i < c.N; ++i) {
    if (!interior(c, i)) continue;
    int a = vprev(c, i), b = i;                       // edge before / after vertex i
    Vec3<T> ea = x[i] - x[vprev(c, i)], eb = x[vnext(c, i)] - x[i];
    Vec3<T> ta = (T(1.0) / norm(ea)) * ea, tb = (T(1.0) / norm(eb)) * eb;
    T k1, k2; material_curvature(ta, tb, d1[a], d1[b], k1, k2);
    T dk1 = k1 - k1b[i], dk2 = k2 - k2b[i];
    U += alpha / (2.0 * lbar) * (dk1 * dk1 + dk2 * dk2);
  }
  return U;
}

// -dU_b/dx with the frames held fixed (App. A step 2, reading B-5); adds into f
template <class T>
void bend_force(const Config& c, const std::vector<Vec3<T>>& x, const std::vector<Vec3<T>>& d1,
                const std::vector<T>& k1b, const std::vector<T>& k2b, const T& alpha, double lbar,
                std::vector<Vec3<T>>& f) {
  for (int i = 0; i < c.N; ++i) {
    if (!interior(c, i)) continue;
    int ip = vprev(c, i), in = vnext(c, i), a = ip, b = i;
    Vec3<T> ea = x[i] - x[ip], eb = x[in] - x[i];
    T La = norm(ea), Lb = norm(eb);
    Vec3<T> ta = (T(1.0) / La) * ea, tb = (T(1.0) / Lb) * eb;
    T chi = 1.0 + dot(ta, tb);
    Vec3<T> kb = (T(2.0) / chi) * cross(ta, tb);                        // Eq.4
    Vec3<T> d2a = cross(ta, d1[a]), d2b = cross(tb, d1[b]);
    Vec3<T> m1 = T(0.5) * (d1[a] + d1[b]), m2 = T(0.5) * (d2a + d2b);
    T dk1 = dot(kb, m2) - k1b[i], dk2 = dot(kb, m1) - k2b[i];           // Eq.5 minus rest curvature
    Vec3<T> q = dk1 * m2 + dk2 * m1;
    T qkb = dot(q, kb);
    Vec3<T> Aa = (T(1.0) / chi) * (T(2.0) * cross(tb, q) - qkb * tb);
    Vec3<T> Ab = (T(1.0) / chi) * (T(2.0) * cross(q, ta) - qkb * ta);
    T s = alpha / lbar;
    Vec3<T> Ga = (s / La) * (Aa - dot(Aa, ta) * ta);
    Vec3<T> Gb = (s / Lb) * (Ab - dot(Ab, tb) * tb);
    // dU/dx_{i-1} = -Ga ; dU/dx_i = Ga - Gb ; dU/dx_{i+1} = Gb ;  f -= dU/dx
    f[ip] = f[ip] + Ga;
    f[i] = f[i] - Ga + Gb;
    f[in] = f[in] - Gb;
  }
}

// Eq.2-3 stretching energy and force (stretch mode 0): U_s = 1/2 sum k_s eps^2 l0
template <class T>
T stretch_energy(const Config& c, const std::vector<Vec3<T>>& x, const T& ks, double l0) {
  T U = T(0.0);
  for (int j = 0; j < c.E(); ++j) {
    if (!edge_exists(c, j)) continue;
    T eps = norm(x[vnext(c, j)] - x[j]) / l0 - 1.0;
    U += 0.5 * ks * eps * eps * l0;
  }
  return U;
}
template <class T>
void stretch_force(const Config& c, const std::vector<Vec3<T>>& x, const T& ks, double l0, std::vector<Vec3<T>>& f) {
  for (int j = 0; j < c.E(); ++j) {
    if (!edge_exists(c, j)) continue;
    int jn = vnext(c, j);
    Vec3<T> e = x[jn] - x[j];
    T L = norm(e);
    Vec3<T> t = (T(1.0) / L) * e;
    T eps = L / l0 - 1.0;
    f[j] = f[j] + (ks * eps) * t;
    f[jn] = f[jn] - (ks * eps) * t;
  }
}

// ---------------------------------------------------------------------------------------------------------
// DIAGNOSTICS ONLY (no arithmetic of the step depends on them): how close the trajectory comes to each branch of the
// piecewise-smooth step, as the smallest relative distance to the threshold seen since the recorder was armed.  The
// gradient of the step jumps where a branch flips (reading B-22: branches frozen at their forward outcome), so a test
// that compares gradients needs to know when a trajectory runs along such a threshold.
enum { MG_APPROACH = 0 /* |u_n| / |u| at the test u_n < 0 of a vertex inside the influence distance (L103) */,
       MG_STICK /* |k| at the Coulomb stick / slide switch k > 0 of the soft coupling */,
       MG_FKINK /* d / eps_s >= 0 on the saturated side of the kink of f = min(exp(d / eps_s), 1) */,
       MG_FTHRESH /* |f - f_thresh| / f_thresh at the influence threshold (a jump of the VALUE, L103 "if f > 0.1") */,
       MG_YIELD /* | |kappa_el| - Y | / Y at the Eq.11 yield test */,
       MG_CONTACT /* |d| / (r_a + r_b) at the Eq.13 penetration test d > 0 of a candidate pair */,
       MG_FRICTION /* |mu_s D_p / h - |v_t|| / |v_t| at the clamp of the self-contact friction (L410) */,
       MG_COUNT };
inline double*& margin_sink() { static thread_local double* p = nullptr; return p; }
inline void note_margin(int cls, double rel) { double* m = margin_sink(); if (m && rel == rel && rel < m[cls]) m[cls] = rel; }

// ---------------------------------------------------------------------------------------------------------
// Eq.10 with XPBD compliance (reading B-8): one edge, in place on the correction accumulators.
// e = current edge vector (x^p_{j+1}-x^p_j)+(dx_{j+1}-dx_j); atil = c/h^2 (0 => Eq.10 verbatim).
template <class T>
inline void project_edge(const Vec3<T>& e, double wj, double wj1, double l0, const T& atil, T& S, Vec3<T>& dxj, Vec3<T>& dxj1) {
  if (wj == 0.0 && wj1 == 0.0) return;
  T L = norm(e);
  Vec3<T> t = (T(1.0) / L) * e;
  T C = L - l0;
  T lam = (C - atil * S) / (wj + wj1 + atil);
  S += lam;
  dxj = dxj + (lam * wj) * t;
  dxj1 = dxj1 - (lam * wj1) * t;
}

// closest points of two segments, rule B-14
template <class T>
inline void closest_points(const Vec3<T>& p1, const Vec3<T>& q1, const Vec3<T>& p2, const Vec3<T>& q2, T& t, T& u) {
  Vec3<T> d1 = q1 - p1, d2 = q2 - p2, r = p1 - p2;
  T a = dot(d1, d1), e = dot(d2, d2), b = dot(d1, d2), c = dot(d1, r), f = dot(d2, r);
  T den = a * e - b * b;
  auto clamp01 = [](const T& s) { if (s < 0.0) return T(0.0); if (s > 1.0) return T(1.0); return s; };
  if (val(den) > 1e-12 * val(a) * val(e)) t = clamp01((b * f - c * e) / den); else t = T(0.0);
  u = (b * t + f) / e;
  if (u < 0.0) { u = T(0.0); t = clamp01(-c / a); }
  else if (u > 1.0) { u = T(1.0); t = clamp01((b - c) / a); }
}

// Eq.13 (denominator typo fixed: readings B-12/B-13).  Returns false if not penetrating.
// x: the four vertices (i,i+1,j,j+1); w: inverse masses; rsum = r_a+r_b.  out[4] corrections, depth d.
template <class T>
inline bool self_contact_correction(const Vec3<T> x[4], const double w[4], double rsum, Vec3<T> out[4], T& d,
                                    T& t, T& u, Vec3<T>& n, T& W) {
  closest_points(x[0], x[1], x[2], x[3], t, u);
  Vec3<T> ca = (1.0 - t) * x[0] + t * x[1], cb = (1.0 - u) * x[2] + u * x[3];
  Vec3<T> dv = ca - cb;
  T delta = norm(dv);
  d = rsum - delta;
  note_margin(MG_CONTACT, std::fabs(val(d)) / rsum);
  if (!(d > 0.0) || !(delta > 1e-12)) return false;
  n = (T(1.0) / delta) * dv;
  W = w[0] * (1.0 - t) * (1.0 - t) + w[1] * t * t + w[2] * (1.0 - u) * (1.0 - u) + w[3] * u * u;
  if (!(val(W) > 0.0)) return false;
  out[0] = (d * w[0] * (1.0 - t) / W) * n;
  out[1] = (d * w[1] * t / W) * n;
  out[2] = -((d * w[2] * (1.0 - u) / W) * n);
  out[3] = -((d * w[3] * u / W) * n);
  return true;
}

// Eq.11: plastic update of the rest curvature; Y = sigma_y * l_bar (reading B-21)
template <class T>
inline void plasticity_update(const T& k1, const T& k2, T& k1b, T& k2b, const T& Y, const T& r_c) {
  T e1 = k1 - k1b, e2 = k2 - k2b;
  T n = sqrt(e1 * e1 + e2 * e2);
  note_margin(MG_YIELD, std::fabs(val(n) - val(Y)) / val(Y));
  if (n > Y) {
    T s = r_c * (n - Y) / n;
    k1b += s * e1;
    k2b += s * e2;
  }
}

// ---------------------------------------------------------------------------------------------------------
// analytic signed distance + gradient of the rigid primitives (reading B-18).  Returns false where the
// gradient is undefined (point on an axis / segment), in which case the primitive is skipped for that vertex.
template <class T>
inline bool sdf(int type, const T* P, const Vec3<T>& y, T& phi, Vec3<T>& n) {
  if (type == PRIM_PLANE) {                       // P = n(3), o : phi = n.y - o
    n = mkv<T>(P[0], P[1], P[2]);
    phi = dot(n, y) - P[3];
    return true;
  }
  if (type == PRIM_CAPSULE) {                     // P = a(3), b(3), R
    Vec3<T> a = mkv<T>(P[0], P[1], P[2]), b = mkv<T>(P[3], P[4], P[5]);
    Vec3<T> ab = b - a;
    T s = dot(y - a, ab) / dot(ab, ab);
    if (s < 0.0) s = T(0.0); else if (s > 1.0) s = T(1.0);
    Vec3<T> dv = y - (a + s * ab);
    T dist = norm(dv);
    if (!(dist > 1e-12)) return false;
    phi = dist - P[6];
    n = (T(1.0) / dist) * dv;
    return true;
  }
  if (type == PRIM_CYLINDER) {                    // P = centre(3), unit axis(3), R, half-height
    Vec3<T> c = mkv<T>(P[0], P[1], P[2]), ax = mkv<T>(P[3], P[4], P[5]);
    Vec3<T> p = y - c;
    T a = dot(p, ax);
    Vec3<T> rv = p - a * ax;
    T rho = norm(rv);
    T sgn = (a < 0.0) ? T(-1.0) : T(1.0);
    T absa = sgn * a;
    T dr = rho - P[6], da = absa - P[7];
    bool radial_ok = rho > 1e-12;
    Vec3<T> er = radial_ok ? (T(1.0) / rho) * rv : zero3<T>();
    if (dr <= 0.0 && da <= 0.0) {                 // inside: nearest face
      if (dr > da) { if (!radial_ok) return false; phi = dr; n = er; }
      else { phi = da; n = sgn * ax; }
    } else if (da <= 0.0) { if (!radial_ok) return false; phi = dr; n = er; }        // beside the side wall
    else if (dr <= 0.0) { phi = da; n = sgn * ax; }                                  // above / below a cap
    else {                                                                           // nearest point on a rim
      phi = sqrt(dr * dr + da * da);
      n = (dr / phi) * er + ((da / phi) * sgn) * ax;
    }
    return true;
  }
  if (type == PRIM_BOX) {                         // P = centre(3), half extents(3), rotation vector(3)
    Vec3<T> c = mkv<T>(P[0], P[1], P[2]);
    Mat3<T> R = rodrigues(mkv<T>(P[6], P[7], P[8]));
    Vec3<T> p = mulT(R, y - c);
    T pc[3] = {p.x, p.y, p.z}, sg[3], q[3];
    for (int k = 0; k < 3; ++k) { sg[k] = (pc[k] < 0.0) ? T(-1.0) : T(1.0); q[k] = sg[k] * pc[k] - P[3 + k]; }
    Vec3<T> nl;
    if (q[0] > 0.0 || q[1] > 0.0 || q[2] > 0.0) {  // outside: distance to the clamped point
      T o[3];
      for (int k = 0; k < 3; ++k) o[k] = (q[k] > 0.0) ? q[k] : T(0.0);
      phi = sqrt(o[0] * o[0] + o[1] * o[1] + o[2] * o[2]);
      nl = mkv<T>(sg[0] * o[0] / phi, sg[1] * o[1] / phi, sg[2] * o[2] / phi);
    } else {                                      // inside: nearest face (first maximum in x,y,z order)
      int k = 0;
      if (q[1] > q[k]) k = 1;
      if (q[2] > q[k]) k = 2;
      phi = q[k];
      nl = zero3<T>();
      if (k == 0) nl.x = sg[0]; else if (k == 1) nl.y = sg[1]; else nl.z = sg[2];
    }
    n = mul(R, nl);
    return true;
  }
  return false;
}

// P:L103 soft coupling response of one sampled position against one primitive (App. A step 7, reading B-17).
// v: running vertex velocity (updated in place); vb: velocity of the body point; d = r - phi.
template <class T>
inline void rigid_response(Vec3<T>& v, const Vec3<T>& vb, const Vec3<T>& n, const T& d, double eps_s,
                           double f_thresh, double e_rest, double mu) {
  T f = exp(d / eps_s);
  note_margin(MG_FTHRESH, std::fabs(val(f) - f_thresh) / f_thresh);
  if (f > 1.0) f = T(1.0);
  if (!(f > f_thresh)) return;
  Vec3<T> u = v - vb;
  T un = dot(u, n);
  note_margin(MG_APPROACH, std::fabs(val(un)) / (std::sqrt(val(dot(u, u))) + 1e-300));
  if (!(un < 0.0)) return;
  if (val(d) >= 0.0) note_margin(MG_FKINK, val(d) / eps_s);   // saturated side only: from below the response is smooth up to the kink
  Vec3<T> ut = u - un * n;
  T J = (1.0 + e_rest) * (-un);
  T utn = norm(ut);
  Vec3<T> utp = zero3<T>();
  if (utn > 1e-12) {
    T k = 1.0 - mu * J / utn;
    if (mu > 0.0) note_margin(MG_STICK, std::fabs(val(k)));
    if (k > 0.0) utp = k * ut;
  }
  Vec3<T> up = (-e_rest * un) * n + utp;
  v = v + f * (up - u);
}

// ---------------------------------------------------------------------------------------------------------
// one gripper at one normalised time tau in [0,1] of the current step (App. A step 1, readings B-19/B-20)
template <class T> struct GripperPose { Vec3<T> p; Mat3<T> R; };
template <class T>
inline GripperPose<T> gripper_pose(const T* a_prev, const T* a_cur, double tau) {
  T xi[6];
  for (int k = 0; k < 6; ++k) xi[k] = (1.0 - tau) * a_prev[k] + tau * a_cur[k];
  GripperPose<T> gp;
  gp.p = mkv<T>(xi[0], xi[1], xi[2]);
  gp.R = rodrigues(mkv<T>(xi[3], xi[4], xi[5]));
  return gp;
}
// velocity of the body point that sits at world position c at time tau (finite difference over the substep)
template <class T>
inline Vec3<T> body_point_velocity(const GripperPose<T>& g0, const GripperPose<T>& g1, const Vec3<T>& c, double h) {
  Vec3<T> local = mulT(g1.R, c - g1.p);
  Vec3<T> before = g0.p + mul(g0.R, local);
  return (T(1.0) / h) * (c - before);
}

// ---------------------------------------------------------------------------------------------------------
template <class T> struct Work {
  std::vector<Vec3<T>> f, v1, xp, dx, acc, t_old;
  std::vector<T> S, Dp;
  std::vector<std::pair<int, int>> cand;
};

inline int cyclic_edge_distance(const Config& c, int a, int b) {
  int d = b - a;
  if (c.topology == TOPO_RING) { int E = c.E(); if (E - d < d) d = E - d; }
  return d;
}

// ONE substep s (0-based) of step t: App. A steps 1-9.  a_prev = a_{t-1}, a_cur = a_t, each [G][6].
template <class T>
void substep(const Config& c, const Scene& sc, const Params<T>& pm, State<T>& st, const T* a_prev, const T* a_cur,
             int s, Work<T>& w) {
  const int N = c.N, E = c.E(), G = c.G;
  const double h = c.dt / c.n_sub, m = sc.m, l0 = sc.l0, lbar = sc.l0;
  const double tau0 = double(s) / c.n_sub, tau1 = double(s + 1) / c.n_sub;
  std::vector<double> winv(N);
  for (int i = 0; i < N; ++i) winv[i] = (sc.kin[i] == KIN_FREE) ? 1.0 / m : 0.0;

  // -- 1. bodies (A1): gripper poses at substep start and end, grasp targets
  std::vector<GripperPose<T>> gp0(G), gp1(G);
  for (int g = 0; g < G; ++g) {
    gp0[g] = gripper_pose(a_prev + 6 * g, a_cur + 6 * g, tau0);
    gp1[g] = gripper_pose(a_prev + 6 * g, a_cur + 6 * g, tau1);
  }
  auto grasp_target = [&](int i) {
    int g = sc.grasp_g[i], k = sc.grasp_k[i];
    return gp1[g].p + mul(gp1[g].R, cst<T>(sc.q[g * c.n_grasp_max + k]));
  };

  // -- 2. forces (A2): gravity, stretch energy (mode 0), bending
  w.f.assign(N, zero3<T>());
  for (int i = 0; i < N; ++i) w.f[i] = mkv<T>(T(m * c.g[0]), T(m * c.g[1]), T(m * c.g[2]));
  if (c.stretch_mode == STRETCH_ENERGY) stretch_force(c, st.x, pm.stretch, l0, w.f);
  bend_force(c, st.x, st.d1, st.k1, st.k2, pm.alpha, lbar, w.f);

  // -- 3. velocity (A3): symplectic Euler with implicit viscous damping (reading B-7)
  w.v1.assign(N, zero3<T>());
  for (int i = 0; i < N; ++i) {
    if (sc.kin[i] == KIN_FREE) w.v1[i] = (T(1.0) / (1.0 + pm.gamma * h)) * (st.v[i] + (T(h / m)) * w.f[i]);
    else if (sc.kin[i] == KIN_PINNED) w.v1[i] = zero3<T>();
    else w.v1[i] = (T(1.0) / h) * (grasp_target(i) - st.x[i]);
  }

  // -- 4. predict (A4)
  w.xp.assign(N, zero3<T>());
  w.dx.assign(N, zero3<T>());
  w.S.assign(E, T(0.0));
  for (int i = 0; i < N; ++i) w.xp[i] = st.x[i] + T(h) * w.v1[i];
  w.cand.clear();
  if (c.self_contact) {
    const double rsum = 2.0 * c.r;
    for (int a = 0; a < E; ++a)
      for (int b = a + 1; b < E; ++b) {
        if (cyclic_edge_distance(c, a, b) < c.self_skip) continue;
        if (!edge_exists(c, a) || !edge_exists(c, b)) continue;
        Vec3<double> p1 = vval(w.xp[a]), q1 = vval(w.xp[vnext(c, a)]), p2 = vval(w.xp[b]), q2 = vval(w.xp[vnext(c, b)]);
        double t, u; closest_points(p1, q1, p2, q2, t, u);
        Vec3<double> dv = ((1.0 - t) * p1 + t * q1) - ((1.0 - u) * p2 + u * q2);
        if (norm(dv) < 2.0 * rsum) w.cand.push_back(std::make_pair(a, b));
      }
  }
  w.Dp.assign(w.cand.size(), T(0.0));

  // -- 5. projection loop (A5)
  auto ycur = [&](int i) { return w.xp[i] + w.dx[i]; };
  auto edge_vec = [&](int j) { int jn = vnext(c, j); return (w.xp[jn] - w.xp[j]) + (w.dx[jn] - w.dx[j]); };
  const bool odd_ring = (c.topology == TOPO_RING) && (E % 2 == 1);
  for (int it = 0; it < c.N_C; ++it) {
    if (c.stretch_mode == STRETCH_PROJECT) {
      T atil = pm.stretch / (h * h);
      for (int colour = 0; colour < 3; ++colour) {
        for (int j = 0; j < E; ++j) {
          int col_j = (odd_ring && j == E - 1) ? 2 : (j & 1);
          if (col_j != colour || !edge_exists(c, j)) continue;
          int jn = vnext(c, j);
          project_edge(edge_vec(j), winv[j], winv[jn], l0, atil, w.S[j], w.dx[j], w.dx[jn]);
        }
      }
    }
    if (c.self_contact && !w.cand.empty()) {     // Jacobi pass: all corrections from the same y, summed
      w.acc.assign(N, zero3<T>());
      const double rsum = 2.0 * c.r;
      for (size_t p = 0; p < w.cand.size(); ++p) {
        int a = w.cand[p].first, b = w.cand[p].second;
        int iv[4] = {a, vnext(c, a), b, vnext(c, b)};
        Vec3<T> xs[4] = {ycur(iv[0]), ycur(iv[1]), ycur(iv[2]), ycur(iv[3])};
        double ws[4] = {winv[iv[0]], winv[iv[1]], winv[iv[2]], winv[iv[3]]};
        Vec3<T> out[4], n; T d, t, u, W;
        if (!self_contact_correction(xs, ws, rsum, out, d, t, u, n, W)) continue;
        for (int k = 0; k < 4; ++k) w.acc[iv[k]] = w.acc[iv[k]] + out[k];
        w.Dp[p] += d;
      }
      for (int i = 0; i < N; ++i) w.dx[i] = w.dx[i] + w.acc[i];
    }
  }

  // -- 6. reconcile velocities with the projected positions + self-contact friction (A6)
  std::vector<Vec3<T>>& vel = w.v1;     // from here on w.v1 holds v^2, v^3, v^4 in turn
  for (int i = 0; i < N; ++i)
    if (sc.kin[i] == KIN_FREE) vel[i] = vel[i] + (T(1.0) / h) * w.dx[i];
  if (c.self_contact && !w.cand.empty()) {
    w.acc.assign(N, zero3<T>());
    for (size_t p = 0; p < w.cand.size(); ++p) {
      if (!(w.Dp[p] > 0.0)) continue;
      int a = w.cand[p].first, b = w.cand[p].second;
      int iv[4] = {a, vnext(c, a), b, vnext(c, b)};
      Vec3<T> xs[4] = {ycur(iv[0]), ycur(iv[1]), ycur(iv[2]), ycur(iv[3])};
      double ws[4] = {winv[iv[0]], winv[iv[1]], winv[iv[2]], winv[iv[3]]};
      T t, u; closest_points(xs[0], xs[1], xs[2], xs[3], t, u);
      Vec3<T> dv = ((1.0 - t) * xs[0] + t * xs[1]) - ((1.0 - u) * xs[2] + u * xs[3]);
      T delta = norm(dv);
      if (!(delta > 1e-12)) continue;
      Vec3<T> n = (T(1.0) / delta) * dv;
      T W = ws[0] * (1.0 - t) * (1.0 - t) + ws[1] * t * t + ws[2] * (1.0 - u) * (1.0 - u) + ws[3] * u * u;
      if (!(val(W) > 0.0)) continue;
      Vec3<T> vrel = ((1.0 - t) * vel[iv[0]] + t * vel[iv[1]]) - ((1.0 - u) * vel[iv[2]] + u * vel[iv[3]]);
      Vec3<T> vt = vrel - dot(vrel, n) * n;
      T vtn = norm(vt);
      if (!(vtn > 1e-12)) continue;
      T cap = sc.mu_s * w.Dp[p] / h;
      note_margin(MG_FRICTION, std::fabs(val(cap) - val(vtn)) / val(vtn));
      T mag = (cap < vtn) ? cap : vtn;
      Vec3<T> D = (-(mag / vtn)) * vt;
      w.acc[iv[0]] = w.acc[iv[0]] + (ws[0] * (1.0 - t) / W) * D;
      w.acc[iv[1]] = w.acc[iv[1]] + (ws[1] * t / W) * D;
      w.acc[iv[2]] = w.acc[iv[2]] - (ws[2] * (1.0 - u) / W) * D;
      w.acc[iv[3]] = w.acc[iv[3]] - (ws[3] * u / W) * D;
    }
    for (int i = 0; i < N; ++i)
      if (sc.kin[i] == KIN_FREE) vel[i] = vel[i] + w.acc[i];
  }

  // -- 7. rigid soft coupling (A7): user primitives in index order, then finger capsules g0f0,g0f1,g1f0,...
  for (int i = 0; i < N; ++i) {
    if (sc.kin[i] != KIN_FREE) continue;
    Vec3<T> y = ycur(i);
    for (int k = 0; k < c.K; ++k) {
      T P[PRIM_NPARAM];
      for (int q = 0; q < PRIM_NPARAM; ++q) P[q] = T(sc.prim_param[k * PRIM_NPARAM + q]);
      T phi; Vec3<T> n;
      if (!sdf(sc.prim_type[k], P, y, phi, n)) continue;
      rigid_response(vel[i], zero3<T>(), n, T(c.r) - phi, c.eps_s, c.f_thresh, c.e_rest, sc.mu_r);
    }
    for (int g = 0; g < G; ++g) {
      const double gap = sc.finger_geom[4 * g + 0], len = sc.finger_geom[4 * g + 1], rf = sc.finger_geom[4 * g + 2];
      for (int fk = 0; fk < 2; ++fk) {
        double sx = (fk == 0 ? 0.5 : -0.5) * gap;
        Vec3<T> A = gp1[g].p + mul(gp1[g].R, mkv<T>(T(sx), T(0.0), T(0.0)));
        Vec3<T> B = gp1[g].p + mul(gp1[g].R, mkv<T>(T(sx), T(0.0), T(len)));
        T P[PRIM_NPARAM] = {A.x, A.y, A.z, B.x, B.y, B.z, T(rf), T(0.0), T(0.0), T(0.0)};
        T phi; Vec3<T> n;
        if (!sdf(PRIM_CAPSULE, P, y, phi, n)) continue;
        Vec3<T> vb = body_point_velocity(gp0[g], gp1[g], y, h);
        rigid_response(vel[i], vb, n, T(c.r) - phi, c.eps_s, c.f_thresh, c.e_rest, sc.mu_r);
      }
    }
  }

  // -- 8. commit (A8)
  w.t_old.assign(E, zero3<T>());
  for (int j = 0; j < E; ++j) {
    if (!edge_exists(c, j)) continue;
    Vec3<T> e = st.x[vnext(c, j)] - st.x[j]; w.t_old[j] = (T(1.0) / norm(e)) * e;
  }
  for (int i = 0; i < N; ++i) {
    if (sc.kin[i] == KIN_FREE) { st.x[i] = st.x[i] + T(h) * vel[i]; st.v[i] = vel[i]; }
    else if (sc.kin[i] == KIN_PINNED) { st.v[i] = zero3<T>(); }
    else { st.x[i] = grasp_target(i); st.v[i] = vel[i]; }
  }

  // -- 9. frames (time-parallel transport, reading B-4) + plasticity (Eq.11)
  for (int j = 0; j < E; ++j) {
    if (!edge_exists(c, j)) continue;
    Vec3<T> e = st.x[vnext(c, j)] - st.x[j];
    Vec3<T> tn = (T(1.0) / norm(e)) * e;
    Vec3<T> d = ptransport(w.t_old[j], tn, st.d1[j]);
    d = d - dot(d, tn) * tn;
    st.d1[j] = (T(1.0) / norm(d)) * d;
  }
  if (c.plasticity) {
    for (int i = 0; i < N; ++i) {
      if (!interior(c, i)) continue;
      int ip = vprev(c, i), in = vnext(c, i);
      Vec3<T> ea = st.x[i] - st.x[ip], eb = st.x[in] - st.x[i];
      Vec3<T> ta = (T(1.0) / norm(ea)) * ea, tb = (T(1.0) / norm(eb)) * eb;
      T k1, k2; material_curvature(ta, tb, st.d1[ip], st.d1[i], k1, k2);
      T Y = pm.sigma_y * lbar;
      plasticity_update(k1, k2, st.k1[i], st.k2[i], Y, pm.r_c);
    }
  }
}

// one env-step = n_sub substeps
template <class T>
void step(const Config& c, const Scene& sc, const Params<T>& pm, State<T>& st, const T* a_prev, const T* a_cur, Work<T>& w) {
  for (int s = 0; s < c.n_sub; ++s) substep(c, sc, pm, st, a_prev, a_cur, s, w);
}

}  // namespace orc
