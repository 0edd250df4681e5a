// rod_ops.cuh — per-element operators of the rod step (forward values), written from PAPER.md.
//
// Each function is one equation of the paper applied to ONE element (an edge, an interior vertex, a segment
// pair, a vertex/primitive pair); the warp kernels in rod_kernels.cu own the data movement between lanes.
// Everything is `T`-generic and host/device so that tests/ can compile this header with g++ in double and
// check every operator (and its hand-written adjoint in rod_adj.cuh) against finite differences on the CPU.
// The GPU only ever instantiates T = float.
//
//   Eq.4   curvature binormal
//   Eq.5   material curvature (as printed)        L360
//   Eq.6-7 bending energy -> force (frames fixed) L363-372
//   Eq.2-3 stretch force                          L344-351
//   Eq.10  inextensibility projection             L383-392   (+ compliance, R-8)
//   Eq.11  plasticity                             L394-398
//   Eq.13  self-contact projection + friction     L406-410
//   soft rigid coupling                           L103
#pragma once
#include <math.h>

#if defined(__CUDACC__)
#define DLO_HD __host__ __device__ __forceinline__
#else
#define DLO_HD inline
#endif

namespace dlo {

template <class T> struct V3 { T x, y, z; };
template <class T> DLO_HD V3<T> mk3(T a, T b, T c) { V3<T> r; r.x = a; r.y = b; r.z = c; return r; }
template <class T> DLO_HD V3<T> zero3() { return mk3<T>(T(0), T(0), T(0)); }
template <class T> DLO_HD V3<T> operator+(const V3<T>& a, const V3<T>& b) { return mk3<T>(a.x + b.x, a.y + b.y, a.z + b.z); }
template <class T> DLO_HD V3<T> operator-(const V3<T>& a, const V3<T>& b) { return mk3<T>(a.x - b.x, a.y - b.y, a.z - b.z); }
template <class T> DLO_HD V3<T> operator-(const V3<T>& a) { return mk3<T>(-a.x, -a.y, -a.z); }
template <class T> DLO_HD V3<T> operator*(T s, const V3<T>& a) { return mk3<T>(s * a.x, s * a.y, s * a.z); }
template <class T> DLO_HD V3<T>& operator+=(V3<T>& a, const V3<T>& b) { a.x += b.x; a.y += b.y; a.z += b.z; return a; }
template <class T> DLO_HD V3<T>& operator-=(V3<T>& a, const V3<T>& b) { a.x -= b.x; a.y -= b.y; a.z -= b.z; return a; }
template <class T> DLO_HD T dot(const V3<T>& a, const V3<T>& b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
template <class T> DLO_HD V3<T> cross(const V3<T>& a, const V3<T>& b) {
  return mk3<T>(a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x);
}
// a + s*b
template <class T> DLO_HD V3<T> axpy(const V3<T>& a, T s, const V3<T>& b) { return mk3<T>(a.x + s * b.x, a.y + s * b.y, a.z + s * b.z); }

DLO_HD float rsqrt_(float a) {
#if defined(__CUDA_ARCH__)
  return rsqrtf(a);
#else
  return 1.0f / sqrtf(a);
#endif
}
DLO_HD double rsqrt_(double a) { return 1.0 / sqrt(a); }
DLO_HD float sqrt_(float a) { return sqrtf(a); }
DLO_HD double sqrt_(double a) { return sqrt(a); }
DLO_HD float exp_(float a) { return expf(a); }
DLO_HD double exp_(double a) { return exp(a); }
DLO_HD void sincos_(float a, float* s, float* c) {
#if defined(__CUDA_ARCH__)
  sincosf(a, s, c);
#else
  *s = sinf(a); *c = cosf(a);
#endif
}
DLO_HD void sincos_(double a, double* s, double* c) { *s = sin(a); *c = cos(a); }
// explicit fused multiply-add: used where the SAME value must come out of every kernel the expression is inlined into
// (forward, replay, reverse pass): an `a * b + c` left to the compiler may be contracted differently in each of them
DLO_HD float fma_(float a, float b, float c) { return fmaf(a, b, c); }
DLO_HD double fma_(double a, double b, double c) { return fma(a, b, c); }
template <class T> DLO_HD T clamp01(T s) { return s < T(0) ? T(0) : (s > T(1) ? T(1) : s); }

// 3x3 rotation, row-major
template <class T> struct M3 { T m[9]; };
template <class T> DLO_HD V3<T> mul(const M3<T>& R, const V3<T>& a) {
  return mk3<T>(R.m[0] * a.x + R.m[1] * a.y + R.m[2] * a.z, R.m[3] * a.x + R.m[4] * a.y + R.m[5] * a.z,
                R.m[6] * a.x + R.m[7] * a.y + R.m[8] * a.z);
}
template <class T> DLO_HD V3<T> mulT(const M3<T>& R, const V3<T>& a) {
  return mk3<T>(R.m[0] * a.x + R.m[3] * a.y + R.m[6] * a.z, R.m[1] * a.x + R.m[4] * a.y + R.m[7] * a.z,
                R.m[2] * a.x + R.m[5] * a.y + R.m[8] * a.z);
}

// Rodrigues coefficients: R = I + A [rho]x + B [rho]x^2, series for |rho|^2 < 1e-8 (R-20)
template <class T> DLO_HD void rodrigues_coeff(T th2, T& A, T& B) {
  if (th2 < T(1e-8)) { A = fma_(th2, T(-1.0 / 6.0), T(1)); B = fma_(th2, T(-1.0 / 24.0), T(0.5)); }
  else { T th = sqrt_(th2), s, c; sincos_(th, &s, &c); A = s / th; B = (T(1) - c) / th2; }
}
template <class T> DLO_HD M3<T> rodrigues(const V3<T>& rho) {
  const T kx = rho.x, ky = rho.y, kz = rho.z;
  T th2 = fma_(kz, kz, fma_(ky, ky, kx * kx)), A, B;
  rodrigues_coeff(th2, A, B);
  const T Bx = B * kx, By = B * ky, Ax = A * kx, Ay = A * ky, Az = A * kz;   // every sum of products below is an explicit fma
  M3<T> R;
  R.m[0] = fma_(B, fma_(kx, kx, -th2), T(1)); R.m[1] = fma_(Bx, ky, -Az);                R.m[2] = fma_(Bx, kz, Ay);
  R.m[3] = fma_(Bx, ky, Az);                 R.m[4] = fma_(B, fma_(ky, ky, -th2), T(1)); R.m[5] = fma_(By, kz, -Ax);
  R.m[6] = fma_(Bx, kz, -Ay);                R.m[7] = fma_(By, kz, Ax);                 R.m[8] = fma_(B, fma_(kz, kz, -th2), T(1));
  return R;
}

// rotation-minimising transport of u from unit tangent a to unit tangent b
template <class T> DLO_HD V3<T> ptransport(const V3<T>& a, const V3<T>& b, const V3<T>& u) {
  V3<T> w = cross(a, b);
  T c = dot(a, b);
  V3<T> wu = cross(w, u);
  return u + wu + (T(1) / (T(1) + c)) * cross(w, wu);
}

// Eq.4 + Eq.5 at one interior vertex: edges a (before) and b (after), unit tangents ta, tb, directors d1a, d1b
template <class T> DLO_HD void material_curvature(const V3<T>& ta, const V3<T>& tb, const V3<T>& d1a, const V3<T>& d1b,
                                                  T& k1, T& k2) {
  T chi = T(1) + dot(ta, tb);
  V3<T> kb = (T(2) / chi) * cross(ta, tb);
  V3<T> m1 = T(0.5) * (d1a + d1b), m2 = T(0.5) * (cross(ta, d1a) + cross(tb, d1b));
  k1 = dot(kb, m2);
  k2 = dot(kb, m1);
}

// -dU_b/dx of the bending element at one interior vertex (Eq.6-7, frames held fixed, R-5).
// s = alpha / l_bar.  The element adds +Ga to vertex i-1, (-Ga + Gb) to vertex i, -Gb to vertex i+1.
template <class T> DLO_HD void bend_element(const V3<T>& ta, const V3<T>& tb, T inv_La, T inv_Lb, const V3<T>& d1a,
                                            const V3<T>& d1b, T k1b, T k2b, T s, V3<T>& Ga, V3<T>& Gb) {
  T ichi = T(1) / (T(1) + dot(ta, tb));
  V3<T> kb = (T(2) * ichi) * cross(ta, tb);
  V3<T> m1 = T(0.5) * (d1a + d1b), m2 = T(0.5) * (cross(ta, d1a) + cross(tb, d1b));
  T dk1 = dot(kb, m2) - k1b, dk2 = dot(kb, m1) - k2b;
  V3<T> q = dk1 * m2 + dk2 * m1;
  T qkb = dot(q, kb);
  V3<T> Aa = ichi * (T(2) * cross(tb, q) - qkb * tb);
  V3<T> Ab = ichi * (T(2) * cross(q, ta) - qkb * ta);
  Ga = (s * inv_La) * (Aa - dot(Aa, ta) * ta);
  Gb = (s * inv_Lb) * (Ab - dot(Ab, tb) * tb);
}

// Eq.10 with compliance on one edge: e = current edge vector, S = accumulated multiplier of this substep.
// Returns lambda and the unit direction; the caller applies dx_j += lam*wj*t, dx_{j+1} -= lam*wj1*t, S += lam.
template <class T> DLO_HD void project_edge(const V3<T>& e, T wsum, T l0, T atil, T S, T& lam, V3<T>& t) {
  T L2 = dot(e, e);
  T iL = rsqrt_(L2);
  T L = L2 * iL;
  t = iL * e;
  lam = ((L - l0) - atil * S) / (wsum + atil);
}

// closest points of segments [p1,q1], [p2,q2] (R-14); `region` records the branch for the adjoint:
// bit0: t from the interior formula (den ok), bit1: u<0 branch, bit2: u>1 branch, bit3: t clamped
template <class T> DLO_HD void closest_points(const V3<T>& p1, const V3<T>& q1, const V3<T>& p2, const V3<T>& q2, T& t, T& u) {
  V3<T> d1 = q1 - p1, d2 = q2 - p2, r = p1 - p2;
  T a = dot(d1, d1), e = dot(d2, d2), b = dot(d1, d2), c = dot(d1, r), f = dot(d2, r);
  T den = a * e - b * b;
  if (den > T(1e-12) * a * e) t = clamp01((b * f - c * e) / den); else t = T(0);
  u = (b * t + f) / e;
  if (u < T(0)) { u = T(0); t = clamp01(-c / a); }
  else if (u > T(1)) { u = T(1); t = clamp01((b - c) / a); }
}

// Eq.13 evaluation on four vertices (i,i+1 | j,j+1).  Returns true when penetrating; corrections are
// out_k = coef[k] * n with coef = d*w_k*beta_k/W, beta = (1-t, t, -(1-u), -u).
template <class T> DLO_HD bool contact_eval(const V3<T> x[4], const T w[4], T rsum, T& d, T& t, T& u, V3<T>& n, T& W) {
  closest_points(x[0], x[1], x[2], x[3], t, u);
  V3<T> dv = (axpy(x[0], t, x[1] - x[0])) - (axpy(x[2], u, x[3] - x[2]));
  T del2 = dot(dv, dv);
  T del = sqrt_(del2);
  d = rsum - del;
  if (!(d > T(0)) || !(del > T(1e-12))) return false;
  n = (T(1) / del) * dv;
  T a0 = T(1) - t, b0 = T(1) - u;
  W = w[0] * a0 * a0 + w[1] * t * t + w[2] * b0 * b0 + w[3] * u * u;
  return W > T(0);
}

// Eq.11: Y = sigma_y * l_bar
template <class T> DLO_HD void plasticity_update(T k1, T k2, T& k1b, T& k2b, T Y, T r_c) {
  T e1 = k1 - k1b, e2 = k2 - k2b;
  T n2 = e1 * e1 + e2 * e2;
  if (n2 > Y * Y) {
    T n = sqrt_(n2);
    T s = r_c * (n - Y) / n;
    k1b += s * e1;
    k2b += s * e2;
  }
}

// oriented box: P = centre(3), half extents(3); R = box-to-world rotation.  Exact Euclidean SDF; inside the
// nearest face wins (first maximum in x,y,z order).
template <class T> DLO_HD bool sdf_box(const T* P, const M3<T>& R, const V3<T>& y, T& phi, V3<T>& n) {
  V3<T> p = mulT(R, y - mk3<T>(P[0], P[1], P[2]));
  T pc[3] = {p.x, p.y, p.z}, sg[3], q[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) { sg[k] = (pc[k] < T(0)) ? T(-1) : T(1); q[k] = sg[k] * pc[k] - P[3 + k]; }
  V3<T> nl;
  if (q[0] > T(0) || q[1] > T(0) || q[2] > T(0)) {
    T o0 = q[0] > T(0) ? q[0] : T(0), o1 = q[1] > T(0) ? q[1] : T(0), o2 = q[2] > T(0) ? q[2] : T(0);
    phi = sqrt_(o0 * o0 + o1 * o1 + o2 * o2);
    nl = mk3<T>(sg[0] * o0 / phi, sg[1] * o1 / phi, sg[2] * o2 / phi);
  } else {
    int k = 0;
    T qk = q[0];   // (no q[k]: a dynamically indexed array lives in local memory)
    if (q[1] > qk) { k = 1; qk = q[1]; }
    if (q[2] > qk) { k = 2; qk = q[2]; }
    phi = qk;
    nl = mk3<T>(k == 0 ? sg[0] : T(0), k == 1 ? sg[1] : T(0), k == 2 ? sg[2] : T(0));
  }
  n = mul(R, nl);
  return true;
}

// analytic SDF + unit gradient of the rigid primitives (R-18); false = gradient undefined, skip
template <class T> DLO_HD bool sdf_eval(int type, const T* P, const V3<T>& y, T& phi, V3<T>& n) {
  if (type == 0) {  // plane: n(3), o
    n = mk3<T>(P[0], P[1], P[2]);
    phi = dot(n, y) - P[3];
    return true;
  }
  if (type == 1) {  // capsule: a(3), b(3), R
    V3<T> a = mk3<T>(P[0], P[1], P[2]), ab = mk3<T>(P[3], P[4], P[5]) - a;
    T s = clamp01(dot(y - a, ab) / dot(ab, ab));
    V3<T> dv = y - axpy(a, s, ab);
    T dist = sqrt_(dot(dv, dv));
    if (!(dist > T(1e-12))) return false;
    phi = dist - P[6];
    n = (T(1) / dist) * dv;
    return true;
  }
  if (type == 2) {  // cylinder: centre(3), unit axis(3), R, half-height
    V3<T> ax = mk3<T>(P[3], P[4], P[5]), p = y - mk3<T>(P[0], P[1], P[2]);
    T a = dot(p, ax);
    V3<T> rv = p - a * ax;
    T rho = sqrt_(dot(rv, rv));
    T sgn = (a < T(0)) ? T(-1) : T(1);
    T dr = rho - P[6], da = sgn * a - P[7];
    bool radial_ok = rho > T(1e-12);
    V3<T> er = radial_ok ? (T(1) / rho) * rv : zero3<T>();
    if (dr <= T(0) && da <= T(0)) {
      if (dr > da) { if (!radial_ok) return false; phi = dr; n = er; }
      else { phi = da; n = sgn * ax; }
    } else if (da <= T(0)) { if (!radial_ok) return false; phi = dr; n = er; }
    else if (dr <= T(0)) { phi = da; n = sgn * ax; }
    else { phi = sqrt_(dr * dr + da * da); n = (dr / phi) * er + ((da / phi) * sgn) * ax; }
    return true;
  }
  if (type == 3) {  // box: centre(3), half extents(3), rotation vector(3)
    return sdf_box<T>(P, rodrigues(mk3<T>(P[6], P[7], P[8])), y, phi, n);
  }
  return false;
}

// same, for parameters pre-expanded by the kernels: a box carries its rotation matrix in P[6..14]
template <class T> DLO_HD bool sdf_eval_pre(int type, const T* P, const V3<T>& y, T& phi, V3<T>& n) {
  if (type == 3) {
    M3<T> R;
#pragma unroll
    for (int k = 0; k < 9; ++k) R.m[k] = P[6 + k];
    return sdf_box<T>(P, R, y, phi, n);
  }
  return sdf_eval<T>(type, P, y, phi, n);
}

// L103 soft coupling response of one vertex against one body (R-17).  v updated in place; returns
// true if the response was applied.  d = r - phi, inv_eps = 1/eps_s.
template <class T> DLO_HD bool rigid_response(V3<T>& v, const V3<T>& vb, const V3<T>& n, T d, T inv_eps, T f_thresh,
                                              T e_rest, T mu) {
  T f = exp_(d * inv_eps);
  if (f > T(1)) f = T(1);
  if (!(f > f_thresh)) return false;
  V3<T> u = v - vb;
  T un = dot(u, n);
  if (!(un < T(0))) return false;
  V3<T> ut = u - un * n;
  T J = (T(1) + e_rest) * (-un);
  T utn = sqrt_(dot(ut, ut));
  V3<T> utp = zero3<T>();
  if (utn > T(1e-12)) {
    T k = T(1) - mu * J / utn;
    if (k > T(0)) utp = k * ut;
  }
  V3<T> up = (-e_rest * un) * n + utp;
  v = v + f * (up - u);
  return true;
}

// gripper pose: p (3), R from the 6-vector xi = (p, rho)
template <class T> struct Pose { V3<T> p; M3<T> R; };
template <class T> DLO_HD Pose<T> make_pose(const T* a_prev, const T* a_cur, T tau) {
  T xi[6];
#pragma unroll
  for (int k = 0; k < 6; ++k) xi[k] = fma_(tau, a_cur[k], (T(1) - tau) * a_prev[k]);
  Pose<T> g;
  g.p = mk3<T>(xi[0], xi[1], xi[2]);
  g.R = rodrigues(mk3<T>(xi[3], xi[4], xi[5]));
  return g;
}
// velocity of the body point sitting at world c at the end of the substep (finite difference over the substep)
template <class T> DLO_HD V3<T> body_point_velocity(const Pose<T>& g0, const Pose<T>& g1, const V3<T>& c, T inv_h) {
  V3<T> local = mulT(g1.R, c - g1.p);
  V3<T> before = g0.p + mul(g0.R, local);
  return inv_h * (c - before);
}

}  // namespace dlo
