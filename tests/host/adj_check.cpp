// Host check of the product's per-element adjoints (paper_2606_04206_b200/csrc/rod_adj.cuh) against central
// finite differences of the matching forward operators (rod_ops.cuh), in double.  Built and run by
// tests/test_adjoint_ops_host.py with g++ (no CUDA).  Prints "name max_rel_err" per operator.
#include <cstdio>
#include <cstdlib>
#include <functional>
#include <random>
#include <string>
#include <vector>
#include "rod_adj.cuh"

using namespace dlo;
typedef std::vector<double> vec;
typedef V3<double> d3;
static std::mt19937_64 rng(1234);
static double U(double a = -1, double b = 1) { return std::uniform_real_distribution<double>(a, b)(rng); }
static d3 g3(const vec& x, int o) { return mk3<double>(x[o], x[o + 1], x[o + 2]); }
static void p3(vec& x, int o, const d3& v) { x[o] = v.x; x[o + 1] = v.y; x[o + 2] = v.z; }
static void a3(vec& x, int o, const d3& v) { x[o] += v.x; x[o + 1] += v.y; x[o + 2] += v.z; }
static d3 unit(d3 v) { return (1.0 / sqrt(dot(v, v))) * v; }

// f: in -> out ; adj: (in, outbar) -> inbar.  Returns max relative error over the inputs.
static double check(const std::string& name, const vec& x0, int nout, std::function<vec(const vec&)> f,
                    std::function<vec(const vec&, const vec&)> adj, double eps = 1e-6) {
  vec ob(nout);
  for (auto& o : ob) o = U();
  vec ib = adj(x0, ob);
  double worst = 0, scale = 1e-12;
  vec fd(x0.size());
  for (size_t i = 0; i < x0.size(); ++i) {
    vec xp = x0, xm = x0;
    double h = eps * std::max(1.0, fabs(x0[i]));
    xp[i] += h; xm[i] -= h;
    vec fp = f(xp), fm = f(xm);
    double s = 0;
    for (int k = 0; k < nout; ++k) s += ob[k] * (fp[k] - fm[k]) / (2 * h);
    fd[i] = s;
    scale = std::max(scale, fabs(s));
  }
  for (size_t i = 0; i < x0.size(); ++i) worst = std::max(worst, fabs(fd[i] - ib[i]) / scale);
  printf("%s %.3e\n", name.c_str(), worst);
  return worst;
}

int main() {
  // ---- bend_element: in = ta(3) tb(3) iLa iLb d1a(3) d1b(3) k1b k2b s  (tangents/directors treated as free vectors)
  for (int rep = 0; rep < 3; ++rep) {
    vec x(17);
    d3 ta = unit(mk3<double>(1, U(-.4, .4), U(-.4, .4))), tb = unit(mk3<double>(1, U(-.4, .4), U(-.4, .4)));
    p3(x, 0, ta); p3(x, 3, tb); x[6] = U(50, 100); x[7] = U(50, 100);
    p3(x, 8, unit(cross(ta, mk3<double>(U(), U(), 1)))); p3(x, 11, unit(cross(tb, mk3<double>(U(), U(), 1))));
    x[14] = U(); x[15] = U(); x[16] = U(0.5, 2);
    check("bend_element", x, 6,
          [](const vec& x) { d3 Ga, Gb; bend_element<double>(g3(x, 0), g3(x, 3), x[6], x[7], g3(x, 8), g3(x, 11), x[14], x[15], x[16], Ga, Gb);
                             vec o(6); p3(o, 0, Ga); p3(o, 3, Gb); return o; },
          [](const vec& x, const vec& ob) { vec ib(17, 0.0); d3 tab = zero3<double>(), tbb = tab, dab = tab, dbb = tab;
                             bend_element_adj<double>(g3(x, 0), g3(x, 3), x[6], x[7], g3(x, 8), g3(x, 11), x[14], x[15], x[16], g3(ob, 0), g3(ob, 3),
                                                      tab, tbb, ib[6], ib[7], dab, dbb, ib[14], ib[15], ib[16]);
                             p3(ib, 0, tab); p3(ib, 3, tbb); p3(ib, 8, dab); p3(ib, 11, dbb); return ib; });
  }
  // ---- material_curvature
  {
    vec x(12);
    d3 ta = unit(mk3<double>(1, U(-.4, .4), U(-.4, .4))), tb = unit(mk3<double>(1, U(-.4, .4), U(-.4, .4)));
    p3(x, 0, ta); p3(x, 3, tb); p3(x, 6, unit(cross(ta, mk3<double>(U(), U(), 1)))); p3(x, 9, unit(cross(tb, mk3<double>(U(), U(), 1))));
    check("material_curvature", x, 2,
          [](const vec& x) { vec o(2); material_curvature<double>(g3(x, 0), g3(x, 3), g3(x, 6), g3(x, 9), o[0], o[1]); return o; },
          [](const vec& x, const vec& ob) { vec ib(12, 0.0); d3 a = zero3<double>(), b = a, c = a, d = a;
                             material_curvature_adj<double>(g3(x, 0), g3(x, 3), g3(x, 6), g3(x, 9), ob[0], ob[1], a, b, c, d);
                             p3(ib, 0, a); p3(ib, 3, b); p3(ib, 6, c); p3(ib, 9, d); return ib; });
  }
  // ---- normalize: e -> (t, iL)
  {
    vec x = {U(), U(), U()};
    check("normalize", x, 4,
          [](const vec& x) { d3 e = g3(x, 0); double iL = 1 / sqrt(dot(e, e)); vec o(4); p3(o, 0, iL * e); o[3] = iL; return o; },
          [](const vec& x, const vec& ob) { d3 e = g3(x, 0); double iL = 1 / sqrt(dot(e, e)); vec ib(3); p3(ib, 0, normalize_adj<double>(iL * e, iL, g3(ob, 0), ob[3])); return ib; });
  }
  // ---- frame update
  {
    vec x(9);
    d3 to = unit(mk3<double>(1, U(-.3, .3), U(-.3, .3))), tn = unit(mk3<double>(1, U(-.3, .3), U(-.3, .3)));
    p3(x, 0, to); p3(x, 3, tn); p3(x, 6, unit(cross(to, mk3<double>(U(), U(), 1))));
    check("frame_update", x, 3,
          [](const vec& x) { d3 d = ptransport<double>(g3(x, 0), g3(x, 3), g3(x, 6)); d = d - dot(d, g3(x, 3)) * g3(x, 3); vec o(3); p3(o, 0, unit(d)); return o; },
          [](const vec& x, const vec& ob) { vec ib(9, 0.0); d3 a = zero3<double>(), b = a, c = a; frame_update_adj<double>(g3(x, 0), g3(x, 3), g3(x, 6), g3(ob, 0), a, b, c);
                             p3(ib, 0, a); p3(ib, 3, b); p3(ib, 6, c); return ib; });
  }
  // ---- plasticity: in = k1 k2 k1b k2b Y rc ; out = new k1b k2b   (active and inactive)
  for (int rep = 0; rep < 2; ++rep) {
    vec x = {0.8, -0.5, 0.1, 0.05, rep == 0 ? 0.3 : 5.0, 0.6};
    check(rep == 0 ? "plasticity_active" : "plasticity_inactive", x, 2,
          [](const vec& x) { vec o = {x[2], x[3]}; plasticity_update<double>(x[0], x[1], o[0], o[1], x[4], x[5]); return o; },
          [](const vec& x, const vec& ob) { vec ib(6, 0.0); double g1 = ob[0], g2 = ob[1];
                             plasticity_adj<double>(x[0], x[1], x[2], x[3], x[4], x[5], g1, g2, ib[0], ib[1], ib[4], ib[5]); ib[2] = g1; ib[3] = g2; return ib; });
  }
  // ---- project_edge: in = e(3) S dxj(3) dxn(3) atil ; out = dxj'(3) dxn'(3) S'
  {
    const double wj = 100, wn = 100, l0 = 0.05;
    vec x(11);
    p3(x, 0, mk3<double>(0.052, 0.004, -0.003)); x[3] = 1e-6; p3(x, 4, mk3<double>(U() * 1e-4, U() * 1e-4, U() * 1e-4)); p3(x, 7, mk3<double>(U() * 1e-4, U() * 1e-4, U() * 1e-4)); x[10] = 30;
    auto fwd = [=](const vec& x) { double lam; d3 t; project_edge<double>(g3(x, 0), wj + wn, l0, x[10], x[3], lam, t);
                                   vec o(7); p3(o, 0, axpy(g3(x, 4), lam * wj, t)); p3(o, 3, axpy(g3(x, 7), -lam * wn, t)); o[6] = x[3] + lam; return o; };
    check("project_edge", x, 7, fwd,
          [=](const vec& x, const vec& ob) { double lam; d3 t; project_edge<double>(g3(x, 0), wj + wn, l0, x[10], x[3], lam, t);
                             d3 e = g3(x, 0); double iL = 1 / sqrt(dot(e, e)); vec ib(11, 0.0); double Sbar = ob[6]; d3 eb;
                             project_edge_adj<double>(t, iL, lam, x[3] + lam, wj, wn, x[10], g3(ob, 0), g3(ob, 3), Sbar, ib[10], eb);
                             p3(ib, 0, eb); ib[3] = Sbar; p3(ib, 4, g3(ob, 0)); p3(ib, 7, g3(ob, 3)); return ib; }, 1e-7);
  }
  // ---- closest points in several regions: in = 4 points ; out = t,u
  {
    double cases[5][12] = {{0, 0, 0, 1, 0, 0, 0.3, -0.5, 0.2, 0.6, 0.5, 0.25},      // interior / interior
                           {0, 0, 0, 1, 0, 0, 1.4, -0.5, 0.2, 1.6, 0.5, 0.3},       // t clamped to 1, u interior
                           {0, 0, 0, 1, 0, 0, 0.3, 0.4, 0.2, 0.5, 0.9, 0.3},        // u < 0 branch, t free
                           {0, 0, 0, 1, 0, 0, 0.3, -0.9, 0.2, 0.5, -0.4, 0.3},      // u > 1 branch, t free
                           {0, 0, 0, 1, 0, 0, -0.5, 0.4, 0.2, -0.3, 0.9, 0.3}};     // both clamped
    for (int c = 0; c < 5; ++c) {
      vec x(cases[c], cases[c] + 12);
      for (auto& v : x) v += 0.01 * U();
      check("closest_points_" + std::to_string(c), x, 2,
            [](const vec& x) { vec o(2); closest_points<double>(g3(x, 0), g3(x, 3), g3(x, 6), g3(x, 9), o[0], o[1]); return o; },
            [](const vec& x, const vec& ob) { vec ib(12, 0.0); d3 a = zero3<double>(), b = a, c = a, d = a;
                               closest_points_adj<double>(g3(x, 0), g3(x, 3), g3(x, 6), g3(x, 9), ob[0], ob[1], a, b, c, d);
                               p3(ib, 0, a); p3(ib, 3, b); p3(ib, 6, c); p3(ib, 9, d); return ib; });
    }
  }
  // ---- Eq.13 contact: in = 4 points ; out = 4 corrections (12) + depth
  for (int c = 0; c < 3; ++c) {
    double base[3][12] = {{0, 0, 0, 1, 0, 0, 0.3, -0.5, 0.05, 0.6, 0.5, 0.08}, {0, 0, 0, 1, 0, 0, 0.7, -0.5, 0.05, 1.1, 0.1, 0.09}, {0, 0, 0, 1, 0, 0, 0.3, 0.02, 0.05, 0.5, 0.9, 0.3}};
    vec x(base[c], base[c] + 12);
    for (auto& v : x) v += 0.005 * U();
    const double w[4] = {100, c == 1 ? 0.0 : 100, 100, 50}, rsum = 0.15;
    check("contact_" + std::to_string(c), x, 13,
          [=](const vec& x) { d3 xs[4] = {g3(x, 0), g3(x, 3), g3(x, 6), g3(x, 9)}; double d, t, u, W; d3 n; vec o(13, 0.0);
                              if (!contact_eval<double>(xs, w, rsum, d, t, u, n, W)) { printf("contact case not penetrating\n"); return o; }
                              double s = d / W; p3(o, 0, (s * w[0] * (1 - t)) * n); p3(o, 3, (s * w[1] * t) * n); p3(o, 6, (-s * w[2] * (1 - u)) * n); p3(o, 9, (-s * w[3] * u) * n); o[12] = d; return o; },
          [=](const vec& x, const vec& ob) { d3 xs[4] = {g3(x, 0), g3(x, 3), g3(x, 6), g3(x, 9)}, obs[4] = {g3(ob, 0), g3(ob, 3), g3(ob, 6), g3(ob, 9)}, xb[4];
                              for (auto& v : xb) v = zero3<double>(); contact_adj<double>(xs, w, rsum, obs, ob[12], xb); vec ib(12); for (int k = 0; k < 4; ++k) p3(ib, 3 * k, xb[k]); return ib; });
  }
  // ---- friction: in = 4 points, 4 velocities, Dp ; out = 4 velocity increments
  for (int c = 0; c < 2; ++c) {
    vec x = {0, 0, 0, 1, 0, 0, 0.3, -0.5, 0.05, 0.6, 0.5, 0.08, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
    for (int k = 0; k < 12; ++k) x[k] += 0.005 * U();
    for (int k = 12; k < 24; ++k) x[k] = U();
    x[24] = c == 0 ? 1e-5 : 1.0;     // capped / not capped
    const double w[4] = {100, 100, 100, 50}, mu = 0.3, inv_h = 5000;
    check(c == 0 ? "friction_capped" : "friction_stick", x, 12,
          [=](const vec& x) { d3 xs[4] = {g3(x, 0), g3(x, 3), g3(x, 6), g3(x, 9)}, vv[4] = {g3(x, 12), g3(x, 15), g3(x, 18), g3(x, 21)}; vec o(12, 0.0);
                              double t, u; closest_points<double>(xs[0], xs[1], xs[2], xs[3], t, u); d3 dv = axpy(xs[0], t, xs[1] - xs[0]) - axpy(xs[2], u, xs[3] - xs[2]);
                              double del = sqrt(dot(dv, dv)), a0 = 1 - t, b0 = 1 - u, W = w[0] * a0 * a0 + w[1] * t * t + w[2] * b0 * b0 + w[3] * u * u; d3 n = (1 / del) * dv;
                              d3 vrel = (a0 * vv[0] + t * vv[1]) - (b0 * vv[2] + u * vv[3]); d3 vt = vrel - dot(vrel, n) * n; double vtn = sqrt(dot(vt, vt));
                              double cap = mu * x[24] * inv_h, mag = cap < vtn ? cap : vtn; d3 D = (-(mag / vtn)) * vt;
                              p3(o, 0, (w[0] * a0 / W) * D); p3(o, 3, (w[1] * t / W) * D); p3(o, 6, (-w[2] * b0 / W) * D); p3(o, 9, (-w[3] * u / W) * D); return o; },
          [=](const vec& x, const vec& ob) { d3 xs[4] = {g3(x, 0), g3(x, 3), g3(x, 6), g3(x, 9)}, vv[4] = {g3(x, 12), g3(x, 15), g3(x, 18), g3(x, 21)};
                              d3 obs[4] = {g3(ob, 0), g3(ob, 3), g3(ob, 6), g3(ob, 9)}, xb[4], vb[4]; for (int k = 0; k < 4; ++k) xb[k] = vb[k] = zero3<double>();
                              vec ib(25, 0.0); friction_adj<double>(xs, vv, w, x[24], mu, inv_h, obs, xb, vb, ib[24]);
                              for (int k = 0; k < 4; ++k) { p3(ib, 3 * k, xb[k]); p3(ib, 12 + 3 * k, vb[k]); } return ib; });
  }
  // ---- rigid response: in = v(3) vb(3) n(3) d ; out = v'(3)   (sliding, sticking, saturated f)
  for (int c = 0; c < 3; ++c) {
    vec x = {0.4, 0.1, -0.3, 0.05, 0, 0.02, 0.1, 0.05, 1.0, c == 2 ? 2e-3 : -5e-4};
    if (c == 1) { x[0] = 0.05; x[1] = 0.01; }
    d3 n = unit(g3(x, 6)); p3(x, 6, n);
    const double inv_eps = 1000, e_rest = 0.2, mu = 0.5;
    check("rigid_response_" + std::to_string(c), x, 3,
          [=](const vec& x) { d3 v = g3(x, 0); bool on = rigid_response<double>(v, g3(x, 3), g3(x, 6), x[9], inv_eps, 0.1, e_rest, mu); if (!on) printf("inactive!\n"); vec o(3); p3(o, 0, v); return o; },
          [=](const vec& x, const vec& ob) { vec ib(10, 0.0); d3 a = zero3<double>(), b = a, c = a;
                              ib[9] = rigid_response_adj<double>(g3(x, 0), g3(x, 3), g3(x, 6), x[9], inv_eps, e_rest, mu, g3(ob, 0), a, b, c); p3(ib, 0, a); p3(ib, 3, b); p3(ib, 6, c); return ib; });
  }
  // ---- SDFs w.r.t. y: out = phi, n(3)
  {
    struct Case { int type; std::vector<double> P; std::vector<d3> ys; };
    M3<double> R = rodrigues<double>(mk3<double>(0.2, -0.3, 0.5));
    std::vector<double> box = {0.1, -0.2, 0.05, 0.3, 0.2, 0.1};
    box.insert(box.end(), R.m, R.m + 9);
    std::vector<Case> cases = {
        {0, {0.0, 0.6, 0.8, 0.1}, {mk3<double>(0.3, 0.2, 0.5)}},
        {1, {0, 0, 0, 1, 0.2, 0.1, 0.05}, {mk3<double>(0.4, 0.5, 0.3), mk3<double>(-0.4, 0.2, 0.1), mk3<double>(1.5, 0.4, 0.3)}},
        {2, {0.1, 0.1, 0.2, 0, 0, 1, 0.3, 0.4}, {mk3<double>(0.8, 0.2, 0.3), mk3<double>(0.2, 0.15, 0.9), mk3<double>(0.7, 0.5, 0.8), mk3<double>(0.15, 0.2, 0.3), mk3<double>(0.12, 0.13, 0.55)}},
        {3, box, {mk3<double>(0.9, 0.2, 0.3), mk3<double>(0.5, 0.6, 0.7), mk3<double>(0.12, -0.18, 0.07), mk3<double>(0.1, -0.2, 0.4)}}};
    for (auto& cs : cases)
      for (size_t k = 0; k < cs.ys.size(); ++k) {
        vec x = {cs.ys[k].x, cs.ys[k].y, cs.ys[k].z};
        const int type = cs.type; const std::vector<double> P = cs.P;
        check("sdf_type" + std::to_string(type) + "_" + std::to_string(k), x, 4,
              [=](const vec& x) { double phi; d3 n; sdf_eval_pre<double>(type, P.data(), g3(x, 0), phi, n); vec o(4); o[0] = phi; p3(o, 1, n); return o; },
              [=](const vec& x, const vec& ob) { d3 yb = zero3<double>(); sdf_pre_adj<double>(type, P.data(), g3(x, 0), ob[0], g3(ob, 1), yb); vec ib(3); p3(ib, 0, yb); return ib; });
      }
  }
  // ---- capsule w.r.t. end points too: in = a b y
  for (int c = 0; c < 2; ++c) {
    vec x = {0, 0, 0, 1, 0.2, 0.1, c == 0 ? 0.4 : -0.4, 0.5, 0.3};
    check("sdf_capsule_endpoints_" + std::to_string(c), x, 4,
          [](const vec& x) { double P[7] = {x[0], x[1], x[2], x[3], x[4], x[5], 0.05}; double phi; d3 n; sdf_eval<double>(1, P, g3(x, 6), phi, n); vec o(4); o[0] = phi; p3(o, 1, n); return o; },
          [](const vec& x, const vec& ob) { d3 yb = zero3<double>(), ab = yb, bb = yb; sdf_capsule_adj<double>(g3(x, 0), g3(x, 3), g3(x, 6), ob[0], g3(ob, 1), yb, ab, bb);
                              vec ib(9); p3(ib, 0, ab); p3(ib, 3, bb); p3(ib, 6, yb); return ib; });
  }
  // ---- rodrigues (both branches) and pose interpolation; body point velocity
  for (int c = 0; c < 2; ++c) {
    vec x = c == 0 ? vec{0.3, -0.8, 0.5} : vec{2e-5, -3e-5, 1e-5};
    check(c == 0 ? "rodrigues" : "rodrigues_series", x, 9,
          [](const vec& x) { M3<double> R = rodrigues<double>(g3(x, 0)); return vec(R.m, R.m + 9); },
          [](const vec& x, const vec& ob) { vec ib(3); p3(ib, 0, rodrigues_adj<double>(g3(x, 0), ob.data())); return ib; }, c == 0 ? 1e-6 : 1e-9);
  }
  {
    vec x(15);   // a_prev(6) a_cur(6) c(3)
    for (auto& v : x) v = U();
    const double inv_h = 5000;
    check("body_point_velocity+make_pose", x, 3,
          [=](const vec& x) { Pose<double> g0 = make_pose<double>(&x[0], &x[6], 0.4), g1 = make_pose<double>(&x[0], &x[6], 0.6); vec o(3); p3(o, 0, body_point_velocity<double>(g0, g1, g3(x, 12), inv_h)); return o; },
          [=](const vec& x, const vec& ob) { Pose<double> g0 = make_pose<double>(&x[0], &x[6], 0.4), g1 = make_pose<double>(&x[0], &x[6], 0.6);
                              PoseBar<double> b0, b1; pose_bar_zero(b0); pose_bar_zero(b1); d3 cb = zero3<double>(); vec ib(15, 0.0);
                              body_point_velocity_adj<double>(g0, g1, g3(x, 12), inv_h, g3(ob, 0), cb, b0, b1);
                              make_pose_adj<double>(&x[0], &x[6], 0.4, b0, &ib[0], &ib[6]); make_pose_adj<double>(&x[0], &x[6], 0.6, b1, &ib[0], &ib[6]); p3(ib, 12, cb); return ib; });
  }
  return 0;
}
