// ORACLE — TEST INFRASTRUCTURE ONLY.  Not part of the product path; shares no code with the CUDA library.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load this.
//
// C entry points around rod_step.hpp: rollout with checkpoints (forward in segments, one state
// per segment cached, reverse replay + backprop) and the reverse pass, one environment at a time in fp64,
// parallel over environments with OpenMP.  Layouts mirror the product's C-ABI so one harness drives both:
//   x, v      [B][3][N]     d1 [B][3][N] (first E columns used)     kappa_bar [B][2][N]
//   actions   [H][B][G][6]  g_material [B][5] = (stretch, bend, damping, yield, creep)
#include <cstdio>
#include <cstring>
#include <memory>
#ifdef _OPENMP
#include <omp.h>
#endif
#include "rod_step.hpp"

using namespace orc;

struct oracle_config {
  int32_t batch, n_verts, topology, n_substeps, n_proj_iters, stretch_mode;
  int32_t enable_plasticity, enable_self_contact, self_skip;
  int32_t n_grippers, n_grasp_max, n_primitives, kappa_bar_from_x0;
  double dt, gravity[3], rope_radius, contact_softness, influence_threshold, restitution;
};

struct EnvD {
  Scene sc;
  Params<double> pm;
  State<double> s0, cur;                 // state after A0 / current state
  std::vector<State<double>> ckpt;       // checkpoint g = state after g*stride steps
  std::vector<State<double>> rec;        // optional per-step record (rec[t] = state after t steps)
  double margin[MG_COUNT];               // diagnostics: closest approach to each branch threshold during the last rollout
  std::vector<uint8_t> cut;              // [N] absent edges of a multi-DLO scene (empty: one rope)
};

struct oracle_sim {
  Config c;
  int B;
  std::vector<EnvD> env;
  std::vector<double> actions;           // [H][B][G][6]
  int H_actions = 0, H_done = 0, stride = 0, record = 0;
  int t_start = 0;                       // frame index of the state in s0 (0 after oracle_set_state; oracle_restore_state sets it)
};

static Config to_config(const oracle_config& o) {
  Config c;
  c.cut = nullptr;
  c.N = o.n_verts; c.topology = o.topology; c.n_sub = o.n_substeps; c.N_C = o.n_proj_iters;
  c.stretch_mode = o.stretch_mode; c.plasticity = o.enable_plasticity; c.self_contact = o.enable_self_contact;
  c.self_skip = o.self_skip; c.G = o.n_grippers; c.n_grasp_max = o.n_grasp_max; c.K = o.n_primitives;
  c.kappa_bar_from_x0 = o.kappa_bar_from_x0;
  c.dt = o.dt; for (int k = 0; k < 3; ++k) c.g[k] = o.gravity[k];
  c.r = o.rope_radius; c.eps_s = o.contact_softness; c.f_thresh = o.influence_threshold; c.e_rest = o.restitution;
  return c;
}

// the env's own view of the shared config (its cuts)
static Config env_config(const oracle_sim* h, int b);
static void recompute_kin(const Config& c, Scene& sc, const std::vector<uint8_t>& pinned) {
  sc.kin.assign(c.N, KIN_FREE); sc.grasp_g.assign(c.N, -1); sc.grasp_k.assign(c.N, -1);
  for (int i = 0; i < c.N; ++i) if (!pinned.empty() && pinned[i]) sc.kin[i] = KIN_PINNED;
  for (int g = 0; g < c.G; ++g)
    for (int k = 0; k < c.n_grasp_max; ++k) {
      if (sc.grasp_vert.empty()) continue;
      int v = sc.grasp_vert[g * c.n_grasp_max + k];
      if (v >= 0 && v < c.N) { sc.kin[v] = KIN_GRASPED; sc.grasp_g[v] = g; sc.grasp_k[v] = k; }
    }
}

static Config env_config(const oracle_sim* h, int b) {
  Config c = h->c;
  c.cut = h->env[b].cut.empty() ? nullptr : h->env[b].cut.data();
  return c;
}

template <class T> static State<T> lift(const State<double>& s) {
  State<T> r;
  r.x.resize(s.x.size()); r.v.resize(s.v.size()); r.d1.resize(s.d1.size()); r.k1.resize(s.k1.size()); r.k2.resize(s.k2.size());
  return r;
}

extern "C" {

oracle_sim* oracle_create(const oracle_config* oc, const double* material /* [B][9]: m,l0,stretch,alpha,gamma,sigma_y,r_c,mu_r,mu_s */) {
  oracle_sim* h = new oracle_sim();
  h->c = to_config(*oc);
  h->B = oc->batch;
  h->env.resize(h->B);
  for (int b = 0; b < h->B; ++b) {
    const double* M = material + 9 * b;
    EnvD& e = h->env[b];
    e.sc.m = M[0]; e.sc.l0 = M[1]; e.sc.mu_r = M[7]; e.sc.mu_s = M[8];
    e.pm.stretch = M[2]; e.pm.alpha = M[3]; e.pm.gamma = M[4]; e.pm.sigma_y = M[5]; e.pm.r_c = M[6];
    e.sc.prim_type.assign(h->c.K, 0); e.sc.prim_param.assign(h->c.K * PRIM_NPARAM, 0.0);
    e.sc.finger_geom.assign(4 * h->c.G, 0.0); e.sc.grasp_vert.assign(h->c.G * h->c.n_grasp_max, -1);
    e.sc.q.assign(h->c.G * h->c.n_grasp_max, zero3<double>()); e.sc.pose0.assign(6 * h->c.G, 0.0);
    recompute_kin(h->c, e.sc, std::vector<uint8_t>());
  }
  return h;
}
void oracle_destroy(oracle_sim* h) { delete h; }

void oracle_set_pins(oracle_sim* h, const uint8_t* pinned /* [B][N] */) {
  for (int b = 0; b < h->B; ++b) {
    std::vector<uint8_t> p(pinned + (size_t)b * h->c.N, pinned + (size_t)(b + 1) * h->c.N);
    // grasp flags are re-applied on top of the pins
    recompute_kin(h->c, h->env[b].sc, p);
  }
}
void oracle_set_primitives(oracle_sim* h, const int32_t* types /* [K] */, const double* params /* [B][K][10] */) {
  const int K = h->c.K;
  for (int b = 0; b < h->B; ++b) {
    Scene& sc = h->env[b].sc;
    for (int k = 0; k < K; ++k) sc.prim_type[k] = types[k];
    for (int q = 0; q < K * PRIM_NPARAM; ++q) sc.prim_param[q] = params[(size_t)b * K * PRIM_NPARAM + q];
  }
}
void oracle_set_grippers(oracle_sim* h, const double* init_pose /* [B][G][6] */, const double* finger_geom /* [B][G][4] */,
                         const int32_t* grasp_verts /* [B][G][n_grasp_max] */) {
  const int G = h->c.G, M = h->c.n_grasp_max;
  for (int b = 0; b < h->B; ++b) {
    Scene& sc = h->env[b].sc;
    for (int q = 0; q < 6 * G; ++q) sc.pose0[q] = init_pose[(size_t)b * 6 * G + q];
    for (int q = 0; q < 4 * G; ++q) sc.finger_geom[q] = finger_geom[(size_t)b * 4 * G + q];
    for (int q = 0; q < G * M; ++q) sc.grasp_vert[q] = grasp_verts[(size_t)b * G * M + q];
    std::vector<uint8_t> pins(h->c.N, 0);
    for (int i = 0; i < h->c.N; ++i) pins[i] = (sc.kin[i] == KIN_PINNED);
    recompute_kin(h->c, sc, pins);
  }
}

// Multi-DLO scenes: cut[b][j] != 0 removes edge (j, j+1) of env b (rod_step.hpp, Config::cut).  Open topology only.
int32_t oracle_set_cuts(oracle_sim* h, const uint8_t* cut /* [B][N] */) {
  if (h->c.topology != TOPO_OPEN) return -1;
  for (int b = 0; b < h->B; ++b) h->env[b].cut.assign(cut + (size_t)b * h->c.N, cut + (size_t)(b + 1) * h->c.N);
  return 0;
}

// A0: frames, rest curvature, grasp-local coordinates.  Call after pins / grippers / cuts are set.
void oracle_set_state(oracle_sim* h, const double* x0, const double* v0, const double* kbar0 /* or NULL */) {
  const int N = h->c.N, E = h->c.E();
#pragma omp parallel for schedule(dynamic)
  for (int b = 0; b < h->B; ++b) {
    const Config c = env_config(h, b);
    EnvD& e = h->env[b];
    State<double>& s = e.s0;
    s.x.resize(N); s.v.resize(N); s.k1.assign(N, 0.0); s.k2.assign(N, 0.0);
    const double* X = x0 + (size_t)b * 3 * N; const double* V = v0 + (size_t)b * 3 * N;
    for (int i = 0; i < N; ++i) { s.x[i] = mkv(X[i], X[N + i], X[2 * N + i]); s.v[i] = mkv(V[i], V[N + i], V[2 * N + i]); }
    frames_init(c, s.x, s.d1, nullptr);
    if (kbar0) {
      const double* Kb = kbar0 + (size_t)b * 2 * N;
      for (int i = 0; i < N; ++i) { s.k1[i] = Kb[i]; s.k2[i] = Kb[N + i]; }
    } else if (c.kappa_bar_from_x0) {
      for (int i = 0; i < N; ++i) {
        if (!interior(c, i)) continue;
        int ip = vprev(c, i), in = vnext(c, i);
        Vec3<double> ea = s.x[i] - s.x[ip], eb = s.x[in] - s.x[i];
        material_curvature((1.0 / norm(ea)) * ea, (1.0 / norm(eb)) * eb, s.d1[ip], s.d1[i], s.k1[i], s.k2[i]);
      }
    }
    // grasp-local coordinates q_k = R_g(0)^T (x_k(0) - p_g(0))
    for (int g = 0; g < c.G; ++g) {
      GripperPose<double> gp = gripper_pose(&e.sc.pose0[6 * g], &e.sc.pose0[6 * g], 0.0);
      for (int k = 0; k < c.n_grasp_max; ++k) {
        int v = e.sc.grasp_vert[g * c.n_grasp_max + k];
        if (v >= 0 && v < N) e.sc.q[g * c.n_grasp_max + k] = mulT(gp.R, s.x[v] - gp.p);
      }
    }
    e.cur = s;
    e.ckpt.clear(); e.rec.clear();
    (void)E;
  }
  h->H_done = 0;
  h->t_start = 0;
}

// Harness plumbing (no arithmetic): put a full state (x, v, d1, kappa_bar as oracle_get_state returns them) back as the
// start state of the next rollout, which then runs frames t_start, t_start+1, ... (a checkpoint is one
// state; the segment is re-run from it).  No A0: the frames are taken as given; the grasp-local coordinates stay those
// of the last oracle_set_state.  The reverse pass then differentiates that segment only (g_actions indexed from t_start).
void oracle_restore_state(oracle_sim* h, const double* x, const double* v, const double* d1, const double* kbar, int32_t t_start) {
  const Config& c = h->c; const int N = c.N, E = c.E();
  for (int b = 0; b < h->B; ++b) {
    EnvD& e = h->env[b];
    State<double>& s = e.s0;
    s.x.resize(N); s.v.resize(N); s.d1.resize(E); s.k1.assign(N, 0.0); s.k2.assign(N, 0.0);
    const double* X = x + (size_t)b * 3 * N; const double* V = v + (size_t)b * 3 * N; const double* D = d1 + (size_t)b * 3 * N;
    const double* Kb = kbar + (size_t)b * 2 * N;
    for (int i = 0; i < N; ++i) { s.x[i] = mkv(X[i], X[N + i], X[2 * N + i]); s.v[i] = mkv(V[i], V[N + i], V[2 * N + i]); s.k1[i] = Kb[i]; s.k2[i] = Kb[N + i]; }
    for (int j = 0; j < E; ++j) s.d1[j] = mkv(D[j], D[N + j], D[2 * N + j]);
    e.cur = s;
    e.ckpt.clear(); e.rec.clear();
  }
  h->H_done = 0;
  h->t_start = t_start;
}

// Test hook: replace the A0 products (initial frames d1 [B][3][N], grasp-local coordinates q [B][G][M][3]) after
// oracle_set_state, so that finite differences in x0 can hold them fixed exactly as the reverse pass does
// ("no gradient through A0", Backward).  Either may be NULL.
void oracle_override_init(oracle_sim* h, const double* d1, const double* q) {
  const Config& c = h->c; const int N = c.N, E = c.E(), GM = c.G * c.n_grasp_max;
  for (int b = 0; b < h->B; ++b) {
    EnvD& e = h->env[b];
    if (d1) for (int j = 0; j < E; ++j) e.s0.d1[j] = mkv(d1[(size_t)b * 3 * N + j], d1[(size_t)b * 3 * N + N + j], d1[(size_t)b * 3 * N + 2 * N + j]);
    if (q) for (int k = 0; k < GM; ++k) e.sc.q[k] = mkv(q[((size_t)b * GM + k) * 3], q[((size_t)b * GM + k) * 3 + 1], q[((size_t)b * GM + k) * 3 + 2]);
    e.cur = e.s0;
  }
}
void oracle_get_grasp_local(oracle_sim* h, double* q /* [B][G][M][3] */) {
  const int GM = h->c.G * h->c.n_grasp_max;
  for (int b = 0; b < h->B; ++b)
    for (int k = 0; k < GM; ++k) { const Vec3<double>& v = h->env[b].sc.q[k]; double* o = q + ((size_t)b * GM + k) * 3; o[0] = v.x; o[1] = v.y; o[2] = v.z; }
}

void oracle_set_actions(oracle_sim* h, const double* actions /* [H][B][G][6] */, int32_t horizon) {
  h->actions.assign(actions, actions + (size_t)horizon * h->B * h->c.G * 6);
  h->H_actions = horizon;
}

static const double* action_ptr(const oracle_sim* h, int b, int t) {   // a_t, t = -1 -> initial pose
  if (t < 0) return h->env[b].sc.pose0.data();
  return h->actions.data() + ((size_t)t * h->B + b) * h->c.G * 6;
}

// forward rollout from the state set by oracle_set_state.  stride>0: keep checkpoint every `stride` steps.
// record != 0: additionally keep the state after every step (for the pins that look at trajectories).
int32_t oracle_rollout_forward(oracle_sim* h, int32_t horizon, int32_t stride, int32_t record) {
  if (h->c.G > 0 && h->t_start + horizon > h->H_actions) return -1;
  const int ts = h->t_start;
  h->stride = stride; h->record = record; h->H_done = horizon;
#pragma omp parallel for schedule(dynamic)
  for (int b = 0; b < h->B; ++b) {
    const Config c = env_config(h, b);
    EnvD& e = h->env[b];
    Work<double> w;
    e.cur = e.s0; e.ckpt.clear(); e.rec.clear();
    for (int k = 0; k < MG_COUNT; ++k) e.margin[k] = 1e300;
    margin_sink() = e.margin;              // diagnostics only (rod_step.hpp, note_margin)
    if (stride > 0) e.ckpt.push_back(e.cur);
    if (record) e.rec.push_back(e.cur);
    static const double none[1] = {0.0};
    for (int t = 0; t < horizon; ++t) {
      const double* ap = c.G ? action_ptr(h, b, ts + t - 1) : none;
      const double* ac = c.G ? action_ptr(h, b, ts + t) : none;
      step(c, e.sc, e.pm, e.cur, ap, ac, w);
      if (stride > 0 && (t + 1) % stride == 0) e.ckpt.push_back(e.cur);
      if (record) e.rec.push_back(e.cur);
    }
    margin_sink() = nullptr;
  }
  return 0;
}

// diagnostics: per env, the smallest relative distance to each branch threshold during the last oracle_rollout_forward
// (classes MG_* of rod_step.hpp; 1e300 = the branch was never evaluated)
int32_t oracle_num_margins(void) { return MG_COUNT; }
void oracle_get_margins(oracle_sim* h, double* out /* [B][MG_COUNT] */) {
  for (int b = 0; b < h->B; ++b)
    for (int k = 0; k < MG_COUNT; ++k) out[(size_t)b * MG_COUNT + k] = h->env[b].margin[k];
}

static void pack_state(const Config& c, const State<double>& s, double* x, double* v, double* d1, double* kb) {
  const int N = c.N, E = c.E();
  for (int i = 0; i < N; ++i) {
    if (x) { x[i] = s.x[i].x; x[N + i] = s.x[i].y; x[2 * N + i] = s.x[i].z; }
    if (v) { v[i] = s.v[i].x; v[N + i] = s.v[i].y; v[2 * N + i] = s.v[i].z; }
    if (kb) { kb[i] = s.k1[i]; kb[N + i] = s.k2[i]; }
    if (d1) { bool ok = i < E; d1[i] = ok ? s.d1[i].x : 0.0; d1[N + i] = ok ? s.d1[i].y : 0.0; d1[2 * N + i] = ok ? s.d1[i].z : 0.0; }
  }
}
void oracle_get_state(oracle_sim* h, double* x, double* v, double* d1, double* kbar) {
  const int N = h->c.N;
  for (int b = 0; b < h->B; ++b)
    pack_state(h->c, h->env[b].cur, x ? x + (size_t)b * 3 * N : nullptr, v ? v + (size_t)b * 3 * N : nullptr,
               d1 ? d1 + (size_t)b * 3 * N : nullptr, kbar ? kbar + (size_t)b * 2 * N : nullptr);
}
int32_t oracle_get_record(oracle_sim* h, int32_t t, double* x, double* v, double* d1, double* kbar) {
  const int N = h->c.N;
  for (int b = 0; b < h->B; ++b) {
    if (t < 0 || t >= (int)h->env[b].rec.size()) return -1;
    pack_state(h->c, h->env[b].rec[t], x ? x + (size_t)b * 3 * N : nullptr, v ? v + (size_t)b * 3 * N : nullptr,
               d1 ? d1 + (size_t)b * 3 * N : nullptr, kbar ? kbar + (size_t)b * 2 * N : nullptr);
  }
  return 0;
}

// Reverse pass: segments in reverse; each is replayed from its checkpoint keeping the state
// at the start of every step, then every step is differentiated with the tape scalar, last step first.
// Seeds dL/dx_T, dL/dv_T [B][3][N] (NULL = 0).  Outputs are written (not accumulated); any may be NULL.
int32_t oracle_backward(oracle_sim* h, const double* gxT, const double* gvT, double* g_actions /* [H][B][G][6] */,
                        double* g_x0, double* g_v0, double* g_d10 /* [B][3][N], extra */, double* g_kbar0 /* [B][2][N], extra */,
                        double* g_material /* [B][5] */) {
  const int N = h->c.N, E = h->c.E(), G = h->c.G, H = h->H_done, stride = h->stride;
  if (stride <= 0 || H <= 0) return -2;
  const int ts = h->t_start;   // frames are ts + t; g_actions is indexed by t (relative to the rollout's start)
  if (g_actions) std::memset(g_actions, 0, sizeof(double) * (size_t)H * h->B * G * 6);
#pragma omp parallel for schedule(dynamic)
  for (int b = 0; b < h->B; ++b) {
    const Config c = env_config(h, b);
    EnvD& e = h->env[b];
    Tape tape; current_tape() = &tape;
    Work<double> wd; Work<AD> wa;
    // running adjoints of the state
    std::vector<double> ax(3 * N, 0.0), av(3 * N, 0.0), ad(3 * E, 0.0), ak(2 * N, 0.0), gm(5, 0.0);
    for (int i = 0; i < N; ++i)
      for (int k = 0; k < 3; ++k) {
        if (gxT) ax[3 * i + k] = gxT[(size_t)b * 3 * N + k * N + i];
        if (gvT) av[3 * i + k] = gvT[(size_t)b * 3 * N + k * N + i];
      }
    const int nseg = (H + stride - 1) / stride;
    static const double none[1] = {0.0};
    for (int g = nseg - 1; g >= 0; --g) {
      const int t0 = g * stride, t1 = (t0 + stride < H) ? t0 + stride : H;
      std::vector<State<double>> starts;              // state at the start of each step of the segment
      State<double> s = e.ckpt[g];
      for (int t = t0; t < t1; ++t) {
        starts.push_back(s);
        step(c, e.sc, e.pm, s, G ? action_ptr(h, b, ts + t - 1) : none, G ? action_ptr(h, b, ts + t) : none, wd);
      }
      for (int t = t1 - 1; t >= t0; --t) {
        tape.clear();
        const State<double>& s0 = starts[t - t0];
        State<AD> sa = lift<AD>(s0);
        for (int i = 0; i < N; ++i) sa.x[i] = mkv(AD::variable(s0.x[i].x), AD::variable(s0.x[i].y), AD::variable(s0.x[i].z));
        for (int i = 0; i < N; ++i) sa.v[i] = mkv(AD::variable(s0.v[i].x), AD::variable(s0.v[i].y), AD::variable(s0.v[i].z));
        for (int j = 0; j < E; ++j) sa.d1[j] = mkv(AD::variable(s0.d1[j].x), AD::variable(s0.d1[j].y), AD::variable(s0.d1[j].z));
        for (int i = 0; i < N; ++i) { sa.k1[i] = AD::variable(s0.k1[i]); sa.k2[i] = AD::variable(s0.k2[i]); }
        std::vector<AD> ap(G ? 6 * G : 1), ac(G ? 6 * G : 1);
        for (int q = 0; q < 6 * G; ++q) { ap[q] = AD::variable(action_ptr(h, b, ts + t - 1)[q]); ac[q] = AD::variable(action_ptr(h, b, ts + t)[q]); }
        Params<AD> pa;
        pa.stretch = AD::variable(e.pm.stretch); pa.alpha = AD::variable(e.pm.alpha); pa.gamma = AD::variable(e.pm.gamma);
        pa.sigma_y = AD::variable(e.pm.sigma_y); pa.r_c = AD::variable(e.pm.r_c);
        const State<AD> in = sa;                       // remember the input nodes
        step(c, e.sc, pa, sa, ap.data(), ac.data(), wa);
        std::vector<double> adj(tape.size(), 0.0);
        auto seed = [&](const AD& o, double g_) { if (o.i >= 0) adj[o.i] += g_; };
        for (int i = 0; i < N; ++i) {
          seed(sa.x[i].x, ax[3 * i]); seed(sa.x[i].y, ax[3 * i + 1]); seed(sa.x[i].z, ax[3 * i + 2]);
          seed(sa.v[i].x, av[3 * i]); seed(sa.v[i].y, av[3 * i + 1]); seed(sa.v[i].z, av[3 * i + 2]);
          seed(sa.k1[i], ak[2 * i]); seed(sa.k2[i], ak[2 * i + 1]);
        }
        for (int j = 0; j < E; ++j) { seed(sa.d1[j].x, ad[3 * j]); seed(sa.d1[j].y, ad[3 * j + 1]); seed(sa.d1[j].z, ad[3 * j + 2]); }
        tape.reverse(adj);
        for (int i = 0; i < N; ++i) {
          ax[3 * i] = adj[in.x[i].x.i]; ax[3 * i + 1] = adj[in.x[i].y.i]; ax[3 * i + 2] = adj[in.x[i].z.i];
          av[3 * i] = adj[in.v[i].x.i]; av[3 * i + 1] = adj[in.v[i].y.i]; av[3 * i + 2] = adj[in.v[i].z.i];
          ak[2 * i] = adj[in.k1[i].i]; ak[2 * i + 1] = adj[in.k2[i].i];
        }
        for (int j = 0; j < E; ++j) { ad[3 * j] = adj[in.d1[j].x.i]; ad[3 * j + 1] = adj[in.d1[j].y.i]; ad[3 * j + 2] = adj[in.d1[j].z.i]; }
        gm[0] += adj[pa.stretch.i]; gm[1] += adj[pa.alpha.i]; gm[2] += adj[pa.gamma.i]; gm[3] += adj[pa.sigma_y.i]; gm[4] += adj[pa.r_c.i];
        if (g_actions)
          for (int q = 0; q < 6 * G; ++q) {
            g_actions[((size_t)t * h->B + b) * G * 6 + q] += adj[ac[q].i];
            if (t > 0) g_actions[((size_t)(t - 1) * h->B + b) * G * 6 + q] += adj[ap[q].i];
          }
      }
    }
    for (int i = 0; i < N; ++i)
      for (int k = 0; k < 3; ++k) {
        if (g_x0) g_x0[(size_t)b * 3 * N + k * N + i] = ax[3 * i + k];
        if (g_v0) g_v0[(size_t)b * 3 * N + k * N + i] = av[3 * i + k];
        if (g_d10) g_d10[(size_t)b * 3 * N + k * N + i] = (i < E) ? ad[3 * i + k] : 0.0;
      }
    if (g_kbar0) for (int i = 0; i < N; ++i) { g_kbar0[(size_t)b * 2 * N + i] = ak[2 * i]; g_kbar0[(size_t)b * 2 * N + N + i] = ak[2 * i + 1]; }
    if (g_material) for (int k = 0; k < 5; ++k) g_material[(size_t)b * 5 + k] = gm[k];
    current_tape() = nullptr;
  }
  return 0;
}

int32_t oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// ------------------------------------------------------------------------------------------------------
// operator-level entry points (the same functions the substep calls), for the pins in tests/
static std::vector<Vec3<double>> unpack3(const double* a, int n, int ld) {
  std::vector<Vec3<double>> r(n);
  for (int i = 0; i < n; ++i) r[i] = mkv(a[i], a[ld + i], a[2 * ld + i]);
  return r;
}
static Config mini_config(int N, int topology) { Config c; std::memset(&c, 0, sizeof(c)); c.N = N; c.topology = topology; return c; }

void oracle_op_curvature_binormal(const double* ta, const double* tb, double* out) {
  Vec3<double> r = curvature_binormal(mkv(ta[0], ta[1], ta[2]), mkv(tb[0], tb[1], tb[2]));
  out[0] = r.x; out[1] = r.y; out[2] = r.z;
}
void oracle_op_frames_init(int32_t N, int32_t topology, const double* x /* [3][N] */, double* d1 /* [3][N] */, double* psiH) {
  Config c = mini_config(N, topology);
  std::vector<Vec3<double>> d;
  frames_init(c, unpack3(x, N, N), d, psiH);
  for (int j = 0; j < N; ++j) { bool ok = j < c.E(); d1[j] = ok ? d[j].x : 0; d1[N + j] = ok ? d[j].y : 0; d1[2 * N + j] = ok ? d[j].z : 0; }
}
void oracle_op_material_curvature(int32_t N, int32_t topology, const double* x, const double* d1, double* kappa /* [2][N] */) {
  Config c = mini_config(N, topology);
  auto X = unpack3(x, N, N); auto D = unpack3(d1, N, N);
  for (int i = 0; i < N; ++i) {
    kappa[i] = kappa[N + i] = 0.0;
    if (!interior(c, i)) continue;
    int ip = vprev(c, i), in = vnext(c, i);
    Vec3<double> ea = X[i] - X[ip], eb = X[in] - X[i];
    material_curvature((1.0 / norm(ea)) * ea, (1.0 / norm(eb)) * eb, D[ip], D[i], kappa[i], kappa[N + i]);
  }
}
double oracle_op_bend_energy(int32_t N, int32_t topology, const double* x, const double* d1, const double* kbar, double alpha, double lbar) {
  Config c = mini_config(N, topology);
  std::vector<double> k1(kbar, kbar + N), k2(kbar + N, kbar + 2 * N);
  return bend_energy(c, unpack3(x, N, N), unpack3(d1, N, N), k1, k2, alpha, lbar);
}
void oracle_op_bend_force(int32_t N, int32_t topology, const double* x, const double* d1, const double* kbar, double alpha, double lbar, double* f) {
  Config c = mini_config(N, topology);
  std::vector<double> k1(kbar, kbar + N), k2(kbar + N, kbar + 2 * N);
  std::vector<Vec3<double>> F(N, zero3<double>());
  bend_force(c, unpack3(x, N, N), unpack3(d1, N, N), k1, k2, alpha, lbar, F);
  for (int i = 0; i < N; ++i) { f[i] = F[i].x; f[N + i] = F[i].y; f[2 * N + i] = F[i].z; }
}
double oracle_op_stretch_energy(int32_t N, int32_t topology, const double* x, double ks, double l0) {
  Config c = mini_config(N, topology);
  return stretch_energy(c, unpack3(x, N, N), ks, l0);
}
void oracle_op_stretch_force(int32_t N, int32_t topology, const double* x, double ks, double l0, double* f) {
  Config c = mini_config(N, topology);
  std::vector<Vec3<double>> F(N, zero3<double>());
  stretch_force(c, unpack3(x, N, N), ks, l0, F);
  for (int i = 0; i < N; ++i) { f[i] = F[i].x; f[N + i] = F[i].y; f[2 * N + i] = F[i].z; }
}
// one application of Eq.10 to an isolated edge: xj, xj1 in/out (positions), S in/out
void oracle_op_project_edge(double* xj, double* xj1, double wj, double wj1, double l0, double atil, double* S) {
  Vec3<double> a = mkv(xj[0], xj[1], xj[2]), b = mkv(xj1[0], xj1[1], xj1[2]);
  Vec3<double> da = zero3<double>(), db = zero3<double>();
  project_edge(b - a, wj, wj1, l0, atil, *S, da, db);
  a = a + da; b = b + db;
  xj[0] = a.x; xj[1] = a.y; xj[2] = a.z; xj1[0] = b.x; xj1[1] = b.y; xj1[2] = b.z;
}
void oracle_op_closest_points(const double* p1, const double* q1, const double* p2, const double* q2, double* t, double* u) {
  closest_points(mkv(p1[0], p1[1], p1[2]), mkv(q1[0], q1[1], q1[2]), mkv(p2[0], p2[1], p2[2]), mkv(q2[0], q2[1], q2[2]), *t, *u);
}
// Eq.13 on four vertices x[4][3] (in/out), w[4]; returns 1 if a correction was applied; tu[2] = (t,u) used
int32_t oracle_op_self_contact(double* x, const double* w, double rsum, double* depth, double* tu) {
  Vec3<double> xs[4], out[4], n; double d, t, u, W;
  for (int k = 0; k < 4; ++k) xs[k] = mkv(x[3 * k], x[3 * k + 1], x[3 * k + 2]);
  bool hit = self_contact_correction(xs, w, rsum, out, d, t, u, n, W);
  *depth = d; tu[0] = t; tu[1] = u;
  if (!hit) return 0;
  for (int k = 0; k < 4; ++k) { x[3 * k] += out[k].x; x[3 * k + 1] += out[k].y; x[3 * k + 2] += out[k].z; }
  return 1;
}
void oracle_op_plasticity(const double* kappa, double* kbar, double Y, double r_c) {
  plasticity_update(kappa[0], kappa[1], kbar[0], kbar[1], Y, r_c);
}
int32_t oracle_op_sdf(int32_t type, const double* params, const double* y, double* phi, double* n) {
  Vec3<double> nn = zero3<double>(); double p = 0.0;
  bool ok = sdf(type, params, mkv(y[0], y[1], y[2]), p, nn);
  *phi = p; n[0] = nn.x; n[1] = nn.y; n[2] = nn.z;
  return ok ? 1 : 0;
}
void oracle_op_rigid_response(double* v, const double* vb, const double* n, double d, double eps_s, double f_thresh, double e_rest, double mu) {
  Vec3<double> vv = mkv(v[0], v[1], v[2]);
  rigid_response(vv, mkv(vb[0], vb[1], vb[2]), mkv(n[0], n[1], n[2]), d, eps_s, f_thresh, e_rest, mu);
  v[0] = vv.x; v[1] = vv.y; v[2] = vv.z;
}
void oracle_op_rodrigues(const double* rho, double* R /* row-major 3x3 */) {
  Mat3<double> M = rodrigues(mkv(rho[0], rho[1], rho[2]));
  for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) R[3 * a + b] = M.m[a][b];
}
void oracle_op_ptransport(const double* a, const double* b, const double* u, double* out) {
  Vec3<double> r = ptransport(mkv(a[0], a[1], a[2]), mkv(b[0], b[1], b[2]), mkv(u[0], u[1], u[2]));
  out[0] = r.x; out[1] = r.y; out[2] = r.z;
}

}  // extern "C"
