// dlo_api.cu — host driver behind the C-ABI of include/dlo.h: handle, device buffers, launch schedule of the
// forward segment kernel and of the replay + adjoint kernels (gradient checkpointing).
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <string>
#include <vector>
#include <algorithm>

#include "../../include/dlo.h"
#include "rod_kernels.cuh"
#include "rod_adjoint.cuh"

using namespace dlo;

static thread_local std::string g_err;
static dlo_status fail(dlo_status code, const std::string& msg) { g_err = msg; return code; }
#define CU(call)                                                                                        \
  do {                                                                                                  \
    cudaError_t e_ = (call);                                                                            \
    if (e_ != cudaSuccess) {                                                                            \
      dlo_status c_ = (e_ == cudaErrorMemoryAllocation) ? DLO_ERR_OOM : DLO_ERR_CUDA;                    \
      return fail(c_, std::string(#call) + ": " + cudaGetErrorString(e_));                              \
    }                                                                                                   \
  } while (0)

struct dlo_sim {
  dlo_config cfg;
  cudaStream_t stream;
  KParams P;                      // kernel parameter block (pointers filled as buffers appear)
  int VPL, smem_fwd, smem_adj;    // dynamic shared memory per CTA
  int wpb_fwd, wpb_adj;           // warps (envs) per CTA
  size_t blk;                     // floats per env state block
  // library-owned device memory
  float *mat = nullptr, *qloc = nullptr, *pose0 = nullptr, *finger = nullptr, *prim = nullptr;
  float *state = nullptr, *state0 = nullptr, *ckpt = nullptr, *tape = nullptr, *acc_tape = nullptr, *adj = nullptr, *replay = nullptr, *gmat = nullptr;
  uint8_t *kin = nullptr, *pins = nullptr, *cuts = nullptr /* absent edges, allocated by dlo_set_cuts */;
  // Tape buffers, one checkpoint segment each (n_tape of them, segment g uses buffer g % n_tape).  The first is required; the
  // others are taken while device memory allows (180 GB of HBM: config 5 fits four of its ten 37 GB segments).  The forward
  // rollout writes the tape of its LAST n_tape segments itself, so the reverse pass replays only the segments before them,
  // and with more than one buffer those replays run on a second stream under the adjoint of a later segment.
  enum { MAX_TAPE = 4 };
  float* tapes[MAX_TAPE] = {};
  uint8_t* tape_flags[MAX_TAPE] = {};
  float* side[MAX_TAPE] = {};          // side-record pools, slot counters and slot indices, per tape buffer
  int *side_count[MAX_TAPE] = {}, *tape_slot[MAX_TAPE] = {};
  int side_cap = 0, side_floats = 0;
  int n_tape = 0, max_tape = MAX_TAPE;   // allocated / wanted at most (DLO_TAPE_BUFFERS)
  cudaStream_t aux = nullptr;
  cudaEvent_t ev_fwd = nullptr, ev_rep[MAX_TAPE] = {}, ev_adj[MAX_TAPE] = {};
  int *grasp = nullptr, *flags = nullptr;
  // env -> warp-slot order (k_sort_envs): work statistics of the last forward chunk / of the tape in each tape buffer, the orders made from them
  int *stat = nullptr, *stat_rep[MAX_TAPE] = {}, *perm_main = nullptr, *perm_rep = nullptr;
  bool stat_valid = false, stat_rep_valid[MAX_TAPE] = {};
  int chunk = 100;                 // frames per forward launch when the forward re-orders (sort_mode bit 0)
  int sort_mode = 6;               // bit 0: forward launches, bit 1: replays, bit 2: adjoint launches take the envs in sorted order
  size_t ckpt_blocks = 0, tape_blocks = 0;
  const float* actions = nullptr;   // borrowed
  int H_actions = 0, H_done = 0, stride = 0;
  int tape_lo = 1 << 30, tape_K = 0;   // segments >= tape_lo of the last forward rollout are on tape already, segment g in buffer g % tape_K
  int device = 0;                  // the CUDA device the handle was created on (every call must be made with it current)
  int t_start = 0;                 // frame index of state0 (0 after dlo_set_state; dlo_restore_state sets it)
  bool have_state = false, have_q = false, have_prims = false, have_grippers = false, have_adj = false;
  int64_t launches = 0;
  // staging of the *_host calls, owned by the handle: pinned host buffers and their device twins
  float *hx0 = nullptr, *hv0 = nullptr, *hkb = nullptr, *hact = nullptr, *hxT = nullptr, *hvT = nullptr;
  float *dx0 = nullptr, *dv0 = nullptr, *dkb = nullptr, *dact = nullptr, *dxT = nullptr, *dvT = nullptr;
  float *dsx = nullptr, *dsv = nullptr, *dga = nullptr, *dgx = nullptr, *dgv = nullptr, *dgm = nullptr;
  size_t hact_n = 0, dact_n = 0, dga_n = 0;
  // optional per-kernel timing (dlo_set_kernel_timing): CUDA event pairs around every launch of the three big kernels,
  // recorded on the stream the kernel is launched on; class 0 = k_forward, 1 = k_forward with tape (replay), 2 = k_adjoint
  bool timing = false;
  std::vector<cudaEvent_t> tev[3];   // start, stop, start, stop, ...
  std::vector<int64_t> tunits[3];    // env-steps processed by each launch
};

struct LaunchTimer {   // brackets one launch with an event pair when timing is on
  dlo_sim* s; int cls; cudaStream_t st; cudaEvent_t stop = nullptr;
  LaunchTimer(dlo_sim* s_, int cls_, cudaStream_t st_, int64_t units) : s(s_), cls(cls_), st(st_) {
    if (!s->timing) return;
    cudaEvent_t a = nullptr;
    if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&stop) != cudaSuccess) { if (a) cudaEventDestroy(a); stop = nullptr; cudaGetLastError(); return; }
    cudaEventRecord(a, st);
    s->tev[cls].push_back(a); s->tev[cls].push_back(stop); s->tunits[cls].push_back(units);
  }
  ~LaunchTimer() { if (stop) cudaEventRecord(stop, st); }
};

// every entry point: the handle's device must be the current one
static dlo_status check_device(const dlo_sim* s) {
  int d = -1;
  if (cudaGetDevice(&d) != cudaSuccess) { cudaGetLastError(); return fail(DLO_ERR_CUDA, "cudaGetDevice failed"); }
  if (d != s->device) return fail(DLO_ERR_BAD_STATE, "the handle was created on CUDA device " + std::to_string(s->device) + " but device " + std::to_string(d) + " is current");
  return DLO_OK;
}
#define ENTER(s)                                                       \
  do {                                                                 \
    if (!(s)) return fail(DLO_ERR_INVALID_ARG, "NULL handle");         \
    if (dlo_status st_ = check_device(s)) return st_;                  \
  } while (0)

static int vpl_for(int N) { return 2 * ((N + 63) / 64); }
static int round_up(int a, int b) { return (a + b - 1) / b * b; }

// per-warp shared-memory layout (float offsets); `adjoint` adds the reverse-pass scratch
static int smem_layout(KParams& P, int VPL, bool adjoint) {
  const int NP = 33 * VPL;   // padded row (vpos)
  int o = 0;
  P.n_guard = 0;
  // DLO_CHECKS=1 (the pool's compute-sanitizer being closed): four guard words behind every region, filled by warp_setup and
  // verified when the kernel ends (FLAG_GUARD); aliased views (sm_blk, sm_xref in the adjoint) share their host region's guard
  auto take = [&](int n) {
    int at = o;
    o += round_up(n, 4);
    if (P.checks && n > 0 && P.n_guard < 24) { P.sm_guard[P.n_guard++] = o; o += 4; }
    return at;
  };
  P.sm_pose = take(P.G * POSE_STRIDE);
  P.sm_prim = take(P.K * PRIM_SM_STRIDE);
  P.sm_q = take(P.G * P.M * 3);
  P.sm_ys = P.sm_acc = P.sm_vs = P.sm_mid = P.sm_dp = P.sm_cand = 0;
  P.sm_lam = P.sm_dpbar = P.sm_ybar = P.sm_vbar = P.sm_posebar = P.sm_blk = P.sm_xref = P.sm_hot = 0;
  if (P.self_contact) {
    P.sm_ys = take(3 * NP); P.sm_acc = take(3 * NP); P.sm_vs = take(3 * NP); P.sm_mid = take(5 * NP);
    P.sm_dp = take(P.cand_cap); P.sm_cand = take(P.cand_cap);   // candidates + prefilter survivors (ushort each)
    P.sm_blk = P.sm_vs;   // block bounding spheres (4 x 32 floats) live only inside build_pair_list; sm.vs is written after it (carry-over, friction)
    P.sm_hot = take(P.hot_cap / 2);   // near pairs (ushort each), kept across substeps
    if (!adjoint) P.sm_xref = take(3 * NP);   // positions at which the pair list was built (must outlive the substep)
  }
  if (adjoint) {
    P.sm_posebar = take(P.G * 24);
    if (P.self_contact) {
      P.sm_dpbar = take(P.cand_cap); P.sm_ybar = take(3 * NP); P.sm_vbar = take(3 * NP);
      P.sm_xref = P.sm_ybar;   // the reverse pass rebuilds the pair list in every recomputed substep; ybar is zeroed before each use
    }
  }
  P.sm_warp_floats = o;
  return o * (int)sizeof(float);   // bytes per warp
}

static dlo_status validate(const dlo_config* c) {
  if (!c) return fail(DLO_ERR_INVALID_ARG, "config is NULL");
  if (c->batch < 1) return fail(DLO_ERR_INVALID_ARG, "batch < 1");
  if (c->n_verts < 3 || c->n_verts > DLO_MAX_VERTS) return fail(DLO_ERR_INVALID_ARG, "n_verts out of [3,256]");
  if (c->topology != DLO_OPEN && c->topology != DLO_RING) return fail(DLO_ERR_INVALID_ARG, "bad topology");
  if (c->topology == DLO_RING && c->n_verts < 4) return fail(DLO_ERR_INVALID_ARG, "ring needs n_verts >= 4");
  if (c->n_substeps < 1 || c->n_proj_iters < 0 || c->n_proj_iters > 32) return fail(DLO_ERR_INVALID_ARG, "n_substeps < 1 or n_proj_iters out of [0,32]");
  if (c->stretch_mode != DLO_STRETCH_ENERGY && c->stretch_mode != DLO_STRETCH_PROJECT) return fail(DLO_ERR_INVALID_ARG, "bad stretch_mode");
  if (c->n_grippers < 0 || c->n_grippers > DLO_MAX_GRIPPERS) return fail(DLO_ERR_INVALID_ARG, "n_grippers out of [0,4]");
  if (c->n_grippers > 0 && (c->n_grasp_max < 1 || c->n_grasp_max > 8)) return fail(DLO_ERR_INVALID_ARG, "n_grasp_max out of [1,8]");
  if (c->n_primitives < 0 || c->n_primitives > DLO_MAX_PRIMITIVES) return fail(DLO_ERR_INVALID_ARG, "n_primitives out of [0,16]");
  if (c->n_primitives + 2 * c->n_grippers > 32) return fail(DLO_ERR_INVALID_ARG, "too many rigid bodies");
  if (!(c->dt > 0.0f) || !(c->contact_softness > 0.0f) || !(c->influence_threshold > 0.0f)) return fail(DLO_ERR_INVALID_ARG, "dt, contact_softness, influence_threshold must be > 0");
  if (c->enable_self_contact && c->self_skip < 2) return fail(DLO_ERR_INVALID_ARG, "self_skip < 2");
  return DLO_OK;
}

static void fill_params(const dlo_config& c, KParams& P) {
  memset(&P, 0, sizeof(P));
  P.B = c.batch; P.N = c.n_verts; P.ring = c.topology == DLO_RING; P.E = P.ring ? P.N : P.N - 1;
  P.NS = round_up(P.N, 4);
  P.odd_ring = P.ring && (P.E & 1);
  P.n_sub = c.n_substeps; P.N_C = c.n_proj_iters; P.stretch_mode = c.stretch_mode; P.plasticity = c.enable_plasticity != 0;
  P.self_contact = c.enable_self_contact != 0; P.self_skip = c.self_skip;
  P.G = c.n_grippers; P.M = P.G ? c.n_grasp_max : 1; P.K = c.n_primitives;
  // 15/4 N pairs: with the block spheres aliased onto sm.vs this brings two 7-warp forward CTAs of config 5 under the
  // 196 KB shared-memory configuration (97.5 KB each), which leaves the SM 60 KB of L1 for the spilled registers instead of 28
  P.cand_cap = round_up(15 * P.N / 4, 32);
  P.hot_cap = 32 * vpl_for(P.N);   // <= a third of the 3 x 33 VPL floats of sm.vs, which holds two such arrays during a mid-loop rebuild
  P.list_margin = c.rope_radius;   // a quarter of the candidate distance 2(r_a+r_b)
  P.vote_mode = 3;
  P.near_dist = 3.0f * c.rope_radius;   // 3/2 (r_a + r_b): half of (r_a + r_b) of slack for the far pairs
  if (const char* ov = getenv("DLO_NEAR")) P.near_dist = c.rope_radius * (float)atof(ov);   // 0: no near list
  if (const char* ov = getenv("DLO_LIST_MARGIN")) P.list_margin = c.rope_radius * (float)atof(ov);   // tuning overrides (no effect on results)
  if (const char* ov = getenv("DLO_VOTE")) P.vote_mode = atoi(ov) & 3;
  P.h = c.dt / (float)c.n_substeps; P.inv_h = 1.0f / P.h;
  for (int k = 0; k < 3; ++k) P.g[k] = c.gravity[k];
  P.r = c.rope_radius; P.inv_eps = 1.0f / c.contact_softness; P.f_thresh = c.influence_threshold; P.e_rest = c.restitution;
  P.log_thresh_lo = logf(c.influence_threshold) - 0.01f;
  P.phase_mask = 0xffffffffu;
  if (const char* ov = getenv("DLO_PHASES")) P.phase_mask = (unsigned)strtoul(ov, nullptr, 0);   // tuning override (no effect on results)
  if (const char* ov = getenv("DLO_CHECKS")) P.checks = atoi(ov);   // 1: checks on; 2: and a deliberate overrun (self-test of the check)
}

size_t dlo_scratch_bytes(const dlo_config* c, int32_t horizon, int32_t stride) {
  if (validate(c) != DLO_OK) return 0;
  KParams P;
  fill_params(*c, P);
  const size_t B = P.B, blk = (size_t)STATE_ROWS * P.NS * sizeof(float);
  size_t n = B * (MAT_N * 4 + P.NS + P.N + 4) + B * P.G * (P.M * 3 * 4 + 6 * 4 + 4 * 4 + P.M * 4) + B * P.K * PRIM_NP * 4;
  n += 2 * B * blk;                                                            // state, state0
  if (stride > 0 && horizon > 0) {
    n += ((size_t)horizon / stride + 1) * B * blk;                             // checkpoints
    const size_t tape = ((size_t)(stride < horizon ? stride : horizon) * P.n_sub + 1) * B * tape_rows(P.N_C) * P.NS * sizeof(float);
    n += tape * (horizon > stride ? 2 : 1);                                     // tape of one segment, double-buffered when there are several
    n += B * blk;                                                              // running adjoint
    if (P.self_contact) {
      n += B * (size_t)P.N_C * 3 * 33 * vpl_for(P.N) * 4;    // self-contact correction tape
      const size_t seg = (size_t)(stride < horizon ? stride : horizon) * P.n_sub + 1, cap = std::max<size_t>(1024, seg * B / 12);
      n += (horizon > stride ? 2 : 1) * (cap * side_record_floats(P, 33 * vpl_for(P.N)) * 4 + seg * B * 4 + 4);   // side-record pools + slot indices
    }
    n += 3 * B * 8 + 2 * B * 4;                                                // work statistics and env orders
  }
  return n;
}

// DLO_CHECKS=1: every library allocation starts as 0xff bytes (NaN as a float, -1 as an int), so that a read of memory
// nothing wrote shows up in the results (the stand-in for compute-sanitizer's initcheck, closed on this pool)
static bool checks_on() { const char* v = getenv("DLO_CHECKS"); return v && atoi(v) != 0; }
template <class T> static cudaError_t dalloc(T** p, size_t n) {
  cudaError_t e = cudaMalloc((void**)p, (n ? n : 1) * sizeof(T));
  if (e == cudaSuccess && checks_on()) e = cudaMemset(*p, 0xff, (n ? n : 1) * sizeof(T));
  return e;
}

extern "C" {

const char* dlo_last_error(void) { return g_err.c_str(); }
const char* dlo_version(void) { return "dlo-b200 0.1 (sm_100a)"; }
int64_t dlo_launch_count(const dlo_sim* s) { return s ? s->launches : 0; }

dlo_status dlo_create(const dlo_config* cfg, const dlo_material* mat, void* stream, dlo_sim** out) {
  if (!out) return fail(DLO_ERR_INVALID_ARG, "out is NULL");
  *out = nullptr;
  dlo_status st = validate(cfg);
  if (st != DLO_OK) return st;
  if (!mat) return fail(DLO_ERR_INVALID_ARG, "material is NULL");
  const float* mp[MAT_N] = {mat->mass_per_vertex, mat->rest_edge_len, mat->stretch, mat->bend_stiffness, mat->damping,
                            mat->yield_curv, mat->creep_rate, mat->mu_rigid, mat->mu_self};
  for (int k = 0; k < MAT_N; ++k) if (!mp[k]) return fail(DLO_ERR_INVALID_ARG, "a material array is NULL");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return fail(DLO_ERR_CUDA, "no CUDA device: this library has no CPU path"); }
  dlo_sim* s = new dlo_sim();
  s->cfg = *cfg;
  s->stream = (cudaStream_t)stream;
  if (cudaGetDevice(&s->device) != cudaSuccess) { cudaGetLastError(); delete s; return fail(DLO_ERR_CUDA, "cudaGetDevice failed"); }
  fill_params(*cfg, s->P);
  KParams& P = s->P;
  s->VPL = vpl_for(P.N);
  s->blk = (size_t)STATE_ROWS * P.NS;
  {
    const int per_fwd = smem_layout(P, s->VPL, false);
    KParams Pa = P;
    const int per_adj = smem_layout(Pa, s->VPL, true);
    const int cap = 227 * 1024;
    if (per_adj > cap) { delete s; return fail(DLO_ERR_UNSUPPORTED, "shared memory per env exceeds 227 KB for this n_verts / n_proj_iters"); }
    // forward: two CTAs per SM; choose the CTA size whose slots (2 * n_SM * warps) split the batch into whole waves
    // (4096 envs on 148 SMs: 7 warps -> 1.98 waves, where 8 warps would leave the second wave 27 % empty)
    int n_sm = 148;
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, s->device);
    // CTA shape: c warps per CTA, as many CTAs per SM as the register file (16 warps at 128 registers) and shared memory allow.  Cost model
    // fitted to a sweep on config 5: time ~ waves * sqrt(warps per SM), larger CTAs slightly
    // better at equal occupancy (more warps share each instruction-cache fill).
    const int max_w = s->VPL <= 4 ? 16 : 8;   // resident warps per SM the register file allows (128 / 255 registers)
    double best = 1e30;
    s->wpb_fwd = 1;
    for (int cw = 1; cw <= DLO_FWD_WARPS; ++cw) {
      const int k = std::min(max_w / cw, cap / std::max(cw * per_fwd, 1));
      if (k < 1) continue;
      const double slots = (double)k * n_sm * cw, waves = ceil(P.B / slots), cost = waves * sqrt((double)(k * cw)) * (1.0 - 0.01 * cw);
      if (cost < best - 1e-9) { best = cost; s->wpb_fwd = cw; }
    }
    if (const char* ov = getenv("DLO_FWD_WARPS")) s->wpb_fwd = std::max(1, std::min(DLO_FWD_WARPS, atoi(ov)));   // tuning override
    s->wpb_adj = std::max(1, std::min(DLO_ADJ_WARPS, cap / std::max(per_adj, 1)));
    if (const char* ov = getenv("DLO_ADJ_WARPS")) s->wpb_adj = std::max(1, std::min(s->wpb_adj, atoi(ov)));   // tuning override
    s->smem_fwd = per_fwd * s->wpb_fwd;
    s->smem_adj = per_adj * s->wpb_adj;
  }
  const size_t B = P.B;
#define CUD(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { dlo_destroy(s); return fail(e_ == cudaErrorMemoryAllocation ? DLO_ERR_OOM : DLO_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e_)); } } while (0)
  CUD(dalloc(&s->mat, B * MAT_N));
  CUD(dalloc(&s->kin, B * P.NS));
  CUD(dalloc(&s->pins, B * P.N));
  CUD(dalloc(&s->qloc, B * P.G * P.M * 3));
  CUD(dalloc(&s->pose0, B * P.G * 6));
  CUD(dalloc(&s->finger, B * P.G * 4));
  CUD(dalloc(&s->grasp, B * P.G * P.M));
  CUD(dalloc(&s->prim, B * P.K * PRIM_NP));
  CUD(dalloc(&s->state, B * s->blk));
  CUD(dalloc(&s->state0, B * s->blk));
  CUD(dalloc(&s->flags, B));
  CUD(dalloc(&s->stat, 2 * B));
  for (int k = 0; k < dlo_sim::MAX_TAPE; ++k) CUD(dalloc(&s->stat_rep[k], 2 * B));
  if (const char* ov = getenv("DLO_TAPE_BUFFERS")) s->max_tape = std::max(1, std::min((int)dlo_sim::MAX_TAPE, atoi(ov)));   // tuning override (no effect on results)
  CUD(dalloc(&s->perm_main, B)); CUD(dalloc(&s->perm_rep, B));
  if (const char* ov = getenv("DLO_CHUNK")) s->chunk = std::max(1, atoi(ov));   // tuning overrides (no effect on results)
  if (const char* ov = getenv("DLO_SORT")) s->sort_mode = atoi(ov) & 7;
  if (!P.self_contact) s->sort_mode = 0;   // the order only matters for the self-contact work
  CUD(cudaMemsetAsync(s->flags, 0, B * sizeof(int), s->stream));
  CUD(cudaMemsetAsync(s->pins, 0, B * P.N, s->stream));
  CUD(cudaMemsetAsync(s->grasp, 0xff, B * P.G * P.M * sizeof(int), s->stream));
  CUD(cudaMemsetAsync(s->pose0, 0, B * P.G * 6 * sizeof(float), s->stream));
  CUD(cudaMemsetAsync(s->finger, 0, B * P.G * 4 * sizeof(float), s->stream));
  CUD(cudaMemsetAsync(s->prim, 0, B * P.K * PRIM_NP * sizeof(float), s->stream));
  MatArgs ma;
  for (int k = 0; k < MAT_N; ++k) ma.a[k] = mp[k];
  k_pack_material<<<(P.B + 127) / 128, 128, 0, s->stream>>>(P.B, ma, s->mat);
  k_build_kin<<<(P.B + 127) / 128, 128, 0, s->stream>>>(P.B, P.N, P.NS, P.G, P.M, s->pins, s->grasp, s->cuts, s->kin);
  s->launches += 2;
  CUD(cudaGetLastError());
  CUD(cudaStreamSynchronize(s->stream));   // the material arrays are the caller's: done with them before returning
#undef CUD
  P.mat = s->mat; P.kin = s->kin; P.qloc = s->qloc; P.pose0 = s->pose0; P.finger = s->finger; P.prim = s->prim;
  P.state = s->state; P.flags = s->flags;
  *out = s;
  return DLO_OK;
}

dlo_status dlo_destroy(dlo_sim* s) {
  if (!s) return DLO_OK;
  int cur = -1;
  cudaGetDevice(&cur);
  if (cur != s->device) cudaSetDevice(s->device);   // free on the handle's own device, whatever is current
  cudaStreamSynchronize(s->stream);
  if (s->aux) cudaStreamSynchronize(s->aux);
  void* dev[] = {s->mat, s->qloc, s->pose0, s->finger, s->prim, s->state, s->state0, s->ckpt, s->acc_tape, s->adj, s->replay, s->gmat,
                 s->kin, s->pins, s->cuts, s->grasp, s->flags, s->stat, s->perm_main, s->perm_rep};
  for (void* p : dev) if (p) cudaFree(p);
  for (int k = 0; k < dlo_sim::MAX_TAPE; ++k) {
    for (void* p : {(void*)s->tapes[k], (void*)s->tape_flags[k], (void*)s->side[k], (void*)s->side_count[k], (void*)s->tape_slot[k], (void*)s->stat_rep[k]}) if (p) cudaFree(p);
    for (cudaEvent_t e : {s->ev_rep[k], s->ev_adj[k]}) if (e) cudaEventDestroy(e);
  }
  if (s->aux) cudaStreamDestroy(s->aux);
  if (s->ev_fwd) cudaEventDestroy(s->ev_fwd);
  for (auto& v : s->tev) for (cudaEvent_t e : v) cudaEventDestroy(e);
  void* stg[] = {s->dx0, s->dv0, s->dkb, s->dact, s->dxT, s->dvT, s->dsx, s->dsv, s->dga, s->dgx, s->dgv, s->dgm};
  for (void* p : stg) if (p) cudaFree(p);
  void* host[] = {s->hx0, s->hv0, s->hkb, s->hact, s->hxT, s->hvT};
  for (void* p : host) if (p) cudaFreeHost(p);
  if (cur >= 0 && cur != s->device) cudaSetDevice(cur);
  delete s;
  return DLO_OK;
}

static dlo_status rebuild_kin(dlo_sim* s) {
  const KParams& P = s->P;
  k_build_kin<<<(P.B + 127) / 128, 128, 0, s->stream>>>(P.B, P.N, P.NS, P.G, P.M, s->pins, s->grasp, s->cuts, s->kin);
  s->launches += 1;
  CU(cudaGetLastError());
  s->have_state = false; s->have_q = false;
  return DLO_OK;
}

dlo_status dlo_set_pins(dlo_sim* s, const uint8_t* pinned) {
  ENTER(s);
  if (!pinned) return fail(DLO_ERR_INVALID_ARG, "NULL argument");
  CU(cudaMemcpyAsync(s->pins, pinned, (size_t)s->P.B * s->P.N, cudaMemcpyDeviceToDevice, s->stream));
  return rebuild_kin(s);
}

dlo_status dlo_set_cuts(dlo_sim* s, const uint8_t* cut) {
  ENTER(s);
  if (!cut) return fail(DLO_ERR_INVALID_ARG, "NULL argument");
  if (s->P.ring) return fail(DLO_ERR_UNSUPPORTED, "dlo_set_cuts needs the open topology (the ropes lie back to back in one vertex array)");
  if (s->P.self_contact && s->P.self_skip != 2) return fail(DLO_ERR_UNSUPPORTED, "dlo_set_cuts with self-contact needs self_skip == 2");
  if (!s->cuts) CU(dalloc(&s->cuts, (size_t)s->P.B * s->P.N));
  CU(cudaMemcpyAsync(s->cuts, cut, (size_t)s->P.B * s->P.N, cudaMemcpyDeviceToDevice, s->stream));
  return rebuild_kin(s);
}

dlo_status dlo_set_primitives(dlo_sim* s, const int32_t* types, const float* params) {
  ENTER(s);
  if (s->P.K == 0) return DLO_OK;
  if (!types || !params) return fail(DLO_ERR_INVALID_ARG, "NULL argument");
  for (int k = 0; k < s->P.K; ++k) {
    if (types[k] < 0 || types[k] > 3) return fail(DLO_ERR_INVALID_ARG, "unknown primitive type");
    s->P.prim_type[k] = types[k];
  }
  s->P.prim_pack = 0u;
  for (int k = 0; k < s->P.K; ++k) s->P.prim_pack |= (unsigned)types[k] << (2 * k);
  CU(cudaMemcpyAsync(s->prim, params, (size_t)s->P.B * s->P.K * PRIM_NP * sizeof(float), cudaMemcpyDeviceToDevice, s->stream));
  s->have_prims = true;
  return DLO_OK;
}

dlo_status dlo_set_grippers(dlo_sim* s, const float* init_pose, const float* finger_geom, const int32_t* grasp_verts) {
  ENTER(s);
  if (s->P.G == 0) return DLO_OK;
  if (!init_pose || !finger_geom || !grasp_verts) return fail(DLO_ERR_INVALID_ARG, "NULL argument");
  const size_t BG = (size_t)s->P.B * s->P.G;
  CU(cudaMemcpyAsync(s->pose0, init_pose, BG * 6 * sizeof(float), cudaMemcpyDeviceToDevice, s->stream));
  CU(cudaMemcpyAsync(s->finger, finger_geom, BG * 4 * sizeof(float), cudaMemcpyDeviceToDevice, s->stream));
  CU(cudaMemcpyAsync(s->grasp, grasp_verts, BG * s->P.M * sizeof(int), cudaMemcpyDeviceToDevice, s->stream));
  s->have_grippers = true;
  return rebuild_kin(s);
}

dlo_status dlo_set_state(dlo_sim* s, const float* x0, const float* v0, const float* kb0) {
  ENTER(s);
  if (!x0 || !v0) return fail(DLO_ERR_INVALID_ARG, "NULL argument");
  const KParams& P = s->P;
  if (P.K > 0 && !s->have_prims) return fail(DLO_ERR_BAD_STATE, "dlo_set_primitives must precede dlo_set_state");
  if (P.G > 0 && !s->have_grippers) return fail(DLO_ERR_BAD_STATE, "dlo_set_grippers must precede dlo_set_state");
  SetupArgs A;
  A.B = P.B; A.N = P.N; A.E = P.E; A.NS = P.NS; A.ring = P.ring; A.G = P.G; A.M = P.M; A.kappa_from_x0 = s->cfg.kappa_bar_from_x0;
  A.x0 = x0; A.v0 = v0; A.kb0 = kb0; A.pose0 = s->pose0; A.grasp_verts = s->grasp; A.state = s->state0; A.qloc = s->qloc; A.cuts = s->cuts;
  k_set_state<<<(P.B + 63) / 64, 64, 0, s->stream>>>(A);
  s->launches += 1;
  CU(cudaGetLastError());
  CU(cudaMemcpyAsync(s->state, s->state0, (size_t)P.B * s->blk * sizeof(float), cudaMemcpyDeviceToDevice, s->stream));
  CU(cudaMemsetAsync(s->flags, 0, (size_t)P.B * sizeof(int), s->stream));
  s->have_state = true; s->have_q = true; s->have_adj = false;
  s->H_done = 0; s->stride = 0; s->t_start = 0;
  return DLO_OK;
}

dlo_status dlo_restore_state(dlo_sim* s, const float* x, const float* x_lo, const float* v, const float* d1, const float* kb, int32_t step_index) {
  ENTER(s);
  if (!x || !v || !d1 || !kb) return fail(DLO_ERR_INVALID_ARG, "NULL argument (x, v, d1 and kappa_bar are all required)");
  if (step_index < 0) return fail(DLO_ERR_INVALID_ARG, "step_index < 0");
  if (!s->have_q) return fail(DLO_ERR_BAD_STATE, "dlo_restore_state needs an earlier dlo_set_state on this scene (grasp-local coordinates are captured there)");
  const KParams& P = s->P;
  const size_t n = (size_t)P.B * s->blk;
  k_put_state<<<(unsigned)((n + 255) / 256), 256, 0, s->stream>>>(P.B, P.N, P.NS, x, v, d1, kb, x_lo, s->state0);
  s->launches += 1;
  CU(cudaGetLastError());
  CU(cudaMemcpyAsync(s->state, s->state0, n * sizeof(float), cudaMemcpyDeviceToDevice, s->stream));
  s->have_state = true; s->have_adj = false;
  s->H_done = 0; s->stride = 0; s->t_start = step_index;
  return DLO_OK;
}

dlo_status dlo_set_actions(dlo_sim* s, const float* actions, int32_t horizon) {
  ENTER(s);
  if (horizon < 0) return fail(DLO_ERR_INVALID_ARG, "horizon < 0");
  if (s->P.G > 0 && horizon > 0 && !actions) return fail(DLO_ERR_INVALID_ARG, "actions is NULL");
  s->actions = actions; s->H_actions = horizon; s->P.actions = actions;
  return DLO_OK;
}

}  // extern "C"

template <int VPL, bool TAPE> static cudaError_t launch_forward_t(dlo_sim* s, const KParams& P, int t0, int t1, int stride, cudaStream_t st) {
  cudaError_t e = cudaFuncSetAttribute(k_forward<VPL, TAPE>, cudaFuncAttributeMaxDynamicSharedMemorySize, s->smem_fwd > 48 * 1024 ? s->smem_fwd : 48 * 1024);
  if (e != cudaSuccess) return e;
  const int grid = (P.B + s->wpb_fwd - 1) / s->wpb_fwd;
  {
    LaunchTimer lt(s, TAPE ? 1 : 0, st, (int64_t)P.B * (t1 - t0));
    k_forward<VPL, TAPE><<<grid, s->wpb_fwd * 32, s->smem_fwd, st>>>(P, t0, t1, stride);
  }
  s->launches += 1;
  return cudaGetLastError();
}
// forward (tape = false) or replay of a segment with tape records (tape = true); P carries the buffers to use
static cudaError_t launch_forward(dlo_sim* s, KParams P, int t0, int t1, int stride, bool tape, cudaStream_t st) {
  smem_layout(P, s->VPL, false);
#define DLO_FWD_CASE(V) return tape ? launch_forward_t<V, true>(s, P, t0, t1, stride, st) : launch_forward_t<V, false>(s, P, t0, t1, stride, st)
  switch (s->VPL) {
#ifdef DLO_VPL_ONLY   /* development builds: one instantiation only */
    default: DLO_FWD_CASE(DLO_VPL_ONLY);
#else
    case 2: DLO_FWD_CASE(2);
    case 4: DLO_FWD_CASE(4);
    case 6: DLO_FWD_CASE(6);
    default: DLO_FWD_CASE(8);
#endif
  }
#undef DLO_FWD_CASE
}

static cudaError_t sort_envs(dlo_sim* s, const int* stat, int col, int shift, int* perm, cudaStream_t st) {
  k_sort_envs<<<1, 1024, 0, st>>>(s->P.B, stat, col, shift, perm);
  s->launches += 1;
  return cudaGetLastError();
}
// frames [t0, t1) of the plain forward rollout.  With sort_mode bit 0: in launches of s->chunk frames, from the second on
// with the envs in the order of the self-contact work they did in the launch before (measured: no gain for the forward,
// whose waiting warps leave their issue slots to the SM's other CTA; off by default)
static cudaError_t forward_chunks(dlo_sim* s, int t0, int t1, int stride) {
  const bool on = (s->sort_mode & 1) != 0;
  for (int a = t0; a < t1;) {
    const int b = (on && a + s->chunk < t1) ? a + s->chunk : t1;
    KParams Pc = s->P;
    Pc.stat = on ? s->stat : nullptr;
    Pc.perm = nullptr;
    if (on && s->stat_valid) {
      cudaError_t e = sort_envs(s, s->stat, 0, 4, s->perm_main, s->stream);
      if (e != cudaSuccess) return e;
      Pc.perm = s->perm_main;
    }
    cudaError_t e = launch_forward(s, Pc, a, b, stride, false, s->stream);
    if (e != cudaSuccess) return e;
    s->stat_valid = on;
    a = b;
  }
  return cudaSuccess;
}

// Tape buffers, one checkpoint segment each: the first is required, up to min(#segments, max_tape) are taken while memory
// allows.  Each comes with its optional side-record pool.
static void free_tape_buffer(dlo_sim* s, int k) {
  for (void* p : {(void*)s->tapes[k], (void*)s->tape_flags[k], (void*)s->side[k], (void*)s->side_count[k], (void*)s->tape_slot[k]}) if (p) cudaFree(p);
  s->tapes[k] = nullptr; s->tape_flags[k] = nullptr; s->side[k] = nullptr; s->side_count[k] = nullptr; s->tape_slot[k] = nullptr;
}
static dlo_status ensure_tape(dlo_sim* s, int H, int stride) {
  const int B = s->P.B;
  const size_t rec = (size_t)tape_rows(s->P.N_C) * s->P.NS, seg = (size_t)(stride < H ? stride : H) * s->P.n_sub + 1;
  const int nseg = (H + stride - 1) / stride;
  if (seg > s->tape_blocks) {   // a longer segment than the buffers hold: start over
    CU(cudaStreamSynchronize(s->stream));
    if (s->aux) CU(cudaStreamSynchronize(s->aux));
    for (int k = 0; k < dlo_sim::MAX_TAPE; ++k) free_tape_buffer(s, k);
    s->n_tape = 0; s->tape_blocks = 0; s->side_cap = 0;
    s->tape_lo = 1 << 30;
    CU(dalloc(&s->tapes[0], seg * B * rec));
    CU(dalloc(&s->tape_flags[0], seg * B));
    s->tape_blocks = seg;
    s->n_tape = 1;
  }
  const bool want_side = s->P.self_contact && !getenv("DLO_NO_SIDE");
  if (want_side) {
    // side records for one substep in twelve (config 5 uses one in thirty); a substep that finds the pool empty is
    // recomputed by the reverse pass instead.  Optional: without the memory the reverse pass recomputes them all.
    s->side_floats = side_record_floats(s->P, 33 * s->VPL);
    s->side_cap = (int)std::min<size_t>((size_t)1 << 30, std::max<size_t>(1024, s->tape_blocks * B / 12));
  }
  auto side_pool = [&](int k) {
    if (!want_side || s->side[k]) return;
    const bool ok = cudaMalloc((void**)&s->side[k], (size_t)s->side_cap * s->side_floats * sizeof(float)) == cudaSuccess &&
                    cudaMalloc((void**)&s->side_count[k], sizeof(int)) == cudaSuccess &&
                    cudaMalloc((void**)&s->tape_slot[k], s->tape_blocks * B * sizeof(int)) == cudaSuccess;
    if (!ok) {
      cudaGetLastError();
      for (void* p : {(void*)s->side[k], (void*)s->side_count[k], (void*)s->tape_slot[k]}) if (p) cudaFree(p);
      s->side[k] = nullptr; s->side_count[k] = nullptr; s->tape_slot[k] = nullptr;
    }
  };
  side_pool(0);
  const int want = std::min(nseg, s->max_tape);
  const size_t tape_bytes = s->tape_blocks * B * rec * sizeof(float);
  const size_t side_bytes = want_side ? (size_t)s->side_cap * s->side_floats * sizeof(float) + s->tape_blocks * B * sizeof(int) : 0;
  while (s->n_tape < want) {
    const int k = s->n_tape;
    if (k >= 2) {   // beyond double buffering: only out of memory nobody else is likely to need (a tenth of the device stays free)
      size_t free_b = 0, total_b = 0;
      if (cudaMemGetInfo(&free_b, &total_b) != cudaSuccess) { cudaGetLastError(); break; }
      if (free_b < tape_bytes + side_bytes + total_b / 10) break;
    }
    if (cudaMalloc((void**)&s->tapes[k], tape_bytes) != cudaSuccess || cudaMalloc((void**)&s->tape_flags[k], s->tape_blocks * B) != cudaSuccess) {
      cudaGetLastError();
      free_tape_buffer(s, k);
      break;
    }
    side_pool(k);
    s->n_tape = k + 1;
  }
  return DLO_OK;
}

extern "C" {

dlo_status dlo_rollout_forward(dlo_sim* s, int32_t horizon, int32_t stride) {
  ENTER(s);
  if (!s->have_state) return fail(DLO_ERR_BAD_STATE, "dlo_set_state has not been called (or the scene changed since)");
  if (horizon < 0 || stride < 0) return fail(DLO_ERR_INVALID_ARG, "horizon < 0 or checkpoint_stride < 0");
  if (s->P.G > 0 && s->t_start + horizon > s->H_actions) return fail(DLO_ERR_INVALID_ARG, "start frame + horizon exceeds the actions given to dlo_set_actions");
  s->P.t_base = s->t_start;
  s->have_adj = false;
  const KParams& P = s->P;
  const size_t blk_bytes = s->blk * sizeof(float) * P.B;
  CU(cudaMemcpyAsync(s->state, s->state0, blk_bytes, cudaMemcpyDeviceToDevice, s->stream));
  s->H_done = 0; s->stride = 0;
  if (stride > 0) {
    const size_t need = (size_t)horizon / stride + 1;
    if (need > s->ckpt_blocks) {
      CU(cudaStreamSynchronize(s->stream));
      if (s->ckpt) cudaFree(s->ckpt);
      s->ckpt = nullptr; s->ckpt_blocks = 0;
      CU(dalloc(&s->ckpt, need * P.B * s->blk));
      s->ckpt_blocks = need;
    }
    s->P.ckpt = s->ckpt;
    CU(cudaMemcpyAsync(s->ckpt, s->state0, blk_bytes, cudaMemcpyDeviceToDevice, s->stream));   // checkpoint 0 = initial state
  }
  s->tape_lo = 1 << 30; s->tape_K = 0;
  s->stat_valid = false;
  for (bool& v : s->stat_rep_valid) v = false;
  if (horizon > 0 && stride > 0) {
    // the last n_tape segments are run in tape mode, so that the reverse pass can start without replaying them
    dlo_status st = ensure_tape(s, horizon, stride);
    if (st) return st;
    const int nseg = (horizon + stride - 1) / stride, K = s->n_tape, lo = nseg - std::min(K, nseg);
    if (lo > 0) CU(forward_chunks(s, 0, lo * stride, stride));
    for (int g = lo; g < nseg; ++g) {
      const int buf = g % K, t0 = g * stride, t1 = std::min(t0 + stride, (int)horizon);
      KParams Pf = s->P;
      Pf.tape = s->tapes[buf];
      Pf.tape_flag = s->tape_flags[buf];
      if (s->side[buf]) {
        CU(cudaMemsetAsync(s->side_count[buf], 0, sizeof(int), s->stream));
        Pf.side = s->side[buf]; Pf.side_count = s->side_count[buf]; Pf.tape_slot = s->tape_slot[buf]; Pf.side_cap = s->side_cap; Pf.side_floats = s->side_floats;
      }
      if (s->sort_mode) {
        Pf.stat = s->stat_rep[buf];
        if ((s->sort_mode & 1) && s->stat_valid) { CU(sort_envs(s, s->stat, 0, 4, s->perm_main, s->stream)); Pf.perm = s->perm_main; }
      }
      CU(launch_forward(s, Pf, t0, t1, stride, true, s->stream));
      s->stat_rep_valid[buf] = s->sort_mode != 0;
    }
    s->tape_lo = lo; s->tape_K = K;
  } else if (horizon > 0) CU(forward_chunks(s, 0, horizon, stride));
  s->H_done = horizon; s->stride = stride;
  return DLO_OK;
}

dlo_status dlo_get_state(dlo_sim* s, float* x, float* v, float* d1, float* kb) {
  ENTER(s);
  if (!s->have_state) return fail(DLO_ERR_BAD_STATE, "no state");
  const KParams& P = s->P;
  const size_t n = (size_t)P.B * STATE_ROWS * P.N;
  k_get_state<<<(unsigned)((n + 255) / 256), 256, 0, s->stream>>>(P.B, P.N, P.NS, s->state, x, v, d1, kb, nullptr);
  s->launches += 1;
  CU(cudaGetLastError());
  return DLO_OK;
}

dlo_status dlo_get_position_residual(dlo_sim* s, float* x_lo) {
  ENTER(s);
  if (!x_lo) return fail(DLO_ERR_INVALID_ARG, "NULL argument");
  if (!s->have_state) return fail(DLO_ERR_BAD_STATE, "no state");
  const KParams& P = s->P;
  const size_t n = (size_t)P.B * STATE_ROWS * P.N;
  k_get_state<<<(unsigned)((n + 255) / 256), 256, 0, s->stream>>>(P.B, P.N, P.NS, s->state, nullptr, nullptr, nullptr, nullptr, x_lo);
  s->launches += 1;
  CU(cudaGetLastError());
  return DLO_OK;
}

dlo_status dlo_check_numerics(dlo_sim* s, int32_t* n_bad) {
  ENTER(s);
  std::vector<int> f(s->P.B);
  CU(cudaMemcpyAsync(f.data(), s->flags, f.size() * sizeof(int), cudaMemcpyDeviceToHost, s->stream));
  CU(cudaStreamSynchronize(s->stream));
  int bad = 0, ovf = 0;
  int grd = 0;
  for (int v : f) { bad += v != 0; ovf += (v & FLAG_CAND_OVERFLOW) != 0; grd += (v & FLAG_GUARD) != 0; }
  if (n_bad) *n_bad = bad;
  if (bad) return fail(DLO_ERR_NUMERIC, std::to_string(bad) + " env(s) flagged (" + std::to_string(ovf) + " self-contact candidate overflow, " +
                                            std::to_string(grd) + " shared-memory guard, rest non-finite)");
  return DLO_OK;
}

}  // extern "C"

#include "dlo_api_backward.inl"
#include "dlo_bench.inl"
#include "dlo_noalloc.inl"
