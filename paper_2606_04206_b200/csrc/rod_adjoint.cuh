// rod_adjoint.cuh — reverse pass of one substep for one env held by one warp, and the segment adjoint kernel.
//
// the rollout is replayed segment by segment from its checkpoints and differentiated backwards.
// Here the replay (k_forward with write_tape) leaves the state at the start of every substep of the segment in
// HBM; k_adjoint then walks the substeps in reverse.  For each it (1) recomputes the substep forward with REC
// (keeping the Eq.10 multipliers in shared memory and the few self-contact corrections in an L2-resident
// scratch), (2) applies the transposed Jacobian of A9..A1 in reverse order using the per-element adjoints of
// rod_adj.cuh.  The Eq.10 sweeps are undone exactly from the stored multipliers (the update of an edge is
// invertible given lambda), so no per-sweep position snapshots are needed.  Lane <-> vertex mapping, shuffles
// and shared-memory use mirror rod_substep.cuh; every forward gather becomes a scatter to the same neighbour.
#pragma once
#include "rod_adj.cuh"
#include "rod_substep.cuh"

namespace dlo {

template <int VPL> struct LaneAdj {
  f3 x[VPL], v[VPL], d1[VPL];
  float kb1[VPL], kb2[VPL];
};
template <int VPL> __device__ __forceinline__ void load_adj(const float* __restrict__ blk, int base, int NS, LaneAdj<VPL>& a) {
  LaneState<VPL> s;
  load_state<VPL>(blk, base, NS, s);
#pragma unroll
  for (int k = 0; k < VPL; ++k) { a.x[k] = s.x[k]; a.v[k] = s.v[k]; a.d1[k] = s.d1[k]; a.kb1[k] = s.kb1[k]; a.kb2[k] = s.kb2[k]; }
}
template <int VPL> __device__ __forceinline__ void store_adj(float* __restrict__ blk, int base, int NS, const LaneAdj<VPL>& a) {
  LaneState<VPL> s;
#pragma unroll
  for (int k = 0; k < VPL; ++k) { s.x[k] = a.x[k]; s.v[k] = a.v[k]; s.d1[k] = a.d1[k]; s.kb1[k] = a.kb1[k]; s.kb2[k] = a.kb2[k]; }
  store_state<VPL>(blk, base, NS, s);
}

enum { GM_STRETCH = 0, GM_ALPHA = 1, GM_GAMMA = 2, GM_SIGY = 3, GM_RC = 4 };
struct GradAcc { double gm[5]; float apbar[6], acbar[6]; };   // material adjoints: sums of cancelling terms over all substeps, kept in double

// add `val` to the array element at the lane's last valid slot
template <int VPL> __device__ __forceinline__ void add_at_last(f3 a[VPL], int ks, const f3& val) {
#pragma unroll
  for (int k = 0; k < VPL; ++k) if (k == ks) a[k] += val;
}
template <int VPL> __device__ __forceinline__ void add_at_last(float a[VPL], int ks, float val) {
#pragma unroll
  for (int k = 0; k < VPL; ++k) if (k == ks) a[k] += val;
}
// scatter an edge-vector adjoint: -= at the edge's own vertex, += at its next vertex (local slot or `send`)
template <int VPL> __device__ __forceinline__ void scatter_edge(f3 a[VPL], f3& send, int k, int ks, const f3& eb) {
  a[k] -= eb;
  if (k == VPL - 1 || k == ks) send += eb;
  else a[k + 1 < VPL ? k + 1 : k] += eb;
}

// pose adjoints live in shared memory: per gripper P0bar (p 3, R 9) then P1bar (p 3, R 9)
__device__ __forceinline__ void posebar_add(float* dst, const PoseBar<float>& g) {
  atomicAdd(dst + 0, g.p.x); atomicAdd(dst + 1, g.p.y); atomicAdd(dst + 2, g.p.z);
#pragma unroll
  for (int k = 0; k < 9; ++k) atomicAdd(dst + 3 + k, g.R[k]);
}
// Adjoint of the grasp targets p1 + R1 q of a lane's kinematic vertices, summed per gripper in registers and added to
// the shared pose adjoint once (flush): consecutive vertices of a lane usually hang on the same gripper, and a
// shared-memory float atomicAdd is a compare-and-swap loop (twelve of them per vertex otherwise).
struct GraspAcc {
  PoseBar<float> b;
  int g;
  __device__ __forceinline__ void init() { pose_bar_zero(b); g = -1; }
  __device__ __forceinline__ void flush(const WarpSmem& sm) {
    if (g >= 0) posebar_add(sm.posebar + g * 24 + 12, b);
    g = -1;
  }
  __device__ __forceinline__ void add(const KParams& P, const WarpSmem& sm, int code, const f3& tbar) {
    const int slot = code - KIN_GRASP0, gg = (slot >= P.M) + (slot >= 2 * P.M) + (slot >= 3 * P.M);
    if (gg != g) { flush(sm); pose_bar_zero(b); g = gg; }
    const float* q = sm.q + 3 * slot;
    rigid_point_adj<float>(mk3<float>(q[0], q[1], q[2]), tbar, b);
  }
};

// one rigid body (primitive b < K, else finger (b-K)) evaluated at y: phi, n, body velocity
__device__ __forceinline__ bool body_eval(const CoupleConst& P, const WarpSmem& sm, int b, const f3& y, float& phi, f3& n, f3& vb) {
  vb = zero3<float>();
  if (b < P.K) return sdf_eval_pre<float>((int)((P.types >> (2 * b)) & 3u), sm.prim + b * PRIM_SM_STRIDE, y, phi, n);
  const int g = (b - P.K) >> 1, fk = (b - P.K) & 1;
  const float* o = sm.pose + g * POSE_STRIDE;
  const float* A = o + (fk ? POSE_FA1 : POSE_FA0);
  const float* Bp = o + (fk ? POSE_FB1 : POSE_FB0);
  const float Pc[7] = {A[0], A[1], A[2], Bp[0], Bp[1], Bp[2], o[POSE_RF]};
  if (!sdf_eval<float>(1, Pc, y, phi, n)) return false;
  vb = finger_body_velocity(o, y, P.inv_h);   // the forward's expression: same bits, same branches
  return true;
}

// reverse of A7 for one free vertex: `active` = bodies that responded (forward order = bit order), v3 = velocity
// before the coupling.  velbar: in = adjoint of v4, out = adjoint of v3.  ybar += adjoint of y.
struct CoupleAdj { f3 velbar, ybar; };
__device__ __noinline__ CoupleAdj rigid_coupling_adj(const KParams& __restrict__ KP, const CoupleConst P, float* smbase, int np, int env, unsigned active, f3 y, f3 v3, float mu_r,
                                                     f3 velbar) {
  WarpSmem sm;
  sm.init(KP, smbase, np);
  f3 ybar = zero3<float>();
  unsigned m = active;
  while (m) {
    const int b = 31 - __clz(m);
    m &= ~(1u << b);
    // velocity seen by body b: replay the earlier active bodies
    f3 v = v3;
    unsigned lo = active & ((1u << b) - 1u);
    while (lo) {
      const int b2 = __ffs(lo) - 1;
      lo &= lo - 1;
      float phi; f3 n, vb;
      if (body_eval(P, sm, b2, y, phi, n, vb)) rigid_response<float>(v, vb, n, P.r - phi, P.inv_eps, P.f_thresh, P.e_rest, mu_r);
    }
    float phi; f3 n, vb;
    if (!body_eval(P, sm, b, y, phi, n, vb)) continue;
    f3 vbar = zero3<float>(), vbbar = zero3<float>(), nbar = zero3<float>();
    const float dbar = rigid_response_adj<float>(v, vb, n, P.r - phi, P.inv_eps, P.e_rest, mu_r, velbar, vbar, vbbar, nbar);
    velbar = vbar;
    const float phibar = -dbar;
    if (b < P.K) sdf_pre_adj<float>((int)((P.types >> (2 * b)) & 3u), sm.prim + b * PRIM_SM_STRIDE, y, phibar, nbar, ybar);
    else {
      const int g = (b - P.K) >> 1, fk = (b - P.K) & 1;
      const float* o = sm.pose + g * POSE_STRIDE;
      const float* A = o + (fk ? POSE_FA1 : POSE_FA0);
      const float* Bp = o + (fk ? POSE_FB1 : POSE_FB0);
      f3 Abar = zero3<float>(), Bbar = zero3<float>();
      sdf_capsule_adj<float>(mk3<float>(A[0], A[1], A[2]), mk3<float>(Bp[0], Bp[1], Bp[2]), y, phibar, nbar, ybar, Abar, Bbar);
      PoseBar<float> b0, b1;
      pose_bar_zero(b0); pose_bar_zero(b1);
      const float* fg = KP.finger + ((size_t)env * P.G + g) * 4;
      const float sx = (fk ? -0.5f : 0.5f) * fg[0];
      rigid_point_adj<float>(mk3<float>(sx, 0.f, 0.f), Abar, b1);
      rigid_point_adj<float>(mk3<float>(sx, 0.f, fg[1]), Bbar, b1);
      body_point_velocity_adj<float>(read_pose(o, 0), read_pose(o, 1), y, P.inv_h, vbbar, ybar, b0, b1);
      posebar_add(sm.posebar + g * 24, b0);
      posebar_add(sm.posebar + g * 24 + 12, b1);
    }
  }
  CoupleAdj out;
  out.velbar = velbar; out.ybar = ybar;
  return out;
}

// serialised scatter of four vertex adjoints (positions -> ybar, optionally velocities -> acc)
__device__ __forceinline__ void ordered_scatter_vec4(unsigned hits, int lane, float* dst, int NP, const int iv[4], const f3 xb[4]) {
  while (hits) {
    const int src = __ffs(hits) - 1;
    hits &= hits - 1;
    if (lane == src) {
#pragma unroll
      for (int k = 0; k < 4; ++k) { dst[iv[k]] += xb[k].x; dst[NP + iv[k]] += xb[k].y; dst[2 * NP + iv[k]] += xb[k].z; }
    }
    __syncwarp();
  }
}
template <int VPL> __device__ __forceinline__ void cand_verts(const WarpSmem& sm, int N, int p, int iv[4]) {
  const unsigned c = sm.cand[p];
  iv[0] = c >> 8; iv[2] = c & 255; iv[1] = (iv[0] + 1 < N) ? iv[0] + 1 : 0; iv[3] = (iv[2] + 1 < N) ? iv[2] + 1 : 0;
#pragma unroll
  for (int k = 0; k < 4; ++k) iv[k] = vpos<VPL>(iv[k]);   // shared-memory positions
}

// reverse of one Eq.13 Jacobi pass: positions y (before the pass) in sm.ys, adjoint of the post-pass corrections
// in sm.vbar, adjoint of D_p in sm.dpbar; position adjoints are summed into sm.ybar
template <int VPL> __device__ __noinline__ void contact_pass_adj(const KParams& __restrict__ P, int lane, float* smbase, int ncand) {
  WarpSmem sm;
  sm.init(P, smbase, 33 * VPL);
  const int NP = sm.NP, N = P.N;
  const float rsum = 2.0f * P.r;
  for (int p0 = 0; p0 < ncand; p0 += 32) {
    const int p = p0 + lane;
    bool hit = false;
    int iv[4] = {0, 0, 0, 0};
    f3 xb[4] = {zero3<float>(), zero3<float>(), zero3<float>(), zero3<float>()};
    if (p < ncand) {
      cand_verts<VPL>(sm, N, p, iv);
      f3 xs[4], ob[4];
      float ws[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) { xs[k] = lds3(sm.ys, NP, iv[k]); ob[k] = lds3(sm.vbar, NP, iv[k]); ws[k] = sm.mid[4 * NP + iv[k]]; }
      f3 ea = xs[1] - xs[0], eb = xs[3] - xs[2];
      f3 dm = (xs[0] + 0.5f * ea) - (xs[2] + 0.5f * eb);
      const float reach = 0.5f * (sqrt_(dot(ea, ea)) + sqrt_(dot(eb, eb))) + rsum;
      if (dot(dm, dm) < reach * reach) hit = contact_adj<float>(xs, ws, rsum, ob, sm.dpbar[p], xb);
    }
    ordered_scatter_vec4(__ballot_sync(DLO_FULL, hit), lane, sm.ybar, NP, iv, xb);
  }
}

// reverse of the friction pass: y in sm.ys, v^2 in sm.vs, adjoint of v^3 in sm.vbar; writes sm.dpbar, sums
// position adjoints into sm.ybar and velocity adjoints into sm.acc
template <int VPL> __device__ __noinline__ void friction_pass_adj(const KParams& __restrict__ P, int lane, float* smbase, int ncand, float mu_s) {
  WarpSmem sm;
  sm.init(P, smbase, 33 * VPL);
  const int NP = sm.NP, N = P.N;
  for (int p0 = 0; p0 < ncand; p0 += 32) {
    const int p = p0 + lane;
    bool hit = false;
    int iv[4] = {0, 0, 0, 0};
    f3 xb[4] = {zero3<float>(), zero3<float>(), zero3<float>(), zero3<float>()};
    f3 vb[4] = {zero3<float>(), zero3<float>(), zero3<float>(), zero3<float>()};
    if (p < ncand && sm.dp[p] > 0.0f) {
      cand_verts<VPL>(sm, N, p, iv);
      f3 xs[4], vv[4], ob[4];
      float ws[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) { xs[k] = lds3(sm.ys, NP, iv[k]); vv[k] = lds3(sm.vs, NP, iv[k]); ob[k] = lds3(sm.vbar, NP, iv[k]); ws[k] = sm.mid[4 * NP + iv[k]]; }
      float dpb = 0.0f;
      hit = friction_adj<float>(xs, vv, ws, sm.dp[p], mu_s, P.inv_h, ob, xb, vb, dpb);
      sm.dpbar[p] = dpb;
    }
    const unsigned hits = __ballot_sync(DLO_FULL, hit);
    ordered_scatter_vec4(hits, lane, sm.ybar, NP, iv, xb);
    ordered_scatter_vec4(hits, lane, sm.acc, NP, iv, vb);
  }
}

}  // namespace dlo
#include "rod_adjoint2.cuh"
