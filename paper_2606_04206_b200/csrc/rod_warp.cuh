// rod_warp.cuh — one warp <-> one env: lane topology, state I/O and the forward substep shared by the forward
// kernel and the replay half of the adjoint kernel.
//
// Mapping.  Lane l owns the VPL consecutive vertices base = l*VPL .. base+VPL-1 and the
// edges with the same indices (edge j joins j and j+1; ring: E-1 joins N-1 and 0).  VPL is even, so an edge's
// red/black colour (j & 1) is a compile-time property of its slot: red (even) edges have both end points in
// the same lane, black (odd) edges cross to slot 0 of the next lane only at the lane's last slot.  The whole
// state lives in registers across all substeps of a launch; lanes talk through warp shuffles only, shared
// memory holds what needs indexed access (gripper poses, primitive parameters, self-contact scratch).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "rod_ops.cuh"

namespace dlo {

typedef V3<float> f3;
enum { KIN_FREE = 0, KIN_PINNED = 1, KIN_GRASP0 = 2 };   // kin code >= 2: grasped, slot = code - 2 = g*M + k
enum { KIN_CUT = 0x80 };   // bit 7 of the kin byte of vertex i: the edge (i, i+1) does not exist (several DLOs in one env, dlo_set_cuts)
enum { MAT_M = 0, MAT_L0, MAT_STRETCH, MAT_ALPHA, MAT_GAMMA, MAT_SIGY, MAT_RC, MAT_MUR, MAT_MUS, MAT_N };
// rows of one env's state block.  Positions are kept as an unevaluated sum x + xl of two floats (xl = what the fp32 rounding
// of x + h v dropped, |xl| <= ulp(x)/2): an fp32 position at 0.5 m carries 3e-8 m of rounding, which the next substep's Eq.10
// projection turns into 3e-8 / h = 3e-4 m/s of velocity noise - as large as the Coulomb stick threshold mu g h of a vertex
// resting on the ground.  With the residual carried along, edge vectors are exact differences (noise 5e-10 m, 2e-6 m/s).
enum { ROW_X = 0, ROW_V = 3, ROW_D1 = 6, ROW_KB = 9, ROW_XL = 11, STATE_ROWS = 14 };
enum { FLAG_NONFINITE = 1, FLAG_CAND_OVERFLOW = 2, FLAG_GUARD = 4 /* DLO_CHECKS: a shared-memory region was written past its end */ };
#define DLO_GUARD_WORD 0x7fc0dead   /* a NaN bit pattern no computation produces */
#define DLO_FULL 0xffffffffu
// primitives in shared memory: [0..14] parameters (boxes expanded to centre(3), half(3), R(9)), [16..18] centre and [19]
// radius of a bounding sphere (radius < 0: unbounded, e.g. a plane) used to cull vertices that are out of reach
enum { PRIM_NP = 10, PRIM_SM_STRIDE = 20, PRIM_BC = 16, PRIM_BR = 19 };

struct KParams {
  int B, N, E, NS /* padded row length */, ring, odd_ring, n_sub, N_C, stretch_mode, plasticity, self_contact, self_skip;
  int G, M, K, cand_cap, hot_cap;
  unsigned phase_mask;   // which of the lockstep phase barriers are taken (tuning: DLO_PHASES; bit = site)
  int checks;            // DLO_CHECKS=1: guard words behind every per-warp shared-memory region, verified when a kernel ends
  int n_guard, sm_guard[24];   // their positions (float offsets from the warp's base)
  int t_base;            // frame index of the rollout's first step: step t of the launch uses actions[t_base + t - 1], actions[t_base + t]
  float h, inv_h, g[3], r, inv_eps, f_thresh, e_rest, log_thresh_lo /* log(f_thresh) - 0.01 */;
  int vote_mode;         // bit 0: the warps of a CTA refresh their contact data together; bit 1: ... and rebuild their pair lists together
  float near_dist;       // pairs closer than this at a full filter go to the near list (measured every substep)
  float list_margin;     // the self-contact pair list stays valid while no vertex has moved further than this since it was built
  int prim_type[16];
  unsigned prim_pack;    // prim_type[k] in bits 2k, 2k+1 (what the non-inlined A7 takes by value)
  const float* mat;      // [B][MAT_N]
  const uint8_t* kin;    // [B][NS]
  const float* qloc;     // [B][G*M][3]
  const float* pose0;    // [B][G][6]
  const float* finger;   // [B][G][4]
  const float* prim;     // [B][K][10]
  const float* actions;  // [H][B][G][6]
  float* state;          // [B][11][NS]
  float* ckpt;           // [n_ckpt][B][11][NS]
  float* tape;           // [stride*n_sub][B][11][NS]
  int* flags;            // [B]
  float* adj;            // [B][11][NS] running state adjoint of the reverse pass
  float* acc_tape;       // [B][N_C][3][32*VPL] self-contact corrections of the substep being reversed
  float* gmat;           // [B][5] running material gradient
  float* g_actions;      // [H][B][G][6] (may be null)
  // side records of the substeps that applied a self-contact correction (written by the replay, read by the adjoint
  // instead of recomputing the substep): pool of side_cap slots of side_floats floats, slot index per tape record
  float* side;
  int* side_count;
  int* tape_slot;        // [stride*n_sub][B]
  int side_cap, side_floats;
  const int* perm;       // [B] env handled by warp slot i (null: identity); set per launch, sorted by the envs' recent self-contact work
  int* stat;             // [B][2] written at the end of a forward launch: self-contact work units, time pattern of the substeps with a correction
  uint8_t* tape_flag;    // [stride*n_sub][B]: 1 if the substep applied a self-contact correction (written by the replay)
  // per-warp shared memory layout (float offsets from the warp's base), set by the host
  int sm_pose, sm_prim, sm_q, sm_ys, sm_acc, sm_vs, sm_mid, sm_dp, sm_cand, sm_lam, sm_dpbar, sm_ybar, sm_vbar, sm_posebar, sm_blk, sm_xref, sm_hot, sm_warp_floats;
};

// per-gripper block in shared memory: p0(3) R0(9) p1(3) R1(9) fingerA0(3) fingerB0(3) fingerA1(3) fingerB1(3) rf(1) pad(3)
enum { POSE_P0 = 0, POSE_R0 = 3, POSE_P1 = 12, POSE_R1 = 15, POSE_FA0 = 24, POSE_FB0 = 27, POSE_FA1 = 30, POSE_FB1 = 33, POSE_RF = 36, POSE_FC0 = 37, POSE_FC1 = 40, POSE_FRAD = 43, POSE_P0L = 44, POSE_P1L = 47, POSE_STRIDE = 52 };   // FC*: finger mid points, FRAD: bounding radius, P*L: low parts of p0, p1 (two-float)

__device__ __forceinline__ float shfl(float v, int src) { return __shfl_sync(DLO_FULL, v, src); }
__device__ __forceinline__ f3 shfl3(const f3& v, int src) { return mk3<float>(shfl(v.x, src), shfl(v.y, src), shfl(v.z, src)); }
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(DLO_FULL, v, o);
  return v;
}
// shared-memory position of vertex i: natural order plus one pad word per 32, so that both access patterns are
// bank-conflict free: the lanes' own vertices (stride VPL across lanes) and runs of consecutive vertices (candidates)
template <int VPL> __device__ __forceinline__ int vpos(int i) { return i + (i >> 5); }
// max / min over the warp of NON-NEGATIVE values (squared lengths): their bit patterns order like unsigned integers,
// so one REDUX replaces five shuffle + compare rounds.  A NaN compares above every number: it survives a max (the
// bounds built on it then fail, which is the conservative side) and is dropped by a min.
__device__ __forceinline__ float warp_max(float v) { return __uint_as_float(__reduce_max_sync(DLO_FULL, __float_as_uint(v))); }
__device__ __forceinline__ float warp_min(float v) { return __uint_as_float(__reduce_min_sync(DLO_FULL, __float_as_uint(v))); }
__device__ __forceinline__ f3 lds3(const float* s, int NP, int i) { return mk3<float>(s[i], s[NP + i], s[2 * NP + i]); }
__device__ __forceinline__ void sts3(float* s, int NP, int i, const f3& v) { s[i] = v.x; s[NP + i] = v.y; s[2 * NP + i] = v.z; }

// layout of a side record (float offsets): header (ncand, jac_mask), v^3 rows (velocity after the self-contact friction),
// candidate codes, depth sums D_p, the summed corrections of every Jacobi pass [N_C][3][33 VPL]
__host__ __device__ inline int side_off_v3() { return 4; }
__host__ __device__ inline int side_off_cand(const KParams& P) { return 4 + 3 * P.NS; }
__host__ __device__ inline int side_off_dp(const KParams& P) { return side_off_cand(P) + P.cand_cap / 2; }
__host__ __device__ inline int side_off_acc(const KParams& P) { return side_off_dp(P) + P.cand_cap; }
__host__ __device__ inline int side_record_floats(const KParams& P, int NP) { return (side_off_acc(P) + P.N_C * 3 * NP + 3) / 4 * 4; }

template <int VPL> struct Topo {
  int lane, base, nv, ks, nl, pl;   // own lane, first vertex, #valid vertices, last valid slot, next / previous lane
  bool vvalid[VPL], evalid[VPL], interior[VPL], remote_edge;   // remote_edge: the edge at slot ks crosses to lane nl
  __device__ __forceinline__ void init(const KParams& P) {
    lane = threadIdx.x & 31;
    base = lane * VPL;
    nv = min(max(P.N - base, 0), VPL);
    ks = nv - 1;
    const int last_lane = (P.N - 1) / VPL;
    nl = (base + VPL < P.N) ? lane + 1 : 0;
    pl = (lane > 0) ? lane - 1 : last_lane;
    if (lane > last_lane) { nl = lane; pl = lane; }
#pragma unroll
    for (int k = 0; k < VPL; ++k) {
      const int i = base + k;
      vvalid[k] = i < P.N;
      evalid[k] = i < P.E;
      interior[k] = vvalid[k] && (P.ring || (i >= 1 && i <= P.N - 2));
    }
    remote_edge = nv > 0 && (base + ks) < P.E && (base + ks + 1 >= P.N || ks == VPL - 1);
  }
};

// one row of a state block: NS is a multiple of 4, base = lane*VPL is even
template <int VPL> __device__ __forceinline__ void load_row(const float* __restrict__ row, int base, int NS, float out[VPL]) {
  if (VPL % 4 == 0) {
#pragma unroll
    for (int k = 0; k < VPL; k += 4) {
      float4 q = (base + k < NS) ? *reinterpret_cast<const float4*>(row + base + k) : make_float4(0.f, 0.f, 0.f, 0.f);
      out[k] = q.x; out[k + 1] = q.y; out[k + 2] = q.z; out[k + 3] = q.w;
    }
  } else {
#pragma unroll
    for (int k = 0; k < VPL; k += 2) {
      float2 q = (base + k < NS) ? *reinterpret_cast<const float2*>(row + base + k) : make_float2(0.f, 0.f);
      out[k] = q.x; out[k + 1] = q.y;
    }
  }
}
template <int VPL> __device__ __forceinline__ void store_row(float* __restrict__ row, int base, int NS, const float in[VPL]) {
  if (VPL % 4 == 0) {
#pragma unroll
    for (int k = 0; k < VPL; k += 4)
      if (base + k < NS) *reinterpret_cast<float4*>(row + base + k) = make_float4(in[k], in[k + 1], in[k + 2], in[k + 3]);
  } else {
#pragma unroll
    for (int k = 0; k < VPL; k += 2)
      if (base + k < NS) *reinterpret_cast<float2*>(row + base + k) = make_float2(in[k], in[k + 1]);
  }
}

// rows of one tape record (per substep and env), each NS floats: the state at the start of the substep, then what the
// reverse pass would otherwise have to recompute: final corrections, the velocity v^1 after the force step (x^p = x + h v^1,
// the predicted edge vectors and, without self-contact friction, v^3 = v^1 + dx/h follow from it with the forward's own
// expressions, bit for bit), Eq.10 multiplier sums, the mask of rigid bodies that responded, and the multipliers of every
// iteration.  (The position residual rows stay in the record: a reverse pass fed fp32-rounded positions was measured to
// lose the 1e-3 gradient bar on ~5 % of the teacher-forced segments.)
enum { TAPE_DX = STATE_ROWS, TAPE_V1 = TAPE_DX + 3, TAPE_S = TAPE_V1 + 3, TAPE_ACT = TAPE_S + 1, TAPE_LAM = TAPE_ACT + 1 };
__host__ __device__ inline int tape_rows(int N_C) { return TAPE_LAM + N_C; }

template <int VPL> __device__ __forceinline__ void store_rows3(float* __restrict__ rows, int base, int NS, const f3 a[VPL]) {
  float r[VPL];
#pragma unroll
  for (int k = 0; k < VPL; ++k) r[k] = a[k].x;
  store_row<VPL>(rows, base, NS, r);
#pragma unroll
  for (int k = 0; k < VPL; ++k) r[k] = a[k].y;
  store_row<VPL>(rows + NS, base, NS, r);
#pragma unroll
  for (int k = 0; k < VPL; ++k) r[k] = a[k].z;
  store_row<VPL>(rows + 2 * NS, base, NS, r);
}
template <int VPL> __device__ __forceinline__ void load_rows3(const float* __restrict__ rows, int base, int NS, f3 a[VPL]) {
  float rx[VPL], ry[VPL], rz[VPL];
  load_row<VPL>(rows, base, NS, rx); load_row<VPL>(rows + NS, base, NS, ry); load_row<VPL>(rows + 2 * NS, base, NS, rz);
#pragma unroll
  for (int k = 0; k < VPL; ++k) a[k] = mk3<float>(rx[k], ry[k], rz[k]);
}

// the per-lane slice of one env's state (x, v per vertex; d1 per edge; rest curvature per vertex)
template <int VPL> struct LaneState {
  f3 x[VPL], v[VPL], d1[VPL];
  float kb1[VPL], kb2[VPL];
  f3 xl[VPL];   // low part of the position (see ROW_XL)
};

template <int VPL> __device__ __forceinline__ void load_state(const float* __restrict__ blk, int base, int NS, LaneState<VPL>& s) {
  float r[STATE_ROWS][VPL];
#pragma unroll
  for (int q = 0; q < STATE_ROWS; ++q) load_row<VPL>(blk + q * NS, base, NS, r[q]);
#pragma unroll
  for (int k = 0; k < VPL; ++k) {
    s.x[k] = mk3<float>(r[0][k], r[1][k], r[2][k]);
    s.v[k] = mk3<float>(r[3][k], r[4][k], r[5][k]);
    s.d1[k] = mk3<float>(r[6][k], r[7][k], r[8][k]);
    s.kb1[k] = r[9][k]; s.kb2[k] = r[10][k];
    s.xl[k] = mk3<float>(r[11][k], r[12][k], r[13][k]);
  }
}
template <int VPL> __device__ __forceinline__ void store_state(float* __restrict__ blk, int base, int NS, const LaneState<VPL>& s) {
  float r[VPL];
#define DLO_ST(q, expr) { _Pragma("unroll") for (int k = 0; k < VPL; ++k) r[k] = (expr); store_row<VPL>(blk + (q) * NS, base, NS, r); }
  DLO_ST(0, s.x[k].x) DLO_ST(1, s.x[k].y) DLO_ST(2, s.x[k].z)
  DLO_ST(3, s.v[k].x) DLO_ST(4, s.v[k].y) DLO_ST(5, s.v[k].z)
  DLO_ST(6, s.d1[k].x) DLO_ST(7, s.d1[k].y) DLO_ST(8, s.d1[k].z)
  DLO_ST(9, s.kb1[k]) DLO_ST(10, s.kb2[k])
  DLO_ST(11, s.xl[k].x) DLO_ST(12, s.xl[k].y) DLO_ST(13, s.xl[k].z)
#undef DLO_ST
}

// per-env constants held in registers for the whole launch
template <int VPL> struct EnvConst {
  float m, inv_m, l0, stretch, alpha, gamma, sigy, rc, mu_r, mu_s;
  float w[VPL];       // inverse mass, 0 for pinned / grasped / padding
  int kin[VPL];
  float wr;           // inverse mass of the remote next vertex (slot 0 of lane nl)
};

template <int VPL> __device__ __forceinline__ void load_env(const KParams& P, int env, Topo<VPL>& tp, EnvConst<VPL>& c) {
  const float* M = P.mat + (size_t)env * MAT_N;
  c.m = M[MAT_M]; c.inv_m = 1.0f / c.m; c.l0 = M[MAT_L0]; c.stretch = M[MAT_STRETCH]; c.alpha = M[MAT_ALPHA];
  c.gamma = M[MAT_GAMMA]; c.sigy = M[MAT_SIGY]; c.rc = M[MAT_RC]; c.mu_r = M[MAT_MUR]; c.mu_s = M[MAT_MUS];
  bool cut[VPL];
#pragma unroll
  for (int k = 0; k < VPL; ++k) {
    const int raw = tp.vvalid[k] ? (int)P.kin[(size_t)env * P.NS + tp.base + k] : KIN_PINNED;
    c.kin[k] = raw & (KIN_CUT - 1);
    cut[k] = (raw & KIN_CUT) != 0;
    c.w[k] = (tp.vvalid[k] && c.kin[k] == KIN_FREE) ? c.inv_m : 0.0f;
  }
  // several DLOs in one env: an absent edge is no edge (no stretch / Eq.10 constraint, no frame, no contact segment), and a
  // vertex next to it is a rope end (no bending element).  The previous lane is always full: its last slot is VPL - 1.
  {
    const bool prev_cut = __shfl_sync(DLO_FULL, (int)cut[VPL - 1], tp.pl) != 0;
#pragma unroll
    for (int k = 0; k < VPL; ++k) {
      if (cut[k]) tp.evalid[k] = false;
      if (cut[k] || (k == 0 ? prev_cut : cut[k > 0 ? k - 1 : 0])) tp.interior[k] = false;
    }
  }
  c.wr = shfl(c.w[0], tp.nl);
  // opaque from here on: otherwise the compiler, short of registers, re-derives w[k] from kin[k], the lane index and N at
  // every use inside the projection loop (4 instructions instead of a register or one reload)
#pragma unroll
  for (int k = 0; k < VPL; ++k) asm volatile("" : "+f"(c.w[k]));
  asm volatile("" : "+f"(c.wr));
}

// cached edge geometry of the CURRENT positions: unit tangent and inverse length per owned edge, plus the copy
// of the previous lane's last edge (tangent, inverse length, director) needed by the bending element at slot 0
template <int VPL> struct EdgeCache {
  f3 t[VPL];
  float iL[VPL];
  f3 pt, pd1;
  float piL;
};

template <int VPL> __device__ __forceinline__ f3 pick_last(const f3 a[VPL], int ks) {
  f3 r = a[0];
#pragma unroll
  for (int k = 1; k < VPL; ++k) if (k == ks) r = a[k];
  return r;
}
template <int VPL> __device__ __forceinline__ float pick_last(const float a[VPL], int ks) {
  float r = a[0];
#pragma unroll
  for (int k = 1; k < VPL; ++k) if (k == ks) r = a[k];
  return r;
}

// next-vertex value of slot k: local slot k+1, or the remote value at the lane's last slot
template <int VPL> __device__ __forceinline__ f3 next_of(const f3 a[VPL], const f3& remote, int k, int ks) {
  if (k == VPL - 1) return remote;
  return (k == ks) ? remote : a[k + 1 < VPL ? k + 1 : k];
}

// exact edge vector of slot k from the two-float positions: the difference of the high parts is exact (neighbours agree in
// their leading bits), the low parts add what the stored fp32 positions had rounded away
template <int VPL> __device__ __forceinline__ f3 edge_vec(const LaneState<VPL>& s, const f3& xr, const f3& xlr, int k, int ks) {
  return (next_of<VPL>(s.x, xr, k, ks) - s.x[k]) + (next_of<VPL>(s.xl, xlr, k, ks) - s.xl[k]);
}
template <int VPL> __device__ __forceinline__ void edge_refresh(const Topo<VPL>& tp, const LaneState<VPL>& s, EdgeCache<VPL>& ec) {
  const f3 xr = shfl3(s.x[0], tp.nl), xlr = shfl3(s.xl[0], tp.nl);
#pragma unroll
  for (int k = 0; k < VPL; ++k) {
    f3 e = edge_vec<VPL>(s, xr, xlr, k, tp.ks);
    float L2 = dot(e, e);
    float iL = tp.evalid[k] ? rsqrt_(L2) : 0.0f;
    ec.iL[k] = iL;
    ec.t[k] = iL * e;
  }
}
template <int VPL> __device__ __forceinline__ void edge_prev_refresh(const Topo<VPL>& tp, const LaneState<VPL>& s, EdgeCache<VPL>& ec) {
  ec.pt = shfl3(pick_last<VPL>(ec.t, tp.ks), tp.pl);
  ec.pd1 = shfl3(pick_last<VPL>(s.d1, tp.ks), tp.pl);
  ec.piL = shfl(pick_last<VPL>(ec.iL, tp.ks), tp.pl);
}

}  // namespace dlo
