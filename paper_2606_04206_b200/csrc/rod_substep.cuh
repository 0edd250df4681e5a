// rod_substep.cuh — ONE substep of the rod step for one env held by one warp (steps A1-A9).
// `REC` = true additionally records what the reverse pass needs (rod_adjoint.cuh): the Eq.10 multipliers, the
// per-iteration self-contact corrections, the pre-coupling velocity and the set of active rigid responses.
#pragma once
#include "rod_warp.cuh"

namespace dlo {

struct WarpSmem {
  float *pose, *prim, *q, *ys, *acc, *vs, *mid, *dp, *lam, *dpbar, *ybar, *vbar, *posebar, *blk, *xref;
  unsigned short* cand;
  unsigned short* hot;   // near pairs of the last full filter (in pair order), kept across substeps
  float* base;        // the warp's shared-memory block (non-inlined helpers rebuild the view from this one pointer)
  unsigned phase_mask;   // KParams::phase_mask
  int sync_threads;   // > 0: warps of the CTA walk the phases in lockstep (named barrier over this many threads)
  int NP;   // row stride of the per-vertex arrays: 33*VPL (32*VPL vertices + pad words, see vpos)
  __device__ __forceinline__ void init(const KParams& P, float* base, int np) {
    pose = base + P.sm_pose; prim = base + P.sm_prim; q = base + P.sm_q; ys = base + P.sm_ys; acc = base + P.sm_acc;
    vs = base + P.sm_vs; mid = base + P.sm_mid; dp = base + P.sm_dp; cand = reinterpret_cast<unsigned short*>(base + P.sm_cand);
    hot = reinterpret_cast<unsigned short*>(base + P.sm_hot);
    lam = base + P.sm_lam; dpbar = base + P.sm_dpbar; ybar = base + P.sm_ybar; vbar = base + P.sm_vbar; posebar = base + P.sm_posebar; blk = base + P.sm_blk; xref = base + P.sm_xref;
    NP = np;
    this->base = base;
    sync_threads = 0;
    phase_mask = P.phase_mask;
  }
};

// Phase barrier of the big kernels.  All warps of a CTA run the same long instruction stream on different envs; kept
// in step, one instruction-cache fill serves all of them.  Must only be called from CTA-uniform control flow.
__device__ __forceinline__ void phase_sync(const WarpSmem& sm, unsigned site_bit = 1u) {
  if (sm.sync_threads > 0 && (sm.phase_mask & site_bit)) asm volatile("bar.sync 1, %0;" ::"r"(sm.sync_threads) : "memory");
}

// Phase barrier that also ORs a per-thread flag over the CTA (bar.red): the warps decide together, at no extra cost
__device__ __forceinline__ bool phase_vote(const WarpSmem& sm, bool v) {
  if (sm.sync_threads <= 0) return v;
  int r;
  asm volatile(
      "{\n\t.reg .pred pin, pout;\n\tsetp.ne.s32 pin, %2, 0;\n\tbar.red.or.pred pout, 1, %1, pin;\n\tselp.s32 %0, 1, 0, pout;\n\t}"
      : "=r"(r) : "r"(sm.sync_threads), "r"((int)v) : "memory");
  return r != 0;
}

// what is known about self-contact from earlier substeps: positions at which the candidate list was last built and
// the exact minimum pair distance there (dref < 0: nothing known, build at first need; huge: never build)
template <int VPL> struct ContactCache {
  f3 xref[VPL];
  float dref;  // minimum distance, at xref, over the pairs that are NOT in the near list
  int nlist;   // size of the pair list in shared memory (build_pair_list); < 0: none yet or truncated, rebuild at next use
  int nhot;    // size of the near list (sm.hot); < 0: none (then dref covers every pair)
  __device__ __forceinline__ void reset(float d) {
#pragma unroll
    for (int k = 0; k < VPL; ++k) xref[k] = zero3<float>();
    dref = d;
    nlist = -1;
    nhot = -1;
  }
};

// intermediates of one substep that outlive it when REC (all per lane)
template <int VPL> struct SubRec {
  f3 v1[VPL], xp[VPL] /* reverse pass only */, dx[VPL], v3[VPL], v4[VPL], t_old[VPL];
  float S[VPL];
  unsigned active[VPL];   // bit k<K: primitive k responded; bit K+2g+f: finger f of gripper g responded
  int ncand, any_pen;
  int side_slot;          // MODE 2: slot of this substep's side record (-1: none)
  int work;               // rough count of the self-contact work this substep did (scheduling hint only)
  unsigned jac_mask;      // bit it: the Jacobi pass of iteration it applied at least one correction
};

// (hi, lo) <- (hi + lo) + a, renormalised so that |lo| <= ulp(hi)/2: Knuth's two-sum of hi and a (exact), the old low part
// added to its error term, then a fast two-sum.  No FMA contraction can change it: there are no products here.
__device__ __forceinline__ void two_float_add(float& hi, float& lo, float a) {
  const float t = __fadd_rn(hi, a);
  const float bb = __fsub_rn(t, hi);
  const float err = __fadd_rn(__fsub_rn(hi, __fsub_rn(t, bb)), __fsub_rn(a, bb));
  const float l2 = __fadd_rn(lo, err);
  hi = __fadd_rn(t, l2);
  lo = __fsub_rn(l2, __fsub_rn(hi, t));
}
__device__ __forceinline__ void two_float_add(f3& hi, f3& lo, const f3& a) {
  two_float_add(hi.x, lo.x, a.x); two_float_add(hi.y, lo.y, a.y); two_float_add(hi.z, lo.z, a.z);
}

// A1 (L129, R-20): lane g < G evaluates gripper g at the substep's start and end and publishes it
// `chain`: the block still holds the previous substep of the same step, whose end pose is this substep's start pose
__device__ __forceinline__ void publish_poses(const KParams& P, int env, int lane, const float ap[6], const float ac[6], int s, float* pose_sm,
                                              bool chain = false) {
  if (lane < P.G) {
    const float tau0 = (float)s / (float)P.n_sub, tau1 = (float)(s + 1) / (float)P.n_sub;
    float* o = pose_sm + lane * POSE_STRIDE;
    // The gripper POSITION is interpolated in double and kept as a two-float sum (hi in P0 / P1, lo in P0L / P1L): grasped
    // vertices are put at p + R q every substep, and an fp32 p at 0.5 m would jitter them by 3e-8 m against their free
    // neighbours, i.e. 3e-8 / h of velocity noise through Eq.10.  R stays fp32: its rounding is scaled by |q| ~ 1 cm.
    auto put_p = [&](float tau, int at, int at_lo) {
      const double td = (double)tau;
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        const double pd = fma(td, (double)ac[k], (1.0 - td) * (double)ap[k]);
        const float hi = (float)pd;
        o[at + k] = hi; o[at_lo + k] = (float)(pd - (double)hi);
      }
    };
    if (chain) {
#pragma unroll
      for (int k = 0; k < 12; ++k) o[POSE_P0 + k] = o[POSE_P1 + k];   // p1, R1 -> p0, R0 (contiguous)
#pragma unroll
      for (int k = 0; k < 3; ++k) o[POSE_P0L + k] = o[POSE_P1L + k];
    } else {
      const Pose<float> g0 = make_pose<float>(ap, ac, tau0);
      put_p(tau0, POSE_P0, POSE_P0L);
#pragma unroll
      for (int k = 0; k < 9; ++k) o[POSE_R0 + k] = g0.R.m[k];
    }
    Pose<float> g1 = make_pose<float>(ap, ac, tau1);
    put_p(tau1, POSE_P1, POSE_P1L);
    g1.p = mk3<float>(o[POSE_P1], o[POSE_P1 + 1], o[POSE_P1 + 2]);
#pragma unroll
    for (int k = 0; k < 9; ++k) o[POSE_R1 + k] = g1.R.m[k];
    const float* fg = P.finger + ((size_t)env * P.G + lane) * 4;
    const float gap = fg[0], len = fg[1];
    f3 A0 = g1.p + mul(g1.R, mk3<float>(0.5f * gap, 0.f, 0.f)), B0 = g1.p + mul(g1.R, mk3<float>(0.5f * gap, 0.f, len));
    f3 A1 = g1.p + mul(g1.R, mk3<float>(-0.5f * gap, 0.f, 0.f)), B1 = g1.p + mul(g1.R, mk3<float>(-0.5f * gap, 0.f, len));
    o[POSE_FA0] = A0.x; o[POSE_FA0 + 1] = A0.y; o[POSE_FA0 + 2] = A0.z; o[POSE_FB0] = B0.x; o[POSE_FB0 + 1] = B0.y; o[POSE_FB0 + 2] = B0.z;
    o[POSE_FA1] = A1.x; o[POSE_FA1 + 1] = A1.y; o[POSE_FA1 + 2] = A1.z; o[POSE_FB1] = B1.x; o[POSE_FB1 + 1] = B1.y; o[POSE_FB1 + 2] = B1.z;
    o[POSE_RF] = fg[2];
    const f3 c0 = 0.5f * (A0 + B0), c1 = 0.5f * (A1 + B1);
    o[POSE_FC0] = c0.x; o[POSE_FC0 + 1] = c0.y; o[POSE_FC0 + 2] = c0.z; o[POSE_FC1] = c1.x; o[POSE_FC1 + 1] = c1.y; o[POSE_FC1 + 2] = c1.z;
    o[POSE_FRAD] = 0.5f * fabsf(len) + fg[2];
  }
  __syncwarp();
}
__device__ __forceinline__ Pose<float> read_pose(const float* o, int which) {
  Pose<float> g;
  const float* p = o + (which ? POSE_P1 : POSE_P0);
  const float* R = o + (which ? POSE_R1 : POSE_R0);
  g.p = mk3<float>(p[0], p[1], p[2]);
#pragma unroll
  for (int k = 0; k < 9; ++k) g.R.m[k] = R[k];
  return g;
}
// target of a grasped vertex at the end of the substep: p1 + R1 q  (L103 kinematic flag, R-19), as a two-float sum hi + lo
__device__ __forceinline__ f3 grasp_target(const KParams& P, const WarpSmem& sm, int code, f3& lo) {
  const int slot = code - KIN_GRASP0, g = (slot >= P.M) + (slot >= 2 * P.M) + (slot >= 3 * P.M);   // slot / M for G <= 4, without the division
  const float* o = sm.pose + g * POSE_STRIDE;
  const float* q = sm.q + 3 * slot;
  Pose<float> g1 = read_pose(o, 1);
  const float* Rm = g1.R.m;   // R q + p_lo, every sum of products an explicit fma (same bits in every kernel)
  const f3 s = mk3<float>(fma_(Rm[0], q[0], fma_(Rm[1], q[1], fma_(Rm[2], q[2], o[POSE_P1L]))),
                          fma_(Rm[3], q[0], fma_(Rm[4], q[1], fma_(Rm[5], q[2], o[POSE_P1L + 1]))),
                          fma_(Rm[6], q[0], fma_(Rm[7], q[1], fma_(Rm[8], q[2], o[POSE_P1L + 2]))));
  f3 hi = g1.p;
  lo = zero3<float>();
  two_float_add(hi, lo, s);
  return hi;
}
// velocity of the finger-body point at world y over the substep (L103): (y - [p0 + R0 R1^T (y - p1)]) / h, evaluated as
// ((p1 - p0) + (R1 - R0) local) / h with local = R1^T (y - p1): the same number without differencing two positions at 0.5 m
__device__ __forceinline__ f3 finger_body_velocity(const float* o, const f3& y, float inv_h) {
  const Pose<float> g0 = read_pose(o, 0), g1 = read_pose(o, 1);
  const f3 local = mulT(g1.R, y - g1.p);
  const f3 dp = (g1.p - g0.p) + (mk3<float>(o[POSE_P1L], o[POSE_P1L + 1], o[POSE_P1L + 2]) - mk3<float>(o[POSE_P0L], o[POSE_P0L + 1], o[POSE_P0L + 2]));
  M3<float> dR;
#pragma unroll
  for (int k = 0; k < 9; ++k) dR.m[k] = g1.R.m[k] - g0.R.m[k];
  return inv_h * (dp + mul(dR, local));
}

// A2 bending (Eq.4-7): per owned interior vertex the element gradients Ga, Gb; returns the gathered force
template <int VPL>
__device__ __forceinline__ void bending_forces(const Topo<VPL>& tp, const LaneState<VPL>& s, const EdgeCache<VPL>& ec, float sc, f3 f[VPL]) {
  f3 Ga[VPL], Gb[VPL];
#pragma unroll
  for (int k = 0; k < VPL; ++k) {
    Ga[k] = zero3<float>(); Gb[k] = zero3<float>();
    if (tp.interior[k]) {
      const f3 ta = (k == 0) ? ec.pt : ec.t[k > 0 ? k - 1 : 0];
      const f3 da = (k == 0) ? ec.pd1 : s.d1[k > 0 ? k - 1 : 0];
      const float ia = (k == 0) ? ec.piL : ec.iL[k > 0 ? k - 1 : 0];
      bend_element<float>(ta, ec.t[k], ia, ec.iL[k], da, s.d1[k], s.kb1[k], s.kb2[k], sc, Ga[k], Gb[k]);
    }
  }
  const f3 Gb_prev = shfl3(pick_last<VPL>(Gb, tp.ks), tp.pl);   // element i-1 of slot 0
  const f3 Ga_next = shfl3(Ga[0], tp.nl);                      // element i+1 of the last slot
#pragma unroll
  for (int k = 0; k < VPL; ++k) {
    const f3 gbp = (k == 0) ? Gb_prev : Gb[k > 0 ? k - 1 : 0];
    const f3 gan = next_of<VPL>(Ga, Ga_next, k, tp.ks);
    f[k] = f[k] - gbp - Ga[k] + Gb[k] + gan;
  }
}

// squared segment-segment distance of an edge pair (pa.. are smem positions of the four end points)
__device__ __forceinline__ float pair_dist2(const float* ys, int NP, int pa, int pan, int pb, int pbn) {
  f3 p1 = lds3(ys, NP, pa), q1 = lds3(ys, NP, pan), p2 = lds3(ys, NP, pb), q2 = lds3(ys, NP, pbn);
  float t, u;
  closest_points<float>(p1, q1, p2, q2, t, u);
  f3 dv = axpy(p1, t, q1 - p1) - axpy(p2, u, q2 - p2);
  return dot(dv, dv);
}

// A4 candidate list (Eq.13 "potentially colliding", R-15): all edge pairs a<b with cyclic index distance >=
// self_skip whose segments are closer than 2(r_a+r_b) at x^p.  The SET equals the oracle's; it is found in two
// stages.  build_pair_list (run only when some vertex has moved more than list_margin since its last run) collects a
// conservative superset, the pairs that can come within 2(r_a+r_b) while no vertex moves further than list_margin:
// (1) bounding spheres of the lanes' edge blocks (VPL edges each) are tested pairwise, (2) edge pairs of the
// surviving block pairs pass a midpoint-sphere test, both with the reach widened by 2 list_margin (segment distance
// is 1-Lipschitz in the end points).  filter_candidates (every substep that needs the list) takes the exact
// segment-segment test at x^p over that superset, 32 pairs at a time.  Every rejection is conservative, so no pair
// is lost.  Order: by (block a, block b, slot a, slot b) - a function of the pair indices only, so the list is the
// same whenever and wherever the superset was built (forward, replay and the recomputing reverse pass agree bit
// for bit); it is not the oracle's lexicographic order (only the fp32 summation order of the Jacobi pass depends
// on it).  mid = (midpoint, half length, w) at the positions the superset was built at.
template <int VPL>
__device__ __noinline__ int build_pair_list(const KParams& __restrict__ P, int lane, float* smbase, float slack, float bx, float by, float bz, float br) {
  WarpSmem sm;
  sm.init(P, smbase, 33 * VPL);
  const int E = P.E, NP = sm.NP, nb = (E + VPL - 1) / VPL;
  // P is read through a reference here (a generic load per access, repeated in every loop iteration because of the stores
  // to shared memory in between): the fields the loops use are taken once
  const int self_skip = P.self_skip, ring = P.ring, cand_cap = P.cand_cap;
  const float lim = 4.0f * P.r + slack;   // 2 (r_a + r_b) + slack
  constexpr int PP = VPL * VPL, NPER = PP <= 32 ? 32 / PP : 1, ITER = (PP + 31) / 32;
  unsigned short* surv = sm.cand + P.cand_cap;
  // (1) block pairs: lane B tests its own block against block A
  sm.blk[lane] = bx; sm.blk[32 + lane] = by; sm.blk[64 + lane] = bz; sm.blk[96 + lane] = br;
  __syncwarp();
  unsigned mymask = 0u;
  for (int A = 0; A < nb; ++A) {
    const float dx = sm.blk[A] - bx, dy = sm.blk[32 + A] - by, dz = sm.blk[64 + A] - bz, reach = sm.blk[96 + A] + br + lim;
    const bool hit = lane >= A && lane < nb && reach > 0.0f && dx * dx + dy * dy + dz * dz < reach * reach;   // (a block of absent edges has radius -1e30)
    const unsigned m = __ballot_sync(DLO_FULL, hit);
    if (lane == A) mymask = m;
  }
  // (2) edge pairs of surviving block pairs -> survivors of the midpoint-sphere test
  int nsurv = 0;
  for (int A = 0; A < nb; ++A) {
    unsigned mask = __shfl_sync(DLO_FULL, mymask, A);
    while (mask) {
#pragma unroll
      for (int j = 0; j < ITER; ++j) {
        const int sub = (PP <= 32) ? lane / PP : 0, idx = (PP <= 32) ? lane % PP : j * 32 + lane;
        unsigned mm = mask, Bsel = 0xffffffffu;   // the (sub+1)-th set bit of mask
#pragma unroll
        for (int q = 0; q < NPER; ++q) { if (q == sub && mm) Bsel = __ffs(mm) - 1; mm &= mm - 1u; }
        const int ka = idx / VPL, kb = idx % VPL, a = A * VPL + ka, b = (int)Bsel * VPL + kb, d = b - a;
        bool hit = false;
        if (Bsel != 0xffffffffu && idx < PP && sub < NPER && b < E && d >= self_skip && (!ring || E - d >= self_skip)) {
          const int pa = vpos<VPL>(a), pb = vpos<VPL>(b);
          const float dx = sm.mid[pb] - sm.mid[pa], dy = sm.mid[NP + pb] - sm.mid[NP + pa], dz = sm.mid[2 * NP + pb] - sm.mid[2 * NP + pa];
          const float reach = sm.mid[3 * NP + pa] + sm.mid[3 * NP + pb] + lim;
          hit = reach > 0.0f && dx * dx + dy * dy + dz * dz < reach * reach;
        }
        const unsigned m = __ballot_sync(DLO_FULL, hit);
        if (hit) {
          const int pos = nsurv + __popc(m & ((1u << lane) - 1u));
          if (pos < cand_cap) surv[pos] = (unsigned short)((a << 8) | b);
        }
        nsurv += __popc(m);
      }
#pragma unroll
      for (int q = 0; q < NPER; ++q) mask &= mask - 1u;
    }
  }
  __syncwarp();
  return nsurv;   // > cand_cap: truncated
}

// exact narrow phase at x^p (in sm.ys) over the pair list, ordered compaction into the candidate list.  The same pass
// splits the pairs into NEAR (closer than 3 r_sum / 2, kept in sm.hot in pair order) and FAR: between full filters
// only the near pairs are measured again (filter_near, every substep), the far ones are covered by the Lipschitz
// bound on dfar.  Too many near pairs for sm.hot: no near list (nhot = -1), dfar covers every pair.
struct CandOut { int ncand, nhot; float dmin, dfar; };   // dmin: exact minimum segment distance over ALL eligible pairs, capped at 2(r_a+r_b); dfar: over the far ones
template <int VPL>
__device__ __noinline__ CandOut filter_candidates(const KParams& __restrict__ P, int lane, float* smbase, int nsurv, bool overflow, bool wide) {
  WarpSmem sm;
  sm.init(P, smbase, 33 * VPL);
  const int N = P.N, NP = sm.NP;
  const float lim = 4.0f * P.r;   // 2 (r_a + r_b)
  const float near2 = P.near_dist * P.near_dist;
  const unsigned short* surv = sm.cand + P.cand_cap;
  int ncand = 0, nhot = 0;
  float d2min = lim * lim, d2far = lim * lim;
  for (int p0 = 0; p0 < nsurv; p0 += 32) {
    const int p = p0 + lane;
    bool hit = false, near = false;
    unsigned c = 0u;
    if (p < nsurv) {
      c = surv[p];
      const int a = c >> 8, b = c & 255, an = (a + 1 < N) ? a + 1 : 0, bn = (b + 1 < N) ? b + 1 : 0;
      const float d2 = pair_dist2(sm.ys, NP, vpos<VPL>(a), vpos<VPL>(an), vpos<VPL>(b), vpos<VPL>(bn));
      near = d2 < near2;
      // Candidates: by definition every pair closer than 2 (r_a + r_b) at x^p.  Only a pair that penetrates contributes, and
      // while the corrections stay below (dfar - r_sum) / 2 no pair beyond the near distance can: the candidate list is then
      // the near pairs alone (a handful instead of every pair of edges two apart), `wide` brings the others in when a
      // projection loop does move that far (substep: far_unsafe after a build)
      hit = wide ? d2 < lim * lim : near;
      d2min = fminf(d2min, d2);
      if (!near) d2far = fminf(d2far, d2);
    }
    const unsigned m = __ballot_sync(DLO_FULL, hit), mh = __ballot_sync(DLO_FULL, near);
    if (hit) sm.cand[ncand + __popc(m & ((1u << lane) - 1u))] = (unsigned short)c;
    if (near) {
      const int pos = nhot + __popc(mh & ((1u << lane) - 1u));
      if (pos < P.hot_cap) sm.hot[pos] = (unsigned short)c;
    }
    ncand += __popc(m);
    nhot += __popc(mh);
  }
  __syncwarp();
  CandOut out;
  out.ncand = ncand;
  out.dmin = overflow ? 0.0f : sqrt_(warp_min(d2min));
  const bool nolist = overflow || nhot > P.hot_cap;
  out.nhot = nolist ? -1 : nhot;
  out.dfar = nolist ? out.dmin : sqrt_(warp_min(d2far));
  return out;
}

// the near pairs measured again at x^p (in sm.ys): candidate list = those closer than 2(r_a+r_b), in pair order
template <int VPL>
__device__ __noinline__ CandOut filter_near(const KParams& __restrict__ P, int lane, float* smbase, int nhot) {
  WarpSmem sm;
  sm.init(P, smbase, 33 * VPL);
  const int N = P.N, NP = sm.NP;
  const float lim = 4.0f * P.r;
  int ncand = 0;
  float d2min = lim * lim;
  for (int p0 = 0; p0 < nhot; p0 += 32) {
    const int p = p0 + lane;
    bool hit = false;
    unsigned c = 0u;
    if (p < nhot) {
      c = sm.hot[p];
      const int a = c >> 8, b = c & 255, an = (a + 1 < N) ? a + 1 : 0, bn = (b + 1 < N) ? b + 1 : 0;
      const float d2 = pair_dist2(sm.ys, NP, vpos<VPL>(a), vpos<VPL>(an), vpos<VPL>(b), vpos<VPL>(bn));
      hit = d2 < lim * lim;
      d2min = fminf(d2min, d2);
    }
    const unsigned m = __ballot_sync(DLO_FULL, hit);
    if (hit) sm.cand[ncand + __popc(m & ((1u << lane) - 1u))] = (unsigned short)c;
    ncand += __popc(m);
  }
  __syncwarp();
  CandOut out;
  out.ncand = ncand; out.nhot = nhot;
  out.dmin = sqrt_(warp_min(d2min));
  out.dfar = 0.0f;
  return out;
}

// serialised (deterministic, candidate-order) accumulation of one lane's four vertex contributions
__device__ __forceinline__ void ordered_scatter4(unsigned hits, int lane, float* acc, int NP, const int iv[4], const float coef[4], const f3& n) {
  while (hits) {
    const int src = __ffs(hits) - 1;
    hits &= hits - 1;
    if (lane == src) {
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        acc[iv[k]] += coef[k] * n.x; acc[NP + iv[k]] += coef[k] * n.y; acc[2 * NP + iv[k]] += coef[k] * n.z;
      }
    }
    __syncwarp();
  }
}

// A5(ii): one Jacobi pass of Eq.13 over the candidates at y (in sm.ys); corrections summed into sm.acc, D_p += d.
// Returns true if any correction was applied.
template <int VPL>
__device__ __noinline__ bool contact_pass(const KParams& __restrict__ P, int lane, float* smbase, int ncand) {
  WarpSmem sm;
  sm.init(P, smbase, 33 * VPL);
  const int NP = sm.NP, N = P.N;
  const float rsum = 2.0f * P.r;
  bool any = false;
  for (int p0 = 0; p0 < ncand; p0 += 32) {
    const int p = p0 + lane;
    bool hit = false;
    int iv[4] = {0, 0, 0, 0};
    float coef[4] = {0.f, 0.f, 0.f, 0.f};
    f3 n = zero3<float>();
    if (p < ncand) {
      const unsigned c = sm.cand[p];
      iv[0] = c >> 8; iv[2] = c & 255; iv[1] = (iv[0] + 1 < N) ? iv[0] + 1 : 0; iv[3] = (iv[2] + 1 < N) ? iv[2] + 1 : 0;
#pragma unroll
      for (int k = 0; k < 4; ++k) iv[k] = vpos<VPL>(iv[k]);
      f3 xs[4];
      float ws[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) { xs[k] = lds3(sm.ys, NP, iv[k]); ws[k] = sm.mid[4 * NP + iv[k]]; }
      // conservative reject: the segments cannot be closer than |midpoint distance| - half lengths
      f3 ea = xs[1] - xs[0], eb = xs[3] - xs[2];
      f3 dm = (xs[0] + 0.5f * ea) - (xs[2] + 0.5f * eb);
      const float reach = 0.5f * (sqrt_(dot(ea, ea)) + sqrt_(dot(eb, eb))) + rsum;
      if (dot(dm, dm) < reach * reach) {
        float d, t, u, W;
        if (contact_eval<float>(xs, ws, rsum, d, t, u, n, W)) {
          hit = true;
          const float s = d / W;
          coef[0] = s * ws[0] * (1.0f - t); coef[1] = s * ws[1] * t; coef[2] = -s * ws[2] * (1.0f - u); coef[3] = -s * ws[3] * u;
          sm.dp[p] += d;
        }
      }
    }
    const unsigned hits = __ballot_sync(DLO_FULL, hit);
    any |= hits != 0u;
    ordered_scatter4(hits, lane, sm.acc, NP, iv, coef, n);
  }
  return any;
}

// A6 self-contact friction (L410, R-16) for candidates with D_p > 0: velocities in sm.vs, positions in sm.ys
template <int VPL>
__device__ __noinline__ void friction_pass(const KParams& __restrict__ P, int lane, float* smbase, int ncand, float mu_s) {
  WarpSmem sm;
  sm.init(P, smbase, 33 * VPL);
  const int NP = sm.NP, N = P.N;
  for (int p0 = 0; p0 < ncand; p0 += 32) {
    const int p = p0 + lane;
    bool hit = false;
    int iv[4] = {0, 0, 0, 0};
    float coef[4] = {0.f, 0.f, 0.f, 0.f};
    f3 D = zero3<float>();
    if (p < ncand && sm.dp[p] > 0.0f) {
      const unsigned c = sm.cand[p];
      iv[0] = c >> 8; iv[2] = c & 255; iv[1] = (iv[0] + 1 < N) ? iv[0] + 1 : 0; iv[3] = (iv[2] + 1 < N) ? iv[2] + 1 : 0;
#pragma unroll
      for (int k = 0; k < 4; ++k) iv[k] = vpos<VPL>(iv[k]);
      f3 xs[4], vv[4];
      float ws[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) { xs[k] = lds3(sm.ys, NP, iv[k]); vv[k] = lds3(sm.vs, NP, iv[k]); ws[k] = sm.mid[4 * NP + iv[k]]; }
      float t, u;
      closest_points<float>(xs[0], xs[1], xs[2], xs[3], t, u);
      f3 dv = axpy(xs[0], t, xs[1] - xs[0]) - axpy(xs[2], u, xs[3] - xs[2]);
      const float del = sqrt_(dot(dv, dv));
      const float a0 = 1.0f - t, b0 = 1.0f - u;
      const float W = ws[0] * a0 * a0 + ws[1] * t * t + ws[2] * b0 * b0 + ws[3] * u * u;
      if (del > 1e-12f && W > 0.0f) {
        f3 n = (1.0f / del) * dv;
        f3 vrel = (a0 * vv[0] + t * vv[1]) - (b0 * vv[2] + u * vv[3]);
        f3 vt = vrel - dot(vrel, n) * n;
        const float vtn = sqrt_(dot(vt, vt));
        if (vtn > 1e-12f) {
          const float cap = mu_s * sm.dp[p] * P.inv_h;
          const float mag = cap < vtn ? cap : vtn;
          D = (-(mag / vtn)) * vt;
          const float iW = 1.0f / W;
          coef[0] = ws[0] * a0 * iW; coef[1] = ws[1] * t * iW; coef[2] = -ws[2] * b0 * iW; coef[3] = -ws[3] * u * iW;
          hit = true;
        }
      }
    }
    const unsigned hits = __ballot_sync(DLO_FULL, hit);
    ordered_scatter4(hits, lane, sm.acc, NP, iv, coef, D);
  }
}

// A7 (L103): soft coupling of one free vertex at y against the K fixed primitives, then the finger capsules.
// Not inlined on purpose: it is called once per vertex slot and is the largest single piece of straight-line code
// (four SDF types + fingers); one copy keeps the kernel inside the instruction cache.
struct CoupleOut { f3 v; unsigned active; };
// the scalars of KParams that A7 needs, passed by value: inside a non-inlined function a field of the kernel's parameter
// block is a generic load through a pointer, in the kernel it is a constant-bank operand
struct CoupleConst {
  int K, G;
  float r, inv_eps, log_thresh_lo, f_thresh, e_rest, inv_h;
  unsigned types;   // prim_type[k] in bits 2k, 2k+1
};
__device__ __forceinline__ CoupleConst couple_const(const KParams& P) {
  CoupleConst q;
  q.K = P.K; q.G = P.G; q.r = P.r; q.inv_eps = P.inv_eps; q.log_thresh_lo = P.log_thresh_lo; q.f_thresh = P.f_thresh; q.e_rest = P.e_rest; q.inv_h = P.inv_h;
  q.types = P.prim_pack;
  return q;
}
__device__ __noinline__ CoupleOut rigid_coupling(const CoupleConst P, const float* __restrict__ prim_sm, const float* __restrict__ pose_sm,
                                                 f3 y, f3 v, float mu_r) {
  unsigned active = 0u;
  // a body whose bounding sphere is farther than reach = r + eps_s |ln f_thresh| cannot pass the f > f_thresh test
  const float reach = P.r - P.log_thresh_lo * (1.0f / P.inv_eps);
  for (int k = 0; k < P.K; ++k) {
    const float* pk = prim_sm + k * PRIM_SM_STRIDE;
    if (pk[PRIM_BR] >= 0.0f) {
      const f3 dc = y - mk3<float>(pk[PRIM_BC], pk[PRIM_BC + 1], pk[PRIM_BC + 2]);
      const float lim = pk[PRIM_BR] + reach;
      if (dot(dc, dc) >= lim * lim) continue;
    }
    float phi;
    f3 n;
    if (!sdf_eval_pre<float>((int)((P.types >> (2 * k)) & 3u), pk, y, phi, n)) continue;
    if ((P.r - phi) * P.inv_eps < P.log_thresh_lo) continue;
    if (rigid_response<float>(v, zero3<float>(), n, P.r - phi, P.inv_eps, P.f_thresh, P.e_rest, mu_r)) active |= 1u << k;
  }
  for (int g = 0; g < P.G; ++g) {
    const float* o = pose_sm + g * POSE_STRIDE;
    for (int fk = 0; fk < 2; ++fk) {
      const float* fc = o + (fk ? POSE_FC1 : POSE_FC0);
      const f3 dc = y - mk3<float>(fc[0], fc[1], fc[2]);
      const float lim = o[POSE_FRAD] + reach;
      if (dot(dc, dc) >= lim * lim) continue;
      const float* A = o + (fk ? POSE_FA1 : POSE_FA0);
      const float* Bp = o + (fk ? POSE_FB1 : POSE_FB0);
      float Pc[7] = {A[0], A[1], A[2], Bp[0], Bp[1], Bp[2], o[POSE_RF]};
      float phi;
      f3 n;
      if (!sdf_eval<float>(1, Pc, y, phi, n)) continue;
      if ((P.r - phi) * P.inv_eps < P.log_thresh_lo) continue;   // f < threshold for sure: v untouched, skip the body velocity
      f3 vb = finger_body_velocity(o, y, P.inv_h);
      if (rigid_response<float>(v, vb, n, P.r - phi, P.inv_eps, P.f_thresh, P.e_rest, mu_r)) active |= 1u << (P.K + 2 * g + fk);
    }
  }
  CoupleOut out;
  out.v = v; out.active = active;
  return out;
}

// Eq.10 with compliance on one edge, loop invariants precomputed: idn = 1 / (w_j + w_j+1 + atil), or 0 for a slot
// that is not projected (then lam = 0 and t is finite: the caller's updates change nothing).
__device__ __forceinline__ void project_edge_pre(const f3& e, float l0, float atil, float S, float idn, float& lam, f3& t) {
  const float L2 = fmaxf(dot(e, e), 1.0e-30f);   // a padding slot has e = 0: keep t finite there, lam * t must be 0
  const float iL = rsqrt_(L2);
  t = iL * e;
  lam = ((L2 * iL - l0) - atil * S) * idn;
}

// ---------------------------------------------------------------------------------------------------------
// One substep.  On entry `ec` holds the edge geometry of s.x (tangents, inverse lengths, previous lane's last
// edge); on exit it holds that of the new positions.  ap/ac: this step's a_{t-1}, a_t of gripper `lane` (lane<G).
// the barriers of substep() for a warp that skips the recompute (it must still take part in them, votes included)
__device__ __forceinline__ void substep_idle_syncs(const KParams& P, const WarpSmem& sm) {
  phase_sync(sm, 1u);
  if ((P.vote_mode & 1) && phase_vote(sm, false) && (P.vote_mode & 2)) phase_vote(sm, false);
  phase_sync(sm, 2u);
  phase_sync(sm, 4u);
}
// MODE 0: plain forward.  MODE 1 (REC): recompute inside the adjoint kernel (contact corrections -> acc_tape).
// MODE 2 (TAPE): replay of a segment.  In both, the Eq.10 multipliers go to the tape rows `lam_rows` [N_C][NS].
template <int VPL, int MODE>
__device__ __forceinline__ void substep(const KParams& P, const Topo<VPL>& tp, const EnvConst<VPL>& c, const WarpSmem& sm, int env,
                                        const float ap[6], const float ac[6], int sub, LaneState<VPL>& s, EdgeCache<VPL>& ec,
                                        SubRec<VPL>& R, float* acc_tape, ContactCache<VPL>& cc, float* lam_rows = nullptr) {
  constexpr bool REC = MODE == 1;
  const float h = P.h, inv_h = P.inv_h;
  // -- A1 bodies
  if (P.G > 0) publish_poses(P, env, tp.lane, ap, ac, sub, sm.pose, MODE != 1 && sub > 0);

  phase_sync(sm, 1u);
  // -- A2 forces: gravity, stretch (mode ENERGY, Eq.2-3), bending (Eq.4-7)
  f3 f[VPL];
#pragma unroll
  for (int k = 0; k < VPL; ++k) f[k] = mk3<float>(c.m * P.g[0], c.m * P.g[1], c.m * P.g[2]);
  if (P.stretch_mode == 0) {
    f3 F[VPL];
#pragma unroll
    for (int k = 0; k < VPL; ++k) {
      const float L = tp.evalid[k] ? 1.0f / ec.iL[k] : 0.0f;
      F[k] = tp.evalid[k] ? (c.stretch * (L / c.l0 - 1.0f)) * ec.t[k] : zero3<float>();
    }
    const f3 Fp = shfl3(pick_last<VPL>(F, tp.ks), tp.pl);
#pragma unroll
    for (int k = 0; k < VPL; ++k) f[k] = f[k] + F[k] - ((k == 0) ? Fp : F[k > 0 ? k - 1 : 0]);
  }
  bending_forces<VPL>(tp, s, ec, c.alpha / c.l0, f);

  // -- A3 velocity (symplectic Euler L97, implicit viscous damping R-7), A4 predict
  const float idamp = 1.0f / (1.0f + c.gamma * h), hm = h * c.inv_m;
#pragma unroll
  for (int k = 0; k < VPL; ++k) {
    f3 v1 = zero3<float>();
    if (c.kin[k] == KIN_FREE) v1 = idamp * axpy(s.v[k], hm, f[k]);
    else if (c.kin[k] >= KIN_GRASP0) { f3 tl; const f3 th = grasp_target(P, sm, c.kin[k], tl); v1 = inv_h * ((th - s.x[k]) + (tl - s.xl[k])); }
    R.v1[k] = v1;
    R.dx[k] = zero3<float>();
    R.S[k] = 0.0f;
  }
  // predicted edge vectors, constant during the projection loop: the exact edge of the two-float positions plus h times the
  // velocity difference - NOT the difference of rounded predicted positions, which would bring back 3e-8 m of noise per vertex
  f3 epred[VPL];
  {
    const f3 xr = shfl3(s.x[0], tp.nl), xlr = shfl3(s.xl[0], tp.nl), v1r = shfl3(R.v1[0], tp.nl);
#pragma unroll
    for (int k = 0; k < VPL; ++k) epred[k] = axpy(edge_vec<VPL>(s, xr, xlr, k, tp.ks), h, next_of<VPL>(R.v1, v1r, k, tp.ks) - R.v1[k]);
  }
  // x^p = x + h v^1 (contact geometry; fp32 positions are ample there): recomputed where it is read, one FFMA per component,
  // instead of held in 3 VPL registers across the projection loop
  auto XP = [&](int k) { return axpy(s.x[k], h, R.v1[k]); };

  // Self-contact is evaluated lazily (exactly): segment distance is 1-Lipschitz in the end points, so with d_ref the
  // minimum distance of a set of pairs at the positions x_ref where they were last measured, none of them can
  // penetrate while d_ref - 2 (max_i |x^p_i - x_ref,i| + max_i |dx_i|) >= r_a + r_b.  A full filter (pair list at
  // x^p, every pair measured) splits the pairs into near ones (closer than 3/2 r_sum, a handful: real contacts
  // and sharp folds) and far ones.  The far ones are covered by that bound with d_ref = their minimum distance, which
  // leaves r_sum / 2 of slack: a full filter every few tens of substeps.  The near ones are measured again at every
  // x^p (filter_near) and swept when they can penetrate within the iteration's max |dx|.  A pass that cannot apply a
  // correction changes nothing, so the state is identical to building the whole list and sweeping it every time.
  R.ncand = 0; R.any_pen = 0; R.jac_mask = 0u; R.work = 0; R.side_slot = -1;
  bool side_tried = false;
  bool built = false, wide_built = false;
  float D1 = 0.0f;
  float dnear = 1.0e30f;   // exact minimum distance at x^p over the pairs of the candidate list in use
  if (P.self_contact) {
    float m2 = 0.0f;
#pragma unroll
    for (int k = 0; k < VPL; ++k)
      if (tp.vvalid[k]) { const f3 d = XP(k) - cc.xref[k]; m2 = fmaxf(m2, dot(d, d)); }
    D1 = sqrt_(warp_max(m2));
  }
  auto build_list = [&](bool vote, bool wide) {
    // is the pair list still a superset?  (no vertex further than list_margin from where it was built)
    // (a list that was truncated is rebuilt at every use: that is this env's own business, the vote is about movement only)
    const bool trunc = cc.nlist < 0;
    bool fresh = false, overflow = false;
    int nuse = cc.nlist;
    if (!trunc) {
      float m2 = 0.0f;
#pragma unroll
      for (int k = 0; k < VPL; ++k)
        if (tp.vvalid[k]) { const f3 d = XP(k) - lds3(sm.xref, sm.NP, vpos<VPL>(tp.base + k)); m2 = fmaxf(m2, dot(d, d)); }
      const float lm = 0.999f * P.list_margin;
      const float wm = warp_max(m2);
      fresh = !(wm <= lm * lm);
    }
    if (vote && (P.vote_mode & 2)) fresh = phase_vote(sm, fresh);   // a warp of the CTA rebuilds: all do (they would wait for it anyway)
    fresh = fresh || trunc;
#pragma unroll
    for (int k = 0; k < VPL; ++k) {
      const int i = vpos<VPL>(tp.base + k);
      sts3(sm.ys, sm.NP, i, XP(k));
      sm.mid[4 * sm.NP + i] = c.w[k];
    }
    if (fresh) {
#pragma unroll
      for (int k = 0; k < VPL; ++k) {
        const int i = vpos<VPL>(tp.base + k);
        sts3(sm.xref, sm.NP, i, XP(k));
        sts3(sm.mid, sm.NP, i, axpy(XP(k), 0.5f, epred[k]));
        sm.mid[3 * sm.NP + i] = tp.evalid[k] ? 0.5f * sqrt_(dot(epred[k], epred[k])) : -1.0e30f;   // an absent edge (cut) is in reach of nothing
      }
      // bounding sphere of this lane's edge block (centre = mean of its edge midpoints)
      f3 bc = zero3<float>();
      float bn = 0.0f, brad = -1.0e30f;
#pragma unroll
      for (int k = 0; k < VPL; ++k)
        if (tp.evalid[k]) { bc += axpy(XP(k), 0.5f, epred[k]); bn += 1.0f; }
      if (bn > 0.0f) {
        bc = (1.0f / bn) * bc;
#pragma unroll
        for (int k = 0; k < VPL; ++k)
          if (tp.evalid[k]) {
            const f3 dm = axpy(XP(k), 0.5f, epred[k]) - bc;
            brad = fmaxf(brad, sqrt_(dot(dm, dm)) + 0.5f * sqrt_(dot(epred[k], epred[k])));
          }
      }
      __syncwarp();
      cc.nlist = build_pair_list<VPL>(P, tp.lane, sm.base, 2.0f * P.list_margin, bc.x, bc.y, bc.z, brad);
      if (cc.nlist > P.cand_cap) {
        // the superset does not fit (a tightly folded rope): list of this substep's positions only, rebuilt at the next use
        nuse = build_pair_list<VPL>(P, tp.lane, sm.base, 0.0f, bc.x, bc.y, bc.z, brad);
        cc.nlist = -1;
        if (nuse > P.cand_cap) {
          overflow = true;
          nuse = P.cand_cap;
          if (tp.lane == 0) atomicOr(P.flags + env, FLAG_CAND_OVERFLOW);
        }
      } else {
        nuse = cc.nlist;
      }
    }
    __syncwarp();
    // a rebuild in the middle of the projection loop, after sweeps over the near pairs have applied corrections: their
    // depth sums D_p move to the pairs' positions in the new list (sm.vs is free until the friction pass)
    const int nold = R.any_pen ? R.ncand : 0;
    unsigned* oldc = reinterpret_cast<unsigned*>(sm.vs);
    float* oldd = sm.vs + P.hot_cap;
    for (int p = tp.lane; p < nold; p += 32) { oldc[p] = sm.cand[p]; oldd[p] = sm.dp[p]; }
    __syncwarp();
    const CandOut co = filter_candidates<VPL>(P, tp.lane, sm.base, nuse, overflow, wide);
    R.work += fresh ? 24 : 8;
    R.ncand = co.ncand;
    cc.dref = co.dfar;
    cc.nhot = co.nhot;
    dnear = co.dmin;
#pragma unroll
    for (int k = 0; k < VPL; ++k) cc.xref[k] = XP(k);
    for (int p = tp.lane; p < R.ncand; p += 32) {
      float d = 0.0f;
      const unsigned code = sm.cand[p];
      for (int q = 0; q < nold; ++q) if (oldc[q] == code) d = oldd[q];
      sm.dp[p] = d;
    }
    __syncwarp();
  };

  // The warps of a CTA walk in lockstep, so a warp that refreshes its contact data stalls the others: they refresh
  // together, whenever one of them has to (refreshing early changes no result), which aligns their next refreshes too.
  {
    const float need = 2.0f * P.r + 1.0e-6f;
    const bool want = P.self_contact && !(cc.dref - 2.0f * D1 >= need);
    const bool go = (P.vote_mode & 1) ? phase_vote(sm, want) : want;
    if (go && P.self_contact) {
      build_list((P.vote_mode & 1) != 0, false);
      built = true;
      D1 = 0.0f;
    } else if (P.self_contact && cc.nhot > 0) {
      // the far pairs are safe where they are: measure the near ones at x^p, they are this substep's candidates
#pragma unroll
      for (int k = 0; k < VPL; ++k) sts3(sm.ys, sm.NP, vpos<VPL>(tp.base + k), XP(k));
      __syncwarp();
      const CandOut co = filter_near<VPL>(P, tp.lane, sm.base, cc.nhot);
      R.work += 1;
      R.ncand = co.ncand;
      dnear = co.dmin;
      for (int p = tp.lane; p < R.ncand; p += 32) sm.dp[p] = 0.0f;
      __syncwarp();
    }
  }
  // -- A5 projection loop
  const float atil = c.stretch * inv_h * inv_h;
  // loop invariants of Eq.10 per owned edge: inverse mass of its far vertex and 1 / (w_j + w_j+1 + atil), 0 for a
  // slot that is not projected (padding, pinned at both ends).  The loop body is then branch-free; with division as
  // MUFU.RCP x numerator (-prec-div=false) the multiplier has the same bits as dividing inside the loop.
  float idn[VPL], wfar[VPL];
#pragma unroll
  for (int k = 0; k < VPL; ++k) {
    const bool red = (k & 1) == 0;
    const bool rem = !red && ((k == VPL - 1) || (k == tp.ks));
    const bool on = red ? ((k + 1 < tp.nv) && tp.evalid[k]) : (tp.evalid[k] && (k <= tp.ks));
    wfar[k] = rem ? c.wr : c.w[k + 1 < VPL ? k + 1 : k];
    const float wsum = c.w[k] + wfar[k];
    idn[k] = (P.stretch_mode == 1 && on && wsum > 0.0f) ? 1.0f / (wsum + atil) : 0.0f;
  }
  for (int it = 0; it < P.N_C; ++it) {
    float lamv[VPL];
#pragma unroll
    for (int k = 0; k < VPL; ++k) lamv[k] = 0.0f;
    if (P.stretch_mode == 1) {
      // red: even slots, both end points local
#pragma unroll
      for (int k = 0; k < VPL; k += 2) {
        float lam;
        f3 t;
        project_edge_pre(epred[k] + (R.dx[k + 1] - R.dx[k]), c.l0, atil, R.S[k], idn[k], lam, t);
        R.S[k] += lam;
        R.dx[k] = axpy(R.dx[k], lam * c.w[k], t);
        R.dx[k + 1] = axpy(R.dx[k + 1], -lam * wfar[k], t);
        lamv[k] = lam;
      }
      // black: odd slots; the lane's last slot crosses to slot 0 of the next lane
      {
        const f3 dxr = shfl3(R.dx[0], tp.nl);
        f3 back = zero3<float>();
#pragma unroll
        for (int k = 1; k < VPL; k += 2) {
          const bool last = (k == VPL - 1), rem = last || (k == tp.ks);
          const f3 dxn = last ? dxr : (rem ? dxr : R.dx[k + 1 < VPL ? k + 1 : k]);
          float lam;
          f3 t;
          project_edge_pre(epred[k] + (dxn - R.dx[k]), c.l0, atil, R.S[k], idn[k], lam, t);
          R.S[k] += lam;
          R.dx[k] = axpy(R.dx[k], lam * c.w[k], t);
          const float cn = lam * wfar[k];
          if (last) back = axpy(back, cn, t);
          else {   // at most one remote edge per lane is projected: `back` receives one non-zero term
            back = axpy(back, rem ? cn : 0.0f, t);
            R.dx[k + 1 < VPL ? k + 1 : k] = axpy(R.dx[k + 1 < VPL ? k + 1 : k], rem ? 0.0f : -cn, t);
          }
          lamv[k] = lam;
        }
        R.dx[0] -= shfl3(back, tp.pl);
      }
      // third colour: the closing edge of an odd ring (slot ks of the last lane, even slot)
      // (written like the red sweep, every even slot with a per-slot flag: a body guarded by `k == tp.ks` makes the
      // compiler index dx / S / epred by ks, which puts those arrays in local memory for the whole kernel)
      if (P.odd_ring) {
        const f3 dxr = shfl3(R.dx[0], tp.nl);
        f3 back = zero3<float>();
#pragma unroll
        for (int k = 0; k < VPL; k += 2) {
          const bool on = (k == tp.ks) && (tp.base + k == P.E - 1);
          const float wsum = c.w[k] + c.wr;
          float lam = 0.0f;
          f3 t = zero3<float>();
          if (on && wsum > 0.0f) project_edge<float>(epred[k] + (dxr - R.dx[k]), wsum, c.l0, atil, R.S[k], lam, t);
          R.S[k] += lam;
          R.dx[k] = axpy(R.dx[k], lam * c.w[k], t);
          back = axpy(back, lam * c.wr, t);
          lamv[k] += lam;   // the closing edge's slot is idle in the red sweep
        }
        R.dx[0] -= shfl3(back, tp.pl);
      }
    }
    if (MODE >= 1 && lam_rows) store_row<VPL>(lam_rows + (size_t)it * P.NS, tp.base, P.NS, lamv);
    bool sweep = false;
    if (P.self_contact) {
      float m2 = 0.0f;
#pragma unroll
      for (int k = 0; k < VPL; ++k) m2 = fmaxf(m2, dot(R.dx[k], R.dx[k]));
      const float Dm = sqrt_(warp_max(m2)), need = 2.0f * P.r + 1.0e-6f;
      bool far_unsafe = !(cc.dref - 2.0f * (D1 + Dm) >= need);
      if (far_unsafe && !built) {
        build_list(false, false);
        built = true;
        D1 = 0.0f;
        far_unsafe = !(cc.dref - 2.0f * Dm >= need);
      }
      if (far_unsafe && !wide_built) {   // corrections so large that pairs beyond the near distance could touch: every pair closer than 2 (r_a + r_b) at x^p becomes a candidate
        build_list(false, true);
        built = true; wide_built = true;
        D1 = 0.0f;
      }
      sweep = far_unsafe || !(dnear - 2.0f * Dm >= need);
    }
    if (sweep && R.ncand > 0) {
#pragma unroll
      for (int k = 0; k < VPL; ++k) sts3(sm.ys, sm.NP, vpos<VPL>(tp.base + k), XP(k) + R.dx[k]);
      __syncwarp();
      const bool any = contact_pass<VPL>(P, tp.lane, sm.base, R.ncand);
      R.work += any ? 3 : 1;
      __syncwarp();
      if (any) {
        if (MODE == 2 && P.side && !side_tried) {   // replay: the corrections go to a side record (if the pool has a slot left)
          side_tried = true;
          int sl = 0;
          if (tp.lane == 0) sl = atomicAdd(P.side_count, 1);
          sl = __shfl_sync(DLO_FULL, sl, 0);
          if (sl < P.side_cap) { R.side_slot = sl; acc_tape = P.side + (size_t)sl * P.side_floats + side_off_acc(P); }
        }
        R.any_pen = 1;
        R.jac_mask |= 1u << it;
#pragma unroll
        for (int k = 0; k < VPL; ++k) {
          const int i = vpos<VPL>(tp.base + k);   // own vertex, slot-major position
          const f3 a = lds3(sm.acc, sm.NP, i);
          R.dx[k] += a;
          if (MODE >= 1 && acc_tape) sts3(acc_tape + (size_t)it * 3 * sm.NP, sm.NP, i, a);
          sts3(sm.acc, sm.NP, i, zero3<float>());
        }
        __syncwarp();
      }
    }
  }

  // -- A6 reconcile v with the projected positions (R-11) + self-contact friction
  f3 vel[VPL];
#pragma unroll
  for (int k = 0; k < VPL; ++k) vel[k] = (c.kin[k] == KIN_FREE) ? axpy(R.v1[k], inv_h, R.dx[k]) : R.v1[k];
  if (P.self_contact && R.any_pen) {
#pragma unroll
    for (int k = 0; k < VPL; ++k) { sts3(sm.ys, sm.NP, vpos<VPL>(tp.base + k), XP(k) + R.dx[k]); sts3(sm.vs, sm.NP, vpos<VPL>(tp.base + k), vel[k]); }
    __syncwarp();
    friction_pass<VPL>(P, tp.lane, sm.base, R.ncand, c.mu_s);
    __syncwarp();
#pragma unroll
    for (int k = 0; k < VPL; ++k) {
      const int i = vpos<VPL>(tp.base + k);   // own vertex, slot-major position
      if (c.kin[k] == KIN_FREE) vel[k] += lds3(sm.acc, sm.NP, i);
      sts3(sm.acc, sm.NP, i, zero3<float>());
    }
    __syncwarp();
  }

  phase_sync(sm, 2u);
  // -- A7 rigid soft coupling at y = x^p + dx
#pragma unroll
  for (int k = 0; k < VPL; ++k) {
    R.v3[k] = vel[k];
    R.active[k] = 0u;
    if (c.kin[k] == KIN_FREE && (P.K > 0 || P.G > 0)) {
      const CoupleOut co = rigid_coupling(couple_const(P), sm.prim, sm.pose, XP(k) + R.dx[k], vel[k], c.mu_r);
      vel[k] = co.v; R.active[k] = co.active;
    }
    R.v4[k] = vel[k];
  }

  // tangents of the positions the substep started from, for the frame transport of A9: recomputed here (the expression of
  // edge_refresh, same bits as ec.t had) rather than held in 3 VPL registers across the projection loop
  {
    const f3 xr = shfl3(s.x[0], tp.nl), xlr = shfl3(s.xl[0], tp.nl);
#pragma unroll
    for (int k = 0; k < VPL; ++k) {
      const f3 e = edge_vec<VPL>(s, xr, xlr, k, tp.ks);
      const float iL = tp.evalid[k] ? rsqrt_(dot(e, e)) : 0.0f;
      R.t_old[k] = iL * e;
    }
  }
  // -- A8 commit: x + xl <- (x + xl) + h v in two-float arithmetic (the rounding error of the sum is kept, not dropped)
#pragma unroll
  for (int k = 0; k < VPL; ++k) {
    if (c.kin[k] == KIN_FREE) { two_float_add(s.x[k], s.xl[k], h * vel[k]); s.v[k] = vel[k]; }
    else if (c.kin[k] >= KIN_GRASP0) { s.x[k] = grasp_target(P, sm, c.kin[k], s.xl[k]); s.v[k] = vel[k]; }
    else if (tp.vvalid[k]) s.v[k] = zero3<float>();
  }

  phase_sync(sm, 4u);
  // -- A9 frames: time-parallel transport (R-4), then plasticity (Eq.11)
  edge_refresh<VPL>(tp, s, ec);
#pragma unroll
  for (int k = 0; k < VPL; ++k) {
    if (tp.evalid[k]) {
      f3 d = ptransport<float>(R.t_old[k], ec.t[k], s.d1[k]);
      d = axpy(d, -dot(d, ec.t[k]), ec.t[k]);
      s.d1[k] = rsqrt_(dot(d, d)) * d;
    }
  }
  edge_prev_refresh<VPL>(tp, s, ec);
  if (P.plasticity) {
    const float Y = c.sigy * c.l0;
#pragma unroll
    for (int k = 0; k < VPL; ++k) {
      if (tp.interior[k]) {
        const f3 ta = (k == 0) ? ec.pt : ec.t[k > 0 ? k - 1 : 0];
        const f3 da = (k == 0) ? ec.pd1 : s.d1[k > 0 ? k - 1 : 0];
        float k1, k2;
        material_curvature<float>(ta, ec.t[k], da, s.d1[k], k1, k2);
        plasticity_update<float>(k1, k2, s.kb1[k], s.kb2[k], Y, c.rc);
      }
    }
  }
  if (P.G > 0) __syncwarp();   // the pose block is rewritten by the next substep
}

}  // namespace dlo
