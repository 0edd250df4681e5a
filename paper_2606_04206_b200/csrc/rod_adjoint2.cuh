// rod_adjoint2.cuh — reverse of one substep (A9 ... A1) and the segment adjoint kernel (second half of rod_adjoint.cuh)
#pragma once

namespace dlo {

// undo + differentiate one Eq.10 edge update.  dxk/dxn: corrections of the edge's own / next vertex AFTER the
// update (restored to their values before it); gk/gn: their adjoints (updated in place); epb: adjoint of the
// predicted edge vector.
__device__ __forceinline__ void edge_reverse(const f3& epred, float lam, float wk, float wn, float atil, f3& dxk, f3& dxn, float& S,
                                             f3& gk, f3& gn, float& Sb, float& atilbar, f3& epb) {
  const f3 ep = epred + (dxn - dxk);                // = (L - lam (wk+wn)) t
  const float iLp = rsqrt_(dot(ep, ep));
  const f3 t = iLp * ep;
  const float L = 1.0f / iLp + lam * (wk + wn);
  const float Spost = S;
  S -= lam;
  dxk = axpy(dxk, -lam * wk, t);
  dxn = axpy(dxn, lam * wn, t);
  f3 eb;
  project_edge_adj<float>(t, 1.0f / L, lam, Spost, wk, wn, atil, gk, gn, Sb, atilbar, eb);
  gn += eb;
  gk -= eb;
  epb += eb;
}

// The same with the loop invariants precomputed (idn = 1 / (wk + wn + atil), 0 for a slot that is not projected) and no
// branch: an idle slot has lam = 0 on the tape and idn = 0, so every update below adds a zero.
__device__ __forceinline__ void edge_reverse_pre(const f3& epred, float lam, float wk, float wn, float idn, float atil, f3& dxk, f3& dxn, float& S,
                                                 f3& gk, f3& gn, float& Sb, double& atilbar, f3& epb) {
  const f3 ep = epred + (dxn - dxk);                // = (L - lam (wk+wn)) t
  const float ep2 = fmaxf(dot(ep, ep), 1.0e-30f);   // (padding slots have ep = 0: keep t finite)
  const float iLp = rsqrt_(ep2);
  const f3 t = iLp * ep;
  const float L = ep2 * iLp + lam * (wk + wn);
  const float Spost = S;
  S -= lam;
  dxk = axpy(dxk, -lam * wk, t);
  dxn = axpy(dxn, lam * wn, t);
  // project_edge_adj (rod_adj.cuh) with the division by (wk + wn + atil) replaced by the stored reciprocal
  const f3 g = wk * gk - wn * gn;
  const float numbar = (dot(g, t) + Sb) * idn;
  atilbar -= (double)numbar * (double)Spost;   // thousands of terms of either sign per substep: summed in double
  Sb -= atil * numbar;
  const f3 tbar = lam * g;
  const f3 eb = numbar * t + (1.0f / L) * (tbar - dot(tbar, t) * t);
  gn += eb;
  gk -= eb;
  epb += eb;
}

// Reverse of one substep.  s0 = state at its start (from the tape); A: in = adjoint of the state at its end,
// out = adjoint of the state at its start.  G accumulates material / action adjoints of this lane.
template <int VPL>
__device__ __forceinline__ void substep_reverse(const KParams& P, const Topo<VPL>& tp, const EnvConst<VPL>& c, const WarpSmem& sm, int env,
                                                const float ap[6], const float ac[6], int sub, const float* __restrict__ s0blk,
                                                const float* __restrict__ s1blk, LaneAdj<VPL>& A, GradAcc& G, float* acc_tape, int contact_flag, int side_slot) {
  const float h = P.h, inv_h = P.inv_h;
  float gm_rc = 0.0f, gm_sigy = 0.0f, gm_gamma = 0.0f;   // this substep's share of the material adjoints (a few terms per lane);
                                                         // the sums over substeps run in double (G.gm): they cancel heavily
  // ---- forward recompute with recording.  The start state is read from the tape twice (here and again for the
  // reverse of A2) rather than held in ~70 registers across the projection loop, the hottest part of the kernel.
  LaneState<VPL> s0;
  load_state<VPL>(s0blk, tp.base, P.NS, s0);
  LaneState<VPL> s = s0;
  EdgeCache<VPL> ec0, ec;
  edge_refresh<VPL>(tp, s0, ec0);
  edge_prev_refresh<VPL>(tp, s0, ec0);
  ec = ec0;
  SubRec<VPL> R;
  if (P.G > 0) {
    for (int k = tp.lane; k < P.G * 24; k += 32) sm.posebar[k] = 0.0f;
  }
  if (contact_flag == 1) {
    // the substep applied a self-contact correction and left no side record: recompute it with recording (candidate list, depth sums, corrections)
    ContactCache<VPL> cc;
    cc.reset(-1.0f);
    substep<VPL, 1>(P, tp, c, sm, env, ap, ac, sub, s, ec, R, acc_tape, cc, const_cast<float*>(s0blk) + (size_t)TAPE_LAM * P.NS);
  } else {
    // common case: everything the reverse needs is on the tape record written by the replay
    load_rows3<VPL>(s0blk + (size_t)TAPE_DX * P.NS, tp.base, P.NS, R.dx);
    load_rows3<VPL>(s0blk + (size_t)TAPE_V1 * P.NS, tp.base, P.NS, R.v1);
    load_row<VPL>(s0blk + (size_t)TAPE_S * P.NS, tp.base, P.NS, R.S);
    float am[VPL];
    load_row<VPL>(s0blk + (size_t)TAPE_ACT * P.NS, tp.base, P.NS, am);
#pragma unroll
    for (int k = 0; k < VPL; ++k) {
      R.active[k] = __float_as_uint(am[k]);
      R.v3[k] = (c.kin[k] == KIN_FREE) ? axpy(R.v1[k], inv_h, R.dx[k]) : R.v1[k];   // v^3 = v^1 + dx/h without friction (the forward's expression)
      R.t_old[k] = ec0.t[k];
    }
    R.ncand = 0; R.any_pen = 0; R.jac_mask = 0u;
    if (contact_flag == 2) {
      // self-contact data of the substep from its side record: candidate list, depth sums, v^3 (which includes friction here);
      // the summed corrections of the Jacobi passes are read from the record in the reverse loop
      const float* sr = P.side + (size_t)side_slot * P.side_floats;
      R.ncand = reinterpret_cast<const int*>(sr)[0];
      R.jac_mask = reinterpret_cast<const unsigned*>(sr)[1];
      R.any_pen = 1;
      load_rows3<VPL>(sr + side_off_v3(), tp.base, P.NS, R.v3);
      const unsigned* cs = reinterpret_cast<const unsigned*>(sr + side_off_cand(P));
      unsigned* cd = reinterpret_cast<unsigned*>(sm.cand);
      for (int p = tp.lane; p < (R.ncand + 1) / 2; p += 32) cd[p] = cs[p];
      for (int p = tp.lane; p < R.ncand; p += 32) sm.dp[p] = sr[side_off_dp(P) + p];
#pragma unroll
      for (int k = 0; k < VPL; ++k) sm.mid[4 * sm.NP + vpos<VPL>(tp.base + k)] = c.w[k];
      acc_tape = const_cast<float*>(sr) + side_off_acc(P);
      __syncwarp();
    }
    // state at the end of the substep = start state of the next record (positions and directors are all that is used)
    load_rows3<VPL>(s1blk + (size_t)ROW_X * P.NS, tp.base, P.NS, s.x);
    load_rows3<VPL>(s1blk + (size_t)ROW_XL * P.NS, tp.base, P.NS, s.xl);
    load_rows3<VPL>(s1blk + (size_t)ROW_D1 * P.NS, tp.base, P.NS, s.d1);
    edge_refresh<VPL>(tp, s, ec);
    edge_prev_refresh<VPL>(tp, s, ec);
    substep_idle_syncs(P, sm);
  }
  if (P.G > 0) publish_poses(P, env, tp.lane, ap, ac, sub, sm.pose);   // keep this substep's poses for the reverse
#pragma unroll
  for (int k = 0; k < VPL; ++k) R.xp[k] = axpy(s0.x[k], h, R.v1[k]);   // x^p by the forward's own expression: same bits

  f3 tbar_old[VPL], tbar_new[VPL];
#pragma unroll
  for (int k = 0; k < VPL; ++k) { tbar_old[k] = zero3<float>(); tbar_new[k] = zero3<float>(); }

  phase_sync(sm, 8u);
  // ---- reverse A9: plasticity (Eq.11), then the frame transport
  if (P.plasticity) {
    const float Y = c.sigy * c.l0;
    f3 ptb = zero3<float>(), pdb = zero3<float>();
#pragma unroll
    for (int k = 0; k < VPL; ++k) {
      if (tp.interior[k]) {
        const f3 ta = (k == 0) ? ec.pt : ec.t[k > 0 ? k - 1 : 0];
        const f3 da = (k == 0) ? ec.pd1 : s.d1[k > 0 ? k - 1 : 0];
        float k1, k2;
        material_curvature<float>(ta, ec.t[k], da, s.d1[k], k1, k2);
        float k1bar = 0.f, k2bar = 0.f, Ybar = 0.f;
        plasticity_adj<float>(k1, k2, s0.kb1[k], s0.kb2[k], Y, c.rc, A.kb1[k], A.kb2[k], k1bar, k2bar, Ybar, gm_rc);
        gm_sigy += Ybar * c.l0;
        f3 tab = zero3<float>(), tbb = zero3<float>(), dab = zero3<float>(), dbb = zero3<float>();
        material_curvature_adj<float>(ta, ec.t[k], da, s.d1[k], k1bar, k2bar, tab, tbb, dab, dbb);
        tbar_new[k] += tbb;
        A.d1[k] += dbb;
        if (k == 0) { ptb += tab; pdb += dab; }
        else { tbar_new[k > 0 ? k - 1 : 0] += tab; A.d1[k > 0 ? k - 1 : 0] += dab; }
      }
    }
    add_at_last<VPL>(tbar_new, tp.ks, shfl3(ptb, tp.nl));
    add_at_last<VPL>(A.d1, tp.ks, shfl3(pdb, tp.nl));
  }
#pragma unroll
  for (int k = 0; k < VPL; ++k) {
    if (tp.evalid[k]) {
      f3 tob = zero3<float>(), tnb = zero3<float>(), dob = zero3<float>();
      frame_update_adj<float>(R.t_old[k], ec.t[k], s0.d1[k], A.d1[k], tob, tnb, dob);
      tbar_old[k] += tob; tbar_new[k] += tnb; A.d1[k] = dob;
    } else A.d1[k] = zero3<float>();
  }
  {   // new tangents -> new positions
    f3 send = zero3<float>();
#pragma unroll
    for (int k = 0; k < VPL; ++k)
      if (tp.evalid[k]) scatter_edge<VPL>(A.x, send, k, tp.ks, normalize_adj<float>(ec.t[k], ec.iL[k], tbar_new[k], 0.0f));
    A.x[0] += shfl3(send, tp.pl);
  }

  phase_sync(sm, 16u);
  // ---- reverse A8 commit
  f3 velbar[VPL];
  GraspAcc ga;
  ga.init();
#pragma unroll
  for (int k = 0; k < VPL; ++k) {
    velbar[k] = zero3<float>();
    if (c.kin[k] == KIN_FREE) velbar[k] = axpy(A.v[k], h, A.x[k]);
    else if (c.kin[k] >= KIN_GRASP0) { ga.add(P, sm, c.kin[k], A.x[k]); velbar[k] = A.v[k]; A.x[k] = zero3<float>(); }
    A.v[k] = zero3<float>();
  }
  ga.flush(sm);

  {   // old tangents (frame transport) -> old positions, while the old edge geometry is still at hand
    f3 send = zero3<float>();
#pragma unroll
    for (int k = 0; k < VPL; ++k)
      if (tp.evalid[k]) scatter_edge<VPL>(A.x, send, k, tp.ks, normalize_adj<float>(ec0.t[k], ec0.iL[k], tbar_old[k], 0.0f));
    A.x[0] += shfl3(send, tp.pl);
  }

  phase_sync(sm, 32u);
  // ---- reverse A7 rigid coupling
  f3 ybar[VPL];
#pragma unroll
  for (int k = 0; k < VPL; ++k) {
    ybar[k] = zero3<float>();
    if (c.kin[k] == KIN_FREE && R.active[k]) {
      const CoupleAdj ca = rigid_coupling_adj(P, couple_const(P), sm.base, sm.NP, env, R.active[k], R.xp[k] + R.dx[k], R.v3[k], c.mu_r, velbar[k]);
      velbar[k] = ca.velbar; ybar[k] = ca.ybar;
    }
  }

  phase_sync(sm, 64u);
  // ---- reverse A6 friction + reconciliation.  velbar is now the adjoint of v^3.
  if (P.self_contact && R.ncand > 0) {
    for (int p = tp.lane; p < R.ncand; p += 32) sm.dpbar[p] = 0.0f;
    __syncwarp();
  }
  if (P.self_contact && R.any_pen) {
#pragma unroll
    for (int k = 0; k < VPL; ++k) {
      const int i = vpos<VPL>(tp.base + k);
      sts3(sm.ys, sm.NP, i, R.xp[k] + R.dx[k]);
      sts3(sm.vs, sm.NP, i, (c.kin[k] == KIN_FREE) ? axpy(R.v1[k], inv_h, R.dx[k]) : R.v1[k]);
      sts3(sm.vbar, sm.NP, i, (c.kin[k] == KIN_FREE) ? velbar[k] : zero3<float>());
      sts3(sm.ybar, sm.NP, i, zero3<float>());
    }
    __syncwarp();
    friction_pass_adj<VPL>(P, tp.lane, sm.base, R.ncand, c.mu_s);
    __syncwarp();
#pragma unroll
    for (int k = 0; k < VPL; ++k) {
      const int i = vpos<VPL>(tp.base + k);
      velbar[k] += lds3(sm.acc, sm.NP, i);
      ybar[k] += lds3(sm.ybar, sm.NP, i);
      sts3(sm.acc, sm.NP, i, zero3<float>());
    }
    __syncwarp();
  }
  f3 v1bar[VPL], dxb[VPL], xpb[VPL], epb[VPL];
  float Sb[VPL];
#pragma unroll
  for (int k = 0; k < VPL; ++k) {
    v1bar[k] = velbar[k];
    dxb[k] = (c.kin[k] == KIN_FREE) ? axpy(ybar[k], inv_h, velbar[k]) : ybar[k];
    xpb[k] = ybar[k];
    epb[k] = zero3<float>();
    Sb[k] = 0.0f;
  }

  phase_sync(sm, 128u);
  // ---- reverse A5: iterations backwards; each Eq.10 update is undone from its stored multiplier
  f3 epred[VPL];   // the forward's predicted edge vectors, by the forward's expression (positions re-read: they are not held across the reverse of A9..A6)
  {
    LaneState<VPL> sx;
    load_rows3<VPL>(s0blk + (size_t)ROW_X * P.NS, tp.base, P.NS, sx.x);
    load_rows3<VPL>(s0blk + (size_t)ROW_XL * P.NS, tp.base, P.NS, sx.xl);
    const f3 xr = shfl3(sx.x[0], tp.nl), xlr = shfl3(sx.xl[0], tp.nl), v1r = shfl3(R.v1[0], tp.nl);
#pragma unroll
    for (int k = 0; k < VPL; ++k) epred[k] = axpy(edge_vec<VPL>(sx, xr, xlr, k, tp.ks), h, next_of<VPL>(R.v1, v1r, k, tp.ks) - R.v1[k]);
  }
  const float atil = c.stretch * inv_h * inv_h;
  double atilbar = 0.0;   // adjoint of the compliance term alpha~ = c / h^2: a sum of nearly cancelling terms
  float idn[VPL], wfar[VPL];   // as in substep(): far-vertex inverse mass, 1 / (w_j + w_j+1 + atil) or 0 for an idle slot
#pragma unroll
  for (int k = 0; k < VPL; ++k) {
    const bool red = (k & 1) == 0;
    const bool rem = !red && ((k == VPL - 1) || (k == tp.ks));
    const bool on = red ? ((k + 1 < tp.nv) && tp.evalid[k]) : (tp.evalid[k] && (k <= tp.ks));
    wfar[k] = rem ? c.wr : c.w[k + 1 < VPL ? k + 1 : k];
    const float wsum = c.w[k] + wfar[k];
    idn[k] = (P.stretch_mode == 1 && on && wsum > 0.0f) ? 1.0f / (wsum + atil) : 0.0f;
  }
  float lam_next[VPL];   // multipliers one iteration ahead: the tape read of iteration it - 1 is in flight while iteration it is reversed
  load_row<VPL>(s0blk + (size_t)(TAPE_LAM + (P.N_C > 0 ? P.N_C - 1 : 0)) * P.NS, tp.base, P.NS, lam_next);
  for (int it = P.N_C - 1; it >= 0; --it) {
    float lamv[VPL];   // multipliers of this iteration, one per owned edge (the odd ring's closing edge sits in its idle red slot)
#pragma unroll
    for (int k = 0; k < VPL; ++k) lamv[k] = lam_next[k];
    if (it > 0) load_row<VPL>(s0blk + (size_t)(TAPE_LAM + it - 1) * P.NS, tp.base, P.NS, lam_next);
    if (P.self_contact && ((R.jac_mask >> it) & 1u)) {
#pragma unroll
      for (int k = 0; k < VPL; ++k) {
        const int i = vpos<VPL>(tp.base + k);
        R.dx[k] -= lds3(acc_tape + (size_t)it * 3 * sm.NP, sm.NP, i);
        sts3(sm.ys, sm.NP, i, R.xp[k] + R.dx[k]);
        sts3(sm.vbar, sm.NP, i, dxb[k]);
        sts3(sm.ybar, sm.NP, i, zero3<float>());
      }
      __syncwarp();
      contact_pass_adj<VPL>(P, tp.lane, sm.base, R.ncand);
      __syncwarp();
#pragma unroll
      for (int k = 0; k < VPL; ++k) {
        const f3 yb = lds3(sm.ybar, sm.NP, vpos<VPL>(tp.base + k));
        dxb[k] += yb;
        xpb[k] += yb;
      }
      __syncwarp();
    }
    if (P.stretch_mode == 1) {
      if (P.odd_ring) {   // third colour
        f3 dxr = shfl3(R.dx[0], tp.nl), gr = shfl3(dxb[0], tp.nl);
        const f3 dxr0 = dxr, gr0 = gr;
#pragma unroll
        for (int k = 0; k < VPL; k += 2) {
          // on copies, written back unconditionally: a body guarded by `k == tp.ks` that updates the arrays in place makes
          // the compiler index them by ks, which puts them in local memory for the whole kernel
          const bool on = (k == tp.ks) && (tp.base + k == P.E - 1) && (c.w[k] + c.wr > 0.0f);
          f3 dxk = R.dx[k], dxn = dxr, gk = dxb[k], gn = gr, eb = epb[k];
          float Sk = R.S[k], sb = Sb[k], ab = 0.0f;
          if (on) edge_reverse(epred[k], lamv[k], c.w[k], c.wr, atil, dxk, dxn, Sk, gk, gn, sb, ab, eb);
          R.dx[k] = dxk; dxr = dxn; R.S[k] = Sk; dxb[k] = gk; gr = gn; Sb[k] = sb; atilbar += (double)ab; epb[k] = eb;
        }
        R.dx[0] += shfl3(dxr - dxr0, tp.pl);
        dxb[0] += shfl3(gr - gr0, tp.pl);
      }
      {   // black
        f3 dxr = shfl3(R.dx[0], tp.nl), gr = shfl3(dxb[0], tp.nl);
        const f3 dxr0 = dxr, gr0 = gr;
#pragma unroll
        for (int k = 1; k < VPL; k += 2) {
          if (k == VPL - 1) {
            edge_reverse_pre(epred[k], lamv[k], c.w[k], wfar[k], idn[k], atil, R.dx[k], dxr, R.S[k], dxb[k], gr, Sb[k], atilbar, epb[k]);
          } else {   // the far vertex is remote when this is the lane's last valid slot
            const int kn = k + 1 < VPL ? k + 1 : k;
            const bool rem = (k == tp.ks);
            f3 dxn = rem ? dxr : R.dx[kn], gn = rem ? gr : dxb[kn];
            edge_reverse_pre(epred[k], lamv[k], c.w[k], wfar[k], idn[k], atil, R.dx[k], dxn, R.S[k], dxb[k], gn, Sb[k], atilbar, epb[k]);
            dxr = rem ? dxn : dxr; gr = rem ? gn : gr;
            R.dx[kn] = rem ? R.dx[kn] : dxn; dxb[kn] = rem ? dxb[kn] : gn;
          }
        }
        R.dx[0] += shfl3(dxr - dxr0, tp.pl);
        dxb[0] += shfl3(gr - gr0, tp.pl);
      }
#pragma unroll
      for (int k = 0; k < VPL; k += 2)   // red (an odd ring keeps the closing edge's multiplier in its idle red slot: not this edge's)
        edge_reverse_pre(epred[k], idn[k] != 0.0f ? lamv[k] : 0.0f, c.w[k], wfar[k], idn[k], atil, R.dx[k], R.dx[k + 1], R.S[k], dxb[k], dxb[k + 1], Sb[k], atilbar, epb[k]);
    }
  }
  G.gm[GM_STRETCH] += (P.stretch_mode == 1) ? atilbar * (double)inv_h * (double)inv_h : 0.0;
  {   // predicted edge vectors -> predicted positions
    f3 send = zero3<float>();
#pragma unroll
    for (int k = 0; k < VPL; ++k)
      if (tp.evalid[k]) scatter_edge<VPL>(xpb, send, k, tp.ks, epb[k]);
    xpb[0] += shfl3(send, tp.pl);
  }

  phase_sync(sm, 256u);
  // ---- reverse A4 predict, A3 velocity
  LaneState<VPL> s0b;
  load_state<VPL>(s0blk, tp.base, P.NS, s0b);
  const float idamp = 1.0f / (1.0f + c.gamma * h), hm = h * c.inv_m;
  f3 fbar[VPL];
#pragma unroll
  for (int k = 0; k < VPL; ++k) {
    v1bar[k] = axpy(v1bar[k], h, xpb[k]);
    if (tp.vvalid[k]) A.x[k] += xpb[k];
    fbar[k] = zero3<float>();
    if (c.kin[k] == KIN_FREE) {
      A.v[k] = idamp * v1bar[k];
      fbar[k] = (hm * idamp) * v1bar[k];
      gm_gamma -= h * idamp * dot(v1bar[k], R.v1[k]);
    } else if (c.kin[k] >= KIN_GRASP0) {
      const f3 tb = inv_h * v1bar[k];
      ga.add(P, sm, c.kin[k], tb);
      A.x[k] -= tb;
    }
  }
  ga.flush(sm);

  phase_sync(sm, 512u);
  // ---- reverse A2 forces: bending elements (and the stretch force in ENERGY mode) -> old edge geometry
  {
    EdgeCache<VPL> eb0;
    edge_refresh<VPL>(tp, s0b, eb0);
    edge_prev_refresh<VPL>(tp, s0b, eb0);
    f3 tb2[VPL];
    float ib2[VPL];
#pragma unroll
    for (int k = 0; k < VPL; ++k) { tb2[k] = zero3<float>(); ib2[k] = 0.0f; }
    const f3 fb_prev = shfl3(pick_last<VPL>(fbar, tp.ks), tp.pl), fb_next = shfl3(fbar[0], tp.nl);
    const float sc = c.alpha / c.l0;
    f3 ptb = zero3<float>(), pdb = zero3<float>();
    float piLb = 0.0f, sbar = 0.0f;
#pragma unroll
    for (int k = 0; k < VPL; ++k) {
      if (tp.interior[k]) {
        const f3 ta = (k == 0) ? eb0.pt : eb0.t[k > 0 ? k - 1 : 0];
        const f3 da = (k == 0) ? eb0.pd1 : s0b.d1[k > 0 ? k - 1 : 0];
        const float ia = (k == 0) ? eb0.piL : eb0.iL[k > 0 ? k - 1 : 0];
        const f3 Gab = ((k == 0) ? fb_prev : fbar[k > 0 ? k - 1 : 0]) - fbar[k];
        const f3 Gbb = fbar[k] - next_of<VPL>(fbar, fb_next, k, tp.ks);
        f3 tab = zero3<float>(), tbb = zero3<float>(), dab = zero3<float>(), dbb = zero3<float>();
        float iab = 0.f, ibb = 0.f;
        bend_element_adj<float>(ta, eb0.t[k], ia, eb0.iL[k], da, s0b.d1[k], s0b.kb1[k], s0b.kb2[k], sc, Gab, Gbb, tab, tbb, iab, ibb, dab, dbb,
                                A.kb1[k], A.kb2[k], sbar);
        tb2[k] += tbb; ib2[k] += ibb; A.d1[k] += dbb;
        if (k == 0) { ptb += tab; pdb += dab; piLb += iab; }
        else { tb2[k > 0 ? k - 1 : 0] += tab; A.d1[k > 0 ? k - 1 : 0] += dab; ib2[k > 0 ? k - 1 : 0] += iab; }
      }
    }
    G.gm[GM_ALPHA] += (double)(sbar / c.l0);
    add_at_last<VPL>(tb2, tp.ks, shfl3(ptb, tp.nl));
    add_at_last<VPL>(A.d1, tp.ks, shfl3(pdb, tp.nl));
    add_at_last<VPL>(ib2, tp.ks, shfl(piLb, tp.nl));
    if (P.stretch_mode == 0) {
#pragma unroll
      for (int k = 0; k < VPL; ++k) {
        if (tp.evalid[k]) {
          const f3 Fb = fbar[k] - next_of<VPL>(fbar, fb_next, k, tp.ks);
          const float L = 1.0f / eb0.iL[k], eps = L / c.l0 - 1.0f, Ft = dot(Fb, eb0.t[k]);
          G.gm[GM_STRETCH] += (double)(eps * Ft);
          tb2[k] += (c.stretch * eps) * Fb;
          ib2[k] -= (c.stretch * Ft / c.l0) * L * L;
        }
      }
    }
    f3 send = zero3<float>();
#pragma unroll
    for (int k = 0; k < VPL; ++k)
      if (tp.evalid[k]) scatter_edge<VPL>(A.x, send, k, tp.ks, normalize_adj<float>(eb0.t[k], eb0.iL[k], tb2[k], ib2[k]));
    A.x[0] += shfl3(send, tp.pl);
  }

  G.gm[GM_RC] += (double)gm_rc; G.gm[GM_SIGY] += (double)gm_sigy; G.gm[GM_GAMMA] += (double)gm_gamma;
  phase_sync(sm, 1024u);
  // ---- reverse A1: pose adjoints -> action adjoints (lane g owns gripper g)
  if (P.G > 0) {
    __syncwarp();
    if (tp.lane < P.G) {
      const float tau0 = (float)sub / (float)P.n_sub, tau1 = (float)(sub + 1) / (float)P.n_sub;
      PoseBar<float> b0, b1;
      const float* pb = sm.posebar + tp.lane * 24;
      b0.p = mk3<float>(pb[0], pb[1], pb[2]); b1.p = mk3<float>(pb[12], pb[13], pb[14]);
#pragma unroll
      for (int k = 0; k < 9; ++k) { b0.R[k] = pb[3 + k]; b1.R[k] = pb[15 + k]; }
      make_pose_adj<float>(ap, ac, tau0, b0, G.apbar, G.acbar);
      make_pose_adj<float>(ap, ac, tau1, b1, G.apbar, G.acbar);
    }
    __syncwarp();
  }
}

// Segment adjoint: walks the substeps of steps t1-1 .. t0 backwards, one warp per env.  P.tape holds the state at
// the start of every substep of the segment (written by k_forward), P.adj the running state adjoint.
template <int VPL>
__global__ void __launch_bounds__(DLO_ADJ_WARPS * 32, 1) k_adjoint(const __grid_constant__ KParams P, int t0, int t1) {
  extern __shared__ __align__(16) float smem[];
  const int wpb = blockDim.x >> 5, wib = threadIdx.x >> 5, slot = blockIdx.x * wpb + wib;
  if (slot >= P.B) return;
  const int env = P.perm ? P.perm[slot] : slot;
  WarpSmem sm;
  sm.init(P, smem + (size_t)wib * P.sm_warp_floats, 33 * VPL);
  sm.sync_threads = 32 * min(wpb, P.B - (int)blockIdx.x * wpb);
  Topo<VPL> tp;
  tp.init(P);
  EnvConst<VPL> c;
  load_env<VPL>(P, env, tp, c);
  warp_setup<VPL>(P, env, tp.lane, sm);
  const size_t blk = (size_t)STATE_ROWS * P.NS;
  LaneAdj<VPL> A;
  load_adj<VPL>(P.adj + (size_t)env * blk, tp.base, P.NS, A);
  GradAcc G;
#pragma unroll
  for (int k = 0; k < 5; ++k) G.gm[k] = 0.0;
  float ap[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f}, ac[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  float* acc_tape = P.acc_tape ? P.acc_tape + (size_t)env * P.N_C * 3 * sm.NP : nullptr;
  for (int t = t1 - 1; t >= t0; --t) {
    if (P.G > 0) load_actions(P, env, tp.lane, t, ap, ac);
#pragma unroll
    for (int k = 0; k < 6; ++k) { G.apbar[k] = 0.0f; G.acbar[k] = 0.0f; }
    for (int sub = P.n_sub - 1; sub >= 0; --sub) {
      const size_t rec = (size_t)tape_rows(P.N_C) * P.NS, idx = (size_t)(t - t0) * P.n_sub + sub;
      const float* s0blk = P.tape + (idx * P.B + env) * rec;
      const float* s1blk = P.tape + ((idx + 1) * P.B + env) * rec;
      // the record of the substep reversed NEXT goes to L2 now (one bulk prefetch, no registers, no shared memory): with two
      // warps per scheduler there is nothing to hide a DRAM round trip behind when its rows are loaded
      if (idx > 0 && tp.lane == 0)
        asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(P.tape + ((idx - 1) * P.B + env) * rec), "r"((unsigned)(rec * sizeof(float))) : "memory");
      const int cflag = P.tape_flag ? (int)P.tape_flag[idx * P.B + env] : 1;
      const int slot = (cflag == 2) ? P.tape_slot[idx * P.B + env] : -1;
      substep_reverse<VPL>(P, tp, c, sm, env, ap, ac, sub, s0blk, s1blk, A, G, acc_tape, cflag, slot);
    }
    if (P.g_actions && tp.lane < P.G) {
      float* gc = P.g_actions + (((size_t)t * P.B + env) * P.G + tp.lane) * 6;
#pragma unroll
      for (int k = 0; k < 6; ++k) gc[k] += G.acbar[k];
      if (t > 0) {
        float* gp = P.g_actions + (((size_t)(t - 1) * P.B + env) * P.G + tp.lane) * 6;
#pragma unroll
        for (int k = 0; k < 6; ++k) gp[k] += G.apbar[k];
      }
    }
  }
  store_adj<VPL>(P.adj + (size_t)env * blk, tp.base, P.NS, A);
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    double v = G.gm[k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(DLO_FULL, v, o);
    if (tp.lane == 0) P.gmat[(size_t)env * 5 + k] += (float)v;
  }
  verify_guards(P, env, tp.lane, sm);
}

// seeds of the reverse pass -> running adjoint block; gradients out of it
__global__ void k_seed_adjoint(int B, int N, int NS, const float* gx, const float* gv, float* adj) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (size_t)B * STATE_ROWS * NS) return;
  const int i = (int)(idx % NS), q = (int)((idx / NS) % STATE_ROWS), env = (int)(idx / ((size_t)NS * STATE_ROWS));
  float val = 0.0f;
  if (i < N) {
    if (q < 3 && gx) val = gx[((size_t)env * 3 + q) * N + i];
    else if (q >= 3 && q < 6 && gv) val = gv[((size_t)env * 3 + q - 3) * N + i];
  }
  adj[idx] = val;
}

}  // namespace dlo
