// rod_kernels.cuh — the __global__ entry points: set-up (A0), state packing, the persistent forward segment
// kernel.  The adjoint kernel lives in rod_adjoint.cuh.  Included once by dlo_api.cu.
#pragma once
#include "rod_substep.cuh"

namespace dlo {

// warps (= envs) per CTA: the CTA's warps walk the kernel in lockstep (phase_sync), so more warps per CTA share each
// instruction-cache fill.  Forward: 2 CTAs of 4..8 warps per SM at <= 128 registers (the register file is split four ways: 16 K registers per scheduler, so more than 3 warps on a scheduler means <= 128 registers each); the host picks the count that fills whole waves; adjoint: 1 CTA of 8 warps at 255.
// (upper bounds: the host lowers them when the per-warp shared memory of a large rope would not fit)
#ifndef DLO_FWD_WARPS
#define DLO_FWD_WARPS 8
#endif
#ifndef DLO_ADJ_WARPS
#define DLO_ADJ_WARPS 8
#endif

// ---------------------------------------------------------------------------------------------------------
// host-side helpers shared with the launcher
struct SetupArgs {
  int B, N, E, NS, ring, G, M, kappa_from_x0;
  const float *x0, *v0, *kb0;      // user arrays [B][3][N], [B][2][N] (kb0 may be null)
  const float* pose0;              // [B][G][6]
  const int* grasp_verts;          // [B][G][M]
  const uint8_t* cuts;             // [B][N] absent edges (dlo_set_cuts) or null
  float* state;                    // [B][11][NS]
  float* qloc;                     // [B][G*M][3]
};

typedef V3<double> d3;

// A0 (L340, L400-404 Eq.12): frames by space-parallel transport from edge 0, ring holonomy correction,
// rest curvature, grasp-local coordinates.  One thread per env; evaluated in fp64 once per rollout.
__global__ void k_set_state(SetupArgs A) {
  const int env = blockIdx.x * blockDim.x + threadIdx.x;
  if (env >= A.B) return;
  const int N = A.N, E = A.E, NS = A.NS;
  const float* X = A.x0 + (size_t)env * 3 * N;
  const float* V = A.v0 + (size_t)env * 3 * N;
  float* S = A.state + (size_t)env * STATE_ROWS * NS;
  for (int q = 0; q < STATE_ROWS; ++q)
    for (int i = 0; i < NS; ++i) S[q * NS + i] = 0.0f;
  for (int i = 0; i < N; ++i)
    for (int k = 0; k < 3; ++k) { S[(ROW_X + k) * NS + i] = X[k * N + i]; S[(ROW_V + k) * NS + i] = V[k * N + i]; }
  auto xv = [&](int i) { return mk3<double>((double)X[i], (double)X[N + i], (double)X[2 * N + i]); };
  auto tang = [&](int j) { d3 e = xv((j + 1 < N) ? j + 1 : 0) - xv(j); return (1.0 / sqrt(dot(e, e))) * e; };
  auto put_d1 = [&](int j, const d3& d) { S[(ROW_D1 + 0) * NS + j] = (float)d.x; S[(ROW_D1 + 1) * NS + j] = (float)d.y; S[(ROW_D1 + 2) * NS + j] = (float)d.z; };
  const uint8_t* cut = A.cuts ? A.cuts + (size_t)env * N : nullptr;   // several DLOs: every rope starts a frame chain of its own
  auto absent = [&](int j) { return cut && cut[j] != 0; };
  d3 zhat = mk3<double>(0, 0, 1), yhat = mk3<double>(0, 1, 0);
  auto first_director = [&](const d3& t) {
    d3 cz = cross(t, zhat);
    d3 ref = (sqrt(dot(cz, cz)) < 1e-6) ? yhat : zhat;
    d3 u = ref - dot(ref, t) * t;
    return (1.0 / sqrt(dot(u, u))) * u;
  };
  d3 t0 = tang(0);
  d3 d0 = first_director(t0), d = d0, tp = t0;
  double psiH = 0.0;
  if (A.ring) {   // first pass: holonomy of the closed loop
    for (int j = 1; j < E; ++j) { d3 tj = tang(j); d = ptransport<double>(tp, tj, d); tp = tj; }
    d3 uu = ptransport<double>(tp, t0, d);
    psiH = atan2(dot(cross(d0, uu), t0), dot(d0, uu));
    d = d0; tp = t0;
  }
  bool fresh = false;
  for (int j = 0; j < E; ++j) {
    if (absent(j)) { fresh = true; continue; }   // no frame on an absent edge (the row stays zero)
    d3 tj = tang(j);
    if (fresh) { d = first_director(tj); tp = tj; fresh = false; }
    else if (j > 0) { d = ptransport<double>(tp, tj, d); tp = tj; }
    d3 out = d;
    if (A.ring) {   // Eq.12: rotate by phi^j = -psiH * j / E about the tangent
      const double phi = -psiH * (double)j / (double)E;
      out = cos(phi) * d + sin(phi) * cross(tj, d);
    }
    put_d1(j, out);
  }
  if (A.kb0) {
    const float* Kb = A.kb0 + (size_t)env * 2 * N;
    for (int i = 0; i < N; ++i) { S[ROW_KB * NS + i] = Kb[i]; S[(ROW_KB + 1) * NS + i] = Kb[N + i]; }
  } else if (A.kappa_from_x0) {
    for (int i = 0; i < N; ++i) {
      if (!(A.ring || (i >= 1 && i <= N - 2))) continue;
      if (absent(i - 1 >= 0 ? i - 1 : 0) || absent(i)) continue;   // a rope end has no bending element
      const int a = (i + N - 1) % N;
      d3 da = mk3<double>(S[ROW_D1 * NS + a], S[(ROW_D1 + 1) * NS + a], S[(ROW_D1 + 2) * NS + a]);
      d3 db = mk3<double>(S[ROW_D1 * NS + i], S[(ROW_D1 + 1) * NS + i], S[(ROW_D1 + 2) * NS + i]);
      double k1, k2;
      material_curvature<double>(tang(a), tang(i), da, db, k1, k2);
      S[ROW_KB * NS + i] = (float)k1; S[(ROW_KB + 1) * NS + i] = (float)k2;
    }
  }
  for (int g = 0; g < A.G; ++g) {   // q_k = R_g(0)^T (x_k(0) - p_g(0))
    const float* a = A.pose0 + ((size_t)env * A.G + g) * 6;
    M3<double> R = rodrigues<double>(mk3<double>(a[3], a[4], a[5]));
    d3 p = mk3<double>(a[0], a[1], a[2]);
    for (int k = 0; k < A.M; ++k) {
      const int v = A.grasp_verts[((size_t)env * A.G + g) * A.M + k];
      float* q = A.qloc + (((size_t)env * A.G + g) * A.M + k) * 3;
      d3 l = (v >= 0 && v < N) ? mulT(R, xv(v) - p) : zero3<double>();
      q[0] = (float)l.x; q[1] = (float)l.y; q[2] = (float)l.z;
    }
  }
}

// kinematic codes from pins and grasp sets (grasp flags on top of pins, like the problem statement R-19)
__global__ void k_build_kin(int B, int N, int NS, int G, int M, const uint8_t* pins, const int* grasp_verts, const uint8_t* cuts, uint8_t* kin) {
  const int env = blockIdx.x * blockDim.x + threadIdx.x;
  if (env >= B) return;
  uint8_t* K = kin + (size_t)env * NS;
  for (int i = 0; i < NS; ++i) K[i] = (i < N && pins && pins[(size_t)env * N + i]) ? KIN_PINNED : (i < N ? KIN_FREE : KIN_PINNED);
  if (grasp_verts)
    for (int g = 0; g < G; ++g)
      for (int k = 0; k < M; ++k) {
        const int v = grasp_verts[((size_t)env * G + g) * M + k];
        if (v >= 0 && v < N) K[v] = (uint8_t)(KIN_GRASP0 + g * M + k);
      }
  if (cuts)
    for (int i = 0; i < N; ++i)
      if (cuts[(size_t)env * N + i]) K[i] |= KIN_CUT;
}

struct MatArgs { const float* a[MAT_N]; };
__global__ void k_pack_material(int B, MatArgs m, float* out) {
  const int env = blockIdx.x * blockDim.x + threadIdx.x;
  if (env >= B) return;
#pragma unroll
  for (int k = 0; k < MAT_N; ++k) out[(size_t)env * MAT_N + k] = m.a[k][env];
}

// internal state block -> user arrays (any may be null)
__global__ void k_get_state(int B, int N, int NS, const float* state, float* x, float* v, float* d1, float* kb, float* xl) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (size_t)B * STATE_ROWS * N) return;
  const int i = (int)(idx % N), q = (int)((idx / N) % STATE_ROWS), env = (int)(idx / ((size_t)N * STATE_ROWS));
  const float val = state[((size_t)env * STATE_ROWS + q) * NS + i];
  if (q < 3) { if (x) x[((size_t)env * 3 + q) * N + i] = val; }
  else if (q < 6) { if (v) v[((size_t)env * 3 + q - 3) * N + i] = val; }
  else if (q < 9) { if (d1) d1[((size_t)env * 3 + q - 6) * N + i] = val; }
  else if (q < 11) { if (kb) kb[((size_t)env * 2 + q - 9) * N + i] = val; }
  else if (xl) xl[((size_t)env * 3 + q - 11) * N + i] = val;
}

// user arrays -> internal state block (exact restore: the inverse of k_get_state; padding columns zeroed)
__global__ void k_put_state(int B, int N, int NS, const float* x, const float* v, const float* d1, const float* kb, const float* xl, float* state) {
  const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (size_t)B * STATE_ROWS * NS) return;
  const int i = (int)(idx % NS), q = (int)((idx / NS) % STATE_ROWS), env = (int)(idx / ((size_t)NS * STATE_ROWS));
  float val = 0.0f;
  if (i < N) {
    if (q < 3) val = x[((size_t)env * 3 + q) * N + i];
    else if (q < 6) val = v[((size_t)env * 3 + q - 3) * N + i];
    else if (q < 9) val = d1[((size_t)env * 3 + q - 6) * N + i];
    else if (q < 11) val = kb[((size_t)env * 2 + q - 9) * N + i];
    else val = xl ? xl[((size_t)env * 3 + q - 11) * N + i] : 0.0f;
  }
  state[idx] = val;
}

// ---------------------------------------------------------------------------------------------------------
// per-warp start-up shared by the forward and adjoint kernels: primitives (boxes expanded to rotation
// matrices), grasp-local coordinates, zeroed accumulators
template <int VPL>
__device__ __forceinline__ void warp_setup(const KParams& P, int env, int lane, const WarpSmem& sm) {
  for (int k = lane; k < P.K; k += 32) {
    const float* src = P.prim + ((size_t)env * P.K + k) * PRIM_NP;
    float* dst = sm.prim + k * PRIM_SM_STRIDE;
    for (int q = 0; q < PRIM_NP; ++q) dst[q] = src[q];
    const int ty = P.prim_type[k];
    if (ty == 3) {
      M3<float> R = rodrigues<float>(mk3<float>(src[6], src[7], src[8]));
      for (int q = 0; q < 9; ++q) dst[6 + q] = R.m[q];
    }
    // bounding sphere
    dst[PRIM_BC] = src[0]; dst[PRIM_BC + 1] = src[1]; dst[PRIM_BC + 2] = src[2];
    dst[PRIM_BR] = -1.0f;
    if (ty == 1) {
      const f3 a = mk3<float>(src[0], src[1], src[2]), b = mk3<float>(src[3], src[4], src[5]), mid = 0.5f * (a + b), hb = 0.5f * (b - a);
      dst[PRIM_BC] = mid.x; dst[PRIM_BC + 1] = mid.y; dst[PRIM_BC + 2] = mid.z;
      dst[PRIM_BR] = sqrt_(dot(hb, hb)) + src[6];
    } else if (ty == 2) dst[PRIM_BR] = sqrt_(src[6] * src[6] + src[7] * src[7]);
    else if (ty == 3) dst[PRIM_BR] = sqrt_(src[3] * src[3] + src[4] * src[4] + src[5] * src[5]);
  }
  for (int k = lane; k < P.G * P.M * 3; k += 32) sm.q[k] = P.qloc[(size_t)env * P.G * P.M * 3 + k];
  if (P.checks)
    for (int k = lane; k < 4 * P.n_guard; k += 32) reinterpret_cast<unsigned*>(sm.base)[P.sm_guard[k >> 2] + (k & 3)] = DLO_GUARD_WORD;
  __syncwarp();
  if (P.checks == 2 && P.K > 0 && lane == 0) sm.prim[P.K * PRIM_SM_STRIDE] = 0.0f;   // self-test of the check: one word past the primitives
  if (P.self_contact)
    for (int k = lane; k < 3 * sm.NP; k += 32) sm.acc[k] = 0.0f;
  __syncwarp();
}

__device__ __forceinline__ void load_actions(const KParams& P, int env, int lane, int t, float ap[6], float ac[6]) {
  if (lane < P.G) {
    const int ta = P.t_base + t;   // absolute frame (a rollout restored by dlo_restore_state starts at t_base > 0)
    const float* cur = P.actions + (((size_t)ta * P.B + env) * P.G + lane) * 6;
    const float* prv = (ta > 0) ? P.actions + (((size_t)(ta - 1) * P.B + env) * P.G + lane) * 6 : P.pose0 + ((size_t)env * P.G + lane) * 6;
#pragma unroll
    for (int k = 0; k < 6; ++k) { ap[k] = prv[k]; ac[k] = cur[k]; }
  }
}

// Env -> warp-slot order of the next launch: envs sorted by a work key, heaviest first (counting sort, one CTA).  The
// warps of a CTA walk in lockstep and wait for their slowest member at every phase barrier, so envs that do the same
// amount of self-contact work belong in the same CTA; envs are independent, the order changes no result.
__global__ void __launch_bounds__(1024, 1) k_sort_envs(int B, const int* __restrict__ stat, int col, int shift, int* __restrict__ perm) {
  __shared__ int hist[1024];
  const int tid = threadIdx.x;
  hist[tid] = 0;
  __syncthreads();
  for (int i = tid; i < B; i += 1024) atomicAdd(&hist[min(max(stat[2 * i + col] >> shift, 0), 1023)], 1);
  __syncthreads();
  if (tid == 0) {   // start offsets, descending keys
    int run = 0;
    for (int k = 1023; k >= 0; --k) { const int n = hist[k]; hist[k] = run; run += n; }
  }
  __syncthreads();
  for (int i = tid; i < B; i += 1024) perm[atomicAdd(&hist[min(max(stat[2 * i + col] >> shift, 0), 1023)], 1)] = i;
}

// DLO_CHECKS: every guard word behind the warp's shared-memory regions must still be there
__device__ __forceinline__ void verify_guards(const KParams& P, int env, int lane, const WarpSmem& sm) {
  if (!P.checks) return;
  __syncwarp();
  bool bad = false;
  for (int k = lane; k < 4 * P.n_guard; k += 32) bad |= reinterpret_cast<const unsigned*>(sm.base)[P.sm_guard[k >> 2] + (k & 3)] != DLO_GUARD_WORD;
  if (__any_sync(DLO_FULL, bad) && lane == 0) atomicOr(P.flags + env, FLAG_GUARD);
}

template <int VPL> __device__ __forceinline__ bool state_finite(const LaneState<VPL>& s) {
  float a = 0.0f;
#pragma unroll
  for (int k = 0; k < VPL; ++k) a += (s.x[k].x + s.x[k].y + s.x[k].z) + (s.v[k].x + s.v[k].y + s.v[k].z) * 0.0f;
  return isfinite(a);
}

// Persistent forward segment: steps t0..t1-1 of every env, one warp per env, state in registers throughout.
// stride > 0: checkpoint (t+1)/stride written after every `stride`-th step (L115).  write_tape: the state at
// the start of every substep goes to P.tape (replay half of the reverse pass).
// Persistent forward segment: steps t0..t1-1 of every env, one warp per env, state in registers throughout.
// stride > 0: checkpoint (t+1)/stride written after every `stride`-th step (L115).  TAPE = true is the replay half of
// the reverse pass: a tape record per substep goes to P.tape, and the segment's final state to record [n_substeps].
template <int VPL, bool TAPE>
__global__ void __launch_bounds__(DLO_FWD_WARPS * 32, VPL <= 4 ? 2 : 1) k_forward(const __grid_constant__ KParams P, int t0, int t1, int stride) {
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
  // work: self-contact work units of this launch; npen: which tenths of the launch's substeps applied a self-contact
  // correction (bit 9 = the last tenth) - envs with the same pattern recompute the same substeps in the adjoint
  int work = 0, npen = 0;
  const size_t blk = (size_t)STATE_ROWS * P.NS, rec = (size_t)tape_rows(P.N_C) * P.NS;
  LaneState<VPL> s;
  load_state<VPL>(P.state + (size_t)env * blk, tp.base, P.NS, s);
  EdgeCache<VPL> ec;
  edge_refresh<VPL>(tp, s, ec);
  edge_prev_refresh<VPL>(tp, s, ec);
  float ap[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f}, ac[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  SubRec<VPL> R;
  ContactCache<VPL> cc;
  cc.reset(-1.0f);
  for (int t = t0; t < t1; ++t) {
    if (P.G > 0) load_actions(P, env, tp.lane, t, ap, ac);
    for (int sub = 0; sub < P.n_sub; ++sub) {
      if (TAPE) {
        const size_t idx = (size_t)(t - t0) * P.n_sub + sub;
        float* tb = P.tape + (idx * P.B + env) * rec;
        store_state<VPL>(tb, tp.base, P.NS, s);
        substep<VPL, 2>(P, tp, c, sm, env, ap, ac, sub, s, ec, R, nullptr, cc, tb + (size_t)TAPE_LAM * P.NS);
        store_rows3<VPL>(tb + (size_t)TAPE_DX * P.NS, tp.base, P.NS, R.dx);
        store_rows3<VPL>(tb + (size_t)TAPE_V1 * P.NS, tp.base, P.NS, R.v1);
        store_row<VPL>(tb + (size_t)TAPE_S * P.NS, tp.base, P.NS, R.S);
        float am[VPL];
#pragma unroll
        for (int k = 0; k < VPL; ++k) am[k] = __uint_as_float(R.active[k]);
        store_row<VPL>(tb + (size_t)TAPE_ACT * P.NS, tp.base, P.NS, am);
        int flag = R.any_pen;
        if (R.any_pen && R.side_slot >= 0) {   // what the reverse pass needs of this substep's self-contact, so that it need not recompute it
          float* sr = P.side + (size_t)R.side_slot * P.side_floats;
          if (tp.lane == 0) { reinterpret_cast<int*>(sr)[0] = R.ncand; reinterpret_cast<unsigned*>(sr)[1] = R.jac_mask; P.tape_slot[idx * P.B + env] = R.side_slot; }
          store_rows3<VPL>(sr + side_off_v3(), tp.base, P.NS, R.v3);
          const unsigned* cs = reinterpret_cast<const unsigned*>(sm.cand);
          unsigned* cd = reinterpret_cast<unsigned*>(sr + side_off_cand(P));
          for (int p = tp.lane; p < (R.ncand + 1) / 2; p += 32) cd[p] = cs[p];
          for (int p = tp.lane; p < R.ncand; p += 32) sr[side_off_dp(P) + p] = sm.dp[p];
          flag = 2;
        }
        if (tp.lane == 0) P.tape_flag[idx * P.B + env] = (uint8_t)flag;
      } else {
        substep<VPL, 0>(P, tp, c, sm, env, ap, ac, sub, s, ec, R, nullptr, cc);
      }
      work += R.work; npen |= R.any_pen << ((((t - t0) * P.n_sub + sub) * 10) / ((t1 - t0) * P.n_sub));
    }
    if (stride > 0 && (t + 1) % stride == 0) store_state<VPL>(P.ckpt + ((size_t)((t + 1) / stride) * P.B + env) * blk, tp.base, P.NS, s);
  }
  if (TAPE) store_state<VPL>(P.tape + ((size_t)(t1 - t0) * P.n_sub * P.B + env) * rec, tp.base, P.NS, s);
  store_state<VPL>(P.state + (size_t)env * blk, tp.base, P.NS, s);
  if (P.stat && tp.lane == 0) { P.stat[2 * env] = work; P.stat[2 * env + 1] = npen; }
  const bool ok = state_finite<VPL>(s);
  if (__any_sync(DLO_FULL, !ok) && tp.lane == 0) atomicOr(P.flags + env, FLAG_NONFINITE);
  verify_guards(P, env, tp.lane, sm);
}

}  // namespace dlo
