/* dlo.h — C-ABI of the B200-native batched differentiable rod step (DLO-Lab hot path).
 *
 * What the library computes.  One "env" is one discretised deformable linear object (rope / band): N vertices
 * x_i with adapted frames per edge (Eq.1), advanced by symplectic Euler (L97) in frames of
 * `dt` made of `n_substeps` substeps (L438).  Each substep is, in this order (paper silent on the order;
 * DESIGN.md reading R-31): gripper kinematics (L129) -> internal forces: gravity, stretching Eq.2-3 (L344-351,
 * stretch mode ENERGY) and bending Eq.4-7 (L353-372) -> damped velocity update -> predict -> N_C iterations of
 * {inextensibility projection Eq.10 (L383-392) with optional compliance, red/black edge order; segment-segment
 * self-contact projection Eq.13 (L406-408)} -> velocity reconciliation + self-contact Coulomb friction (L410)
 * -> soft coupling against rigid primitives and gripper fingers (L103) -> commit -> frame transport and
 * bending plasticity Eq.11 (L394-398).  Ring topology initialises frames with the holonomy correction Eq.12
 * (L400-404).  `dlo_backward` is the exact reverse-mode derivative of that discrete map (branches frozen at
 * their forward outcome) under gradient checkpointing: one state per `checkpoint_stride` steps kept, segments
 * replayed in reverse (L115).
 *
 * Conventions
 *   - All arithmetic on the GPU is fp32; vertex positions are carried as an unevaluated sum of two fp32 numbers (x plus
 *     the residual x_lo that the rounding of x + h v dropped), so that edge vectors are exact differences.  B = batch, N = n_verts, E = N-1 (open) or N (ring), G = n_grippers,
 *     M = n_grasp_max, K = n_primitives, H = horizon (steps = frames).
 *   - Every array argument says "dev" (CUDA device pointer, 16-byte aligned) or "host".  Layouts are dense,
 *     row-major, last index fastest: x, v, d1 are [B][3][N] (SoA per env; d1 uses the first E columns);
 *     kappa_bar is [B][2][N]; actions are [H][B][G][6] = (position p, rotation vector rho) of each gripper
 *     reached exactly at the END of step t (R-20).
 *   - Ownership: the caller owns every buffer it passes.  The library reads / writes them asynchronously on
 *     the stream given at create and keeps no pointer after the call returns, except `actions` (borrowed until
 *     the next dlo_set_actions / dlo_destroy: dlo_backward replays them).  Checkpoints, tape and per-env
 *     constants live in library-owned device memory (size: dlo_scratch_bytes); so does the staging of the *_host
 *     calls (per handle, freed by dlo_destroy).
 *   - Device: a handle belongs to the CUDA device that was current at dlo_create; every later call on it must be
 *     made with that device current (DLO_ERR_BAD_STATE otherwise).
 *   - Errors: every call returns a dlo_status; nothing aborts or throws across the ABI; a failed call leaves
 *     the handle usable.  dlo_last_error() returns a thread-local message for the last failing call.
 *   - Threading: one handle <-> one stream; calls are stream-ordered and (except the *_host calls and
 *     dlo_check_numerics) do not synchronise the host.
 *   - There is no CPU fallback: without a CUDA device dlo_create returns DLO_ERR_CUDA.
 */
#ifndef DLO_H_
#define DLO_H_
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dlo_sim dlo_sim;   /* opaque, library-owned */
typedef int32_t dlo_status;

enum { DLO_OK = 0, DLO_ERR_INVALID_ARG = -1, DLO_ERR_BAD_STATE = -2 /* call order */, DLO_ERR_CUDA = -3,
       DLO_ERR_OOM = -4, DLO_ERR_UNSUPPORTED = -5, DLO_ERR_NUMERIC = -6 /* non-finite state / candidate overflow */ };
enum { DLO_OPEN = 0, DLO_RING = 1 };
enum { DLO_STRETCH_ENERGY = 0 /* Eq.2-3 force */, DLO_STRETCH_PROJECT = 1 /* Eq.10 projection (+compliance) */ };
enum { DLO_PRIM_PLANE = 0, DLO_PRIM_CAPSULE = 1, DLO_PRIM_CYLINDER = 2, DLO_PRIM_BOX = 3 };

#define DLO_MAX_VERTS 256       /* one warp per env, <= 8 vertices per lane */
#define DLO_MAX_GRIPPERS 4
#define DLO_MAX_PRIMITIVES 16
#define DLO_PRIM_NPARAM 10
#define DLO_N_MATERIAL_GRADS 5  /* stretch, bend, damping, yield, creep */

/* Host POD, copied at create.  Limits: 3 <= n_verts <= DLO_MAX_VERTS (ring: >= 4), n_grippers <= 4,
 * n_primitives <= 16, n_substeps >= 1, n_proj_iters >= 0. */
typedef struct {
  int32_t batch, n_verts, topology, n_substeps /* 5, L438 */, n_proj_iters /* N_C, L392 */, stretch_mode;
  int32_t enable_plasticity /* Eq.11 */, enable_self_contact /* Eq.13 */, self_skip /* min cyclic edge-index distance, 2 */;
  int32_t n_grippers, n_grasp_max, n_primitives;
  int32_t kappa_bar_from_x0;   /* 1: dlo_set_state(kappa_bar0 = NULL) takes the rest curvature of x0 instead of 0 */
  float dt, gravity[3], rope_radius, contact_softness /* eps_s of L103 */, influence_threshold /* 0.1, L103 */,
      restitution;
} dlo_config;

/* DEVICE pointers, each [B] fp32, copied at create.  `stretch` is k_s (mode ENERGY, Eq.3) or the compliance c in
 * m/N (mode PROJECT; 0 = Eq.10 verbatim).  bend_stiffness is alpha = E A r^2 / 4 of Eq.7.  yield_curv in rad/m
 * (compared as sigma_y * l_bar with the integrated curvature of Eq.5), creep_rate = r_c of Eq.11. */
typedef struct {
  const float *mass_per_vertex, *rest_edge_len, *stretch, *bend_stiffness, *damping, *yield_curv, *creep_rate,
      *mu_rigid, *mu_self;
} dlo_material;

/* Create a simulator for `batch` independent envs on `cuda_stream` (a cudaStream_t, NULL = default stream).
 * Fails with DLO_ERR_INVALID_ARG on out-of-range sizes, DLO_ERR_CUDA without a device, DLO_ERR_OOM. */
dlo_status dlo_create(const dlo_config* cfg, const dlo_material* mat, void* cuda_stream, dlo_sim** out);
dlo_status dlo_destroy(dlo_sim* sim);

/* Scene.  Call before dlo_set_state (A0 captures grasp-local coordinates there).
 * pins: dev [B][N] uint8, non-zero = vertex fixed in space (w = 0).
 * primitives: types host [K] (same for all envs), params dev [B][K][10]:
 *   PLANE n(3), o          CAPSULE a(3), b(3), R          CYLINDER centre(3), unit axis(3), R, half-height
 *   BOX centre(3), half-extents(3), rotation vector(3).   All fixed in space (L103, kinematic bodies only).
 * grippers: init_pose dev [B][G][6] = a_{-1}; finger_geom dev [B][G][4] = gap, length, radius, pad (two capsule
 *   fingers from p + R(+-gap/2,0,0) to p + R(+-gap/2,0,length)); grasp_verts dev [B][G][M] int32, -1 = none:
 *   vertices carried rigidly by the gripper (kinematic, L103). */
dlo_status dlo_set_pins(dlo_sim* sim, const uint8_t* pinned);
/* Several DLOs in one env (PAPER.md L145 Separation, L155 Letter Art: Eq.13 acts between different ropes, L406).  The ropes
 * lie back to back in the env's vertex array; cut: dev [B][N] uint8, non-zero at vertex j = the edge (j, j+1) does not exist
 * (the last entry is ignored).  An absent edge carries no stretch force / Eq.10 constraint, no frame (its d1 column stays 0)
 * and is no self-contact segment; the vertices next to it are rope ends (no bending element, no rest curvature); the frames
 * of A0 start afresh at the first edge of every rope.  All ropes of an env share its material, radius and rest edge length;
 * every pair of existing edges at index distance >= self_skip is a contact pair, within a rope or across ropes.  Call
 * before dlo_set_state.  DLO_ERR_UNSUPPORTED for the ring topology (one closed band per env) or self_skip != 2. */
dlo_status dlo_set_cuts(dlo_sim* sim, const uint8_t* cut);
dlo_status dlo_set_primitives(dlo_sim* sim, const int32_t* types, const float* params);
dlo_status dlo_set_grippers(dlo_sim* sim, const float* init_pose, const float* finger_geom, const int32_t* grasp_verts);

/* A0: initial state x0, v0 dev [B][3][N]; kappa_bar0 dev [B][2][N] or NULL.  Builds the frames by parallel
 * transport (ring: Eq.12) and the grasp-local coordinates. */
dlo_status dlo_set_state(dlo_sim* sim, const float* x0, const float* v0, const float* kappa_bar0);

/* actions dev [H][B][G][6]; borrowed (see Ownership).  Ignored when n_grippers == 0 (may be NULL). */
dlo_status dlo_set_actions(dlo_sim* sim, const float* actions, int32_t horizon);

/* Roll the state set by dlo_set_state forward by `horizon` steps.  checkpoint_stride > 0 keeps the state every
 * `stride` steps for dlo_backward (L115); 0 = forward only.  DLO_ERR_INVALID_ARG if horizon exceeds the actions. */
dlo_status dlo_rollout_forward(dlo_sim* sim, int32_t horizon, int32_t checkpoint_stride);

/* Current state; each pointer dev, may be NULL.  x, v, d1: [B][3][N]; kappa_bar: [B][2][N]. */
dlo_status dlo_get_state(dlo_sim* sim, float* x, float* v, float* d1, float* kappa_bar);

/* Low part of the positions (dev [B][3][N]): the state's positions are x + x_lo with x as dlo_get_state returns them and
 * |x_lo| <= ulp(x)/2.  Needed only to put a state back EXACTLY (dlo_restore_state). */
dlo_status dlo_get_position_residual(dlo_sim* sim, float* x_lo);

/* Exact restore (a checkpoint is "a single state"; the segment is re-run from it).  Puts back a
 * state as dlo_get_state (+ dlo_get_position_residual) returned it, bit for bit: x, v, d1 dev [B][3][N], kappa_bar dev
 * [B][2][N] (all four required), x_lo dev [B][3][N] or NULL (= 0: the positions are then exactly x), and `step_index`, the frame the next dlo_rollout_forward starts at: its step k uses the actions
 * a_{step_index+k-1} -> a_{step_index+k} of the array given to dlo_set_actions (a_{-1} = init_pose), so
 * step_index + horizon must not exceed that array.  No A0 runs: the frames are taken as given, and the grasp-local
 * coordinates stay those captured by the last dlo_set_state (DLO_ERR_BAD_STATE if there was none, or if the scene
 * changed since).  dlo_get_state + dlo_get_position_residual -> dlo_restore_state -> rollout of k steps equals k more steps of the original
 * rollout bitwise.  dlo_backward after such a rollout differentiates that segment only: g_actions [horizon][B][G][6]
 * is indexed from step_index (the gradient with respect to a_{step_index-1} is dropped, like that of init_pose),
 * g_x0 / g_v0 are with respect to the restored x, v.  dlo_set_state resets step_index to 0. */
dlo_status dlo_restore_state(dlo_sim* sim, const float* x, const float* x_lo, const float* v, const float* d1,
                             const float* kappa_bar, int32_t step_index);

/* Reverse pass of the last checkpointed rollout.  Seeds dL/dx_T, dL/dv_T dev [B][3][N] (NULL = 0).  Outputs
 * (dev, each may be NULL, WRITTEN not accumulated): g_actions [H][B][G][6], g_x0, g_v0 [B][3][N],
 * g_material [B][5] = d/d(stretch, bend_stiffness, damping, yield_curv, creep_rate).  The initial frames and
 * rest curvature are independent inputs (no gradient through A0).  DLO_ERR_BAD_STATE without a checkpointed
 * rollout. */
dlo_status dlo_backward(dlo_sim* sim, const float* dL_dx_T, const float* dL_dv_T, float* g_actions, float* g_x0,
                        float* g_v0, float* g_material);

/* After dlo_backward: the adjoint of the WHOLE start state of the rollout (what a chained segment-wise reverse pass
 * hands to the segment before, L115).  Each pointer dev, may be NULL: g_x, g_v, g_d1 [B][3][N], g_kappa_bar [B][2][N].
 * g_x, g_v equal dlo_backward's g_x0, g_v0.  DLO_ERR_BAD_STATE without a completed dlo_backward. */
dlo_status dlo_get_state_adjoint(dlo_sim* sim, float* g_x, float* g_v, float* g_d1, float* g_kappa_bar);

/* Host-buffer convenience calls (the end-to-end path): pageable or pinned HOST pointers, copies included, and
 * the call returns after the results have landed.  dlo_rollout_forward_host = set_state + set_actions +
 * rollout_forward + read-back of x_T, v_T (either may be NULL).  dlo_backward_host = seeds up, dlo_backward,
 * gradients down (any may be NULL). */
dlo_status dlo_rollout_forward_host(dlo_sim* sim, const float* x0, const float* v0, const float* kappa_bar0,
                                    const float* actions, int32_t horizon, int32_t checkpoint_stride, float* x_T,
                                    float* v_T);
dlo_status dlo_backward_host(dlo_sim* sim, const float* dL_dx_T, const float* dL_dv_T, float* g_actions, float* g_x0,
                             float* g_v0, float* g_material);

/* Synchronises the stream; DLO_ERR_NUMERIC if any env saw a non-finite state or overflowed its self-contact
 * candidate list since dlo_set_state; n_bad (host, may be NULL) receives the number of such envs. */
dlo_status dlo_check_numerics(dlo_sim* sim, int32_t* n_bad);

/* Device bytes the library allocates for this config / rollout shape (constants + checkpoints + tape; the tape of one
 * checkpoint segment, twice when there are several).  While more than a tenth of the device's memory stays free the handle
 * takes up to two more tape buffers of the same size (DLO_TAPE_BUFFERS = 1..4 caps the total): the forward rollout then
 * leaves its last segments on tape and the reverse pass skips their replay.  A handle that
 * is driven through the *_host calls additionally holds their device staging: 4 + 4 arrays [B][3][N], one [B][2][N],
 * one [B][5] and two [H][B][G][6] (actions, action gradients). */
size_t dlo_scratch_bytes(const dlo_config* cfg, int32_t horizon, int32_t checkpoint_stride);

/* Measurement.  dlo_set_kernel_timing(on != 0) makes the handle bracket every launch of its three big kernels with a
 * CUDA event pair on the launching stream (and clears what was recorded before); dlo_get_kernel_timing synchronises and
 * returns, for kernel_class 0 = forward segment kernel, 1 = the same with tape records (replay), 2 = segment adjoint
 * kernel: the launches recorded, the sum of their durations and the env-steps they processed (each pointer host, may be
 * NULL).  dlo_measure_fp32_peak runs an FFMA-chain microbenchmark (8 independent chains per thread, 2048 threads per SM,
 * ~70 ms, best of 3) on the current device and returns the fp32 rate in TFLOP/s: the denominator of the ALU roofline
 * (SURVEY.md section 8(d)); elapsed_ms, n_sm host, may be NULL. */
dlo_status dlo_set_kernel_timing(dlo_sim* sim, int32_t on);
dlo_status dlo_get_kernel_timing(dlo_sim* sim, int32_t kernel_class, int32_t* n_launches, double* total_ms, int64_t* env_steps);
dlo_status dlo_measure_fp32_peak(void* cuda_stream, double* tflops, double* elapsed_ms, int32_t* n_sm);

/* Forward rollout WITHOUT any allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid it).  No handle: one call = dlo_create + scene + dlo_set_state + dlo_rollout_forward
 * (stride 0) + dlo_get_state of a problem small enough that everything the handle would allocate (packed material,
 * kinematic codes, grasp-local coordinates, the working state, per-env flags) fits a device array of
 * DLO_STATIC_SCRATCH_BYTES that is part of the library image (every GPU that loads the library holds it until exit).
 * dlo_static_scratch_bytes(cfg) = the bytes a config needs (0 for an invalid config); a config that needs more is refused
 * with DLO_ERR_UNSUPPORTED (4 MiB holds e.g. 1024 envs x 64 vertices or 256 x 256).  Same kernels and results as the
 * handle path.  The call issues a memset, five kernels and at most one device-to-device copy on `cuda_stream` and
 * returns without synchronising; it calls no cudaMalloc / cudaFree / allocating routine.  (The very first call on a device
 * resolves the array's address with cudaGetSymbolAddress: make that one outside graph capture.)
 *   cfg, mat: as dlo_create (mat: dev pointers, each [B]).  scene: may be NULL when there are no pins, primitives or
 *   grippers; otherwise the arguments of dlo_set_pins / dlo_set_primitives / dlo_set_grippers / dlo_set_actions (actions
 *   [>= horizon][B][G][6]); pointers that the config does not need are ignored.  x0, v0 dev [B][3][N]; kappa_bar0 dev
 *   [B][2][N] or NULL.  Outputs (dev, caller-owned, each may be NULL): x_T, v_T [B][3][N]; env_flags [B] int32, 0 = fine,
 *   else the per-env bits dlo_check_numerics counts (1 non-finite, 2 candidate overflow, 4 guard).
 * The scratch array is SHARED by all calls and keeps the last call's contents: the part a call uses is cleared when the call
 * starts.  Calls whose work overlaps on the GPU (two streams without an event between them, two host threads) race on it;
 * calls on one stream, or ordered by events, are safe. */
#define DLO_STATIC_SCRATCH_BYTES (4u << 20)
typedef struct {
  const uint8_t* pinned;       /* dev [B][N] or NULL */
  const int32_t* prim_types;   /* host [K] */
  const float* prim_params;    /* dev [B][K][10] */
  const float *init_pose, *finger_geom;   /* dev [B][G][6], [B][G][4] */
  const int32_t* grasp_verts;  /* dev [B][G][M] */
  const float* actions;        /* dev [H][B][G][6] */
} dlo_scene;
size_t dlo_static_scratch_bytes(const dlo_config* cfg);
dlo_status dlo_rollout_forward_static(const dlo_config* cfg, const dlo_material* mat, const dlo_scene* scene, const float* x0,
                                      const float* v0, const float* kappa_bar0, int32_t horizon, float* x_T, float* v_T,
                                      int32_t* env_flags, void* cuda_stream);

/* Number of kernel launches issued on this handle since create (bench.py's gpu_launches). */
int64_t dlo_launch_count(const dlo_sim* sim);

const char* dlo_last_error(void);
const char* dlo_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DLO_H_ */
