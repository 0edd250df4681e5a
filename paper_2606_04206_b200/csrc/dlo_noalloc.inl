// dlo_noalloc.inl — dlo_rollout_forward_static: the forward rollout for callers that cannot allocate (code under CUDA
// graph capture, serving loops, harnesses that forbid cudaMalloc).  Same kernels as dlo_rollout_forward (k_pack_material,
// k_build_kin, k_set_state, k_forward<VPL,false>, k_get_state); what the handle keeps in cudaMalloc'ed buffers - packed
// material, kinematic codes, grasp-local coordinates, the working state block, the per-env flags - lives in ONE file-scope
// device array of DLO_STATIC_SCRATCH_BYTES.  Included by dlo_api.cu (the array, the cudaGetSymbolAddress that turns its
// name into a device address, and every launch that uses it are in that one translation unit).
//
// The array is part of the library image: every GPU that loads the library holds it until the process exits.  All
// calls share it and it keeps the last call's contents: the part a call uses is cleared when the call starts, and two
// calls whose kernels overlap on the GPU (different streams without an event between them, or two host threads) race.
#include <mutex>

static __device__ __align__(256) unsigned char g_static_scratch[DLO_STATIC_SCRATCH_BYTES];

namespace {

constexpr int kMaxDevices = 64;
std::mutex g_static_mutex;
unsigned char* g_static_ptr[kMaxDevices] = {};   // device address of g_static_scratch on each device (null: not asked yet)

// In host code `g_static_scratch` is the host-side shadow of the symbol, not a device address; this asks the runtime for the
// address on the CURRENT device, once per device.
dlo_status static_scratch_address(unsigned char** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return fail(DLO_ERR_CUDA, "no CUDA device: this library has no CPU path"); }
  if (dev < 0 || dev >= kMaxDevices) return fail(DLO_ERR_UNSUPPORTED, "dlo_rollout_forward_static: device ordinal " + std::to_string(dev) + " beyond " + std::to_string(kMaxDevices - 1));
  std::lock_guard<std::mutex> lock(g_static_mutex);
  if (!g_static_ptr[dev]) {
    void* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
    if (e != cudaSuccess || !p) {
      cudaGetLastError();
      return fail(DLO_ERR_CUDA, std::string("cudaGetSymbolAddress(g_static_scratch): ") + cudaGetErrorString(e));
    }
    g_static_ptr[dev] = static_cast<unsigned char*>(p);
  }
  *out = g_static_ptr[dev];
  return DLO_OK;
}

struct StaticLayout { size_t mat, kin, qloc, state, flags, total; };
size_t up256(size_t n) { return (n + 255) / 256 * 256; }
StaticLayout static_layout(const KParams& P) {
  StaticLayout L;
  const size_t B = P.B;
  size_t o = 0;
  L.mat = o;   o += up256(B * MAT_N * sizeof(float));
  L.kin = o;   o += up256(B * P.NS);
  L.qloc = o;  o += up256(B * P.G * P.M * 3 * sizeof(float));
  L.state = o; o += up256(B * STATE_ROWS * P.NS * sizeof(float));
  L.flags = o; o += up256(B * sizeof(int));
  L.total = o;
  return L;
}

}  // namespace

extern "C" {

size_t dlo_static_scratch_bytes(const dlo_config* c) {
  if (validate(c) != DLO_OK) return 0;
  KParams P;
  fill_params(*c, P);
  return static_layout(P).total;
}

dlo_status dlo_rollout_forward_static(const dlo_config* cfg, const dlo_material* mat, const dlo_scene* scene, const float* x0, const float* v0,
                                      const float* kappa_bar0, int32_t horizon, float* x_T, float* v_T, int32_t* env_flags, void* cuda_stream) {
  dlo_status vs = validate(cfg);
  if (vs != DLO_OK) return vs;
  if (!mat || !x0 || !v0) return fail(DLO_ERR_INVALID_ARG, "NULL argument (material, x0 and v0 are required)");
  if (horizon < 0) return fail(DLO_ERR_INVALID_ARG, "horizon < 0");
  const float* mp[MAT_N] = {mat->mass_per_vertex, mat->rest_edge_len, mat->stretch, mat->bend_stiffness, mat->damping,
                            mat->yield_curv, mat->creep_rate, mat->mu_rigid, mat->mu_self};
  for (int k = 0; k < MAT_N; ++k) if (!mp[k]) return fail(DLO_ERR_INVALID_ARG, "a material array is NULL");
  if (cfg->n_primitives > 0 && (!scene || !scene->prim_types || !scene->prim_params)) return fail(DLO_ERR_INVALID_ARG, "n_primitives > 0 needs scene->prim_types and scene->prim_params");
  if (cfg->n_grippers > 0 && (!scene || !scene->init_pose || !scene->finger_geom || !scene->grasp_verts)) return fail(DLO_ERR_INVALID_ARG, "n_grippers > 0 needs scene->init_pose, finger_geom and grasp_verts");
  if (cfg->n_grippers > 0 && horizon > 0 && !scene->actions) return fail(DLO_ERR_INVALID_ARG, "n_grippers > 0 needs scene->actions [horizon][B][G][6]");
  KParams P;
  fill_params(*cfg, P);
  for (int k = 0; k < P.K; ++k) {
    if (scene->prim_types[k] < 0 || scene->prim_types[k] > 3) return fail(DLO_ERR_INVALID_ARG, "unknown primitive type");
    P.prim_type[k] = scene->prim_types[k];
    P.prim_pack |= (unsigned)scene->prim_types[k] << (2 * k);
  }
  const StaticLayout L = static_layout(P);
  if (L.total > (size_t)DLO_STATIC_SCRATCH_BYTES)
    return fail(DLO_ERR_UNSUPPORTED, "dlo_rollout_forward_static: batch " + std::to_string(P.B) + " x n_verts " + std::to_string(P.N) + " needs " + std::to_string(L.total) +
                                         " bytes of scratch, the static array holds " + std::to_string((size_t)DLO_STATIC_SCRATCH_BYTES) + " (DLO_STATIC_SCRATCH_BYTES); use dlo_create / dlo_rollout_forward");
  // launch shape: like dlo_create, without its wave-count model (the problems that fit here are a fraction of one wave)
  dlo_sim shape;   // carries the launch shape to launch_forward; owns nothing
  shape.VPL = vpl_for(P.N);
  const int per_fwd = smem_layout(P, shape.VPL, false), cap = 227 * 1024;
  if (per_fwd > cap) return fail(DLO_ERR_UNSUPPORTED, "shared memory per env exceeds 227 KB for this n_verts");
  shape.wpb_fwd = std::max(1, std::min({4, DLO_FWD_WARPS, cap / 2 / std::max(per_fwd, 1)}));
  shape.smem_fwd = per_fwd * shape.wpb_fwd;
  unsigned char* base = nullptr;
  dlo_status as = static_scratch_address(&base);
  if (as != DLO_OK) return as;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  float* d_mat = reinterpret_cast<float*>(base + L.mat);
  uint8_t* d_kin = base + L.kin;
  float* d_qloc = reinterpret_cast<float*>(base + L.qloc);
  float* d_state = reinterpret_cast<float*>(base + L.state);
  int* d_flags = reinterpret_cast<int*>(base + L.flags);
  // the last call's contents are still there: everything this call uses starts at zero
  CU(cudaMemsetAsync(base, 0, L.total, st));
  MatArgs ma;
  for (int k = 0; k < MAT_N; ++k) ma.a[k] = mp[k];
  k_pack_material<<<(P.B + 127) / 128, 128, 0, st>>>(P.B, ma, d_mat);
  k_build_kin<<<(P.B + 127) / 128, 128, 0, st>>>(P.B, P.N, P.NS, P.G, P.M, scene ? scene->pinned : nullptr, P.G > 0 ? scene->grasp_verts : nullptr, nullptr, d_kin);
  SetupArgs A;
  A.B = P.B; A.N = P.N; A.E = P.E; A.NS = P.NS; A.ring = P.ring; A.G = P.G; A.M = P.M; A.kappa_from_x0 = cfg->kappa_bar_from_x0;
  A.x0 = x0; A.v0 = v0; A.kb0 = kappa_bar0; A.pose0 = P.G > 0 ? scene->init_pose : nullptr; A.grasp_verts = P.G > 0 ? scene->grasp_verts : nullptr;
  A.state = d_state; A.qloc = d_qloc; A.cuts = nullptr;
  k_set_state<<<(P.B + 63) / 64, 64, 0, st>>>(A);
  CU(cudaGetLastError());
  P.mat = d_mat; P.kin = d_kin; P.qloc = d_qloc; P.state = d_state; P.flags = d_flags;
  P.pose0 = P.G > 0 ? scene->init_pose : nullptr; P.finger = P.G > 0 ? scene->finger_geom : nullptr; P.actions = P.G > 0 ? scene->actions : nullptr;
  P.prim = P.K > 0 ? scene->prim_params : nullptr;
  P.t_base = 0;
  if (horizon > 0) CU(launch_forward(&shape, P, 0, horizon, 0, false, st));
  if (x_T || v_T) {
    const size_t n = (size_t)P.B * STATE_ROWS * P.N;
    k_get_state<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(P.B, P.N, P.NS, d_state, x_T, v_T, nullptr, nullptr, nullptr);
    CU(cudaGetLastError());
  }
  if (env_flags) CU(cudaMemcpyAsync(env_flags, d_flags, (size_t)P.B * sizeof(int), cudaMemcpyDeviceToDevice, st));
  return DLO_OK;
}

}  // extern "C"
