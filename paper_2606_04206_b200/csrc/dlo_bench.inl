// dlo_bench.inl — measurement helpers behind the C-ABI (included by dlo_api.cu): per-kernel timing of a handle's launches
// and an FFMA-chain microbenchmark that measures the fp32 (non-tensor) peak of the current device, the denominator of
// the ALU roofline in bench.py ("to be confirmed with an FFMA-chain microbenchmark on the box").

namespace dlo {
// 8 independent FFMA chains per thread, `iters` rounds of 8 unrolled steps each: 2 * 8 * 8 * iters flop per thread.  The
// result is stored only if it is NaN (never, but the compiler cannot know), so nothing is optimised away and nothing is written.
__global__ void __launch_bounds__(256, 8) k_fma_chain(int iters, float a, float b, float* sink) {
  float x[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) x[k] = (float)(threadIdx.x + k) * 1.0e-3f;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
#pragma unroll
      for (int k = 0; k < 8; ++k) x[k] = fmaf(x[k], a, b);
    }
  }
  float acc = 0.0f;
#pragma unroll
  for (int k = 0; k < 8; ++k) acc += x[k];
  if (acc != acc) sink[blockIdx.x * blockDim.x + threadIdx.x] = acc;
}
}  // namespace dlo

extern "C" {

dlo_status dlo_measure_fp32_peak(void* cuda_stream, double* tflops, double* elapsed_ms, int32_t* n_sm_out) {
  if (!tflops) return fail(DLO_ERR_INVALID_ARG, "NULL argument");
  int dev = 0, n_sm = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return fail(DLO_ERR_CUDA, "no CUDA device: this library has no CPU path"); }
  CU(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  float* sink = nullptr;
  const int threads = 256, blocks = n_sm * 8;   // 2048 resident threads per SM, one wave
  CU(cudaMalloc((void**)&sink, (size_t)blocks * threads * sizeof(float)));
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int iters = 1 << 17;   // 2 * 64 * 2^17 = 1.7e7 flop per thread: ~70 ms at 74 TFLOP/s
  k_fma_chain<<<blocks, threads, 0, st>>>(1 << 10, 0.999f, 1.0e-3f, sink);   // warm-up
  double best = 0.0, best_ms = 0.0;
  for (int rep = 0; rep < 3; ++rep) {
    cudaEventRecord(e0, st);
    k_fma_chain<<<blocks, threads, 0, st>>>(iters, 0.999f, 1.0e-3f, sink);
    cudaEventRecord(e1, st);
    cudaError_t e = cudaEventSynchronize(e1);
    if (e != cudaSuccess) { cudaFree(sink); cudaEventDestroy(e0); cudaEventDestroy(e1); return fail(DLO_ERR_CUDA, cudaGetErrorString(e)); }
    float ms = 0.0f;
    cudaEventElapsedTime(&ms, e0, e1);
    const double tf = 2.0 * 64.0 * (double)iters * (double)blocks * threads / (ms * 1e-3) / 1e12;
    if (tf > best) { best = tf; best_ms = ms; }
  }
  cudaFree(sink); cudaEventDestroy(e0); cudaEventDestroy(e1);
  *tflops = best;
  if (elapsed_ms) *elapsed_ms = best_ms;
  if (n_sm_out) *n_sm_out = n_sm;
  return DLO_OK;
}

dlo_status dlo_set_kernel_timing(dlo_sim* s, int32_t on) {
  ENTER(s);
  CU(cudaStreamSynchronize(s->stream));
  if (s->aux) CU(cudaStreamSynchronize(s->aux));
  for (int c = 0; c < 3; ++c) { for (cudaEvent_t e : s->tev[c]) cudaEventDestroy(e); s->tev[c].clear(); s->tunits[c].clear(); }
  s->timing = on != 0;
  return DLO_OK;
}

dlo_status dlo_get_kernel_timing(dlo_sim* s, int32_t kernel_class, int32_t* n_launches, double* total_ms, int64_t* env_steps) {
  ENTER(s);
  if (kernel_class < 0 || kernel_class > 2) return fail(DLO_ERR_INVALID_ARG, "kernel_class out of [0,2]");
  CU(cudaStreamSynchronize(s->stream));
  if (s->aux) CU(cudaStreamSynchronize(s->aux));
  double tot = 0.0; int64_t units = 0;
  const auto& v = s->tev[kernel_class];
  for (size_t k = 0; k + 1 < v.size(); k += 2) {
    float ms = 0.0f;
    CU(cudaEventElapsedTime(&ms, v[k], v[k + 1]));
    tot += ms; units += s->tunits[kernel_class][k / 2];
  }
  if (n_launches) *n_launches = (int32_t)(v.size() / 2);
  if (total_ms) *total_ms = tot;
  if (env_steps) *env_steps = units;
  return DLO_OK;
}

}  // extern "C"
