// pd_probe.cu -- pd_measure_pair_exchange (include/pd.h): measured issue rates behind DESIGN.md 5.1 "why every directed
// bond is evaluated from both ends".  Eq. 2.2 makes the bond term t_ij = t_ji, so one end could
// compute it and hand it to the other end -- over lanes of a warp by a shuffle, over warps by shared memory.  Whether
// that pays is a question of issue rates: what a handed-over double costs against the FP64 instructions it saves.
// Three kernels at the launch shape of pd_measure_fp64_rate (4 CTAs of 256 threads per SM, 8 independent chains per
// thread, no global traffic):
//   0  FP64 fused multiply-adds alone                                       (the figure of pd_measure_fp64_rate)
//   1  64-bit lane shifts alone (__shfl_up_sync of a double = 2 SHFL.32)
//   2  both interleaved, 5 DFMA per shifted double: the trade of the force pass (5 FP64 saved per directed bond
//      for half a shifted double); shows whether the shuffles hide under the FP64 pipe
//   3  8-byte shared-memory store + load of another lane's slot, alone      (the route between warps)
// No step kernel lives here and nothing on the step path calls into this file.
#include <algorithm>

#include "../pd_internal.cuh"

namespace {

constexpr int THREADS = 256, CHAINS = 8, ITERS = 2048;

static __device__ double g_sink[1];   // never written in practice: keeps the chains alive

template <int MODE>
__global__ void __launch_bounds__(THREADS) k_probe(int iters, double a, double b, double magic) {
  __shared__ double sm[THREADS * 2];
  double x[CHAINS];
#pragma unroll
  for (int k = 0; k < CHAINS; ++k) x[k] = (double)(threadIdx.x + k) * 1e-3;
  const int other = (threadIdx.x & ~31) | ((threadIdx.x + 1) & 31);   // the next lane's slot
  for (int it = 0; it < iters; ++it) {
    if constexpr (MODE == 0) {
#pragma unroll
      for (int u = 0; u < 5; ++u)
#pragma unroll
        for (int k = 0; k < CHAINS; ++k) x[k] = fma(x[k], a, b);
    } else if constexpr (MODE == 1) {
#pragma unroll
      for (int k = 0; k < CHAINS; ++k) x[k] = __shfl_up_sync(0xffffffffu, x[k], 1 + (k & 1));
    } else if constexpr (MODE == 2) {
#pragma unroll
      for (int k = 0; k < CHAINS; ++k) {
        x[k] = __shfl_up_sync(0xffffffffu, x[k], 1 + (k & 1));
#pragma unroll
        for (int u = 0; u < 5; ++u) x[k] = fma(x[k], a, b);
      }
    } else {
#pragma unroll
      for (int k = 0; k < CHAINS; k += 2) {
        sm[threadIdx.x] = x[k];
        sm[THREADS + threadIdx.x] = x[k + 1];
        __syncwarp();
        x[k] = sm[other];
        x[k + 1] = sm[THREADS + other];
        __syncwarp();
      }
    }
  }
  double sum = 0.0;
#pragma unroll
  for (int k = 0; k < CHAINS; ++k) sum += x[k];
  if (sum == magic) g_sink[0] = sum;
}

template <int MODE>
int run(int reps, cudaStream_t st, int blocks, double *best_ms) {
  cudaEvent_t e0, e1;
  PD_CUDA(cudaEventCreate(&e0));
  PD_CUDA(cudaEventCreate(&e1));
  float best = 0.f;
  cudaError_t err = cudaSuccess;
  for (int r = 0; r < reps + 1 && err == cudaSuccess; ++r) {   // (the first launch is a warm-up)
    cudaEventRecord(e0, st);
    k_probe<MODE><<<blocks, THREADS, 0, st>>>(ITERS, 0.999999, 1e-9, -12345.678);
    cudaEventRecord(e1, st);
    err = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (err == cudaSuccess) cudaEventElapsedTime(&ms, e0, e1);
    if (r > 0 && ms > 0.f) best = best == 0.f ? ms : std::min(best, ms);
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  if (err != cudaSuccess) return pdi::cuda_fail(err, "pd_measure_pair_exchange");
  PD_CUDA(cudaGetLastError());
  *best_ms = best;
  return PD_OK;
}

}  // namespace

extern "C" int pd_measure_pair_exchange(int reps, void *stream, double per_s[4]) {
  if (reps <= 0 || !per_s) { pdi::set_error("bad argument"); return PD_ERR_ARG; }
  int dev = 0, nsm = 0;
  PD_CUDA(cudaGetDevice(&dev));
  PD_CUDA(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
  const cudaStream_t st = (cudaStream_t)stream;
  const int blocks = nsm * 4;
  const double threads = (double)blocks * THREADS;
  double ms[4] = {0, 0, 0, 0};
  if (int rc = run<0>(reps, st, blocks, &ms[0])) return rc;
  if (int rc = run<1>(reps, st, blocks, &ms[1])) return rc;
  if (int rc = run<2>(reps, st, blocks, &ms[2])) return rc;
  if (int rc = run<3>(reps, st, blocks, &ms[3])) return rc;
  for (int m = 0; m < 4; ++m)
    if (!(ms[m] > 0.0)) { pdi::set_error("pd_measure_pair_exchange: no timing"); return PD_ERR_CUDA; }
  per_s[0] = threads * ITERS * CHAINS * 5.0 / (ms[0] * 1e-3);   // DFMA / s
  per_s[1] = threads * ITERS * CHAINS / (ms[1] * 1e-3);         // shifted doubles / s
  per_s[2] = threads * ITERS * CHAINS / (ms[2] * 1e-3);         // {1 shifted double + 5 DFMA} groups / s
  per_s[3] = threads * ITERS * CHAINS / (ms[3] * 1e-3);         // doubles through shared memory (store + load) / s
  return PD_OK;
}
