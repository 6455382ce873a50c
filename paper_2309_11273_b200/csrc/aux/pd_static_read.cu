// pd_static_read.cu -- pd_get_u_static (include/pd.h): the read-back of the displacement u^n of Eq. 2.11
// (`U` of App. A/B) for callers that may not allocate device memory (code under
// CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).
//
// pd_get_u gathers u^n from the internal node order and component order into user order in a scratch buffer that it
// allocates and frees on every call, and copies that buffer to the caller.  Here the scratch is the file-scope device
// array g_scratch below: PD_STATIC_MAX_DOUBLES doubles = 8 MiB, held by every GPU that loads libpd.so until the process
// exits.  The entry point allocates nothing: no cudaMalloc / cudaMallocAsync / cudaFree, no pd_runtime callback, no
// library routine that allocates; it launches one kernel and one copy on the handle's stream and synchronises with it.
//
// Every call shares g_scratch.  The kernel overwrites the first dim*n doubles (each user node exactly once: perm is a
// bijection of the non-phantom nodes onto 0..n-1), the copy reads exactly those, so nothing needs clearing and what an
// earlier call left behind is never read.  Two calls that OVERLAP on the GPU (two handles on different streams, two
// host threads) race on the array: serialise them.
//
// A translation unit of its own: no step kernel lives here and nothing on the step path calls into this file.
#include <mutex>

#include "../pd_internal.cuh"

namespace {

constexpr int TPB = 256;
constexpr int MAX_DEVICES = 64;

static __device__ __align__(256) double g_scratch[PD_STATIC_MAX_DOUBLES];

// In host code `g_scratch` is a host-side stand-in, not a device address: the kernel gets the address that
// cudaGetSymbolAddress returns for the CURRENT device, looked up once per device.
std::mutex g_mu;
double *g_scratch_dev[MAX_DEVICES] = {};

int scratch_address(double **out) {
  int dev = -1;
  PD_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= MAX_DEVICES) { pdi::set_error("pd_get_u_static: device ordinal out of range"); return PD_ERR_CUDA; }
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_scratch_dev[dev]) {
    void *p = nullptr;
    PD_CUDA(cudaGetSymbolAddress(&p, g_scratch));
    if (!p) { pdi::set_error("pd_get_u_static: cudaGetSymbolAddress returned a null address"); return PD_ERR_CUDA; }
    g_scratch_dev[dev] = (double *)p;
  }
  *out = g_scratch_dev[dev];
  return PD_OK;
}

struct Ax3 { int a[3]; };

// final order -> user AoS (the variant of k_gather_field of pd_api.cu that writes the static scratch).  u^n lives in
// the {u_0, u_1} / u_2 arrays of the uniform lattice layout (uxy, uz) or in the u half of the position pairs of the
// neighbour-record buffer nb (pd_internal.cuh "Data layout").
__global__ void __launch_bounds__(TPB) k_gather_u_static(int64_t npad, int dim, Ax3 ax, const int32_t *__restrict__ perm,
                                                         const double2 *__restrict__ uxy, const double *__restrict__ uz,
                                                         const double2 *__restrict__ nb, bool lattice, double *__restrict__ dst) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= npad) return;
  const int32_t uidx = perm[i];
  if (uidx < 0) return;   // phantom
  for (int k = 0; k < dim; ++k) {
    double val;
    if (uxy) val = k == 0 ? uxy[i].x : (k == 1 ? uxy[i].y : uz[i]);
    else val = nb[pd_pair_index(lattice, npad, i, k)].y;
    dst[(int64_t)dim * uidx + ax.a[k]] = val;
  }
}

}  // namespace

extern "C" int pd_get_u_static(pd_sim *s, double *dst) {
  if (!s || !dst) { pdi::set_error("null argument"); return PD_ERR_ARG; }
  const int64_t count = (int64_t)s->dim * s->n;
  if (count > (int64_t)PD_STATIC_MAX_DOUBLES) {
    pdi::set_error("pd_get_u_static: dim*n = " + std::to_string(count) + " doubles exceed the static scratch of " +
                   std::to_string((long long)PD_STATIC_MAX_DOUBLES) + " doubles (PD_STATIC_MAX_DOUBLES); use pd_get_u");
    return PD_ERR_LIMIT;
  }
  double *scratch = nullptr;
  if (int rc = scratch_address(&scratch)) return rc;
  const bool ulat = s->lat.on && s->lat.uniform;
  const unsigned blocks = (unsigned)((s->npad + TPB - 1) / TPB);
  k_gather_u_static<<<blocks, TPB, 0, s->stream>>>(s->npad, s->dim, Ax3{{s->ax[0], s->ax[1], s->ax[2]}}, s->perm,
                                                   ulat ? s->lat.uxy[s->cur] : nullptr, ulat ? s->lat.uz[s->cur] : nullptr,
                                                   ulat ? nullptr : s->nb[s->cur], s->lat.on, scratch);
  PD_CUDA(cudaGetLastError());
  PD_CUDA(cudaMemcpyAsync(dst, scratch, sizeof(double) * (size_t)count, cudaMemcpyDefault, s->stream));
  PD_CUDA(cudaStreamSynchronize(s->stream));
  return PD_OK;
}
