// pd_api.cu -- the C-ABI entry points of include/pd.h: argument checks, staging of caller data,
// the step loop, and read-back in user node order.  No numerics of the method live here except
// the three mode constants A, K, G (Eqs. 1.8, 1.15, 1.16).
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>

#include "pd_internal.cuh"

namespace {
thread_local std::string g_err;
constexpr int TPB = 256;
inline unsigned nblk(int64_t n) { return (unsigned)((n + TPB - 1) / TPB); }

// user AoS (dim*n) -> final order; dst is either the u half of the position pairs of a neighbour-record
// buffer (nb != NULL) or SoA arrays
struct Ax { int a[3]; };
// where a vector field lives: the u half of the position pairs of a neighbour-record buffer (nb), the
// {u_0, u_1} / u_2 arrays of the uniform lattice layout (uxy, uz), or SoA arrays (d)
struct FieldView {
  double2 *nb; bool lattice;
  double2 *uxy; double *uz;
  double *d[3];
};
__device__ __forceinline__ double &field_ref(const FieldView &f, int64_t npad, int64_t i, int k) {
  if (f.nb) return f.nb[pd_pair_index(f.lattice, npad, i, k)].y;
  if (f.uxy) return k == 0 ? f.uxy[i].x : (k == 1 ? f.uxy[i].y : f.uz[i]);
  return f.d[k][i];
}
__global__ void k_scatter_field(int64_t npad, int dim, Ax ax, const int32_t *__restrict__ perm, const double *__restrict__ src,
                                const uint8_t *__restrict__ flags, bool clamp_zero, FieldView f) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= npad) return;
  int32_t uidx = perm[i];
  unsigned fl = flags[i];
  for (int k = 0; k < dim; ++k) {
    double val = (src && uidx >= 0) ? src[(int64_t)dim * uidx + ax.a[k]] : 0.0;
    if (clamp_zero && (fl & (1u << k))) val = 0.0;
    field_ref(f, npad, i, k) = val;
  }
}

// final order -> user AoS; source is the u half of a neighbour-record buffer or SoA arrays
__global__ void k_gather_field(int64_t npad, int dim, Ax ax, const int32_t *__restrict__ perm, FieldView f, double *dst) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= npad) return;
  int32_t uidx = perm[i];
  if (uidx < 0) return;
  for (int k = 0; k < dim; ++k) dst[(int64_t)dim * uidx + ax.a[k]] = field_ref(f, npad, i, k);
}

// halo pack / unpack of the slab decomposition: rows idx[q] (user indices) of u <-> a dense (count x dim) AoS buffer
__global__ void k_pack_u(int64_t count, int dim, Ax ax, int64_t npad, const int32_t *__restrict__ idx, const int32_t *__restrict__ iperm,
                         FieldView u, double *buf, bool unpack) {
  int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= count) return;
  const int64_t i = iperm[idx[q]];
  for (int k = 0; k < dim; ++k) {
    if (unpack) field_ref(u, npad, i, k) = buf[q * dim + ax.a[k]];
    else buf[q * dim + ax.a[k]] = field_ref(u, npad, i, k);
  }
}

FieldView view_u(pd_sim *s, int buf) {
  FieldView f{};
  if (s->lat.on && s->lat.uniform) { f.uxy = s->lat.uxy[buf]; f.uz = s->lat.uz[buf]; }
  else { f.nb = s->nb[buf]; f.lattice = s->lat.on; }
  return f;
}
FieldView view_soa(double *const *d) {
  FieldView f{};
  for (int k = 0; k < 3; ++k) f.d[k] = d[k];
  return f;
}

// scalar per node
__global__ void k_gather_scalar(int64_t npad, const int32_t *__restrict__ perm, const double *__restrict__ src, double *dst) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= npad) return;
  int32_t uidx = perm[i];
  if (uidx < 0) return;
  dst[uidx] = src[i];
}


// ---- adaptive dynamic relaxation (pd_adr_step, Underwood 1983 / Kilic & Madenci 2010) ----
// The step kernels run with rho = 1, dt = 1 and v zeroed before the force pass, so v holds the total force density
// R^n = f(U^n) + g b on return.  Then (pseudo time step 1, Lambda = lam I):
//   1K_ii = -(R_i^n - R_i^{n-1}) / (lam Ud_i^{n-1/2}),   c^n = 2 sqrt((U . 1K U) / (U . U))   over the free dofs
//   Ud^{n+1/2} = ((2 - c^n) Ud^{n-1/2} + 2 R^n / lam) / (2 + c^n)   (n = 0: R^0 / (2 lam));   U^{n+1} = U^n + Ud^{n+1/2}
__global__ void k_adr_reduce(int64_t npad, int dim, const int32_t *__restrict__ perm, const uint8_t *__restrict__ flags, FieldView u,
                             FieldView r, FieldView rprev, FieldView ud, double lam, double *scal) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  double num = 0.0, den = 0.0;
  if (i < npad && perm[i] >= 0) {
    const unsigned fl = flags[i];
    for (int k = 0; k < dim; ++k) {
      if (fl & ((1u << k) | (8u << k))) continue;   // clamped / prescribed dofs are not free
      const double U = field_ref(u, npad, i, k), d = field_ref(ud, npad, i, k);
      const double k1 = d != 0.0 ? -(field_ref(r, npad, i, k) - field_ref(rprev, npad, i, k)) / (lam * d) : 0.0;
      num += U * k1 * U;
      den += U * U;
    }
  }
  for (int o = 16; o > 0; o >>= 1) {
    num += __shfl_xor_sync(0xffffffffu, num, o);
    den += __shfl_xor_sync(0xffffffffu, den, o);
  }
  if ((threadIdx.x & 31) == 0 && (num != 0.0 || den != 0.0)) { atomicAdd(&scal[0], num); atomicAdd(&scal[1], den); }
}
__global__ void k_adr_update(int64_t npad, int dim, const int32_t *__restrict__ perm, const uint8_t *__restrict__ flags, FieldView u,
                             FieldView unext, FieldView r, FieldView rprev, FieldView ud, FieldView bval, double lam, int first,
                             const double *__restrict__ scal) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= npad || perm[i] < 0) return;
  double c = 0.0;
  if (!first && scal[1] > 0.0 && scal[0] / scal[1] > 0.0) c = 2.0 * sqrt(scal[0] / scal[1]);
  const unsigned fl = flags[i];
  for (int k = 0; k < dim; ++k) {
    const double R = field_ref(r, npad, i, k);
    double d = first ? 0.5 * R / lam : ((2.0 - c) * field_ref(ud, npad, i, k) + 2.0 * R / lam) / (2.0 + c);
    if (fl & (1u << k)) d = 0.0;                                   // clamped
    else if (fl & (8u << k)) d = field_ref(bval, npad, i, k);      // prescribed displacement increment per iteration
    field_ref(unext, npad, i, k) = field_ref(u, npad, i, k) + d;
    field_ref(ud, npad, i, k) = d;
    field_ref(rprev, npad, i, k) = R;
  }
}

struct DevTmp {  // RAII temp allocation through the sim's allocator
  pd_sim *s;
  void *p;
  DevTmp(pd_sim *s_, size_t bytes) : s(s_), p(pdi::dev_alloc(s_, bytes ? bytes : 1)) {}
  ~DevTmp() {
    if (p) {
      cudaStreamSynchronize(s->stream);
      pdi::dev_free(s, p);
    }
  }
};

// copy caller memory (host or device) into a fresh device buffer
int stage(pd_sim *s, const void *src, size_t bytes, void **out) {
  *out = nullptr;
  if (!src || bytes == 0) return PD_OK;
  void *p = pdi::dev_alloc(s, bytes);
  if (!p) { pdi::set_error("device allocation failed while staging inputs"); return PD_ERR_ALLOC; }
  cudaError_t e = cudaMemcpyAsync(p, src, bytes, cudaMemcpyDefault, s->stream);
  if (e != cudaSuccess) { pdi::dev_free(s, p); return pdi::cuda_fail(e, "cudaMemcpyAsync(stage)"); }
  *out = p;
  return PD_OK;
}

int flush_break(pd_sim *s) {  // deferred step 5: decide rho^{n} from u^{n} before anything reads it
  if (s->fracture && s->break_pending) {
    const int rc = pdi::launch_dilatation(s, nullptr, true);
    if (rc) return rc;
    s->break_pending = false;
  }
  return PD_OK;
}

int copy_out(pd_sim *s, void *dst, const void *src_dev, size_t bytes) {
  PD_CUDA(cudaMemcpyAsync(dst, src_dev, bytes, cudaMemcpyDefault, s->stream));
  PD_CUDA(cudaStreamSynchronize(s->stream));
  return PD_OK;
}

int get_field(pd_sim *s, double *dst, bool velocity) {
  if (!s || !dst) { pdi::set_error("null argument"); return PD_ERR_ARG; }
  DevTmp tmp(s, sizeof(double) * s->dim * s->n);
  if (!tmp.p) { pdi::set_error("device allocation failed"); return PD_ERR_ALLOC; }
  k_gather_field<<<nblk(s->npad), TPB, 0, s->stream>>>(s->npad, s->dim, Ax{{s->ax[0], s->ax[1], s->ax[2]}}, s->perm,
                                                       velocity ? view_soa(s->v) : view_u(s, s->cur), (double *)tmp.p);
  PD_CUDA(cudaGetLastError());
  return copy_out(s, dst, tmp.p, sizeof(double) * s->dim * s->n);
}
}  // namespace

namespace pdi {
void set_error(const std::string &msg) { g_err = msg; }
int cuda_fail(cudaError_t e, const char *what) {
  g_err = std::string("CUDA error: ") + cudaGetErrorString(e) + " in " + what;
  return PD_ERR_CUDA;
}
void *dev_alloc(pd_sim *s, size_t bytes) {
  void *p = nullptr;
  if (s->own_alloc) {
    if (cudaMallocAsync(&p, bytes, s->stream) != cudaSuccess) { cudaGetLastError(); return nullptr; }
  } else {
    p = s->rt.alloc(bytes, s->rt.ctx);
    if (!p) return nullptr;
  }
  s->allocs.emplace_back(p, bytes);
  s->bytes_held += bytes;
  return p;
}
void dev_free(pd_sim *s, void *p) {
  if (!p) return;
  for (size_t q = 0; q < s->allocs.size(); ++q)
    if (s->allocs[q].first == p) {
      s->bytes_held -= s->allocs[q].second;
      s->allocs.erase(s->allocs.begin() + q);
      break;
    }
  if (s->own_alloc) cudaFreeAsync(p, s->stream); else s->rt.free(p, s->rt.ctx);
}
void dev_free_all(pd_sim *s) {
  cudaStreamSynchronize(s->stream);
  while (!s->allocs.empty()) dev_free(s, s->allocs.back().first);
}
}  // namespace pdi

extern "C" {

const char *pd_last_error(void) { return g_err.c_str(); }
// 8 independent DFMA chains per thread, 4096 x 8 x 4 fused multiply-adds each
__global__ void __launch_bounds__(256) k_fp64_rate(double *out, int iters, double a, double b) {
  double x[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) x[k] = (double)(threadIdx.x + k) * 1e-3;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 4; ++u)
#pragma unroll
      for (int k = 0; k < 8; ++k) x[k] = fma(x[k], a, b);
  }
  double sum = 0.0;
#pragma unroll
  for (int k = 0; k < 8; ++k) sum += x[k];
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = sum;
}

int pd_measure_fp64_rate(int reps, void *stream, double *fma_per_s) {
  if (reps <= 0 || !fma_per_s) { pdi::set_error("bad argument"); return PD_ERR_ARG; }
  int dev = 0, nsm = 0;
  PD_CUDA(cudaGetDevice(&dev));
  PD_CUDA(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
  const cudaStream_t st = (cudaStream_t)stream;
  const int blocks = nsm * 4, threads = 256, iters = 4096;
  double *out = nullptr;
  if (cudaMalloc(&out, sizeof(double) * blocks * threads) != cudaSuccess) { cudaGetLastError(); pdi::set_error("device allocation failed"); return PD_ERR_ALLOC; }
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  double best = 0.0;
  for (int r = 0; r < reps + 1; ++r) {   // (the first launch is a warm-up)
    cudaEventRecord(e0, st);
    k_fp64_rate<<<blocks, threads, 0, st>>>(out, iters, 0.999999, 1e-9);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) break;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (r > 0 && ms > 0.f) best = std::max(best, (double)blocks * threads * iters * 32.0 / (ms * 1e-3));
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(out);
  PD_CUDA(cudaGetLastError());
  *fma_per_s = best;
  return PD_OK;
}

const char *pd_version(void) {
  return "pd-b200 0.6 (sm_100a, FP64; layouts: uniform lattice [compiled-in 122-offset (3-D) and 28-offset (2-D) stencils over "
         "TMA-staged planes; any stencil: table-driven], dense lattice with per-bond geometry, windowed sliced ELL)";
}

int pd_create(pd_sim **out, int64_t n, const double *coords, const double *volumes, double horizon,
              const pd_material *mat, const pd_boundary *bc, const pd_runtime *rt) {
  if (out) *out = nullptr;
  if (!out || !coords || !volumes || !mat) { pdi::set_error("null argument"); return PD_ERR_ARG; }
  if (n <= 0 || n >= (1ll << 31) - 64) { pdi::set_error("n must be in (0, 2^31)"); return PD_ERR_ARG; }
  if (!(mat->dim == 2 || mat->dim == 3) || (mat->dim == 3) != (mat->mode == PD_MODE_3D) || mat->mode < 0 ||
      mat->mode > 2) { pdi::set_error("dim/mode mismatch"); return PD_ERR_ARG; }
  if (!(mat->E > 0) || !(mat->nu > -1.0) || !(mat->nu < 0.5) || !(mat->rho > 0) || !(mat->dt > 0) ||
      !(horizon > 0) || !std::isfinite(horizon) || !std::isfinite(mat->E) || !std::isfinite(mat->rho) ||
      !std::isfinite(mat->dt)) { pdi::set_error("E, rho, dt, horizon must be > 0 and nu in (-1, 0.5)"); return PD_ERR_ARG; }
  if (mat->extension != PD_EXT_LINEARIZED && mat->extension != PD_EXT_GEOMETRIC) { pdi::set_error("unknown extension"); return PD_ERR_ARG; }
  if (bc && bc->n_precut < 0) { pdi::set_error("n_precut < 0"); return PD_ERR_ARG; }
  if (bc && bc->n_precut > 0 && !bc->precut) { pdi::set_error("precut is NULL"); return PD_ERR_ARG; }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    pdi::set_error("no CUDA device: this library has no CPU path");
    return PD_ERR_CUDA;
  }
  pd_sim *s = new (std::nothrow) pd_sim();
  if (!s) { pdi::set_error("host allocation failed"); return PD_ERR_ALLOC; }
  s->n = n; s->dim = mat->dim; s->mode = mat->mode; s->horizon = horizon;
  s->rho = mat->rho; s->dt = mat->dt; s->ramp_time = mat->ramp_time;
  s->geom = mat->extension == PD_EXT_GEOMETRIC;
  s->fracture = (mat->s_c > 0.0) && std::isfinite(mat->s_c);
  s->s_c = s->fracture ? mat->s_c : 0.0;
  if (rt && rt->alloc && rt->free) { s->rt = *rt; s->own_alloc = false; }
  s->stream = rt ? (cudaStream_t)rt->stream : (cudaStream_t)0;
  {  // mode constants
    const double nu = mat->nu, kappa = mat->E / (3.0 * (1.0 - 2.0 * nu)), mu = mat->E / (2.0 * (1.0 + nu));
    if (s->mode == PD_MODE_3D) { s->A = 3.0; s->K = 3.0 * kappa; s->G = 15.0 * mu; }
    else if (s->mode == PD_MODE_PLANE_STRESS) {
      s->A = 2.0 * (1.0 - 2.0 * nu) / (1.0 - nu);
      s->K = 2.0 * kappa * (1.0 - 2.0 * nu) / (1.0 - nu) -
             (2.0 / 3.0) * mu * ((1.0 + nu) * (1.0 - 3.0 * nu)) / ((1.0 - nu) * (1.0 - 2.0 * nu));
      s->G = 8.0 * mu;
    } else { s->A = 2.0; s->K = 2.0 * kappa - (2.0 / 3.0) * mu; s->G = 8.0 * mu; }
    s->c1 = s->K - s->G / 3.0;
  }
  int rc = PD_OK;
  void *d_coords = nullptr, *d_vol = nullptr, *d_flags = nullptr, *d_precut = nullptr, *d_u0 = nullptr, *d_v0 = nullptr,
       *d_val = nullptr;
  const int dim = s->dim;
  auto fail = [&](int code) { pdi::lat_free_cache(s); pdi::dev_free_all(s); delete s; return code; };
  if ((rc = stage(s, coords, sizeof(double) * dim * n, &d_coords))) return fail(rc);
  if ((rc = stage(s, volumes, sizeof(double) * n, &d_vol))) return fail(rc);
  if (bc) {
    if ((rc = stage(s, bc->flags, (size_t)n, &d_flags))) return fail(rc);
    if ((rc = stage(s, bc->precut, sizeof(int32_t) * 2 * bc->n_precut, &d_precut))) return fail(rc);
    if ((rc = stage(s, bc->u0, sizeof(double) * dim * n, &d_u0))) return fail(rc);
    if ((rc = stage(s, bc->v0, sizeof(double) * dim * n, &d_v0))) return fail(rc);
    if ((rc = stage(s, bc->value, sizeof(double) * dim * n, &d_val))) return fail(rc);
  }
  rc = pdi::build_family(s, (const double *)d_coords, (const double *)d_vol, (const uint8_t *)d_flags,
                         (const int32_t *)d_precut, bc ? bc->n_precut : 0);
  if (rc) return fail(rc);

  // ---- state arrays (u, cth live in the neighbour records built above) ----
  auto alloc_d = [&](double **p) {
    *p = (double *)pdi::dev_alloc(s, sizeof(double) * s->npad);
    if (*p) cudaMemsetAsync(*p, 0, sizeof(double) * s->npad, s->stream);
    return *p != nullptr;
  };
  bool ok = true;
  for (int k = 0; k < dim && ok; ++k) ok = alloc_d(&s->v[k]) && alloc_d(&s->bval[k]);
  ok = ok && alloc_d(&s->phi);
  if (ok) {
    s->stats_dev = (unsigned long long *)pdi::dev_alloc(s, 4 * sizeof(unsigned long long));
    ok = s->stats_dev != nullptr;
  }
  if (!ok) { pdi::set_error("device allocation failed for the state arrays"); return fail(PD_ERR_ALLOC); }
  const Ax axv{{s->ax[0], s->ax[1], s->ax[2]}};
  k_scatter_field<<<nblk(s->npad), TPB, 0, s->stream>>>(s->npad, dim, axv, s->perm, (const double *)d_u0, s->flags, true, view_u(s, 0));
  k_scatter_field<<<nblk(s->npad), TPB, 0, s->stream>>>(s->npad, dim, axv, s->perm, (const double *)d_v0, s->flags, true, view_soa(s->v));
  k_scatter_field<<<nblk(s->npad), TPB, 0, s->stream>>>(s->npad, dim, axv, s->perm, (const double *)d_val, s->flags, false,
                                                         view_soa(s->bval));
  cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
  if (e != cudaSuccess) return fail(pdi::cuda_fail(e, "pd_create state initialisation"));
  for (void *p : {d_coords, d_vol, d_flags, d_precut, d_u0, d_v0, d_val}) pdi::dev_free(s, p);
  s->cur = 0; s->step = 0; s->break_pending = false;  // u^0 is not break-checked (reading C-5)
  // graphs pay where the step is launch-bound (the 2-D configs: 10-20 us of kernel time per step); with more than
  // 2e7 directed bonds a launch is 0.1 ms and longer and the plain launches cost nothing
  s->use_graph = s->Z < 20000000;
  if (const char *env = getenv("PD_GRAPH")) s->use_graph = atoi(env) != 0;
  if (const char *env = getenv("PD_GRAPH_STEPS")) s->graph_len = std::max(2, std::min(atoi(env) & ~1, 256));
  *out = s;
  return PD_OK;
}

// one explicit step by plain launches: rows a1, a2 (+ deferred a5), then a1, a3, a4
static int step_once(pd_sim *s) {
  int rc = pdi::launch_dilatation(s, nullptr, s->break_pending);
  if (rc) return rc;
  if ((rc = pdi::launch_force_update(s))) return rc;
  s->cur ^= 1;
  s->step += 1;
  s->break_pending = s->fracture;
  s->launches += 2;
  return PD_OK;
}

// The step loop without per-step host work: 2 g steps (g = 1 or PD_GRAPH_STEPS / 2) are captured once into a CUDA
// graph and replayed.  A graph bakes its kernel arguments, so it is only used in the STEADY state -- buffer parity
// cur = 0 at its start, the deferred break test pending (or no fracture), the load ramp g(t) finished -- and every
// other step takes plain launches.  Capture runs on a private stream (the caller's may be the legacy default
// stream, which cannot be captured); replay is enqueued on the caller's stream.
static bool graph_steady(const pd_sim *s) {
  return s->cur == 0 && s->break_pending == s->fracture &&
         (s->ramp_time <= 0.0 || (double)s->step * s->dt >= s->ramp_time);
}
static int graph_build(pd_sim *s, int which, int nsteps) {
  if (!s->cap_stream && cudaStreamCreateWithFlags(&s->cap_stream, cudaStreamNonBlocking) != cudaSuccess) {
    cudaGetLastError();
    return PD_ERR_CUDA;
  }
  const cudaStream_t user = s->stream;
  const int cur0 = s->cur;
  const int64_t step0 = s->step, launches0 = s->launches;
  s->stream = s->cap_stream;
  cudaGraph_t g = nullptr;
  int rc = PD_OK;
  if (cudaStreamBeginCapture(s->cap_stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) rc = PD_ERR_CUDA;
  for (int it = 0; it < nsteps && rc == PD_OK; ++it) rc = step_once(s);
  if (cudaStreamEndCapture(s->cap_stream, &g) != cudaSuccess) rc = rc ? rc : PD_ERR_CUDA;
  s->stream = user;
  const int64_t captured = s->launches - launches0;
  s->cur = cur0; s->step = step0; s->launches = launches0;   // nothing ran
  if (rc == PD_OK && cudaGraphInstantiate(&s->graph[which], g, 0) != cudaSuccess) rc = PD_ERR_CUDA;
  if (g) cudaGraphDestroy(g);
  if (rc != PD_OK) { cudaGetLastError(); s->graph[which] = nullptr; }
  else { s->graph_steps[which] = nsteps; s->graph_launches[which] = captured; }
  return rc;
}

int pd_step(pd_sim *s, int64_t nsteps) {
  if (!s || nsteps < 0) { pdi::set_error("bad argument"); return PD_ERR_ARG; }
  int64_t left = nsteps;
  while (left > 0) {
    if (s->use_graph && left >= 2 && graph_steady(s)) {
      // which graph: the long one when enough steps are left
      const int big = s->graph_len;
      const int which = (left >= big && big > 2) ? 1 : 0;
      const int len = which ? big : 2;
      if (!s->graph[which] && !s->graph_failed) {
        // the first steps run by plain launches (they also prepare the launch arguments); a graph is only built
        // when enough steps are left to pay for its instantiation
        if (s->step < 4 || left < 64) {
          if (int rc = step_once(s)) return rc;
          --left;
          continue;
        }
        if (graph_build(s, which, len) != PD_OK) s->graph_failed = true;
      }
      if (s->graph[which]) {
        PD_CUDA(cudaGraphLaunch(s->graph[which], s->stream));
        s->step += len; s->launches += s->graph_launches[which];   // cur is back at 0 after an even number of steps
        left -= len;
        continue;
      }
    }
    if (int rc = step_once(s)) return rc;
    --left;
  }
  PD_CUDA(cudaGetLastError());
  return PD_OK;
}

int pd_step_timed(pd_sim *s, int64_t nsteps, double ms[2]) {
  if (!s || nsteps < 0 || !ms) { pdi::set_error("bad argument"); return PD_ERR_ARG; }
  ms[0] = ms[1] = 0.0;
  cudaEvent_t ev[3];
  for (auto &e : ev) PD_CUDA(cudaEventCreate(&e));
  int rc = PD_OK;
  for (int64_t it = 0; it < nsteps && rc == PD_OK; ++it) {
    cudaEventRecord(ev[0], s->stream);
    if ((rc = pdi::launch_dilatation(s, nullptr, s->break_pending))) break;
    cudaEventRecord(ev[1], s->stream);
    if ((rc = pdi::launch_force_update(s))) break;
    cudaEventRecord(ev[2], s->stream);
    s->cur ^= 1; s->step += 1; s->break_pending = s->fracture; s->launches += 2;
    cudaError_t e = cudaEventSynchronize(ev[2]);
    if (e != cudaSuccess) { rc = pdi::cuda_fail(e, "pd_step_timed"); break; }
    float a = 0, b = 0;
    cudaEventElapsedTime(&a, ev[0], ev[1]);
    cudaEventElapsedTime(&b, ev[1], ev[2]);
    ms[0] += a; ms[1] += b;
  }
  for (auto &e : ev) cudaEventDestroy(e);
  return rc;
}

int pd_gather_u(pd_sim *s, const int32_t *idx, int64_t count, double *dst) {
  if (!s || count < 0 || (count > 0 && (!idx || !dst))) { pdi::set_error("bad argument"); return PD_ERR_ARG; }
  if (count == 0) return PD_OK;
  k_pack_u<<<nblk(count), TPB, 0, s->stream>>>(count, s->dim, Ax{{s->ax[0], s->ax[1], s->ax[2]}}, s->npad, idx, s->iperm,
                                               view_u(s, s->cur), dst, false);
  PD_CUDA(cudaGetLastError());
  return PD_OK;
}

int pd_scatter_u(pd_sim *s, const int32_t *idx, int64_t count, const double *src) {
  if (!s || count < 0 || (count > 0 && (!idx || !src))) { pdi::set_error("bad argument"); return PD_ERR_ARG; }
  if (count == 0) return PD_OK;
  k_pack_u<<<nblk(count), TPB, 0, s->stream>>>(count, s->dim, Ax{{s->ax[0], s->ax[1], s->ax[2]}}, s->npad, idx, s->iperm,
                                               view_u(s, s->cur), const_cast<double *>(src), true);
  PD_CUDA(cudaGetLastError());
  return PD_OK;
}

int pd_adr_step(pd_sim *s, int64_t niter, double lam) {
  if (!s || niter < 0 || !(lam > 0.0)) { pdi::set_error("bad argument"); return PD_ERR_ARG; }
  if (s->rho != 1.0 || s->dt != 1.0) { pdi::set_error("pd_adr_step needs a handle created with rho = 1 and dt = 1 (pseudo time)"); return PD_ERR_ARG; }
  const int dim = s->dim;
  if (!s->adr_ud[0]) {
    for (int k = 0; k < dim; ++k) {
      s->adr_ud[k] = (double *)pdi::dev_alloc(s, sizeof(double) * s->npad);
      s->adr_rprev[k] = (double *)pdi::dev_alloc(s, sizeof(double) * s->npad);
      if (!s->adr_ud[k] || !s->adr_rprev[k]) { pdi::set_error("device allocation failed"); return PD_ERR_ALLOC; }
      cudaMemsetAsync(s->adr_ud[k], 0, sizeof(double) * s->npad, s->stream);
      cudaMemsetAsync(s->adr_rprev[k], 0, sizeof(double) * s->npad, s->stream);
    }
    s->adr_scal = (double *)pdi::dev_alloc(s, 2 * sizeof(double));
    if (!s->adr_scal) { pdi::set_error("device allocation failed"); return PD_ERR_ALLOC; }
  }
  const FieldView ud = view_soa(s->adr_ud), rprev = view_soa(s->adr_rprev), r = view_soa(s->v), bval = view_soa(s->bval);
  for (int64_t it = 0; it < niter; ++it) {
    int rc = pdi::launch_dilatation(s, nullptr, s->break_pending);
    if (rc) return rc;
    for (int k = 0; k < dim; ++k) cudaMemsetAsync(s->v[k], 0, sizeof(double) * s->npad, s->stream);
    if ((rc = pdi::launch_force_update(s))) return rc;   // v = R^n; the other u buffer is overwritten below
    const int first = s->adr_it == 0;
    const FieldView u = view_u(s, s->cur), unext = view_u(s, s->cur ^ 1);
    if (!first) {
      cudaMemsetAsync(s->adr_scal, 0, 2 * sizeof(double), s->stream);
      k_adr_reduce<<<nblk(s->npad), TPB, 0, s->stream>>>(s->npad, dim, s->perm, s->flags, u, r, rprev, ud, lam, s->adr_scal);
    }
    k_adr_update<<<nblk(s->npad), TPB, 0, s->stream>>>(s->npad, dim, s->perm, s->flags, u, unext, r, rprev, ud, bval, lam, first,
                                                       s->adr_scal);
    s->cur ^= 1; s->step += 1; s->adr_it += 1; s->break_pending = s->fracture; s->launches += 2;
  }
  PD_CUDA(cudaGetLastError());
  return PD_OK;
}

int pd_get_u(pd_sim *s, double *dst) { return s ? get_field(s, dst, false) : PD_ERR_ARG; }
int pd_get_v(pd_sim *s, double *dst) { return s ? get_field(s, dst, true) : PD_ERR_ARG; }

int pd_get_damage(pd_sim *s, double *dst) {
  if (!s || !dst) { pdi::set_error("null argument"); return PD_ERR_ARG; }
  if (int rc = flush_break(s)) return rc;
  if (int rc = pdi::launch_damage(s)) return rc;
  DevTmp tmp(s, sizeof(double) * s->n);
  if (!tmp.p) { pdi::set_error("device allocation failed"); return PD_ERR_ALLOC; }
  k_gather_scalar<<<nblk(s->npad), TPB, 0, s->stream>>>(s->npad, s->perm, s->phi, (double *)tmp.p);
  PD_CUDA(cudaGetLastError());
  return copy_out(s, dst, tmp.p, sizeof(double) * s->n);
}

int pd_get_stats(pd_sim *s, int64_t *nbonds, int64_t *nbroken, double *max_damage, int64_t *n_ge_half, int64_t *step) {
  if (!s) { pdi::set_error("null argument"); return PD_ERR_ARG; }
  if (int rc = flush_break(s)) return rc;
  if (int rc = pdi::launch_damage(s)) return rc;
  unsigned long long h[3];
  PD_CUDA(cudaMemcpyAsync(h, s->stats_dev, sizeof(h), cudaMemcpyDeviceToHost, s->stream));
  PD_CUDA(cudaStreamSynchronize(s->stream));
  if (nbonds) *nbonds = s->Z;
  if (nbroken) *nbroken = (int64_t)h[0];
  if (max_damage) { double d; memcpy(&d, &h[1], 8); *max_damage = d; }
  if (n_ge_half) *n_ge_half = (int64_t)h[2];
  if (step) *step = s->step;
  return PD_OK;
}

int pd_get_node_fields(pd_sim *s, double *m, double *theta) {
  if (!s) { pdi::set_error("null argument"); return PD_ERR_ARG; }
  DevTmp tmp(s, sizeof(double) * s->n), th(s, sizeof(double) * s->npad);
  if (!tmp.p || !th.p) { pdi::set_error("device allocation failed"); return PD_ERR_ALLOC; }
  if (m) {
    k_gather_scalar<<<nblk(s->npad), TPB, 0, s->stream>>>(s->npad, s->perm, s->m, (double *)tmp.p);
    int rc = copy_out(s, m, tmp.p, sizeof(double) * s->n);
    if (rc) return rc;
  }
  if (theta) {
    if (int rc = flush_break(s)) return rc;
    if (int rc = pdi::launch_dilatation(s, (double *)th.p, false)) return rc;
    k_gather_scalar<<<nblk(s->npad), TPB, 0, s->stream>>>(s->npad, s->perm, (const double *)th.p, (double *)tmp.p);
    PD_CUDA(cudaGetLastError());
    int rc = copy_out(s, theta, tmp.p, sizeof(double) * s->n);
    if (rc) return rc;
  }
  return PD_OK;
}

int pd_get_bond_mask(pd_sim *s, int64_t *rowptr, int32_t *col, uint8_t *intact) {
  if (!s || !rowptr || ((col == nullptr) != (intact == nullptr))) { pdi::set_error("bad argument"); return PD_ERR_ARG; }
  if (int rc = flush_break(s)) return rc;
  DevTmp rp(s, sizeof(long long) * (s->n + 1)), c(s, col ? sizeof(int32_t) * s->Z : 1), it(s, col ? (size_t)s->Z : 1);
  if (!rp.p || !c.p || !it.p) { pdi::set_error("device allocation failed"); return PD_ERR_ALLOC; }
  int rc = pdi::export_bond_mask(s, (long long *)rp.p, col ? (int32_t *)c.p : nullptr, col ? (uint8_t *)it.p : nullptr);
  if (rc) return rc;
  if ((rc = copy_out(s, rowptr, rp.p, sizeof(long long) * (s->n + 1)))) return rc;
  if (col) {
    if ((rc = copy_out(s, col, c.p, sizeof(int32_t) * s->Z))) return rc;
    if ((rc = copy_out(s, intact, it.p, (size_t)s->Z))) return rc;
  }
  return PD_OK;
}

int pd_get_layout(pd_sim *s, int64_t counts[8]) {
  if (!s || !counts) { pdi::set_error("null argument"); return PD_ERR_ARG; }
  counts[0] = s->n; counts[1] = s->npad; counts[2] = s->Z; counts[3] = s->nentries * 32;
  counts[4] = s->launches; counts[5] = (int64_t)s->bytes_held; counts[6] = s->uniform_v ? 1 : 0;
  counts[7] = s->lat.on ? (s->lat.uniform ? (pdi::ball_eligible(s) || pdi::disc_eligible(s) ? 3 : 2) : 1) : 0;
  return PD_OK;
}

int pd_destroy(pd_sim *s) {
  if (!s) return PD_OK;
  cudaStreamSynchronize(s->stream);
  for (auto &g : s->graph) if (g) cudaGraphExecDestroy(g);
  if (s->cap_stream) cudaStreamDestroy(s->cap_stream);
  pdi::lat_free_cache(s);
  pdi::dev_free_all(s);
  delete s;
  return PD_OK;
}

}  // extern "C"
