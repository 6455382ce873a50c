// pd_build.cu -- GPU cell-list family builder.
//
// Runs once in pd_create, entirely on the device:
//   1. bounding box, fine uniform cell grid (cell edge = horizon / kdiv, kdiv ~ horizon/spacing)
//   2. brick-raster sort key per node (bricks of BX x BY x BZ fine cells, raster inside a brick)
//      -> radix sort -> permutation perm[sorted] = user.  Consecutive sorted nodes are consecutive
//      along x inside a brick row, so a warp (32 lanes = 32 nodes) gathers contiguous neighbour data
//      and a CTA covers a compact spatial tile.
//   3. dense cell table (start/end in sorted order)
//   4. count pass  -> row length per node -> slice length (warp max, rounded to PD_SLOT_ALIGN)
//      -> exclusive scan -> slice offsets (SELL-32)
//   5. fill pass   -> col (neighbour sorted index per slot), intact mask, m_i (Eq. 1.9), sum_j V_j
//   6. pre-cut pairs clear their two mask bits; no-fail bit mask (only if some node is no-fail)
// The horizon test is ||xi||^2 <= horizon^2 (inclusive) with the products and
// sums rounded individually in component order (no FMA contraction), so it is reproducible.
#include <cub/device/device_radix_sort.cuh>
#include <cub/device/device_reduce.cuh>
#include <cub/device/device_scan.cuh>
#include <cub/iterator/transform_input_iterator.cuh>

#include <algorithm>
#include <cmath>

#include "pd_internal.cuh"

namespace {

constexpr int TPB = 256;

struct Grid {
  double lo[3];
  double inv_c;  // 1 / cell edge
  int nc[3];     // fine cells per dim
  int nb[3];     // bricks per dim
  int B[3];      // brick size in cells
  int R;         // search radius in cells
  int dim;
};

__device__ __forceinline__ void cell_of(const Grid &g, const double *p, int *q) {
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    if (k < g.dim) {
      int c = (int)floor((p[k] - g.lo[k]) * g.inv_c);
      q[k] = min(max(c, 0), g.nc[k] - 1);
    } else {
      q[k] = 0;
    }
  }
}

__device__ __forceinline__ double dist2_exact(int dim, const double *a, const double *b) {
  double s = 0.0;
  for (int k = 0; k < dim; ++k) {
    double d = __dsub_rn(b[k], a[k]);
    s = __dadd_rn(s, __dmul_rn(d, d));
  }
  return s;
}

// ---- 1. bounding box ------------------------------------------------------------------------
__device__ __forceinline__ unsigned long long enc(double x) {  // order-preserving double -> u64
  unsigned long long b = (unsigned long long)__double_as_longlong(x);
  return (b & 0x8000000000000000ull) ? ~b : (b | 0x8000000000000000ull);
}
static double dec_host(unsigned long long e) {
  unsigned long long b = (e & 0x8000000000000000ull) ? (e & 0x7fffffffffffffffull) : ~e;
  double x;
  memcpy(&x, &b, 8);
  return x;
}

__global__ void k_bbox(int64_t n, int dim, const double *__restrict__ coords, const double *__restrict__ vol,
                       unsigned long long *out /* [0..2]=min, [3..5]=max, [6]=vmin, [7]=vmax */) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  for (int k = 0; k < dim; ++k) {
    unsigned long long e = enc(coords[dim * i + k]);
    atomicMin(&out[k], e);
    atomicMax(&out[3 + k], e);
  }
  unsigned long long ev = enc(vol[i]);
  atomicMin(&out[6], ev);
  atomicMax(&out[7], ev);
}

// ---- 2. sort keys -----------------------------------------------------------------------------
__global__ void k_keys(int64_t n, Grid g, const double *__restrict__ coords, unsigned long long *keys,
                       int32_t *ids) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double p[3] = {0, 0, 0};
  for (int k = 0; k < g.dim; ++k) p[k] = coords[g.dim * i + k];
  int q[3];
  cell_of(g, p, q);
  unsigned long long brick = ((unsigned long long)(q[2] / g.B[2]) * g.nb[1] + (q[1] / g.B[1])) * g.nb[0] + (q[0] / g.B[0]);
  unsigned long long inner = ((unsigned long long)(q[2] % g.B[2]) * g.B[1] + (q[1] % g.B[1])) * g.B[0] + (q[0] % g.B[0]);
  keys[i] = brick * (unsigned long long)(g.B[0] * g.B[1] * g.B[2]) + inner;
  ids[i] = (int32_t)i;
}

// ---- gather user -> sorted --------------------------------------------------------------------
__global__ void k_gather_nodes(int64_t n, int64_t npad, int dim, const int32_t *__restrict__ perm,
                               const double *__restrict__ coords, const double *__restrict__ vol,
                               const uint8_t *__restrict__ flags, double *x0, double *x1, double *x2,
                               double *volS, uint8_t *flagsS, int32_t *iperm) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= npad) return;
  double *xs[3] = {x0, x1, x2};
  if (i < n) {
    int32_t uidx = perm[i];
    for (int k = 0; k < dim; ++k) xs[k][i] = coords[(int64_t)dim * uidx + k];
    volS[i] = vol[uidx];
    flagsS[i] = flags ? flags[uidx] : (uint8_t)0;
    iperm[uidx] = (int32_t)i;
  } else {  // padding nodes: never referenced as neighbours, never written back
    for (int k = 0; k < dim; ++k) xs[k][i] = 0.0;
    volS[i] = 0.0;
    flagsS[i] = 0;
  }
}

// ---- 3. cell table ----------------------------------------------------------------------------
__device__ __forceinline__ int64_t raster_cell(const Grid &g, const int *q) {
  return ((int64_t)q[2] * g.nc[1] + q[1]) * g.nc[0] + q[0];
}

__global__ void k_cell_table(int64_t n, Grid g, const double *__restrict__ x0, const double *__restrict__ x1,
                             const double *__restrict__ x2, int32_t *cell_start, int32_t *cell_end) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double *xs[3] = {x0, x1, x2};
  int q[3];
  double p[3] = {0, 0, 0};
  for (int k = 0; k < g.dim; ++k) p[k] = xs[k][i];
  cell_of(g, p, q);
  int64_t c = raster_cell(g, q);
  int64_t cprev = -1, cnext = -1;
  if (i > 0) {
    for (int k = 0; k < g.dim; ++k) p[k] = xs[k][i - 1];
    cell_of(g, p, q);
    cprev = raster_cell(g, q);
  }
  if (i + 1 < n) {
    for (int k = 0; k < g.dim; ++k) p[k] = xs[k][i + 1];
    cell_of(g, p, q);
    cnext = raster_cell(g, q);
  }
  if (c != cprev) cell_start[c] = (int32_t)i;
  if (c != cnext) cell_end[c] = (int32_t)(i + 1);
}

// ---- 4./5. family traversal ---------------------------------------------------------------------
// Visits the family of sorted node i in a fixed order (cells dz, dy, dx ascending; sorted index
// ascending inside a cell) and calls f(j, r2).
template <typename F>
__device__ __forceinline__ void for_family(const Grid &g, int64_t i, double h2, const double *__restrict__ x0,
                                           const double *__restrict__ x1, const double *__restrict__ x2,
                                           const int32_t *__restrict__ cell_start,
                                           const int32_t *__restrict__ cell_end, F f) {
  const double *xs[3] = {x0, x1, x2};
  double pi[3] = {0, 0, 0};
  for (int k = 0; k < g.dim; ++k) pi[k] = xs[k][i];
  int q[3];
  cell_of(g, pi, q);
  int z0 = g.dim > 2 ? max(q[2] - g.R, 0) : 0, z1 = g.dim > 2 ? min(q[2] + g.R, g.nc[2] - 1) : 0;
  int y0 = max(q[1] - g.R, 0), y1 = min(q[1] + g.R, g.nc[1] - 1);
  int xa = max(q[0] - g.R, 0), xb = min(q[0] + g.R, g.nc[0] - 1);
  for (int cz = z0; cz <= z1; ++cz)
    for (int cy = y0; cy <= y1; ++cy) {
      int64_t base = ((int64_t)cz * g.nc[1] + cy) * g.nc[0];
      for (int cx = xa; cx <= xb; ++cx) {
        int32_t s = cell_start[base + cx], e = cell_end[base + cx];
        for (int32_t j = s; j < e; ++j) {
          if (j == i) continue;
          double pj[3] = {0, 0, 0};
          for (int k = 0; k < g.dim; ++k) pj[k] = xs[k][j];
          double r2 = dist2_exact(g.dim, pi, pj);
          if (r2 <= h2) f(j, r2);
        }
      }
    }
}

__global__ void k_count(int64_t n, int64_t npad, Grid g, double h2, const double *__restrict__ x0,
                        const double *__restrict__ x1, const double *__restrict__ x2,
                        const int32_t *__restrict__ cell_start, const int32_t *__restrict__ cell_end,
                        int32_t *rowlen, int32_t *slice_len, int32_t *slice_words) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= npad) return;
  int cnt = 0;
  if (i < n) for_family(g, i, h2, x0, x1, x2, cell_start, cell_end, [&](int32_t, double) { ++cnt; });
  rowlen[i] = cnt;
  int mx = cnt;
  for (int o = 16; o > 0; o >>= 1) mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  if ((threadIdx.x & 31) == 0) {
    int len = (mx + PD_SLOT_ALIGN - 1) / PD_SLOT_ALIGN * PD_SLOT_ALIGN;
    slice_len[i >> 5] = len;
    slice_words[i >> 5] = (len + 31) / 32;
  }
}

__global__ void k_fill(int64_t n, int64_t npad, Grid g, double h2, const double *__restrict__ x0,
                       const double *__restrict__ x1, const double *__restrict__ x2,
                       const double *__restrict__ vol, const int32_t *__restrict__ cell_start,
                       const int32_t *__restrict__ cell_end, const int32_t *__restrict__ slice_len,
                       const uint32_t *__restrict__ slice_off, const uint32_t *__restrict__ mask_off,
                       int32_t *col, uint32_t *mask, double *m_out, double *fvol_out) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= npad) return;
  int lane = threadIdx.x & 31;
  int64_t s = i >> 5;
  int64_t off = (int64_t)slice_off[s] * 32 + lane;
  int len = slice_len[s];
  int k = 0;
  double m = 0.0, fv = 0.0;
  if (i < n)
    for_family(g, i, h2, x0, x1, x2, cell_start, cell_end, [&](int32_t j, double r2) {
      col[off + (int64_t)k * 32] = j;
      double vj = vol[j];
      m = fma(r2, vj, m);  // m_i = sum ||xi||^2 V_j   (Eq. 1.9, w = 1)
      fv += vj;            // sum V_j                   (Eq. 1.31 denominator)
      ++k;
    });
  int cnt = k;
  for (; k < len; ++k) col[off + (int64_t)k * 32] = (int32_t)i;  // padding slots: self, bit 0
  int64_t moff = (int64_t)mask_off[s] * 32 + lane;
  for (int w = 0; w * 32 < len; ++w) {
    int nb = min(max(cnt - w * 32, 0), 32);
    mask[moff + (int64_t)w * 32] = nb == 32 ? 0xffffffffu : ((1u << nb) - 1u);
  }
  m_out[i] = m;
  fvol_out[i] = fv;
}

// ---- 6. pre-cuts and no-fail mask ---------------------------------------------------------------
__global__ void k_precut(int64_t np, int64_t n, const int32_t *__restrict__ pairs, const int32_t *__restrict__ iperm,
                         const int32_t *__restrict__ rowlen, const uint32_t *__restrict__ slice_off,
                         const uint32_t *__restrict__ mask_off, const int32_t *__restrict__ col, uint32_t *mask,
                         unsigned long long *err) {
  int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= 2 * np) return;
  int64_t pa = pairs[2 * (p >> 1) + (p & 1)], pb = pairs[2 * (p >> 1) + 1 - (p & 1)];
  if (pa < 0 || pa >= n || pb < 0 || pb >= n || pa == pb) { atomicExch(err, 1ull); return; }
  int32_t a = iperm[pa], b = iperm[pb];
  int64_t s = a >> 5;
  int lane = a & 31;
  int64_t off = (int64_t)slice_off[s] * 32 + lane, moff = (int64_t)mask_off[s] * 32 + lane;
  int len = rowlen[a];
  for (int k = 0; k < len; ++k)
    if (col[off + (int64_t)k * 32] == b) {
      atomicAnd(&mask[moff + (int64_t)(k >> 5) * 32], ~(1u << (k & 31)));
      return;
    }
  atomicExch(err, 1ull);  // not a bond
}

__global__ void k_nofail(int64_t npad, const uint8_t *__restrict__ flags, const int32_t *__restrict__ rowlen,
                         const int32_t *__restrict__ slice_len, const uint32_t *__restrict__ slice_off,
                         const uint32_t *__restrict__ mask_off, const int32_t *__restrict__ col, uint32_t *nofail) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= npad) return;
  int lane = threadIdx.x & 31;
  int64_t s = i >> 5;
  int64_t off = (int64_t)slice_off[s] * 32 + lane, moff = (int64_t)mask_off[s] * 32 + lane;
  int len = slice_len[s], cnt = rowlen[i];
  unsigned fi = flags[i];
  for (int w = 0; w * 32 < len; ++w) {
    uint32_t word = 0;
    for (int b = 0; b < 32 && w * 32 + b < cnt; ++b) {
      int32_t j = col[off + (int64_t)(w * 32 + b) * 32];
      if ((fi | flags[j]) & PD_NO_FAIL) word |= 1u << b;
    }
    nofail[moff + (int64_t)w * 32] = word;
  }
}

__global__ void k_any_empty_row(int64_t n, const int32_t *__restrict__ rowlen, unsigned long long *out) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  if (rowlen[i] == 0) atomicExch(&out[0], 1ull);  // some node has an empty family
}

__global__ void k_any_flag(int64_t n, const uint8_t *__restrict__ flags, unsigned long long *out) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  unsigned f = flags[i];
  if (f & PD_NO_FAIL) atomicOr(&out[0], 1ull);
  if (f) atomicOr(&out[0], 2ull);
}

__global__ void k_node_consts(int64_t npad, int64_t n, double G, const double *__restrict__ m, double *minv,
                              double *gmu) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= npad) return;
  double mi = i < n ? m[i] : 1.0;
  minv[i] = i < n ? 1.0 / mi : 0.0;
  gmu[i] = i < n ? G / mi : 0.0;
}

__global__ void k_rowlen_user(int64_t n, const int32_t *__restrict__ iperm, const int32_t *__restrict__ rowlen,
                              long long *out) {
  int64_t uidx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (uidx >= n) return;
  out[uidx] = rowlen[iperm[uidx]];
}

__global__ void k_export_rows(int64_t n, const int32_t *__restrict__ perm, const long long *__restrict__ rowptr,
                              const int32_t *__restrict__ rowlen, const uint32_t *__restrict__ slice_off,
                              const uint32_t *__restrict__ mask_off, const int32_t *__restrict__ col,
                              const uint32_t *__restrict__ mask, int32_t *col_out, uint8_t *intact_out) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int lane = (int)(i & 31);
  int64_t s = i >> 5;
  int64_t off = (int64_t)slice_off[s] * 32 + lane, moff = (int64_t)mask_off[s] * 32 + lane;
  long long base = rowptr[perm[i]];
  int len = rowlen[i];
  for (int k = 0; k < len; ++k) {
    col_out[base + k] = perm[col[off + (int64_t)k * 32]];
    intact_out[base + k] = (uint8_t)((mask[moff + (int64_t)(k >> 5) * 32] >> (k & 31)) & 1u);
  }
}

inline unsigned nblk(int64_t n) { return (unsigned)((n + TPB - 1) / TPB); }

}  // namespace

namespace pdi {

#define BUILD_ALLOC(ptr, type, count)                                        \
  do {                                                                       \
    ptr = (type *)dev_alloc(s, sizeof(type) * (size_t)(count));              \
    if (!ptr) { set_error("device allocation failed in pd_create"); return PD_ERR_ALLOC; } \
  } while (0)

int build_family(pd_sim *s, const double *coords, const double *vol, const uint8_t *flags,
                 const int32_t *precut, int64_t n_precut) {
  cudaStream_t st = s->stream;
  const int64_t n = s->n;
  const int dim = s->dim;
  s->npad = (n + 31) / 32 * 32;
  s->nslices = s->npad / 32;

  // ---- scratch (freed at the end through the same allocator) ----
  std::vector<void *> scratch;
  auto salloc = [&](size_t bytes) -> void * {
    void *p = dev_alloc(s, bytes);
    if (p) scratch.push_back(p);
    return p;
  };
  auto sfree_all = [&]() {
    cudaStreamSynchronize(st);
    for (void *p : scratch) dev_free(s, p);
    scratch.clear();
  };
  struct Guard { decltype(sfree_all) &f; ~Guard() { f(); } } guard{sfree_all};

  // ---- 1. bbox + volume range ----
  unsigned long long *red = (unsigned long long *)salloc(8 * sizeof(unsigned long long));
  if (!red) { set_error("device allocation failed"); return PD_ERR_ALLOC; }
  unsigned long long init[8];
  for (int k = 0; k < 3; ++k) { init[k] = ~0ull; init[3 + k] = 0ull; }
  init[6] = ~0ull; init[7] = 0ull;
  PD_CUDA(cudaMemcpyAsync(red, init, sizeof(init), cudaMemcpyHostToDevice, st));
  k_bbox<<<nblk(n), TPB, 0, st>>>(n, dim, coords, vol, red);
  unsigned long long hred[8];
  PD_CUDA(cudaMemcpyAsync(hred, red, sizeof(hred), cudaMemcpyDeviceToHost, st));
  PD_CUDA(cudaStreamSynchronize(st));
  double lo[3] = {0, 0, 0}, hi[3] = {0, 0, 0};
  for (int k = 0; k < dim; ++k) { lo[k] = dec_host(hred[k]); hi[k] = dec_host(hred[3 + k]); }
  double vmin = dec_host(hred[6]), vmax = dec_host(hred[7]);
  for (int k = 0; k < dim; ++k)
    if (!std::isfinite(lo[k]) || !std::isfinite(hi[k])) { set_error("non-finite coordinate"); return PD_ERR_ARG; }
  if (!(vmin > 0.0) || !std::isfinite(vmax)) { set_error("volumes must be finite and > 0"); return PD_ERR_ARG; }
  s->uniform_v = (vmin == vmax);
  s->vol_uniform = vmin;

  // ---- fine cell grid: edge = horizon/kdiv (slightly enlarged so that a neighbour is never more
  //      than kdiv cells away in spite of rounding in the cell computation) ----
  double meas = 1.0;
  int nd = 0;
  for (int k = 0; k < dim; ++k)
    if (hi[k] > lo[k]) { meas *= (hi[k] - lo[k]); ++nd; }
  int kdiv = 1;
  if (nd > 0) {
    double spacing = std::pow(meas / (double)n, 1.0 / nd);
    if (spacing > 0) kdiv = (int)std::lround(s->horizon / spacing);
  }
  kdiv = std::min(std::max(kdiv, 1), 4);
  Grid g{};
  g.dim = dim;
  for (;;) {
    double c = (s->horizon / kdiv) * (1.0 + 1e-9);
    g.inv_c = 1.0 / c;
    double ncell = 1.0;
    for (int k = 0; k < 3; ++k) {
      g.lo[k] = lo[k];
      double cnt = k < dim ? std::floor((hi[k] - lo[k]) * g.inv_c) + 1.0 : 1.0;
      ncell *= cnt;
      g.nc[k] = cnt < 2.0e9 ? (int)cnt : 2000000000;
    }
    if (ncell <= (double)(1ll << 28)) break;
    if (kdiv == 1) { set_error("cell table too large: domain extent / horizon exceeds 2^28 cells"); return PD_ERR_LIMIT; }
    --kdiv;
  }
  g.R = kdiv;
  s->kdiv = kdiv;
  // brick = one CTA's spatial tile: 32 cells along x (one warp per row), 8 rows
  g.B[0] = 32;
  g.B[1] = dim == 2 ? 8 : 4;
  g.B[2] = dim == 2 ? 1 : 2;
  for (int k = 0; k < 3; ++k) g.nb[k] = (g.nc[k] + g.B[k] - 1) / g.B[k];
  const int64_t ncell = (int64_t)g.nc[0] * g.nc[1] * g.nc[2];

  // ---- 2. sort by brick-raster key ----
  unsigned long long *keys = (unsigned long long *)salloc(sizeof(unsigned long long) * n);
  unsigned long long *keys2 = (unsigned long long *)salloc(sizeof(unsigned long long) * n);
  int32_t *ids = (int32_t *)salloc(sizeof(int32_t) * n);
  if (!keys || !keys2 || !ids) { set_error("device allocation failed"); return PD_ERR_ALLOC; }
  BUILD_ALLOC(s->perm, int32_t, n);
  BUILD_ALLOC(s->iperm, int32_t, n);
  k_keys<<<nblk(n), TPB, 0, st>>>(n, g, coords, keys, ids);
  {
    double maxkey = (double)g.nb[0] * g.nb[1] * g.nb[2] * (g.B[0] * g.B[1] * g.B[2]);
    int bits = std::min(64, (int)std::ceil(std::log2(maxkey + 1.0)) + 1);
    size_t tb = 0;
    PD_CUDA(cub::DeviceRadixSort::SortPairs(nullptr, tb, keys, keys2, ids, s->perm, (int)n, 0, bits, st));
    void *tmp = salloc(tb ? tb : 1);
    if (!tmp) { set_error("device allocation failed"); return PD_ERR_ALLOC; }
    PD_CUDA(cub::DeviceRadixSort::SortPairs(tmp, tb, keys, keys2, ids, s->perm, (int)n, 0, bits, st));
  }

  // ---- node arrays in sorted order ----
  for (int k = 0; k < 3; ++k) {
    if (k < dim) BUILD_ALLOC(s->x[k], double, s->npad); else s->x[k] = nullptr;
  }
  BUILD_ALLOC(s->vol, double, s->npad);
  BUILD_ALLOC(s->flags, uint8_t, s->npad);
  k_gather_nodes<<<nblk(s->npad), TPB, 0, st>>>(n, s->npad, dim, s->perm, coords, vol, flags, s->x[0], s->x[1],
                                                 s->x[2], s->vol, s->flags, s->iperm);

  // ---- 3. cell table ----
  int32_t *cell_start = (int32_t *)salloc(sizeof(int32_t) * ncell);
  int32_t *cell_end = (int32_t *)salloc(sizeof(int32_t) * ncell);
  if (!cell_start || !cell_end) { set_error("device allocation failed"); return PD_ERR_ALLOC; }
  PD_CUDA(cudaMemsetAsync(cell_start, 0, sizeof(int32_t) * ncell, st));
  PD_CUDA(cudaMemsetAsync(cell_end, 0, sizeof(int32_t) * ncell, st));
  k_cell_table<<<nblk(n), TPB, 0, st>>>(n, g, s->x[0], s->x[1], s->x[2], cell_start, cell_end);

  // ---- 4. count -> slice lengths -> offsets ----
  const double h2 = s->horizon * s->horizon;
  BUILD_ALLOC(s->rowlen, int32_t, s->npad);
  BUILD_ALLOC(s->slice_len, int32_t, s->nslices);
  BUILD_ALLOC(s->slice_off, uint32_t, s->nslices + 1);
  BUILD_ALLOC(s->mask_off, uint32_t, s->nslices + 1);
  int32_t *slice_words = (int32_t *)salloc(sizeof(int32_t) * s->nslices);
  if (!slice_words) { set_error("device allocation failed"); return PD_ERR_ALLOC; }
  k_count<<<nblk(s->npad), TPB, 0, st>>>(n, s->npad, g, h2, s->x[0], s->x[1], s->x[2], cell_start, cell_end,
                                          s->rowlen, s->slice_len, slice_words);
  {
    size_t tb1 = 0, tb2 = 0;
    PD_CUDA(cub::DeviceScan::ExclusiveSum(nullptr, tb1, s->slice_len, s->slice_off, (int)s->nslices, st));
    PD_CUDA(cub::DeviceScan::ExclusiveSum(nullptr, tb2, slice_words, s->mask_off, (int)s->nslices, st));
    size_t tb = std::max(tb1, tb2);
    void *tmp = salloc(tb ? tb : 1);
    if (!tmp) { set_error("device allocation failed"); return PD_ERR_ALLOC; }
    // widen on the fly: inputs are int32 lengths, outputs uint32 offsets (in slots)
    PD_CUDA(cub::DeviceScan::ExclusiveSum(tmp, tb, s->slice_len, s->slice_off, (int)s->nslices, st));
    PD_CUDA(cub::DeviceScan::ExclusiveSum(tmp, tb, slice_words, s->mask_off, (int)s->nslices, st));
  }
  // totals (last offset + last length) and the sum of row lengths
  uint32_t last_off[2];
  int32_t last_len[2];
  PD_CUDA(cudaMemcpyAsync(&last_off[0], s->slice_off + (s->nslices - 1), 4, cudaMemcpyDeviceToHost, st));
  PD_CUDA(cudaMemcpyAsync(&last_off[1], s->mask_off + (s->nslices - 1), 4, cudaMemcpyDeviceToHost, st));
  PD_CUDA(cudaMemcpyAsync(&last_len[0], s->slice_len + (s->nslices - 1), 4, cudaMemcpyDeviceToHost, st));
  PD_CUDA(cudaMemcpyAsync(&last_len[1], slice_words + (s->nslices - 1), 4, cudaMemcpyDeviceToHost, st));
  long long *zsum = (long long *)salloc(sizeof(long long));
  if (!zsum) { set_error("device allocation failed"); return PD_ERR_ALLOC; }
  {
    // int32 row lengths summed into a 64-bit accumulator
    cub::TransformInputIterator<long long, cub::CastOp<long long>, const int32_t *> it(s->rowlen, cub::CastOp<long long>());
    size_t tb = 0;
    PD_CUDA(cub::DeviceReduce::Sum(nullptr, tb, it, zsum, (int)s->npad, st));
    void *tmp = salloc(tb ? tb : 1);
    if (!tmp) { set_error("device allocation failed"); return PD_ERR_ALLOC; }
    PD_CUDA(cub::DeviceReduce::Sum(tmp, tb, it, zsum, (int)s->npad, st));
  }
  long long hz = 0;
  PD_CUDA(cudaMemcpyAsync(&hz, zsum, sizeof(long long), cudaMemcpyDeviceToHost, st));
  PD_CUDA(cudaMemsetAsync(red, 0, 8 * sizeof(unsigned long long), st));
  k_any_empty_row<<<nblk(n), TPB, 0, st>>>(n, s->rowlen, red);
  if (flags) k_any_flag<<<nblk(n), TPB, 0, st>>>(n, flags, red + 1);
  PD_CUDA(cudaMemcpyAsync(hred, red, 2 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
  PD_CUDA(cudaStreamSynchronize(st));
  s->Z = hz;
  s->nslots = (int64_t)last_off[0] + last_len[0];
  s->nmaskwords = (int64_t)last_off[1] + last_len[1];
  if (hred[0]) { set_error("a node has an empty family (m_i = 0); enlarge the horizon"); return PD_ERR_ISOLATED; }
  if (s->nslots >= (1ll << 32) - 4096 || s->Z >= (1ll << 31)) {
    set_error("more than 2^31 directed bonds");
    return PD_ERR_LIMIT;
  }
  s->has_nofail = (hred[1] & 1ull) != 0;
  s->has_bc = (hred[1] & 2ull) != 0;

  // ---- 5. fill ----
  BUILD_ALLOC(s->col, int32_t, s->nslots * 32);
  BUILD_ALLOC(s->mask, uint32_t, s->nmaskwords * 32);
  BUILD_ALLOC(s->fvol, double, s->npad);
  BUILD_ALLOC(s->minv, double, s->npad);
  BUILD_ALLOC(s->gmu, double, s->npad);
  BUILD_ALLOC(s->m, double, s->npad);
  double *mtmp = s->m;
  k_fill<<<nblk(s->npad), TPB, 0, st>>>(n, s->npad, g, h2, s->x[0], s->x[1], s->x[2], s->vol, cell_start, cell_end,
                                         s->slice_len, s->slice_off, s->mask_off, s->col, s->mask, mtmp, s->fvol);
  k_node_consts<<<nblk(s->npad), TPB, 0, st>>>(s->npad, n, s->G, mtmp, s->minv, s->gmu);

  // ---- 6. pre-cuts, no-fail ----
  if (n_precut > 0) {
    PD_CUDA(cudaMemsetAsync(red, 0, sizeof(unsigned long long), st));
    k_precut<<<nblk(2 * n_precut), TPB, 0, st>>>(n_precut, n, precut, s->iperm, s->rowlen, s->slice_off, s->mask_off,
                                                  s->col, s->mask, red);
    PD_CUDA(cudaMemcpyAsync(hred, red, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
    PD_CUDA(cudaStreamSynchronize(st));
    if (hred[0]) { set_error("a pre-cut pair is out of range or not a bond"); return PD_ERR_ARG; }
  }
  if (s->has_nofail && s->fracture) {
    BUILD_ALLOC(s->nofail, uint32_t, s->nmaskwords * 32);
    k_nofail<<<nblk(s->npad), TPB, 0, st>>>(s->npad, s->flags, s->rowlen, s->slice_len, s->slice_off, s->mask_off,
                                             s->col, s->nofail);
  }
  PD_CUDA(cudaGetLastError());
  PD_CUDA(cudaStreamSynchronize(st));
  return PD_OK;
}

// rowptr_dev: n+1 int64 (user order); col_dev / intact_dev: Z entries or both NULL
int export_bond_mask(pd_sim *s, long long *rowptr_dev, int32_t *col_dev, uint8_t *intact_dev) {
  cudaStream_t st = s->stream;
  const int64_t n = s->n;
  long long *cnt = (long long *)dev_alloc(s, sizeof(long long) * (n + 1));
  if (!cnt) { set_error("device allocation failed"); return PD_ERR_ALLOC; }
  int rc = PD_OK;
  void *tmp = nullptr;
  do {
    if (cudaMemsetAsync(cnt + n, 0, sizeof(long long), st) != cudaSuccess) { rc = PD_ERR_CUDA; break; }
    k_rowlen_user<<<nblk(n), TPB, 0, st>>>(n, s->iperm, s->rowlen, cnt);
    size_t tb = 0;
    if (cub::DeviceScan::ExclusiveSum(nullptr, tb, cnt, rowptr_dev, (int)(n + 1), st) != cudaSuccess) { rc = PD_ERR_CUDA; break; }
    tmp = dev_alloc(s, tb ? tb : 1);
    if (!tmp) { set_error("device allocation failed"); rc = PD_ERR_ALLOC; break; }
    if (cub::DeviceScan::ExclusiveSum(tmp, tb, cnt, rowptr_dev, (int)(n + 1), st) != cudaSuccess) { rc = PD_ERR_CUDA; break; }
    if (col_dev && intact_dev)
      k_export_rows<<<nblk(n), TPB, 0, st>>>(n, s->perm, rowptr_dev, s->rowlen, s->slice_off, s->mask_off, s->col,
                                              s->mask, col_dev, intact_dev);
    if (cudaGetLastError() != cudaSuccess) rc = PD_ERR_CUDA;
  } while (0);
  cudaStreamSynchronize(st);
  if (tmp) dev_free(s, tmp);
  dev_free(s, cnt);
  if (rc == PD_ERR_CUDA) set_error("CUDA error in pd_get_bond_mask");
  return rc;
}

}  // namespace pdi
