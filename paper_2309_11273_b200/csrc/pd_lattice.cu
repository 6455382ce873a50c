// pd_lattice.cu -- dense LATTICE layout: the builder
// for bodies discretised on a (jittered) lattice, which is the paper's discretisation.
//
// When every cell of the builder's cell grid holds at most one node, the volumes are uniform and
// the union of all families is a stencil of <= 128 relative cell offsets, nothing per bond has to
// be stored but ONE BIT: the neighbour of cell c at stencil offset o is cell c + o.  Nodes live in
// dense 3-D arrays over the cell grid (pd_internal.cuh, PdLattice); the family of a node is a
// 128-bit mask over the stencil (bond exists and is unbroken, Eq. 1.30).  Exactly the same families
// as the general layout: membership is decided by the same exact distance test per node pair.
//
// This file is the builder of that layout; the step kernels are in pd_lattice_step.cu.
#include <cub/device/device_reduce.cuh>
#include <cub/iterator/transform_input_iterator.cuh>

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <vector>

#include "pd_bond.cuh"

namespace {

using pdb::FULL;
constexpr int TPB = 256;
inline unsigned nblk(int64_t n) { return (unsigned)((n + TPB - 1) / TPB); }

__device__ __forceinline__ double dist2_exact(int dim, const double *a, const double *b) {
  double s = 0.0;
  for (int k = 0; k < dim; ++k) {
    double d = __dsub_rn(b[k], a[k]);
    s = __dadd_rn(s, __dmul_rn(d, d));
  }
  return s;
}

// double -> unsigned integer with the same order (and back)
__host__ __device__ __forceinline__ unsigned long long enc_ordered(double d) {
  unsigned long long b;
  memcpy(&b, &d, 8);
  return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}
inline double dec_ordered(unsigned long long e) {
  const unsigned long long b = (e >> 63) ? (e & 0x7fffffffffffffffull) : ~e;
  double d;
  memcpy(&d, &b, 8);
  return d;
}

struct LatDims {
  int DX, DY, DZ, HX, HY, HZ;
  int64_t npad;
};
__device__ __forceinline__ int64_t lat_index(const LatDims &L, int x, int y, int z) {
  return ((int64_t)(z + L.HZ) * L.DY + (y + L.HY)) * L.DX + (x + L.HX);
}

// ---- builder kernels --------------------------------------------------------------------------
__global__ void k_lat_dup(int64_t n, const uint32_t *__restrict__ keys, int *flag) {
  int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p + 1 < n && keys[p] == keys[p + 1]) *flag = 1;   // two nodes share a cell
}

// union of all families as a set of relative cell offsets: bitmap over the (2S+1)^3 box
__global__ void k_lat_offsets(int64_t n, PdGrid g, double h2, const double *__restrict__ coords,
                              const uint32_t *__restrict__ keys, const int32_t *__restrict__ ids,
                              const int32_t *__restrict__ cell_start, const int32_t *__restrict__ cell_end,
                              unsigned int *bitmap) {
  int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n) return;
  const uint32_t key = keys[p];
  const int cx = (int)(key % g.nc[0]), cy = (int)((key / g.nc[0]) % g.nc[1]), cz = (int)(key / ((uint32_t)g.nc[0] * g.nc[1]));
  double pi[3] = {0, 0, 0};
  for (int k = 0; k < g.dim; ++k) pi[k] = coords[(int64_t)g.dim * ids[p] + g.ax[k]];
  const int wx = 2 * g.S[0] + 1, wy = 2 * g.S[1] + 1;
  for (int dz = -g.S[2]; dz <= g.S[2]; ++dz)
    for (int dy = -g.S[1]; dy <= g.S[1]; ++dy)
      for (int dx = -g.S[0]; dx <= g.S[0]; ++dx) {
        const int x = cx + dx, y = cy + dy, z = cz + dz;
        if (x < 0 || y < 0 || z < 0 || x >= g.nc[0] || y >= g.nc[1] || z >= g.nc[2]) continue;
        if (dx == 0 && dy == 0 && dz == 0) continue;
        const int o = ((dz + g.S[2]) * wy + (dy + g.S[1])) * wx + (dx + g.S[0]);
        if ((bitmap[o >> 5] >> (o & 31)) & 1u) continue;   // already known to occur
        {   // nodes sit within half a cell of their cell centre: coordinates differ by >= (|d| - 1) cell edges
          const double lx = max(abs(dx) - 1, 0) / g.inv_c[0], ly = max(abs(dy) - 1, 0) / g.inv_c[1],
                       lz = g.dim > 2 ? max(abs(dz) - 1, 0) / g.inv_c[2] : 0.0;
          if (lx * lx + ly * ly + lz * lz > h2 * (1.0 + 1e-9)) continue;
        }
        const int64_t cell = ((int64_t)z * g.nc[1] + y) * g.nc[0] + x;
        const int32_t q = cell_start[cell];
        if (cell_end[cell] <= q) continue;
        double pj[3] = {0, 0, 0};
        for (int k = 0; k < g.dim; ++k) pj[k] = coords[(int64_t)g.dim * ids[q] + g.ax[k]];
        if (dist2_exact(g.dim, pi, pj) <= h2) atomicOr(&bitmap[o >> 5], 1u << (o & 31));
      }
}

// nodes into the dense arrays (arrays pre-zeroed / perm pre-filled with -1)
__global__ void k_lat_place(int64_t n, PdGrid g, LatDims L, const double *__restrict__ coords,
                            const double *__restrict__ vol, const uint8_t *__restrict__ flags,
                            const uint32_t *__restrict__ keys, const int32_t *__restrict__ ids, int32_t *perm,
                            int32_t *iperm, double2 *nb0, double2 *nb1, double *volF, uint8_t *flagsF, uint32_t *flags32,
                            uint8_t *rgocc, int nxc, int nyq) {
  int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n) return;
  const uint32_t key = keys[p];
  const int cx = (int)(key % g.nc[0]), cy = (int)((key / g.nc[0]) % g.nc[1]), cz = (int)(key / ((uint32_t)g.nc[0] * g.nc[1]));
  const int64_t i = lat_index(L, cx, cy, cz);
  const int32_t uidx = ids[p];
  perm[i] = uidx;
  iperm[uidx] = (int32_t)i;
  for (int k = 0; k < g.dim; ++k) {
    const double x = coords[(int64_t)g.dim * uidx + g.ax[k]];
    nb0[(int64_t)k * L.npad + i].x = x;
    nb1[(int64_t)k * L.npad + i].x = x;
  }
  volF[i] = vol[uidx];
  unsigned f = flags ? flags[uidx] : 0u, fi = f & 0xC0u;   // per-dof bits move with their component
  for (int k = 0; k < g.dim; ++k) {
    if (f & (1u << g.ax[k])) fi |= 1u << k;
    if (f & (8u << g.ax[k])) fi |= 8u << k;
  }
  flagsF[i] = (uint8_t)fi;
  flags32[i] = fi;
  rgocc[((int64_t)cz * nyq + (cy >> 2)) * nxc + (cx >> 5)] = 1;
}

// family masks, m_i (Eq. 1.9, w = 1), sum_j V_j (Eq. 1.31 denominator), family size
__global__ void k_lat_masks(LatDims L, int dim, int nbits, double h2, double G, const int4 *__restrict__ offs,
                            const int32_t *__restrict__ perm, double2 *nb0, double2 *nb1,
                            const double *__restrict__ vol, double *mF, double *minvF, double *fvolF, int32_t *rowlen,
                            uint32_t *member, unsigned long long *r2lb, unsigned long long *xirange) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= L.npad || perm[i] < 0) return;
  double pi[3] = {0, 0, 0};
  for (int k = 0; k < dim; ++k) pi[k] = nb0[(int64_t)k * L.npad + i].x;
  uint32_t w[4] = {0, 0, 0, 0};
  double m = 0.0, fv = 0.0;
  int cnt = 0;
  for (int b = 0; b < nbits; ++b) {
    const int4 o = offs[b];
    if (!o.w) continue;
    const int64_t j = i + ((int64_t)o.z * L.DY + o.y) * L.DX + o.x;
    if (perm[j] < 0) continue;
    double pj[3] = {0, 0, 0};
    for (int k = 0; k < dim; ++k) pj[k] = nb0[(int64_t)k * L.npad + j].x;
    const double r2 = dist2_exact(dim, pi, pj);
    if (r2 <= h2) {
      w[b >> 5] |= 1u << (b & 31);
      {   // lower bound of ||xi||^2 per stencil offset, in the step kernels' own arithmetic (pd_bond.cuh dot3)
        double xi[3] = {0, 0, 0};
        for (int k = 0; k < dim; ++k) xi[k] = pj[k] - pi[k];
        double rk = __dmul_rn(xi[0], xi[0]);
        for (int k = 1; k < dim; ++k) rk = fma(xi[k], xi[k], rk);
        const unsigned long long bitsr = (unsigned long long)__double_as_longlong(rk);   // rk > 0: bit order = value order
        if (bitsr < r2lb[b]) atomicMin(&r2lb[b], bitsr);
        // range of every component of xi over the bonds of this stencil offset (uniform-lattice test)
        for (int k = 0; k < dim; ++k) {
          const unsigned long long e = enc_ordered(xi[k]);
          unsigned long long *mm = xirange + (b * 3 + k) * 2;
          if (e < mm[0]) atomicMin(&mm[0], e);
          if (e > mm[1]) atomicMax(&mm[1], e);
        }
      }
      const double vj = vol[j];
      m = fma(r2, vj, m);
      fv += vj;
      ++cnt;
    }
  }
  for (int q = 0; q < 4; ++q) member[(int64_t)q * L.npad + i] = w[q];
  mF[i] = m;
  fvolF[i] = fv;
  minvF[i] = m > 0.0 ? 1.0 / m : 0.0;
  rowlen[i] = cnt;
  const double gmu = m > 0.0 ? G / m : 0.0;
  nb0[(int64_t)PD_P_AUX * L.npad + i].x = gmu;
  nb1[(int64_t)PD_P_AUX * L.npad + i].x = gmu;
}

// uniform lattice: the static half of the {G/m, cth} pairs
__global__ void k_ulat_aux(int64_t npad, double G, const double *__restrict__ minv, double2 *aux) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < npad) aux[i] = make_double2(G * minv[i], 0.0);
}

__global__ void k_lat_checks(int64_t npad, const int32_t *__restrict__ perm, const int32_t *__restrict__ rowlen,
                             const uint8_t *__restrict__ flags, unsigned long long *out) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= npad || perm[i] < 0) return;
  if (rowlen[i] == 0) atomicOr(&out[0], 1ull);  // some node has an empty family
  unsigned f = flags[i];
  if (f & PD_NO_FAIL) atomicOr(&out[1], 1ull);
  if (f) atomicOr(&out[1], 2ull);
}

// dense index -> cell offset of b relative to a -> bit (or -1)
__device__ __forceinline__ int lat_pair_bit(const LatDims &L, const int *S, const int32_t *off2bit, int64_t a, int64_t b) {
  const int ax_ = (int)(a % L.DX), ay = (int)((a / L.DX) % L.DY), az = (int)(a / ((int64_t)L.DX * L.DY));
  const int bx = (int)(b % L.DX), by = (int)((b / L.DX) % L.DY), bz = (int)(b / ((int64_t)L.DX * L.DY));
  const int dx = bx - ax_, dy = by - ay, dz = bz - az;
  if (abs(dx) > S[0] || abs(dy) > S[1] || abs(dz) > S[2]) return -1;
  return off2bit[((dz + S[2]) * (2 * S[1] + 1) + (dy + S[1])) * (2 * S[0] + 1) + (dx + S[0])];
}

struct S3 { int s[3]; };
__global__ void k_lat_precut(int64_t np, int64_t n, LatDims L, S3 S, const int32_t *__restrict__ pairs,
                             const int32_t *__restrict__ iperm, const int32_t *__restrict__ off2bit,
                             const uint32_t *__restrict__ member, uint32_t *mask, unsigned long long *err) {
  int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= 2 * np) return;
  int64_t pa = pairs[2 * (p >> 1) + (p & 1)], pb = pairs[2 * (p >> 1) + 1 - (p & 1)];
  if (pa < 0 || pa >= n || pb < 0 || pb >= n || pa == pb) { atomicExch(err, 1ull); return; }
  const int64_t a = iperm[pa], b = iperm[pb];
  const int bit = lat_pair_bit(L, S.s, off2bit, a, b);
  if (bit < 0 || !((member[(int64_t)(bit >> 5) * L.npad + a] >> (bit & 31)) & 1u)) { atomicExch(err, 1ull); return; }  // not a bond
  atomicAnd(&mask[(int64_t)(bit >> 5) * L.npad + a], ~(1u << (bit & 31)));
}

__global__ void k_lat_nofail(LatDims L, int nbits, const int4 *__restrict__ offs, const int32_t *__restrict__ perm,
                             const uint8_t *__restrict__ flags, const uint32_t *__restrict__ member, uint32_t *nofail) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= L.npad || perm[i] < 0) return;
  const bool own = flags[i] & PD_NO_FAIL;
  for (int q = 0; q < 4; ++q) {
    const uint32_t mb = member[(int64_t)q * L.npad + i];
    uint32_t w = 0;
    for (int b = 32 * q; b < min(nbits, 32 * q + 32); ++b) {
      if (!((mb >> (b & 31)) & 1u)) continue;
      const int4 o = offs[b];
      const int64_t j = i + ((int64_t)o.z * L.DY + o.y) * L.DX + o.x;
      if (own || (flags[j] & PD_NO_FAIL)) w |= 1u << (b & 31);
    }
    nofail[(int64_t)q * L.npad + i] = w;
  }
}

__global__ void k_lat_export(LatDims L, int nbits, const int4 *__restrict__ offs, const int32_t *__restrict__ perm,
                             const long long *__restrict__ rowptr, const uint32_t *__restrict__ member,
                             const uint32_t *__restrict__ mask, int32_t *col_out, uint8_t *intact_out) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= L.npad || perm[i] < 0) return;
  long long base = rowptr[perm[i]];
  for (int b = 0; b < nbits; ++b) {
    if (!((member[(int64_t)(b >> 5) * L.npad + i] >> (b & 31)) & 1u)) continue;
    const int4 o = offs[b];
    const int64_t j = i + ((int64_t)o.z * L.DY + o.y) * L.DX + o.x;
    col_out[base] = perm[j];
    intact_out[base] = (uint8_t)((mask[(int64_t)(b >> 5) * L.npad + i] >> (b & 31)) & 1u);
    ++base;
  }
}

LatDims lat_dims(const pd_sim *s) {
  const PdLattice &l = s->lat;
  return LatDims{l.DX, l.DY, l.DZ, l.HX, l.HY, l.HZ, s->npad};
}

// device copy of the per-bit offset table {dx, dy, dz, valid}; freed by the caller
int4 *make_offs_dev(pd_sim *s) {
  const PdLattice &l = s->lat;
  std::vector<int4> h(std::max(l.nbits, 1), int4{0, 0, 0, 0});
  for (int c = 0; c < l.ncol; ++c)
    for (int t = 0; t < l.cols[c].n; ++t)
      h[l.cols[c].word * 32 + l.cols[c].bit0 + t] = int4{l.cols[c].dx, l.cols[c].dy0 + t, l.cols[c].dz, 1};
  int4 *d = (int4 *)pdi::dev_alloc(s, sizeof(int4) * h.size());
  if (!d) return nullptr;
  if (cudaMemcpyAsync(d, h.data(), sizeof(int4) * h.size(), cudaMemcpyHostToDevice, s->stream) != cudaSuccess ||
      cudaStreamSynchronize(s->stream) != cudaSuccess) {
    pdi::dev_free(s, d);
    return nullptr;
  }
  return d;
}

}  // namespace

namespace pdi {

#define LAT_ALLOC(ptr, type, count)                                          \
  do {                                                                       \
    ptr = (type *)dev_alloc(s, sizeof(type) * (size_t)(count));              \
    if (!ptr) { set_error("device allocation failed in pd_create"); return PD_ERR_ALLOC; } \
  } while (0)

int build_lattice(pd_sim *s, const PdGrid &g, const double *coords, const double *vol, const uint8_t *flags,
                  const int32_t *precut, int64_t n_precut, const uint32_t *keys, const int32_t *ids,
                  const int32_t *cell_start, const int32_t *cell_end) {
  cudaStream_t st = s->stream;
  const int64_t n = s->n;
  const int dim = s->dim;
  PdLattice &l = s->lat;
  l.on = false;
  if (!s->uniform_v) return 0;
  if (const char *env = getenv("PD_FORCE_GENERIC")) { if (atoi(env)) return 0; }
  const double ncell = (double)g.nc[0] * g.nc[1] * g.nc[2];
  if ((double)n < 0.2 * ncell) return 0;                      // too sparse for a dense array
  std::vector<void *> scratch;
  auto salloc = [&](size_t bytes) -> void * {
    void *p = dev_alloc(s, bytes ? bytes : 1);
    if (p) scratch.push_back(p);
    return p;
  };
  struct Guard {
    pd_sim *s; std::vector<void *> &v;
    ~Guard() { cudaStreamSynchronize(s->stream); for (void *p : v) dev_free(s, p); }
  } guard{s, scratch};

  // ---- one node per cell? ----
  int *dflag = (int *)salloc(sizeof(int));
  if (!dflag) { set_error("device allocation failed"); return PD_ERR_ALLOC; }
  PD_CUDA(cudaMemsetAsync(dflag, 0, sizeof(int), st));
  k_lat_dup<<<nblk(n), TPB, 0, st>>>(n, keys, dflag);
  int hflag = 0;
  PD_CUDA(cudaMemcpyAsync(&hflag, dflag, sizeof(int), cudaMemcpyDeviceToHost, st));
  PD_CUDA(cudaStreamSynchronize(st));
  if (hflag) return 0;

  // ---- the stencil: union of all families as relative cell offsets ----
  const double h2 = s->horizon * s->horizon;
  for (int k = 0; k < 3; ++k) l.S[k] = g.S[k];
  const int wx = 2 * g.S[0] + 1, wy = 2 * g.S[1] + 1, wz = 2 * g.S[2] + 1;
  const int nbox = wx * wy * wz, nbw = (nbox + 31) / 32;
  unsigned int *bitmap = (unsigned int *)salloc(sizeof(unsigned int) * nbw);
  if (!bitmap) { set_error("device allocation failed"); return PD_ERR_ALLOC; }
  PD_CUDA(cudaMemsetAsync(bitmap, 0, sizeof(unsigned int) * nbw, st));
  k_lat_offsets<<<nblk(n), TPB, 0, st>>>(n, g, h2, coords, keys, ids, cell_start, cell_end, bitmap);
  std::vector<unsigned int> hb(nbw);
  PD_CUDA(cudaMemcpyAsync(hb.data(), bitmap, sizeof(unsigned int) * nbw, cudaMemcpyDeviceToHost, st));
  PD_CUDA(cudaStreamSynchronize(st));
  auto has = [&](int dx, int dy, int dz) {
    if (abs(dx) > g.S[0] || abs(dy) > g.S[1] || abs(dz) > g.S[2]) return false;
    const int o = ((dz + g.S[2]) * wy + (dy + g.S[1])) * wx + (dx + g.S[0]);
    return ((hb[o >> 5] >> (o & 31)) & 1u) != 0;
  };
  // columns (dz, dx) of runs along y, cut at 7 steps; the bits of a column stay inside one word
  l.ncol = 0;
  int bit = 0;
  l.HX = l.HY = l.HZ = 0;
  std::vector<int32_t> off2bit(nbox, -1);
  for (int dz = -g.S[2]; dz <= g.S[2]; ++dz)
    for (int dx = -g.S[0]; dx <= g.S[0]; ++dx) {
      int dy = -g.S[1];
      while (dy <= g.S[1]) {
        if (!has(dx, dy, dz)) { ++dy; continue; }
        int nrun = 0;
        while (nrun < PD_MAXSTEP && has(dx, dy + nrun, dz)) ++nrun;
        if ((bit & 31) + nrun > 32) bit = (bit + 31) & ~31;
        if (l.ncol >= PD_LAT_MAXCOL || bit + nrun > 128) return 0;   // stencil too large for this layout
        PdLatCol &c = l.cols[l.ncol++];
        c.dx = (int16_t)dx; c.dy0 = (int16_t)dy; c.dz = (int16_t)dz;
        c.n = (uint8_t)nrun; c.word = (uint8_t)(bit >> 5); c.bit0 = (uint8_t)(bit & 31); c.split = 0; c.pad0 = c.pad1 = 0;
        for (int t = 0; t < nrun; ++t)
          off2bit[((dz + g.S[2]) * wy + (dy + t + g.S[1])) * wx + (dx + g.S[0])] = bit + t;
        l.HX = std::max(l.HX, abs(dx));
        l.HY = std::max(l.HY, std::max(abs(dy), abs(dy + nrun - 1)));
        l.HZ = std::max(l.HZ, abs(dz));
        bit += nrun;
        dy += nrun;
      }
    }
  if (l.ncol == 0) return 0;
  l.nbits = bit;
  l.nw = (bit + 31) / 32;
  for (int q = 0; q < 4; ++q) l.fullw[q] = 0;
  for (int c = 0; c < l.ncol; ++c)
    for (int t = 0; t < l.cols[c].n; ++t) l.fullw[l.cols[c].word] |= 1u << (l.cols[c].bit0 + t);

  // ---- dense dims ----
  // (tiles may overrun PY / PZ by up to 8 cells: the dense arrays carry that much zero-filled slack)
  l.PX = (g.nc[0] + 31) / 32 * 32;
  l.PY = (g.nc[1] + 3) / 4 * 4;
  l.PZ = dim == 3 ? g.nc[2] : 1;
  l.DX = l.PX + 2 * l.HX; l.DY = l.PY + 2 * l.HY + 8; l.DZ = l.PZ + 2 * l.HZ + (dim == 3 ? 8 : 0);
  const double npad_d = (double)l.DX * l.DY * l.DZ;
  if (npad_d >= 2.0e9 || npad_d * PD_NP >= 4.0e9) return 0;
  s->npad = (int64_t)l.DX * l.DY * l.DZ;
  s->ngroups = 0; s->nslices = 0;
  const LatDims L = lat_dims(s);
  const int nxc = l.PX / 32, nyq = (l.PY + 8) / 4;

  // ---- arrays ----
  for (int q = 0; q < 2; ++q) {
    LAT_ALLOC(s->nb[q], double2, s->npad * PD_NP);
    PD_CUDA(cudaMemsetAsync(s->nb[q], 0, sizeof(double2) * s->npad * PD_NP, st));
  }
  LAT_ALLOC(s->perm, int32_t, s->npad);
  LAT_ALLOC(s->iperm, int32_t, n);
  LAT_ALLOC(s->vol, double, s->npad);
  LAT_ALLOC(s->m, double, s->npad);
  LAT_ALLOC(s->minv, double, s->npad);
  LAT_ALLOC(s->fvol, double, s->npad);
  LAT_ALLOC(s->flags, uint8_t, s->npad);
  LAT_ALLOC(s->rowlen, int32_t, s->npad);
  LAT_ALLOC(l.member, uint32_t, 4 * s->npad);
  LAT_ALLOC(l.mask, uint32_t, 4 * s->npad);
  LAT_ALLOC(l.rgocc, uint8_t, (size_t)(l.PZ + 8) * nyq * nxc);
  LAT_ALLOC(l.off2bit, int32_t, nbox);
  LAT_ALLOC(l.flags32, uint32_t, s->npad);
  PD_CUDA(cudaMemsetAsync(l.flags32, 0, sizeof(uint32_t) * s->npad, st));
  PD_CUDA(cudaMemsetAsync(s->perm, 0xff, sizeof(int32_t) * s->npad, st));
  for (double *p : {s->vol, s->m, s->minv, s->fvol}) PD_CUDA(cudaMemsetAsync(p, 0, sizeof(double) * s->npad, st));
  PD_CUDA(cudaMemsetAsync(s->flags, 0, s->npad, st));
  PD_CUDA(cudaMemsetAsync(s->rowlen, 0, sizeof(int32_t) * s->npad, st));
  PD_CUDA(cudaMemsetAsync(l.member, 0, sizeof(uint32_t) * 4 * s->npad, st));
  PD_CUDA(cudaMemsetAsync(l.rgocc, 0, (size_t)(l.PZ + 8) * nyq * nxc, st));
  PD_CUDA(cudaMemcpyAsync(l.off2bit, off2bit.data(), sizeof(int32_t) * nbox, cudaMemcpyHostToDevice, st));
  k_lat_place<<<nblk(n), TPB, 0, st>>>(n, g, L, coords, vol, flags, keys, ids, s->perm, s->iperm, s->nb[0], s->nb[1],
                                       s->vol, s->flags, l.flags32, l.rgocc, nxc, nyq);
  l.on = true;   // from here on the allocations belong to the lattice layout (freed by pd_destroy / fail path)
  int4 *offs = make_offs_dev(s);
  if (!offs) { set_error("device allocation failed"); return PD_ERR_ALLOC; }
  scratch.push_back(offs);
  unsigned long long *r2lb_d = (unsigned long long *)salloc(sizeof(unsigned long long) * 128);
  if (!r2lb_d) { set_error("device allocation failed"); return PD_ERR_ALLOC; }
  PD_CUDA(cudaMemsetAsync(r2lb_d, 0xff, sizeof(unsigned long long) * 128, st));
  unsigned long long *xir_d = (unsigned long long *)salloc(sizeof(unsigned long long) * 128 * 6);
  if (!xir_d) { set_error("device allocation failed"); return PD_ERR_ALLOC; }
  {
    std::vector<unsigned long long> init(128 * 6);
    for (int q = 0; q < 128 * 3; ++q) { init[2 * q] = ~0ull; init[2 * q + 1] = 0ull; }
    PD_CUDA(cudaMemcpyAsync(xir_d, init.data(), sizeof(unsigned long long) * 128 * 6, cudaMemcpyHostToDevice, st));
    PD_CUDA(cudaStreamSynchronize(st));
  }
  k_lat_masks<<<nblk(s->npad), TPB, 0, st>>>(L, dim, l.nbits, h2, s->G, offs, s->perm, s->nb[0], s->nb[1], s->vol, s->m,
                                             s->minv, s->fvol, s->rowlen, l.member, r2lb_d, xir_d);
  std::vector<unsigned long long> xir(128 * 6);
  PD_CUDA(cudaMemcpyAsync(xir.data(), xir_d, sizeof(unsigned long long) * 128 * 6, cudaMemcpyDeviceToHost, st));
  {
    unsigned long long hb2[128];
    PD_CUDA(cudaMemcpyAsync(hb2, r2lb_d, sizeof(hb2), cudaMemcpyDeviceToHost, st));
    PD_CUDA(cudaStreamSynchronize(st));
    for (int b = 0; b < 128; ++b) {
      double v = 0.0;
      if (hb2[b] != ~0ull) memcpy(&v, &hb2[b], 8);
      l.r2lb[b] = v;   // 0: no bond with this offset -> the filter never passes it
    }
  }
  PD_CUDA(cudaMemcpyAsync(l.mask, l.member, sizeof(uint32_t) * 4 * s->npad, cudaMemcpyDeviceToDevice, st));

  // ---- Z, checks ----
  long long *zsum = (long long *)salloc(sizeof(long long));
  unsigned long long *red = (unsigned long long *)salloc(4 * sizeof(unsigned long long));
  if (!zsum || !red) { set_error("device allocation failed"); return PD_ERR_ALLOC; }
  {
    cub::TransformInputIterator<long long, cub::CastOp<long long>, const int32_t *> it(s->rowlen, cub::CastOp<long long>());
    size_t tb = 0;
    PD_CUDA(cub::DeviceReduce::Sum(nullptr, tb, it, zsum, (int)s->npad, st));
    void *tmp = salloc(tb);
    if (!tmp) { set_error("device allocation failed"); return PD_ERR_ALLOC; }
    PD_CUDA(cub::DeviceReduce::Sum(tmp, tb, it, zsum, (int)s->npad, st));
  }
  long long hz = 0;
  unsigned long long hred[4] = {0, 0, 0, 0};
  PD_CUDA(cudaMemcpyAsync(&hz, zsum, sizeof(long long), cudaMemcpyDeviceToHost, st));
  PD_CUDA(cudaMemsetAsync(red, 0, 4 * sizeof(unsigned long long), st));
  k_lat_checks<<<nblk(s->npad), TPB, 0, st>>>(s->npad, s->perm, s->rowlen, s->flags, red);
  PD_CUDA(cudaMemcpyAsync(hred, red, 2 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
  PD_CUDA(cudaStreamSynchronize(st));
  s->Z = hz;
  s->nentries = 0; s->nsegs = 0;
  if (hred[0]) { set_error("a node has an empty family (m_i = 0); enlarge the horizon"); return PD_ERR_ISOLATED; }
  if (s->Z >= (1ll << 31)) { set_error("more than 2^31 directed bonds"); return PD_ERR_LIMIT; }
  s->has_nofail = (hred[1] & 1ull) != 0;
  s->has_bc = (hred[1] & 2ull) != 0;

  // ---- pre-cuts, no-fail ----
  if (n_precut > 0) {
    PD_CUDA(cudaMemsetAsync(red, 0, sizeof(unsigned long long), st));
    k_lat_precut<<<nblk(2 * n_precut), TPB, 0, st>>>(n_precut, n, L, S3{{l.S[0], l.S[1], l.S[2]}}, precut, s->iperm, l.off2bit,
                                                    l.member, l.mask, red);
    PD_CUDA(cudaMemcpyAsync(hred, red, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
    PD_CUDA(cudaStreamSynchronize(st));
    if (hred[0]) { set_error("a pre-cut pair is out of range or not a bond"); return PD_ERR_ARG; }
  }
  if (s->has_nofail && s->fracture) {
    LAT_ALLOC(l.nofail, uint32_t, 4 * s->npad);
    PD_CUDA(cudaMemsetAsync(l.nofail, 0, sizeof(uint32_t) * 4 * s->npad, st));
    k_lat_nofail<<<nblk(s->npad), TPB, 0, st>>>(L, l.nbits, offs, s->perm, s->flags, l.member, l.nofail);
  }
  PD_CUDA(cudaGetLastError());
  PD_CUDA(cudaStreamSynchronize(st));

  // ---- uniform lattice?  Every bond of a stencil offset o has xi = (o_k h_k) to within the rounding of the
  //      coordinates (8 ulp of the largest coordinate per axis): the bond geometry becomes a per-offset constant
  //      and the step kernels of pd_lattice_uniform.cu gather displacements only.  h_k = midpoint of the range
  //      of xi_k over the bonds of the unit offset e_k (antisymmetric by construction: xi_ji = -xi_ij exactly).
  for (int w = 0; w <= 4; ++w) {
    int c = 0;
    while (c < l.ncol && l.cols[c].word < w) ++c;
    l.wbeg[w] = c;
  }
  l.uniform = false;
  bool want_uniform = !s->geom;   // (the geometric-extension variant needs xi + eta per bond)
  if (const char *env = getenv("PD_LAT_UNIFORM")) want_uniform = atoi(env) != 0;
  if (want_uniform) {
    bool ok = true;
    double h[3] = {0, 0, 0}, tol[3] = {0, 0, 0};
    auto range = [&](int b, int k, double &lo, double &hi) {
      const unsigned long long e0 = xir[(size_t)(b * 3 + k) * 2], e1 = xir[(size_t)(b * 3 + k) * 2 + 1];
      if (e0 == ~0ull) return false;   // no bond with this offset
      lo = dec_ordered(e0); hi = dec_ordered(e1);
      return true;
    };
    for (int k = 0; k < dim && ok; ++k) {
      const int e[3] = {k == 0, k == 1, k == 2};
      const int b = has(e[0], e[1], e[2]) ? off2bit[((e[2] + g.S[2]) * wy + (e[1] + g.S[1])) * wx + (e[0] + g.S[0])] : -1;
      double lo = 0, hi = 0;
      if (b < 0 || !range(b, k, lo, hi) || !(lo > 0.0)) { ok = false; break; }
      h[k] = 0.5 * (lo + hi);
      const double cmax = std::max(std::fabs(g.lo[k]), std::fabs(g.lo[k] + (g.nc[k] - 1) / g.inv_c[k])) + h[k];
      tol[k] = 8.0 * 2.220446049250313e-16 * cmax;
    }
    for (int c = 0; c < l.ncol && ok; ++c)
      for (int t = 0; t < l.cols[c].n && ok; ++t) {
        const int b = l.cols[c].word * 32 + l.cols[c].bit0 + t;
        const int o[3] = {l.cols[c].dx, l.cols[c].dy0 + t, l.cols[c].dz};
        for (int k = 0; k < dim; ++k) {
          double lo = 0, hi = 0;
          if (!range(b, k, lo, hi)) continue;
          const double nominal = (double)o[k] * h[k];
          if (std::fabs(lo - nominal) > tol[k] || std::fabs(hi - nominal) > tol[k]) ok = false;
        }
      }
    if (ok) {
      for (int k = 0; k < 3; ++k) l.h[k] = h[k];
      for (int q = 0; q < 2; ++q) {
        LAT_ALLOC(l.uxy[q], double2, s->npad);
        PD_CUDA(cudaMemsetAsync(l.uxy[q], 0, sizeof(double2) * s->npad, st));
        if (dim == 3) {
          LAT_ALLOC(l.uz[q], double, s->npad);
          PD_CUDA(cudaMemsetAsync(l.uz[q], 0, sizeof(double) * s->npad, st));
        }
      }
      LAT_ALLOC(l.aux, double2, s->npad);
      k_ulat_aux<<<nblk(s->npad), TPB, 0, st>>>(s->npad, s->G, s->minv, l.aux);
      PD_CUDA(cudaGetLastError());
      PD_CUDA(cudaStreamSynchronize(st));
      for (int q = 0; q < 2; ++q) { dev_free(s, s->nb[q]); s->nb[q] = nullptr; }   // positions are not needed any more
      l.uniform = true;
    }
  }
  return 1;
}

int lat_export_bond_mask(pd_sim *s, const long long *rowptr_dev, int32_t *col_dev, uint8_t *intact_dev) {
  int4 *offs = make_offs_dev(s);
  if (!offs) { set_error("device allocation failed"); return PD_ERR_ALLOC; }
  k_lat_export<<<nblk(s->npad), TPB, 0, s->stream>>>(lat_dims(s), s->lat.nbits, offs, s->perm, rowptr_dev, s->lat.member,
                                                     s->lat.mask, col_dev, intact_dev);
  cudaError_t e = cudaGetLastError();
  cudaStreamSynchronize(s->stream);
  dev_free(s, offs);
  return e == cudaSuccess ? PD_OK : cuda_fail(e, "k_lat_export");
}

}  // namespace pdi

