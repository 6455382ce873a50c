// pd_lattice.cu -- dense LATTICE layout: builder and step kernels (rows a1-a5)
// for bodies discretised on a (jittered) lattice, which is the paper's discretisation.
//
// When every cell of the builder's cell grid holds at most one node, the volumes are uniform and
// the union of all families is a stencil of <= 128 relative cell offsets, nothing per bond has to
// be stored but ONE BIT: the neighbour of cell c at stencil offset o is cell c + o.  Nodes live in
// dense 3-D arrays over the cell grid (pd_internal.cuh, PdLattice); the family of a node is a
// 128-bit mask over the stencil (bond exists and is unbroken, Eq. 1.30).  Exactly the same families
// as the general layout: membership is decided by the same exact distance test per node pair.
//
// Step kernels: one CTA per spatial TILE of 32 x TY x TZ cells.  The neighbour records of the tile
// plus a halo of the stencil radius are staged in shared memory with 16-byte asynchronous copies
// (cp.async) -- every HBM/L2 access of the step is a coalesced bulk row copy, the ~120 gathers per
// node are shared-memory reads.  A warp owns a ROW GROUP (32 lanes x 4 rows adjacent in y); the
// stencil columns (dx, dy0..dy0+n-1, dz) are walked with a 4-entry register window sliding along y
// exactly as in pd_step.cu (one shared-memory record per 4 bonds), NSPLIT warps share a row group
// by splitting the columns between them and add their partial sums through shared memory.
#include <cub/device/device_reduce.cuh>
#include <cub/iterator/transform_input_iterator.cuh>

#include <algorithm>
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
        const int64_t cell = ((int64_t)z * g.nc[1] + y) * g.nc[0] + x;
        const int32_t q = cell_start[cell];
        if (cell_end[cell] <= q) continue;
        double pj[3] = {0, 0, 0};
        for (int k = 0; k < g.dim; ++k) pj[k] = coords[(int64_t)g.dim * ids[q] + g.ax[k]];
        if (dist2_exact(g.dim, pi, pj) <= h2) {
          const int o = ((dz + g.S[2]) * wy + (dy + g.S[1])) * wx + (dx + g.S[0]);
          if (!((bitmap[o >> 5] >> (o & 31)) & 1u)) atomicOr(&bitmap[o >> 5], 1u << (o & 31));
        }
      }
}

// nodes into the dense arrays (arrays pre-zeroed / perm pre-filled with -1)
__global__ void k_lat_place(int64_t n, PdGrid g, LatDims L, const double *__restrict__ coords,
                            const double *__restrict__ vol, const uint8_t *__restrict__ flags,
                            const uint32_t *__restrict__ keys, const int32_t *__restrict__ ids, int32_t *perm,
                            int32_t *iperm, double2 *nb0, double2 *nb1, double *volF, uint8_t *flagsF, uint8_t *rgocc,
                            int nxc, int nyq) {
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
  rgocc[((int64_t)cz * nyq + (cy >> 2)) * nxc + (cx >> 5)] = 1;
}

// family masks, m_i (Eq. 1.9, w = 1), sum_j V_j (Eq. 1.31 denominator), family size
__global__ void k_lat_masks(LatDims L, int dim, int nbits, double h2, double G, const int4 *__restrict__ offs,
                            const int32_t *__restrict__ perm, double2 *nb0, double2 *nb1,
                            const double *__restrict__ vol, double *mF, double *minvF, double *fvolF, int32_t *rowlen,
                            uint32_t *member) {
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
  PD_CUDA(cudaMemsetAsync(s->perm, 0xff, sizeof(int32_t) * s->npad, st));
  for (double *p : {s->vol, s->m, s->minv, s->fvol}) PD_CUDA(cudaMemsetAsync(p, 0, sizeof(double) * s->npad, st));
  PD_CUDA(cudaMemsetAsync(s->flags, 0, s->npad, st));
  PD_CUDA(cudaMemsetAsync(s->rowlen, 0, sizeof(int32_t) * s->npad, st));
  PD_CUDA(cudaMemsetAsync(l.member, 0, sizeof(uint32_t) * 4 * s->npad, st));
  PD_CUDA(cudaMemsetAsync(l.rgocc, 0, (size_t)(l.PZ + 8) * nyq * nxc, st));
  PD_CUDA(cudaMemcpyAsync(l.off2bit, off2bit.data(), sizeof(int32_t) * nbox, cudaMemcpyHostToDevice, st));
  k_lat_place<<<nblk(n), TPB, 0, st>>>(n, g, L, coords, vol, flags, keys, ids, s->perm, s->iperm, s->nb[0], s->nb[1],
                                       s->vol, s->flags, l.rgocc, nxc, nyq);
  l.on = true;   // from here on the allocations belong to the lattice layout (freed by pd_destroy / fail path)
  int4 *offs = make_offs_dev(s);
  if (!offs) { set_error("device allocation failed"); return PD_ERR_ALLOC; }
  scratch.push_back(offs);
  k_lat_masks<<<nblk(s->npad), TPB, 0, st>>>(L, dim, l.nbits, h2, s->G, offs, s->perm, s->nb[0], s->nb[1], s->vol, s->m,
                                             s->minv, s->fvol, s->rowlen, l.member);
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

// ================================================================================================
// step kernels
namespace {

struct LatCol8 { int off; uint8_t n, word, bit0, pad; };   // off: smem offset (double2 units) of entry 0 relative to row 0's own cell

struct LatArgs {
  int DX, DY, HX, HY, HZ;
  int nxc, nyt, nyq;                 // tiles along x and y; row groups along y (rgocc stride)
  int TY, TZ, SX, SY, SZ;            // tile and shared-memory tile dims
  int nsplit, nw;
  int cbeg[5];                       // split s walks cols[cbeg[s] .. cbeg[s+1])
  int64_t npad;
  uint32_t fullw[4];
  const double2 *nbr;                // pair arrays [PD_NP][npad] holding u^n (and cth^n)
  double2 *nbw;                      // dilatation: the same buffer (pair AUX written); force: the other buffer
  uint32_t *mask;
  const uint32_t *nofail;
  const uint8_t *rgocc;
  const double *minv;
  double *v[3];
  const double *bval[3];
  double *theta_out;
  const uint8_t *flags;
  const int32_t *perm;
  double A, c1, G, s_c, vol_uniform, rho, dt, ramp_time;
  int64_t step;
  LatCol8 cols[PD_LAT_MAXCOL];
};

__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gsrc) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async4(void *smem_dst, const void *gsrc) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// predicated 16-byte shared-memory load: no branch, so the four bonds of a step stay in one basic block
__device__ __forceinline__ void lds_if(double2 &v, const double2 *ptr, uint32_t pred) {
  const unsigned a = (unsigned)__cvta_generic_to_shared(ptr);
  asm("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %3, 0;\n\t@p ld.shared.v2.f64 {%0, %1}, [%2];\n\t}"
      : "+d"(v.x), "+d"(v.y) : "r"(a), "r"(pred));
}

template <int NPAIR, class E>
__device__ __forceinline__ void lds_ent(E &e, const double2 *tile, int tsz, int idx) {
  constexpr int DIMP = sizeof(e.p) / sizeof(double2);
#pragma unroll
  for (int k = 0; k < DIMP; ++k) e.p[k] = tile[k * tsz + idx];
  if (NPAIR > DIMP) e.g = tile[DIMP * tsz + idx];
}
template <int NPAIR, class E>
__device__ __forceinline__ void lds_ent_if(E &e, const double2 *tile, int tsz, int idx, uint32_t pred) {
  constexpr int DIMP = sizeof(e.p) / sizeof(double2);
#pragma unroll
  for (int k = 0; k < DIMP; ++k) lds_if(e.p[k], tile + k * tsz + idx, pred);
  if (NPAIR > DIMP) lds_if(e.g, tile + DIMP * tsz + idx, pred);
}

// one stencil column: n steps, row r of step t pairs with the record at base + (t + r) * SX
template <bool MASKED, int NPAIR, class P>
__device__ __forceinline__ void lat_run_col(P &p, const double2 *tile, int tsz, int base, int SX, int n,
                                            const uint32_t (&bits)[4], const uint32_t (&nfb)[4], uint32_t (&clr)[4]) {
  typename P::E S[4];
#pragma unroll
  for (int q = 0; q < 4; ++q) lds_ent<NPAIR>(S[q], tile, tsz, base + q * SX);
  uint32_t anyp = 0;
  if (MASKED) anyp = __reduce_or_sync(FULL, bits[0] | (bits[1] << 7) | (bits[2] << 14) | (bits[3] << 21));
  auto bond = [&](int r, const typename P::E &e, int t) {
    if (p.template bond<MASKED>(r, e, (bits[r] >> t) & 1u, (nfb[r] >> t) & 1u)) clr[r] |= 1u << t;
  };
#pragma unroll
  for (int t = 0; t < PD_MAXSTEP; ++t) {
    if (t < n) {
      const bool live = !MASKED || (anyp & (0x204081u << t)) != 0;   // warp-uniform
      if (live) bond(0, S[t % 4], t);
      lds_ent_if<NPAIR>(S[t % 4], tile, tsz, base + (t + 4) * SX, (t + 1 < n) ? 1u : 0u);   // record t+4: row 3 of step t+1
      if (live) {
        bond(1, S[(t + 1) % 4], t);
        bond(2, S[(t + 2) % 4], t);
        bond(3, S[(t + 3) % 4], t);
      }
    }
  }
}

// stages the tile, walks the columns of this warp's split, returns false if the warp has nothing to finish
// (NPAIR pairs per record: DIM position pairs + the aux pair for the force pass)
template <int DIM, int NPAIR, int MAXT, class P>
__device__ __forceinline__ bool lat_tile(P &p, const LatArgs &a, double2 *sm, int64_t (&inode)[4], int &rg, int &sp,
                                         uint32_t *&smask, int *&sflag, int &NT) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
  const int xc = blockIdx.x, yt = blockIdx.y, zt = blockIdx.z;
  const int x0 = xc * 32, y0 = yt * a.TY, z0 = zt * a.TZ;
  const int nrgy = a.TY >> 2, nrg = nrgy * a.TZ;
  NT = 32 * a.TY * a.TZ;
  const int tsz = a.SZ * a.SY * a.SX;
  smask = (uint32_t *)(sm + NPAIR * tsz + 4 * a.SX);
  sflag = (int *)(smask + 4 * NT);
  // ---- empty tile? ----
  int occ = 0;
  if ((int)threadIdx.x < nrg) {
    const int rgy = threadIdx.x % nrgy, rgz = threadIdx.x / nrgy;
    occ = a.rgocc[((int64_t)(z0 + rgz) * a.nyq + ((y0 >> 2) + rgy)) * a.nxc + xc];
  }
  if (!__syncthreads_or(occ)) return false;
  // ---- stage the tile + halo: rows of SX records, 16-byte asynchronous copies ----
  // (loops arranged so that no integer division by a run-time value is needed per row)
  const int tyshift = a.TY == 8 ? 3 : 2;
  for (int pl = warp; pl < NPAIR * a.SZ; pl += nwarp) {   // plane = (pair, z level)
    int pp = 0, zz = pl;
    while (zz >= a.SZ) { zz -= a.SZ; ++pp; }
    const int gp = pp < DIM ? pp : PD_P_AUX;
    const double2 *src = a.nbr + (int64_t)gp * a.npad + ((int64_t)(z0 + zz) * a.DY + y0) * a.DX + x0 + lane;
    double2 *dst = sm + (int64_t)pl * a.SY * a.SX + lane;
    const bool two = lane + 32 < a.SX;
    for (int yy = 0; yy < a.SY; ++yy) {
      cp_async16(dst, src);
      if (two) cp_async16(dst + 32, src + 32);
      src += a.DX;
      dst += a.SX;
    }
  }
  for (int w = 0; w < a.nw; ++w)
    for (int tn = threadIdx.x; tn < NT; tn += blockDim.x) {
      const int x = tn & 31, row = tn >> 5, y = row & (a.TY - 1), z = row >> tyshift;
      const int64_t i = ((int64_t)(z0 + z + a.HZ) * a.DY + (y0 + y + a.HY)) * a.DX + (x0 + x + a.HX);
      cp_async4(smask + w * NT + tn, a.mask + (int64_t)w * a.npad + i);
    }
  if (threadIdx.x == 0) *sflag = 0;
  cp_async_wait_all();
  __syncthreads();
  // ---- this warp's row group and column split ----
  rg = warp / a.nsplit;
  sp = warp % a.nsplit;
  const int rgy = rg % nrgy, rgz = rg / nrgy;
  const bool active = a.rgocc[((int64_t)(z0 + rgz) * a.nyq + ((y0 >> 2) + rgy)) * a.nxc + xc] != 0;
  int own0 = ((rgz + a.HZ) * a.SY + (rgy * 4 + a.HY)) * a.SX + lane + a.HX;
  int tn0 = ((rgz * a.TY) + rgy * 4) * 32 + lane;
#pragma unroll
  for (int r = 0; r < 4; ++r)
    inode[r] = ((int64_t)(z0 + rgz + a.HZ) * a.DY + (y0 + rgy * 4 + r + a.HY)) * a.DX + (x0 + lane + a.HX);
  if (!active) return true;   // (still takes part in the reduction barriers; its sums are zero)
#pragma unroll
  for (int r = 0; r < 4; ++r) {
#pragma unroll
    for (int k = 0; k < DIM; ++k) {
      const double2 xu = sm[k * tsz + own0 + r * a.SX];
      p.xo[r][k] = xu.x;
      p.uo[r][k] = xu.y;
    }
  }
  for (int c = a.cbeg[sp]; c < a.cbeg[sp + 1]; ++c) {
    const LatCol8 col = a.cols[c];
    const int n = col.n;
    const uint32_t nmask = (1u << n) - 1u;
    uint32_t bits[4], nfb[4] = {0, 0, 0, 0}, clr[4] = {0, 0, 0, 0};
#pragma unroll
    for (int r = 0; r < 4; ++r) bits[r] = (smask[col.word * NT + tn0 + r * 32] >> col.bit0) & nmask;
    const bool full = __all_sync(FULL, (bits[0] & bits[1] & bits[2] & bits[3]) == nmask);
    bool slow = !full;
    const int base = own0 + col.off;
    if (!slow) {
      p.fast_begin();
      lat_run_col<false, NPAIR>(p, sm, tsz, base, a.SX, n, bits, nfb, clr);
      slow = p.fast_failed();
    }
    if (slow) {
      if (P::kFrac && a.nofail) {
#pragma unroll
        for (int r = 0; r < 4; ++r) nfb[r] = (a.nofail[(int64_t)col.word * a.npad + inode[r]] >> col.bit0) & nmask;
      }
      lat_run_col<true, NPAIR>(p, sm, tsz, base, a.SX, n, bits, nfb, clr);
      if (P::kFrac) {
        uint32_t anyclr = 0;
#pragma unroll
        for (int r = 0; r < 4; ++r) {
          if (clr[r]) atomicAnd(&smask[col.word * NT + tn0 + r * 32], ~(clr[r] << col.bit0));
          anyclr |= clr[r];
        }
        if (anyclr) *sflag = 1;
      }
    }
  }
  return true;
}

// partial sums of the NSPLIT warps of a row group are added through shared memory (the tile is dead by then)
template <int NACC>
__device__ __forceinline__ void lat_reduce(const LatArgs &a, double *red, int rg, int sp, double (&acc)[NACC]) {
  const int lane = threadIdx.x & 31;
  __syncthreads();   // every warp is done reading the tile
  if (a.nsplit > 1) {
    if (sp > 0) {
#pragma unroll
      for (int q = 0; q < NACC; ++q) red[((rg * (a.nsplit - 1) + sp - 1) * NACC + q) * 32 + lane] = acc[q];
    }
    __syncthreads();
    if (sp == 0) {
      for (int s2 = 1; s2 < a.nsplit; ++s2)
#pragma unroll
        for (int q = 0; q < NACC; ++q) acc[q] += red[((rg * (a.nsplit - 1) + s2 - 1) * NACC + q) * 32 + lane];
    }
  }
}

// broken bits back to HBM (only if some bond of the tile broke in this pass)
__device__ __forceinline__ void lat_flush_masks(const LatArgs &a, const uint32_t *smask, const int *sflag, int NT) {
  if (!*sflag) return;
  const int xc = blockIdx.x, yt = blockIdx.y, zt = blockIdx.z;
  const int x0 = xc * 32, y0 = yt * a.TY, z0 = zt * a.TZ;
  const int tyshift = a.TY == 8 ? 3 : 2;
  for (int w = 0; w < a.nw; ++w)
    for (int tn = threadIdx.x; tn < NT; tn += blockDim.x) {
      const int x = tn & 31, row = tn >> 5, y = row & (a.TY - 1), z = row >> tyshift;
      const int64_t i = ((int64_t)(z0 + z + a.HZ) * a.DY + (y0 + y + a.HY)) * a.DX + (x0 + x + a.HX);
      a.mask[(int64_t)w * a.npad + i] = smask[w * NT + tn];
    }
}

template <int DIM, bool FRAC, int MAXT>
__global__ void __launch_bounds__(MAXT) k_lat_dilatation(const __grid_constant__ LatArgs a) {
  extern __shared__ __align__(16) double2 sm[];
  const int lane = threadIdx.x & 31;
  pdb::DilPolicy<DIM, FRAC, true, 4> p;
  p.s_c = a.s_c;
#pragma unroll
  for (int r = 0; r < 4; ++r) p.acc[r] = 0.0;
  int64_t inode[4];
  int rg, sp, NT;
  uint32_t *smask;
  int *sflag;
  if (!lat_tile<DIM, DIM, MAXT>(p, a, sm, inode, rg, sp, smask, sflag, NT)) return;
  // the mask words must leave shared memory before the reduction reuses it
  __syncthreads();
  if (FRAC) lat_flush_masks(a, smask, sflag, NT);
  lat_reduce<4>(a, (double *)sm, rg, sp, p.acc);
  if (sp != 0) return;
#pragma unroll
  for (int r = 0; r < 4; ++r) {
    const int64_t i = inode[r];
    const double mi = a.minv[i];   // 0 for phantoms
    const double theta = a.A * mi * (p.acc[r] * a.vol_uniform);
    a.nbw[(int64_t)PD_P_AUX * a.npad + i] = make_double2(a.G * mi, a.c1 * theta * mi);
    if (a.theta_out) a.theta_out[i] = theta;
  }
  (void)lane;
}

template <int DIM, int MAXT>
__global__ void __launch_bounds__(MAXT) k_lat_force_update(const __grid_constant__ LatArgs a) {
  extern __shared__ __align__(16) double2 sm[];
  pdb::ForcePolicy<DIM, true, 4> p;
#pragma unroll
  for (int r = 0; r < 4; ++r) {
    p.gmu_i[r] = p.cth_i[r] = 0.0;
#pragma unroll
    for (int k = 0; k < DIM; ++k) { p.f[r][k] = 0.0; p.xo[r][k] = p.uo[r][k] = 0.0; }
  }
  int64_t inode[4];
  int rg, sp, NT;
  uint32_t *smask;
  int *sflag;
  // own aux pair {G/m_i, cth_i}: read from HBM before the tile walk (coalesced; the copy in the tile is the same data)
  {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int xc = blockIdx.x, yt = blockIdx.y, zt = blockIdx.z;
    const int nrgy = a.TY >> 2;
    const int rg0 = warp / a.nsplit, rgy = rg0 % nrgy, rgz = rg0 / nrgy;
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      const int64_t i = ((int64_t)(zt * a.TZ + rgz + a.HZ) * a.DY + (yt * a.TY + rgy * 4 + r + a.HY)) * a.DX + (xc * 32 + lane + a.HX);
      const double2 g = a.nbr[(int64_t)PD_P_AUX * a.npad + i];
      p.gmu_i[r] = g.x;
      p.cth_i[r] = g.y;
    }
  }
  if (!lat_tile<DIM, DIM + 1, MAXT>(p, a, sm, inode, rg, sp, smask, sflag, NT)) return;
  double acc[4 * DIM];
#pragma unroll
  for (int r = 0; r < 4; ++r)
#pragma unroll
    for (int k = 0; k < DIM; ++k) acc[r * DIM + k] = p.f[r][k];
  lat_reduce<4 * DIM>(a, (double *)sm, rg, sp, acc);
  if (sp != 0) return;
  // ---- Eq. 2.11 + boundary dofs (App. B) ----
  double g = 1.0;
  if (a.ramp_time > 0.0) g = fmin(1.0, __ddiv_rn(__dmul_rn((double)a.step, a.dt), a.ramp_time));
#pragma unroll
  for (int r = 0; r < 4; ++r) {
    const int64_t i = inode[r];
    if (a.perm[i] < 0) continue;   // phantom
    const unsigned fl = a.flags[i];
#pragma unroll
    for (int k = 0; k < DIM; ++k) {
      const double fk = acc[r * DIM + k] * a.vol_uniform;
      double vk = a.v[k][i];
      double uk = p.uo[r][k];
      if (fl & (1u << k)) {                       // clamped: u stays, v = 0
        vk = 0.0;
      } else if (fl & (8u << k)) {                // prescribed velocity
        vk = a.bval[k][i];
        uk = __dadd_rn(uk, __dmul_rn(a.dt, vk));
      } else {
        const double bk = (fl & PD_BODY_FORCE) ? a.bval[k][i] : 0.0;
        const double ac = __ddiv_rn(__dadd_rn(fk, __dmul_rn(g, bk)), a.rho);
        vk = __dadd_rn(vk, __dmul_rn(a.dt, ac));
        uk = __dadd_rn(uk, __dmul_rn(a.dt, vk));
      }
      a.v[k][i] = vk;
      a.nbw[(int64_t)k * a.npad + i] = make_double2(p.xo[r][k], uk);
    }
  }
}

}  // namespace

namespace {

// phi_i = 1 - sum_j rho_ij V_j / sum_j V_j (Eq. 1.31) and the three damage scalars
__global__ void k_lat_damage(int64_t npad, int nw, double vol_uniform, const int32_t *__restrict__ perm,
                             const uint32_t *__restrict__ mask, const int32_t *__restrict__ rowlen,
                             const double *__restrict__ fvol, double *phi_out, unsigned long long *stats) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  unsigned long long broken = 0, ge_half = 0;
  double phimax = 0.0;
  if (i < npad && perm[i] >= 0) {
    int cnt = 0;
    for (int w = 0; w < nw; ++w) cnt += __popc(mask[(int64_t)w * npad + i]);
    double sum = 0.0;   // the sum of cnt equal volumes, added one by one like sum_j V_j was
    for (int q = 0; q < cnt; ++q) sum += vol_uniform;
    const double phi = 1.0 - sum / fvol[i];
    phi_out[i] = phi;
    broken = (unsigned long long)(rowlen[i] - cnt);
    ge_half = phi >= 0.5 ? 1ull : 0ull;
    phimax = phi;
  }
  unsigned long long pbits = (unsigned long long)__double_as_longlong(fmax(phimax, 0.0));  // phi >= 0: bit order = value order
  for (int o = 16; o > 0; o >>= 1) {
    broken += __shfl_xor_sync(FULL, broken, o);
    ge_half += __shfl_xor_sync(FULL, ge_half, o);
    unsigned long long other = __shfl_xor_sync(FULL, pbits, o);
    pbits = other > pbits ? other : pbits;
  }
  if ((threadIdx.x & 31) == 0) {
    if (broken) atomicAdd(&stats[0], broken);
    if (pbits) atomicMax(&stats[1], pbits);
    if (ge_half) atomicAdd(&stats[2], ge_half);
  }
}

int env_int(const char *name, int dflt) {
  const char *e = getenv(name);
  return e ? atoi(e) : dflt;
}

// tile shape, column table (shared-memory offsets, split between the warps of a row group) and pointers
// npair = records pairs staged per node.  Returns the dynamic shared-memory size, 0 if nothing fits.
size_t lat_make_args(pd_sim *s, LatArgs &a, int npair, int TY, int TZ, int nsplit) {
  const PdLattice &l = s->lat;
  a.DX = l.DX; a.DY = l.DY; a.HX = l.HX; a.HY = l.HY; a.HZ = l.HZ;
  a.TY = TY; a.TZ = TZ;
  a.SX = 32 + 2 * l.HX; a.SY = TY + 2 * l.HY; a.SZ = TZ + 2 * l.HZ;
  a.nxc = l.PX / 32; a.nyt = (l.PY + TY - 1) / TY; a.nyq = (l.PY + 8) / 4;
  a.nsplit = nsplit; a.nw = l.nw;
  a.npad = s->npad;
  for (int q = 0; q < 4; ++q) a.fullw[q] = l.fullw[q];
  // greedy balance of the columns over the splits (by steps), longest first
  std::vector<int> order(l.ncol), owner(l.ncol), load(nsplit, 0);
  for (int c = 0; c < l.ncol; ++c) order[c] = c;
  std::stable_sort(order.begin(), order.end(), [&](int x, int y) { return l.cols[x].n > l.cols[y].n; });
  for (int c : order) {
    int best = 0;
    for (int q = 1; q < nsplit; ++q) if (load[q] < load[best]) best = q;
    owner[c] = best;
    load[best] += l.cols[c].n + 1;
  }
  int k = 0;
  for (int q = 0; q < nsplit; ++q) {
    a.cbeg[q] = k;
    for (int c = 0; c < l.ncol; ++c)
      if (owner[c] == q) {
        const PdLatCol &src = l.cols[c];
        a.cols[k].off = (src.dz * a.SY + src.dy0) * a.SX + src.dx;
        a.cols[k].n = src.n; a.cols[k].word = src.word; a.cols[k].bit0 = src.bit0; a.cols[k].pad = 0;
        ++k;
      }
  }
  for (int q = nsplit; q < 5; ++q) a.cbeg[q] = k;
  a.nbr = s->nb[s->cur]; a.nbw = s->nb[s->cur];
  a.mask = l.mask; a.nofail = l.nofail; a.rgocc = l.rgocc; a.minv = s->minv;
  for (int q = 0; q < 3; ++q) { a.v[q] = s->v[q]; a.bval[q] = s->bval[q]; }
  a.theta_out = nullptr; a.flags = s->flags; a.perm = s->perm;
  a.A = s->A; a.c1 = s->c1; a.G = s->G; a.s_c = s->s_c; a.vol_uniform = s->vol_uniform; a.rho = s->rho; a.dt = s->dt;
  a.ramp_time = s->ramp_time; a.step = s->step;
  const size_t tile = (size_t)npair * a.SZ * a.SY * a.SX * sizeof(double2);
  return tile + 4 * a.SX * sizeof(double2) + 4 * (size_t)(32 * TY * TZ) * sizeof(uint32_t) + 64;
}

constexpr size_t SMEM_MAX = 232448;   // 227 KB opt-in per CTA on sm_100

// largest tile that fits: TZ from the preferred value down; TY = 4 (one row group along y) unless 2-D
bool lat_pick(pd_sim *s, LatArgs &a, int npair, const char *env_prefix, int &TY, int &TZ, int &nsplit, size_t &smem) {
  const int dim = s->dim;
  char nm[64];
  snprintf(nm, sizeof nm, "%s_TY", env_prefix); TY = env_int(nm, dim == 3 ? 4 : 8);
  snprintf(nm, sizeof nm, "%s_TZ", env_prefix); TZ = env_int(nm, dim == 3 ? 4 : 1);
  snprintf(nm, sizeof nm, "%s_NSPLIT", env_prefix); nsplit = env_int(nm, 0);
  if (TY != 4 && TY != 8) TY = 4;
  if (dim == 2) TZ = 1;
  TZ = std::max(1, std::min(TZ, 8));
  for (;; --TZ) {
    smem = lat_make_args(s, a, npair, TY, TZ, 1);
    if (smem <= SMEM_MAX) break;
    if (TZ == 1) { if (TY == 8) { TY = 4; TZ = 2; continue; } return false; }
  }
  const int nrg = (TY / 4) * TZ;
  if (nsplit <= 0) nsplit = std::max(1, std::min(4, 12 / nrg));   // about 8-12 warps per CTA
  nsplit = std::max(1, std::min(nsplit, 4));
  smem = lat_make_args(s, a, npair, TY, TZ, nsplit);
  return true;
}

template <typename K>
int lat_launch(K kernel, pd_sim *s, const LatArgs &a, int TY, int TZ, int nsplit, size_t smem) {
  const PdLattice &l = s->lat;
  const int nzt = (l.PZ + TZ - 1) / TZ;
  const dim3 grid((unsigned)a.nxc, (unsigned)a.nyt, (unsigned)nzt);
  const unsigned threads = (unsigned)((TY / 4) * TZ * nsplit * 32);
  PD_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  kernel<<<grid, threads, smem, s->stream>>>(a);
  return PD_OK;
}

}  // namespace

namespace pdi {

int lat_launch_dilatation(pd_sim *s, double *theta_out, bool do_break) {
  LatArgs a;
  int TY, TZ, nsplit;
  size_t smem;
  if (!lat_pick(s, a, s->dim, "PD_LAT_DIL", TY, TZ, nsplit, smem)) { set_error("lattice tile does not fit shared memory"); return PD_ERR_LIMIT; }
  a.theta_out = theta_out;
  const bool frac = do_break && s->fracture;
  constexpr int MT = 384;
  if ((TY / 4) * TZ * nsplit * 32 > MT) { set_error("lattice dilatation: too many threads per tile"); return PD_ERR_LIMIT; }
  if (s->dim == 2) return frac ? lat_launch(k_lat_dilatation<2, true, MT>, s, a, TY, TZ, nsplit, smem)
                               : lat_launch(k_lat_dilatation<2, false, MT>, s, a, TY, TZ, nsplit, smem);
  return frac ? lat_launch(k_lat_dilatation<3, true, MT>, s, a, TY, TZ, nsplit, smem)
              : lat_launch(k_lat_dilatation<3, false, MT>, s, a, TY, TZ, nsplit, smem);
}

int lat_launch_force_update(pd_sim *s) {
  LatArgs a;
  int TY, TZ, nsplit;
  size_t smem;
  if (!lat_pick(s, a, s->dim + 1, "PD_LAT_FRC", TY, TZ, nsplit, smem)) { set_error("lattice tile does not fit shared memory"); return PD_ERR_LIMIT; }
  a.nbw = s->nb[s->cur ^ 1];
  constexpr int MT = 384;
  while ((TY / 4) * TZ * nsplit * 32 > MT && nsplit > 1) { --nsplit; smem = lat_make_args(s, a, s->dim + 1, TY, TZ, nsplit); a.nbw = s->nb[s->cur ^ 1]; }
  if ((TY / 4) * TZ * nsplit * 32 > MT) { set_error("lattice force: too many threads per tile"); return PD_ERR_LIMIT; }
  if (s->dim == 2) return lat_launch(k_lat_force_update<2, MT>, s, a, TY, TZ, nsplit, smem);
  return lat_launch(k_lat_force_update<3, MT>, s, a, TY, TZ, nsplit, smem);
}

int lat_launch_damage(pd_sim *s) {
  cudaMemsetAsync(s->stats_dev, 0, 3 * sizeof(unsigned long long), s->stream);
  k_lat_damage<<<nblk(s->npad), TPB, 0, s->stream>>>(s->npad, s->lat.nw, s->vol_uniform, s->perm, s->lat.mask, s->rowlen,
                                                     s->fvol, s->phi, s->stats_dev);
  return PD_OK;
}

}  // namespace pdi
