// pd_build.cu -- GPU cell-list family builder.
//
// Runs once in pd_create, entirely on the device:
//   1. bounding box; node spacing from the median nearest-neighbour distance of a node sample;
//      uniform cell grid whose edge per dimension is extent/round(extent/spacing), origin shifted by
//      half a cell: on a (jittered) lattice body every cell holds exactly one node.  Nothing below
//      depends on that for correctness -- any point cloud gives the right families, a lattice
//      (the paper's discretisation) gives the compact layout.
//   2. radix sort by cell id (z, y, x) -> every (z, y) CELL ROW is a run sorted along x
//   3. final node order: a TILE = (BZ z-levels) x (R cell rows in y) x (32 cells in x, counted from
//      the first occupied cell of the tile row); lane = x cell inside the tile (nodes sharing a
//      cell are pushed to the next free lane).  Tiles that hold a node are numbered in raster
//      order; slice = tile*BZ*R + (z % BZ)*R + (y % R), final index = slice*32 + lane.  Absent
//      nodes are phantoms.  Lane l of a group (= R slices = one warp) therefore owns R nodes that
//      are adjacent in y at the same x: their families overlap, so one gathered neighbour
//      serves up to R bonds (register blocking of the neighbour list).
//   4. count pass -> entries per group -> exclusive scan -> group offsets ("SELL-32xR")
//   5. fill pass  -> col (neighbour element index per entry), member bits, m_i (Eq. 1.9), sum_j V_j
//   6. pre-cut pairs clear their two intact bits; no-fail bit mask (only if some node is no-fail)
// Passes 4 and 5 run one warp per group in LOCKSTEP over the cells of a box around the lanes'
// nominal cells: an entry is created for (relative cell, k-th node in it) whenever that node is a
// family member for ANY lane, and lanes without a bond there get a padding entry.  So all lanes of
// a warp meet the same relative neighbour in the same entry: the gathers of an entry are
// contiguous, and which (entry, r) pairs are bonds is warp-uniform in the bulk.
// The horizon test is ||xi||^2 <= horizon^2 (inclusive) with the products and
// sums rounded individually in component order (no FMA contraction), so it is reproducible.
#include <cub/device/device_radix_sort.cuh>
#include <cub/device/device_reduce.cuh>
#include <cub/device/device_scan.cuh>
#include <cub/iterator/transform_input_iterator.cuh>

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>

#include "pd_internal.cuh"

namespace {

constexpr int TPB = 256;

using Grid = PdGrid;

__device__ __forceinline__ void cell_of(const Grid &g, const double *p, int *q) {
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    if (k < g.dim) {
      int c = (int)floor((p[k] - g.lo[k]) * g.inv_c[k] + 0.5);
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
  __shared__ unsigned long long sh[8];
  if (threadIdx.x < 8) sh[threadIdx.x] = (threadIdx.x < 3 || threadIdx.x == 6) ? ~0ull : 0ull;
  __syncthreads();
  unsigned long long mn[4] = {~0ull, ~0ull, ~0ull, ~0ull}, mx[4] = {0, 0, 0, 0};
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    for (int k = 0; k < dim; ++k) {
      unsigned long long e = enc(coords[dim * i + k]);
      mn[k] = min(mn[k], e);
      mx[k] = max(mx[k], e);
    }
    unsigned long long ev = enc(vol[i]);
    mn[3] = min(mn[3], ev);
    mx[3] = max(mx[3], ev);
  }
  for (int k = 0; k < 4; ++k)
    for (int o = 16; o > 0; o >>= 1) {
      mn[k] = min(mn[k], __shfl_xor_sync(0xffffffffu, mn[k], o));
      mx[k] = max(mx[k], __shfl_xor_sync(0xffffffffu, mx[k], o));
    }
  if ((threadIdx.x & 31) == 0) {
    for (int k = 0; k < 3; ++k) { atomicMin(&sh[k], mn[k]); atomicMax(&sh[3 + k], mx[k]); }
    atomicMin(&sh[6], mn[3]);
    atomicMax(&sh[7], mx[3]);
  }
  __syncthreads();
  if (threadIdx.x < 8) {
    if (threadIdx.x < 3 || threadIdx.x == 6) atomicMin(&out[threadIdx.x], sh[threadIdx.x]);
    else atomicMax(&out[threadIdx.x], sh[threadIdx.x]);
  }
}

// nearest-neighbour distance^2 of sample nodes (brute force; one block per sample)
__global__ void k_nn_sample(int64_t n, int dim, const double *__restrict__ coords, int64_t stride, double *out) {
  const int64_t i = (int64_t)blockIdx.x * stride;
  double pi[3] = {0, 0, 0};
  for (int k = 0; k < dim; ++k) pi[k] = coords[dim * i + k];
  double best = 1.0e300;
  for (int64_t j = threadIdx.x; j < n; j += blockDim.x) {
    double r2 = 0.0;
    for (int k = 0; k < dim; ++k) { double d = coords[dim * j + k] - pi[k]; r2 += d * d; }
    if (j != i && r2 > 0.0) best = fmin(best, r2);
  }
  __shared__ double sh[TPB / 32];
  for (int o = 16; o > 0; o >>= 1) best = fmin(best, __shfl_xor_sync(0xffffffffu, best, o));
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = best;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < TPB / 32; ++w) best = fmin(best, sh[w]);
    out[blockIdx.x] = best;
  }
}

// ---- 2. sort keys: raster cell id, x fastest ------------------------------------------------------
__global__ void k_keys(int64_t n, Grid g, const double *__restrict__ coords, uint32_t *keys, int32_t *ids) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double p[3] = {0, 0, 0};
  for (int k = 0; k < g.dim; ++k) p[k] = coords[g.dim * i + g.ax[k]];
  int q[3];
  cell_of(g, p, q);
  keys[i] = (uint32_t)(((int64_t)q[2] * g.nc[1] + q[1]) * g.nc[0] + q[0]);
  ids[i] = (int32_t)i;
}

// cell and row tables over the sorted keys (start/end positions; empty = 0/0)
__global__ void k_tables(int64_t n, int ncx, const uint32_t *__restrict__ keys, int32_t *cell_start, int32_t *cell_end,
                         int32_t *row_start, int32_t *row_end) {
  int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n) return;
  uint32_t c = keys[p];
  uint32_t cp = p > 0 ? keys[p - 1] : 0xffffffffu, cn = p + 1 < n ? keys[p + 1] : 0xffffffffu;
  if (p == 0 || c != cp) cell_start[c] = (int32_t)p;
  if (p + 1 == n || c != cn) cell_end[c] = (int32_t)(p + 1);
  uint32_t r = c / ncx;
  if (p == 0 || r != cp / ncx) row_start[r] = (int32_t)p;
  if (p + 1 == n || r != cn / ncx) row_end[r] = (int32_t)(p + 1);
}

// t_p = cx_p - rank_p: its running maximum along a row places nodes that share a cell on the next free lane
__global__ void k_row_t(int64_t n, int ncx, const uint32_t *__restrict__ keys, const int32_t *__restrict__ row_start,
                        int32_t *rowid, int32_t *t) {
  int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n) return;
  uint32_t c = keys[p];
  int32_t row = (int32_t)(c / ncx);
  rowid[p] = row;
  t[p] = (int32_t)(c % ncx) - (int32_t)(p - row_start[row]);
}

// first occupied x cell of every tile row = (BZ z-levels) x (R cell rows)
__global__ void k_tilerow_x0(int64_t ntr, Grid g, const uint32_t *__restrict__ keys, const int32_t *__restrict__ row_start,
                             const int32_t *__restrict__ row_end, int32_t *x0) {
  int64_t tr = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (tr >= ntr) return;
  int yg = (int)(tr % g.ncyg), zt = (int)(tr / g.ncyg);
  int best = 0x7fffffff;
  for (int dz = 0; dz < g.BZ; ++dz)
    for (int dy = 0; dy < g.R; ++dy) {
      int cz = zt * g.BZ + dz, cy = yg * g.R + dy;
      if (cz >= g.nc[2] || cy >= g.nc[1]) continue;
      int64_t row = (int64_t)cz * g.nc[1] + cy;
      if (row_end[row] > row_start[row]) best = min(best, (int)(keys[row_start[row]] % g.nc[0]));
    }
  x0[tr] = best;
}

// virtual x (lane + 32*chunk) of every node inside its tile row, and its maximum
__global__ void k_vx(int64_t n, Grid g, const int32_t *__restrict__ rowid, const int32_t *__restrict__ row_start,
                     const int32_t *__restrict__ tmax, const int32_t *__restrict__ x0, int32_t *vx, int *maxvx) {
  int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  int v = 0;
  if (p < n) {
    int row = rowid[p];
    int cy = row % g.nc[1], cz = row / g.nc[1];
    int64_t tr = (int64_t)(cz / g.BZ) * g.ncyg + cy / g.R;
    v = (int)(p - row_start[row]) + tmax[p] - x0[tr];
    vx[p] = v;
  }
  for (int o = 16; o > 0; o >>= 1) v = max(v, __shfl_xor_sync(0xffffffffu, v, o));
  if ((threadIdx.x & 31) == 0) atomicMax(maxvx, v);
}

__device__ __forceinline__ int64_t tile_dense_of(const Grid &g, int row, int vx) {
  int cy = row % g.nc[1], cz = row / g.nc[1];
  return ((int64_t)(cz / g.BZ) * g.ncyg + cy / g.R) * g.maxchunk + (vx >> 5);
}

__global__ void k_tile_mark(int64_t n, Grid g, const int32_t *__restrict__ rowid, const int32_t *__restrict__ vx,
                            int32_t *flag) {
  int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n) return;
  flag[tile_dense_of(g, rowid[p], vx[p])] = 1;
}

__global__ void k_final_index(int64_t n, Grid g, const int32_t *__restrict__ rowid, const int32_t *__restrict__ vx,
                              const int32_t *__restrict__ ord1, const int32_t *__restrict__ tile_ord,
                              int32_t *tile_inv, int32_t *fin1, int32_t *perm, int32_t *iperm) {
  int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n) return;
  int row = rowid[p];
  int cy = row % g.nc[1], cz = row / g.nc[1];
  int64_t td = tile_dense_of(g, row, vx[p]);
  int32_t t = tile_ord[td];
  tile_inv[t] = (int32_t)td;
  int64_t slice = (int64_t)t * (g.BZ * g.R) + (cz % g.BZ) * g.R + (cy % g.R);
  int32_t fin = (int32_t)(slice * 32 + (vx[p] & 31));
  fin1[p] = fin;
  int32_t uidx = ord1[p];
  perm[fin] = uidx;
  iperm[uidx] = fin;
}

// node data in final order (arrays pre-zeroed; phantoms stay zero): reference positions into the x half
// of the position pairs of BOTH neighbour-record buffers, volumes, flags
__global__ void k_records(int64_t npad, Grid g, const int32_t *__restrict__ perm, const double *__restrict__ coords,
                          const double *__restrict__ vol, const uint8_t *__restrict__ flags, double2 *nb0, double2 *nb1,
                          double *volF, uint8_t *flagsF) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= npad) return;
  int32_t uidx = perm[i];
  if (uidx < 0) return;
  const int dim = g.dim;
  const uint32_t e = pd_elem(i);
  for (int k = 0; k < dim; ++k) {
    const double x = coords[(int64_t)dim * uidx + g.ax[k]];
    nb0[e + 32 * k].x = x;
    nb1[e + 32 * k].x = x;
  }
  volF[i] = vol[uidx];
  unsigned f = flags ? flags[uidx] : 0u, fi = f & 0xC0u;   // per-dof bits move with their component
  for (int k = 0; k < dim; ++k) {
    if (f & (1u << g.ax[k])) fi |= 1u << k;
    if (f & (8u << g.ax[k])) fi |= 8u << k;
  }
  flagsF[i] = (uint8_t)fi;
}

// ---- 4./5. lockstep family traversal of one group (one warp; lane = 4 nodes) -----------------------
// The group's neighbourhood is walked COLUMN by column: a column = the cells (cz, bx + dx, *) along
// internal axis 1 (the axis along which the lane's 4 rows are adjacent).  Per column and lane the
// bond bits of every cell are found by the exact distance test; then
//   * if no lane meets a cell with more than one node: SHIFT segments.  With c the cell index along
//     the column, bond (row r, cell c) belongs to step T = c - r; steps that are a bond for no lane
//     are dropped, runs of consecutive steps are cut into segments of <= 7 steps, a segment of n
//     steps lists the n + 3 cells T0 .. T0 + n + 2 as entries (lanes without a node there get
//     their own node 0 and no bit);
//   * otherwise FLAT segments: one entry per (cell, k-th node in it) that is a bond for some lane.
// All lanes of a warp meet the same relative neighbour in the same entry, so the gathers of an
// entry are contiguous and the segment structure (the CODE nibble) is warp-uniform.
constexpr int MAXCY = 32;   // cells scanned per column: 4 + 2 S[1] <= 32 (S <= 9 because cell edge >= horizon/8)

struct GroupOut {
  int ecnt = 0, scnt = 0;
  int rl[PD_R] = {0, 0, 0, 0};
  double m[PD_R] = {0, 0, 0, 0}, fv[PD_R] = {0, 0, 0, 0};
};

template <bool FILL>
__device__ __forceinline__ void scan_group(const Grid &g, int64_t grp, int lane, double h2,
                                           const double2 *__restrict__ nb0, const double *__restrict__ vol,
                                           const int32_t *__restrict__ perm,
                                           const int32_t *__restrict__ cell_start,
                                           const int32_t *__restrict__ cell_end,
                                           const int32_t *__restrict__ fin1,
                                           const int32_t *__restrict__ tile_inv,
                                           const int32_t *__restrict__ tile_x0, uint32_t *colp, uint32_t *memp,
                                           GroupOut &o) {
  constexpr unsigned FULL = 0xffffffffu;
  constexpr int R = PD_R;
  // nominal cell of the lane
  const int64_t td = tile_inv[grp / g.BZ];
  const int chunk = (int)(td % g.maxchunk);
  const int64_t tr = td / g.maxchunk;
  const int by0 = (int)(tr % g.ncyg) * R, bz = (int)(tr / g.ncyg) * g.BZ + (int)(grp % g.BZ);
  const int bx = tile_x0[tr] + 32 * chunk + lane;
  const uint32_t self = pd_elem(grp * R * 32 + lane);
  double pi[R][3];
  int64_t ir[R];
  unsigned valid = 0;
  int dl = 1 << 30, dh = -(1 << 30);
#pragma unroll
  for (int r = 0; r < R; ++r) {
    ir[r] = (grp * R + r) * 32 + lane;
    pi[r][0] = pi[r][1] = pi[r][2] = 0.0;
    if (perm[ir[r]] >= 0) {
      valid |= 1u << r;
      const double2 *p = nb0 + pd_elem(ir[r]);
      for (int k = 0; k < g.dim; ++k) pi[r][k] = p[32 * k].x;
      int q[3];
      cell_of(g, pi[r], q);
      dl = min(dl, q[0] - bx);
      dh = max(dh, q[0] - bx);
    }
  }
  for (int s = 16; s > 0; s >>= 1) {
    dl = min(dl, __shfl_xor_sync(FULL, dl, s));
    dh = max(dh, __shfl_xor_sync(FULL, dh, s));
  }
  if (dh < dl) return;  // no node in this group
  const int z0 = g.dim > 2 ? max(bz - g.S[2], 0) : 0, z1 = g.dim > 2 ? min(bz + g.S[2], g.nc[2] - 1) : 0;
  const int y0 = max(by0 - g.S[1], 0), y1 = min(by0 + R - 1 + g.S[1], g.nc[1] - 1);
  const int ny = min(y1 - y0 + 1, MAXCY);

  auto bond_bits = [&](int64_t j, double *r2) -> unsigned {
    unsigned bits = 0;
    const double2 *q = nb0 + pd_elem(j);
    double pj[3] = {0, 0, 0};
    for (int k = 0; k < g.dim; ++k) pj[k] = q[32 * k].x;
#pragma unroll
    for (int r = 0; r < R; ++r) {
      r2[r] = dist2_exact(g.dim, pi[r], pj);
      if (((valid >> r) & 1u) && j != ir[r] && r2[r] <= h2) bits |= 1u << r;
    }
    return bits;
  };
  auto emit_entry = [&](int64_t j) {
    if (FILL) colp[(int64_t)o.ecnt * 32] = j >= 0 ? pd_elem(j) : self;
    ++o.ecnt;
  };
  auto emit_seg = [&](unsigned code, uint32_t word) {
    if (FILL) memp[(int64_t)o.scnt * 32] = (code << 28) | word;
    ++o.scnt;
  };
  auto account = [&](int64_t j, unsigned bits, const double *r2) {   // m_i (Eq. 1.9, w = 1), sum_j V_j (Eq. 1.31)
#pragma unroll
    for (int r = 0; r < R; ++r) o.rl[r] += (bits >> r) & 1u;
    if (FILL && bits) {
      const double vj = vol[j];
#pragma unroll
      for (int r = 0; r < R; ++r)
        if ((bits >> r) & 1u) {
          o.m[r] = fma(r2[r], vj, o.m[r]);
          o.fv[r] += vj;
        }
    }
  };

  for (int cz = z0; cz <= z1; ++cz)
    for (int dx = dl - g.S[0]; dx <= dh + g.S[0]; ++dx) {
      const int cx = bx + dx;
      const bool inx = valid && cx >= 0 && cx < g.nc[0];
      // ---- phase 1: bond bits of the first node of every cell of the column ----
      unsigned char bits[MAXCY];
      int jj[MAXCY];
      int maxcnt = 0;
      unsigned anyb = 0;
      for (int c = 0; c < ny; ++c) {
        bits[c] = 0;
        jj[c] = -1;
        if (inx) {
          const int64_t cell = ((int64_t)cz * g.nc[1] + (y0 + c)) * g.nc[0] + cx;
          const int32_t s = cell_start[cell], cnt = cell_end[cell] - s;
          maxcnt = max(maxcnt, cnt);
          if (cnt >= 1) {
            double r2[R];
            jj[c] = fin1[s];
            bits[c] = (unsigned char)bond_bits(jj[c], r2);
            anyb |= bits[c];
          }
        }
      }
      if (!__any_sync(FULL, anyb != 0 || maxcnt > 1)) continue;
      for (int s = 16; s > 0; s >>= 1) maxcnt = max(maxcnt, __shfl_xor_sync(FULL, maxcnt, s));
      if (maxcnt <= 1) {
        // ---- SHIFT segments ----
        int tmin = 1 << 30, tmax = -(1 << 30);
        for (int c = 0; c < ny; ++c)
          for (int r = 0; r < R; ++r)
            if ((bits[c] >> r) & 1u) { tmin = min(tmin, c - r); tmax = max(tmax, c - r); }
        for (int s = 16; s > 0; s >>= 1) {
          tmin = min(tmin, __shfl_xor_sync(FULL, tmin, s));
          tmax = max(tmax, __shfl_xor_sync(FULL, tmax, s));
        }
        auto step_bits = [&](int T) -> unsigned {   // bit r: bond (row r, cell T + r)
          unsigned b = 0;
          for (int r = 0; r < R; ++r) {
            const int c = T + r;
            if (c >= 0 && c < ny && ((bits[c] >> r) & 1u)) b |= 1u << r;
          }
          return b;
        };
        int T = tmin;
        while (T <= tmax) {
          unsigned sb = step_bits(T);
          if (!__any_sync(FULL, sb != 0)) { ++T; continue; }
          const int Ta = T;
          int n = 0;
          uint32_t word = 0;
          while (n < PD_MAXSTEP) {
            word |= sb << (4 * n);
            ++n;
            ++T;
            if (T > tmax) break;
            sb = step_bits(T);
            if (!__any_sync(FULL, sb != 0)) break;
          }
          for (int c = Ta; c < Ta + n + 3; ++c) emit_entry((c >= 0 && c < ny) ? (int64_t)jj[c] : -1);
          emit_seg((unsigned)n, word);
          for (int t = 0; t < n; ++t)
            for (int r = 0; r < R; ++r)
              if ((word >> (4 * t + r)) & 1u) {
                double r2[R];
                const int64_t j = jj[Ta + t + r];
                bond_bits(j, r2);
                account(j, 1u << r, r2);
              }
        }
      } else {
        // ---- FLAT segments: every (cell, k-th node) that is a bond for some lane ----
        int n = 0;
        uint32_t word = 0;
        for (int c = 0; c < ny; ++c) {
          int32_t s = 0, cnt = 0;
          if (inx) {
            const int64_t cell = ((int64_t)cz * g.nc[1] + (y0 + c)) * g.nc[0] + cx;
            s = cell_start[cell];
            cnt = cell_end[cell] - s;
          }
          int mx = cnt;
          for (int q = 16; q > 0; q >>= 1) mx = max(mx, __shfl_xor_sync(FULL, mx, q));
          for (int idx = 0; idx < mx; ++idx) {
            unsigned b = 0;
            double r2[R];
            int64_t j = -1;
            if (idx < cnt) { j = fin1[s + idx]; b = bond_bits(j, r2); }
            if (!__any_sync(FULL, b != 0)) continue;
            emit_entry(b ? j : -1);
            account(j, b, r2);
            word |= b << (4 * n);
            if (++n == PD_MAXSTEP) { emit_seg(8u + n, word); n = 0; word = 0; }
          }
        }
        if (n) emit_seg(8u + n, word);
      }
    }
}

__global__ void k_count(int64_t ngroups, Grid g, double h2, const double2 *__restrict__ nb0,
                        const int32_t *__restrict__ perm, const int32_t *__restrict__ cell_start,
                        const int32_t *__restrict__ cell_end, const int32_t *__restrict__ fin1,
                        const int32_t *__restrict__ tile_inv, const int32_t *__restrict__ tile_x0, int32_t *rowlen,
                        uint32_t *glen, uint32_t *slen) {
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  int64_t grp = t >> 5;
  if (grp >= ngroups) return;
  int lane = threadIdx.x & 31;
  GroupOut o;
  scan_group<false>(g, grp, lane, h2, nb0, nullptr, perm, cell_start, cell_end, fin1, tile_inv, tile_x0, nullptr, nullptr, o);
#pragma unroll
  for (int r = 0; r < PD_R; ++r) rowlen[(grp * PD_R + r) * 32 + lane] = o.rl[r];
  if (lane == 0) { glen[grp] = (uint32_t)o.ecnt; slen[grp] = (uint32_t)o.scnt; }  // the same on all lanes
}

__global__ void k_fill(int64_t ngroups, Grid g, double h2, double G, double2 *__restrict__ nb0, double2 *__restrict__ nb1,
                       const double *__restrict__ vol, double *__restrict__ mF, double *__restrict__ minvF,
                       double *__restrict__ fvolF, const int32_t *__restrict__ perm,
                       const int32_t *__restrict__ cell_start, const int32_t *__restrict__ cell_end,
                       const int32_t *__restrict__ fin1, const int32_t *__restrict__ tile_inv,
                       const int32_t *__restrict__ tile_x0, const uint32_t *__restrict__ goff,
                       const uint32_t *__restrict__ soff, uint32_t *col, uint32_t *member) {
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  int64_t grp = t >> 5;
  if (grp >= ngroups) return;
  int lane = threadIdx.x & 31;
  GroupOut o;
  scan_group<true>(g, grp, lane, h2, nb0, vol, perm, cell_start, cell_end, fin1, tile_inv, tile_x0,
                   col + (int64_t)goff[grp] * 32 + lane, member + (int64_t)soff[grp] * 32 + lane, o);
#pragma unroll
  for (int r = 0; r < PD_R; ++r) {
    int64_t i = (grp * PD_R + r) * 32 + lane;
    if (perm[i] < 0) continue;
    mF[i] = o.m[r];
    fvolF[i] = o.fv[r];
    minvF[i] = o.m[r] > 0.0 ? 1.0 / o.m[r] : 0.0;
    const double gmu = o.m[r] > 0.0 ? G / o.m[r] : 0.0;
    nb0[pd_elem(i) + 32 * PD_P_AUX].x = gmu;
    nb1[pd_elem(i) + 32 * PD_P_AUX].x = gmu;
  }
}

// ---- 6. pre-cuts and no-fail mask ---------------------------------------------------------------
__global__ void k_precut(int64_t np, int64_t n, const int32_t *__restrict__ pairs,
                         const int32_t *__restrict__ iperm, const uint32_t *__restrict__ goff,
                         const uint32_t *__restrict__ soff, const uint32_t *__restrict__ col,
                         const uint32_t *__restrict__ member, uint32_t *seg, unsigned long long *err) {
  int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= 2 * np) return;
  int64_t pa = pairs[2 * (p >> 1) + (p & 1)], pb = pairs[2 * (p >> 1) + 1 - (p & 1)];
  if (pa < 0 || pa >= n || pb < 0 || pb >= n || pa == pb) { atomicExch(err, 1ull); return; }
  int32_t a = iperm[pa];
  const uint32_t eb = pd_elem(iperm[pb]);
  int64_t slice = a >> 5;
  int lane = a & 31, ra = (int)(slice % PD_R);
  int64_t grp = slice / PD_R;
  const uint32_t *c = col + (int64_t)goff[grp] * 32 + lane;
  const uint32_t *mb = member + (int64_t)soff[grp] * 32 + lane;
  uint32_t *sg = seg + (int64_t)soff[grp] * 32 + lane;
  bool found = false;
  pd_for_lane_slots(mb, (int)(soff[grp + 1] - soff[grp]), [&](int s, int bit, int r, int k) {
    if (!found && r == ra && ((mb[(int64_t)s * 32] >> bit) & 1u) && c[(int64_t)k * 32] == eb) {
      atomicAnd(&sg[(int64_t)s * 32], ~(1u << bit));
      found = true;
    }
  });
  if (!found) atomicExch(err, 1ull);  // not a bond
}

__global__ void k_nofail(int64_t ngroups, const uint8_t *__restrict__ flags, const uint32_t *__restrict__ goff,
                         const uint32_t *__restrict__ soff, const uint32_t *__restrict__ col,
                         const uint32_t *__restrict__ member, uint32_t *nofail) {
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  int64_t grp = t >> 5;
  if (grp >= ngroups) return;
  int lane = threadIdx.x & 31;
  const int nseg = (int)(soff[grp + 1] - soff[grp]);
  const uint32_t *c = col + (int64_t)goff[grp] * 32 + lane;
  const uint32_t *mb = member + (int64_t)soff[grp] * 32 + lane;
  uint32_t *nf = nofail + (int64_t)soff[grp] * 32 + lane;
  unsigned fi = 0;  // bit r: node r is no-fail
  for (int r = 0; r < PD_R; ++r)
    if (flags[(grp * PD_R + r) * 32 + lane] & PD_NO_FAIL) fi |= 1u << r;
  for (int s = 0; s < nseg; ++s) nf[(int64_t)s * 32] = mb[(int64_t)s * 32] & 0xf0000000u;
  pd_for_lane_slots(mb, nseg, [&](int s, int bit, int r, int k) {
    if (!((mb[(int64_t)s * 32] >> bit) & 1u)) return;
    if (((fi >> r) & 1u) || (flags[pd_elem_inv(c[(int64_t)k * 32])] & PD_NO_FAIL)) nf[(int64_t)s * 32] |= 1u << bit;
  });
}

__global__ void k_checks(int64_t npad, const int32_t *__restrict__ perm, const int32_t *__restrict__ rowlen,
                         const uint8_t *__restrict__ flags, unsigned long long *out) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= npad || perm[i] < 0) return;
  if (rowlen[i] == 0) atomicOr(&out[0], 1ull);  // some node has an empty family
  unsigned f = flags[i];
  if (f & PD_NO_FAIL) atomicOr(&out[1], 1ull);
  if (f) atomicOr(&out[1], 2ull);
}

__global__ void k_rowlen_user(int64_t n, const int32_t *__restrict__ iperm, const int32_t *__restrict__ rowlen,
                              long long *out) {
  int64_t uidx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (uidx >= n) return;
  out[uidx] = rowlen[iperm[uidx]];
}

__global__ void k_export_rows(int64_t ngroups, const int32_t *__restrict__ perm,
                              const long long *__restrict__ rowptr, const uint32_t *__restrict__ goff,
                              const uint32_t *__restrict__ soff, const uint32_t *__restrict__ col,
                              const uint32_t *__restrict__ member, const uint32_t *__restrict__ seg,
                              int32_t *col_out, uint8_t *intact_out) {
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  int64_t grp = t >> 5;
  if (grp >= ngroups) return;
  int lane = threadIdx.x & 31;
  const int nseg = (int)(soff[grp + 1] - soff[grp]);
  const uint32_t *c = col + (int64_t)goff[grp] * 32 + lane;
  const uint32_t *mb = member + (int64_t)soff[grp] * 32 + lane;
  const uint32_t *sg = seg + (int64_t)soff[grp] * 32 + lane;
  long long base[PD_R];
  for (int r = 0; r < PD_R; ++r) {
    int32_t uidx = perm[(grp * PD_R + r) * 32 + lane];
    base[r] = uidx >= 0 ? rowptr[uidx] : -1;
  }
  pd_for_lane_slots(mb, nseg, [&](int s, int bit, int r, int k) {
    if (base[r] < 0 || !((mb[(int64_t)s * 32] >> bit) & 1u)) return;
    col_out[base[r]] = perm[pd_elem_inv(c[(int64_t)k * 32])];
    intact_out[base[r]] = (uint8_t)((sg[(int64_t)s * 32] >> bit) & 1u);
    ++base[r];
  });
}

inline unsigned nblk(int64_t n) { return (unsigned)((n + TPB - 1) / TPB); }

template <typename T>
int scan_exclusive(pd_sim *s, std::vector<void *> &scratch, const T *in, T *out, int64_t cnt) {
  size_t tb = 0;
  PD_CUDA(cub::DeviceScan::ExclusiveSum(nullptr, tb, in, out, (int)cnt, s->stream));
  void *tmp = pdi::dev_alloc(s, tb ? tb : 1);
  if (!tmp) { pdi::set_error("device allocation failed"); return PD_ERR_ALLOC; }
  scratch.push_back(tmp);
  PD_CUDA(cub::DeviceScan::ExclusiveSum(tmp, tb, in, out, (int)cnt, s->stream));
  return PD_OK;
}

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
  const int R = PD_R;

  // ---- scratch (freed at the end through the same allocator) ----
  std::vector<void *> scratch;
  auto salloc = [&](size_t bytes) -> void * {
    void *p = dev_alloc(s, bytes ? bytes : 1);
    if (p) scratch.push_back(p);
    return p;
  };
  auto sfree_all = [&]() {
    cudaStreamSynchronize(st);
    for (void *p : scratch) dev_free(s, p);
    scratch.clear();
  };
  struct Guard { decltype(sfree_all) &f; ~Guard() { f(); } } guard{sfree_all};
#define SCRATCH(ptr, type, count)                                            \
  type *ptr = (type *)salloc(sizeof(type) * (size_t)(count));                \
  if (!ptr) { set_error("device allocation failed in pd_create"); return PD_ERR_ALLOC; }

  // ---- 1. bbox + volume range ----
  SCRATCH(red, unsigned long long, 8);
  unsigned long long init[8];
  for (int k = 0; k < 3; ++k) { init[k] = ~0ull; init[3 + k] = 0ull; }
  init[6] = ~0ull; init[7] = 0ull;
  PD_CUDA(cudaMemcpyAsync(red, init, sizeof(init), cudaMemcpyHostToDevice, st));
  k_bbox<<<std::min<unsigned>(nblk(n), 1184u), TPB, 0, st>>>(n, dim, coords, vol, red);
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

  // ---- node spacing: median nearest-neighbour distance of up to 1024 sample nodes ----
  double spacing = s->horizon;
  {
    const int nsamp = (int)std::min<int64_t>(n, 1024);
    SCRATCH(nn_d, double, nsamp);
    k_nn_sample<<<nsamp, TPB, 0, st>>>(n, dim, coords, n / nsamp, nn_d);
    std::vector<double> nn(nsamp);
    PD_CUDA(cudaMemcpyAsync(nn.data(), nn_d, sizeof(double) * nsamp, cudaMemcpyDeviceToHost, st));
    PD_CUDA(cudaStreamSynchronize(st));
    std::vector<double> ok;
    for (double v : nn) if (v > 0.0 && v < 1.0e299 && std::isfinite(v)) ok.push_back(std::sqrt(v));
    if (!ok.empty()) {
      std::nth_element(ok.begin(), ok.begin() + ok.size() / 2, ok.end());
      spacing = ok[ok.size() / 2];
    }
  }
  // ---- cell grid: edge_k = extent_k / round(extent_k / spacing), kept inside [horizon/8, horizon];
  //      cell index = round((x - lo)/edge): a lattice node sits in the middle of its own cell ----
  spacing = std::min(std::max(spacing, s->horizon / 8.0), s->horizon);
  // lane axis = the axis whose cell count fills whole 32-lane chunks best (ties: the longer one)
  {
    int best = 0;
    double bfill = -1.0, bcnt = 0.0;
    for (int k = 0; k < dim; ++k) {
      double cnt = std::floor((hi[k] - lo[k]) / spacing + 0.5) + 1.0;
      double fill = cnt / (32.0 * std::ceil(cnt / 32.0));
      if (fill > bfill + 1e-12 || (std::fabs(fill - bfill) <= 1e-12 && cnt > bcnt)) { best = k; bfill = fill; bcnt = cnt; }
    }
    if (const char *env = getenv("PD_LANE_AXIS")) { int a = atoi(env); if (a >= 0 && a < dim) best = a; }
    int q = 0;
    s->ax[q++] = best;
    for (int k = 0; k < dim; ++k) if (k != best) s->ax[q++] = k;
    for (; q < 3; ++q) s->ax[q] = q;
    double lo2[3] = {0, 0, 0}, hi2[3] = {0, 0, 0};
    for (int k = 0; k < dim; ++k) { lo2[k] = lo[s->ax[k]]; hi2[k] = hi[s->ax[k]]; }
    for (int k = 0; k < 3; ++k) { lo[k] = lo2[k]; hi[k] = hi2[k]; }
  }
  Grid g{};
  g.dim = dim;
  for (int k = 0; k < 3; ++k) g.ax[k] = s->ax[k];
  for (;;) {
    double ncell = 1.0;
    for (int k = 0; k < 3; ++k) {
      g.lo[k] = lo[k];
      double ext = k < dim ? hi[k] - lo[k] : 0.0;
      double cnt = std::floor(ext / spacing + 0.5);
      double c = cnt >= 1.0 ? ext / cnt : spacing;
      g.inv_c[k] = 1.0 / c;
      ncell *= cnt + 1.0;
      g.nc[k] = cnt + 1.0 < 2.0e9 ? (int)cnt + 1 : 2000000000;
      // |round(a) - round(b)| <= floor(|a - b|) + 1
      g.S[k] = k < dim ? (int)std::floor(s->horizon / c) + 1 : 0;
    }
    if (ncell <= (double)(1ll << 28)) break;
    if (spacing >= s->horizon) { set_error("cell table too large: domain extent / horizon exceeds 2^28 cells"); return PD_ERR_LIMIT; }
    spacing = std::min(spacing * 2.0, s->horizon);
  }
  s->kdiv = g.S[0];
  g.R = R;
  g.BZ = dim == 3 ? PD_GROUPS_PER_CTA : 1;
  g.ncyg = (g.nc[1] + R - 1) / R;
  g.nczt = (g.nc[2] + g.BZ - 1) / g.BZ;
  const int64_t ncell = (int64_t)g.nc[0] * g.nc[1] * g.nc[2];
  const int64_t nrow = (int64_t)g.nc[1] * g.nc[2];
  const int64_t ntr = (int64_t)g.nczt * g.ncyg;

  // ---- 2. sort by cell id ----
  SCRATCH(keys, uint32_t, n);
  SCRATCH(keys2, uint32_t, n);
  SCRATCH(ids, int32_t, n);
  SCRATCH(ord1, int32_t, n);
  k_keys<<<nblk(n), TPB, 0, st>>>(n, g, coords, keys, ids);
  {
    int bits = 1;
    while (bits < 32 && (1ll << bits) < ncell) ++bits;
    size_t tb = 0;
    PD_CUDA(cub::DeviceRadixSort::SortPairs(nullptr, tb, keys, keys2, ids, ord1, (int)n, 0, bits, st));
    void *tmp = salloc(tb);
    if (!tmp) { set_error("device allocation failed"); return PD_ERR_ALLOC; }
    PD_CUDA(cub::DeviceRadixSort::SortPairs(tmp, tb, keys, keys2, ids, ord1, (int)n, 0, bits, st));
  }
  SCRATCH(cell_start, int32_t, ncell);
  SCRATCH(cell_end, int32_t, ncell);
  SCRATCH(row_start, int32_t, nrow);
  SCRATCH(row_end, int32_t, nrow);
  PD_CUDA(cudaMemsetAsync(cell_start, 0, sizeof(int32_t) * ncell, st));
  PD_CUDA(cudaMemsetAsync(cell_end, 0, sizeof(int32_t) * ncell, st));
  PD_CUDA(cudaMemsetAsync(row_start, 0, sizeof(int32_t) * nrow, st));
  PD_CUDA(cudaMemsetAsync(row_end, 0, sizeof(int32_t) * nrow, st));
  k_tables<<<nblk(n), TPB, 0, st>>>(n, g.nc[0], keys2, cell_start, cell_end, row_start, row_end);

  // ---- lattice body (one node per cell, uniform volume, small stencil)?  then the dense layout of
  //      pd_lattice.cu replaces everything below ----
  {
    int rc = build_lattice(s, g, coords, vol, flags, precut, n_precut, keys2, ord1, cell_start, cell_end);
    if (rc < 0) return rc;
    if (rc == 1) return PD_OK;
  }

  // ---- 3. lanes, tiles, final order ----
  SCRATCH(rowid, int32_t, n);
  SCRATCH(tval, int32_t, n);
  SCRATCH(tmax, int32_t, n);
  SCRATCH(vx, int32_t, n);
  SCRATCH(tile_x0, int32_t, ntr);
  k_row_t<<<nblk(n), TPB, 0, st>>>(n, g.nc[0], keys2, row_start, rowid, tval);
  {
    size_t tb = 0;
    PD_CUDA(cub::DeviceScan::InclusiveScanByKey(nullptr, tb, rowid, tval, tmax, cub::Max(), (int)n, cub::Equality(), st));
    void *tmp = salloc(tb);
    if (!tmp) { set_error("device allocation failed"); return PD_ERR_ALLOC; }
    PD_CUDA(cub::DeviceScan::InclusiveScanByKey(tmp, tb, rowid, tval, tmax, cub::Max(), (int)n, cub::Equality(), st));
  }
  k_tilerow_x0<<<nblk(ntr), TPB, 0, st>>>(ntr, g, keys2, row_start, row_end, tile_x0);
  int *maxvx_d = (int *)(red + 2);
  PD_CUDA(cudaMemsetAsync(red, 0, 8 * sizeof(unsigned long long), st));
  k_vx<<<nblk(n), TPB, 0, st>>>(n, g, rowid, row_start, tmax, tile_x0, vx, maxvx_d);
  int maxvx = 0;
  PD_CUDA(cudaMemcpyAsync(&maxvx, maxvx_d, sizeof(int), cudaMemcpyDeviceToHost, st));
  PD_CUDA(cudaStreamSynchronize(st));
  g.maxchunk = maxvx / 32 + 1;

  const int64_t ntile_dense = ntr * g.maxchunk;
  if (ntile_dense >= (1ll << 31) - 1) { set_error("tile table too large"); return PD_ERR_LIMIT; }
  SCRATCH(tile_flag, int32_t, ntile_dense + 1);
  SCRATCH(tile_ord, int32_t, ntile_dense + 1);
  PD_CUDA(cudaMemsetAsync(tile_flag, 0, sizeof(int32_t) * (ntile_dense + 1), st));
  k_tile_mark<<<nblk(n), TPB, 0, st>>>(n, g, rowid, vx, tile_flag);
  {
    int rc = scan_exclusive<int32_t>(s, scratch, tile_flag, tile_ord, ntile_dense + 1);
    if (rc) return rc;
  }
  int32_t ntile = 0;
  PD_CUDA(cudaMemcpyAsync(&ntile, tile_ord + ntile_dense, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  PD_CUDA(cudaStreamSynchronize(st));
  s->ngroups = (int64_t)ntile * g.BZ;
  s->nslices = s->ngroups * R;
  s->npad = s->nslices * 32;
  if (s->npad >= (1ll << 31) - 64 || s->npad * PD_NP >= (1ll << 32)) { set_error("too many nodes after padding"); return PD_ERR_LIMIT; }

  SCRATCH(fin1, int32_t, n);
  SCRATCH(tile_inv, int32_t, ntile);
  BUILD_ALLOC(s->perm, int32_t, s->npad);
  BUILD_ALLOC(s->iperm, int32_t, n);
  PD_CUDA(cudaMemsetAsync(s->perm, 0xff, sizeof(int32_t) * s->npad, st));
  k_final_index<<<nblk(n), TPB, 0, st>>>(n, g, rowid, vx, ord1, tile_ord, tile_inv, fin1, s->perm, s->iperm);

  for (int q = 0; q < 2; ++q) {
    BUILD_ALLOC(s->nb[q], double2, s->npad * PD_NP);
    PD_CUDA(cudaMemsetAsync(s->nb[q], 0, sizeof(double2) * s->npad * PD_NP, st));
  }
  BUILD_ALLOC(s->vol, double, s->npad);
  BUILD_ALLOC(s->m, double, s->npad);
  BUILD_ALLOC(s->minv, double, s->npad);
  BUILD_ALLOC(s->fvol, double, s->npad);
  BUILD_ALLOC(s->flags, uint8_t, s->npad);
  for (double *p : {s->vol, s->m, s->minv, s->fvol}) PD_CUDA(cudaMemsetAsync(p, 0, sizeof(double) * s->npad, st));
  PD_CUDA(cudaMemsetAsync(s->flags, 0, s->npad, st));
  k_records<<<nblk(s->npad), TPB, 0, st>>>(s->npad, g, s->perm, coords, vol, flags, s->nb[0], s->nb[1], s->vol, s->flags);

  // ---- 4. count -> group lengths -> offsets ----
  const double h2 = s->horizon * s->horizon;
  BUILD_ALLOC(s->rowlen, int32_t, s->npad);
  BUILD_ALLOC(s->goff, uint32_t, s->ngroups + 1);
  BUILD_ALLOC(s->soff, uint32_t, s->ngroups + 1);
  SCRATCH(glen, uint32_t, s->ngroups + 1);
  SCRATCH(slen, uint32_t, s->ngroups + 1);
  PD_CUDA(cudaMemsetAsync(glen + s->ngroups, 0, sizeof(uint32_t), st));
  PD_CUDA(cudaMemsetAsync(slen + s->ngroups, 0, sizeof(uint32_t), st));
  const unsigned gblk = nblk(s->ngroups * 32);
  k_count<<<gblk, TPB, 0, st>>>(s->ngroups, g, h2, s->nb[0], s->perm, cell_start, cell_end, fin1, tile_inv, tile_x0,
                                s->rowlen, glen, slen);
  {
    int rc = scan_exclusive<uint32_t>(s, scratch, glen, s->goff, s->ngroups + 1);
    if (rc) return rc;
    rc = scan_exclusive<uint32_t>(s, scratch, slen, s->soff, s->ngroups + 1);
    if (rc) return rc;
  }
  uint32_t total_entries = 0, total_segs = 0;
  PD_CUDA(cudaMemcpyAsync(&total_entries, s->goff + s->ngroups, sizeof(uint32_t), cudaMemcpyDeviceToHost, st));
  PD_CUDA(cudaMemcpyAsync(&total_segs, s->soff + s->ngroups, sizeof(uint32_t), cudaMemcpyDeviceToHost, st));
  SCRATCH(zsum, long long, 1);
  {
    cub::TransformInputIterator<long long, cub::CastOp<long long>, const int32_t *> it(s->rowlen, cub::CastOp<long long>());
    size_t tb = 0;
    PD_CUDA(cub::DeviceReduce::Sum(nullptr, tb, it, zsum, (int)s->npad, st));
    void *tmp = salloc(tb);
    if (!tmp) { set_error("device allocation failed"); return PD_ERR_ALLOC; }
    PD_CUDA(cub::DeviceReduce::Sum(tmp, tb, it, zsum, (int)s->npad, st));
  }
  long long hz = 0;
  PD_CUDA(cudaMemcpyAsync(&hz, zsum, sizeof(long long), cudaMemcpyDeviceToHost, st));
  PD_CUDA(cudaMemsetAsync(red, 0, 8 * sizeof(unsigned long long), st));
  k_checks<<<nblk(s->npad), TPB, 0, st>>>(s->npad, s->perm, s->rowlen, s->flags, red);
  PD_CUDA(cudaMemcpyAsync(hred, red, 2 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
  PD_CUDA(cudaStreamSynchronize(st));
  s->Z = hz;
  s->nentries = total_entries;
  s->nsegs = total_segs;
  if (hred[0]) { set_error("a node has an empty family (m_i = 0); enlarge the horizon"); return PD_ERR_ISOLATED; }
  if (s->Z >= (1ll << 31)) {
    set_error("more than 2^31 directed bonds");
    return PD_ERR_LIMIT;
  }
  if ((uint64_t)total_entries * 32 >= (1ull << 32) - 32 * (PD_COL_SLACK + 1)) {
    set_error("neighbour list too long for 32-bit offsets");
    return PD_ERR_LIMIT;
  }
  s->has_nofail = (hred[1] & 1ull) != 0;
  s->has_bc = (hred[1] & 2ull) != 0;

  // ---- 5. fill ----
  const size_t ncol = ((size_t)total_entries + PD_COL_SLACK) * 32, nwords = ((size_t)total_segs + 8) * 32;
  BUILD_ALLOC(s->col, uint32_t, ncol);
  BUILD_ALLOC(s->member, uint32_t, nwords);
  BUILD_ALLOC(s->seg, uint32_t, nwords);
  PD_CUDA(cudaMemsetAsync(s->col + (size_t)total_entries * 32, 0, sizeof(uint32_t) * 32 * PD_COL_SLACK, st));  // slack: node 0
  PD_CUDA(cudaMemsetAsync(s->member + (size_t)total_segs * 32, 0, sizeof(uint32_t) * 8 * 32, st));
  k_fill<<<gblk, TPB, 0, st>>>(s->ngroups, g, h2, s->G, s->nb[0], s->nb[1], s->vol, s->m, s->minv, s->fvol, s->perm,
                               cell_start, cell_end, fin1, tile_inv, tile_x0, s->goff, s->soff, s->col, s->member);
  PD_CUDA(cudaMemcpyAsync(s->seg, s->member, sizeof(uint32_t) * nwords, cudaMemcpyDeviceToDevice, st));

  // ---- 6. pre-cuts, no-fail ----
  if (n_precut > 0) {
    PD_CUDA(cudaMemsetAsync(red, 0, sizeof(unsigned long long), st));
    k_precut<<<nblk(2 * n_precut), TPB, 0, st>>>(n_precut, n, precut, s->iperm, s->goff, s->soff, s->col, s->member, s->seg, red);
    PD_CUDA(cudaMemcpyAsync(hred, red, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
    PD_CUDA(cudaStreamSynchronize(st));
    if (hred[0]) { set_error("a pre-cut pair is out of range or not a bond"); return PD_ERR_ARG; }
  }
  if (s->has_nofail && s->fracture) {
    BUILD_ALLOC(s->nofail, uint32_t, nwords);
    PD_CUDA(cudaMemsetAsync(s->nofail, 0, sizeof(uint32_t) * nwords, st));
    k_nofail<<<gblk, TPB, 0, st>>>(s->ngroups, s->flags, s->goff, s->soff, s->col, s->member, s->nofail);
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
    if (col_dev && intact_dev && s->lat.on) {
      cudaStreamSynchronize(st);
      rc = lat_export_bond_mask(s, rowptr_dev, col_dev, intact_dev);
    } else if (col_dev && intact_dev)
      k_export_rows<<<nblk(s->ngroups * 32), TPB, 0, st>>>(s->ngroups, s->perm, rowptr_dev, s->goff, s->soff, s->col,
                                                            s->member, s->seg, col_dev, intact_dev);
    if (cudaGetLastError() != cudaSuccess) rc = PD_ERR_CUDA;
  } while (0);
  cudaStreamSynchronize(st);
  if (tmp) dev_free(s, tmp);
  dev_free(s, cnt);
  if (rc == PD_ERR_CUDA) set_error("CUDA error in pd_get_bond_mask");
  return rc;
}

}  // namespace pdi
