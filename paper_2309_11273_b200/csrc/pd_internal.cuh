// pd_internal.cuh -- private state of libpd.so (not part of the boundary; see include/pd.h).
//
// Data layout in HBM.  Nodes are renumbered by the builder into a
// FINAL order made of 32-node SLICES (one warp lane per node); PD_R = 4 consecutive slices form a
// GROUP (one warp): lane l of group g owns the 4 nodes (g*4 + r)*32 + l, r = 0..3, which the
// builder chooses to be the l-th nodes of 4 lattice rows adjacent along internal axis 1.
// Missing nodes are PHANTOMS (perm = -1, zero records, no bonds).
// Vector components are stored in INTERNAL order: component k = user component ax[k]; internal
// axis 0 is the lane axis chosen by the builder.
//
//   nb[b], b = 0, 1 : NEIGHBOUR RECORDS, the data a bond gathers from its far end, as 16-byte pairs
//         in AoSoA-32: pair p of node i sits at double2 index  pd_elem(i) + 32 p,
//         pd_elem(i) = (i >> 5) * (32 * PD_NP) + (i & 31), so a warp reads 512 contiguous bytes per
//         pair with one LDG.128 per lane.
//           pair k < 3 : { x_k (reference position, static), u_k }      (buffer b holds u^n for cur = b)
//           pair 3     : { G/m_i (static),  cth_i = (K - G/3) theta_i / m_i of the u in this buffer }
//   own-node statics (SoA [npad]): vol = V_i, minv = 1/m_i, m = m_i, fvol = sum_j V_j
//   v, bval : SoA [dim][npad];  flags, rowlen, phi : [npad]
//
//   neighbour lists ("windowed SELL-32x4"): group g owns the ENTRIES goff[g] .. goff[g+1]-1 and the
//   SEGMENTS soff[g] .. soff[g+1]-1.
//     col[(goff[g] + k)*32 + l]   = pd_elem() of the node lane l gathers in entry k (own node 0 if none)
//     seg[(soff[g] + s)*32 + l]   = one 32-bit word per lane and segment:
//           bits 28-31  CODE, the same on all 32 lanes:
//                 1..7   SHIFT segment of n = CODE steps over n + 3 consecutive entries: in step t
//                        row r pairs with entry t + r (a window sliding along the rows' axis: the
//                        4 rows are adjacent lattice rows, so entry t + r is the same RELATIVE
//                        neighbour for every row; one gathered neighbour serves up to 4 bonds)
//                 9..15  FLAT segment of n = CODE - 8 steps over n entries: in step t all rows pair
//                        with entry t (general point clouds, cells holding several nodes)
//                 0      padding (skipped)
//           bits 0-27   bit 4 t + r : the bond (row r, step t) exists and is unbroken (Eq. 1.30)
//     member / nofail : same shape as seg, static: the bond exists / may never break
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <utility>
#include <vector>

#include "../../include/pd.h"

#define PD_MAX_DIM 3
#define PD_R 4            // rows (nodes) per lane
#define PD_NP 4           // 16-byte pairs per node in a neighbour record
#define PD_P_AUX 3        // pair {G/m, cth}
#define PD_MAXSTEP 7      // steps per segment (28 mask bits)
#define PD_GROUPS_PER_CTA 4   // 128 threads; in 3D the 4 groups of a CTA are 4 levels (internal axis 2) of one tile
#define PD_COL_SLACK 64   // readable entries past the end of col (the kernels prefetch indices ahead)

__host__ __device__ __forceinline__ uint32_t pd_elem(int64_t i) {
  return (uint32_t)((i >> 5) * (32 * PD_NP) + (i & 31));
}
__host__ __device__ __forceinline__ int64_t pd_elem_inv(uint32_t e) {
  return ((int64_t)(e / (32 * PD_NP)) << 5) | (e & 31);
}

// double2 index of pair p of node i in a neighbour-record buffer, for either layout
__host__ __device__ __forceinline__ int64_t pd_pair_index(bool lattice, int64_t npad, int64_t i, int p) {
  return lattice ? (int64_t)p * npad + i : (int64_t)pd_elem(i) + 32 * p;
}

// Calls f(s, bit, r, k) for every bond slot of one lane: s = segment index inside the group,
// bit = 4 t + r, k = entry index inside the group.  `words` = the lane's segment words (any of
// seg / member / nofail: only the CODE nibble is read here), stride 32.
template <typename F>
__host__ __device__ __forceinline__ void pd_for_lane_slots(const uint32_t *words, int nseg, F f) {
  int e = 0;
  for (int s = 0; s < nseg; ++s) {
    const uint32_t code = words[(int64_t)s * 32] >> 28;
    if (code == 0) continue;
    if (code < 8) {
      const int n = (int)code;
      for (int t = 0; t < n; ++t)
        for (int r = 0; r < PD_R; ++r) f(s, 4 * t + r, r, e + t + r);
      e += n + 3;
    } else {
      const int n = (int)code - 8;
      for (int t = 0; t < n; ++t)
        for (int r = 0; r < PD_R; ++r) f(s, 4 * t + r, r, e + t);
      e += n;
    }
  }
}

// ---- dense lattice layout (pd_lattice.cu), used when the body is a (jittered) lattice with one node
// per cell, uniform volume and a family stencil of <= 128 relative offsets.  Nodes live in a dense
// array over the cell grid (internal axes 0 = lane axis X, 1 = Y, 2 = Z) with a margin of the
// stencil radius on every side (zero-filled PHANTOM cells):
//     cell (x, y, z) -> final index  ((z + HZ) * DY + (y + HY)) * DX + (x + HX)
//   neighbour-record pair p of node i sits at nb[b][p * npad + i]  (each pair a dense 3-D array)
//   lmask / lmember / lnofail [w * npad + i], w < 4: one bit per stencil offset (bit order = the
//   column table below), so no neighbour index is stored at all.
// The stencil is a table of COLUMNS: offsets (dx, dy0 .. dy0 + n - 1, dz), n <= 7, whose bits
// bit0 .. bit0 + n - 1 lie inside one mask word.
#define PD_LAT_MAXCOL 160
struct PdLatCol {
  int16_t dx, dy0, dz;
  uint8_t n, word, bit0, split, pad0, pad1;   // split: which warp of a row group walks this column
};
struct PdGrid {
  double lo[3];
  double inv_c[3];  // 1 / cell edge per dimension
  int nc[3];        // cells per dim
  int S[3];         // search radius in cells per dim
  int dim;
  int ax[3];        // internal axis k = user axis ax[k]
  int R, BZ;        // rows per thread, z-levels per tile
  int ncyg, nczt, maxchunk;
};
struct PdLattice {
  bool on = false;
  // UNIFORM lattice (pd_lattice_uniform.cu): every bond of a stencil offset o has the same xi = (o_k h_k) up to
  // the rounding of the coordinates, so the bond geometry is a per-offset constant and the step kernels
  // gather displacements only:  uxy[b] = {u_0, u_1}, uz[b] = u_2 (3-D), aux = {G/m, cth}; nb[] is released.
  bool uniform = false;
  double h[3] = {0, 0, 0};         // lattice spacing per internal axis
  double2 *uxy[2] = {nullptr, nullptr};
  double *uz[2] = {nullptr, nullptr};
  double2 *aux = nullptr;
  double *ctab[2] = {nullptr, nullptr};   // device: per stencil bit, the constants of the dilatation / force pass
  void *ucols = nullptr;           // device: the column table of the uniform kernels
  int wbeg[5] = {0, 0, 0, 0, 0};   // columns whose bits lie in mask word w: wbeg[w] .. wbeg[w + 1] - 1
  int DX = 0, DY = 0, DZ = 0;      // dense dims incl. margins
  int HX = 0, HY = 0, HZ = 0;      // margins = stencil radius per axis
  int PX = 0, PY = 0, PZ = 0;      // padded cell counts (PX multiple of 32, PY of 4)
  int ncol = 0, nbits = 0, nw = 0; // columns, mask bits used (incl. padding), mask words
  uint32_t fullw[4] = {0, 0, 0, 0};
  PdLatCol cols[PD_LAT_MAXCOL];
  uint32_t *mask = nullptr, *member = nullptr, *nofail = nullptr;   // [4][npad]
  uint8_t *rgocc = nullptr;        // [PZ + 8][(PY + 8)/4][PX/32]: the 32x4 row group holds a node
  uint32_t *flags32 = nullptr;     // [npad] the node flags as 32-bit words (4-byte asynchronous copies)
  int32_t *off2bit = nullptr;      // [(2S2+1)(2S1+1)(2S0+1)] offset -> bit index or -1
  double r2lb[128];                // per stencil bit: min over all bonds of ||xi||^2 exactly as the step kernels
                                   // compute it (break-test filter: dot < s_c * r2lb  =>  the bond cannot break)
  void *cache[8] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};   // host: prepared launch arguments of the step
                                   // kernels ([0], [1]: pd_lattice_uniform.cu; [2], [3]: pd_lattice_step.cu; [4], [5]: pd_lattice_ball.cu; [6], [7]: pd_lattice_disc.cu)
  // pd_lattice_ball.cu: octant words of mask / nofail [8][npad] and the exact-pass tables (device)
  uint32_t *mask8 = nullptr, *nf8 = nullptr;
  void *ball_q8 = nullptr, *ball_wl = nullptr;   // table of the octant copies; worklist of the break test
  int *ball_wl_count = nullptr;
  uint8_t *ball_tfull = nullptr;   // per warp tile: every family complete, intact and allowed to break
  int32_t *thr_dir = nullptr;      // device: per (column, step) filter thresholds of the dilatation kernel (pd_lattice_step.cu)
  int S[3] = {0, 0, 0};
};

struct pd_sim {
  PdLattice lat;
  // scalars
  int dim = 0, mode = 0;
  int ax[3] = {0, 1, 2};        // internal component k = user component ax[k]; internal 0 is the lane axis
  int64_t n = 0, npad = 0, nslices = 0, ngroups = 0;
  int64_t Z = 0, nentries = 0, nsegs = 0;  // directed bonds; stored entries / segments per lane
  double horizon = 0, A = 0, K = 0, G = 0, c1 = 0;  // c1 = K - G/3
  double rho = 0, dt = 0, s_c = 0, ramp_time = 0, vol_uniform = 0;
  bool fracture = false, uniform_v = false, has_nofail = false, has_bc = false;
  bool geom = false;            // variant: geometric extension e = ||xi + eta|| - ||xi|| (App. C) instead of the linearized one
  int kdiv = 1;
  // runtime
  pd_runtime rt{};
  bool own_alloc = true;
  cudaStream_t stream = 0;
  std::vector<std::pair<void *, size_t>> allocs;
  size_t bytes_held = 0;
  // node arrays (final order)
  int32_t *perm = nullptr, *iperm = nullptr;  // perm[final] = user or -1, iperm[user] = final
  double2 *nb[2] = {nullptr, nullptr};
  double *vol = nullptr, *minv = nullptr, *m = nullptr, *fvol = nullptr;
  double *v[PD_MAX_DIM] = {}, *bval[PD_MAX_DIM] = {};
  double *phi = nullptr;
  uint8_t *flags = nullptr;
  int32_t *rowlen = nullptr;
  // windowed SELL
  uint32_t *goff = nullptr, *soff = nullptr;   // [ngroups + 1] entry / segment offsets
  uint32_t *col = nullptr;
  uint32_t *seg = nullptr, *member = nullptr, *nofail = nullptr;
  // state
  int cur = 0;            // which buffer holds u^n
  int64_t step = 0;       // n
  int64_t launches = 0;   // kernels launched by pd_step
  bool break_pending = false;  // u^n has not been break-checked yet (deferred step 5)
  // CUDA graphs of the step loop (pd_api.cu): [0] = 2 steps, [1] = graph_len steps
  bool use_graph = true, graph_failed = false;
  int graph_len = 32;
  int graph_steps[2] = {0, 0};
  int64_t graph_launches[2] = {0, 0};   // kernels inside one replay of the graph
  cudaGraphExec_t graph[2] = {nullptr, nullptr};
  cudaStream_t cap_stream = nullptr;
  unsigned long long *stats_dev = nullptr;  // [0]=broken directed, [1]=max phi bits, [2]=#phi>=.5
  // adaptive dynamic relaxation (pd_adr_step): Ud^{n-1/2}, R^{n-1} (SoA, internal component order), {num, den} of c^n
  double *adr_ud[PD_MAX_DIM] = {}, *adr_rprev[PD_MAX_DIM] = {}, *adr_scal = nullptr;
  int64_t adr_it = 0;
};

namespace pdi {
void set_error(const std::string &msg);
int cuda_fail(cudaError_t e, const char *what);
void *dev_alloc(pd_sim *s, size_t bytes);  // through pd_runtime; tracked; nullptr on failure
void dev_free(pd_sim *s, void *p);         // untracks and releases one allocation
void dev_free_all(pd_sim *s);
// pd_build.cu
int build_family(pd_sim *s, const double *coords_user_dev, const double *vol_user_dev,
                 const uint8_t *flags_user_dev, const int32_t *precut_dev, int64_t n_precut);
int export_bond_mask(pd_sim *s, long long *rowptr_dev, int32_t *col_dev, uint8_t *intact_dev);
// pd_lattice.cu: returns 1 if the lattice layout was built, 0 if the body does not qualify, < 0 on error
int build_lattice(pd_sim *s, const PdGrid &g, const double *coords_user_dev, const double *vol_user_dev,
                  const uint8_t *flags_user_dev, const int32_t *precut_dev, int64_t n_precut,
                  const uint32_t *keys_sorted, const int32_t *ids_sorted, const int32_t *cell_start,
                  const int32_t *cell_end);
int lat_export_bond_mask(pd_sim *s, const long long *rowptr_dev, int32_t *col_dev, uint8_t *intact_dev);
int lat_launch_dilatation(pd_sim *s, double *theta_out, bool do_break);
int lat_launch_force_update(pd_sim *s);
int lat_launch_damage(pd_sim *s);
void lat_free_cache(pd_sim *s);
// pd_lattice_uniform.cu
int ulat_launch_dilatation(pd_sim *s, double *theta_out, bool do_break);
int ulat_launch_force_update(pd_sim *s);
void ulat_free_cache(pd_sim *s);
// pd_lattice_ball.cu: return 1 if launched, 0 if the lattice's stencil is not the compiled-in ball, < 0 on error
int ball_launch_dilatation(pd_sim *s, double *theta_out, bool do_break);
int ball_launch_force_update(pd_sim *s);
void ball_free_cache(pd_sim *s);
bool ball_eligible(const pd_sim *s);
// pd_lattice_disc.cu: the same for the 2-D 28-offset stencil
int disc_launch_dilatation(pd_sim *s, double *theta_out, bool do_break);
int disc_launch_force_update(pd_sim *s);
void disc_free_cache(pd_sim *s);
bool disc_eligible(const pd_sim *s);
// pd_step.cu
int launch_dilatation(pd_sim *s, double *theta_out, bool do_break);
int launch_force_update(pd_sim *s);
int launch_damage(pd_sim *s);
}  // namespace pdi

#define PD_CUDA(call)                                                       \
  do {                                                                      \
    cudaError_t e__ = (call);                                               \
    if (e__ != cudaSuccess) return pdi::cuda_fail(e__, #call);              \
  } while (0)
