// pd_internal.cuh -- private state of libpd.so (not part of the boundary; see include/pd.h).
//
// Data layout in HBM.  Nodes are renumbered by the builder into a
// FINAL order made of 32-node SLICES (one warp lane per node); R consecutive slices form a
// GROUP (one warp): lane l of group g owns the R nodes (g*R + r)*32 + l, r = 0..R-1, which the
// builder chooses to be the l-th nodes of R adjacent lattice rows.  Missing nodes are PHANTOMS
// (perm = -1, zero record, no bonds).
//
//   rec : node records, AoSoA-32 with PD_NF = 16 FP64 fields per node:
//         element index elem(i) = (i >> 5) * (32*PD_NF) + (i & 31); field f lives at elem + 32 f
//         (so a warp reads 256 contiguous bytes per field and one address serves all fields).
//         (vector components are stored in INTERNAL order: component k = user component ax[k],
//          internal axis 0 = the lane axis chosen by the builder)
//         fields: 0-2 x (reference position)   3 gmu = G/m_i      4 vol = V_i     5 minv = 1/m_i
//                 6 m_i                        7 fvol = sum_j V_j
//                 8-10 u (buffer 0)  11 cth (buffer 0)   12-14 u (buffer 1)  15 cth (buffer 1)
//         cth_i = (K - G/3) theta_i / m_i belongs to the u buffer it was computed from.
//   blocked sliced ELL ("SELL-32xR"): group g has glen[g] ENTRIES starting at goff[g]; entry k of
//         lane l is ONE neighbour shared by the lane's R nodes:
//           col   [(goff[g] + k)*32 + l]            elem() of the neighbour
//           intact[(goff[g] + k)/EPW*32 + l]        bit ((k % EPW)*R + r): bond (node r, neighbour)
//                                                   exists and is unbroken (Eq. 1.30); EPW = 32/R
//           member[...]  same shape, static: the bond exists (family membership)
//           nofail[...]  same shape, static, only if some node is no-fail
//         padding entries point at the lane's own node 0 and have all bits 0.
//   v, bval : SoA [dim][npad];  flags, rowlen, phi : [npad]
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <utility>
#include <vector>

#include "../../include/pd.h"

#define PD_MAX_DIM 3
#define PD_NF 16          // FP64 fields per node record
#define PD_F_X 0
#define PD_F_GMU 3
#define PD_F_VOL 4
#define PD_F_MINV 5
#define PD_F_M 6
#define PD_F_FVOL 7
#define PD_F_U(buf) (8 + 4 * (buf))
#define PD_F_CTH(buf) (11 + 4 * (buf))
#define PD_GROUPS_PER_CTA 4   // 128 threads; in 3D the 4 groups of a CTA are 4 z-levels of one tile

__host__ __device__ __forceinline__ uint32_t pd_elem(int64_t i) {
  return (uint32_t)((i >> 5) * (32 * PD_NF) + (i & 31));
}
__host__ __device__ __forceinline__ int64_t pd_elem_inv(uint32_t e) {
  return ((int64_t)(e / (32 * PD_NF)) << 5) | (e & 31);
}

struct pd_sim {
  // scalars
  int dim = 0, mode = 0;
  int R = 4;                    // rows (nodes) per thread
  int ax[3] = {0, 1, 2};        // internal component k = user component ax[k]; internal 0 is the lane axis
  int64_t n = 0, npad = 0, nslices = 0, ngroups = 0;
  int64_t Z = 0, nentries = 0;  // directed bonds; stored entries per lane (sum of glen)
  double horizon = 0, A = 0, K = 0, G = 0, c1 = 0;  // c1 = K - G/3
  double rho = 0, dt = 0, s_c = 0, ramp_time = 0, vol_uniform = 0;
  bool fracture = false, uniform_v = false, has_nofail = false, has_bc = false;
  int kdiv = 1;
  // runtime
  pd_runtime rt{};
  bool own_alloc = true;
  cudaStream_t stream = 0;
  std::vector<std::pair<void *, size_t>> allocs;
  size_t bytes_held = 0;
  // node arrays (final order)
  int32_t *perm = nullptr, *iperm = nullptr;  // perm[final] = user or -1, iperm[user] = final
  double *rec = nullptr;
  double *v[PD_MAX_DIM] = {}, *bval[PD_MAX_DIM] = {};
  double *phi = nullptr;
  uint8_t *flags = nullptr;
  int32_t *rowlen = nullptr;
  // blocked SELL
  uint32_t *goff = nullptr;   // [ngroups + 1] entry offsets (multiples of EPW)
  uint32_t *col = nullptr;
  uint32_t *intact = nullptr, *member = nullptr, *nofail = nullptr;
  // state
  int cur = 0;            // which u buffer holds u^n
  int64_t step = 0;       // n
  int64_t launches = 0;   // kernels launched by pd_step
  bool break_pending = false;  // u^n has not been break-checked yet (deferred step 5)
  unsigned long long *stats_dev = nullptr;  // [0]=broken directed, [1]=max phi bits, [2]=#phi>=.5
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
