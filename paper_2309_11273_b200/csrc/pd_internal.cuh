// pd_internal.cuh -- private state of libpd.so (not part of the boundary; see include/pd.h).
//
// Data layout in HBM (all node arrays in the library's SORTED node order, padded to a
// multiple of 32 nodes):
//   x[k], u[b][k], v[k], bval[k] : SoA FP64, one array per component k (u double-buffered, b = 0/1)
//   vol, minv (=1/m_i), gmu (=G/m_i), cth (=(K-G/3) theta_i/m_i, rewritten every step), fvol
//   sliced ELL ("SELL-32"): slice s = sorted nodes 32s .. 32s+31 (one warp, one lane per node);
//     col [(slice_off[s] + k)*32 + lane]  : neighbour (sorted index) in slot k of that lane's row
//     mask[(mask_off[s]  + w)*32 + lane]  : bit b of word w = bond in slot 32w+b intact (Eq. 1.30)
//   slots past a row's length point at the node itself and have mask bit 0.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <utility>
#include <vector>

#include "../../include/pd.h"

#define PD_MAX_DIM 3
#define PD_SLOT_ALIGN 4  // slice lengths are rounded up to a multiple of this (inner unroll)

struct pd_sim {
  // scalars
  int dim = 0, mode = 0;
  int64_t n = 0, npad = 0, nslices = 0;
  int64_t Z = 0, nslots = 0, nmaskwords = 0;  // directed bonds, stored slots (per lane), mask words (per lane)
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
  // node arrays (sorted order)
  int32_t *perm = nullptr, *iperm = nullptr;  // perm[sorted] = user, iperm[user] = sorted
  double *x[PD_MAX_DIM] = {}, *u[2][PD_MAX_DIM] = {}, *v[PD_MAX_DIM] = {}, *bval[PD_MAX_DIM] = {};
  double *vol = nullptr, *m = nullptr, *minv = nullptr, *gmu = nullptr, *cth = nullptr, *fvol = nullptr, *phi = nullptr;
  uint8_t *flags = nullptr;
  int32_t *rowlen = nullptr;
  // SELL
  uint32_t *slice_off = nullptr, *mask_off = nullptr;
  int32_t *slice_len = nullptr;
  int32_t *col = nullptr;
  uint32_t *mask = nullptr, *nofail = nullptr;
  // state
  int cur = 0;            // which u buffer holds u^n
  int64_t step = 0;       // n
  int64_t launches = 0;   // kernels launched by pd_step
  bool break_pending = false;  // u^n has not been break-checked yet (deferred step 5)
  unsigned long long *stats_dev = nullptr;  // [0]=broken directed, [1]=max phi bits, [2]=#phi>=.5, [3]=err flag
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
void launch_dilatation(pd_sim *s, const double *const *ucur, double *theta_out, bool do_break);
void launch_force_update(pd_sim *s);
void launch_damage(pd_sim *s);
}  // namespace pdi

#define PD_CUDA(call)                                                       \
  do {                                                                      \
    cudaError_t e__ = (call);                                               \
    if (e__ != cudaSuccess) return pdi::cuda_fail(e__, #call);              \
  } while (0)
