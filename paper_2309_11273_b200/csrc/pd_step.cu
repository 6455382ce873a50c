// pd_step.cu -- the per-step kernels.
//
// One warp per GROUP of the blocked sliced-ELL layout (pd_internal.cuh): lane l owns R nodes (the
// l-th nodes of R adjacent lattice rows) and walks the lane's entry list.  An entry is one
// neighbour j; x_j, u_j (and G/m_j, cth_j) are gathered ONCE and serve the up-to-R bonds
// (i_r, j), r = 0..R-1, whose bits are set -- register blocking of the gather, which is what
// the L1 data pipe, the index stream and the instruction issue are all short of (profiles/).
// In the bulk of a lattice body the 32 lanes of a warp see the same relative neighbour in entry
// k, so every gather of a warp is 256 contiguous bytes per field, and which (entry, r) pairs
// are bonds is warp-uniform: pairs that are a bond for no lane are skipped with a uniform
// branch (the OR of the mask word over the warp, one REDUX per word).
//
//   k_dilatation  (rows a1, a2, and a5's break test folded in):
//        for each intact bond  dot = xi . eta            [= xbar * e, sqrt-free]
//        FRAC: if dot >= s_c * ||xi||^2 (<=> e/xbar >= s_c, Eq. 1.17/1.30) clear the bit first
//        theta_i = (A/m_i) sum_j rho_ij dot V_j           (Eq. 1.6 / 2.3)
//        writes cth_i = (K - G/3) theta_i / m_i
//   k_force_update (rows a1, a3, a4):
//        f_i = sum_j rho_ij V_j [ cth_i + cth_j + (G/m_i + G/m_j) dot/||xi||^2 ] xi   (Eq. 2.2 / 2.1)
//        then Eq. 2.11 + boundary dofs, u^{n+1} into the other u buffer
//   k_damage (row a5): phi_i (Eq. 1.31) + device-side reduction of the three damage scalars
//
// The break test of step n (on u^{n+1}) runs at the start of step n+1's dilatation pass, which
// needs the same xi . eta; pd_api.cu flushes it before any state is read back.  Both ends of a
// bond take the identical decision because -a*-b == a*b exactly in every product and the sums
// run in the same component order.
#include "pd_internal.cuh"

namespace {

constexpr int TPB = 32 * PD_GROUPS_PER_CTA;
constexpr unsigned FULL = 0xffffffffu;
constexpr int EB = 8;   // entries per pipelined block (a whole mask word when R = 4)

struct StepArgs {
  int64_t ngroups;
  double *rec;
  const uint32_t *goff;
  const uint32_t *col;
  uint32_t *intact;
  const uint32_t *nofail;
  double *v[3];
  const double *bval[3];
  double *theta_out;
  double *phi;
  const uint8_t *flags;
  const int32_t *rowlen;
  const int32_t *perm;
  unsigned long long *stats;
  double A, c1, s_c, vol_uniform, rho, dt, ramp_time;
  int64_t step;
};

// 1/x to ~1 ulp: hardware seed (MUFU.RCP64H, rel. err 2^-23) + one cubic Newton step:
// y (1 + e + e^2) with e = 1 - x y  leaves (1/x)(1 - e^3).
__device__ __forceinline__ double rcp_fast(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double e = fma(-x, y, 1.0);
  double t = fma(e, e, e);
  return fma(y, t, y);
}

template <int DIM>
__device__ __forceinline__ double dot_xi_eta(const double *xi, const double *eta) {
  double d = xi[0] * eta[0];
#pragma unroll
  for (int k = 1; k < DIM; ++k) d = fma(xi[k], eta[k], d);
  return d;
}

// ---------------------------------------------------------------------------------------------
template <int DIM, int R, bool FRAC, bool UNIV, int CUR>
__global__ void __launch_bounds__(TPB) k_dilatation(StepArgs a) {
  constexpr int EPW = 32 / R;
  constexpr uint32_t RMASK = (1u << R) - 1u;
  constexpr uint32_t BMASK = EB * R == 32 ? 0xffffffffu : ((1u << (EB * R)) - 1u);
  const int lane = threadIdx.x & 31;
  const int64_t grp = ((int64_t)blockIdx.x * TPB + threadIdx.x) >> 5;
  if (grp >= a.ngroups) return;
  double *rec = a.rec;
  const uint32_t e0 = pd_elem(grp * R * 32 + lane);

  double xi_[R][DIM], ui_[R][DIM], acc[R];
#pragma unroll
  for (int r = 0; r < R; ++r) {
    acc[r] = 0.0;
#pragma unroll
    for (int k = 0; k < DIM; ++k) {
      xi_[r][k] = rec[e0 + r * 32 * PD_NF + 32 * (PD_F_X + k)];
      ui_[r][k] = rec[e0 + r * 32 * PD_NF + 32 * (PD_F_U(CUR) + k)];
    }
  }
  const uint32_t off = a.goff[grp];
  const uint32_t nwords = (a.goff[grp + 1] - off) / EPW;
  const uint32_t *col = a.col + (int64_t)off * 32 + lane;
  uint32_t *bits = a.intact + (int64_t)(off / EPW) * 32 + lane;
  const uint32_t *nofail = (FRAC && a.nofail) ? a.nofail + (int64_t)(off / EPW) * 32 + lane : nullptr;

  // entries are walked in blocks of EB = 8: the 8 neighbour indices of the NEXT block are loaded
  // before the current block is processed, and the node data of entry q+1 before entry q is used
  // (software pipeline in registers; the index stream comes from HBM, the node data from L1/L2).
  const uint32_t nblocks = nwords * (EPW / EB);
  uint32_t cn[EB], mwn = 0;
  if (nblocks) {
#pragma unroll
    for (int q = 0; q < EB; ++q) cn[q] = col[q * 32];
    mwn = bits[0];
  }
  for (uint32_t blk = 0; blk < nblocks; ++blk) {
    const uint32_t w = blk / (EPW / EB), sh = (blk % (EPW / EB)) * (EB * R);
    uint32_t c[EB];
#pragma unroll
    for (int q = 0; q < EB; ++q) c[q] = cn[q];
    uint32_t mwfull = (EPW == EB) ? mwn : bits[w * 32];
    if (blk + 1 < nblocks) {
#pragma unroll
      for (int q = 0; q < EB; ++q) cn[q] = col[((blk + 1) * EB + q) * 32];
      if (EPW == EB) mwn = bits[(w + 1) * 32];
    }
    uint32_t mw = (mwfull >> sh) & BMASK;
    const uint32_t anyw = __reduce_or_sync(FULL, mw);   // warp-uniform: pairs that are a bond for some lane
    if (anyw == 0) continue;
    const uint32_t mw0 = mw;
    uint32_t nf = 0;
    if (FRAC && nofail) nf = (nofail[w * 32] >> sh) & BMASK;
    double xj[DIM], uj[DIM], vj = 0.0, xn[DIM], un[DIM], vn = 0.0;
    {
      const double *p = rec + c[0];
#pragma unroll
      for (int k = 0; k < DIM; ++k) { xn[k] = __ldg(p + 32 * (PD_F_X + k)); un[k] = __ldg(p + 32 * (PD_F_U(CUR) + k)); }
      if (!UNIV) vn = __ldg(p + 32 * PD_F_VOL);
    }
#pragma unroll
    for (int q = 0; q < EB; ++q) {
#pragma unroll
      for (int k = 0; k < DIM; ++k) { xj[k] = xn[k]; uj[k] = un[k]; }
      vj = vn;
      if (q + 1 < EB) {
        const double *p = rec + c[q + 1];
#pragma unroll
        for (int k = 0; k < DIM; ++k) { xn[k] = __ldg(p + 32 * (PD_F_X + k)); un[k] = __ldg(p + 32 * (PD_F_U(CUR) + k)); }
        if (!UNIV) vn = __ldg(p + 32 * PD_F_VOL);
      }
      if (((anyw >> (q * R)) & RMASK) == 0) continue;
#pragma unroll
      for (int r = 0; r < R; ++r) {
        const uint32_t bit = 1u << (q * R + r);
        if (anyw & bit) {
          double xi[DIM], eta[DIM];
#pragma unroll
          for (int k = 0; k < DIM; ++k) {
            xi[k] = xj[k] - xi_[r][k];
            eta[k] = uj[k] - ui_[r][k];
          }
          const double dot = dot_xi_eta<DIM>(xi, eta);
          const bool in = (mw & bit) != 0;
          bool brk = false;
          if (FRAC) {
            // s >= s_c breaks (Eq. 1.30): xi.eta - s_c ||xi||^2 >= 0, one rounding, sign read off the high word
            const double t = fma(-a.s_c, dot_xi_eta<DIM>(xi, xi), dot);
            brk = in && __double2hiint(t) >= 0 && !(nf & bit);
            if (brk) mw ^= bit;
          }
          if (in && !brk) {
            if (UNIV) acc[r] += dot; else acc[r] = fma(vj, dot, acc[r]);
          }
        }
      }
    }
    if (FRAC && mw != mw0) bits[w * 32] = mwfull & ~((mw0 & ~mw) << sh);
  }
#pragma unroll
  for (int r = 0; r < R; ++r) {
    const uint32_t e = e0 + r * 32 * PD_NF;
    if (UNIV) acc[r] *= a.vol_uniform;
    const double mi = rec[e + 32 * PD_F_MINV];   // 0 for phantoms
    const double theta = a.A * mi * acc[r];
    rec[e + 32 * PD_F_CTH(CUR)] = a.c1 * theta * mi;
    if (a.theta_out) a.theta_out[(grp * R + r) * 32 + lane] = theta;
  }
}

// ---------------------------------------------------------------------------------------------
template <int DIM, int R, bool UNIV, int CUR>
__global__ void __launch_bounds__(TPB) k_force_update(StepArgs a) {
  constexpr int EPW = 32 / R;
  constexpr uint32_t RMASK = (1u << R) - 1u;
  constexpr uint32_t BMASK = EB * R == 32 ? 0xffffffffu : ((1u << (EB * R)) - 1u);
  const int lane = threadIdx.x & 31;
  const int64_t grp = ((int64_t)blockIdx.x * TPB + threadIdx.x) >> 5;
  if (grp >= a.ngroups) return;
  double *rec = a.rec;
  const uint32_t e0 = pd_elem(grp * R * 32 + lane);

  double xi_[R][DIM], ui_[R][DIM], f[R][DIM], cth_i[R], gmu_i[R];
#pragma unroll
  for (int r = 0; r < R; ++r) {
    const uint32_t e = e0 + r * 32 * PD_NF;
#pragma unroll
    for (int k = 0; k < DIM; ++k) {
      xi_[r][k] = rec[e + 32 * (PD_F_X + k)];
      ui_[r][k] = rec[e + 32 * (PD_F_U(CUR) + k)];
      f[r][k] = 0.0;
    }
    cth_i[r] = rec[e + 32 * PD_F_CTH(CUR)];
    gmu_i[r] = rec[e + 32 * PD_F_GMU];
  }
  const uint32_t off = a.goff[grp];
  const uint32_t nwords = (a.goff[grp + 1] - off) / EPW;
  const uint32_t *col = a.col + (int64_t)off * 32 + lane;
  const uint32_t *bits = a.intact + (int64_t)(off / EPW) * 32 + lane;

  const uint32_t nblocks = nwords * (EPW / EB);
  uint32_t cn[EB], mwn = 0;
  if (nblocks) {
#pragma unroll
    for (int q = 0; q < EB; ++q) cn[q] = col[q * 32];
    mwn = bits[0];
  }
  for (uint32_t blk = 0; blk < nblocks; ++blk) {
    const uint32_t w = blk / (EPW / EB), sh = (blk % (EPW / EB)) * (EB * R);
    uint32_t c[EB];
#pragma unroll
    for (int q = 0; q < EB; ++q) c[q] = cn[q];
    const uint32_t mwfull = (EPW == EB) ? mwn : bits[w * 32];
    if (blk + 1 < nblocks) {
#pragma unroll
      for (int q = 0; q < EB; ++q) cn[q] = col[((blk + 1) * EB + q) * 32];
      if (EPW == EB) mwn = bits[(w + 1) * 32];
    }
    const uint32_t mw = (mwfull >> sh) & BMASK;
    const uint32_t anyw = __reduce_or_sync(FULL, mw);
    if (anyw == 0) continue;
    double xj[DIM], uj[DIM], gj, cj, vj = 0.0, xn[DIM], un[DIM], gn, cnx, vn = 0.0;
    {
      const double *p = rec + c[0];
#pragma unroll
      for (int k = 0; k < DIM; ++k) { xn[k] = __ldg(p + 32 * (PD_F_X + k)); un[k] = __ldg(p + 32 * (PD_F_U(CUR) + k)); }
      gn = __ldg(p + 32 * PD_F_GMU);
      cnx = __ldg(p + 32 * PD_F_CTH(CUR));
      if (!UNIV) vn = __ldg(p + 32 * PD_F_VOL);
    }
#pragma unroll
    for (int q = 0; q < EB; ++q) {
#pragma unroll
      for (int k = 0; k < DIM; ++k) { xj[k] = xn[k]; uj[k] = un[k]; }
      gj = gn; cj = cnx; vj = vn;
      if (q + 1 < EB) {
        const double *p = rec + c[q + 1];
#pragma unroll
        for (int k = 0; k < DIM; ++k) { xn[k] = __ldg(p + 32 * (PD_F_X + k)); un[k] = __ldg(p + 32 * (PD_F_U(CUR) + k)); }
        gn = __ldg(p + 32 * PD_F_GMU);
        cnx = __ldg(p + 32 * PD_F_CTH(CUR));
        if (!UNIV) vn = __ldg(p + 32 * PD_F_VOL);
      }
      if (((anyw >> (q * R)) & RMASK) == 0) continue;
#pragma unroll
      for (int r = 0; r < R; ++r) {
        const uint32_t bit = 1u << (q * R + r);
        if (anyw & bit) {
          double xi[DIM], eta[DIM];
#pragma unroll
          for (int k = 0; k < DIM; ++k) {
            xi[k] = xj[k] - xi_[r][k];
            eta[k] = uj[k] - ui_[r][k];
          }
          const double dot = dot_xi_eta<DIM>(xi, eta);
          const double r2 = dot_xi_eta<DIM>(xi, xi);
          const double d = dot * rcp_fast(r2);                       // e / xbar
          double t = fma(gmu_i[r] + gj, d, cth_i[r] + cj);
          if (!UNIV) t *= vj;
          t = (mw & bit) ? t : 0.0;                                  // rho_ij
#pragma unroll
          for (int k = 0; k < DIM; ++k) f[r][k] = fma(t, xi[k], f[r][k]);
        }
      }
    }
  }
  // ---- Eq. 2.11 + boundary dofs (App. B) ----
  double g = 1.0;
  if (a.ramp_time > 0.0) g = fmin(1.0, __ddiv_rn(__dmul_rn((double)a.step, a.dt), a.ramp_time));
#pragma unroll
  for (int r = 0; r < R; ++r) {
    const int64_t i = (grp * R + r) * 32 + lane;
    if (a.perm[i] < 0) continue;   // phantom
    const uint32_t e = e0 + r * 32 * PD_NF;
    const unsigned fl = a.flags[i];
#pragma unroll
    for (int k = 0; k < DIM; ++k) {
      double fk = f[r][k];
      if (UNIV) fk *= a.vol_uniform;
      double vk = a.v[k][i];
      double uk = ui_[r][k];
      if (fl & (1u << k)) {                       // clamped: u stays, v = 0
        vk = 0.0;
      } else if (fl & (8u << k)) {                // prescribed velocity
        vk = a.bval[k][i];
        uk = __dadd_rn(uk, __dmul_rn(a.dt, vk));
      } else {
        const double bk = (fl & PD_BODY_FORCE) ? a.bval[k][i] : 0.0;
        const double acc = __ddiv_rn(__dadd_rn(fk, __dmul_rn(g, bk)), a.rho);
        vk = __dadd_rn(vk, __dmul_rn(a.dt, acc));
        uk = __dadd_rn(uk, __dmul_rn(a.dt, vk));
      }
      a.v[k][i] = vk;
      rec[e + 32 * (PD_F_U(CUR ^ 1) + k)] = uk;
    }
  }
}

// ---------------------------------------------------------------------------------------------
// phi_i = 1 - sum_j rho_ij V_j / sum_j V_j (Eq. 1.31) and the three damage scalars.
template <int R>
__global__ void __launch_bounds__(TPB) k_damage(StepArgs a, bool univ) {
  constexpr int EPW = 32 / R;
  const int lane = threadIdx.x & 31;
  const int64_t grp = ((int64_t)blockIdx.x * TPB + threadIdx.x) >> 5;
  unsigned long long broken = 0, ge_half = 0;
  double phimax = 0.0;
  if (grp < a.ngroups) {
    const double *rec = a.rec;
    const uint32_t off = a.goff[grp];
    const uint32_t nwords = (a.goff[grp + 1] - off) / EPW;
    const uint32_t *col = a.col + (int64_t)off * 32 + lane;
    const uint32_t *bits = a.intact + (int64_t)(off / EPW) * 32 + lane;
    double sum[R];
    int cnt[R];
#pragma unroll
    for (int r = 0; r < R; ++r) { sum[r] = 0.0; cnt[r] = 0; }
    for (uint32_t w = 0; w < nwords; ++w) {
      const uint32_t mw = bits[w * 32];
      if (mw == 0) continue;
      for (int q = 0; q < EPW; ++q) {
        const uint32_t nib = (mw >> (q * R)) & ((R == 32) ? 0xffffffffu : ((1u << R) - 1u));
        if (!nib) continue;
        double vj = a.vol_uniform;
        if (!univ) vj = rec[col[(w * EPW + q) * 32] + 32 * PD_F_VOL];
#pragma unroll
        for (int r = 0; r < R; ++r)
          if ((nib >> r) & 1u) { sum[r] += vj; ++cnt[r]; }
      }
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
      const int64_t i = (grp * R + r) * 32 + lane;
      if (a.perm[i] < 0) continue;
      const double fvol = rec[pd_elem(i) + 32 * PD_F_FVOL];
      const double phi = 1.0 - sum[r] / fvol;
      a.phi[i] = phi;
      broken += (unsigned long long)(a.rowlen[i] - cnt[r]);
      ge_half += phi >= 0.5 ? 1ull : 0ull;
      phimax = fmax(phimax, phi);
    }
  }
  // warp reduce, then one atomic per warp
  unsigned long long pbits = (unsigned long long)__double_as_longlong(fmax(phimax, 0.0));  // phi >= 0: bit order = value order
  for (int o = 16; o > 0; o >>= 1) {
    broken += __shfl_xor_sync(FULL, broken, o);
    ge_half += __shfl_xor_sync(FULL, ge_half, o);
    unsigned long long other = __shfl_xor_sync(FULL, pbits, o);
    pbits = other > pbits ? other : pbits;
  }
  if (lane == 0) {
    if (broken) atomicAdd(&a.stats[0], broken);
    atomicMax(&a.stats[1], pbits);
    if (ge_half) atomicAdd(&a.stats[2], ge_half);
  }
}

StepArgs make_args(pd_sim *s) {
  StepArgs a{};
  a.ngroups = s->ngroups;
  a.rec = s->rec; a.goff = s->goff; a.col = s->col; a.intact = s->intact; a.nofail = s->nofail;
  for (int k = 0; k < 3; ++k) { a.v[k] = s->v[k]; a.bval[k] = s->bval[k]; }
  a.theta_out = nullptr; a.phi = s->phi; a.flags = s->flags; a.rowlen = s->rowlen; a.perm = s->perm;
  a.stats = s->stats_dev;
  a.A = s->A; a.c1 = s->c1; a.s_c = s->s_c; a.vol_uniform = s->vol_uniform; a.rho = s->rho; a.dt = s->dt;
  a.ramp_time = s->ramp_time; a.step = s->step;
  return a;
}

inline unsigned ngrid(const pd_sim *s) { return (unsigned)((s->ngroups + PD_GROUPS_PER_CTA - 1) / PD_GROUPS_PER_CTA); }

template <int DIM, int R, bool FRAC, bool UNIV>
void dil_cur(const StepArgs &a, int cur, unsigned grid, cudaStream_t st) {
  if (cur) k_dilatation<DIM, R, FRAC, UNIV, 1><<<grid, TPB, 0, st>>>(a);
  else k_dilatation<DIM, R, FRAC, UNIV, 0><<<grid, TPB, 0, st>>>(a);
}
template <int DIM, int R>
void dil_dispatch(const StepArgs &a, bool frac, bool univ, int cur, unsigned grid, cudaStream_t st) {
  if (frac) { if (univ) dil_cur<DIM, R, true, true>(a, cur, grid, st); else dil_cur<DIM, R, true, false>(a, cur, grid, st); }
  else { if (univ) dil_cur<DIM, R, false, true>(a, cur, grid, st); else dil_cur<DIM, R, false, false>(a, cur, grid, st); }
}
template <int DIM, int R>
void force_dispatch(const StepArgs &a, bool univ, int cur, unsigned grid, cudaStream_t st) {
  if (univ) { if (cur) k_force_update<DIM, R, true, 1><<<grid, TPB, 0, st>>>(a); else k_force_update<DIM, R, true, 0><<<grid, TPB, 0, st>>>(a); }
  else { if (cur) k_force_update<DIM, R, false, 1><<<grid, TPB, 0, st>>>(a); else k_force_update<DIM, R, false, 0><<<grid, TPB, 0, st>>>(a); }
}

}  // namespace

namespace pdi {

int launch_dilatation(pd_sim *s, double *theta_out, bool do_break) {
  StepArgs a = make_args(s);
  a.theta_out = theta_out;
  const bool frac = do_break && s->fracture;
  const unsigned grid = ngrid(s);
  if (s->dim == 2) {
    if (s->R == 1) dil_dispatch<2, 1>(a, frac, s->uniform_v, s->cur, grid, s->stream);
    else if (s->R == 2) dil_dispatch<2, 2>(a, frac, s->uniform_v, s->cur, grid, s->stream);
    else dil_dispatch<2, 4>(a, frac, s->uniform_v, s->cur, grid, s->stream);
  } else {
    if (s->R == 1) dil_dispatch<3, 1>(a, frac, s->uniform_v, s->cur, grid, s->stream);
    else if (s->R == 2) dil_dispatch<3, 2>(a, frac, s->uniform_v, s->cur, grid, s->stream);
    else dil_dispatch<3, 4>(a, frac, s->uniform_v, s->cur, grid, s->stream);
  }
  return PD_OK;
}

int launch_force_update(pd_sim *s) {
  StepArgs a = make_args(s);
  const unsigned grid = ngrid(s);
  if (s->dim == 2) {
    if (s->R == 1) force_dispatch<2, 1>(a, s->uniform_v, s->cur, grid, s->stream);
    else if (s->R == 2) force_dispatch<2, 2>(a, s->uniform_v, s->cur, grid, s->stream);
    else force_dispatch<2, 4>(a, s->uniform_v, s->cur, grid, s->stream);
  } else {
    if (s->R == 1) force_dispatch<3, 1>(a, s->uniform_v, s->cur, grid, s->stream);
    else if (s->R == 2) force_dispatch<3, 2>(a, s->uniform_v, s->cur, grid, s->stream);
    else force_dispatch<3, 4>(a, s->uniform_v, s->cur, grid, s->stream);
  }
  return PD_OK;
}

int launch_damage(pd_sim *s) {
  StepArgs a = make_args(s);
  cudaMemsetAsync(s->stats_dev, 0, 3 * sizeof(unsigned long long), s->stream);
  const unsigned grid = ngrid(s);
  if (s->R == 1) k_damage<1><<<grid, TPB, 0, s->stream>>>(a, s->uniform_v);
  else if (s->R == 2) k_damage<2><<<grid, TPB, 0, s->stream>>>(a, s->uniform_v);
  else k_damage<4><<<grid, TPB, 0, s->stream>>>(a, s->uniform_v);
  return PD_OK;
}

}  // namespace pdi
