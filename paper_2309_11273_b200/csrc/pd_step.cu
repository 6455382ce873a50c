// pd_step.cu -- the per-step kernels.
//
// One thread per node, one warp per SELL-32 slice; lane l of slice s owns sorted node 32s+l and
// walks its row slot by slot.  In the bulk of a lattice-like body all 32 lanes of a warp see the
// same neighbour offset in slot k, so the gathers x[col], u[col], ... of a warp are 256 contiguous
// bytes per array (coalesced), and the col / mask streams are read exactly once, coalesced.
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

constexpr int TPB = 256;

struct StepArgs {
  int64_t n, npad;
  const uint32_t *slice_off, *mask_off;
  const int32_t *slice_len;
  const int32_t *col;
  uint32_t *mask;
  const uint32_t *nofail;
  const double *x[3];
  const double *u[3];   // u^n
  double *unew[3];      // u^{n+1}
  double *v[3];
  const double *bval[3];
  const double *vol, *minv, *gmu, *fvol;
  double *cth;
  double *theta_out;
  double *phi;
  const uint8_t *flags;
  const int32_t *rowlen;
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
__device__ __forceinline__ void load_vec(const double *const *a, int64_t i, double *o) {
#pragma unroll
  for (int k = 0; k < DIM; ++k) o[k] = __ldg(a[k] + i);
}

template <int DIM>
__device__ __forceinline__ double dot_xi_eta(const double *xi, const double *eta) {
  double d = xi[0] * eta[0];
#pragma unroll
  for (int k = 1; k < DIM; ++k) d = fma(xi[k], eta[k], d);
  return d;
}

// ---------------------------------------------------------------------------------------------
template <int DIM, bool FRAC, bool UNIV>
__global__ void __launch_bounds__(TPB) k_dilatation(StepArgs a) {
  const int64_t i = (int64_t)blockIdx.x * TPB + threadIdx.x;
  if (i >= a.npad) return;
  const int lane = threadIdx.x & 31;
  const int64_t s = i >> 5;
  const int len = a.slice_len[s];
  const int32_t *col = a.col + (int64_t)a.slice_off[s] * 32 + lane;
  uint32_t *mask = a.mask + (int64_t)a.mask_off[s] * 32 + lane;
  const uint32_t *nofail = (FRAC && a.nofail) ? a.nofail + (int64_t)a.mask_off[s] * 32 + lane : nullptr;

  double xi_[DIM], ui_[DIM];
  load_vec<DIM>(a.x, i, xi_);
  load_vec<DIM>(a.u, i, ui_);
  double acc = 0.0;

  for (int k0 = 0; k0 < len; k0 += 32) {
    uint32_t mw = mask[(int64_t)(k0 >> 5) * 32];
    const uint32_t mw0 = mw;
    uint32_t nf = 0;
    if (FRAC && nofail) nf = nofail[(int64_t)(k0 >> 5) * 32];
    const int kend = min(32, len - k0);
    for (int b0 = 0; b0 < kend; b0 += PD_SLOT_ALIGN) {
#pragma unroll
      for (int q = 0; q < PD_SLOT_ALIGN; ++q) {
        const int b = b0 + q;
        const int64_t j = col[(int64_t)(k0 + b) * 32];
        double xi[DIM], eta[DIM];
#pragma unroll
        for (int k = 0; k < DIM; ++k) {
          xi[k] = __ldg(a.x[k] + j) - xi_[k];
          eta[k] = __ldg(a.u[k] + j) - ui_[k];
        }
        const double dot = dot_xi_eta<DIM>(xi, eta);
        bool bit = (mw >> b) & 1u;
        if (FRAC) {
          const double r2 = dot_xi_eta<DIM>(xi, xi);
          if (bit && dot >= a.s_c * r2 && !((nf >> b) & 1u)) {  // s >= s_c breaks (Eq. 1.30)
            mw &= ~(1u << b);
            bit = false;
          }
        }
        if (UNIV) {
          acc = bit ? acc + dot : acc;
        } else {
          const double vj = __ldg(a.vol + j);
          acc = bit ? fma(vj, dot, acc) : acc;
        }
      }
    }
    if (FRAC && mw != mw0) mask[(int64_t)(k0 >> 5) * 32] = mw;
  }
  if (i < a.n) {
    if (UNIV) acc *= a.vol_uniform;
    const double mi = a.minv[i];
    const double theta = a.A * mi * acc;
    a.cth[i] = a.c1 * theta * mi;
    if (a.theta_out) a.theta_out[i] = theta;
  }
}

// ---------------------------------------------------------------------------------------------
template <int DIM, bool UNIV>
__global__ void __launch_bounds__(TPB) k_force_update(StepArgs a) {
  const int64_t i = (int64_t)blockIdx.x * TPB + threadIdx.x;
  if (i >= a.npad) return;
  const int lane = threadIdx.x & 31;
  const int64_t s = i >> 5;
  const int len = a.slice_len[s];
  const int32_t *col = a.col + (int64_t)a.slice_off[s] * 32 + lane;
  const uint32_t *mask = a.mask + (int64_t)a.mask_off[s] * 32 + lane;

  double xi_[DIM], ui_[DIM], f[DIM];
  load_vec<DIM>(a.x, i, xi_);
  load_vec<DIM>(a.u, i, ui_);
  const double cth_i = a.cth[i], gmu_i = a.gmu[i];
#pragma unroll
  for (int k = 0; k < DIM; ++k) f[k] = 0.0;

  for (int k0 = 0; k0 < len; k0 += 32) {
    const uint32_t mw = mask[(int64_t)(k0 >> 5) * 32];
    const int kend = min(32, len - k0);
    for (int b0 = 0; b0 < kend; b0 += PD_SLOT_ALIGN) {
#pragma unroll
      for (int q = 0; q < PD_SLOT_ALIGN; ++q) {
        const int b = b0 + q;
        const int64_t j = col[(int64_t)(k0 + b) * 32];
        double xi[DIM], eta[DIM];
#pragma unroll
        for (int k = 0; k < DIM; ++k) {
          xi[k] = __ldg(a.x[k] + j) - xi_[k];
          eta[k] = __ldg(a.u[k] + j) - ui_[k];
        }
        const double dot = dot_xi_eta<DIM>(xi, eta);
        const double r2 = dot_xi_eta<DIM>(xi, xi);
        const double d = dot * rcp_fast(r2);                       // e / xbar
        double t = fma(gmu_i + __ldg(a.gmu + j), d, cth_i + __ldg(a.cth + j));
        if (!UNIV) t *= __ldg(a.vol + j);
        t = ((mw >> b) & 1u) ? t : 0.0;                            // rho_ij; padding slots too
#pragma unroll
        for (int k = 0; k < DIM; ++k) f[k] = fma(t, xi[k], f[k]);
      }
    }
  }
  if (i >= a.n) return;
  if (UNIV) {
#pragma unroll
    for (int k = 0; k < DIM; ++k) f[k] *= a.vol_uniform;
  }
  // ---- Eq. 2.11 + boundary dofs (App. B) ----
  const unsigned fl = a.flags[i];
  double g = 1.0;
  if (a.ramp_time > 0.0) g = fmin(1.0, __ddiv_rn(__dmul_rn((double)a.step, a.dt), a.ramp_time));
#pragma unroll
  for (int k = 0; k < DIM; ++k) {
    double vk = a.v[k][i];
    double uk = ui_[k];
    if (fl & (1u << k)) {                       // clamped: u stays, v = 0
      vk = 0.0;
    } else if (fl & (8u << k)) {                // prescribed velocity
      vk = a.bval[k][i];
      uk = __dadd_rn(uk, __dmul_rn(a.dt, vk));
    } else {
      const double bk = (fl & PD_BODY_FORCE) ? a.bval[k][i] : 0.0;
      const double acc = __ddiv_rn(__dadd_rn(f[k], __dmul_rn(g, bk)), a.rho);
      vk = __dadd_rn(vk, __dmul_rn(a.dt, acc));
      uk = __dadd_rn(uk, __dmul_rn(a.dt, vk));
    }
    a.v[k][i] = vk;
    a.unew[k][i] = uk;
  }
}

// ---------------------------------------------------------------------------------------------
// phi_i = 1 - sum_j rho_ij V_j / sum_j V_j (Eq. 1.31) and the three damage scalars.
__global__ void __launch_bounds__(TPB) k_damage(StepArgs a) {
  const int64_t i = (int64_t)blockIdx.x * TPB + threadIdx.x;
  const int lane = threadIdx.x & 31;
  unsigned long long broken = 0, ge_half = 0;
  double phi = 0.0;
  if (i < a.npad) {
    const int64_t s = i >> 5;
    const int len = a.slice_len[s];
    const int32_t *col = a.col + (int64_t)a.slice_off[s] * 32 + lane;
    const uint32_t *mask = a.mask + (int64_t)a.mask_off[s] * 32 + lane;
    double sum = 0.0;
    int intact = 0;
    for (int k0 = 0; k0 < len; k0 += 32) {
      const uint32_t mw = mask[(int64_t)(k0 >> 5) * 32];
      intact += __popc(mw);
      const int kend = min(32, len - k0);
      for (int b = 0; b < kend; ++b) {
        const int64_t j = col[(int64_t)(k0 + b) * 32];
        const double vj = __ldg(a.vol + j);
        sum = ((mw >> b) & 1u) ? sum + vj : sum;
      }
    }
    if (i < a.n) {
      phi = 1.0 - sum / a.fvol[i];
      a.phi[i] = phi;
      broken = (unsigned long long)(a.rowlen[i] - intact);
      ge_half = phi >= 0.5 ? 1ull : 0ull;
    }
  }
  // warp reduce, then one atomic per warp
  unsigned long long pbits = (unsigned long long)__double_as_longlong(fmax(phi, 0.0));  // phi >= 0: bit order = value order
  for (int o = 16; o > 0; o >>= 1) {
    broken += __shfl_xor_sync(0xffffffffu, broken, o);
    ge_half += __shfl_xor_sync(0xffffffffu, ge_half, o);
    unsigned long long other = __shfl_xor_sync(0xffffffffu, pbits, o);
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
  a.n = s->n; a.npad = s->npad;
  a.slice_off = s->slice_off; a.mask_off = s->mask_off; a.slice_len = s->slice_len;
  a.col = s->col; a.mask = s->mask; a.nofail = s->nofail;
  for (int k = 0; k < 3; ++k) {
    a.x[k] = s->x[k]; a.u[k] = s->u[s->cur][k]; a.unew[k] = s->u[s->cur ^ 1][k];
    a.v[k] = s->v[k]; a.bval[k] = s->bval[k];
  }
  a.vol = s->vol; a.minv = s->minv; a.gmu = s->gmu; a.fvol = s->fvol; a.cth = s->cth;
  a.theta_out = nullptr; a.phi = s->phi; a.flags = s->flags; a.rowlen = s->rowlen; a.stats = s->stats_dev;
  a.A = s->A; a.c1 = s->c1; a.s_c = s->s_c; a.vol_uniform = s->vol_uniform; a.rho = s->rho; a.dt = s->dt;
  a.ramp_time = s->ramp_time; a.step = s->step;
  return a;
}

inline unsigned nblk(int64_t n) { return (unsigned)((n + TPB - 1) / TPB); }

template <int DIM>
void dispatch_dilatation(const StepArgs &a, bool frac, bool univ, unsigned grid, cudaStream_t st) {
  if (frac) {
    if (univ) k_dilatation<DIM, true, true><<<grid, TPB, 0, st>>>(a);
    else k_dilatation<DIM, true, false><<<grid, TPB, 0, st>>>(a);
  } else {
    if (univ) k_dilatation<DIM, false, true><<<grid, TPB, 0, st>>>(a);
    else k_dilatation<DIM, false, false><<<grid, TPB, 0, st>>>(a);
  }
}

}  // namespace

namespace pdi {

void launch_dilatation(pd_sim *s, const double *const *ucur, double *theta_out, bool do_break) {
  StepArgs a = make_args(s);
  if (ucur) for (int k = 0; k < s->dim; ++k) a.u[k] = ucur[k];
  a.theta_out = theta_out;
  const bool frac = do_break && s->fracture;
  if (s->dim == 2) dispatch_dilatation<2>(a, frac, s->uniform_v, nblk(s->npad), s->stream);
  else dispatch_dilatation<3>(a, frac, s->uniform_v, nblk(s->npad), s->stream);
}

void launch_force_update(pd_sim *s) {
  StepArgs a = make_args(s);
  const unsigned grid = nblk(s->npad);
  if (s->dim == 2) {
    if (s->uniform_v) k_force_update<2, true><<<grid, TPB, 0, s->stream>>>(a);
    else k_force_update<2, false><<<grid, TPB, 0, s->stream>>>(a);
  } else {
    if (s->uniform_v) k_force_update<3, true><<<grid, TPB, 0, s->stream>>>(a);
    else k_force_update<3, false><<<grid, TPB, 0, s->stream>>>(a);
  }
}

void launch_damage(pd_sim *s) {
  StepArgs a = make_args(s);
  cudaMemsetAsync(s->stats_dev, 0, 3 * sizeof(unsigned long long), s->stream);
  k_damage<<<nblk(s->npad), TPB, 0, s->stream>>>(a);
}

}  // namespace pdi
