// pd_bond.cuh -- the per-bond arithmetic of the two step kernels, shared by the two neighbour-list
// layouts (pd_step.cu: windowed sliced ELL for any point cloud; pd_lattice.cu: dense lattice tiles).
//
//   dilatation (+ break):  dot = xi . eta  [= xbar * e, sqrt-free; rows a1, a2 of SURVEY.md 8(a)]
//        FRAC: dot - s_c ||xi||^2 >= 0  <=>  e / xbar >= s_c  (Eqs. 1.17, 1.30): the bond breaks
//        theta_i = (A/m_i) sum_j rho_ij dot V_j           (Eq. 1.6 / 2.3)
//   force:  f_i = sum_j rho_ij V_j [ cth_i + cth_j + (G/m_i + G/m_j) dot/||xi||^2 ] xi   (Eq. 2.2 / 2.1)
//
// Both ends of a bond take the identical break decision because -a*-b == a*b exactly in every
// product and the sums run in the same component order; every code path (fast / masked, ELL /
// lattice) uses exactly this arithmetic.
#pragma once
#include "pd_internal.cuh"

namespace pdb {

constexpr unsigned FULL = 0xffffffffu;

// one gathered neighbour: DIM pairs {x_k, u_k} (+ {G/m, cth}) (+ V_j)
template <int DIM, bool AUX, bool VOL>
struct Ent {
  double2 p[DIM];
  double2 g;
  double vj;
};

template <int DIM>
__device__ __forceinline__ double dot3(const double *x, const double *y) {
  double d = __dmul_rn(x[0], y[0]);
#pragma unroll
  for (int k = 1; k < DIM; ++k) d = fma(x[k], y[k], d);
  return d;
}

// GEOM (variant): the geometric extension of the paper's loop code, e = ||xi + eta|| - ||xi||
// (App. C), in place of the linearized M . eta.  Returned as xbar * e, the quantity the
// linearized path calls dot = xi . eta, so that everything downstream (theta, break test, e / xbar = dot / ||xi||^2)
// is unchanged.  Evaluated like the listing (and the oracle): squares summed in component order, individually
// rounded, two square roots.
template <int DIM>
__device__ __forceinline__ double dot_geom(const double *xi, const double *eta) {
  double r2 = __dmul_rn(xi[0], xi[0]), y2;
  {
    const double y = __dadd_rn(xi[0], eta[0]);
    y2 = __dmul_rn(y, y);
  }
#pragma unroll
  for (int k = 1; k < DIM; ++k) {
    const double y = __dadd_rn(xi[k], eta[k]);
    r2 = __dadd_rn(r2, __dmul_rn(xi[k], xi[k]));
    y2 = __dadd_rn(y2, __dmul_rn(y, y));
  }
  const double xbar = sqrt(r2);
  return __dmul_rn(xbar, __dsub_rn(sqrt(y2), xbar));
}

// dilatation (+ break) policy: R rows per lane.
// FILT (lattice layout): the fast pass does not evaluate dot - s_c ||xi||^2 per bond; it keeps the
// maximum of the HIGH WORDS of dot over a step and compares it with the high word of
// thr = s_c * min ||xi||^2 of that stencil offset (a static lower bound over all bonds, pd_lattice.cu):
// hi(dot) < hi(thr) => dot < thr <= s_c ||xi||^2 => the exact test is negative.  Anything else sends
// the bonds to the masked variant, which evaluates the exact test.  (Integer compares on the ALU pipe
// instead of 4 FP64 instructions per bond.)
template <int DIM, bool FRAC, bool UNIV, int R, bool FILT = false, bool GEOM = false>
struct DilPolicy {
  using E = Ent<DIM, false, !UNIV>;
  static constexpr bool kFrac = FRAC;
  double xo[R][DIM], uo[R][DIM], acc[R], snap[R];
  double s_c;
  int sg;   // AND of the sign words of dot - s_c r2 over the fast path's bonds
  int mxhi; // FILT: max high word of dot over the bonds of the current step

  __device__ __forceinline__ void fast_begin() {
    if (FRAC) {
#pragma unroll
      for (int r = 0; r < R; ++r) snap[r] = acc[r];
      sg = (int)0x80000000;
      mxhi = (int)0x80000000;
    }
  }
  // FILT: end of a fast step whose bonds share the threshold high word thr_hi
  __device__ __forceinline__ void step_end(int thr_hi) {
    if (FRAC && FILT) {
      if (mxhi >= thr_hi) sg = 0;
      mxhi = (int)0x80000000;
    }
  }
  // true: some bond of the fast pass met the break criterion on some lane; the accumulators are
  // rolled back and the caller redoes the same bonds with the masked variant
  __device__ __forceinline__ bool fast_failed() {
    if (!FRAC) return false;
    if (!__any_sync(FULL, sg >= 0)) return false;
#pragma unroll
    for (int r = 0; r < R; ++r) acc[r] = snap[r];
    return true;
  }
  // returns true if the bond breaks now (MASKED && FRAC only)
  template <bool MASKED>
  __device__ __forceinline__ bool bond(int r, const E &e, bool in, bool nofail) {
    double xi[DIM], eta[DIM];
#pragma unroll
    for (int k = 0; k < DIM; ++k) {
      xi[k] = e.p[k].x - xo[r][k];
      eta[k] = e.p[k].y - uo[r][k];
    }
    const double dot = GEOM ? dot_geom<DIM>(xi, eta) : dot3<DIM>(xi, eta);
    bool brk = false;
    if (!MASKED) in = true;
    if (FRAC && FILT && !MASKED) {
      mxhi = max(mxhi, __double2hiint(dot));
    } else if (FRAC) {
      // s >= s_c breaks (Eq. 1.30): xi.eta - s_c ||xi||^2 >= 0, one rounding, sign read off the high word
      const double t = fma(-s_c, dot3<DIM>(xi, xi), dot);
      if (MASKED) {
        brk = in && __double2hiint(t) >= 0 && !nofail;
        if (brk) in = false;
      } else {
        sg &= __double2hiint(t);
      }
    }
    if (in) {
      if (UNIV) acc[r] += dot; else acc[r] = fma(e.vj, dot, acc[r]);
    }
    return brk;
  }

  // ---- staged form of one STEP (the R bonds of the R rows with R records), written phase by phase
  // over the rows so that every instruction has R - 1 independent ones between it and its consumer.
  // Same arithmetic, operand by operand, as bond().
  double xi_[R][DIM], eta_[R][DIM];
  __device__ __forceinline__ void diffs(int r, const E &e) {
#pragma unroll
    for (int k = 0; k < DIM; ++k) {
      xi_[r][k] = e.p[k].x - xo[r][k];
      eta_[r][k] = e.p[k].y - uo[r][k];
    }
  }
  // in / nofail: bit r = row r (MASKED only); returns the rows whose bond breaks now
  template <bool MASKED>
  __device__ __forceinline__ uint32_t finish(uint32_t in, uint32_t nofail) {
    static_assert(UNIV, "staged form: uniform volume only");   // (never taken with GEOM: the lattice kernels launch GEOM unstaged)
    double dot[R], r2[R];
#pragma unroll
    for (int r = 0; r < R; ++r) dot[r] = __dmul_rn(xi_[r][0], eta_[r][0]);
    constexpr bool EXACT = FRAC && (MASKED || !FILT);
    if (EXACT) {
#pragma unroll
      for (int r = 0; r < R; ++r) r2[r] = __dmul_rn(xi_[r][0], xi_[r][0]);
    }
#pragma unroll
    for (int k = 1; k < DIM; ++k) {
#pragma unroll
      for (int r = 0; r < R; ++r) dot[r] = fma(xi_[r][k], eta_[r][k], dot[r]);
      if (EXACT) {
#pragma unroll
        for (int r = 0; r < R; ++r) r2[r] = fma(xi_[r][k], xi_[r][k], r2[r]);
      }
    }
    uint32_t brk = 0;
    if (!MASKED) in = (1u << R) - 1u;
    if (FRAC && FILT && !MASKED) {
#pragma unroll
      for (int r = 0; r < R; ++r) mxhi = max(mxhi, __double2hiint(dot[r]));
    } else if (FRAC) {
      double t[R];
#pragma unroll
      for (int r = 0; r < R; ++r) t[r] = fma(-s_c, r2[r], dot[r]);
      if (MASKED) {
#pragma unroll
        for (int r = 0; r < R; ++r)
          if (((in >> r) & 1u) && __double2hiint(t[r]) >= 0 && !((nofail >> r) & 1u)) brk |= 1u << r;
        in &= ~brk;
      } else {
#pragma unroll
        for (int r = 0; r < R; ++r) sg &= __double2hiint(t[r]);
      }
    }
#pragma unroll
    for (int r = 0; r < R; ++r)
      if ((in >> r) & 1u) acc[r] += dot[r];
    return brk;
  }
};

// 1/x seed: MUFU.RCP64H (relative error about 2^-20)
__device__ __forceinline__ double rcp_seed(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  return y;
}

// force policy
template <int DIM, bool UNIV, int R, bool GEOM = false>
struct ForcePolicy {
  using E = Ent<DIM, true, !UNIV>;
  static constexpr bool kFrac = false;
  double xo[R][DIM], uo[R][DIM], f[R][DIM], cth_i[R], gmu_i[R];

  __device__ __forceinline__ void fast_begin() {}
  __device__ __forceinline__ void step_end(int) {}
  __device__ __forceinline__ bool fast_failed() { return false; }
  template <bool MASKED>
  __device__ __forceinline__ bool bond(int r, const E &e, bool in, bool) {
    double xi[DIM], eta[DIM];
#pragma unroll
    for (int k = 0; k < DIM; ++k) {
      xi[k] = e.p[k].x - xo[r][k];
      eta[k] = e.p[k].y - uo[r][k];
    }
    const double dot = GEOM ? dot_geom<DIM>(xi, eta) : dot3<DIM>(xi, eta);
    const double r2 = dot3<DIM>(xi, xi);
    // d = dot / r2 = e / xbar: seed y, err = 1 - r2 y, d = dot y (1 + err + err^2)  (relative error err^3 ~ 2^-60)
    const double y = rcp_seed(r2);
    const double err = fma(-r2, y, 1.0);
    const double q = __dmul_rn(dot, y);
    const double d = fma(q, fma(err, err, err), q);
    double t = fma(gmu_i[r] + e.g.x, d, cth_i[r] + e.g.y);
    if (!UNIV) t *= e.vj;
    if (!MASKED) in = true;   // rho_ij
    if (in) {
#pragma unroll
      for (int k = 0; k < DIM; ++k) f[r][k] = fma(t, xi[k], f[r][k]);
    }
    return false;
  }

  // ---- staged form of one step (see DilPolicy): same arithmetic as bond(), phase by phase over the rows
  double xi_[R][DIM], eta_[R][DIM], gs_[R], cs_[R];
  __device__ __forceinline__ void diffs(int r, const E &e) {
#pragma unroll
    for (int k = 0; k < DIM; ++k) {
      xi_[r][k] = e.p[k].x - xo[r][k];
      eta_[r][k] = e.p[k].y - uo[r][k];
    }
    gs_[r] = gmu_i[r] + e.g.x;
    cs_[r] = cth_i[r] + e.g.y;
  }
  template <bool MASKED>
  __device__ __forceinline__ uint32_t finish(uint32_t in, uint32_t) {
    static_assert(UNIV, "staged form: uniform volume only");   // (never taken with GEOM: the lattice kernels launch GEOM unstaged)
    double dot[R], r2[R], y[R], err[R], q[R], t[R];
#pragma unroll
    for (int r = 0; r < R; ++r) r2[r] = __dmul_rn(xi_[r][0], xi_[r][0]);
#pragma unroll
    for (int r = 0; r < R; ++r) dot[r] = __dmul_rn(xi_[r][0], eta_[r][0]);
#pragma unroll
    for (int k = 1; k < DIM; ++k) {
#pragma unroll
      for (int r = 0; r < R; ++r) r2[r] = fma(xi_[r][k], xi_[r][k], r2[r]);
#pragma unroll
      for (int r = 0; r < R; ++r) dot[r] = fma(xi_[r][k], eta_[r][k], dot[r]);
    }
#pragma unroll
    for (int r = 0; r < R; ++r) y[r] = rcp_seed(r2[r]);
#pragma unroll
    for (int r = 0; r < R; ++r) err[r] = fma(-r2[r], y[r], 1.0);
#pragma unroll
    for (int r = 0; r < R; ++r) q[r] = __dmul_rn(dot[r], y[r]);
#pragma unroll
    for (int r = 0; r < R; ++r) err[r] = fma(err[r], err[r], err[r]);
#pragma unroll
    for (int r = 0; r < R; ++r) q[r] = fma(q[r], err[r], q[r]);
#pragma unroll
    for (int r = 0; r < R; ++r) t[r] = fma(gs_[r], q[r], cs_[r]);
    if (!MASKED) in = (1u << R) - 1u;   // rho_ij
#pragma unroll
    for (int k = 0; k < DIM; ++k)
#pragma unroll
      for (int r = 0; r < R; ++r)
        if ((in >> r) & 1u) f[r][k] = fma(t[r], xi_[r][k], f[r][k]);
    return 0u;
  }
};

}  // namespace pdb
