// pd_lattice_uniform.cu -- step kernels of the UNIFORM lattice layout, the
// default for the paper's own discretisation, a uniform grid.
//
// On a uniform lattice every bond of one stencil offset o has the same reference vector
// xi = (o_0 h_0, o_1 h_1, o_2 h_2) (pd_lattice.cu checks this to a few ulp of the coordinates), so the
// bond geometry the paper stores per bond (`xi`, `Xi` of App. C) collapses into a table of
// <= 128 constants: per offset xi, w = xi / ||xi||^2 and thr = s_c ||xi||^2.  Per directed bond and step
//
//   dilatation (+ break):  eta = u_j - u_i,  dot = xi . eta  [= xbar e]            7 FP64 instructions
//        breaks iff dot >= thr  (<=> e / xbar >= s_c, Eqs. 1.17, 1.30): a 64-bit INTEGER compare of the
//        bit patterns (thr > 0), no FP64 instruction; theta_i = (A / m_i) V sum_j rho_ij dot  (Eq. 1.6 / 2.3)
//   force:  d = w . eta [= e / xbar],  t = (cth_i + cth_j) + (G/m_i + G/m_j) d,  f_i += t xi      12 FP64
//        (Eq. 2.2 / 2.1), then Eq. 2.11 and the boundary dofs (App. B) fused into the epilogue,
//
// against 10-14 + 22 when xi has to be formed per bond (pd_lattice_step.cu), and a gathered neighbour
// is 24 (dilatation) / 40 (force) bytes {u, G/m, cth} instead of 48 / 64.
//
// Kernel shape = the direct kernels of pd_lattice_step.cu: one warp owns a ROW GROUP (32 lanes x R rows
// adjacent in y) at one level and walks the stencil COLUMNS (dx, dy0 .. dy0 + n - 1, dz) with a register
// window of R (+ PF prefetched) records sliding along y: in step t row r pairs with record t + r, so one
// gathered record serves up to R bonds and the R bonds of a step are independent FP64 chains.  Records
// come straight from the dense arrays by arithmetic addressing (no neighbour index exists), shared
// between warps through L1; no shared-memory staging, one CTA barrier (tables).  The mask words of the
// row group are walked word by word in registers.  A column whose R n bonds are intact on all lanes runs
// FAST (no mask test; the break test is a running integer max of the high words of dot against the high
// word of thr, any hit sends the column to the exact variant); any other column runs MASKED (predicated
// accumulation, exact break test, bits cleared).
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <vector>

#include "pd_internal.cuh"

namespace {

constexpr unsigned FULL = 0xffffffffu;

struct UCol { int off; uint8_t n, word, bit0, pad; };   // off = (dz*DY + dy0)*DX + dx (dense cells)

struct UArgs {
  int DX, DY, HX, HY, HZ, PZ;
  int nxc, nyq, nyq_used;            // x chunks; rgocc stride; row groups along y that can hold nodes
  int ncol, nw, nbits, cy, cz;       // columns; mask words; stencil bits; row groups (y) and levels (z) per CTA
  int wbeg[5];                       // columns of mask word w
  int64_t npad;
  const double2 *uxy;                // {u_0, u_1} of u^n
  const double *uz;                  // u_2 of u^n (3-D)
  double2 *uxy_w;                    // force: u^{n+1}
  double *uz_w;
  double2 *aux;                      // {G/m_i, cth_i}: written by the dilatation pass, gathered by the force pass
  uint32_t *mask;
  const uint32_t *nofail;
  const uint8_t *rgocc;
  const uint32_t *flags32;
  const double *minv;
  const double *ctab;                // [nbits][TS] per-offset constants (see ulat_tables)
  double *v[3];
  const double *bval[3];
  double *theta_out;
  double A, c1, G, vol_uniform, rrho, dt, gramp;   // gramp = g(t_n) = min(1, n dt / ramp_time)
  UCol cols[PD_LAT_MAXCOL];
};

// predicated read-only loads: no branch, so the bonds of a step stay in one basic block
__device__ __forceinline__ void ldg2_if(double2 &v, const double2 *ptr, uint32_t pred) {
  asm("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %3, 0;\n\t@p ld.global.nc.v2.f64 {%0, %1}, [%2];\n\t}"
      : "+d"(v.x), "+d"(v.y) : "l"(ptr), "r"(pred));
}
__device__ __forceinline__ void ldg1_if(double &v, const double *ptr, uint32_t pred) {
  asm("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %2, 0;\n\t@p ld.global.nc.f64 %0, [%1];\n\t}" : "+d"(v) : "l"(ptr), "r"(pred));
}

// a gathered neighbour: {u_0, u_1}, u_2 (3-D), {G/m, cth} (force pass)
struct URec { double2 xy; double z; double2 g; };

template <int DIM, bool FORCE>
__device__ __forceinline__ void u_load(URec &s, const double2 *pxy, const double *pz, const double2 *pg, int off) {
  s.xy = __ldg(pxy + off);
  if (DIM == 3) s.z = __ldg(pz + off);
  if (FORCE) s.g = __ldg(pg + off);
}
template <int DIM, bool FORCE>
__device__ __forceinline__ void u_load_if(URec &s, const double2 *pxy, const double *pz, const double2 *pg, int off, uint32_t pred) {
  ldg2_if(s.xy, pxy + off, pred);
  if (DIM == 3) ldg1_if(s.z, pz + off, pred);
  if (FORCE) ldg2_if(s.g, pg + off, pred);
}

// own-node state of the R rows of a lane
template <int DIM, bool FORCE, int R>
struct UState {
  double uo[R][DIM];
  double f[R][DIM], gmu[R], cth[R];   // force pass
  double acc[R], snap[R];             // dilatation pass
  int bad;                            // FAST dilatation: some bond may meet the break criterion
};

// constants of one stencil offset in shared memory: dilatation {xi_0, xi_1, xi_2, thr}; force {xi_0, xi_1, xi_2, -, w_0, w_1, w_2, -}
template <bool FORCE> struct UTab { static constexpr int TS = FORCE ? 8 : 4; };

// one stencil column: n steps, row r of step t pairs with record t + r (record q at base + q*DX)
template <bool MASKED, int DIM, bool FORCE, bool FRAC, int R, int PF>
__device__ __forceinline__ void u_run_col(UState<DIM, FORCE, R> &p, const double2 *pxy, const double *pz, const double2 *pg, int base,
                                          int DX, int n, const double *cst, const uint32_t (&bits)[R], const uint32_t (&nfb)[R],
                                          uint32_t (&clr)[R]) {
  constexpr int W = R + PF, TS = UTab<FORCE>::TS;
  URec S[W];
#pragma unroll
  for (int q = 0; q < W; ++q) {
    if (q < R) u_load<DIM, FORCE>(S[q], pxy, pz, pg, base + q * DX);
    else u_load_if<DIM, FORCE>(S[q], pxy, pz, pg, base + q * DX, (q - R + 2 <= n) ? 1u : 0u);
  }
  uint32_t anyp = 0;
  if (MASKED) {
    uint32_t pkd = 0;
#pragma unroll
    for (int r = 0; r < R; ++r) pkd |= bits[r] << (7 * r);
    anyp = __reduce_or_sync(FULL, pkd);
  }
  constexpr uint32_t STEPBITS = R == 4 ? 0x204081u : (R == 2 ? 0x81u : 0x1u);
#pragma unroll
  for (int t = 0; t < PD_MAXSTEP; ++t) {
    if (t < n) {
      const bool live = !MASKED || (anyp & (STEPBITS << t)) != 0;   // warp-uniform
      double eta[R][DIM], gs[R], cs[R];
      if (live) {
#pragma unroll
        for (int r = 0; r < R; ++r) {
          const URec &e = S[(t + r) % W];
          eta[r][0] = e.xy.x - p.uo[r][0];
          eta[r][1] = e.xy.y - p.uo[r][1];
          if (DIM == 3) eta[r][2] = e.z - p.uo[r][2];
          if (FORCE) { gs[r] = p.gmu[r] + e.g.x; cs[r] = p.cth[r] + e.g.y; }
        }
      }
      // record t + W takes the slot of record t (last used by row 0 just now); first needed in step t + PF + 1
      u_load_if<DIM, FORCE>(S[t % W], pxy, pz, pg, base + (t + W) * DX, (t + PF + 1 < n) ? 1u : 0u);
      if (live) {
        const double *c = cst + t * TS;
        double xi[DIM];
#pragma unroll
        for (int k = 0; k < DIM; ++k) xi[k] = c[k];
        uint32_t in = (1u << R) - 1u;
        if (MASKED) {
          in = 0;
#pragma unroll
          for (int r = 0; r < R; ++r) in |= ((bits[r] >> t) & 1u) << r;
        }
        if constexpr (!FORCE) {
          double dot[R];
#pragma unroll
          for (int r = 0; r < R; ++r) dot[r] = __dmul_rn(xi[0], eta[r][0]);
#pragma unroll
          for (int k = 1; k < DIM; ++k)
#pragma unroll
            for (int r = 0; r < R; ++r) dot[r] = fma(xi[k], eta[r][k], dot[r]);
          if (FRAC) {
            const long long thr = __double_as_longlong(c[3]);   // s_c ||xi||^2 > 0: bit order = value order
            if (!MASKED) {
              int mx = __double2hiint(dot[0]);
#pragma unroll
              for (int r = 1; r < R; ++r) mx = max(mx, __double2hiint(dot[r]));
              if (mx >= (int)(thr >> 32)) p.bad = 1;   // hi(dot) < hi(thr) => dot < thr
            } else {
              // s >= s_c breaks (Eq. 1.30): dot >= thr, exact, identical at both ends of the bond
              uint32_t brk = 0;
#pragma unroll
              for (int r = 0; r < R; ++r)
                if (((in >> r) & 1u) && __double_as_longlong(dot[r]) >= thr && !((nfb[r] >> t) & 1u)) brk |= 1u << r;
              in &= ~brk;
#pragma unroll
              for (int r = 0; r < R; ++r) clr[r] |= ((brk >> r) & 1u) << t;
            }
          }
#pragma unroll
          for (int r = 0; r < R; ++r)
            if ((in >> r) & 1u) p.acc[r] += dot[r];
        } else {
          double w[DIM], d[R], tt[R];
#pragma unroll
          for (int k = 0; k < DIM; ++k) w[k] = c[4 + k];
#pragma unroll
          for (int r = 0; r < R; ++r) d[r] = __dmul_rn(w[0], eta[r][0]);
#pragma unroll
          for (int k = 1; k < DIM; ++k)
#pragma unroll
            for (int r = 0; r < R; ++r) d[r] = fma(w[k], eta[r][k], d[r]);
#pragma unroll
          for (int r = 0; r < R; ++r) tt[r] = fma(gs[r], d[r], cs[r]);
#pragma unroll
          for (int k = 0; k < DIM; ++k)
#pragma unroll
            for (int r = 0; r < R; ++r)
              if ((in >> r) & 1u) p.f[r][k] = fma(tt[r], xi[k], p.f[r][k]);
        }
      }
    }
  }
}

// MAXT only sets the register budget (65536 / MAXT per thread: 256 -> 255, 384 -> 168, 512 -> 128); CTAs are smaller
template <int DIM, bool FORCE, bool FRAC, int R, int PF, int MAXT>
__global__ void __launch_bounds__(MAXT, 1) k_ulat(const __grid_constant__ UArgs a) {
  extern __shared__ __align__(16) unsigned char smraw[];
  constexpr int TS = UTab<FORCE>::TS;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  // shared: per-offset constants, column table
  double *stab = (double *)smraw;
  UCol *scol = (UCol *)(stab + a.nbits * TS);
  for (int c = tid; c < a.nbits * TS; c += blockDim.x) stab[c] = a.ctab[c];
  for (int c = tid; c < a.ncol; c += blockDim.x) scol[c] = a.cols[c];
  // this warp's row group: (xc, yq, z)
  const int wy = warp % a.cy, wz = warp / a.cy;
  const int xc = blockIdx.x, yq = blockIdx.y * a.cy + wy, z = blockIdx.z * a.cz + wz;   // yq counts groups of R rows
  const bool active = yq < a.nyq_used && z < a.PZ && a.rgocc[((int64_t)z * a.nyq + ((yq * R) >> 2)) * a.nxc + xc] != 0;
  const int64_t i0 = ((int64_t)(z + a.HZ) * a.DY + (yq * R + a.HY)) * a.DX + (xc * 32 + lane + a.HX);   // row 0's cell
  __syncthreads();   // tables visible (the only CTA barrier)
  if (!active) return;
  UState<DIM, FORCE, R> p;
  const double2 *pxy = a.uxy + i0;
  const double *pz = DIM == 3 ? a.uz + i0 : nullptr;
  const double2 *pg = a.aux + i0;
#pragma unroll
  for (int r = 0; r < R; ++r) {
    const double2 xy = pxy[r * a.DX];
    p.uo[r][0] = xy.x;
    p.uo[r][1] = xy.y;
    if (DIM == 3) p.uo[r][2] = pz[r * a.DX];
  }
  if constexpr (FORCE) {
#pragma unroll
    for (int r = 0; r < R; ++r) {
      const double2 g = pg[r * a.DX];
      p.gmu[r] = g.x;
      p.cth[r] = g.y;
#pragma unroll
      for (int k = 0; k < DIM; ++k) p.f[r][k] = 0.0;
    }
  } else {
#pragma unroll
    for (int r = 0; r < R; ++r) p.acc[r] = 0.0;
  }
  int c = 0;
  for (int w = 0; w < a.nw; ++w) {
    uint32_t mw[R];
#pragma unroll
    for (int r = 0; r < R; ++r) mw[r] = a.mask[(int64_t)w * a.npad + i0 + r * a.DX];
    bool dirty = false;
    const int cend = a.wbeg[w + 1];
    for (; c < cend; ++c) {
      const UCol col = scol[c];
      const int n = col.n;
      const uint32_t nmask = (1u << n) - 1u;
      uint32_t bits[R], nfb[R], clr[R];
#pragma unroll
      for (int r = 0; r < R; ++r) { nfb[r] = clr[r] = 0; bits[r] = (mw[r] >> col.bit0) & nmask; }
      uint32_t ball = bits[0];
#pragma unroll
      for (int r = 1; r < R; ++r) ball &= bits[r];
      bool slow = !__all_sync(FULL, ball == nmask);
      const double *cst = stab + (w * 32 + col.bit0) * TS;
      if (!slow) {
        if (!FORCE && FRAC) {
          p.bad = 0;
#pragma unroll
          for (int r = 0; r < R; ++r) p.snap[r] = p.acc[r];
        }
        u_run_col<false, DIM, FORCE, FRAC, R, PF>(p, pxy, pz, pg, col.off, a.DX, n, cst, bits, nfb, clr);
        if (!FORCE && FRAC) {
          if (__any_sync(FULL, p.bad)) {   // redo the column with the exact test
            slow = true;
#pragma unroll
            for (int r = 0; r < R; ++r) p.acc[r] = p.snap[r];
          }
        }
      }
      if (slow) {
        if (!FORCE && FRAC && a.nofail) {
#pragma unroll
          for (int r = 0; r < R; ++r) nfb[r] = (a.nofail[(int64_t)w * a.npad + i0 + r * a.DX] >> col.bit0) & nmask;
        }
        u_run_col<true, DIM, FORCE, FRAC, R, PF>(p, pxy, pz, pg, col.off, a.DX, n, cst, bits, nfb, clr);
        if (!FORCE && FRAC) {
#pragma unroll
          for (int r = 0; r < R; ++r)
            if (clr[r]) { mw[r] &= ~(clr[r] << col.bit0); dirty = true; }
        }
      }
    }
    if (!FORCE && FRAC && dirty) {   // broken bits back to HBM
#pragma unroll
      for (int r = 0; r < R; ++r) a.mask[(int64_t)w * a.npad + i0 + r * a.DX] = mw[r];
    }
  }
  if constexpr (!FORCE) {
    double mi[R];
#pragma unroll
    for (int r = 0; r < R; ++r) mi[r] = a.minv[i0 + r * a.DX];
#pragma unroll
    for (int r = 0; r < R; ++r) {
      const int64_t i = i0 + r * a.DX;
      const double theta = a.A * mi[r] * (p.acc[r] * a.vol_uniform);   // minv = 0 for phantoms
      a.aux[i] = make_double2(a.G * mi[r], a.c1 * theta * mi[r]);
      if (a.theta_out) a.theta_out[i] = theta;
    }
  } else {
    // ---- Eq. 2.11 + boundary dofs (App. B) ----
    double vk[R][DIM];
    unsigned fl[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
      fl[r] = a.flags32[i0 + r * a.DX];
#pragma unroll
      for (int k = 0; k < DIM; ++k) vk[r][k] = a.v[k][i0 + r * a.DX];
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
      if (p.gmu[r] == 0.0) continue;   // phantom (a node has m_i > 0)
      const int64_t i = i0 + r * a.DX;
      double un[DIM];
#pragma unroll
      for (int k = 0; k < DIM; ++k) {
        const double fk = p.f[r][k] * a.vol_uniform;
        double vv = vk[r][k];
        double uk = p.uo[r][k];
        if (fl[r] & (1u << k)) {                       // clamped: u stays, v = 0
          vv = 0.0;
        } else if (fl[r] & (8u << k)) {                // prescribed velocity
          vv = a.bval[k][i];
          uk = __dadd_rn(uk, __dmul_rn(a.dt, vv));
        } else {
          const double bk = (fl[r] & PD_BODY_FORCE) ? a.bval[k][i] : 0.0;
          const double ac = __dmul_rn(__dadd_rn(fk, __dmul_rn(a.gramp, bk)), a.rrho);   // (f + g b) / rho
          vv = __dadd_rn(vv, __dmul_rn(a.dt, ac));
          uk = __dadd_rn(uk, __dmul_rn(a.dt, vv));
        }
        a.v[k][i] = vv;
        un[k] = uk;
      }
      a.uxy_w[i] = make_double2(un[0], un[1]);
      if (DIM == 3) a.uz_w[i] = un[DIM - 1];
    }
  }
}

int env_int(const char *name, int dflt) {
  const char *e = getenv(name);
  return e ? atoi(e) : dflt;
}

struct UPrepared {
  UArgs a;
  size_t smem = 0;
  dim3 grid, block;
  int rows = 4, pf = 0, regs = 168;
};

// per stencil bit: xi = o h, w = xi / ||xi||^2, thr = s_c ||xi||^2, in the kernels' own operation order
std::vector<double> ulat_tables(const pd_sim *s, bool force) {
  const PdLattice &l = s->lat;
  const int TS = force ? 8 : 4, dim = s->dim;
  std::vector<double> h((size_t)std::max(l.nbits, 1) * TS, 0.0);
  for (int c = 0; c < l.ncol; ++c)
    for (int t = 0; t < l.cols[c].n; ++t) {
      const int b = l.cols[c].word * 32 + l.cols[c].bit0 + t;
      const int o[3] = {l.cols[c].dx, l.cols[c].dy0 + t, l.cols[c].dz};
      double xi[3] = {0, 0, 0};
      for (int k = 0; k < dim; ++k) xi[k] = (double)o[k] * l.h[k];
      double r2 = xi[0] * xi[0];
      for (int k = 1; k < dim; ++k) r2 = std::fma(xi[k], xi[k], r2);
      double *e = &h[(size_t)b * TS];
      for (int k = 0; k < dim; ++k) e[k] = xi[k];
      if (force) {
        const double ir2 = 1.0 / r2;
        for (int k = 0; k < dim; ++k) e[4 + k] = xi[k] * ir2;
      } else {
        e[3] = s->s_c * r2;
      }
    }
  return h;
}

UPrepared *ulat_prepare(pd_sim *s, bool force) {
  PdLattice &l = s->lat;
  void *&slot = l.cache[force ? 1 : 0];
  if (slot) return (UPrepared *)slot;
  UPrepared *pp = new UPrepared();
  UArgs &a = pp->a;
  a.DX = l.DX; a.DY = l.DY; a.HX = l.HX; a.HY = l.HY; a.HZ = l.HZ; a.PZ = l.PZ;
  {   // rows per lane: 4 in 3-D, 2 in 2-D (small families: more, shorter warps); -1 = the other one
    const int dflt = s->dim == 2 ? 2 : 4, r = env_int(force ? "PD_ULAT_FRC_ROWS" : "PD_ULAT_DIL_ROWS", 0);
    pp->rows = r == -1 ? 6 - dflt : ((r == 2 || r == 4) ? r : dflt);
  }
  pp->pf = std::max(0, std::min(env_int(force ? "PD_ULAT_FRC_PF" : "PD_ULAT_DIL_PF", 0), 1));
  pp->regs = env_int(force ? "PD_ULAT_FRC_REGS" : "PD_ULAT_DIL_REGS", force && s->dim == 3 ? 168 : 128);
  a.nxc = l.PX / 32; a.nyq = (l.PY + 8) / 4; a.nyq_used = l.PY / pp->rows;
  a.ncol = l.ncol; a.nw = l.nw; a.nbits = l.nbits;
  a.cy = std::max(1, std::min(env_int(force ? "PD_ULAT_FRC_CY" : "PD_ULAT_DIL_CY", 2), 8));
  a.cz = s->dim == 3 ? std::max(1, std::min(env_int(force ? "PD_ULAT_FRC_CZ" : "PD_ULAT_DIL_CZ", 2), 8)) : 1;
  while (a.cy * a.cz > 8) { if (a.cz > 1) --a.cz; else --a.cy; }   // <= 256 threads per CTA
  for (int w = 0; w < 5; ++w) a.wbeg[w] = l.wbeg[w];
  a.npad = s->npad;
  for (int c = 0; c < l.ncol; ++c) {
    const PdLatCol &src = l.cols[c];
    a.cols[c].off = (src.dz * l.DY + src.dy0) * l.DX + src.dx;
    a.cols[c].n = src.n; a.cols[c].word = src.word; a.cols[c].bit0 = src.bit0; a.cols[c].pad = 0;
  }
  a.aux = l.aux;
  a.mask = l.mask; a.nofail = l.nofail; a.rgocc = l.rgocc; a.flags32 = l.flags32; a.minv = s->minv;
  for (int q = 0; q < 3; ++q) { a.v[q] = s->v[q]; a.bval[q] = s->bval[q]; }
  a.theta_out = nullptr;
  a.A = s->A; a.c1 = s->c1; a.G = s->G; a.vol_uniform = s->vol_uniform; a.rrho = 1.0 / s->rho; a.dt = s->dt;
  a.gramp = 1.0;
  const int TS = force ? 8 : 4;
  if (!l.ctab[force]) {
    const std::vector<double> h = ulat_tables(s, force);
    l.ctab[force] = (double *)pdi::dev_alloc(s, sizeof(double) * h.size());
    if (!l.ctab[force]) { delete pp; return nullptr; }
    if (cudaMemcpyAsync(l.ctab[force], h.data(), sizeof(double) * h.size(), cudaMemcpyHostToDevice, s->stream) != cudaSuccess ||
        cudaStreamSynchronize(s->stream) != cudaSuccess) { delete pp; return nullptr; }
  }
  a.ctab = l.ctab[force];
  const int nwarp = a.cy * a.cz;
  pp->smem = (size_t)l.nbits * TS * sizeof(double) + (size_t)l.ncol * sizeof(UCol);
  pp->block = dim3((unsigned)(nwarp * 32));
  pp->grid = dim3((unsigned)a.nxc, (unsigned)((a.nyq_used + a.cy - 1) / a.cy), (unsigned)((l.PZ + a.cz - 1) / a.cz));
  slot = pp;
  return pp;
}

template <int DIM, bool FORCE, bool FRAC, int R, int PF>
void ulat_dispatch2(const UPrepared *pp, cudaStream_t st) {
  if (pp->regs >= 255) k_ulat<DIM, FORCE, FRAC, R, PF, 256><<<pp->grid, pp->block, pp->smem, st>>>(pp->a);
  else if (pp->regs >= 168) k_ulat<DIM, FORCE, FRAC, R, PF, 384><<<pp->grid, pp->block, pp->smem, st>>>(pp->a);
  else k_ulat<DIM, FORCE, FRAC, R, PF, 512><<<pp->grid, pp->block, pp->smem, st>>>(pp->a);
}
template <int DIM, bool FORCE, bool FRAC>
void ulat_dispatch(const UPrepared *pp, cudaStream_t st) {
  if (pp->rows == 2) { if (pp->pf) ulat_dispatch2<DIM, FORCE, FRAC, 2, 1>(pp, st); else ulat_dispatch2<DIM, FORCE, FRAC, 2, 0>(pp, st); }
  else { if (pp->pf) ulat_dispatch2<DIM, FORCE, FRAC, 4, 1>(pp, st); else ulat_dispatch2<DIM, FORCE, FRAC, 4, 0>(pp, st); }
}

}  // namespace

namespace pdi {

void ulat_free_cache(pd_sim *s) {
  for (int q = 0; q < 2; ++q) {
    delete (UPrepared *)s->lat.cache[q];
    s->lat.cache[q] = nullptr;
  }
}

int ulat_launch_dilatation(pd_sim *s, double *theta_out, bool do_break) {
  UPrepared *pp = ulat_prepare(s, false);
  if (!pp) { set_error("device allocation failed"); return PD_ERR_ALLOC; }
  const PdLattice &l = s->lat;
  UArgs &a = pp->a;
  a.uxy = l.uxy[s->cur]; a.uz = l.uz[s->cur]; a.uxy_w = nullptr; a.uz_w = nullptr;
  a.theta_out = theta_out;
  const bool frac = do_break && s->fracture;
  if (s->dim == 2) { if (frac) ulat_dispatch<2, false, true>(pp, s->stream); else ulat_dispatch<2, false, false>(pp, s->stream); }
  else { if (frac) ulat_dispatch<3, false, true>(pp, s->stream); else ulat_dispatch<3, false, false>(pp, s->stream); }
  return PD_OK;
}

int ulat_launch_force_update(pd_sim *s) {
  UPrepared *pp = ulat_prepare(s, true);
  if (!pp) { set_error("device allocation failed"); return PD_ERR_ALLOC; }
  const PdLattice &l = s->lat;
  UArgs &a = pp->a;
  a.uxy = l.uxy[s->cur]; a.uz = l.uz[s->cur]; a.uxy_w = l.uxy[s->cur ^ 1]; a.uz_w = l.uz[s->cur ^ 1];
  a.gramp = 1.0;
  if (s->ramp_time > 0.0) a.gramp = std::min(1.0, ((double)s->step * s->dt) / s->ramp_time);
  if (s->dim == 2) ulat_dispatch<2, true, false>(pp, s->stream); else ulat_dispatch<3, true, false>(pp, s->stream);
  return PD_OK;
}

}  // namespace pdi
