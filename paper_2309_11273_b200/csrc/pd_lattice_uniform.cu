// pd_lattice_uniform.cu -- step kernels of the UNIFORM lattice layout, the
// default for the paper's own discretisation, a uniform grid.
//
// On a uniform lattice every bond of one stencil offset o has the same reference vector
// xi = (o_0 h_0, o_1 h_1, o_2 h_2) (pd_lattice.cu checks this to a few ulp of the coordinates), so the
// bond geometry the paper stores per bond (`xi`, `Xi` of App. C) collapses into a table of
// <= 128 constants: per offset xi, 1 / ||xi||^2 and thr = s_c ||xi||^2.  Per directed bond and step
//
//   dilatation (+ break):  eta = u_j - u_i,  dot = xi . eta  [= xbar e]            7 FP64 instructions
//        breaks iff dot >= thr  (<=> e / xbar >= s_c, Eqs. 1.17, 1.30): a 64-bit INTEGER compare of the
//        bit patterns (thr > 0), no FP64 instruction; theta_i = (A / m_i) V sum_j rho_ij dot  (Eq. 1.6 / 2.3)
//   force:  d = dot / ||xi||^2 [= e / xbar],  t = (cth_i + cth_j) + (G/m_i + G/m_j) d,  f_i += t xi   12 FP64
//        (Eq. 2.2 / 2.1; the x and z parts of t xi are summed per column: xi_x, xi_z are column constants),
//        then Eq. 2.11 and the boundary dofs (App. B) fused into the epilogue,
//
// against 10-14 + 22 when xi has to be formed per bond (pd_lattice_step.cu), and a gathered neighbour
// is 24 (dilatation) / 40 (force) bytes {u, G/m, cth} instead of 48 / 64.
//
// Kernel shape: one warp owns a ROW GROUP (32 lanes x R rows adjacent in y) at one level z and walks the
// stencil COLUMNS (dx, dy0 .. dy0 + n - 1, dz) with a register window of R records sliding along y: in
// step t row r pairs with record t + r, so one gathered record serves up to R bonds and the R bonds of a
// step are independent FP64 chains.  A column whose R n bonds are intact on all lanes runs FAST (no mask
// test; the break test is a running integer max of the high words of dot against the high word of thr,
// any hit sends the column to the exact variant); any other column runs MASKED (bond terms zeroed by
// select, exact break test, bits cleared).  The mask words of a row group are walked in registers.
//
// Where the records come from:
//   STAGED (default): the warps of a CTA are row groups adjacent in y at ONE level z.  For every plane
//     z + dz of the stencil the cells the CTA can reach (USX x sy) are brought into shared memory by TMA
//     (cp.async.bulk.tensor, NB buffers in flight, completion on an mbarrier; a buffer is handed back by
//     the last warp that leaves it -- a shared counter, no CTA barrier), and every record address is a
//     compile-time offset from one shared-memory pointer.
//   DIRECT (stencils wider than the staged halo, or no tensor maps): records are read from the dense
//     arrays by arithmetic addressing through L1, as in pd_lattice_step.cu.

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <type_traits>
#include <vector>

#include "pd_internal.cuh"
#include "pd_stage.cuh"

namespace {

using namespace pdstage;

constexpr unsigned FULL = 0xffffffffu;
constexpr int UH = 3;              // STAGED kernels: halo of a staged plane = largest stencil radius in x and y they take
constexpr int USX = 32 + 2 * UH;   // cells per staged row (compile-time pitch: every record address is an immediate offset)
constexpr int UMAXSEG = 16;

// one stencil column; 32 bytes, read with two 16-byte shared-memory loads
struct __align__(16) UCol {
  int off;             // DIRECT: (dz*DY + dy0)*DX + dx (dense cells)
  int soff;            // STAGED: dy0*USX + dx
  uint8_t n, word, bit0, pad;
  int tab;             // index of the column's first step in the per-step constant table
  double xi0, xi2;     // x and z components of xi: constant along the column
};
// a run of columns inside one plane and one mask word
struct USeg { int16_t plane, word; int16_t cbeg, cend; };

struct UArgs {
  int DX, DY, HX, HY, HZ, PZ;
  int nxc, nyq, nyq_used;            // x chunks; rgocc stride; row groups along y that can hold nodes
  int ncol, nbits, nw, cy, cz;       // columns; stencil bits; mask words; row groups (y) and levels (z) per CTA
  int np, nseg, sy;                  // planes (distinct dz), segments; STAGED: rows of a staged plane = R cy + 2 UH
  int pdz[8];                        // dz of plane p
  USeg seg[UMAXSEG];                 // plane-major, word-minor
  uint32_t fullw[4];                 // all stencil bits of mask word w
  uint32_t o_col, o_buf, o_z, o_g, plane_bytes, tx_bytes;   // shared-memory carve-up (bytes), see ulat_smem
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
  const double2 *ctab;               // [nbits + 8] per stencil bit {xi_1, thr} (dilatation) / {xi_1, 1 / ||xi||^2} (force)
  const UCol *cols;                  // [ncol] device copy of the column table
  double *v[3];
  const double *bval[3];
  double *theta_out;
  double A, c1, G, vol_uniform, rrho, dt, gramp;   // gramp = g(t_n) = min(1, n dt / ramp_time)
  alignas(64) CUtensorMap tm_xy, tm_z, tm_g;       // STAGED: 3-D tiled maps of uxy (as doubles), uz, aux (as doubles)
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

// where the records of a column come from.  Record q of the current column:
//   SrcGlobal: the dense arrays, cell i0 + off + q DX (L1-cached read-only loads, DX known at run time)
//   SrcShared: the staged plane in shared memory, cell s0 + soff + q USX (USX a compile-time constant)
template <int DIM, bool FORCE>
struct SrcGlobal {
  const double2 *pxy; const double *pz; const double2 *pg;
  int DX, base;
  __device__ __forceinline__ void column(int off, int) { base = off; }
  __device__ __forceinline__ void load(URec &s, int q) const {
    const int off = base + q * DX;
    s.xy = __ldg(pxy + off);
    if (DIM == 3) s.z = __ldg(pz + off);
    if (FORCE) s.g = __ldg(pg + off);
  }
  __device__ __forceinline__ void load_if(URec &s, int q, bool pred) const {
    const int off = base + q * DX;
    ldg2_if(s.xy, pxy + off, pred);
    if (DIM == 3) ldg1_if(s.z, pz + off, pred);
    if (FORCE) ldg2_if(s.g, pg + off, pred);
  }
};
template <int DIM, bool FORCE>
struct SrcShared {
  const double2 *sxy; const double *sz; const double2 *sg;   // the thread's row-0 own cell inside the staged plane
  const double2 *cxy; const double *cz; const double2 *cg;   // ... shifted to record 0 of the current column
  __device__ __forceinline__ void column(int, int soff) {
    cxy = sxy + soff;
    if (DIM == 3) cz = sz + soff;
    if (FORCE) cg = sg + soff;
  }
  __device__ __forceinline__ void load(URec &s, int q) const {
    s.xy = cxy[q * USX];
    if (DIM == 3) s.z = cz[q * USX];
    if (FORCE) s.g = cg[q * USX];
  }
  __device__ __forceinline__ void load_if(URec &s, int q, bool pred) const {
    if (pred) load(s, q);
  }
};

// own-node state of the R rows of a lane
template <int DIM, bool FORCE, int R>
struct UState {
  double uo[R][DIM];
  double f[R][DIM], gmu[R], cth[R];   // force pass
  double acc[R], snap[R];             // dilatation pass
  int bad;                            // FAST dilatation: some bond may meet the break criterion
};

// one stencil column: n steps, row r of step t pairs with record t + r.
// xi0, xi2: the column's x and z components of xi; cst[t] = {xi_1, thr | 1/||xi||^2} of step t.
template <bool MASKED, int DIM, bool FORCE, bool FRAC, int R, class SRC>
__device__ __forceinline__ void u_run_col(UState<DIM, FORCE, R> &p, const SRC &src, int n, double xi0, double xi2, const double2 *cst,
                                          const uint32_t (&bits)[R], const uint32_t (&nfb)[R], uint32_t (&clr)[R]) {
  URec S[R];
#pragma unroll
  for (int q = 0; q < R; ++q) src.load(S[q], q);
  uint32_t anyp = 0;
  if (MASKED) {
    uint32_t pkd = 0;
#pragma unroll
    for (int r = 0; r < R; ++r) pkd |= bits[r] << (7 * r);
    anyp = __reduce_or_sync(FULL, pkd);
  }
  constexpr uint32_t STEPBITS = R == 4 ? 0x204081u : (R == 2 ? 0x81u : 0x1u);
  double ts[R];   // force: sum of t over the column (the x and z parts of t xi are added at the end)
#pragma unroll
  for (int r = 0; r < R; ++r) ts[r] = 0.0;
  double2 cbuf[2];
  cbuf[0] = cst[0];
#pragma unroll
  for (int t = 0; t < PD_MAXSTEP; ++t) {
    if (t >= n) break;
    const bool live = !MASKED || (anyp & (STEPBITS << t)) != 0;   // warp-uniform
    const double2 cc = cbuf[t & 1];
    if (t + 1 < PD_MAXSTEP) cbuf[(t + 1) & 1] = cst[t + 1];   // the next step's constants, one step ahead (the table has slack)
    double eta[R][DIM], gs[R], cs[R];
    if (live) {
#pragma unroll
      for (int r = 0; r < R; ++r) {
        const URec &e = S[(t + r) % R];
        eta[r][0] = e.xy.x - p.uo[r][0];
        eta[r][1] = e.xy.y - p.uo[r][1];
        if (DIM == 3) eta[r][2] = e.z - p.uo[r][2];
        if (FORCE) { gs[r] = p.gmu[r] + e.g.x; cs[r] = p.cth[r] + e.g.y; }
      }
    }
    // record t + R takes the slot of record t (last used by row 0 just now); first needed in step t + 1
    src.load_if(S[t % R], t + R, t + 1 < n);
    if (live) {
      double dot[R];
#pragma unroll
      for (int r = 0; r < R; ++r) dot[r] = __dmul_rn(xi0, eta[r][0]);
#pragma unroll
      for (int r = 0; r < R; ++r) dot[r] = fma(cc.x, eta[r][1], dot[r]);
      if (DIM == 3) {
#pragma unroll
        for (int r = 0; r < R; ++r) dot[r] = fma(xi2, eta[r][2], dot[r]);
      }
      if constexpr (!FORCE) {
        if (FRAC && !MASKED) {
          const int thr_hi = __double2hiint(cc.y);   // s_c ||xi||^2 > 0: bit order = value order
          int mx = __double2hiint(dot[0]);
#pragma unroll
          for (int r = 1; r < R; ++r) mx = max(mx, __double2hiint(dot[r]));
          if (mx >= thr_hi) p.bad = 1;   // hi(dot) < hi(thr) => dot < thr
        }
        if (MASKED) {
          const long long thr = __double_as_longlong(cc.y);
#pragma unroll
          for (int r = 0; r < R; ++r) {
            bool in = (bits[r] >> t) & 1u;
            if (FRAC) {   // s >= s_c breaks (Eq. 1.30): dot >= thr, exact, identical at both ends of the bond
              const bool brk = in && __double_as_longlong(dot[r]) >= thr && !((nfb[r] >> t) & 1u);
              if (brk) { clr[r] |= 1u << t; in = false; }
            }
            p.acc[r] += in ? dot[r] : 0.0;   // + 0.0 leaves the sum as it is
          }
        } else {
#pragma unroll
          for (int r = 0; r < R; ++r) p.acc[r] += dot[r];
        }
      } else {
        double tt[R];
#pragma unroll
        for (int r = 0; r < R; ++r) tt[r] = __dmul_rn(dot[r], cc.y);   // d = e / xbar
#pragma unroll
        for (int r = 0; r < R; ++r) tt[r] = fma(gs[r], tt[r], cs[r]);
        if (MASKED) {   // rho_ij = 0: t = 0
#pragma unroll
          for (int r = 0; r < R; ++r) tt[r] = ((bits[r] >> t) & 1u) ? tt[r] : 0.0;
        }
#pragma unroll
        for (int r = 0; r < R; ++r) ts[r] += tt[r];
#pragma unroll
        for (int r = 0; r < R; ++r) p.f[r][1] = fma(tt[r], cc.x, p.f[r][1]);
      }
    }
  }
  if constexpr (FORCE) {
#pragma unroll
    for (int r = 0; r < R; ++r) {
      p.f[r][0] = fma(ts[r], xi0, p.f[r][0]);
      if (DIM == 3) p.f[r][2] = fma(ts[r], xi2, p.f[r][2]);
    }
  }
}
// shared-memory carve-up (bytes): [0, 128) mbarriers + counters | per-step constants | column table | NB plane buffers
struct USmem { uint32_t tab, col, buf, z, g, plane, total; };
inline USmem ulat_smem(int dim, bool force, bool staged, int nbits, int ncol, int sy, int nb) {
  USmem m;
  auto up = [](uint32_t x) { return (x + 127u) & ~127u; };
  m.tab = 128;
  m.col = up(m.tab + (nbits + 8) * 16);
  m.buf = up(m.col + ncol * (uint32_t)sizeof(UCol));
  m.z = up((uint32_t)sy * USX * 16);
  m.g = m.z + (dim == 3 ? up((uint32_t)sy * USX * 8) : 0);
  m.plane = m.g + (force ? up((uint32_t)sy * USX * 16) : 0);
  m.total = m.buf + (staged ? nb * m.plane : 0);
  return m;
}

// MAXT only sets the register budget (65536 / MAXT per thread: 256 -> 255, 384 -> 168, 512 -> 128, 640 -> 102); CTAs are smaller.
template <int DIM, bool FORCE, bool FRAC, int R, bool STAGED, int NB, int MAXT>
__global__ void __launch_bounds__(MAXT, 1) k_ulat(const __grid_constant__ UArgs a) {
  extern __shared__ __align__(128) unsigned char smraw[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  uint64_t *full = (uint64_t *)smraw;           // [NB] plane has landed
  int *left = (int *)(smraw + 64);              // [NB] warps that have not left the buffer yet
  double2 *stab = (double2 *)(smraw + 128);
  UCol *scol = (UCol *)(smraw + a.o_col);
  for (int c = tid; c < a.nbits + 8; c += blockDim.x) stab[c] = a.ctab[c];
  {
    const int4 *src = (const int4 *)a.cols;
    int4 *dst = (int4 *)scol;
    for (int c = tid; c < a.ncol * 2; c += blockDim.x) dst[c] = src[c];
  }
  const int nwarp = blockDim.x >> 5;
  if (STAGED && tid == 0) {
#pragma unroll
    for (int b = 0; b < NB; ++b) { mbar_init(&full[b], 1); left[b] = nwarp; }
    mbar_fence_init();
  }
  // this warp's row group: (xc, yq, z)
  const int wy = warp % a.cy, wz = warp / a.cy;
  const int xc = blockIdx.x, yq = blockIdx.y * a.cy + wy, z = blockIdx.z * a.cz + wz;   // yq counts groups of R rows
  const bool active = yq < a.nyq_used && z < a.PZ && a.rgocc[((int64_t)z * a.nyq + ((yq * R) >> 2)) * a.nxc + xc] != 0;
  const int64_t i0 = ((int64_t)(z + a.HZ) * a.DY + (yq * R + a.HY)) * a.DX + (xc * 32 + lane + a.HX);   // row 0's cell
  if (STAGED) {
    if (!__syncthreads_or(active)) return;   // tables and barriers visible; nothing to do for the whole CTA?
  } else {
    __syncthreads();                         // tables visible (the only CTA barrier)
    if (!active) return;
  }
  // STAGED: plane p = the box [xc 32 + HX - UH, +USX) x [y0 + HY - UH, +sy) of level z + HZ + pdz[p]
  auto issue = [&](int pl) {
    const int b = pl % NB;
    unsigned char *dst = smraw + a.o_buf + b * a.plane_bytes;
    const int cx = xc * 32 + a.HX - UH, cyy = blockIdx.y * a.cy * R + a.HY - UH, czz = z + a.HZ + a.pdz[pl];
    mbar_expect_tx(&full[b], a.tx_bytes);
    tma_load_3d(dst, &a.tm_xy, 2 * cx, cyy, czz, &full[b]);
    if (DIM == 3) tma_load_3d(dst + a.o_z, &a.tm_z, cx, cyy, czz, &full[b]);
    if (FORCE) tma_load_3d(dst + a.o_g, &a.tm_g, 2 * cx, cyy, czz, &full[b]);
  };
  if (STAGED && tid == 0) {
#pragma unroll
    for (int b = 0; b < NB; ++b)
      if (b < a.np) issue(b);
  }
  UState<DIM, FORCE, R> p;
  const double2 *pxy = a.uxy + i0;
  const double *pz = DIM == 3 ? a.uz + i0 : nullptr;
  const double2 *pg = a.aux + i0;
  if (active) {
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
  }
  using SRC = typename std::conditional<STAGED, SrcShared<DIM, FORCE>, SrcGlobal<DIM, FORCE>>::type;
  SRC src;
  if constexpr (!STAGED) { src.pxy = pxy; src.pz = pz; src.pg = pg; src.DX = a.DX; }
  const int s0 = (wy * R + UH) * USX + lane + UH;   // STAGED: row 0's own cell inside a staged plane
  int plane = -1, curw = -1;
  uint32_t mw[R], mwn[R], comb = 0;   // mask words of the row group: the word in use, the next one (in flight)
  bool wfull = false, dirty = false;
  if (active) {
#pragma unroll
    for (int r = 0; r < R; ++r) mwn[r] = a.mask[i0 + r * a.DX];
  }
  for (int sg = 0; sg < a.nseg; ++sg) {
    const USeg seg = a.seg[sg];
    if (STAGED && seg.plane != plane) {
      if (plane >= 0) {   // leave the buffer of the previous plane; the last warp out refills it
        __syncwarp();
        if (lane == 0) {
          __threadfence_block();
          const int b = plane % NB;
          if (atomicSub(&left[b], 1) == 1) {
            left[b] = nwarp;
            __threadfence_block();
            if (plane + NB < a.np) issue(plane + NB);
          }
        }
      }
      plane = seg.plane;
      const int b = plane % NB;
      mbar_wait(&full[b], (plane / NB) & 1);
      if constexpr (STAGED) {
        const unsigned char *buf = smraw + a.o_buf + b * a.plane_bytes;
        src.sxy = (const double2 *)buf + s0;
        src.sz = (const double *)(buf + a.o_z) + s0;
        src.sg = (const double2 *)(buf + a.o_g) + s0;
      }
    }
    if (!active) continue;
    const int w = seg.word;
    if (w != curw) {   // the mask words are walked in order: word w arrived while word w - 1 was in use
      if (!FORCE && FRAC && dirty) {   // broken bits back to HBM
#pragma unroll
        for (int r = 0; r < R; ++r) a.mask[(int64_t)curw * a.npad + i0 + r * a.DX] = mw[r];
      }
      dirty = false;
      curw = w;
#pragma unroll
      for (int r = 0; r < R; ++r) mw[r] = mwn[r];
      if (w + 1 < a.nw) {
#pragma unroll
        for (int r = 0; r < R; ++r) mwn[r] = a.mask[(int64_t)(w + 1) * a.npad + i0 + r * a.DX];
      }
      comb = mw[0];
#pragma unroll
      for (int r = 1; r < R; ++r) comb &= mw[r];
      wfull = __all_sync(FULL, comb == a.fullw[w]);   // every bond of this word is intact on the whole row group
    }
    for (int c = seg.cbeg; c < seg.cend; ++c) {
      const UCol col = scol[c];
      const int n = col.n;
      const double2 *cst = stab + col.tab;
      uint32_t bits[R], nfb[R], clr[R];
#pragma unroll
      for (int r = 0; r < R; ++r) nfb[r] = clr[r] = bits[r] = 0;
      src.column(col.off, col.soff);
      bool slow = false;
      if (!wfull) {
        const uint32_t nmask = (1u << n) - 1u;
        slow = !__all_sync(FULL, ((comb >> col.bit0) & nmask) == nmask);
      }
      if (!slow) {
        if (!FORCE && FRAC) {
          p.bad = 0;
#pragma unroll
          for (int r = 0; r < R; ++r) p.snap[r] = p.acc[r];
        }
        u_run_col<false, DIM, FORCE, FRAC, R>(p, src, n, col.xi0, col.xi2, cst, bits, nfb, clr);
        if (!FORCE && FRAC) {
          if (__any_sync(FULL, p.bad)) {   // redo the column with the exact test
            slow = true;
#pragma unroll
            for (int r = 0; r < R; ++r) p.acc[r] = p.snap[r];
          }
        }
      }
      if (slow) {
        const uint32_t nmask = (1u << n) - 1u;
#pragma unroll
        for (int r = 0; r < R; ++r) bits[r] = (mw[r] >> col.bit0) & nmask;
        if (!FORCE && FRAC && a.nofail) {
#pragma unroll
          for (int r = 0; r < R; ++r) nfb[r] = (a.nofail[(int64_t)w * a.npad + i0 + r * a.DX] >> col.bit0) & nmask;
        }
        u_run_col<true, DIM, FORCE, FRAC, R>(p, src, n, col.xi0, col.xi2, cst, bits, nfb, clr);
        if (!FORCE && FRAC) {
          bool any = false;
#pragma unroll
          for (int r = 0; r < R; ++r)
            if (clr[r]) { mw[r] &= ~(clr[r] << col.bit0); any = true; }
          if (any) {
            dirty = true;
            comb = mw[0];
#pragma unroll
            for (int r = 1; r < R; ++r) comb &= mw[r];
          }
          if (__any_sync(FULL, any)) wfull = false;   // (warp-uniform: it guards warp votes)
        }
      }
    }
  }
  if (!active) return;
  if (!FORCE && FRAC && dirty) {   // broken bits back to HBM
#pragma unroll
    for (int r = 0; r < R; ++r) a.mask[(int64_t)curw * a.npad + i0 + r * a.DX] = mw[r];
  }
  if (!active) return;
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
  int rows = 4, regs = 168, nb = 2;
  bool staged = false;
  CUtensorMap tm_xy[2], tm_z[2], tm_g;   // per displacement buffer
};

// device tables: per stencil bit {xi_1, thr = s_c ||xi||^2} (dilatation) or {xi_1, 1 / ||xi||^2} (force), ||xi||^2 in the
// kernels' own operation order; per column the UCol record (xi_0, xi_2 are constant along a column)
bool ulat_tables(pd_sim *s, bool force, UArgs &a) {
  PdLattice &l = s->lat;
  const int dim = s->dim;
  if (!l.ctab[force]) {
    std::vector<double2> h((size_t)l.nbits + 8, make_double2(0.0, 0.0));
    for (int c = 0; c < l.ncol; ++c)
      for (int t = 0; t < l.cols[c].n; ++t) {
        const int b = l.cols[c].word * 32 + l.cols[c].bit0 + t;
        const int o[3] = {l.cols[c].dx, l.cols[c].dy0 + t, l.cols[c].dz};
        double xi[3] = {0, 0, 0};
        for (int k = 0; k < dim; ++k) xi[k] = (double)o[k] * l.h[k];
        double r2 = xi[0] * xi[0];
        for (int k = 1; k < dim; ++k) r2 = std::fma(xi[k], xi[k], r2);
        h[b] = make_double2(xi[1], force ? 1.0 / r2 : s->s_c * r2);
      }
    l.ctab[force] = (double *)pdi::dev_alloc(s, sizeof(double2) * h.size());
    if (!l.ctab[force]) return false;
    if (cudaMemcpyAsync(l.ctab[force], h.data(), sizeof(double2) * h.size(), cudaMemcpyHostToDevice, s->stream) != cudaSuccess ||
        cudaStreamSynchronize(s->stream) != cudaSuccess) return false;
  }
  if (!l.ucols) {
    std::vector<UCol> h(std::max(l.ncol, 1));
    memset(h.data(), 0, sizeof(UCol) * h.size());
    for (int c = 0; c < l.ncol; ++c) {
      const PdLatCol &src = l.cols[c];
      UCol &u = h[c];
      u.off = (src.dz * l.DY + src.dy0) * l.DX + src.dx;
      u.soff = src.dy0 * USX + src.dx;
      u.n = src.n; u.word = src.word; u.bit0 = src.bit0; u.pad = 0;
      u.tab = src.word * 32 + src.bit0;
      u.xi0 = (double)src.dx * l.h[0];
      u.xi2 = dim == 3 ? (double)src.dz * l.h[2] : 0.0;
    }
    l.ucols = pdi::dev_alloc(s, sizeof(UCol) * h.size());
    if (!l.ucols) return false;
    if (cudaMemcpyAsync(l.ucols, h.data(), sizeof(UCol) * h.size(), cudaMemcpyHostToDevice, s->stream) != cudaSuccess ||
        cudaStreamSynchronize(s->stream) != cudaSuccess) return false;
  }
  a.ctab = (const double2 *)l.ctab[force];
  a.cols = (const UCol *)l.ucols;
  return true;
}

UPrepared *ulat_prepare(pd_sim *s, bool force, bool allow_staged = true) {
  PdLattice &l = s->lat;
  void *&slot = l.cache[force ? 1 : 0];
  if (slot) return (UPrepared *)slot;
  UPrepared *pp = new UPrepared();
  UArgs &a = pp->a;
  memset(&a, 0, sizeof a);
  a.DX = l.DX; a.DY = l.DY; a.HX = l.HX; a.HY = l.HY; a.HZ = l.HZ; a.PZ = l.PZ;
  {   // rows per lane: 2 (measured: 16-20 resident warps per SM beat the longer record reuse of 4); -1 = 4
    const int dflt = 2, r = env_int(force ? "PD_ULAT_FRC_ROWS" : "PD_ULAT_DIL_ROWS", 0);
    pp->rows = r == -1 ? 6 - dflt : ((r == 2 || r == 4) ? r : dflt);
  }
  pp->regs = env_int(force ? "PD_ULAT_FRC_REGS" : "PD_ULAT_DIL_REGS", force ? 168 : 102);
  pp->nb = env_int("PD_ULAT_NB", 2) == 3 ? 3 : 2;
  // STAGED (TMA planes in shared memory) whenever the stencil radius in x and y is within the staged halo
  pp->staged = allow_staged && env_int("PD_ULAT_STAGED", 1) != 0 && l.HX <= UH && l.HY <= UH && (l.DX % 2 == 0);
  a.nxc = l.PX / 32; a.nyq = (l.PY + 8) / 4; a.nyq_used = l.PY / pp->rows;
  a.ncol = l.ncol; a.nbits = l.nbits; a.nw = l.nw;
  if (pp->staged) {   // one level per CTA, cy row groups adjacent in y
    a.cy = std::max(1, std::min(env_int(force ? "PD_ULAT_FRC_CY" : "PD_ULAT_DIL_CY", 4), 8));
    a.cz = 1;
  } else {
    a.cy = std::max(1, std::min(env_int(force ? "PD_ULAT_FRC_CY" : "PD_ULAT_DIL_CY", 2), 8));
    a.cz = s->dim == 3 ? std::max(1, std::min(env_int(force ? "PD_ULAT_FRC_CZ" : "PD_ULAT_DIL_CZ", 2), 8)) : 1;
    while (a.cy * a.cz > 8) { if (a.cz > 1) --a.cz; else --a.cy; }   // <= 256 threads per CTA
  }
  a.sy = pp->rows * a.cy + 2 * UH;
  for (int w = 0; w < 4; ++w) a.fullw[w] = l.fullw[w];
  // planes (distinct dz; the column table is dz-major) and segments (runs of columns inside one plane and one mask word)
  a.np = 0; a.nseg = 0;
  for (int c = 0; c < l.ncol; ++c) {
    const bool newp = a.np == 0 || l.cols[c].dz != a.pdz[a.np - 1];
    if (newp) {
      if (a.np == 8) { delete pp; return nullptr; }
      a.pdz[a.np++] = l.cols[c].dz;
    }
    if (newp || l.cols[c].word != a.seg[a.nseg - 1].word) {
      if (a.nseg == UMAXSEG) { delete pp; return nullptr; }
      USeg &g = a.seg[a.nseg++];
      g.plane = (int16_t)(a.np - 1); g.word = l.cols[c].word; g.cbeg = (int16_t)c; g.cend = (int16_t)c;
    }
    a.seg[a.nseg - 1].cend = (int16_t)(c + 1);
  }
  a.npad = s->npad;
  a.aux = l.aux;
  a.mask = l.mask; a.nofail = l.nofail; a.rgocc = l.rgocc; a.flags32 = l.flags32; a.minv = s->minv;
  for (int q = 0; q < 3; ++q) { a.v[q] = s->v[q]; a.bval[q] = s->bval[q]; }
  a.theta_out = nullptr;
  a.A = s->A; a.c1 = s->c1; a.G = s->G; a.vol_uniform = s->vol_uniform; a.rrho = 1.0 / s->rho; a.dt = s->dt;
  a.gramp = 1.0;
  if (!ulat_tables(s, force, a)) { delete pp; return nullptr; }
  const int nwarp = a.cy * a.cz;
  const USmem lay = ulat_smem(s->dim, force, pp->staged, l.nbits, l.ncol, a.sy, pp->nb);
  a.o_col = lay.col; a.o_buf = lay.buf; a.o_z = lay.z; a.o_g = lay.g; a.plane_bytes = lay.plane;
  a.tx_bytes = (uint32_t)a.sy * USX * (16 + (s->dim == 3 ? 8 : 0) + (force ? 16 : 0));
  pp->smem = lay.total;
  if (pp->staged) {
    bool ok = true;
    for (int q = 0; q < 2 && ok; ++q) {
      ok = make_plane_map(&pp->tm_xy[q], l.uxy[q], 2, l.DX, l.DY, l.DZ, USX, a.sy);
      if (ok && s->dim == 3) ok = make_plane_map(&pp->tm_z[q], l.uz[q], 1, l.DX, l.DY, l.DZ, USX, a.sy);
    }
    if (ok) ok = make_plane_map(&pp->tm_g, l.aux, 2, l.DX, l.DY, l.DZ, USX, a.sy);
    if (!ok || pp->smem > 232448 - 1024) {   // no tensor maps on this driver / planes do not fit: the direct variant
      delete pp;
      return ulat_prepare(s, force, false);
    }
  }
  pp->block = dim3((unsigned)(nwarp * 32));
  pp->grid = dim3((unsigned)a.nxc, (unsigned)((a.nyq_used + a.cy - 1) / a.cy), (unsigned)((l.PZ + a.cz - 1) / a.cz));
  slot = pp;
  return pp;
}

template <int DIM, bool FORCE, bool FRAC, int R, bool STAGED, int NB, int MAXT>
void ulat_dispatch3(const UPrepared *pp, cudaStream_t st) {
  auto kern = k_ulat<DIM, FORCE, FRAC, R, STAGED, NB, MAXT>;
  static bool attr_done = false;   // per instantiation: opt in to > 48 KB of dynamic shared memory
  if (!attr_done) {
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 232448 - 1024);
    attr_done = true;
  }
  kern<<<pp->grid, pp->block, pp->smem, st>>>(pp->a);
}
template <int DIM, bool FORCE, bool FRAC, int R, bool STAGED, int NB>
void ulat_dispatch2(const UPrepared *pp, cudaStream_t st) {
  if (pp->regs >= 255) ulat_dispatch3<DIM, FORCE, FRAC, R, STAGED, NB, 256>(pp, st);
  else if (pp->regs >= 168) ulat_dispatch3<DIM, FORCE, FRAC, R, STAGED, NB, 384>(pp, st);
  else if (pp->regs >= 128) ulat_dispatch3<DIM, FORCE, FRAC, R, STAGED, NB, 512>(pp, st);
  else ulat_dispatch3<DIM, FORCE, FRAC, R, STAGED, NB, 640>(pp, st);
}
template <int DIM, bool FORCE, bool FRAC, int R>
void ulat_dispatch1(const UPrepared *pp, cudaStream_t st) {
  if (!pp->staged) ulat_dispatch2<DIM, FORCE, FRAC, R, false, 2>(pp, st);
  else if (pp->nb == 3) ulat_dispatch2<DIM, FORCE, FRAC, R, true, 3>(pp, st);
  else ulat_dispatch2<DIM, FORCE, FRAC, R, true, 2>(pp, st);
}
template <int DIM, bool FORCE, bool FRAC>
void ulat_dispatch(const UPrepared *pp, cudaStream_t st) {
  if (pp->rows == 2) ulat_dispatch1<DIM, FORCE, FRAC, 2>(pp, st); else ulat_dispatch1<DIM, FORCE, FRAC, 4>(pp, st);
}

}  // namespace

namespace pdi {

void ulat_free_cache(pd_sim *s) {
  ball_free_cache(s);
  disc_free_cache(s);
  for (int q = 0; q < 2; ++q) {
    delete (UPrepared *)s->lat.cache[q];
    s->lat.cache[q] = nullptr;
  }
}

int ulat_launch_dilatation(pd_sim *s, double *theta_out, bool do_break) {
  if (int rc = ball_launch_dilatation(s, theta_out, do_break)) return rc > 0 ? PD_OK : rc;   // the compiled-in 122-offset stencil (3-D)
  if (int rc = disc_launch_dilatation(s, theta_out, do_break)) return rc > 0 ? PD_OK : rc;   // the compiled-in 28-offset stencil (2-D)
  UPrepared *pp = ulat_prepare(s, false);
  if (!pp) { set_error("device allocation failed"); return PD_ERR_ALLOC; }
  const PdLattice &l = s->lat;
  UArgs &a = pp->a;
  a.uxy = l.uxy[s->cur]; a.uz = l.uz[s->cur]; a.uxy_w = nullptr; a.uz_w = nullptr;
  if (pp->staged) { a.tm_xy = pp->tm_xy[s->cur]; a.tm_z = pp->tm_z[s->cur]; a.tm_g = pp->tm_g; }
  a.theta_out = theta_out;
  const bool frac = do_break && s->fracture;
  if (s->dim == 2) { if (frac) ulat_dispatch<2, false, true>(pp, s->stream); else ulat_dispatch<2, false, false>(pp, s->stream); }
  else { if (frac) ulat_dispatch<3, false, true>(pp, s->stream); else ulat_dispatch<3, false, false>(pp, s->stream); }
  return PD_OK;
}

int ulat_launch_force_update(pd_sim *s) {
  if (int rc = ball_launch_force_update(s)) return rc > 0 ? PD_OK : rc;
  if (int rc = disc_launch_force_update(s)) return rc > 0 ? PD_OK : rc;
  UPrepared *pp = ulat_prepare(s, true);
  if (!pp) { set_error("device allocation failed"); return PD_ERR_ALLOC; }
  const PdLattice &l = s->lat;
  UArgs &a = pp->a;
  a.uxy = l.uxy[s->cur]; a.uz = l.uz[s->cur]; a.uxy_w = l.uxy[s->cur ^ 1]; a.uz_w = l.uz[s->cur ^ 1];
  if (pp->staged) { a.tm_xy = pp->tm_xy[s->cur]; a.tm_z = pp->tm_z[s->cur]; a.tm_g = pp->tm_g; }
  a.gramp = 1.0;
  if (s->ramp_time > 0.0) a.gramp = std::min(1.0, ((double)s->step * s->dt) / s->ramp_time);
  if (s->dim == 2) ulat_dispatch<2, true, false>(pp, s->stream); else ulat_dispatch<3, true, false>(pp, s->stream);
  return PD_OK;
}

}  // namespace pdi
