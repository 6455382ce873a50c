// pd_lattice_disc.cu -- step kernels of the UNIFORM lattice layout for the 2-D stencil of the paper's examples: an
// isotropic 2-D lattice with horizon delta = 3.015 dx, whose family is the DISC of the 28 integer
// offsets 0 < |o|^2 <= 9.  The 2-D counterpart of pd_lattice_ball.cu, and much simpler: the whole walk of a lane, 28
// offsets x RY rows, is some hundred straight-line instructions, and the RY + 6 rows a warp reaches fit one TMA box.
//
//   dilatation (+ break):  eta = u_j - u_i,  dot = xi . eta  [= xbar e];  theta_i = (A / m_i) V sum_j rho_ij dot
//        (Eq. 1.6 / 2.3); s >= s_c <=> dot >= thr = s_c ||xi||^2 (Eqs. 1.17, 1.30,
//        PAPER.md:297-300, 417-425).  The walk FILTERS (per class |o|^2 a running integer max of the high words of dot
//        against the high word of the smallest thr of the class); a warp whose filter fires tests its bonds one by one
//        against thr on the bit patterns, from the box still in shared memory, clears the bits and takes the broken
//        bonds out of the sum.  Both ends of a bond compute the same dot bit for bit, so they decide alike (C-6).
//   force:  d = dot / ||xi||^2,  t = (cth_i + cth_j) + (G/m_i + G/m_j) d,  f_i += t xi   (Eq. 2.2 / 2.1),
//        then Eq. 2.11 and the boundary dofs of App. B in the epilogue.
//
// Kernel shape: one warp per CTA = 32 lanes along x, RY rows per lane; the box [x0 - 3, x0 + 35) x [y0 - 3, y0 + RY + 3)
// of {u_0, u_1} (and {G/m, cth} in the force pass) comes by one TMA load; every record address and every mask bit is a
// compile-time constant.  A warp whose nodes all have their full family intact and breakable runs the FAST body, any
// other the MASKED body.  The 2-D configs are latency bound (a few thousand warps in all): what counts is the length of
// the one dependent chain TMA -> walk -> epilogue, not throughput.
//
// Taken only when the lattice's stencil and mask-bit layout are exactly the disc's (checked in disc_prepare); every
// other uniform lattice takes the table-driven kernels of pd_lattice_uniform.cu.
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
constexpr int S = 3;                // stencil radius
constexpr int M2 = 9;               // |o|^2 <= M2
constexpr int DSX = 32 + 2 * S;     // cells per staged row
constexpr int NBITS = 28;

__host__ __device__ constexpr bool indisc(int dx, int dy) {
  const int r = dx * dx + dy * dy;
  return r > 0 && r <= M2 && dx >= -S && dx <= S && dy >= -S && dy <= S;
}
// mask bit of an offset: the builder's layout (pd_lattice.cu: columns by dx, runs along y of <= 7 bits)
__host__ __device__ constexpr int disc_bit(int qx, int qy) {
  int bit = 0;
  for (int dx = -S; dx <= S; ++dx) {
    int dy = -S;
    while (dy <= S) {
      if (!indisc(dx, dy)) { ++dy; continue; }
      int n = 0;
      while (n < PD_MAXSTEP && indisc(dx, dy + n)) ++n;
      if ((bit & 31) + n > 32) bit = (bit + 31) & ~31;
      if (dx == qx && qy >= dy && qy < dy + n) return bit + (qy - dy);
      bit += n;
      dy += n;
    }
  }
  return -1;
}
static_assert(disc_bit(3, 0) == NBITS - 1 && disc_bit(-3, 0) == 0, "disc stencil bit layout");
constexpr uint32_t DISC_FULL = (1u << NBITS) - 1u;

template <int B, int E, class F>
__device__ __forceinline__ void sfor(F &&f) {
  if constexpr (B < E) {
    f(std::integral_constant<int, B>{});
    sfor<B + 1, E>(f);
  }
}
#define CV(x) (std::remove_reference_t<decltype(x)>::value)

struct DArgs {
  int DX, DY, PY, HX, HY, nxc;
  const uint8_t *rgocc;              // [(PY + 8) / 4][nxc]: the 32 x 4 row group holds a node
  int64_t npad;
  const double2 *uxy;                // u^n
  double2 *uxy_w;                    // force: u^{n+1}
  double2 *aux;                      // {G/m_i, cth_i}
  uint32_t *mask;                    // [npad] one word per node
  const uint32_t *nofail;            // [npad] or null
  const uint32_t *flags32;
  const double *minv;
  double *v[2];
  const double *bval[2];
  double *theta_out;
  double A, c1, G, vol_uniform, rrho, dt, gramp;
  double xi[2][4];                   // xi[k][a] = a h_k
  double rinv[4][4];                 // 1 / ||xi||^2 of offset (+-a, +-b)
  double thr[4][4];                  // s_c ||xi||^2
  int thr_hi[M2 + 1];                // per class: min over the class of hi(thr)
  int8_t odx[32], ody[32];           // offset of mask bit q (exact test)
  alignas(64) CUtensorMap tm_xy, tm_g;
};

template <bool FORCE, int RY>
struct DState {
  double uo[RY][2];
  double acc[RY];
  double f[RY][2], gmu[RY], cth[RY];
  int mx[M2 + 1];
  uint32_t mw[RY], bw[RY];           // intact; intact and allowed to break
};

template <bool FORCE, bool FRAC, bool MASKED, int DXo, int DYo, int R, class ST>
__device__ __forceinline__ void disc_bond(const DArgs &a, ST &p, const double2 &xy, const double2 &g) {
  constexpr int b = disc_bit(DXo, DYo), ax = DXo < 0 ? -DXo : DXo, ay = DYo < 0 ? -DYo : DYo;
  const double x0 = DXo > 0 ? a.xi[0][ax] : -a.xi[0][ax];
  const double x1 = DYo > 0 ? a.xi[1][ay] : -a.xi[1][ay];
  double dot = 0.0;
  if constexpr (DXo != 0) dot = __dmul_rn(x0, xy.x - p.uo[R][0]);
  if constexpr (DYo != 0) {
    const double e1 = xy.y - p.uo[R][1];
    if constexpr (DXo != 0) dot = fma(x1, e1, dot); else dot = __dmul_rn(x1, e1);
  }
  if constexpr (!FORCE) {
    if (!MASKED || ((p.mw[R] >> b) & 1u)) p.acc[R] += dot;   // rho_ij = 0 leaves the sum as it is
    if constexpr (FRAC) {
      const int h = __double2hiint(dot);
      if (!MASKED || ((p.bw[R] >> b) & 1u)) p.mx[ax * ax + ay * ay] = max(p.mx[ax * ax + ay * ay], h);
    }
  } else {
    const double gs = p.gmu[R] + g.x, cs = p.cth[R] + g.y;
    const double d = __dmul_rn(dot, a.rinv[ax][ay]);   // e / xbar
    double t = fma(gs, d, cs);
    if constexpr (MASKED) t = ((p.mw[R] >> b) & 1u) ? t : 0.0;   // rho_ij = 0
    if constexpr (DXo != 0) p.f[R][0] = fma(t, x0, p.f[R][0]);
    if constexpr (DYo != 0) p.f[R][1] = fma(t, x1, p.f[R][1]);
  }
}

template <int RY>
__host__ __device__ constexpr bool disc_used(int dx, int yy) {
  for (int r = 0; r < RY; ++r)
    if (indisc(dx, yy - r)) return true;
  return false;
}

// the whole family walk of the lane: every record of the box is read once
template <bool FORCE, bool FRAC, bool MASKED, int RY, class ST>
__device__ __forceinline__ void disc_walk(const DArgs &a, ST &p, const double2 *sxy, const double2 *sg) {
  sfor<0, RY + 2 * S>([&](auto Yc) {
    sfor<0, 2 * S + 1>([&](auto Xc) {
      constexpr int dx = CV(Xc) - S, yy = CV(Yc) - S;
      if constexpr (disc_used<RY>(dx, yy)) {
        const double2 xy = sxy[yy * DSX + dx];
        double2 g = make_double2(0.0, 0.0);
        if constexpr (FORCE) g = sg[yy * DSX + dx];
        sfor<0, RY>([&](auto Rc) {
          constexpr int dx = CV(Xc) - S, dy = CV(Yc) - S - CV(Rc);
          if constexpr (indisc(dx, dy)) disc_bond<FORCE, FRAC, MASKED, dx, dy, CV(Rc)>(a, p, xy, g);
        });
      }
    });
  });
}

__host__ __device__ constexpr uint32_t up128(uint32_t x) { return (x + 127u) & ~127u; }

template <bool FORCE, bool FRAC, int RY>
__global__ void __launch_bounds__(32) k_disc(const __grid_constant__ DArgs a) {
  constexpr int sy = RY + 2 * S;
  constexpr uint32_t o_g = up128((uint32_t)sy * DSX * 16);
  __shared__ __align__(128) unsigned char sm[128 + o_g + (FORCE ? o_g : 0u)];
  uint64_t *full = (uint64_t *)sm;
  unsigned char *box = sm + 128;
  const int lane = threadIdx.x, xc = blockIdx.x, y0 = blockIdx.y * RY;
  if (lane == 0) {
    mbar_init(full, 1);
    mbar_fence_init();
    mbar_expect_tx(full, (uint32_t)sy * DSX * 16u * (FORCE ? 2u : 1u));
    tma_load_3d(box, &a.tm_xy, 2 * (xc * 32 + a.HX - S), y0 + a.HY - S, 0, full);
    if (FORCE) tma_load_3d(box + o_g, &a.tm_g, 2 * (xc * 32 + a.HX - S), y0 + a.HY - S, 0, full);
  }
  const int64_t i0 = (int64_t)(y0 + a.HY) * a.DX + (xc * 32 + lane + a.HX);
  auto cell = [&](int r) { return i0 + (int64_t)r * a.DX; };
  auto dead = [&](int r) { return y0 + r >= a.PY; };
  DState<FORCE, RY> p;
  constexpr bool BRK = !FORCE && FRAC;
  uint32_t notfull = 0;
  {
    double2 xy[RY], g[RY];
#pragma unroll
    for (int r = 0; r < RY; ++r) {
      const int64_t i = dead(r) ? i0 : cell(r);
      xy[r] = a.uxy[i];
      if constexpr (FORCE) g[r] = a.aux[i];
      p.mw[r] = dead(r) ? 0u : a.mask[i];
      const uint32_t nf = (BRK && a.nofail && !dead(r)) ? a.nofail[i] : 0u;
      p.bw[r] = p.mw[r] & ~nf;
      notfull |= (p.mw[r] ^ DISC_FULL) | (p.mw[r] & nf);
    }
#pragma unroll
    for (int r = 0; r < RY; ++r) {
      p.uo[r][0] = xy[r].x;
      p.uo[r][1] = xy[r].y;
      if constexpr (FORCE) {
        p.gmu[r] = dead(r) ? 0.0 : g[r].x;
        p.cth[r] = g[r].y;
        p.f[r][0] = p.f[r][1] = 0.0;
      } else {
        p.acc[r] = 0.0;
      }
    }
  }
  const bool fast = __all_sync(FULL, notfull == 0u);
  bool occ = false;   // does the row group hold a node at all?
#pragma unroll
  for (int r = 0; r < RY; r += 4) occ = occ || (!dead(r) && a.rgocc[(int64_t)((y0 + r) >> 2) * a.nxc + xc] != 0);
  if (!occ) {   // phantom cells only (the box in flight must land before the CTA may go)
    mbar_wait(full, 0);
    return;
  }
  if constexpr (BRK) {
#pragma unroll
    for (int c = 0; c <= M2; ++c) p.mx[c] = (int)0x80000000;
  }
  __syncwarp();
  mbar_wait(full, 0);
  const double2 *sxy = (const double2 *)box + S * DSX + lane + S;
  const double2 *sg = (const double2 *)(box + o_g) + S * DSX + lane + S;
  if (fast) disc_walk<FORCE, FRAC, false, RY>(a, p, sxy, sg);
  else disc_walk<FORCE, FRAC, true, RY>(a, p, sxy, sg);
  if constexpr (!FORCE) {
    if constexpr (FRAC) {
      // ---- break test proper (Eq. 1.30): only where the filter fired, bond by bond from the box in shared memory ----
      bool fired = false;
#pragma unroll
      for (int c = 1; c <= M2; ++c) fired = fired || p.mx[c] >= a.thr_hi[c];
      if (__any_sync(FULL, fired)) {
#pragma unroll 1
        for (int q = 0; q < NBITS; ++q) {
          const int dx = a.odx[q], dy = a.ody[q];   // (uniform index)
          const double x0 = (double)dx * a.xi[0][1], x1 = (double)dy * a.xi[1][1];
          const double thr = a.thr[abs(dx)][abs(dy)];
#pragma unroll
          for (int r = 0; r < RY; ++r) {
            if (!((p.bw[r] >> q) & 1u)) continue;
            const double2 xy = sxy[(r + dy) * DSX + dx];
            // the dot of the walk, bit for bit (a vanishing component of xi adds an exact zero)
            double dot = __dmul_rn(x0, xy.x - p.uo[r][0]);
            dot = fma(x1, xy.y - p.uo[r][1], dot);
            if (__double_as_longlong(dot) >= __double_as_longlong(thr)) {   // s >= s_c: identical at both ends of the bond
              p.mw[r] &= ~(1u << q);
              p.bw[r] &= ~(1u << q);
              p.acc[r] -= dot;   // rho_ij <- 0: the bond leaves the sum of Eq. 2.3
            }
          }
        }
#pragma unroll
        for (int r = 0; r < RY; ++r)
          if (!dead(r)) a.mask[cell(r)] = p.mw[r];
      }
    }
    double mi[RY];
#pragma unroll
    for (int r = 0; r < RY; ++r) mi[r] = a.minv[dead(r) ? i0 : cell(r)];
#pragma unroll
    for (int r = 0; r < RY; ++r) {
      if (dead(r)) continue;
      const int64_t i = cell(r);
      const double theta = a.A * mi[r] * (p.acc[r] * a.vol_uniform);   // minv = 0 for phantoms
      a.aux[i] = make_double2(a.G * mi[r], a.c1 * theta * mi[r]);
      if (a.theta_out) a.theta_out[i] = theta;
    }
  } else {
    // ---- Eq. 2.11 + boundary dofs (App. B); the loads of all RY nodes first ----
    unsigned fl[RY];
    double vk[RY][2];
#pragma unroll
    for (int r = 0; r < RY; ++r) {
      const int64_t i = dead(r) ? i0 : cell(r);
      fl[r] = a.flags32[i];
#pragma unroll
      for (int k = 0; k < 2; ++k) vk[r][k] = a.v[k][i];
    }
#pragma unroll
    for (int r = 0; r < RY; ++r) {
      if (p.gmu[r] == 0.0) continue;   // phantom or dead (a node has m_i > 0)
      const int64_t i = cell(r);
      double un[2];
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        const double fk = p.f[r][k] * a.vol_uniform;
        double vv = vk[r][k];
        double uk = p.uo[r][k];
        if (fl[r] & (1u << k)) {                    // clamped: u stays, v = 0
          vv = 0.0;
        } else if (fl[r] & (8u << k)) {             // prescribed velocity
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
    }
  }
}

// ---------------------------------------------------------------- host side ----------------------------------------------------------------

int env_int(const char *name, int dflt) {
  const char *e = getenv(name);
  return e ? atoi(e) : dflt;
}

constexpr int DRY = 2;   // rows per lane (measured: 1 and 4 are slower on configs 2 and 3)

struct DPrepared {
  DArgs a;
  bool ok = false;
  dim3 grid;
  CUtensorMap tm_xy[2], tm_g;   // per displacement buffer
};

// is the lattice's stencil the disc, bit for bit in the builder's layout?
bool disc_layout_matches(const pd_sim *s) {
  const PdLattice &l = s->lat;
  if (s->dim != 2 || !l.uniform || l.nbits != NBITS || l.nw != 1) return false;
  if (l.HX != S || l.HY != S || l.HZ != 0 || l.PZ != 1) return false;
  int cnt = 0;
  for (int c = 0; c < l.ncol; ++c)
    for (int t = 0; t < l.cols[c].n; ++t, ++cnt)
      if (l.cols[c].dz != 0 || disc_bit(l.cols[c].dx, l.cols[c].dy0 + t) != l.cols[c].word * 32 + l.cols[c].bit0 + t) return false;
  return cnt == NBITS && l.fullw[0] == DISC_FULL;
}

DPrepared *disc_prepare(pd_sim *s, bool force) {
  PdLattice &l = s->lat;
  void *&slot = l.cache[force ? 7 : 6];
  if (slot) return (DPrepared *)slot;
  DPrepared *pp = new DPrepared();
  slot = pp;
  if (env_int("PD_DISC", 1) == 0 || !disc_layout_matches(s)) return pp;   // ok = false: the table-driven kernels
  DArgs &a = pp->a;
  memset(&a, 0, sizeof a);
  a.DX = l.DX; a.DY = l.DY; a.PY = l.PY; a.HX = l.HX; a.HY = l.HY; a.nxc = l.PX / 32;
  a.rgocc = l.rgocc;
  a.npad = s->npad;
  a.aux = l.aux;
  a.mask = l.mask; a.nofail = l.nofail; a.flags32 = l.flags32; a.minv = s->minv;
  for (int q = 0; q < 2; ++q) { a.v[q] = s->v[q]; a.bval[q] = s->bval[q]; }
  a.A = s->A; a.c1 = s->c1; a.G = s->G; a.vol_uniform = s->vol_uniform; a.rrho = 1.0 / s->rho; a.dt = s->dt;
  a.gramp = 1.0;
  // constants, in the operation order of the walk (and of pd_lattice_uniform.cu): xi_k = o_k h_k, ||xi||^2 = fma chain
  for (int k = 0; k < 2; ++k)
    for (int q = 0; q < 4; ++q) a.xi[k][q] = (double)q * l.h[k];
  for (int c = 0; c <= M2; ++c) a.thr_hi[c] = 0x7ff00000;
  for (int i = 0; i < 4; ++i)
    for (int j = 0; j < 4; ++j) {
      const double x0 = (double)i * l.h[0], x1 = (double)j * l.h[1];
      const double r2 = std::fma(x1, x1, x0 * x0);
      a.rinv[i][j] = (i | j) ? 1.0 / r2 : 0.0;
      a.thr[i][j] = s->s_c * r2;
      if (!indisc(i, j)) continue;
      long long bits;
      memcpy(&bits, &a.thr[i][j], 8);
      a.thr_hi[i * i + j * j] = std::min(a.thr_hi[i * i + j * j], (int)(bits >> 32));
    }
  for (int dy = -S; dy <= S; ++dy)
    for (int dx = -S; dx <= S; ++dx)
      if (indisc(dx, dy)) { a.odx[disc_bit(dx, dy)] = (int8_t)dx; a.ody[disc_bit(dx, dy)] = (int8_t)dy; }
  const int sy = DRY + 2 * S;
  bool ok = true;
  for (int q = 0; q < 2 && ok; ++q) ok = make_plane_map(&pp->tm_xy[q], l.uxy[q], 2, l.DX, l.DY, l.DZ, DSX, sy);
  if (ok) ok = make_plane_map(&pp->tm_g, l.aux, 2, l.DX, l.DY, l.DZ, DSX, sy);
  if (!ok) return pp;   // no tensor maps on this driver: the table-driven kernels
  pp->grid = dim3((unsigned)a.nxc, (unsigned)((l.PY + DRY - 1) / DRY), 1u);
  pp->ok = true;
  return pp;
}

}  // namespace

namespace pdi {

bool disc_eligible(const pd_sim *s) { return env_int("PD_DISC", 1) != 0 && disc_layout_matches(s); }

void disc_free_cache(pd_sim *s) {
  for (int q = 6; q < 8; ++q) {
    delete (DPrepared *)s->lat.cache[q];
    s->lat.cache[q] = nullptr;
  }
}

// 1: launched; 0: the lattice is not the disc (the caller takes the table-driven kernels)
int disc_launch_dilatation(pd_sim *s, double *theta_out, bool do_break) {
  DPrepared *pp = disc_prepare(s, false);
  if (!pp->ok) return 0;
  const PdLattice &l = s->lat;
  DArgs &a = pp->a;
  a.uxy = l.uxy[s->cur]; a.uxy_w = nullptr;
  a.tm_xy = pp->tm_xy[s->cur]; a.tm_g = pp->tm_g;
  a.theta_out = theta_out;
  if (do_break && s->fracture) k_disc<false, true, DRY><<<pp->grid, 32, 0, s->stream>>>(a);
  else k_disc<false, false, DRY><<<pp->grid, 32, 0, s->stream>>>(a);
  return 1;
}

int disc_launch_force_update(pd_sim *s) {
  DPrepared *pp = disc_prepare(s, true);
  if (!pp->ok) return 0;
  const PdLattice &l = s->lat;
  DArgs &a = pp->a;
  a.uxy = l.uxy[s->cur]; a.uxy_w = l.uxy[s->cur ^ 1];
  a.tm_xy = pp->tm_xy[s->cur]; a.tm_g = pp->tm_g;
  a.gramp = 1.0;
  if (s->ramp_time > 0.0) a.gramp = std::min(1.0, ((double)s->step * s->dt) / s->ramp_time);
  k_disc<true, false, DRY><<<pp->grid, 32, 0, s->stream>>>(a);
  return 1;
}

}  // namespace pdi
