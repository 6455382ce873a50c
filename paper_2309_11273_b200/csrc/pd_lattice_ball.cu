// pd_lattice_ball.cu -- step kernels of the UNIFORM lattice layout for the stencil every example of the paper uses:
// an isotropic 3-D lattice with horizon delta = 3.015 dx, whose family is the BALL of the
// 122 integer offsets 0 < |o|^2 <= 9.  The stencil is known when the kernel is compiled: no column table, no loop
// control per bond, xi = (o_k h_k), 1/||xi||^2 and the break thresholds are per-class constants, and vanishing
// components of xi cost nothing.
//
//   dilatation (+ break filter):  eta = u_j - u_i,  dot = xi . eta  [= xbar e]      3 / 5 / 7 FP64 for 1 / 2 / 3 non-zero o_k
//        theta_i = (A / m_i) V sum_j rho_ij dot  (Eq. 1.6 / 2.3)
//        s >= s_c  <=>  dot >= thr = s_c ||xi||^2 (Eqs. 1.17, 1.30).  The walk only FILTERS:
//        per class |o|^2 a running integer max of the high words of dot against the high word of the smallest thr of
//        the class (hi(dot) < hi(thr) => dot < thr).  A lane whose filter fires leaves a worklist entry; k_ball_exact,
//        launched after the pass, tests the bonds of the fired classes with dot >= thr on the bit patterns, clears the
//        bits and takes the broken bonds out of theta (the walk never waits for the rare event).  Both ends of a bond
//        compute the same dot bit for bit (negating xi and eta is exact), so they decide alike (C-6).
//   force:  d = dot / ||xi||^2,  t = (cth_i + cth_j) + (G/m_i + G/m_j) d,  f_i += t xi          7 / 10 / 13 FP64
//        (Eq. 2.2 / 2.1), then Eq. 2.11 and the boundary dofs of App. B in the epilogue.
//
// Kernel shape: lanes along x, a lane owns RZ nodes adjacent in z (one row), so a gathered record serves up to RZ bonds
// from registers (0.43 shared-memory records per bond at RZ = 4); a CTA is CY warps adjacent in y and consumes the
// RZ + 4 planes z0 - 2 .. z0 + RZ + 1, each brought into shared memory once by TMA (NB buffers in flight, completion on
// an mbarrier, a buffer handed back by the last warp that leaves it: no CTA barrier); the two outermost planes of the
// stencil serve one bond per lane each, and that record is read from global memory instead.
//
// The MIRRORED walk.  Unrolling all 122 RZ bonds of a lane gives 8-17 k instructions, which do not fit the instruction
// cache: that version ran at one instruction per clock and SM (profiles/r02b_ball_kernels.md, stall_no_instruction 7-8
// per issue).  The ball is symmetric under x -> -x, y -> -y and z -> -z; with one row per lane the first two need no
// exchange of node state, the third only the exchange of the lane's levels l <-> RZ - 1 - l, once per tile.  So the
// straight-line code covers one octant -- offsets (+a, +b, dz) against the planes of the first half -- and runs eight
// times with run-time signs (sx, sy, sz): about 1-2 k instructions per kernel.  Offsets with a = 0 (b = 0) are their
// own mirror image and are walked in the sx = +1 (sy = +1) pass only.
//
// A warp whose nodes all have their full family intact and breakable runs the FAST body; any other the MASKED body,
// where a missing or broken bond is zeroed by a select on the integer pipe (no extra FP64 work).  The MASKED body needs
// the bond bit of offset (sx a, sy b, sz c) at a compile-time position: the OCTANT words mask8[oct][cell], oct = the
// three sign bits, bit = index of (a, b, c) among the 28 magnitudes (an offset with a zero component sits in both
// words of that sign).  They are derived from the 128-bit masks of the lattice layout (which stay the truth for every
// other kernel) when the kernels are prepared and are kept in step by k_ball_exact.
//
// Taken only when the lattice's stencil and mask-bit layout are exactly the ball's (checked in ball_prepare);
// every other uniform lattice takes the table-driven kernels of pd_lattice_uniform.cu.
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
constexpr int BSX = 32 + 2 * S;     // cells per staged row
constexpr int NBITS = 123;          // mask bits of the ball in the builder's layout (one padding bit)

__host__ __device__ constexpr bool inball(int dx, int dy, int dz) {
  const int r = dx * dx + dy * dy + dz * dz;
  return r > 0 && r <= M2 && dx >= -S && dx <= S && dy >= -S && dy <= S && dz >= -S && dz <= S;
}
// mask bit of an offset: the builder's layout (pd_lattice.cu: columns dz-major, then dx, runs along y of <= 7 bits,
// a run never straddles a 32-bit word), evaluated at compile time
__host__ __device__ constexpr int ball_bit(int qx, int qy, int qz) {
  int bit = 0;
  for (int dz = -S; dz <= S; ++dz)
    for (int dx = -S; dx <= S; ++dx) {
      int dy = -S;
      while (dy <= S) {
        if (!inball(dx, dy, dz)) { ++dy; continue; }
        int n = 0;
        while (n < PD_MAXSTEP && inball(dx, dy + n, dz)) ++n;
        if ((bit & 31) + n > 32) bit = (bit + 31) & ~31;
        if (dz == qz && dx == qx && qy >= dy && qy < dy + n) return bit + (qy - dy);
        bit += n;
        dy += n;
      }
    }
  return -1;
}
static_assert(ball_bit(3, 0, 3) == -1 && ball_bit(0, 0, 3) == NBITS - 1, "ball stencil bit layout");
// all stencil bits of mask word w
__host__ __device__ constexpr uint32_t ball_fullw(int w) {
  int bit = 0;
  uint32_t m = 0;
  for (int dz = -S; dz <= S; ++dz)
    for (int dx = -S; dx <= S; ++dx) {
      int dy = -S;
      while (dy <= S) {
        if (!inball(dx, dy, dz)) { ++dy; continue; }
        int n = 0;
        while (n < PD_MAXSTEP && inball(dx, dy + n, dz)) ++n;
        if ((bit & 31) + n > 32) bit = (bit + 31) & ~31;
        for (int t = 0; t < n; ++t)
          if (((bit + t) >> 5) == w) m |= 1u << ((bit + t) & 31);
        bit += n;
        dy += n;
      }
    }
  return m;
}
// bit of the magnitudes (a, b, c) inside an octant word: their index among the 28 triples of the ball
__host__ __device__ constexpr int canon(int qa, int qb, int qc) {
  int k = 0;
  for (int a = 0; a <= S; ++a)
    for (int b = 0; b <= S; ++b)
      for (int c = 0; c <= S; ++c) {
        if (!inball(a, b, c)) continue;
        if (a == qa && b == qb && c == qc) return k;
        ++k;
      }
  return -1;
}
static_assert(canon(3, 0, 0) == 27, "28 magnitudes per octant");

template <int B, int E, class F>
__device__ __forceinline__ void sfor(F &&f) {
  if constexpr (B < E) {
    f(std::integral_constant<int, B>{});
    sfor<B + 1, E>(f);
  }
}
#define CV(x) (std::remove_reference_t<decltype(x)>::value)


struct BArgs {
  int DX, DY, PY, PZ, HX, HY, HZ;
  int nxc, nyq, nbits;
  int64_t npad;
  const double2 *uxy;                // {u_0, u_1} of u^n
  const double *uz;                  // u_2 of u^n
  double2 *uxy_w;                    // force: u^{n+1}
  double *uz_w;
  double2 *aux;                      // {G/m_i, cth_i}: written by the dilatation pass, gathered by the force pass
  uint32_t *mask;                    // [4][npad] the lattice layout's bond bits
  const uint32_t *nofail;            // [4][npad] or null
  uint32_t *mask8;                   // [8][npad] octant words of mask
  const uint32_t *nf8;               // [8][npad] octant words of nofail, or null
  const uint8_t *rgocc;
  uint8_t *tfull;                    // [PZ / RZ][PY][nxc] 1: every node of the warp tile has its full family intact and breakable
  const uint32_t *flags32;
  const double *minv;
  const int2 *q8;                    // [128] exact pass: {bit inside the octant words, set of octant words} of mask bit q
  void *wl;                          // worklist of k_ball_exact: BEntry per warp tile whose filter fired
  int *wl_count;
  double *v[3];
  const double *bval[3];
  double *theta_out;
  double A, c1, G, vol_uniform, rrho, dt, gramp;   // gramp = g(t_n) = min(1, n dt / ramp_time)
  double xi[3][4];                   // xi[k][a] = a h_k
  double rinv[4][4][4];              // 1 / ||xi||^2 of offset (+-a, +-b, +-c), in the operation order of the walk
  double thr[4][4][4];               // s_c ||xi||^2 of offset (+-a, +-b, +-c)
  uint32_t pk[128];                  // mask bit q -> its offset, packed (dx + 3) | (dy + 3) << 4 | (dz + 3) << 8
  int thr_hi[M2 + 1];                // per class |o|^2: min over the class of hi(s_c ||xi||^2)
  uint32_t cmask[M2 + 1][4];         // per class: its bonds in the four mask words
  alignas(64) CUtensorMap tm_xy, tm_z, tm_g;   // 3-D tiled maps of uxy (as doubles), uz, aux (as doubles)
};

// worklist entry of a lane whose break filter fired
template <int RZ>
struct BEntry {
  int64_t i0;             // cell of the lane's node at level z0
  int z0, tile;           // first level; index of the warp tile in tfull
  uint32_t cm, pad;       // the classes |o|^2 that reached the threshold
  double acc[RZ];         // per node: sum_j rho_ij dot before the break test
};

// own-node state of the RZ nodes of a lane (slot l = level z0 + l, or z0 + RZ - 1 - l while sz = -1)
template <int RZ>
struct BState {
  double uo[RZ][3];
  double acc[RZ];                           // dilatation pass
  double f[RZ][3], gmu[RZ], cth[RZ];        // force pass
  int mx[M2 + 1];                           // dilatation pass: running max of hi(dot) per class
  uint32_t wpos[RZ], wneg[RZ];              // MASKED: octant words of the current pass for dz >= 0 / dz < 0 (intact bits)
  uint32_t bpos[RZ], bneg[RZ];              // MASKED dilatation: intact and allowed to break
};

// run-time signs of a pass.  (The values are made opaque to the optimiser where they are set -- keep(): otherwise the
// sign selects are re-derived at every use instead of being held in 26 registers.)
__device__ __forceinline__ void prefetch_l1(const void *ptr) { asm volatile("prefetch.global.L1 [%0];" ::"l"(ptr)); }
__device__ __forceinline__ void keep(double &v) { asm volatile("" : "+d"(v)); }
__device__ __forceinline__ void keep(int &v) { asm volatile("" : "+r"(v)); }
// x or -x by flipping the sign bit on the integer pipe (neg = 0 or 0x80000000)
__device__ __forceinline__ double signed_const(double x, int neg) {
  return __hiloint2double(__double2hiint(x) ^ neg, __double2loint(x));
}
struct BSign {
  double xs0[4], xs1[4], xs2[4];   // sx a h_0, sy b h_1, sz c h_2
  int ry[4], cx[4];                // byte offsets inside the staged xy plane: sy b BSX 16, sx a 16
};

// node slot L of the lane with the neighbour at offset (sx A, sy B, sz DZ)
template <bool FORCE, bool FRAC, bool MASKED, int A, int B, int DZ, int L, class ST>
__device__ __forceinline__ void ball_bond(const BArgs &a, ST &p, const BSign &sg, const double2 &xy, const double z, const double2 &g) {
  constexpr int az = DZ < 0 ? -DZ : DZ, k = canon(A, B, az);
  const double x0 = sg.xs0[A], x1 = sg.xs1[B], x2 = DZ > 0 ? sg.xs2[az] : -sg.xs2[az];
  double dot = 0.0;
  if constexpr (A != 0) dot = __dmul_rn(x0, xy.x - p.uo[L][0]);
  if constexpr (B != 0) {
    const double e1 = xy.y - p.uo[L][1];
    if constexpr (A != 0) dot = fma(x1, e1, dot); else dot = __dmul_rn(x1, e1);
  }
  if constexpr (DZ != 0) {
    const double e2 = z - p.uo[L][2];
    if constexpr (A != 0 || B != 0) dot = fma(x2, e2, dot); else dot = __dmul_rn(x2, e2);
  }
  const uint32_t mw = MASKED ? (DZ < 0 ? p.wneg[L] : p.wpos[L]) : 0u;
  if constexpr (!FORCE) {
    // (MASKED: the bond's term and its filter entry under a predicate -- rho_ij = 0 leaves the sum as it is)
    if (!MASKED || ((mw >> k) & 1u)) p.acc[L] += dot;
    if constexpr (FRAC) {
      const int h = __double2hiint(dot);
      if (!MASKED || (((DZ < 0 ? p.bneg[L] : p.bpos[L]) >> k) & 1u))
        p.mx[A * A + B * B + az * az] = max(p.mx[A * A + B * B + az * az], h);
    }
  } else {
    const double gs = p.gmu[L] + g.x, cs = p.cth[L] + g.y;
    const double d = __dmul_rn(dot, a.rinv[A][B][az]);   // e / xbar
    double t = fma(gs, d, cs);
    if constexpr (MASKED) t = ((mw >> k) & 1u) ? t : 0.0;      // rho_ij = 0 (a select: three predicated DFMAs measured slower)
    if constexpr (A != 0) p.f[L][0] = fma(t, x0, p.f[L][0]);
    if constexpr (B != 0) p.f[L][1] = fma(t, x1, p.f[L][1]);
    if constexpr (DZ != 0) p.f[L][2] = fma(t, x2, p.f[L][2]);
  }
}

template <int RZ>
__host__ __device__ constexpr bool rec_used(int a, int b, int pz) {
  for (int l = 0; l < RZ; ++l)
    if (inball(a, b, pz - l)) return true;
  return false;
}

// plane J of the first half (pz = J - S relative to slot 0), one (sx, sy) pass: records (sx a, sy b), a, b >= 0
template <bool FORCE, bool FRAC, bool MASKED, int J, int RZ, class ST>
__device__ __forceinline__ void ball_plane(const BArgs &a, ST &p, const BSign &sg, const unsigned char *bxy, const unsigned char *bz,
                                           const uint32_t o_g, const bool xpos, const bool ypos) {
  sfor<0, S + 1>([&](auto Ac) {
    if (CV(Ac) == 0 && !xpos) return;   // a = 0 is its own mirror image
    sfor<0, S + 1>([&](auto Bc) {
      constexpr int A = CV(Ac), B = CV(Bc), pz = J - S;
      if constexpr (rec_used<RZ>(A, B, pz)) {
        if (B == 0 && !ypos) return;    // b = 0 is its own mirror image
        const int o = sg.ry[B] + sg.cx[A];
        const double2 xy = *(const double2 *)(bxy + o);
        const double z = *(const double *)(bz + (o >> 1));
        double2 g = make_double2(0.0, 0.0);
        if constexpr (FORCE) g = *(const double2 *)(bxy + o_g + o);
        sfor<0, RZ>([&](auto Lc) {
          constexpr int A = CV(Ac), B = CV(Bc), dz = J - S - CV(Lc);
          if constexpr (inball(A, B, dz)) ball_bond<FORCE, FRAC, MASKED, A, B, dz, CV(Lc)>(a, p, sg, xy, z, g);
        });
      }
    });
  });
}

constexpr uint32_t up128(uint32_t x) { return (x + 127u) & ~127u; }
// shared memory: [0, 64) mbarriers | [64, 128) counters | NB plane buffers {xy | z | g} | octant words of the CTA's
// nodes [8][RZ][threads] (intact) | the same for intact-and-breakable (dilatation pass with fracture)
template <bool FORCE, bool FRAC, int RZ, int CY, int NB>
struct BSmem {
  static constexpr int sy = CY + 2 * S;
  static constexpr uint32_t o_z = up128((uint32_t)sy * BSX * 16);
  static constexpr uint32_t o_g = o_z + up128((uint32_t)sy * BSX * 8);
  static constexpr uint32_t plane = o_g + (FORCE ? up128((uint32_t)sy * BSX * 16) : 0u);
  static constexpr uint32_t tx = (uint32_t)sy * BSX * (16 + 8 + (FORCE ? 16 : 0));
  static constexpr uint32_t o_buf = 128;
  static constexpr uint32_t words = 8u * RZ * CY * 32u * 4u;
  static constexpr uint32_t o_m8 = o_buf + NB * plane;
  static constexpr uint32_t o_b8 = o_m8 + words;
  static constexpr uint32_t total = o_b8 + (!FORCE && FRAC ? words : 0u);
};

template <int RZ, class ST>
__device__ __forceinline__ void swap_levels(ST &p, bool force) {
#pragma unroll
  for (int l = 0; l < RZ / 2; ++l) {
    auto sw = [](double &x, double &y) { const double t = x; x = y; y = t; };
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      sw(p.uo[l][k], p.uo[RZ - 1 - l][k]);
      if (force) sw(p.f[l][k], p.f[RZ - 1 - l][k]);
    }
    if (force) { sw(p.gmu[l], p.gmu[RZ - 1 - l]); sw(p.cth[l], p.cth[RZ - 1 - l]); }
    else sw(p.acc[l], p.acc[RZ - 1 - l]);
  }
}

template <bool FORCE, bool FRAC, int RZ, int CY, int NB, int MINB>
__global__ void __launch_bounds__(CY * 32, MINB) k_ball(const __grid_constant__ BArgs a) {
  using SM = BSmem<FORCE, FRAC, RZ, CY, NB>;
  // planes z0 - S + 1 .. z0 + RZ + S - 2: the two outermost planes of the stencil would each serve ONE bond of the lane
  // (offset (0, 0, -+S) of its first / last node), which is read from global memory instead
  constexpr int NP = RZ + 2 * S - 2, NT = CY * 32;
  constexpr bool BRK = !FORCE && FRAC;
  static_assert(RZ % 2 == 0, "the mirrored walk needs an even number of levels per lane");
  extern __shared__ __align__(128) unsigned char smraw[];
  const int tid = threadIdx.x, lane = tid & 31, wy = tid >> 5;
  uint64_t *full = (uint64_t *)smraw;           // [NB] plane has landed
  int *left = (int *)(smraw + 64);              // [NB] warps that have not left the buffer yet
  uint32_t *m8s = (uint32_t *)(smraw + SM::o_m8) + tid, *b8s = (uint32_t *)(smraw + SM::o_b8) + tid;
  if (tid == 0) {
#pragma unroll
    for (int b = 0; b < NB; ++b) { mbar_init(&full[b], 1); left[b] = CY; }
    mbar_fence_init();
  }
  // this warp's nodes: x chunk xc, row y0, levels z0 .. z0 + RZ - 1
  const int xc = blockIdx.x, y0 = blockIdx.y * CY + wy, z0 = blockIdx.z * RZ;
  bool active = false;
  if (y0 < a.PY) {
#pragma unroll
    for (int l = 0; l < RZ; ++l)
      if (z0 + l < a.PZ) active |= a.rgocc[((int64_t)(z0 + l) * a.nyq + (y0 >> 2)) * a.nxc + xc] != 0;
  }
  if (!__syncthreads_or(active)) return;   // barriers visible; nothing to do for the whole CTA?
  // the planes are consumed in the order NP/2 - 1 .. 0, NP/2 .. NP - 1 (the planes with most bonds first in each half,
  // so their walk hides the next loads; plane q is level z0 - S + 1 + q); position k of that order holds the box
  // [xc 32 + HX - S, +BSX) x [yt + HY - S, +sy) of level z0 + HZ - S + plane(k)
  auto issue = [&](int k) {
    const int b = k % NB;
    unsigned char *dst = smraw + SM::o_buf + b * SM::plane;
    const int plane = k < NP / 2 ? NP / 2 - 1 - k : k;
    const int cx = xc * 32 + a.HX - S, cyy = blockIdx.y * CY + a.HY - S, czz = z0 + a.HZ - S + 1 + plane;
    mbar_expect_tx(&full[b], SM::tx);
    tma_load_3d(dst, &a.tm_xy, 2 * cx, cyy, czz, &full[b]);
    tma_load_3d(dst + SM::o_z, &a.tm_z, cx, cyy, czz, &full[b]);
    if (FORCE) tma_load_3d(dst + SM::o_g, &a.tm_g, 2 * cx, cyy, czz, &full[b]);
  };
  if (tid == 0) {
#pragma unroll
    for (int b = 0; b < NB; ++b)
      if (b < NP) issue(b);
  }
  // cells of the lane's nodes; a node beyond the padded body (levels >= PZ) is DEAD: never loaded or stored
  const int64_t i0 = ((int64_t)(z0 + a.HZ) * a.DY + (y0 + a.HY)) * a.DX + (xc * 32 + lane + a.HX);
  const int64_t zstr = (int64_t)a.DY * a.DX;
  auto cell = [&](int l) { return i0 + l * zstr; };
  auto dead = [&](int l) { return z0 + l >= a.PZ; };
  BState<RZ> p;
  bool fast = active;
  if (active) {
    // every load of the prologue is issued before the first use (no branch in between): one memory latency, not RZ;
    // what the epilogue reads is pulled towards L1 now
    double2 xy[RZ], g[RZ];
    double uz[RZ];
    fast = a.tfull[((int64_t)blockIdx.z * a.PY + y0) * a.nxc + xc] != 0;
#pragma unroll
    for (int l = 0; l < RZ; ++l) {
      const int64_t i = dead(l) ? i0 : cell(l);
      xy[l] = a.uxy[i];
      uz[l] = a.uz[i];
      if constexpr (FORCE) {
        g[l] = a.aux[i];
        prefetch_l1(a.flags32 + i);
#pragma unroll
        for (int k = 0; k < 3; ++k) prefetch_l1(a.v[k] + i);
      } else {
        prefetch_l1(a.minv + i);
      }
    }
#pragma unroll
    for (int l = 0; l < RZ; ++l) {
      const bool dd = dead(l);
      p.uo[l][0] = xy[l].x;
      p.uo[l][1] = xy[l].y;
      p.uo[l][2] = uz[l];
      if constexpr (FORCE) {
        p.gmu[l] = dd ? 0.0 : g[l].x;
        p.cth[l] = g[l].y;
#pragma unroll
        for (int k = 0; k < 3; ++k) p.f[l][k] = 0.0;
      } else {
        p.acc[l] = 0.0;
      }
    }
    if (!fast) {   // MASKED: the octant words of the lane's nodes, parked in shared memory [oct][node][thread]
#pragma unroll
      for (int l = 0; l < RZ; ++l) {
        const bool dd = dead(l);
        const int64_t i = dd ? i0 : cell(l);
#pragma unroll
        for (int o = 0; o < 8; ++o) {
          const uint32_t mo = dd ? 0u : a.mask8[(int64_t)o * a.npad + i];
          m8s[(o * RZ + l) * NT] = mo;
          if constexpr (BRK) b8s[(o * RZ + l) * NT] = a.nf8 ? mo & ~a.nf8[(int64_t)o * a.npad + i] : mo;
        }
      }
    }
  }
  if constexpr (BRK) {
#pragma unroll
    for (int c = 0; c <= M2; ++c) p.mx[c] = (int)0x80000000;
  }
  int s0 = (wy + S) * BSX + lane + S;   // the lane's node inside a staged plane
  keep(s0);
  // leave the buffer of the plane consumed before position k; the last warp out refills it
  auto leave = [&](int k) {
    const int pb = (k - 1) % NB;
    __syncwarp();
    if (lane == 0) {
      __threadfence_block();
      if (atomicSub(&left[pb], 1) == 1) {
        left[pb] = CY;
        __threadfence_block();
        if (k - 1 + NB < NP) issue(k - 1 + NB);
      }
    }
  };
  BSign sg;
#pragma unroll 1
  for (int mz = 0; mz < 2; ++mz) {
    if (active) {
      if (mz) swap_levels<RZ>(p, FORCE);   // z -> -z: the lane's levels change places
#pragma unroll
      for (int c = 1; c < 4; ++c) { sg.xs2[c] = signed_const(a.xi[2][c], mz << 31); keep(sg.xs2[c]); }
    }
    // the record three levels beyond the lane's first node (its last node while sz = -1): on its way during the planes
    double2 fxy = make_double2(0.0, 0.0), fg = make_double2(0.0, 0.0);
    double fz = 0.0;
    if (active) {
      const int nl = mz ? RZ - 1 : 0;
      const int64_t j = dead(nl) ? i0 : cell(nl) + (mz ? S : -S) * zstr;
      fxy = a.uxy[j];
      fz = a.uz[j];
      if constexpr (FORCE) fg = a.aux[j];
    }
    sfor<0, NP / 2>([&](auto Jc) {
      constexpr int J = NP / 2 - CV(Jc);   // plane of the stencil (pz = J - S relative to slot 0), or its mirror image
      const int k = mz * (NP / 2) + CV(Jc), b = k % NB;
      if (k > 0) leave(k);
      mbar_wait(&full[b], (k / NB) & 1);
      if (active) {
        const unsigned char *buf = smraw + SM::o_buf + b * SM::plane;
        const unsigned char *bxy = buf + s0 * 16, *bz = buf + SM::o_z + s0 * 8;
#pragma unroll 1
        for (int my = 0; my < 2; ++my) {
#pragma unroll
          for (int c = 1; c < 4; ++c) {
            sg.xs1[c] = signed_const(a.xi[1][c], my << 31); sg.ry[c] = (my ? -c : c) * (BSX * 16);
            keep(sg.xs1[c]); keep(sg.ry[c]);
          }
          sg.ry[0] = 0;
#pragma unroll 1
          for (int mx = 0; mx < 2; ++mx) {
#pragma unroll
            for (int c = 1; c < 4; ++c) {
              sg.xs0[c] = signed_const(a.xi[0][c], mx << 31); sg.cx[c] = (mx ? -c : c) * 16;
              keep(sg.xs0[c]); keep(sg.cx[c]);
            }
            sg.cx[0] = 0;
            if (fast) {
              ball_plane<FORCE, FRAC, false, J, RZ>(a, p, sg, bxy, bz, SM::o_g, mx == 0, my == 0);
            } else {
              // octant words of this pass: sign bits (sx, sy) and, per bond, sz xor (dz < 0); slot l holds node nl
              const int op = (mx + 2 * my + 4 * mz) * RZ, on = (mx + 2 * my + 4 * (mz ^ 1)) * RZ;
#pragma unroll
              for (int l = 0; l < RZ; ++l) {
                const int nl = mz ? RZ - 1 - l : l;
                p.wpos[l] = m8s[(op + nl) * NT];
                p.wneg[l] = m8s[(on + nl) * NT];
                if constexpr (BRK) { p.bpos[l] = b8s[(op + nl) * NT]; p.bneg[l] = b8s[(on + nl) * NT]; }
              }
              ball_plane<FORCE, FRAC, true, J, RZ>(a, p, sg, bxy, bz, SM::o_g, mx == 0, my == 0);
            }
          }
        }
      }
    });
    if (active) {   // offset (0, 0, -S) of slot 0
      if (fast) {
        ball_bond<FORCE, FRAC, false, 0, 0, -S, 0>(a, p, sg, fxy, fz, fg);
      } else {
        const int nl = mz ? RZ - 1 : 0, on = 4 * (mz ^ 1) * RZ;
        p.wneg[0] = m8s[(on + nl) * NT];
        if constexpr (BRK) p.bneg[0] = b8s[(on + nl) * NT];
        ball_bond<FORCE, FRAC, true, 0, 0, -S, 0>(a, p, sg, fxy, fz, fg);
      }
    }
  }
  if (!active) return;
  swap_levels<RZ>(p, FORCE);   // the levels back in place
  if constexpr (!FORCE) {
    if constexpr (FRAC) {
      uint32_t cm = 0;   // classes |o|^2 whose running max reached the threshold
#pragma unroll
      for (int c = 1; c <= M2; ++c)
        if (c != 7 && p.mx[c] >= a.thr_hi[c]) cm |= 1u << c;
      // A lane whose filter fired leaves an entry for k_ball_exact (its nodes, the fired classes, its sums): the walk
      // never waits for the rare event, and the warps of its CTA are not held up at the plane buffers.
      const uint32_t fire = __ballot_sync(FULL, cm != 0u);
      if (fire) {
        int base = 0;
        if (lane == 0) base = atomicAdd(a.wl_count, __popc(fire));
        base = __shfl_sync(FULL, base, 0);
        if (cm != 0u) {
          BEntry<RZ> *e = (BEntry<RZ> *)a.wl + base + __popc(fire & ((1u << lane) - 1u));
          e->i0 = i0; e->z0 = z0; e->tile = (int)(((int64_t)blockIdx.z * a.PY + y0) * a.nxc + xc); e->cm = cm;
#pragma unroll
          for (int l = 0; l < RZ; ++l) e->acc[l] = p.acc[l];
        }
      }
    }
    double mi[RZ];
#pragma unroll
    for (int l = 0; l < RZ; ++l) mi[l] = a.minv[dead(l) ? i0 : cell(l)];
#pragma unroll
    for (int l = 0; l < RZ; ++l) {
      if (dead(l)) continue;
      const int64_t i = cell(l);
      const double theta = a.A * mi[l] * (p.acc[l] * a.vol_uniform);   // minv = 0 for phantoms
      a.aux[i] = make_double2(a.G * mi[l], a.c1 * theta * mi[l]);
      if (a.theta_out) a.theta_out[i] = theta;
    }
  } else {
    // ---- Eq. 2.11 + boundary dofs (App. B); the loads of all RZ nodes first ----
    unsigned fl[RZ];
    double vk[RZ][3];
#pragma unroll
    for (int l = 0; l < RZ; ++l) {
      const int64_t i = dead(l) ? i0 : cell(l);
      fl[l] = a.flags32[i];
#pragma unroll
      for (int k = 0; k < 3; ++k) vk[l][k] = a.v[k][i];
    }
#pragma unroll
    for (int l = 0; l < RZ; ++l) {
      if (p.gmu[l] == 0.0) continue;   // phantom or dead (a node has m_i > 0)
      const int64_t i = cell(l);
      double un[3];
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        const double fk = p.f[l][k] * a.vol_uniform;
        double vv = vk[l][k];
        double uk = p.uo[l][k];
        if (fl[l] & (1u << k)) {                    // clamped: u stays, v = 0
          vv = 0.0;
        } else if (fl[l] & (8u << k)) {             // prescribed velocity
          vv = a.bval[k][i];
          uk = __dadd_rn(uk, __dmul_rn(a.dt, vv));
        } else {
          const double bk = (fl[l] & PD_BODY_FORCE) ? a.bval[k][i] : 0.0;
          const double ac = __dmul_rn(__dadd_rn(fk, __dmul_rn(a.gramp, bk)), a.rrho);   // (f + g b) / rho
          vv = __dadd_rn(vv, __dmul_rn(a.dt, ac));
          uk = __dadd_rn(uk, __dmul_rn(a.dt, vv));
        }
        a.v[k][i] = vv;
        un[k] = uk;
      }
      a.uxy_w[i] = make_double2(un[0], un[1]);
      a.uz_w[i] = un[2];
    }
  }
}

// ---- the break test proper (Eq. 1.30) for the lanes whose filter fired: one warp per entry and node.
// Lane t tests bit t of each mask word of the node, so all its candidate bonds (those of the fired classes) are in
// flight together: dot >= thr on the bit patterns, bits cleared in the 128-bit masks and in every octant
// copy, the broken bonds taken out of the sum of Eq. 2.3, theta and {G/m, cth} of the nodes written again.
template <int RZ>
__global__ void __launch_bounds__(128, 6) k_ball_exact(const __grid_constant__ BArgs a) {
  const int lane = threadIdx.x & 31;
  const int nwarp = (int)((gridDim.x * blockDim.x) >> 5), count = *a.wl_count;
  if (count == 0) return;
  const int64_t zstr = (int64_t)a.DY * a.DX;
  // per mask bit q: xi, thr and the cell offset, in shared memory (thread q fills entry q: a lane-dependent index into the
  // constant bank is serialised, so it is paid once per CTA, not per candidate bond)
  __shared__ double tx0[128], tx1[128], tx2[128], tthr[128];
  __shared__ int64_t toff[128];
  {
    const int q = threadIdx.x;
    const uint32_t pk = a.pk[q];
    const int dx = (int)(pk & 15u) - S, dy = (int)((pk >> 4) & 15u) - S, dz = (int)((pk >> 8) & 15u) - S;
    tx0[q] = signed_const(a.xi[0][abs(dx)], dx < 0 ? (int)0x80000000 : 0);
    tx1[q] = signed_const(a.xi[1][abs(dy)], dy < 0 ? (int)0x80000000 : 0);
    tx2[q] = signed_const(a.xi[2][abs(dz)], dz < 0 ? (int)0x80000000 : 0);
    tthr[q] = a.thr[abs(dx)][abs(dy)][abs(dz)];
    toff[q] = ((int64_t)dz * a.DY + dy) * a.DX + dx;
  }
  __syncthreads();
  for (int task = (int)((blockIdx.x * blockDim.x + threadIdx.x) >> 5); task < count * RZ; task += nwarp) {
    const BEntry<RZ> *e = (const BEntry<RZ> *)a.wl + task / RZ;
    const int l = task % RZ;
    const int64_t i0 = e->i0;
    const int z0 = e->z0;
    const uint32_t cm = e->cm;
    uint32_t cand[4] = {0u, 0u, 0u, 0u};   // the bonds of the fired classes, per mask word
    for (int c = 1; c <= M2; ++c)
      if ((cm >> c) & 1u) {
#pragma unroll
        for (int w = 0; w < 4; ++w) cand[w] |= a.cmask[c][w];
      }
    {
      if (z0 + l >= a.PZ) continue;   // dead
      const int64_t i = i0 + l * zstr;
      const double2 uxy = a.uxy[i];
      const double u0 = uxy.x, u1 = uxy.y, u2 = a.uz[i];
      uint32_t m[4];
      bool has[4];
      double x0[4], x1[4], x2[4], thr[4];
      double2 xy[4];
      double z[4];
#pragma unroll
      for (int w = 0; w < 4; ++w) {   // this lane's candidate of each word: offset and geometry from the packed table
        m[w] = a.mask[(int64_t)w * a.npad + i];
        const uint32_t nf = a.nofail ? a.nofail[(int64_t)w * a.npad + i] : 0u;
        has[w] = ((m[w] & ~nf & cand[w]) >> lane) & 1u;
        const int q = w * 32 + lane;
        x0[w] = tx0[q]; x1[w] = tx1[q]; x2[w] = tx2[q]; thr[w] = tthr[q];
        const int64_t j = has[w] ? i + toff[q] : i;
        xy[w] = a.uxy[j];
        z[w] = a.uz[j];
      }
      double sub = 0.0;
      bool brokel = false;
#pragma unroll
      for (int w = 0; w < 4; ++w) {
        // the dot of the walk, bit for bit (a vanishing component of xi adds an exact zero)
        double dot = __dmul_rn(x0[w], xy[w].x - u0);
        dot = fma(x1[w], xy[w].y - u1, dot);
        dot = fma(x2[w], z[w] - u2, dot);
        // s >= s_c breaks: dot >= thr on the bit patterns (thr > 0), identical at both ends of the bond
        const bool brk = has[w] && __double_as_longlong(dot) >= __double_as_longlong(thr[w]);
        const uint32_t bb = __ballot_sync(FULL, brk);
        if (bb) {
          if (brk) {   // the bond's copies in the octant words (several lanes may share a word)
            const int2 o8 = a.q8[w * 32 + lane];
            for (int o = 0; o < 8; ++o)
              if ((o8.y >> o) & 1) atomicAnd(&a.mask8[(int64_t)o * a.npad + i], ~(1u << o8.x));
          }
          if (lane == 0) a.mask[(int64_t)w * a.npad + i] = m[w] & ~bb;
          double d = brk ? dot : 0.0;   // rho_ij <- 0: the bonds leave the sum of Eq. 2.3 (fixed summation order)
#pragma unroll
          for (int off = 16; off; off >>= 1) d += __shfl_xor_sync(FULL, d, off);
          sub += d;
          brokel = true;
        }
      }
      if (brokel && lane == 0) {
        const double mi = a.minv[i];
        const double theta = a.A * mi * ((e->acc[l] - sub) * a.vol_uniform);   // as in the epilogue of the walk
        a.aux[i] = make_double2(a.G * mi, a.c1 * theta * mi);
        if (a.theta_out) a.theta_out[i] = theta;
        a.tfull[e->tile] = 0;
      }
    }
  }
}

// octant words of the 128-bit masks: out[o][i] bit k <- in[q >> 5][i] bit (q & 31) for every octant o of q8[q].y
__global__ void k_ball_octants(int64_t npad, int nbits, const int2 *__restrict__ q8, const uint32_t *__restrict__ in,
                               uint32_t *__restrict__ out) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= npad) return;
  uint32_t o8[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  for (int w = 0; w < 4; ++w) {
    uint32_t rem = in[(int64_t)w * npad + i];
    while (rem) {
      const int bb = __ffs(rem) - 1;
      rem &= rem - 1u;
      const int q = w * 32 + bb;
      if (q >= nbits) continue;
      const int2 e = q8[q];
#pragma unroll
      for (int o = 0; o < 8; ++o)
        if ((e.y >> o) & 1) o8[o] |= 1u << e.x;
    }
  }
#pragma unroll
  for (int o = 0; o < 8; ++o) out[(int64_t)o * npad + i] = o8[o];
}

// warp tile (x chunk, row, RZ levels): every node has its full family, intact and allowed to break?
template <int RZ>
__global__ void k_ball_tileflags(BArgs a, int ntiles) {
  const int t = (int)(((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
  if (t >= ntiles) return;
  const int xc = t % a.nxc, y0 = (t / a.nxc) % a.PY, zt = t / (a.nxc * a.PY);
  const int64_t i0 = ((int64_t)(zt * RZ + a.HZ) * a.DY + (y0 + a.HY)) * a.DX + (xc * 32 + lane + a.HX);
  uint32_t notfull = 0;
  for (int l = 0; l < RZ; ++l) {
    if (zt * RZ + l >= a.PZ) { notfull = 1; break; }
    const int64_t i = i0 + (int64_t)l * a.DY * a.DX;
    for (int w = 0; w < 4; ++w)
      notfull |= (a.mask[(int64_t)w * a.npad + i] ^ ball_fullw(w)) | (a.nofail ? a.nofail[(int64_t)w * a.npad + i] : 0u);
  }
  const bool full = __all_sync(FULL, notfull == 0u);
  if (lane == 0) a.tfull[t] = full ? 1 : 0;
}

// ---------------------------------------------------------------- host side ----------------------------------------------------------------

int env_int(const char *name, int dflt) {
  const char *e = getenv(name);
  return e ? atoi(e) : dflt;
}

constexpr int BRZ = 4;   // levels per lane (the rows per CTA, 4 or 8, and the plane buffers, 2 or 3, are launch options)

struct BPrepared {
  BArgs a;
  bool ok = false;
  dim3 grid, block;
  int nb = 2, cy = 8;
  CUtensorMap tm_xy[2], tm_z[2], tm_g;   // per displacement buffer
};

// is the lattice's stencil the ball, bit for bit in the builder's layout?
bool ball_layout_matches(const pd_sim *s) {
  const PdLattice &l = s->lat;
  if (s->dim != 3 || !l.uniform || l.nbits != NBITS || l.nw != 4) return false;
  if (l.HX != S || l.HY != S || l.HZ != S || (l.DX & 1)) return false;
  int cnt = 0;
  for (int c = 0; c < l.ncol; ++c)
    for (int t = 0; t < l.cols[c].n; ++t, ++cnt)
      if (ball_bit(l.cols[c].dx, l.cols[c].dy0 + t, l.cols[c].dz) != l.cols[c].word * 32 + l.cols[c].bit0 + t) return false;
  if (cnt != 122) return false;
  for (int w = 0; w < 4; ++w)
    if (l.fullw[w] != ball_fullw(w)) return false;
  return true;
}

template <bool FORCE, bool FRAC, int CY, int NB, int MINB>
void ball_launch2(const BPrepared *pp, cudaStream_t st) {
  using SM = BSmem<FORCE, FRAC, BRZ, CY, NB>;
  auto kern = k_ball<FORCE, FRAC, BRZ, CY, NB, MINB>;
  static bool attr_done = false;   // per instantiation: opt in to > 48 KB of dynamic shared memory
  if (!attr_done) {
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SM::total);
    attr_done = true;
  }
  kern<<<pp->grid, pp->block, SM::total, st>>>(pp->a);
}
template <bool FORCE, bool FRAC>
void ball_launch(const BPrepared *pp, cudaStream_t st) {
  // (MINB = 512 / threads: 128 registers per thread)
  if (pp->cy == 8) { if (pp->nb == 3) ball_launch2<FORCE, FRAC, 8, 3, 2>(pp, st); else ball_launch2<FORCE, FRAC, 8, 2, 2>(pp, st); }
  else { if (pp->nb == 3) ball_launch2<FORCE, FRAC, 4, 3, 4>(pp, st); else ball_launch2<FORCE, FRAC, 4, 2, 4>(pp, st); }
}

// the device tables and the octant words, shared by the two passes
bool ball_tables(pd_sim *s) {
  PdLattice &l = s->lat;
  if (l.ball_q8) return true;
  std::vector<int2> q8(128, make_int2(0, 0));
  for (int dz = -S; dz <= S; ++dz)
    for (int dy = -S; dy <= S; ++dy)
      for (int dx = -S; dx <= S; ++dx) {
        if (!inball(dx, dy, dz)) continue;
        const int b = ball_bit(dx, dy, dz);
        int octs = 0;
        for (int o = 0; o < 8; ++o) {
          const int sx = o & 1, sy = (o >> 1) & 1, sz = (o >> 2) & 1;
          if ((dx == 0 || (dx < 0) == (sx != 0)) && (dy == 0 || (dy < 0) == (sy != 0)) && (dz == 0 || (dz < 0) == (sz != 0)))
            octs |= 1 << o;
        }
        q8[b] = make_int2(canon(abs(dx), abs(dy), abs(dz)), octs);
      }
  int2 *q8_d = (int2 *)pdi::dev_alloc(s, sizeof(int2) * 128);
  uint32_t *m8 = (uint32_t *)pdi::dev_alloc(s, sizeof(uint32_t) * 8 * s->npad);
  uint32_t *n8 = l.nofail ? (uint32_t *)pdi::dev_alloc(s, sizeof(uint32_t) * 8 * s->npad) : nullptr;
  if (!q8_d || !m8 || (l.nofail && !n8)) return false;
  if (cudaMemcpyAsync(q8_d, q8.data(), sizeof(int2) * 128, cudaMemcpyHostToDevice, s->stream) != cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  const unsigned nblk = (unsigned)((s->npad + 255) / 256);
  k_ball_octants<<<nblk, 256, 0, s->stream>>>(s->npad, l.nbits, q8_d, l.mask, m8);
  if (n8) k_ball_octants<<<nblk, 256, 0, s->stream>>>(s->npad, l.nbits, q8_d, l.nofail, n8);
  if (cudaGetLastError() != cudaSuccess || cudaStreamSynchronize(s->stream) != cudaSuccess) { cudaGetLastError(); return false; }
  l.ball_q8 = q8_d; l.mask8 = m8; l.nf8 = n8;
  return true;
}

BPrepared *ball_prepare(pd_sim *s, bool force) {
  PdLattice &l = s->lat;
  void *&slot = l.cache[force ? 5 : 4];
  if (slot) return (BPrepared *)slot;
  BPrepared *pp = new BPrepared();
  slot = pp;
  if (env_int("PD_BALL", 1) == 0 || !ball_layout_matches(s)) return pp;   // ok = false: the table-driven kernels
  BArgs &a = pp->a;
  memset(&a, 0, sizeof a);
  pp->nb = env_int("PD_BALL_NB", 2) == 3 ? 3 : 2;
  pp->cy = env_int("PD_BALL_CY", 8) == 4 ? 4 : 8;
  a.DX = l.DX; a.DY = l.DY; a.PY = l.PY; a.PZ = l.PZ; a.HX = l.HX; a.HY = l.HY; a.HZ = l.HZ;
  a.nxc = l.PX / 32; a.nyq = (l.PY + 8) / 4; a.nbits = l.nbits;
  a.npad = s->npad;
  a.aux = l.aux;
  a.mask = l.mask; a.nofail = l.nofail; a.rgocc = l.rgocc; a.flags32 = l.flags32; a.minv = s->minv;
  for (int q = 0; q < 3; ++q) { a.v[q] = s->v[q]; a.bval[q] = s->bval[q]; }
  a.A = s->A; a.c1 = s->c1; a.G = s->G; a.vol_uniform = s->vol_uniform; a.rrho = 1.0 / s->rho; a.dt = s->dt;
  a.gramp = 1.0;
  // constants, in the operation order of the walk (and of pd_lattice_uniform.cu): xi_k = o_k h_k, ||xi||^2 = fma chain
  for (int k = 0; k < 3; ++k)
    for (int q = 0; q < 4; ++q) a.xi[k][q] = (double)q * l.h[k];
  auto r2of = [&](int dx, int dy, int dz) {
    const double x0 = (double)dx * l.h[0], x1 = (double)dy * l.h[1], x2 = (double)dz * l.h[2];
    double r2 = x0 * x0;
    r2 = std::fma(x1, x1, r2);
    r2 = std::fma(x2, x2, r2);
    return r2;
  };
  for (int c = 0; c <= M2; ++c) a.thr_hi[c] = 0x7ff00000;
  for (int q = 0; q < 128; ++q) a.pk[q] = (uint32_t)S | (uint32_t)S << 4 | (uint32_t)S << 8;   // (unused bits: the zero offset)
  for (int dz = -S; dz <= S; ++dz)
    for (int dy = -S; dy <= S; ++dy)
      for (int dx = -S; dx <= S; ++dx)
        if (inball(dx, dy, dz)) {
          a.cmask[dx * dx + dy * dy + dz * dz][ball_bit(dx, dy, dz) >> 5] |= 1u << (ball_bit(dx, dy, dz) & 31);
          a.pk[ball_bit(dx, dy, dz)] = (uint32_t)(dx + S) | (uint32_t)(dy + S) << 4 | (uint32_t)(dz + S) << 8;
        }
  for (int i = 0; i < 4; ++i)
    for (int j = 0; j < 4; ++j)
      for (int k = 0; k < 4; ++k) {
        a.rinv[i][j][k] = (i | j | k) ? 1.0 / r2of(i, j, k) : 0.0;
        a.thr[i][j][k] = s->s_c * r2of(i, j, k);
        if (!inball(i, j, k)) continue;
        const double thr = s->s_c * r2of(i, j, k);
        long long bits;
        memcpy(&bits, &thr, 8);
        a.thr_hi[i * i + j * j + k * k] = std::min(a.thr_hi[i * i + j * j + k * k], (int)(bits >> 32));
      }
  if (!ball_tables(s)) { slot = nullptr; delete pp; return nullptr; }   // device allocation failed: nothing cached
  a.q8 = (const int2 *)l.ball_q8;
  a.mask8 = l.mask8; a.nf8 = l.nf8;
  if (!l.ball_tfull) {   // the warp-tile flags (kept in step by the exact pass)
    const int ntiles = ((l.PZ + BRZ - 1) / BRZ) * l.PY * a.nxc;
    uint8_t *tf = (uint8_t *)pdi::dev_alloc(s, (size_t)ntiles);
    if (!tf) { slot = nullptr; delete pp; return nullptr; }
    a.tfull = tf;
    k_ball_tileflags<BRZ><<<(unsigned)(((int64_t)ntiles * 32 + 255) / 256), 256, 0, s->stream>>>(a, ntiles);
    if (cudaGetLastError() != cudaSuccess || cudaStreamSynchronize(s->stream) != cudaSuccess) { cudaGetLastError(); return pp; }
    l.ball_tfull = tf;
  }
  a.tfull = l.ball_tfull;
  if (!l.ball_wl && s->fracture) {   // worklist of the break test: at most one entry per lane and launch
    const size_t ntiles = (size_t)((l.PZ + BRZ - 1) / BRZ) * l.PY * a.nxc;
    void *wl = pdi::dev_alloc(s, ntiles * 32 * sizeof(BEntry<BRZ>));
    int *cnt = (int *)pdi::dev_alloc(s, sizeof(int));
    if (!wl || !cnt) { slot = nullptr; delete pp; return nullptr; }
    l.ball_wl = wl; l.ball_wl_count = cnt;
  }
  a.wl = l.ball_wl; a.wl_count = l.ball_wl_count;
  const int sy = pp->cy + 2 * S;
  bool ok = true;
  for (int q = 0; q < 2 && ok; ++q)
    ok = make_plane_map(&pp->tm_xy[q], l.uxy[q], 2, l.DX, l.DY, l.DZ, BSX, sy) &&
         make_plane_map(&pp->tm_z[q], l.uz[q], 1, l.DX, l.DY, l.DZ, BSX, sy);
  if (ok) ok = make_plane_map(&pp->tm_g, l.aux, 2, l.DX, l.DY, l.DZ, BSX, sy);
  if (!ok) return pp;   // no tensor maps on this driver: the table-driven kernels
  pp->block = dim3((unsigned)(pp->cy * 32));
  pp->grid = dim3((unsigned)a.nxc, (unsigned)((l.PY + pp->cy - 1) / pp->cy), (unsigned)((l.PZ + BRZ - 1) / BRZ));
  pp->ok = true;
  return pp;
}

}  // namespace

namespace pdi {

// does this handle take the kernels of this file?  (the layout pd_get_layout reports)
bool ball_eligible(const pd_sim *s) { return env_int("PD_BALL", 1) != 0 && ball_layout_matches(s); }

void ball_free_cache(pd_sim *s) {
  for (int q = 4; q < 6; ++q) {
    delete (BPrepared *)s->lat.cache[q];
    s->lat.cache[q] = nullptr;
  }
}

// 1: launched; 0: the lattice is not the ball (the caller takes the table-driven kernels); < 0: error
int ball_launch_dilatation(pd_sim *s, double *theta_out, bool do_break) {
  BPrepared *pp = ball_prepare(s, false);
  if (!pp) { set_error("device allocation failed"); return PD_ERR_ALLOC; }
  if (!pp->ok) return 0;
  const PdLattice &l = s->lat;
  BArgs &a = pp->a;
  a.uxy = l.uxy[s->cur]; a.uz = l.uz[s->cur]; a.uxy_w = nullptr; a.uz_w = nullptr;
  a.tm_xy = pp->tm_xy[s->cur]; a.tm_z = pp->tm_z[s->cur]; a.tm_g = pp->tm_g;
  a.theta_out = theta_out;
  if (do_break && s->fracture) {
    if (cudaMemsetAsync(a.wl_count, 0, sizeof(int), s->stream) != cudaSuccess) { cudaGetLastError(); return 0; }
    ball_launch<false, true>(pp, s->stream);
    k_ball_exact<BRZ><<<148 * 12, 128, 0, s->stream>>>(a);   // (exits at once while no filter fires)
    s->launches += 1;
  } else {
    ball_launch<false, false>(pp, s->stream);
  }
  return 1;
}

int ball_launch_force_update(pd_sim *s) {
  BPrepared *pp = ball_prepare(s, true);
  if (!pp) { set_error("device allocation failed"); return PD_ERR_ALLOC; }
  if (!pp->ok) return 0;
  const PdLattice &l = s->lat;
  BArgs &a = pp->a;
  a.uxy = l.uxy[s->cur]; a.uz = l.uz[s->cur]; a.uxy_w = l.uxy[s->cur ^ 1]; a.uz_w = l.uz[s->cur ^ 1];
  a.tm_xy = pp->tm_xy[s->cur]; a.tm_z = pp->tm_z[s->cur]; a.tm_g = pp->tm_g;
  a.gramp = 1.0;
  if (s->ramp_time > 0.0) a.gramp = std::min(1.0, ((double)s->step * s->dt) / s->ramp_time);
  ball_launch<true, false>(pp, s->stream);
  return 1;
}

}  // namespace pdi
