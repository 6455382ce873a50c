// pd_lattice_step.cu -- step kernels of the dense lattice layout (pd_lattice.cu, PdLattice):
// SURVEY.md 8(a) rows a1-a5 for (jittered) lattice bodies.  Two families, same layout, same per-bond
// arithmetic (pd_bond.cuh, shared with pd_step.cu):
//
// (1) DIRECT kernels `k_lat_direct` -- the default.  One warp owns a ROW GROUP (32 lanes x R rows
//     adjacent in y, R = 4 in 3-D) at one level and walks all stencil COLUMNS (dx, dy0..dy0+n-1, dz)
//     with an R-record register window sliding along y: in step t row r pairs with record t + r, one
//     gathered record serves up to R bonds, the R bonds of a step are independent FP64 chains in one
//     basic block.  Records are read straight from the dense pair arrays by arithmetic addressing
//     (16-byte loads, 512 contiguous bytes per pair and warp, shared between warps through L1); there
//     is no shared-memory staging and no CTA barrier.  A column whose R n bonds are intact on all 32
//     lanes runs without a single mask test (FAST); otherwise the MASKED variant predicates the
//     accumulation and, in the dilatation pass, clears the bits of the bonds that break (Eq. 1.30).
//
// (2) MARCHING kernels `k_lat_march` (PD_LAT_KERNEL=march; kept as the measured alternative, see
//     profiles/r01b_design_history.md).  "2.5-D" marching: a CTA owns a column of cells, 32 (x) by
//     TY (y), and marches through LZ levels of z.  Shared memory holds a RING of 2 HZ + 2 z-PLANES of
//     neighbour records (the column's cells plus a halo of the stencil radius in x and y).  While
//     level z is computed from the planes z - HZ .. z + HZ, plane z + HZ + 1 and the mask words and
//     update operands of level z + 1 arrive through asynchronous copies (cp.async); NSPLIT warps
//     share a row group by splitting the stencil columns, their partial sums meet in shared memory.
#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>

#include "pd_bond.cuh"

namespace {

using pdb::FULL;
constexpr int TPB = 256;
constexpr int MAXSPLIT = 8;
inline unsigned nblk(int64_t n) { return (unsigned)((n + TPB - 1) / TPB); }

struct LatCol8 { int off; uint8_t n, word, bit0, dzi; };   // off = dy0 * SX + dx (records); dzi = dz + HZ

struct LatArgs {
  int DX, DY, DZ, HX, HY, HZ, PZ;
  int nxc, nyq;                      // x chunks; row groups along y (rgocc stride)
  int TY, LZ, SX, SY, NP;            // column height, levels per CTA, plane dims, planes in the ring
  int nsplit, nw;
  int cbeg[MAXSPLIT + 1];            // split s walks cols[cbeg[s] .. cbeg[s+1])
  int64_t npad;
  const double2 *nbr;                // pair arrays [PD_NP][npad] holding u^n (and cth^n)
  double2 *nbw;                      // dilatation: the same buffer (pair AUX written); force: the other buffer
  uint32_t *mask;
  const uint32_t *nofail;
  const uint8_t *rgocc;
  const uint32_t *flags32;
  const double *minv;
  const int32_t *thr;                // [ncol][8] filter thresholds (high words), in the order of cols[]
  double *v[3];
  const double *bval[3];
  double *theta_out;
  long long *trace;                  // PD_TRACE builds: per-warp clock64 stamps of one CTA
  double A, c1, G, s_c, vol_uniform, rrho, dt, gramp;   // gramp = g(t_n) = min(1, n dt / ramp_time)
  LatCol8 cols[PD_LAT_MAXCOL];
};

__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gsrc) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async8(void *smem_dst, const void *gsrc) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async4(void *smem_dst, const void *gsrc) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait0() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// predicated 16-byte shared-memory load: no branch, so the four bonds of a step stay in one basic block
__device__ __forceinline__ void lds_if(double2 &v, const double2 *ptr, uint32_t pred) {
  const unsigned a = (unsigned)__cvta_generic_to_shared(ptr);
  asm("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %3, 0;\n\t@p ld.shared.v2.f64 {%0, %1}, [%2];\n\t}"
      : "+d"(v.x), "+d"(v.y) : "r"(a), "r"(pred));
}

// a record = NPAIR pairs, pair k at plane + k * psz + idx
template <int NPAIR, class E>
__device__ __forceinline__ void lds_ent(E &e, const double2 *plane, int psz, int idx) {
  constexpr int DIMP = sizeof(e.p) / sizeof(double2);
#pragma unroll
  for (int k = 0; k < DIMP; ++k) e.p[k] = plane[k * psz + idx];
  if (NPAIR > DIMP) e.g = plane[DIMP * psz + idx];
}
template <int NPAIR, class E>
__device__ __forceinline__ void lds_ent_if(E &e, const double2 *plane, int psz, int idx, uint32_t pred) {
  constexpr int DIMP = sizeof(e.p) / sizeof(double2);
#pragma unroll
  for (int k = 0; k < DIMP; ++k) lds_if(e.p[k], plane + k * psz + idx, pred);
  if (NPAIR > DIMP) lds_if(e.g, plane + DIMP * psz + idx, pred);
}

// one stencil column: n steps, row r of step t pairs with the record at base + (t + r) * SX
template <bool MASKED, int NPAIR, class P>
__device__ __forceinline__ void lat_run_col(P &p, const double2 *plane, int psz, int base, int SX, int n,
                                            const uint32_t (&bits)[4], const uint32_t (&nfb)[4], uint32_t (&clr)[4],
                                            const int *thr) {
  typename P::E S[4];
#pragma unroll
  for (int q = 0; q < 4; ++q) lds_ent<NPAIR>(S[q], plane, psz, base + q * SX);
  uint32_t anyp = 0;
  if (MASKED) anyp = __reduce_or_sync(FULL, bits[0] | (bits[1] << 7) | (bits[2] << 14) | (bits[3] << 21));
  auto bond = [&](int r, const typename P::E &e, int t) {
    if (p.template bond<MASKED>(r, e, (bits[r] >> t) & 1u, (nfb[r] >> t) & 1u)) clr[r] |= 1u << t;
  };
#pragma unroll
  for (int t = 0; t < PD_MAXSTEP; ++t) {
    if (t < n) {
      const bool live = !MASKED || (anyp & (0x204081u << t)) != 0;   // warp-uniform
      if (live) bond(0, S[t % 4], t);
      lds_ent_if<NPAIR>(S[t % 4], plane, psz, base + (t + 4) * SX, (t + 1 < n) ? 1u : 0u);   // record t+4: row 3 of step t+1
      if (live) {
        bond(1, S[(t + 1) % 4], t);
        bond(2, S[(t + 2) % 4], t);
        bond(3, S[(t + 3) % 4], t);
      }
      if (!MASKED && P::kFrac) p.step_end(thr[t]);
    }
  }
}

}  // namespace

namespace {

template <int DIM, bool FORCE, bool FRAC> struct PolicyOf { using type = pdb::DilPolicy<DIM, FRAC, true, 4, true>; };
template <int DIM, bool FRAC> struct PolicyOf<DIM, true, FRAC> { using type = pdb::ForcePolicy<DIM, true, 4>; };
template <int DIM, bool FORCE, bool FRAC, int R> struct PolicyOfR { using type = pdb::DilPolicy<DIM, FRAC, true, R, true>; };
template <int DIM, bool FRAC, int R> struct PolicyOfR<DIM, true, FRAC, R> { using type = pdb::ForcePolicy<DIM, true, R>; };

// shared-memory carve-up (bytes), the same on host and device
struct LatSmem {
  size_t ring, smask, sepi, sfl, red, scol, sthr, sdirty, total;
};
__host__ __device__ inline LatSmem lat_smem(int npair, int epi, bool force, int NP, int SY, int SX, int TY, int nsplit, int nacc,
                                            int ncol) {
  LatSmem m;
  const size_t NTL = 32 * (size_t)TY;
  m.ring = 0;
  m.smask = m.ring + (size_t)NP * npair * SY * SX * sizeof(double2);
  m.sepi = m.smask + 2 * 4 * NTL * sizeof(uint32_t);
  m.sfl = m.sepi + 2 * (size_t)epi * NTL * sizeof(double);
  m.red = m.sfl + (force ? 2 * NTL * sizeof(uint32_t) : 0);
  m.scol = m.red + (size_t)(TY / 4) * nsplit * nacc * 32 * sizeof(double);
  m.sthr = m.scol + (size_t)ncol * sizeof(LatCol8);                  // column table
  m.sdirty = m.sthr + (force ? 0 : (size_t)ncol * 8 * sizeof(int));  // filter thresholds (dilatation)
  m.total = m.sdirty + 16;
  return m;
}

template <int DIM, bool FORCE, bool FRAC, int MAXT>
__global__ void __launch_bounds__(MAXT) k_lat_march(const __grid_constant__ LatArgs a) {
  extern __shared__ __align__(16) unsigned char smraw[];
  constexpr int NPAIR = FORCE ? DIM + 1 : DIM;
  constexpr int NACC = FORCE ? 4 * DIM : 4;
  constexpr int EPI = FORCE ? DIM : 1;
  using P = typename PolicyOf<DIM, FORCE, FRAC>::type;
  const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, warp = tid >> 5, nwarp = nthr >> 5;
  const int xc = blockIdx.x, x0 = xc * 32, y0 = blockIdx.y * a.TY, z_lo = blockIdx.z * a.LZ, z_hi = min(z_lo + a.LZ, a.PZ);
  const int nrg = a.TY >> 2, NTL = 32 * a.TY;
  const int psz = a.SY * a.SX, plsz = NPAIR * psz;
  const LatSmem lay = lat_smem(NPAIR, EPI, FORCE, a.NP, a.SY, a.SX, a.TY, a.nsplit, NACC, a.cbeg[MAXSPLIT]);
  double2 *ring = (double2 *)(smraw + lay.ring);
  uint32_t *smask = (uint32_t *)(smraw + lay.smask);   // [2][4][NTL]
  double *sepi = (double *)(smraw + lay.sepi);         // [2][EPI][NTL]: minv (dilatation) / v (force)
  uint32_t *sfl = (uint32_t *)(smraw + lay.sfl);       // [2][NTL] flags (force)
  double *red = (double *)(smraw + lay.red);           // [nrg][nsplit][NACC][32]
  int *sdirty = (int *)(smraw + lay.sdirty);           // [2]
  LatCol8 *scol = (LatCol8 *)(smraw + lay.scol);       // the column table (shared-memory copy: short, fixed latency)
  int *sthr = (int *)(smraw + lay.sthr);               // [ncol][8] break-filter thresholds

  // ---- nothing to do in this column segment? ----
  int occ = 0;
  for (int z = z_lo + tid; z < z_hi; z += nthr)
    for (int q = 0; q < nrg; ++q) occ |= a.rgocc[((int64_t)z * a.nyq + ((y0 >> 2) + q)) * a.nxc + xc];
  if (!__syncthreads_or(occ)) return;
  {
    const int ncol = a.cbeg[MAXSPLIT];
    for (int c = tid; c < ncol; c += nthr) scol[c] = a.cols[c];
    if (!FORCE && a.thr)
      for (int c = tid; c < ncol * 8; c += nthr) sthr[c] = a.thr[c];
  }

  auto load_plane = [&](int pz, int slot) {   // cell level pz (may be in the margin) -> ring slot
    for (int pp = 0; pp < NPAIR; ++pp) {
      const int gp = pp < DIM ? pp : PD_P_AUX;
      const double2 *src = a.nbr + (int64_t)gp * a.npad + ((int64_t)(pz + a.HZ) * a.DY + y0) * a.DX + x0 + lane;
      double2 *dst = ring + (int64_t)slot * plsz + pp * psz + lane;
      const bool two = lane + 32 < a.SX;
      for (int yy = warp; yy < a.SY; yy += nwarp) {
        cp_async16(dst + yy * a.SX, src + (int64_t)yy * a.DX);
        if (two) cp_async16(dst + yy * a.SX + 32, src + (int64_t)yy * a.DX + 32);
      }
    }
  };
  auto load_level = [&](int z, int buf) {   // mask words and update operands of the owned nodes of level z
    for (int tn = tid; tn < NTL; tn += nthr) {
      const int64_t i = ((int64_t)(z + a.HZ) * a.DY + (y0 + (tn >> 5) + a.HY)) * a.DX + (x0 + (tn & 31) + a.HX);
      for (int w = 0; w < a.nw; ++w) cp_async4(smask + (buf * 4 + w) * NTL + tn, a.mask + (int64_t)w * a.npad + i);
      if (FORCE) {
#pragma unroll
        for (int k = 0; k < DIM; ++k) cp_async8(sepi + (buf * EPI + k) * NTL + tn, a.v[k] + i);
        cp_async4(sfl + buf * NTL + tn, a.flags32 + i);
      } else {
        cp_async8(sepi + buf * NTL + tn, a.minv + i);
      }
    }
    if (tid == 0) sdirty[buf] = 0;
  };

  // ---- this warp's row group and column split ----
  const int rg = warp / a.nsplit, sp = warp - rg * a.nsplit;
  const int own0 = (rg * 4 + a.HY) * a.SX + lane + a.HX;   // row 0's own record inside a plane
  const int tn0 = rg * 4 * 32 + lane;                      // row 0's node inside a level

  // ---- prologue: planes z_lo - HZ .. z_lo + HZ, level z_lo ----
  for (int q = 0; q <= 2 * a.HZ; ++q) load_plane(z_lo - a.HZ + q, q);
  load_level(z_lo, 0);
  cp_async_commit();
  int slot_lo = 0, buf = 0;   // ring slot of plane z - HZ; buffer of level z
#ifdef PD_TRACE
  const bool tr = a.trace && blockIdx.x == 2 && blockIdx.y == gridDim.y / 2 && blockIdx.z == gridDim.z / 2 && lane == 0;
#define STAMP(k) if (tr) a.trace[((z - z_lo) * 16 + warp) * 8 + (k)] = clock64();
#else
#define STAMP(k)
#endif
  // which levels hold a node of this warp's row group (read once: no global load inside the level loop)
  unsigned long long actbits = 0;
  for (int z = z_lo; z < z_hi; ++z)
    if (a.rgocc[((int64_t)z * a.nyq + ((y0 >> 2) + rg)) * a.nxc + xc]) actbits |= 1ull << (z - z_lo);
  // which sums this warp finishes after the level's barrier: q = sp, sp + nsplit, ...
  uint32_t mine = 0;
  for (int q = sp; q < NACC; q += a.nsplit) mine |= 1u << q;
  for (int z = z_lo; z < z_hi; ++z) {
    STAMP(0)
    cp_async_wait0();
    __syncthreads();   // level z's planes and operands have landed; every warp is done with level z - 1
    STAMP(1)
    {   // one level ahead: plane z + HZ + 1 into the slot of plane z - HZ - 1, operands of level z + 1
      int ns = slot_lo + 2 * a.HZ + 1;
      if (ns >= a.NP) ns -= a.NP;
      if (z + 2 * a.HZ + 1 < a.DZ) load_plane(z + a.HZ + 1, ns);
      if (z + 1 < z_hi) load_level(z + 1, buf ^ 1);
      cp_async_commit();
    }
    STAMP(2)
    const bool active = (actbits >> (z - z_lo)) & 1ull;
    P p;
    double acc[NACC];
    if (active) {
      int sz = slot_lo + a.HZ;
      if (sz >= a.NP) sz -= a.NP;
      const double2 *pl0 = ring + (int64_t)sz * plsz;
#pragma unroll
      for (int r = 0; r < 4; ++r) {
#pragma unroll
        for (int k = 0; k < DIM; ++k) {
          const double2 xu = pl0[k * psz + own0 + r * a.SX];
          p.xo[r][k] = xu.x;
          p.uo[r][k] = xu.y;
        }
      }
      if constexpr (FORCE) {
#pragma unroll
        for (int r = 0; r < 4; ++r) {
          const double2 g = pl0[DIM * psz + own0 + r * a.SX];
          p.gmu_i[r] = g.x;
          p.cth_i[r] = g.y;
#pragma unroll
          for (int k = 0; k < DIM; ++k) p.f[r][k] = 0.0;
        }
      } else {
        p.s_c = a.s_c;
#pragma unroll
        for (int r = 0; r < 4; ++r) p.acc[r] = 0.0;
      }
      const uint32_t *mk = smask + buf * 4 * NTL + tn0;
      for (int c = a.cbeg[sp]; c < a.cbeg[sp + 1]; ++c) {
        const LatCol8 col = scol[c];
        const int n = col.n;
        const uint32_t nmask = (1u << n) - 1u;
        uint32_t bits[4], nfb[4] = {0, 0, 0, 0}, clr[4] = {0, 0, 0, 0};
#pragma unroll
        for (int r = 0; r < 4; ++r) bits[r] = (mk[col.word * NTL + r * 32] >> col.bit0) & nmask;
        bool slow = !__all_sync(FULL, (bits[0] & bits[1] & bits[2] & bits[3]) == nmask);
        int s2 = slot_lo + col.dzi;
        if (s2 >= a.NP) s2 -= a.NP;
        const double2 *pl = ring + (int64_t)s2 * plsz;
        const int base = own0 + col.off;
        const int *thr = sthr + 8 * c;   // filter thresholds of the column's steps
        if (!slow) {
          p.fast_begin();
          lat_run_col<false, NPAIR>(p, pl, psz, base, a.SX, n, bits, nfb, clr, thr);
          slow = p.fast_failed();
        }
        if (slow) {
          if (P::kFrac && a.nofail) {
#pragma unroll
            for (int r = 0; r < 4; ++r) {
              const int64_t i = ((int64_t)(z + a.HZ) * a.DY + (y0 + rg * 4 + r + a.HY)) * a.DX + (x0 + lane + a.HX);
              nfb[r] = (a.nofail[(int64_t)col.word * a.npad + i] >> col.bit0) & nmask;
            }
          }
          lat_run_col<true, NPAIR>(p, pl, psz, base, a.SX, n, bits, nfb, clr, thr);
          if (P::kFrac) {
            uint32_t anyclr = 0;
#pragma unroll
            for (int r = 0; r < 4; ++r) {
              if (clr[r]) atomicAnd(smask + (buf * 4 + col.word) * NTL + tn0 + r * 32, ~(clr[r] << col.bit0));
              anyclr |= clr[r];
            }
            if (anyclr) sdirty[buf] = 1;
          }
        }
      }
      if constexpr (FORCE) {
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
          for (int k = 0; k < DIM; ++k) acc[r * DIM + k] = p.f[r][k];
      } else {
#pragma unroll
        for (int r = 0; r < 4; ++r) acc[r] = p.acc[r];
      }
#pragma unroll
      for (int q = 0; q < NACC; ++q) red[((rg * a.nsplit + sp) * NACC + q) * 32 + lane] = acc[q];
    }
    STAMP(3)
    __syncthreads();   // the level's planes are no longer read; partial sums and broken bits are visible
    STAMP(4)
    if (active) {
      // every warp of the row group finishes the sums `mine`: fixed summation order over the splits
      const int64_t i0 = ((int64_t)(z + a.HZ) * a.DY + (y0 + rg * 4 + a.HY)) * a.DX + (x0 + lane + a.HX);
      const double *rd = red + (size_t)rg * a.nsplit * NACC * 32 + lane;
      if (FRAC && sp == 0 && sdirty[buf]) {   // broken bits back to HBM
#pragma unroll
        for (int r = 0; r < 4; ++r)
          for (int w = 0; w < a.nw; ++w)
            a.mask[(int64_t)w * a.npad + i0 + (int64_t)r * a.DX] = smask[(buf * 4 + w) * NTL + tn0 + r * 32];
      }
#pragma unroll
      for (int q = 0; q < NACC; ++q) {
        if (!((mine >> q) & 1u)) continue;   // warp-uniform
        double part[MAXSPLIT];
#pragma unroll
        for (int s3 = 0; s3 < MAXSPLIT; ++s3) part[s3] = s3 < a.nsplit ? rd[(s3 * NACC + q) * 32] : 0.0;
        double sum = part[0];
#pragma unroll
        for (int s3 = 1; s3 < MAXSPLIT; ++s3) sum += part[s3];   // fixed order; absent splits add +0
        if constexpr (!FORCE) {
          const int r = q;
          const int64_t i = i0 + (int64_t)r * a.DX;
          const double mi = sepi[buf * NTL + tn0 + r * 32];   // 0 for phantoms
          const double theta = a.A * mi * (sum * a.vol_uniform);
          a.nbw[(int64_t)PD_P_AUX * a.npad + i] = make_double2(a.G * mi, a.c1 * theta * mi);
          if (a.theta_out) a.theta_out[i] = theta;
        } else {
          // ---- Eq. 2.11 + boundary dofs (App. B) ----
          const int r = q / DIM, k = q - r * DIM;
          if (p.gmu_i[r] == 0.0) continue;   // phantom (a node has m_i > 0)
          const int64_t i = i0 + (int64_t)r * a.DX;
          const unsigned fl = sfl[buf * NTL + tn0 + r * 32];
          const double fk = sum * a.vol_uniform;
          double vk = sepi[(buf * EPI + k) * NTL + tn0 + r * 32];
          double uk = p.uo[r][k];
          if (fl & (1u << k)) {                       // clamped: u stays, v = 0
            vk = 0.0;
          } else if (fl & (8u << k)) {                // prescribed velocity
            vk = a.bval[k][i];
            uk = __dadd_rn(uk, __dmul_rn(a.dt, vk));
          } else {
            const double bk = (fl & PD_BODY_FORCE) ? a.bval[k][i] : 0.0;
            const double ac = __dmul_rn(__dadd_rn(fk, __dmul_rn(a.gramp, bk)), a.rrho);   // (f + g b) / rho
            vk = __dadd_rn(vk, __dmul_rn(a.dt, ac));
            uk = __dadd_rn(uk, __dmul_rn(a.dt, vk));
          }
          a.v[k][i] = vk;
          a.nbw[(int64_t)k * a.npad + i] = make_double2(p.xo[r][k], uk);
        }
      }
    }
    STAMP(5)
    slot_lo = slot_lo + 1 == a.NP ? 0 : slot_lo + 1;
    buf ^= 1;
  }
}

}  // namespace

// ================================================================================================
// DIRECT variant: no shared-memory staging and no CTA barriers.  One warp owns a row group
// (32 lanes x 4 rows) at one level and walks ALL stencil columns for it; the neighbour records are
// read straight from the dense pair arrays with 16-byte loads (a warp reads 512 contiguous bytes per
// pair; the records of a stencil neighbourhood are shared between the warps of a CTA through L1).
// Addresses are arithmetic (cell + stencil offset): nothing is read to find a neighbour.
namespace {

// predicated 16-byte read-only load: no branch, so the four bonds of a step stay in one basic block
__device__ __forceinline__ void ldg_if(double2 &v, const double2 *ptr, uint32_t pred) {
  asm("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %3, 0;\n\t@p ld.global.nc.v2.f64 {%0, %1}, [%2];\n\t}"
      : "+d"(v.x), "+d"(v.y) : "l"(ptr), "r"(pred));
}
// a record = NPAIR pairs; pk[k] points at pair k of the warp's own row-0 cell, off is the (32-bit) cell offset
template <int NPAIR, class E>
__device__ __forceinline__ void ldg_ent(E &e, const double2 *const (&pk)[NPAIR], int off) {
  constexpr int DIMP = sizeof(e.p) / sizeof(double2);
#pragma unroll
  for (int k = 0; k < DIMP; ++k) e.p[k] = __ldg(pk[k] + off);
  if (NPAIR > DIMP) e.g = __ldg(pk[DIMP] + off);
}
template <int NPAIR, class E>
__device__ __forceinline__ void ldg_ent_if(E &e, const double2 *const (&pk)[NPAIR], int off, uint32_t pred) {
  constexpr int DIMP = sizeof(e.p) / sizeof(double2);
#pragma unroll
  for (int k = 0; k < DIMP; ++k) ldg_if(e.p[k], pk[k] + off, pred);
  if (NPAIR > DIMP) ldg_if(e.g, pk[DIMP] + off, pred);
}

// R rows per lane (R = 4: one record serves up to 4 bonds; R = 2: half the registers, twice the warps)
template <bool MASKED, bool STAGED, int NPAIR, int R, class P>
__device__ __forceinline__ void dir_run_col(P &p, const double2 *const (&pk)[NPAIR], int base, int DX, int n,
                                            const uint32_t (&bits)[R], const uint32_t (&nfb)[R], uint32_t (&clr)[R],
                                            const int *thr) {
  typename P::E S[R];
#pragma unroll
  for (int q = 0; q < R; ++q) ldg_ent<NPAIR>(S[q], pk, base + q * DX);
  uint32_t anyp = 0;
  if (MASKED) {
    uint32_t pkd = 0;
#pragma unroll
    for (int r = 0; r < R; ++r) pkd |= bits[r] << (7 * r);
    anyp = __reduce_or_sync(FULL, pkd);
  }
  constexpr uint32_t STEPBITS = R == 4 ? 0x204081u : (R == 2 ? 0x81u : 0x1u);
  auto bond = [&](int r, const typename P::E &e, int t) {
    if (p.template bond<MASKED>(r, e, (bits[r] >> t) & 1u, (nfb[r] >> t) & 1u)) clr[r] |= 1u << t;
  };
#pragma unroll
  for (int t = 0; t < PD_MAXSTEP; ++t) {
    if (t < n) {
      const bool live = !MASKED || (anyp & (STEPBITS << t)) != 0;   // warp-uniform
      if (STAGED) {
        // differences of the R rows first (row 0 frees its slot for the next record), then the products
        // phase by phase over the rows (pd_bond.cuh, finish)
        if (live) p.diffs(0, S[t % R]);
        ldg_ent_if<NPAIR>(S[t % R], pk, base + (t + R) * DX, (t + 1 < n) ? 1u : 0u);
        if (live) {
#pragma unroll
          for (int r = 1; r < R; ++r) p.diffs(r, S[(t + r) % R]);
          uint32_t in4 = (1u << R) - 1u, nf4 = 0u;
          if (MASKED) {
            in4 = 0;
#pragma unroll
            for (int r = 0; r < R; ++r) { in4 |= ((bits[r] >> t) & 1u) << r; nf4 |= ((nfb[r] >> t) & 1u) << r; }
          }
          const uint32_t brk = p.template finish<MASKED>(in4, nf4);
          if (MASKED && P::kFrac) {
#pragma unroll
            for (int r = 0; r < R; ++r) clr[r] |= ((brk >> r) & 1u) << t;
          }
        }
      } else {
        if (live) bond(0, S[t % R], t);
        ldg_ent_if<NPAIR>(S[t % R], pk, base + (t + R) * DX, (t + 1 < n) ? 1u : 0u);   // record t+R: last row of step t+1
        if (live) {
#pragma unroll
          for (int r = 1; r < R; ++r) bond(r, S[(t + r) % R], t);
        }
      }
      if (!MASKED && P::kFrac) p.step_end(thr[t]);
    }
  }
}

struct DirArgs {
  int DX, DY, HX, HY, HZ, PZ;
  int nxc, nyq, nyq_used;            // x chunks; rgocc stride; row groups along y that can hold nodes
  int ncol, nw, cy, cz, rows;        // columns; mask words; row groups (y) and levels (z) per CTA; rows per lane
  int64_t npad;
  const double2 *nbr;
  double2 *nbw;
  uint32_t *mask;
  const uint32_t *nofail;
  const uint8_t *rgocc;
  const uint32_t *flags32;
  const double *minv;
  const int32_t *thr;
  double *v[3];
  const double *bval[3];
  double *theta_out;
  double A, c1, G, s_c, vol_uniform, rrho, dt, gramp;
  struct Col { int off; uint8_t n, word, bit0, pad; } cols[PD_LAT_MAXCOL];   // off = (dz*DY + dy0)*DX + dx (dense cells)
};

template <int DIM, bool FORCE, bool FRAC, int MAXT, int MINB, bool STAGED, int R>
__global__ void __launch_bounds__(MAXT, MINB) k_lat_direct(const __grid_constant__ DirArgs a) {
  extern __shared__ __align__(16) unsigned char smraw[];
  constexpr int NPAIR = FORCE ? DIM + 1 : DIM;
  using P = typename PolicyOfR<DIM, FORCE, FRAC, R>::type;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarp = blockDim.x >> 5;
  // shared: column table, thresholds, per-warp mask words [nwarp][4 words][4 rows][32]
  DirArgs::Col *scol = (DirArgs::Col *)smraw;
  int *sthr = (int *)(scol + a.ncol);
  uint32_t *smk = (uint32_t *)(sthr + (FORCE ? 0 : a.ncol * 8)) + warp * (128 * R);
  for (int c = tid; c < a.ncol; c += blockDim.x) scol[c] = a.cols[c];
  if (!FORCE && a.thr)
    for (int c = tid; c < a.ncol * 8; c += blockDim.x) sthr[c] = a.thr[c];
  // this warp's row group: (xc, yq, z)
  const int wy = warp % a.cy, wz = warp / a.cy;
  const int xc = blockIdx.x, yq = blockIdx.y * a.cy + wy, z = blockIdx.z * a.cz + wz;   // yq counts groups of R rows
  const bool active = yq < a.nyq_used && z < a.PZ && a.rgocc[((int64_t)z * a.nyq + ((yq * R) >> 2)) * a.nxc + xc] != 0;
  const int64_t i0 = ((int64_t)(z + a.HZ) * a.DY + (yq * R + a.HY)) * a.DX + (xc * 32 + lane + a.HX);   // row 0's cell
  if (active) {
#pragma unroll
    for (int r = 0; r < R; ++r)
      for (int w = 0; w < a.nw; ++w) smk[(w * R + r) * 32 + lane] = a.mask[(int64_t)w * a.npad + i0 + (int64_t)r * a.DX];
  }
  __syncthreads();   // tables visible (the only CTA barrier)
  if (!active) return;
  P p;
#pragma unroll
  for (int r = 0; r < R; ++r) {
#pragma unroll
    for (int k = 0; k < DIM; ++k) {
      const double2 xu = a.nbr[(int64_t)k * a.npad + i0 + (int64_t)r * a.DX];
      p.xo[r][k] = xu.x;
      p.uo[r][k] = xu.y;
    }
  }
  if constexpr (FORCE) {
#pragma unroll
    for (int r = 0; r < R; ++r) {
      const double2 g = a.nbr[(int64_t)PD_P_AUX * a.npad + i0 + (int64_t)r * a.DX];
      p.gmu_i[r] = g.x;
      p.cth_i[r] = g.y;
#pragma unroll
      for (int k = 0; k < DIM; ++k) p.f[r][k] = 0.0;
    }
  } else {
    p.s_c = a.s_c;
#pragma unroll
    for (int r = 0; r < R; ++r) p.acc[r] = 0.0;
  }
  const double2 *pk[NPAIR];   // pair k of the warp's own row-0 cell: a record is pk[k] + (32-bit cell offset)
#pragma unroll
  for (int k = 0; k < NPAIR; ++k) pk[k] = a.nbr + (int64_t)(k < DIM ? k : PD_P_AUX) * a.npad + i0;
  bool dirty = false;
  for (int c = 0; c < a.ncol; ++c) {
    const DirArgs::Col col = scol[c];
    const int n = col.n;
    const uint32_t nmask = (1u << n) - 1u;
    uint32_t bits[R], nfb[R], clr[R];
#pragma unroll
    for (int r = 0; r < R; ++r) nfb[r] = clr[r] = 0;
#pragma unroll
    for (int r = 0; r < R; ++r) bits[r] = (smk[(col.word * R + r) * 32 + lane] >> col.bit0) & nmask;
    uint32_t ball = bits[0];
#pragma unroll
    for (int r = 1; r < R; ++r) ball &= bits[r];
    bool slow = !__all_sync(FULL, ball == nmask);
    const int base = col.off;
    const int *thr = sthr + 8 * c;
    if (!slow) {
      p.fast_begin();
      dir_run_col<false, STAGED, NPAIR, R>(p, pk, base, a.DX, n, bits, nfb, clr, thr);
      slow = p.fast_failed();
    }
    if (slow) {
      if (P::kFrac && a.nofail) {
#pragma unroll
        for (int r = 0; r < R; ++r) nfb[r] = (a.nofail[(int64_t)col.word * a.npad + i0 + (int64_t)r * a.DX] >> col.bit0) & nmask;
      }
      dir_run_col<true, STAGED, NPAIR, R>(p, pk, base, a.DX, n, bits, nfb, clr, thr);
      if (P::kFrac) {
#pragma unroll
        for (int r = 0; r < R; ++r)
          if (clr[r]) { smk[(col.word * R + r) * 32 + lane] &= ~(clr[r] << col.bit0); dirty = true; }
      }
    }
  }
  if (FRAC && __any_sync(FULL, dirty)) {   // broken bits back to HBM
    if (dirty) {
#pragma unroll
      for (int r = 0; r < R; ++r)
        for (int w = 0; w < a.nw; ++w) a.mask[(int64_t)w * a.npad + i0 + (int64_t)r * a.DX] = smk[(w * R + r) * 32 + lane];
    }
  }
  if constexpr (!FORCE) {
    double mi[R];
#pragma unroll
    for (int r = 0; r < R; ++r) mi[r] = a.minv[i0 + (int64_t)r * a.DX];
#pragma unroll
    for (int r = 0; r < R; ++r) {
      const int64_t i = i0 + (int64_t)r * a.DX;
      const double theta = a.A * mi[r] * (p.acc[r] * a.vol_uniform);   // minv = 0 for phantoms
      a.nbw[(int64_t)PD_P_AUX * a.npad + i] = make_double2(a.G * mi[r], a.c1 * theta * mi[r]);
      if (a.theta_out) a.theta_out[i] = theta;
    }
  } else {
    // ---- Eq. 2.11 + boundary dofs (App. B) ----
    double vk[R][DIM];
    unsigned fl[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
      fl[r] = a.flags32[i0 + (int64_t)r * a.DX];
#pragma unroll
      for (int k = 0; k < DIM; ++k) vk[r][k] = a.v[k][i0 + (int64_t)r * a.DX];
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
      if (p.gmu_i[r] == 0.0) continue;   // phantom (a node has m_i > 0)
      const int64_t i = i0 + (int64_t)r * a.DX;
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
        a.nbw[(int64_t)k * a.npad + i] = make_double2(p.xo[r][k], uk);
      }
    }
  }
}

}  // namespace

namespace {

// phi_i = 1 - sum_j rho_ij V_j / sum_j V_j (Eq. 1.31) and the three damage scalars
__global__ void k_lat_damage(int64_t npad, int nw, double vol_uniform, const int32_t *__restrict__ perm,
                             const uint32_t *__restrict__ mask, const int32_t *__restrict__ rowlen,
                             const double *__restrict__ fvol, double *phi_out, unsigned long long *stats) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  unsigned long long broken = 0, ge_half = 0;
  double phimax = 0.0;
  if (i < npad && perm[i] >= 0) {
    int cnt = 0;
    for (int w = 0; w < nw; ++w) cnt += __popc(mask[(int64_t)w * npad + i]);
    double sum = 0.0;   // the sum of cnt equal volumes, added one by one like sum_j V_j was
    for (int q = 0; q < cnt; ++q) sum += vol_uniform;
    const double phi = 1.0 - sum / fvol[i];
    phi_out[i] = phi;
    broken = (unsigned long long)(rowlen[i] - cnt);
    ge_half = phi >= 0.5 ? 1ull : 0ull;
    phimax = phi;
  }
  unsigned long long pbits = (unsigned long long)__double_as_longlong(fmax(phimax, 0.0));  // phi >= 0: bit order = value order
  for (int o = 16; o > 0; o >>= 1) {
    broken += __shfl_xor_sync(FULL, broken, o);
    ge_half += __shfl_xor_sync(FULL, ge_half, o);
    unsigned long long other = __shfl_xor_sync(FULL, pbits, o);
    pbits = other > pbits ? other : pbits;
  }
  if ((threadIdx.x & 31) == 0) {
    if (broken) atomicAdd(&stats[0], broken);
    if (pbits) atomicMax(&stats[1], pbits);
    if (ge_half) atomicAdd(&stats[2], ge_half);
  }
}

int env_int(const char *name, int dflt) {
  const char *e = getenv(name);
  return e ? atoi(e) : dflt;
}

constexpr size_t SMEM_MAX = 232448;   // 227 KB opt-in per CTA on sm_100

// column geometry, column table split between the warps of a row group, pointers.
// Returns the dynamic shared-memory size.
size_t lat_make_args(pd_sim *s, LatArgs &a, bool force, int TY, int LZ, int nsplit) {
  const PdLattice &l = s->lat;
  const int dim = s->dim, npair = force ? dim + 1 : dim;
  a.DX = l.DX; a.DY = l.DY; a.DZ = l.DZ; a.HX = l.HX; a.HY = l.HY; a.HZ = l.HZ; a.PZ = l.PZ;
  a.TY = TY; a.LZ = LZ;
  a.SX = 32 + 2 * l.HX; a.SY = TY + 2 * l.HY; a.NP = 2 * l.HZ + 2;
  a.nxc = l.PX / 32; a.nyq = (l.PY + 8) / 4;
  a.nsplit = nsplit; a.nw = l.nw;
  a.npad = s->npad;
  // greedy balance of the columns over the splits (by steps + a fixed cost per column), longest first
  std::vector<int> order(l.ncol), owner(l.ncol), load(nsplit, 0);
  for (int c = 0; c < l.ncol; ++c) order[c] = c;
  std::stable_sort(order.begin(), order.end(), [&](int x, int y) { return l.cols[x].n > l.cols[y].n; });
  for (int c : order) {
    int best = 0;
    for (int q = 1; q < nsplit; ++q) if (load[q] < load[best]) best = q;
    owner[c] = best;
    load[best] += 4 * l.cols[c].n + 3;
  }
  int k = 0;
  for (int q = 0; q < nsplit; ++q) {
    a.cbeg[q] = k;
    for (int c = 0; c < l.ncol; ++c)
      if (owner[c] == q) {
        const PdLatCol &src = l.cols[c];
        a.cols[k].off = src.dy0 * a.SX + src.dx;
        a.cols[k].n = src.n; a.cols[k].word = src.word; a.cols[k].bit0 = src.bit0; a.cols[k].dzi = (uint8_t)(src.dz + l.HZ);
        ++k;
      }
  }
  for (int q = nsplit; q <= MAXSPLIT; ++q) a.cbeg[q] = k;
  a.nbr = s->nb[s->cur]; a.nbw = s->nb[force ? s->cur ^ 1 : s->cur];
  a.mask = l.mask; a.nofail = l.nofail; a.rgocc = l.rgocc; a.flags32 = l.flags32; a.minv = s->minv;
  for (int q = 0; q < 3; ++q) { a.v[q] = s->v[q]; a.bval[q] = s->bval[q]; }
  a.theta_out = nullptr;
  a.trace = nullptr;
  a.A = s->A; a.c1 = s->c1; a.G = s->G; a.s_c = s->s_c; a.vol_uniform = s->vol_uniform; a.rrho = 1.0 / s->rho; a.dt = s->dt;
  a.gramp = 1.0;
  if (s->ramp_time > 0.0) a.gramp = std::min(1.0, ((double)s->step * s->dt) / s->ramp_time);
  return lat_smem(npair, force ? dim : 1, force, a.NP, a.SY, a.SX, TY, nsplit, force ? 4 * dim : 4, k).total;
}

// TY, NSPLIT, LZ: environment overrides (tuning), else the largest configuration that fits
bool lat_pick(pd_sim *s, LatArgs &a, bool force, int maxthreads, int &TY, int &LZ, int &nsplit, size_t &smem) {
  const PdLattice &l = s->lat;
  const char *pre = force ? "PD_LAT_FRC" : "PD_LAT_DIL";
  char nm[64];
  snprintf(nm, sizeof nm, "%s_TY", pre); TY = env_int(nm, 0);
  snprintf(nm, sizeof nm, "%s_NSPLIT", pre); int ns_env = env_int(nm, 0);
  snprintf(nm, sizeof nm, "%s_LZ", pre); LZ = env_int(nm, 0);
  bool ok = false;
  for (int ty : {8, 4}) {
    if (TY != 0 && TY != ty) continue;
    int ns = ns_env > 0 ? std::min(ns_env, MAXSPLIT) : MAXSPLIT;
    ns = std::min(ns, std::max(1, maxthreads / (32 * (ty / 4))));
    for (; ns >= 1; --ns) {
      smem = lat_make_args(s, a, force, ty, 1, ns);
      if (smem <= SMEM_MAX) break;
    }
    if (ns >= 1) { TY = ty; nsplit = ns; ok = true; break; }
  }
  if (!ok) return false;
  if (LZ <= 0) {   // about 4 CTAs per SM over the run, at least 6 levels per CTA (the ring is filled once per CTA)
    const int ncols = (l.PX / 32) * ((l.PY + TY - 1) / TY);
    int nzs = std::max(1, std::min(l.PZ / 6, (592 + ncols - 1) / ncols));
    LZ = (l.PZ + nzs - 1) / nzs;
  }
  LZ = std::max(1, std::min(std::min(LZ, 64), l.PZ));   // (a 64-bit activity mask per CTA)
  smem = lat_make_args(s, a, force, TY, LZ, nsplit);
  return true;
}

#ifdef PD_TRACE
long long *g_trace = nullptr;
void trace_dump(const char *name) {
  static int count[2] = {0, 0};
  if (++count[name[18] == 'r'] != 20) return;   // one warmed-up launch of each kind
  cudaDeviceSynchronize();
  std::vector<long long> h(64 * 16 * 8);
  cudaMemcpy(h.data(), g_trace, h.size() * 8, cudaMemcpyDeviceToHost);
  FILE *f = fopen(name, "w");
  for (int lv = 0; lv < 64; ++lv)
    for (int w = 0; w < 16; ++w) {
      const long long *t = &h[(lv * 16 + w) * 8];
      if (!t[0]) continue;
      fprintf(f, "%d %d %lld %lld %lld %lld %lld %lld\n", lv, w, t[0], t[1], t[2], t[3], t[4], t[5]);
    }
  fclose(f);
}
#endif

template <typename K>
int lat_launch(K kernel, pd_sim *s, const LatArgs &a, size_t smem) {
  const PdLattice &l = s->lat;
  const dim3 grid((unsigned)a.nxc, (unsigned)((l.PY + a.TY - 1) / a.TY), (unsigned)((l.PZ + a.LZ - 1) / a.LZ));
  const unsigned threads = (unsigned)((a.TY / 4) * a.nsplit * 32);
  PD_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
#ifdef PD_TRACE
  if (!g_trace) { cudaMalloc(&g_trace, 64 * 16 * 8 * 8); }
  cudaMemsetAsync(g_trace, 0, 64 * 16 * 8 * 8, s->stream);
  LatArgs a2 = a;
  a2.trace = g_trace;
  kernel<<<grid, threads, smem, s->stream>>>(a2);
  trace_dump(a.nbw == a.nbr ? "gpurun_out/trace_dil.txt" : "gpurun_out/trace_frc.txt");
#else
  kernel<<<grid, threads, smem, s->stream>>>(a);
#endif
  return PD_OK;
}

constexpr int MT_DIL = 384, MT_FRC = 256;

// launch arguments are prepared once per kernel kind and cached on the host (PdLattice::cache)
struct LatPrepared {
  LatArgs a;
  size_t smem = 0;
  bool ok = false;
};

LatPrepared *lat_prepare(pd_sim *s, bool force) {
  PdLattice &l = s->lat;
  if (l.cache[force]) return (LatPrepared *)l.cache[force];
  LatPrepared *pp = new LatPrepared();
  l.cache[force] = pp;
  int TY, LZ, nsplit;
  pp->ok = lat_pick(s, pp->a, force, force ? MT_FRC : MT_DIL, TY, LZ, nsplit, pp->smem);
  if (!pp->ok) return pp;
  pp->a.thr = nullptr;
  if (!force) {   // break-test filter thresholds (pd_bond.cuh, DilPolicy FILT): high word of s_c * min ||xi||^2, a shade low
    std::vector<int32_t> h((size_t)PD_LAT_MAXCOL * 8, 0);
    const int ncol = pp->a.cbeg[MAXSPLIT];
    for (int c = 0; c < ncol; ++c)
      for (int t = 0; t < pp->a.cols[c].n; ++t) {
        const double lb = l.r2lb[pp->a.cols[c].word * 32 + pp->a.cols[c].bit0 + t];
        const double thr = s->s_c * lb * (1.0 - 1.0 / 1099511627776.0);
        long long bits;
        memcpy(&bits, &thr, 8);
        h[(size_t)c * 8 + t] = (int32_t)(bits >> 32);
      }
    if (!l.thr_dev) l.thr_dev = (int32_t *)pdi::dev_alloc(s, sizeof(int32_t) * h.size());
    if (!l.thr_dev) { pp->ok = false; return pp; }
    cudaMemcpyAsync(l.thr_dev, h.data(), sizeof(int32_t) * h.size(), cudaMemcpyHostToDevice, s->stream);
    cudaStreamSynchronize(s->stream);
    pp->a.thr = l.thr_dev;
  }
  return pp;
}

// ---- direct variant: arguments (cached next to the marching ones) and launch ----
struct DirPrepared {
  DirArgs a;
  size_t smem = 0;
  dim3 grid, block;
};

DirPrepared *dir_prepare(pd_sim *s, bool force) {
  PdLattice &l = s->lat;
  static_assert(sizeof(void *) == 8, "");
  void *&slot = l.cache[2 + (force ? 1 : 0)];
  if (slot) return (DirPrepared *)slot;
  DirPrepared *pp = new DirPrepared();
  slot = pp;
  DirArgs &a = pp->a;
  a.DX = l.DX; a.DY = l.DY; a.HX = l.HX; a.HY = l.HY; a.HZ = l.HZ; a.PZ = l.PZ;
  a.rows = env_int(force ? "PD_DIR_FRC_ROWS" : "PD_DIR_DIL_ROWS", s->dim == 2 ? 2 : 4);   // rows per lane
  if (a.rows != 2 && !(a.rows == 1 && s->dim == 2)) a.rows = 4;
  a.nxc = l.PX / 32; a.nyq = (l.PY + 8) / 4; a.nyq_used = l.PY / a.rows;
  a.ncol = l.ncol; a.nw = l.nw;
  a.cy = std::max(1, std::min(env_int(force ? "PD_DIR_FRC_CY" : "PD_DIR_DIL_CY", 2), 4));
  a.cz = s->dim == 3 ? std::max(1, std::min(env_int(force ? "PD_DIR_FRC_CZ" : "PD_DIR_DIL_CZ", 2), 4)) : 1;
  while (a.cy * a.cz > 4) { if (a.cz > 1) --a.cz; else --a.cy; }   // 128 threads per CTA
  a.npad = s->npad;
  for (int c = 0; c < l.ncol; ++c) {
    const PdLatCol &src = l.cols[c];
    a.cols[c].off = (src.dz * l.DY + src.dy0) * l.DX + src.dx;
    a.cols[c].n = src.n; a.cols[c].word = src.word; a.cols[c].bit0 = src.bit0; a.cols[c].pad = 0;
  }
  a.mask = l.mask; a.nofail = l.nofail; a.rgocc = l.rgocc; a.flags32 = l.flags32; a.minv = s->minv;
  for (int q = 0; q < 3; ++q) { a.v[q] = s->v[q]; a.bval[q] = s->bval[q]; }
  a.theta_out = nullptr;
  a.A = s->A; a.c1 = s->c1; a.G = s->G; a.s_c = s->s_c; a.vol_uniform = s->vol_uniform; a.rrho = 1.0 / s->rho; a.dt = s->dt;
  a.gramp = 1.0;
  a.thr = nullptr;
  if (!force) {   // break-test filter thresholds (pd_bond.cuh, DilPolicy FILT): high word of s_c * min ||xi||^2, a shade low
    std::vector<int32_t> h((size_t)PD_LAT_MAXCOL * 8, 0);
    for (int c = 0; c < l.ncol; ++c)
      for (int t = 0; t < l.cols[c].n; ++t) {
        const double thr = s->s_c * l.r2lb[l.cols[c].word * 32 + l.cols[c].bit0 + t] * (1.0 - 1.0 / 1099511627776.0);
        long long bits;
        memcpy(&bits, &thr, 8);
        h[(size_t)c * 8 + t] = (int32_t)(bits >> 32);
      }
    if (!l.thr_dir) l.thr_dir = (int32_t *)pdi::dev_alloc(s, sizeof(int32_t) * h.size());
    if (l.thr_dir) {
      cudaMemcpyAsync(l.thr_dir, h.data(), sizeof(int32_t) * h.size(), cudaMemcpyHostToDevice, s->stream);
      cudaStreamSynchronize(s->stream);
    }
    a.thr = l.thr_dir;
  }
  const int nwarp = a.cy * a.cz;
  pp->smem = (size_t)l.ncol * 8 + (force ? 0 : (size_t)l.ncol * 32) + (size_t)nwarp * 512 * a.rows;
  pp->block = dim3((unsigned)(nwarp * 32));
  pp->grid = dim3((unsigned)a.nxc, (unsigned)((a.nyq_used + a.cy - 1) / a.cy), (unsigned)((l.PZ + a.cz - 1) / a.cz));
  return pp;
}

int dir_launch(pd_sim *s, bool force, double *theta_out, bool frac) {
  DirPrepared *pp = dir_prepare(s, force);
  DirArgs &a = pp->a;
  a.nbr = s->nb[s->cur]; a.nbw = s->nb[force ? s->cur ^ 1 : s->cur];
  a.theta_out = theta_out;
  if (force) {
    a.gramp = 1.0;
    if (s->ramp_time > 0.0) a.gramp = std::min(1.0, ((double)s->step * s->dt) / s->ramp_time);
  } else if (frac && !a.thr) {
    pdi::set_error("device allocation failed");
    return PD_ERR_ALLOC;
  }
  static const int staged = env_int("PD_DIR_STAGED", 2);   // bit 0: dilatation, bit 1: force (phase-ordered step, pd_bond.cuh)
#define DIR_LAUNCH(DIM_, FORCE_, FRAC_, MINB_, ST_)                                                                        \
  do {                                                                                                                     \
    if (a.rows == 1 && DIM_ == 2) k_lat_direct<2, FORCE_, FRAC_, 128, 4, false, 1><<<pp->grid, pp->block, pp->smem, s->stream>>>(a); \
    else if (a.rows == 2) k_lat_direct<DIM_, FORCE_, FRAC_, 128, (FORCE_ ? 3 : 4), false, 2><<<pp->grid, pp->block, pp->smem, s->stream>>>(a); \
    else if (ST_) k_lat_direct<DIM_, FORCE_, FRAC_, 128, MINB_, true, 4><<<pp->grid, pp->block, pp->smem, s->stream>>>(a);  \
    else k_lat_direct<DIM_, FORCE_, FRAC_, 128, MINB_, false, 4><<<pp->grid, pp->block, pp->smem, s->stream>>>(a);          \
  } while (0)
  if (force) {
    if (s->dim == 2) DIR_LAUNCH(2, true, false, 2, staged & 2); else DIR_LAUNCH(3, true, false, 2, staged & 2);
  } else if (frac) {
    if (s->dim == 2) DIR_LAUNCH(2, false, true, 3, staged & 1); else DIR_LAUNCH(3, false, true, 3, staged & 1);
  } else {
    if (s->dim == 2) DIR_LAUNCH(2, false, false, 3, staged & 1); else DIR_LAUNCH(3, false, false, 3, staged & 1);
  }
#undef DIR_LAUNCH
  return PD_OK;
}

}  // namespace

namespace pdi {

void lat_free_cache(pd_sim *s) {
  for (int q = 2; q < 4; ++q) {
    delete (DirPrepared *)s->lat.cache[q];
    s->lat.cache[q] = nullptr;
  }
  for (int q = 0; q < 2; ++q) {
    delete (LatPrepared *)s->lat.cache[q];
    s->lat.cache[q] = nullptr;
  }
}

int lat_launch_dilatation(pd_sim *s, double *theta_out, bool do_break) {
  if (s->lat.kernel == 0) return dir_launch(s, false, theta_out, do_break && s->fracture);
  LatPrepared *pp = lat_prepare(s, false);
  if (!pp->ok) { set_error("lattice plane ring does not fit shared memory"); return PD_ERR_LIMIT; }
  LatArgs &a = pp->a;
  a.nbr = s->nb[s->cur]; a.nbw = s->nb[s->cur];
  a.theta_out = theta_out;
  const bool frac = do_break && s->fracture;
  if (s->dim == 2) return frac ? lat_launch(k_lat_march<2, false, true, MT_DIL>, s, a, pp->smem)
                               : lat_launch(k_lat_march<2, false, false, MT_DIL>, s, a, pp->smem);
  return frac ? lat_launch(k_lat_march<3, false, true, MT_DIL>, s, a, pp->smem)
              : lat_launch(k_lat_march<3, false, false, MT_DIL>, s, a, pp->smem);
}

int lat_launch_force_update(pd_sim *s) {
  if (s->lat.kernel == 0) return dir_launch(s, true, nullptr, false);
  LatPrepared *pp = lat_prepare(s, true);
  if (!pp->ok) { set_error("lattice plane ring does not fit shared memory"); return PD_ERR_LIMIT; }
  LatArgs &a = pp->a;
  a.nbr = s->nb[s->cur]; a.nbw = s->nb[s->cur ^ 1];
  a.gramp = 1.0;
  if (s->ramp_time > 0.0) a.gramp = std::min(1.0, ((double)s->step * s->dt) / s->ramp_time);
  if (s->dim == 2) return lat_launch(k_lat_march<2, true, false, MT_FRC>, s, a, pp->smem);
  return lat_launch(k_lat_march<3, true, false, MT_FRC>, s, a, pp->smem);
}

int lat_launch_damage(pd_sim *s) {
  cudaMemsetAsync(s->stats_dev, 0, 3 * sizeof(unsigned long long), s->stream);
  k_lat_damage<<<nblk(s->npad), TPB, 0, s->stream>>>(s->npad, s->lat.nw, s->vol_uniform, s->perm, s->lat.mask, s->rowlen,
                                                     s->fvol, s->phi, s->stats_dev);
  return PD_OK;
}

}  // namespace pdi
