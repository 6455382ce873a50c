// pd_lattice_step.cu -- step kernels of the dense lattice layout (pd_lattice.cu, PdLattice):
// SURVEY.md 8(a) rows a1-a5 for lattice bodies whose bond geometry differs from bond to bond (jittered
// lattices; uniform lattices take the constant-geometry kernels of pd_lattice_uniform.cu).  Same per-bond
// arithmetic as the sliced-ELL kernels (pd_bond.cuh, shared with pd_step.cu).
//
//     DIRECT kernels `k_lat_direct`.  One warp owns a ROW GROUP (32 lanes x R rows
//     adjacent in y, R = 4 in 3-D) at one level and walks all stencil COLUMNS (dx, dy0..dy0+n-1, dz)
//     with an R-record register window sliding along y: in step t row r pairs with record t + r, one
//     gathered record serves up to R bonds, the R bonds of a step are independent FP64 chains in one
//     basic block.  Records are read straight from the dense pair arrays by arithmetic addressing
//     (16-byte loads, 512 contiguous bytes per pair and warp, shared between warps through L1); there
//     is no shared-memory staging and no CTA barrier.  A column whose R n bonds are intact on all 32
//     lanes runs without a single mask test (FAST); otherwise the MASKED variant predicates the
//     accumulation and, in the dilatation pass, clears the bits of the bonds that break (Eq. 1.30).
//
#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>

#include "pd_bond.cuh"

namespace {

using pdb::FULL;
constexpr int TPB = 256;
inline unsigned nblk(int64_t n) { return (unsigned)((n + TPB - 1) / TPB); }

template <int DIM, bool FORCE, bool FRAC, int R, bool GEOM> struct PolicyOfR { using type = pdb::DilPolicy<DIM, FRAC, true, R, true, GEOM>; };
template <int DIM, bool FRAC, int R, bool GEOM> struct PolicyOfR<DIM, true, FRAC, R, GEOM> { using type = pdb::ForcePolicy<DIM, true, R, GEOM>; };

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

template <int DIM, bool FORCE, bool FRAC, int MAXT, int MINB, bool STAGED, int R, bool GEOM = false>
__global__ void __launch_bounds__(MAXT, MINB) k_lat_direct(const __grid_constant__ DirArgs a) {
  extern __shared__ __align__(16) unsigned char smraw[];
  constexpr int NPAIR = FORCE ? DIM + 1 : DIM;
  using P = typename PolicyOfR<DIM, FORCE, FRAC, R, GEOM>::type;
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
  if (s->geom) a.rows = 2;
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
    if (s->geom) /* geometric extension (variant): 2 rows per lane (dir_prepare), bond by bond */                          \
      k_lat_direct<DIM_, FORCE_, FRAC_, 128, 2, false, 2, true><<<pp->grid, pp->block, pp->smem, s->stream>>>(a);          \
    else if (a.rows == 1 && DIM_ == 2) k_lat_direct<2, FORCE_, FRAC_, 128, 4, false, 1><<<pp->grid, pp->block, pp->smem, s->stream>>>(a); \
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
  ulat_free_cache(s);
  for (int q = 2; q < 4; ++q) {
    delete (DirPrepared *)s->lat.cache[q];
    s->lat.cache[q] = nullptr;
  }
}

int lat_launch_dilatation(pd_sim *s, double *theta_out, bool do_break) {
  if (s->lat.uniform) return ulat_launch_dilatation(s, theta_out, do_break);
  return dir_launch(s, false, theta_out, do_break && s->fracture);
}

int lat_launch_force_update(pd_sim *s) {
  if (s->lat.uniform) return ulat_launch_force_update(s);
  return dir_launch(s, true, nullptr, false);
}

int lat_launch_damage(pd_sim *s) {
  cudaMemsetAsync(s->stats_dev, 0, 3 * sizeof(unsigned long long), s->stream);
  k_lat_damage<<<nblk(s->npad), TPB, 0, s->stream>>>(s->npad, s->lat.nw, s->vol_uniform, s->perm, s->lat.mask, s->rowlen,
                                                     s->fvol, s->phi, s->stats_dev);
  return PD_OK;
}

}  // namespace pdi