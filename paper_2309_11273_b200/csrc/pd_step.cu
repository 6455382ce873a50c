// pd_step.cu -- the per-step kernels.
//
// One warp per GROUP of the windowed sliced-ELL layout (pd_internal.cuh): lane l owns 4 nodes (the
// l-th nodes of 4 adjacent lattice rows) and walks the group's SEGMENTS.  A SHIFT segment of n
// steps covers n + 3 consecutive entries of one lattice column; in step t row r pairs with entry
// t + r, so the four bonds of a step are the SAME relative neighbour for the four rows: a window of
// 4 gathered neighbour records slides along the column in registers, one new record per step
// serves 4 bonds (register blocking of the gather), the four bonds of a step are independent
// FP64 chains in one basic block (ILP 4), and -- when every lane has all 4 n bonds of the
// segment intact, the normal case in the bulk -- there is not a single mask test or branch per
// bond (FAST path).  Segments with missing / broken bonds on some lane run the MASKED variant
// (predicated accumulation, steps that are empty for the whole warp skipped).
//
//   k_dilatation  (rows a1, a2, and a5's break test folded in):
//        for each intact bond  dot = xi . eta            [= xbar * e, sqrt-free]
//        FRAC: a bond with dot - s_c ||xi||^2 >= 0 (<=> e/xbar >= s_c, Eq. 1.17/1.30) breaks first.
//              The fast path only ANDs the sign words of these values; if any of them is
//              non-negative on any lane the segment is redone by the masked variant, which
//              clears the bits.
//        theta_i = (A/m_i) sum_j rho_ij dot V_j           (Eq. 1.6 / 2.3)
//        writes the pair { G/m_i, cth_i = (K - G/3) theta_i / m_i }
//   k_force_update (rows a1, a3, a4):
//        f_i = sum_j rho_ij V_j [ cth_i + cth_j + (G/m_i + G/m_j) dot/||xi||^2 ] xi   (Eq. 2.2 / 2.1)
//        then Eq. 2.11 + boundary dofs, {x, u^{n+1}} into the other neighbour-record buffer
//   k_damage (row a5): phi_i (Eq. 1.31) + device-side reduction of the three damage scalars
//
// The break test of step n (on u^{n+1}) runs at the start of step n+1's dilatation pass, which
// needs the same xi . eta; pd_api.cu flushes it before any state is read back.  Both ends of a
// bond take the identical decision because -a*-b == a*b exactly in every product and the sums
// run in the same component order; fast and masked variants use the same arithmetic.
#include "pd_bond.cuh"

namespace {

using pdb::Ent;

constexpr int TPB = 32 * PD_GROUPS_PER_CTA;
using pdb::FULL;
constexpr int NCQ = PD_MAXSTEP + 3;   // entries of the longest segment

struct StepArgs {
  int64_t ngroups;
  const double2 *nbr;   // neighbour records holding u^n (and, for the force pass, cth^n)
  double2 *nbw;         // dilatation: the same buffer (pair AUX is written); force: the other buffer
  const uint32_t *goff, *soff, *col;
  uint32_t *seg;
  const uint32_t *member, *nofail;
  const double *vol, *minv, *fvol;
  double *v[3];
  const double *bval[3];
  double *theta_out;
  double *phi;
  const uint8_t *flags;
  const int32_t *rowlen;
  const int32_t *perm;
  unsigned long long *stats;
  double A, c1, G, s_c, vol_uniform, rho, dt, ramp_time;
  int64_t step;
};

template <int DIM, bool AUX, bool VOL>
__device__ __forceinline__ void load_ent(Ent<DIM, AUX, VOL> &E, const StepArgs &a, uint32_t c) {
  const double2 *q = a.nbr + c;
#pragma unroll
  for (int k = 0; k < DIM; ++k) E.p[k] = __ldg(q + 32 * k);
  if (AUX) E.g = __ldg(q + 32 * PD_P_AUX);
  if (VOL) E.vj = __ldg(a.vol + (((c >> 7) << 5) | (c & 31)));
}

// ---------------------------------------------------------------------------------------------
// predicated 16-byte read-only load: no branch, so the four bonds of a step stay in one basic block
__device__ __forceinline__ void ldg_if(double2 &v, const double2 *ptr, uint32_t pred) {
  asm("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %3, 0;\n\t@p ld.global.nc.v2.f64 {%0, %1}, [%2];\n\t}"
      : "+d"(v.x), "+d"(v.y) : "l"(ptr), "r"(pred));
}
template <int DIM, bool AUX, bool VOL>
__device__ __forceinline__ void load_ent_if(Ent<DIM, AUX, VOL> &E, const StepArgs &a, uint32_t c, uint32_t pred) {
  const double2 *q = a.nbr + c;
#pragma unroll
  for (int k = 0; k < DIM; ++k) ldg_if(E.p[k], q + 32 * k, pred);
  if (AUX) ldg_if(E.g, q + 32 * PD_P_AUX, pred);
  if (VOL) { if (pred) E.vj = __ldg(a.vol + (((c >> 7) << 5) | (c & 31))); }
}

// one SHIFT segment: n steps over the entries cc[0 .. n+2].  The window S[4] lives across segments:
// in step t row r uses S[(t + r) % 4]; the slot of row 0 is refilled with entry t + 4 as soon as
// row 0 is done.  In the LAST step every slot dies as its row finishes and is refilled with one of
// the first four entries of the NEXT segment (cq[0..3], slot j <- cq[j]), so the next segment
// finds its window already in flight (`preloaded`).
template <bool MASKED, class P>
__device__ __forceinline__ void run_shift(P &p, const StepArgs &a, int n, uint32_t mask, uint32_t nf, uint32_t &clr,
                                          const uint32_t (&cc)[NCQ], const uint32_t (&cq)[NCQ], typename P::E (&S)[4],
                                          bool preloaded) {
  if (!preloaded) {
#pragma unroll
    for (int q = 0; q < 4; ++q) load_ent(S[q], a, cc[q]);
  }
  uint32_t anyw = 0;
  if (MASKED) anyw = __reduce_or_sync(FULL, mask);
  auto bond = [&](int r, const typename P::E &e, int bit) {
    if (p.template bond<MASKED>(r, e, (mask >> bit) & 1u, (nf >> bit) & 1u)) clr |= 1u << bit;
  };
#pragma unroll
  for (int t = 0; t < PD_MAXSTEP; ++t) {
    if (t < n) {
      const uint32_t last = (t + 1 == n) ? 1u : 0u;                    // warp-uniform
      const bool live = !MASKED || ((anyw >> (4 * t)) & 15u) != 0;   // warp-uniform
      if (live) bond(0, S[t % 4], 4 * t + 0);
      load_ent(S[t % 4], a, last ? cq[t % 4] : cc[(t + 4) % NCQ]);
      if (live) bond(1, S[(t + 1) % 4], 4 * t + 1);
      load_ent_if(S[(t + 1) % 4], a, cq[(t + 1) % 4], last);
      if (live) bond(2, S[(t + 2) % 4], 4 * t + 2);
      load_ent_if(S[(t + 2) % 4], a, cq[(t + 2) % 4], last);
      if (live) bond(3, S[(t + 3) % 4], 4 * t + 3);
      load_ent_if(S[(t + 3) % 4], a, cq[(t + 3) % 4], last);
    }
  }
}

constexpr int PF_AHEAD = 24;   // entries
constexpr int PF_SEG = 4;      // segments
__device__ __forceinline__ void prefetch_l2(const void *p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// walks all segments of the warp's group
template <class P>
__device__ __forceinline__ void walk_group(P &p, const StepArgs &a, int64_t grp, int lane) {
  const uint32_t s0 = a.soff[grp], nseg = a.soff[grp + 1] - s0;
  const uint32_t *colp = a.col + (int64_t)a.goff[grp] * 32 + lane;
  const int64_t wbase = (int64_t)s0 * 32 + lane;
  // the segment word and the NCQ neighbour indices of the NEXT segment are loaded while the current
  // one is processed (the index stream comes from HBM; the node data from L1/L2)
  uint32_t wn = 0, cq[NCQ];
  prefetch_l2(colp + (int64_t)(NCQ + lane) * 32 - lane);
  if (lane < PF_SEG) prefetch_l2(a.seg + wbase - lane + (int64_t)lane * 32);
  if (nseg) wn = a.seg[wbase];
#pragma unroll
  for (int q = 0; q < NCQ; ++q) cq[q] = colp[q * 32];
  uint32_t e = 0;
  typename P::E S[4];
  bool pre = false;   // S already holds (in flight) the first four entries of the segment about to start
  for (uint32_t s = 0; s < nseg; ++s) {
    const uint32_t w = wn;
    uint32_t cc[NCQ];
#pragma unroll
    for (int q = 0; q < NCQ; ++q) cc[q] = cq[q];
    const uint32_t code = w >> 28;
    const uint32_t nent = code == 0 ? 0u : (code < 8 ? code + 3 : code - 8);
    const uint32_t en = e + nent;
    if (s + 1 < nseg) wn = a.seg[wbase + (int64_t)(s + 1) * 32];
    // the index and mask streams are read once, line by line, straight from HBM: pull the lines of the
    // entries PF_AHEAD .. PF_AHEAD + nent - 1 past the next segment (one line per lane) and of the
    // segment word PF_SEG ahead into L2, so the loads above find them there
    if ((uint32_t)lane < nent) prefetch_l2(colp + (int64_t)(en + PF_AHEAD + lane) * 32 - lane);
    if (lane == 0 && s + PF_SEG < nseg) prefetch_l2(a.seg + wbase + (int64_t)(s + PF_SEG) * 32);
#pragma unroll
    for (int q = 0; q < NCQ; ++q) cq[q] = colp[(int64_t)(en + q) * 32];   // col has PD_COL_SLACK readable entries past its end
    const uint32_t mask = w & 0x0fffffffu;
    if (code >= 1 && code < 8) {
      const int n = (int)code;
      const uint32_t fullmask = (1u << (4 * n)) - 1u;
      bool slow = !__all_sync(FULL, mask == fullmask);
      uint32_t clr = 0;
      if (!slow) {
        p.fast_begin();
        run_shift<false>(p, a, n, mask, 0u, clr, cc, cq, S, pre);
        slow = p.fast_failed();
        pre = false;   // (only matters if the segment is redone: the window now holds the next segment's entries)
      }
      if (slow) {
        const uint32_t nf = (P::kFrac && a.nofail) ? a.nofail[wbase + (int64_t)s * 32] : 0u;
        run_shift<true>(p, a, n, mask, nf, clr, cc, cq, S, pre);
        if (clr) a.seg[wbase + (int64_t)s * 32] = w & ~clr;
      }
      pre = true;
    } else if (code > 8) {
      pre = false;
      const int n = (int)code - 8;
      const uint32_t nf = (P::kFrac && a.nofail) ? a.nofail[wbase + (int64_t)s * 32] : 0u;
      uint32_t clr = 0;
#pragma unroll 1
      for (int t = 0; t < n; ++t) {
        typename P::E S1;
        load_ent(S1, a, colp[(int64_t)(e + t) * 32]);
#pragma unroll
        for (int r = 0; r < PD_R; ++r) {
          const int bit = 4 * t + r;
          if (p.template bond<true>(r, S1, (mask >> bit) & 1u, (nf >> bit) & 1u)) clr |= 1u << bit;
        }
      }
      if (clr) a.seg[wbase + (int64_t)s * 32] = w & ~clr;
    }
    e = en;
  }
}

// ---------------------------------------------------------------------------------------------
template <int DIM, bool FRAC, bool UNIV, bool GEOM>
__global__ void __launch_bounds__(TPB, 3) k_dilatation(StepArgs a) {
  const int lane = threadIdx.x & 31;
  const int64_t grp = ((int64_t)blockIdx.x * TPB + threadIdx.x) >> 5;
  if (grp >= a.ngroups) return;
  const uint32_t e0 = pd_elem(grp * PD_R * 32 + lane);
  pdb::DilPolicy<DIM, FRAC, UNIV, PD_R, false, GEOM> p;
  p.s_c = a.s_c;
#pragma unroll
  for (int r = 0; r < PD_R; ++r) {
    p.acc[r] = 0.0;
#pragma unroll
    for (int k = 0; k < DIM; ++k) {
      const double2 xu = a.nbr[e0 + r * 32 * PD_NP + 32 * k];
      p.xo[r][k] = xu.x;
      p.uo[r][k] = xu.y;
    }
  }
  walk_group(p, a, grp, lane);
#pragma unroll
  for (int r = 0; r < PD_R; ++r) {
    const int64_t i = (grp * PD_R + r) * 32 + lane;
    double s = p.acc[r];
    if (UNIV) s *= a.vol_uniform;
    const double mi = a.minv[i];   // 0 for phantoms
    const double theta = a.A * mi * s;
    a.nbw[e0 + r * 32 * PD_NP + 32 * PD_P_AUX] = make_double2(a.G * mi, a.c1 * theta * mi);
    if (a.theta_out) a.theta_out[i] = theta;
  }
}

// ---------------------------------------------------------------------------------------------
template <int DIM, bool UNIV, bool GEOM>
__global__ void __launch_bounds__(TPB, 2) k_force_update(StepArgs a) {
  const int lane = threadIdx.x & 31;
  const int64_t grp = ((int64_t)blockIdx.x * TPB + threadIdx.x) >> 5;
  if (grp >= a.ngroups) return;
  const uint32_t e0 = pd_elem(grp * PD_R * 32 + lane);
  pdb::ForcePolicy<DIM, UNIV, PD_R, GEOM> p;
#pragma unroll
  for (int r = 0; r < PD_R; ++r) {
    const uint32_t e = e0 + r * 32 * PD_NP;
#pragma unroll
    for (int k = 0; k < DIM; ++k) {
      const double2 xu = a.nbr[e + 32 * k];
      p.xo[r][k] = xu.x;
      p.uo[r][k] = xu.y;
      p.f[r][k] = 0.0;
    }
    const double2 g = a.nbr[e + 32 * PD_P_AUX];
    p.gmu_i[r] = g.x;
    p.cth_i[r] = g.y;
  }
  walk_group(p, a, grp, lane);
  // ---- Eq. 2.11 + boundary dofs (App. B) ----
  double g = 1.0;
  if (a.ramp_time > 0.0) g = fmin(1.0, __ddiv_rn(__dmul_rn((double)a.step, a.dt), a.ramp_time));
#pragma unroll
  for (int r = 0; r < PD_R; ++r) {
    const int64_t i = (grp * PD_R + r) * 32 + lane;
    if (a.perm[i] < 0) continue;   // phantom
    const uint32_t e = e0 + r * 32 * PD_NP;
    const unsigned fl = a.flags[i];
#pragma unroll
    for (int k = 0; k < DIM; ++k) {
      double fk = p.f[r][k];
      if (UNIV) fk *= a.vol_uniform;
      double vk = a.v[k][i];
      double uk = p.uo[r][k];
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
      a.nbw[e + 32 * k] = make_double2(p.xo[r][k], uk);
    }
  }
}

// ---------------------------------------------------------------------------------------------
// phi_i = 1 - sum_j rho_ij V_j / sum_j V_j (Eq. 1.31) and the three damage scalars.
__global__ void __launch_bounds__(TPB) k_damage(StepArgs a, bool univ) {
  const int lane = threadIdx.x & 31;
  const int64_t grp = ((int64_t)blockIdx.x * TPB + threadIdx.x) >> 5;
  unsigned long long broken = 0, ge_half = 0;
  double phimax = 0.0;
  if (grp < a.ngroups) {
    const uint32_t s0 = a.soff[grp];
    const int nseg = (int)(a.soff[grp + 1] - s0);
    const uint32_t *sg = a.seg + (int64_t)s0 * 32 + lane;
    const uint32_t *mb = a.member + (int64_t)s0 * 32 + lane;
    const uint32_t *col = a.col + (int64_t)a.goff[grp] * 32 + lane;
    double sum[PD_R];
    int cnt[PD_R];
#pragma unroll
    for (int r = 0; r < PD_R; ++r) { sum[r] = 0.0; cnt[r] = 0; }
    if (univ) {
      for (int s = 0; s < nseg; ++s) {
        const uint32_t w = sg[(int64_t)s * 32] & 0x0fffffffu;
#pragma unroll
        for (int r = 0; r < PD_R; ++r) cnt[r] += __popc(w & (0x01111111u << r));
      }
#pragma unroll
      for (int r = 0; r < PD_R; ++r)   // the sum of cnt equal volumes, added one by one like sum_j V_j was (pd_build.cu)
        for (int q = 0; q < cnt[r]; ++q) sum[r] += a.vol_uniform;
    } else {
      pd_for_lane_slots(mb, nseg, [&](int s, int bit, int r, int k) {
        if (!((sg[(int64_t)s * 32] >> bit) & 1u)) return;
        const uint32_t c = col[(int64_t)k * 32];
        const double vj = a.vol[((c >> 7) << 5) | (c & 31)];
#pragma unroll
        for (int q = 0; q < PD_R; ++q)
          if (q == r) { sum[q] += vj; ++cnt[q]; }
      });
    }
#pragma unroll
    for (int r = 0; r < PD_R; ++r) {
      const int64_t i = (grp * PD_R + r) * 32 + lane;
      if (a.perm[i] < 0) continue;
      const double phi = 1.0 - sum[r] / a.fvol[i];
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
  a.nbr = s->nb[s->cur]; a.nbw = s->nb[s->cur];
  a.goff = s->goff; a.soff = s->soff; a.col = s->col; a.seg = s->seg; a.member = s->member; a.nofail = s->nofail;
  a.vol = s->vol; a.minv = s->minv; a.fvol = s->fvol;
  for (int k = 0; k < 3; ++k) { a.v[k] = s->v[k]; a.bval[k] = s->bval[k]; }
  a.theta_out = nullptr; a.phi = s->phi; a.flags = s->flags; a.rowlen = s->rowlen; a.perm = s->perm;
  a.stats = s->stats_dev;
  a.A = s->A; a.c1 = s->c1; a.G = s->G; a.s_c = s->s_c; a.vol_uniform = s->vol_uniform; a.rho = s->rho; a.dt = s->dt;
  a.ramp_time = s->ramp_time; a.step = s->step;
  return a;
}

inline unsigned ngrid(const pd_sim *s) { return (unsigned)((s->ngroups + PD_GROUPS_PER_CTA - 1) / PD_GROUPS_PER_CTA); }

template <int DIM, bool GEOM>
void dil_dispatch(const StepArgs &a, bool frac, bool univ, unsigned grid, cudaStream_t st) {
  if (frac) { if (univ) k_dilatation<DIM, true, true, GEOM><<<grid, TPB, 0, st>>>(a); else k_dilatation<DIM, true, false, GEOM><<<grid, TPB, 0, st>>>(a); }
  else { if (univ) k_dilatation<DIM, false, true, GEOM><<<grid, TPB, 0, st>>>(a); else k_dilatation<DIM, false, false, GEOM><<<grid, TPB, 0, st>>>(a); }
}
template <int DIM, bool GEOM>
void force_dispatch(const StepArgs &a, bool univ, unsigned grid, cudaStream_t st) {
  if (univ) k_force_update<DIM, true, GEOM><<<grid, TPB, 0, st>>>(a); else k_force_update<DIM, false, GEOM><<<grid, TPB, 0, st>>>(a);
}

}  // namespace

namespace pdi {

int launch_dilatation(pd_sim *s, double *theta_out, bool do_break) {
  if (s->lat.on) return lat_launch_dilatation(s, theta_out, do_break);
  StepArgs a = make_args(s);
  a.theta_out = theta_out;
  const bool frac = do_break && s->fracture;
  if (s->geom) {
    if (s->dim == 2) dil_dispatch<2, true>(a, frac, s->uniform_v, ngrid(s), s->stream);
    else dil_dispatch<3, true>(a, frac, s->uniform_v, ngrid(s), s->stream);
  } else {
    if (s->dim == 2) dil_dispatch<2, false>(a, frac, s->uniform_v, ngrid(s), s->stream);
    else dil_dispatch<3, false>(a, frac, s->uniform_v, ngrid(s), s->stream);
  }
  return PD_OK;
}

int launch_force_update(pd_sim *s) {
  if (s->lat.on) return lat_launch_force_update(s);
  StepArgs a = make_args(s);
  a.nbw = s->nb[s->cur ^ 1];
  if (s->geom) {
    if (s->dim == 2) force_dispatch<2, true>(a, s->uniform_v, ngrid(s), s->stream);
    else force_dispatch<3, true>(a, s->uniform_v, ngrid(s), s->stream);
  } else {
    if (s->dim == 2) force_dispatch<2, false>(a, s->uniform_v, ngrid(s), s->stream);
    else force_dispatch<3, false>(a, s->uniform_v, ngrid(s), s->stream);
  }
  return PD_OK;
}

int launch_damage(pd_sim *s) {
  if (s->lat.on) return lat_launch_damage(s);
  StepArgs a = make_args(s);
  cudaMemsetAsync(s->stats_dev, 0, 3 * sizeof(unsigned long long), s->stream);
  k_damage<<<ngrid(s), TPB, 0, s->stream>>>(a, s->uniform_v);
  return PD_OK;
}

}  // namespace pdi
