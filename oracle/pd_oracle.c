/*
 * pd_oracle.c -- CPU ORACLE for the explicit linearized OSB-PD time step.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares
 * no code, header, table or helper with the CUDA path (paper_2309_11273_b200/csrc) and
 * neither includes the other.
 *
 * What it is: the method of Ni, Zaccariotto, Zhu, Galvanetto, "Matrix-based implementation
 * and GPU acceleration of linearized ordinary state-based peridynamic models in MATLAB"
 * (arXiv 2309.11273), written out step by step in the paper's own order and notation, in
 * FP64, gather form of Eq. 2.1, user node order, with sqrt and unit
 * vectors M exactly as printed (no sqrt-free rearrangement, no blocking, no fusion).
 * Citations are PAPER.md line numbers + equation numbers.  Where the paper is silent the
 * reading is the one listed in DESIGN.md ("Readings", ids C-1 .. C-21 from SURVEY.md 8(c)).
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): 1058 bonds of PAPER.md:623, closed-form
 * dilatation theta = A*eps, rigid-body zero force, momentum balance, hand-computed 2- and
 * 3-node forces, classical strain energies, the exact discrete invariant of Eq. 2.11, the
 * constant-force closed form, failure/damage special cases.  Full trajectories of the five
 * synthetic configs are "parity unpinned" by the paper itself (it prints no values); they are
 * pinned only through those properties and a second, independent pair-scatter formulation
 * (oracle/pd_appc.py, App. C of the paper with its typos fixed).
 *
 * Layout conventions (all plain C arrays, caller-owned):
 *   coords, u, v, f, bval : AoS, dim doubles per node (x0,y0[,z0],x1,...), user node order
 *   rowptr[n+1], col[Z]   : CSR of DIRECTED bonds, rows sorted by ascending j
 *   rho[Z]                : uint8 bond status (1 intact, 0 broken), Eq. 1.30
 * OpenMP is used only as "parallel for" over nodes i; every node's sum runs sequentially in
 * ascending-j order, so results do not depend on the thread count.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define PDO_MODE_3D 0
#define PDO_MODE_PLANE_STRESS 1
#define PDO_MODE_PLANE_STRAIN 2

/* flag bits of the boundary description (same meaning as include/pd.h, restated here
 * because the two sides share no header) */
#define PDO_CLAMP(k) (1u << (k))        /* bits 0-2: clamp dof k                        */
#define PDO_PRESC(k) (1u << (3 + (k)))  /* bits 3-5: prescribed-velocity dof k          */
#define PDO_BODYF (1u << 6)             /* bit 6   : body-force node                    */
#define PDO_NOFAIL (1u << 7)            /* bit 7   : bonds touching the node never break */

int pdo_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* ------------------------------------------------------------------------------------------
 * Constants A, K, G by mode.  kappa = E/(3(1-2nu)), mu = E/(2(1+nu)).
 * A: Eq. 1.8; K: Eq. 1.15; G: Eq. 1.16.
 * Returns 0, or -1 on inadmissible input.
 * ---------------------------------------------------------------------------------------- */
int pdo_constants(int mode, double E, double nu, double *A, double *K, double *G,
                  double *kappa, double *mu) {
  if (!(E > 0.0) || !(nu > -1.0) || !(nu < 0.5)) return -1;
  double ka = E / (3.0 * (1.0 - 2.0 * nu));
  double m_ = E / (2.0 * (1.0 + nu));
  *kappa = ka;
  *mu = m_;
  if (mode == PDO_MODE_3D) {
    *A = 3.0;
    *K = 3.0 * ka;
    *G = 15.0 * m_;
  } else if (mode == PDO_MODE_PLANE_STRESS) {
    *A = 2.0 * (1.0 - 2.0 * nu) / (1.0 - nu);
    *K = 2.0 * ka * (1.0 - 2.0 * nu) / (1.0 - nu) -
         (2.0 / 3.0) * m_ * ((1.0 + nu) * (1.0 - 3.0 * nu)) / ((1.0 - nu) * (1.0 - 2.0 * nu));
    *G = 8.0 * m_;
  } else if (mode == PDO_MODE_PLANE_STRAIN) {
    *A = 2.0;
    *K = 2.0 * ka - (2.0 / 3.0) * m_;
    *G = 8.0 * m_;
  } else {
    return -1;
  }
  return 0;
}

/* squared reference bond length ||xi_ij||^2, xi = x_j - x_i (Eq. 1.3);
 * products and sums in this fixed order (the build uses -ffp-contract=off), so the
 * inclusive horizon test below is reproducible. */
static double dist2(int dim, const double *xi, const double *xj) {
  double s = 0.0;
  for (int k = 0; k < dim; ++k) {
    double d = xj[k] - xi[k];
    s = s + d * d;
  }
  return s;
}

/* ------------------------------------------------------------------------------------------
 * Family H_i = { j != i : ||x_j - x_i|| <= delta }, inclusive (reading
 * C-11), tested on squared distances.  Brute force O(N^2): the definition written out.
 * count: fills rowptr[n+1], returns Z.   fill: fills col[Z] ascending in j.
 * ---------------------------------------------------------------------------------------- */
int64_t pdo_family_count_brute(int64_t n, int dim, const double *coords, double horizon,
                               int64_t *rowptr) {
  double h2 = horizon * horizon;
  rowptr[0] = 0;
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t i = 0; i < n; ++i) {
    int64_t c = 0;
    for (int64_t j = 0; j < n; ++j)
      if (j != i && dist2(dim, coords + dim * i, coords + dim * j) <= h2) ++c;
    rowptr[i + 1] = c;
  }
  for (int64_t i = 0; i < n; ++i) rowptr[i + 1] += rowptr[i];
  return rowptr[n];
}

void pdo_family_fill_brute(int64_t n, int dim, const double *coords, double horizon,
                           const int64_t *rowptr, int32_t *col) {
  double h2 = horizon * horizon;
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t i = 0; i < n; ++i) {
    int64_t p = rowptr[i];
    for (int64_t j = 0; j < n; ++j)
      if (j != i && dist2(dim, coords + dim * i, coords + dim * j) <= h2) col[p++] = (int32_t)j;
  }
}

/* Same family, found through a simple uniform cell list (cell edge = horizon, 3^dim cells
 * searched).  Must agree with the brute-force version entry for entry (tests pin this);
 * it exists only so that the oracle can build 10^5..10^6-node families in reasonable time.
 * Uses the identical distance test.  Returns Z, or -1 on allocation failure. */
typedef struct {
  double lo[3];
  int64_t nc[3];
  double inv;
  int64_t *start; /* ncell+1 */
  int32_t *items; /* n, node ids grouped by cell, ascending id inside a cell */
} pdo_cells;

static int64_t cell_of(const pdo_cells *c, int dim, const double *x, int64_t *idx) {
  int64_t id = 0, stride = 1;
  for (int k = 0; k < dim; ++k) {
    int64_t q = (int64_t)floor((x[k] - c->lo[k]) * c->inv);
    if (q < 0) q = 0;
    if (q >= c->nc[k]) q = c->nc[k] - 1;
    idx[k] = q;
    id += q * stride;
    stride *= c->nc[k];
  }
  return id;
}

static int cells_build(pdo_cells *c, int64_t n, int dim, const double *coords, double horizon) {
  double hi[3] = {0, 0, 0};
  for (int k = 0; k < 3; ++k) { c->lo[k] = 0; c->nc[k] = 1; }
  for (int k = 0; k < dim; ++k) { c->lo[k] = coords[k]; hi[k] = coords[k]; }
  for (int64_t i = 0; i < n; ++i)
    for (int k = 0; k < dim; ++k) {
      double x = coords[dim * i + k];
      if (x < c->lo[k]) c->lo[k] = x;
      if (x > hi[k]) hi[k] = x;
    }
  c->inv = 1.0 / horizon;
  int64_t ncell = 1;
  for (int k = 0; k < dim; ++k) {
    c->nc[k] = (int64_t)floor((hi[k] - c->lo[k]) * c->inv) + 1;
    ncell *= c->nc[k];
  }
  c->start = (int64_t *)calloc((size_t)ncell + 1, sizeof(int64_t));
  c->items = (int32_t *)malloc((size_t)n * sizeof(int32_t));
  if (!c->start || !c->items) return -1;
  int64_t idx[3];
  for (int64_t i = 0; i < n; ++i) c->start[cell_of(c, dim, coords + dim * i, idx) + 1]++;
  for (int64_t q = 0; q < ncell; ++q) c->start[q + 1] += c->start[q];
  int64_t *fill = (int64_t *)malloc((size_t)ncell * sizeof(int64_t));
  if (!fill) return -1;
  memcpy(fill, c->start, (size_t)ncell * sizeof(int64_t));
  for (int64_t i = 0; i < n; ++i) c->items[fill[cell_of(c, dim, coords + dim * i, idx)]++] = (int32_t)i;
  free(fill);
  return 0;
}

static int cmp_i32(const void *a, const void *b) {
  int32_t x = *(const int32_t *)a, y = *(const int32_t *)b;
  return (x > y) - (x < y);
}

/* visits the 3^dim cells around node i; if col==NULL only counts */
static int64_t cells_row(const pdo_cells *c, int dim, const double *coords, double h2, int64_t i,
                         int32_t *out) {
  int64_t idx[3] = {0, 0, 0};
  cell_of(c, dim, coords + dim * i, idx);
  int64_t cnt = 0;
  int64_t z0 = dim > 2 ? idx[2] - 1 : 0, z1 = dim > 2 ? idx[2] + 1 : 0;
  for (int64_t cz = z0; cz <= z1; ++cz) {
    if (cz < 0 || cz >= c->nc[2]) continue;
    for (int64_t cy = idx[1] - 1; cy <= idx[1] + 1; ++cy) {
      if (cy < 0 || cy >= c->nc[1]) continue;
      for (int64_t cx = idx[0] - 1; cx <= idx[0] + 1; ++cx) {
        if (cx < 0 || cx >= c->nc[0]) continue;
        int64_t q = cx + c->nc[0] * (cy + c->nc[1] * cz);
        for (int64_t p = c->start[q]; p < c->start[q + 1]; ++p) {
          int64_t j = c->items[p];
          if (j != i && dist2(dim, coords + dim * i, coords + dim * j) <= h2) {
            if (out) out[cnt] = (int32_t)j;
            ++cnt;
          }
        }
      }
    }
  }
  if (out) qsort(out, (size_t)cnt, sizeof(int32_t), cmp_i32);
  return cnt;
}

int64_t pdo_family_cells(int64_t n, int dim, const double *coords, double horizon,
                         int64_t *rowptr, int32_t *col /* NULL: count only */) {
  pdo_cells c;
  if (cells_build(&c, n, dim, coords, horizon) != 0) return -1;
  double h2 = horizon * horizon;
  if (!col) {
    rowptr[0] = 0;
#pragma omp parallel for schedule(dynamic, 256)
    for (int64_t i = 0; i < n; ++i) rowptr[i + 1] = cells_row(&c, dim, coords, h2, i, NULL);
    for (int64_t i = 0; i < n; ++i) rowptr[i + 1] += rowptr[i];
  } else {
#pragma omp parallel for schedule(dynamic, 256)
    for (int64_t i = 0; i < n; ++i) cells_row(&c, dim, coords, h2, i, col + rowptr[i]);
  }
  free(c.start);
  free(c.items);
  return rowptr[n];
}

/* position of directed bond (i -> j) in the CSR, or -1 */
int64_t pdo_find_bond(const int64_t *rowptr, const int32_t *col, int64_t i, int64_t j) {
  int64_t lo = rowptr[i], hi = rowptr[i + 1] - 1;
  while (lo <= hi) {
    int64_t mid = (lo + hi) / 2;
    if (col[mid] == j) return mid;
    if (col[mid] < j) lo = mid + 1; else hi = mid - 1;
  }
  return -1;
}

/* ------------------------------------------------------------------------------------------
 * Weighted volume m_i = sum_{j in H_i} w xbar_ij^2 V_j with w = 1 (Eq. 1.9, PAPER.md:206-210;
 * w = 1 per PAPER.md:385), over the FULL geometric family, never updated (reading C-10), and
 * the family volume vol_i = sum_j V_j, the denominator of Eq. 1.31.
 * ---------------------------------------------------------------------------------------- */
void pdo_weighted_volume(int64_t n, int dim, const double *coords, const double *V,
                         const int64_t *rowptr, const int32_t *col, double *m, double *fvol) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    double mi = 0.0, vi = 0.0;
    for (int64_t p = rowptr[i]; p < rowptr[i + 1]; ++p) {
      int64_t j = col[p];
      double xbar = sqrt(dist2(dim, coords + dim * i, coords + dim * j)); /* Eq. 1.5 */
      mi += xbar * xbar * V[j];
      vi += V[j];
    }
    m[i] = mi;
    fvol[i] = vi;
  }
}

/* ------------------------------------------------------------------------------------------
 * Step 6: linearized extension of every directed bond,
 *   e_ij = rho_ij * M_ij . (u_j - u_i),  M_ij = xi_ij / ||xi_ij||   (Eq. 2.4 /
 *   Eq. 2.7; broken bonds give 0).
 * Also returns xbar_ij = ||xi_ij|| per bond if xbar != NULL.
 * ---------------------------------------------------------------------------------------- */
void pdo_extension(int64_t n, int dim, const double *coords, const int64_t *rowptr,
                   const int32_t *col, const uint8_t *rho, const double *u, double *e,
                   double *xbar_out) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    for (int64_t p = rowptr[i]; p < rowptr[i + 1]; ++p) {
      int64_t j = col[p];
      double xi[3] = {0, 0, 0}, M[3] = {0, 0, 0};
      for (int k = 0; k < dim; ++k) xi[k] = coords[dim * j + k] - coords[dim * i + k];
      double xbar = sqrt(dist2(dim, coords + dim * i, coords + dim * j));
      for (int k = 0; k < dim; ++k) M[k] = xi[k] / xbar;
      double ext = 0.0;
      for (int k = 0; k < dim; ++k) ext += M[k] * (u[dim * j + k] - u[dim * i + k]);
      e[p] = rho[p] ? ext : 0.0;
      if (xbar_out) xbar_out[p] = xbar;
    }
  }
}

/* ------------------------------------------------------------------------------------------
 * Step 7: dilatation theta_i = (A/m_i) sum_j w xbar_ij e_ij V_j (Eq. 1.6, PAPER.md:179-182;
 * discrete form Eq. 2.3).  e already carries rho.
 * ---------------------------------------------------------------------------------------- */
void pdo_dilatation(int64_t n, const double *V, const int64_t *rowptr, const int32_t *col,
                    const double *e, const double *xbar, double A, const double *m,
                    double *theta) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    double s = 0.0;
    for (int64_t p = rowptr[i]; p < rowptr[i + 1]; ++p) s += xbar[p] * e[p] * V[col[p]];
    theta[i] = (A / m[i]) * s;
  }
}

/* ------------------------------------------------------------------------------------------
 * Step 8: internal force DENSITY at node i (Eq. 2.1 gather form):
 *   f_i = sum_j rho_ij [ (K - G/3) (theta_i/m_i + theta_j/m_j) xbar_ij
 *                        + G e_ij (1/m_i + 1/m_j) ] M_ij V_j
 * which is Eq. 2.2 divided by V_i, i.e. (t_i<xi> + t_j<-xi>) M_ij V_j with
 * the force scalar state t of Eq. 1.14.  The division of theta by m a
 * second time is what Eq. 2.2 prints (reading C-12).  Sign: enters the equation of motion
 * with "+" (reading C-2; "RF=EXF+PDF").
 * ---------------------------------------------------------------------------------------- */
void pdo_force_density(int64_t n, int dim, const double *coords, const double *V,
                       const int64_t *rowptr, const int32_t *col, const uint8_t *rho,
                       const double *e, const double *xbar, const double *theta,
                       const double *m, double K, double G, double *f) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    double acc[3] = {0, 0, 0};
    for (int64_t p = rowptr[i]; p < rowptr[i + 1]; ++p) {
      if (!rho[p]) continue;
      int64_t j = col[p];
      double theta_t = theta[i] / m[i] + theta[j] / m[j];  /* theta~_ij */
      double e_t = e[p] / m[i] + e[p] / m[j];              /* e~_ij, */
      double t = (K - G / 3.0) * theta_t * xbar[p] + G * e_t;
      for (int k = 0; k < dim; ++k) {
        double Mk = (coords[dim * j + k] - coords[dim * i + k]) / xbar[p];
        acc[k] += t * Mk * V[j];
      }
    }
    for (int k = 0; k < dim; ++k) f[dim * i + k] = acc[k];
  }
}

/* ------------------------------------------------------------------------------------------
 * Step 9: explicit "modified central difference" update (Eq. 2.11; App. B
 * PAPER.md:872-880):
 *   a_i = (f_i + g(t_n) b_i) / rho_mass ;  v_i <- v_i + dt a_i ;  u_i <- u_i + dt v_i
 * with g(t_n) = min(1, (n dt)/ramp_time), g = 1 if ramp_time <= 0 (reading C-14).
 * Boundary conditions per dof (readings C-3, C-4): clamped: u stays, v = 0; prescribed
 * velocity: v = vbar, u += dt vbar; clamp wins if both are set.  b_i = bval on body-force
 * nodes (bit 6) for dofs that are not prescribed-velocity dofs.
 * ---------------------------------------------------------------------------------------- */
void pdo_update(int64_t n, int dim, const double *f, const uint8_t *flags, const double *bval,
                double rho_mass, double dt, double ramp_time, int64_t step, double *u,
                double *v) {
  double g = 1.0;
  if (ramp_time > 0.0) {
    g = ((double)step * dt) / ramp_time;
    if (g > 1.0) g = 1.0;
  }
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    unsigned fl = flags ? flags[i] : 0u;
    for (int k = 0; k < dim; ++k) {
      int64_t q = dim * i + k;
      if (fl & PDO_CLAMP(k)) {
        v[q] = 0.0;
        continue;
      }
      if (fl & PDO_PRESC(k)) {
        v[q] = bval[q];
        u[q] = u[q] + dt * v[q];
        continue;
      }
      double b = (fl & PDO_BODYF) ? bval[q] : 0.0;
      double a = (f[q] + g * b) / rho_mass;
      v[q] = v[q] + dt * a;
      u[q] = u[q] + dt * v[q];
    }
  }
}

/* ------------------------------------------------------------------------------------------
 * Step 10: critical-stretch bond breaking on the NEW displacement (readings C-5, C-6, C-7):
 *   s_ij = e_ij / xbar_ij (Eq. 1.17), e linearized (reading C-1);
 *   rho_ij <- 0 if s_ij >= s_c (Eq. 1.30 keeps s < s_c), irreversible,
 *   unless either end node carries the no-fail bit.  Returns the number of directed bonds
 *   broken in this call.  near[0] counts intact bonds with |s - s_c| <= near_tol * s_c
 *   (the "near-threshold" events the parity report lists).
 * ---------------------------------------------------------------------------------------- */
int64_t pdo_break(int64_t n, int dim, const double *coords, const int64_t *rowptr,
                  const int32_t *col, const uint8_t *flags, const double *u, double s_c,
                  uint8_t *rho, double near_tol, int64_t *near) {
  int64_t broken = 0, nnear = 0;
#pragma omp parallel for schedule(static) reduction(+ : broken, nnear)
  for (int64_t i = 0; i < n; ++i) {
    for (int64_t p = rowptr[i]; p < rowptr[i + 1]; ++p) {
      if (!rho[p]) continue;
      int64_t j = col[p];
      double xbar = sqrt(dist2(dim, coords + dim * i, coords + dim * j));
      double ext = 0.0;
      for (int k = 0; k < dim; ++k) {
        double Mk = (coords[dim * j + k] - coords[dim * i + k]) / xbar;
        ext += Mk * (u[dim * j + k] - u[dim * i + k]);
      }
      double s = ext / xbar;
      if (fabs(s - s_c) <= near_tol * s_c) ++nnear;
      int nofail = flags && ((flags[i] | flags[j]) & PDO_NOFAIL);
      if (s >= s_c && !nofail) {
        rho[p] = 0;
        ++broken;
      }
    }
  }
  if (near) *near = nnear;
  return broken;
}

/* ------------------------------------------------------------------------------------------
 * Step 11: damage phi_i = 1 - (sum_j rho_ij V_j) / (sum_j V_j) (Eq. 1.31),
 * denominator over the full geometric family (reading C-10).
 * ---------------------------------------------------------------------------------------- */
void pdo_damage(int64_t n, const double *V, const int64_t *rowptr, const int32_t *col,
                const uint8_t *rho, const double *fvol, double *phi) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    double s = 0.0;
    for (int64_t p = rowptr[i]; p < rowptr[i + 1]; ++p)
      if (rho[p]) s += V[col[p]];
    phi[i] = 1.0 - s / fvol[i];
  }
}

/* strain energy density at every node, Eq. 1.20 written with the mode
 * constants: W_i = ((K - G/3)/(2A)) theta_i^2 + (G/(2 m_i)) sum_j rho_ij e_ij^2 V_j.
 * (3D: K-G/3 = 3kappa-5mu, A = 3, G = 15mu gives Eq. 1.20 as printed.)  Used by the pins
 * only (energy checks), never by a time step. */
void pdo_energy_density(int64_t n, const double *V, const int64_t *rowptr, const int32_t *col,
                        const double *e, const double *theta, const double *m, double A,
                        double K, double G, double *W) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    double s = 0.0;
    for (int64_t p = rowptr[i]; p < rowptr[i + 1]; ++p) s += e[p] * e[p] * V[col[p]];
    W[i] = ((K - G / 3.0) / (2.0 * A)) * theta[i] * theta[i] + (G / (2.0 * m[i])) * s;
  }
}

/* ------------------------------------------------------------------------------------------
 * The whole step, steps 6..11 in order, for nsteps steps starting at step index step0.
 * Scratch e, xbar (Z doubles each), theta, f are caller-provided.  s_c <= 0 or +inf disables
 * steps 10-11.  Returns the number of directed bonds broken during the call.
 * If break_log != NULL (capacity log_cap entries of 3 int64: step, i, j) every break is
 * recorded in (step, i, j) order; *log_n receives the count (may exceed log_cap: truncated).
 * ---------------------------------------------------------------------------------------- */
int64_t pdo_run(int64_t n, int dim, const double *coords, const double *V, const int64_t *rowptr,
                const int32_t *col, uint8_t *rho, const double *m, const double *fvol,
                const uint8_t *flags, const double *bval, double A, double K, double G,
                double rho_mass, double dt, double ramp_time, double s_c, int64_t step0,
                int64_t nsteps, double *u, double *v, double *phi, double *e, double *xbar,
                double *theta, double *f, double near_tol, int64_t *near_total,
                int64_t *break_log, int64_t log_cap, int64_t *log_n) {
  int fracture = (s_c > 0.0) && isfinite(s_c);
  int64_t total = 0, nlog = 0, near_sum = 0;
  int64_t Z = rowptr[n];
  uint8_t *before = NULL;
  if (fracture && break_log) before = (uint8_t *)malloc((size_t)Z);
  for (int64_t s = 0; s < nsteps; ++s) {
    int64_t step = step0 + s;
    pdo_extension(n, dim, coords, rowptr, col, rho, u, e, xbar);             /* step 6  */
    pdo_dilatation(n, V, rowptr, col, e, xbar, A, m, theta);                  /* step 7  */
    pdo_force_density(n, dim, coords, V, rowptr, col, rho, e, xbar, theta, m, K, G, f); /* 8 */
    pdo_update(n, dim, f, flags, bval, rho_mass, dt, ramp_time, step, u, v);  /* step 9  */
    if (fracture) {
      if (before) memcpy(before, rho, (size_t)Z);
      int64_t nn = 0;
      total += pdo_break(n, dim, coords, rowptr, col, flags, u, s_c, rho, near_tol, &nn); /* 10 */
      near_sum += nn;
      if (before) {
        for (int64_t i = 0; i < n; ++i)
          for (int64_t p = rowptr[i]; p < rowptr[i + 1]; ++p)
            if (before[p] && !rho[p]) {
              if (nlog < log_cap) {
                break_log[3 * nlog + 0] = step;
                break_log[3 * nlog + 1] = i;
                break_log[3 * nlog + 2] = col[p];
              }
              ++nlog;
            }
      }
    }
  }
  if (phi) pdo_damage(n, V, rowptr, col, rho, fvol, phi);                     /* step 11 */
  if (near_total) *near_total = near_sum;
  if (log_n) *log_n = nlog;
  free(before);
  return total;
}

/* ==========================================================================================
 * VARIANT: the GEOMETRIC extension of the paper's own loop code,
 *   e_ij = || xi_ij + eta_ij || - || xi_ij ||,  eta_ij = u_j - u_i       (App. C),
 * used in place of the linearized M . eta in the dilatation, the force AND the failure stretch
 * s = e / xbar; the direction stays M = xi / xbar (App. C).  Everything else
 * (steps 7, 8, 9, 11) is the code above, unchanged.  Evaluation order as in the listing:
 * Eta_k = Xi_k + (U_j,k - U_i,k), eta = sqrt(sum_k Eta_k^2) summed in k order, E = eta - xi.
 * Pins (tests/test_oracle_pins.py): a FINITE rigid rotation gives e = 0 and zero force (the linearized
 * model does not), transverse hand value sqrt(r^2 + b^2) - r, e_geo -> e_lin quadratically for small
 * eta, the App. C pair-scatter code with its printed (geometric) extension.
 * ======================================================================================== */
void pdo_extension_geom(int64_t n, int dim, const double *coords, const int64_t *rowptr,
                        const int32_t *col, const uint8_t *rho, const double *u, double *e,
                        double *xbar_out) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    for (int64_t p = rowptr[i]; p < rowptr[i + 1]; ++p) {
      int64_t j = col[p];
      double xbar = sqrt(dist2(dim, coords + dim * i, coords + dim * j));
      double s = 0.0;
      for (int k = 0; k < dim; ++k) {
        double Eta = (coords[dim * j + k] - coords[dim * i + k]) + (u[dim * j + k] - u[dim * i + k]);
        s += Eta * Eta;
      }
      double ext = sqrt(s) - xbar;
      e[p] = rho[p] ? ext : 0.0;
      if (xbar_out) xbar_out[p] = xbar;
    }
  }
}

int64_t pdo_break_geom(int64_t n, int dim, const double *coords, const int64_t *rowptr,
                       const int32_t *col, const uint8_t *flags, const double *u, double s_c,
                       uint8_t *rho, double near_tol, int64_t *near) {
  int64_t broken = 0, nnear = 0;
#pragma omp parallel for schedule(static) reduction(+ : broken, nnear)
  for (int64_t i = 0; i < n; ++i) {
    for (int64_t p = rowptr[i]; p < rowptr[i + 1]; ++p) {
      if (!rho[p]) continue;
      int64_t j = col[p];
      double xbar = sqrt(dist2(dim, coords + dim * i, coords + dim * j));
      double sq = 0.0;
      for (int k = 0; k < dim; ++k) {
        double Eta = (coords[dim * j + k] - coords[dim * i + k]) + (u[dim * j + k] - u[dim * i + k]);
        sq += Eta * Eta;
      }
      double s = (sqrt(sq) - xbar) / xbar;
      if (fabs(s - s_c) <= near_tol * s_c) ++nnear;
      int nofail = flags && ((flags[i] | flags[j]) & PDO_NOFAIL);
      if (s >= s_c && !nofail) {
        rho[p] = 0;
        ++broken;
      }
    }
  }
  if (near) *near = nnear;
  return broken;
}

/* the whole step with the geometric extension: pdo_run with steps 6 and 10 replaced */
int64_t pdo_run_geom(int64_t n, int dim, const double *coords, const double *V, const int64_t *rowptr,
                     const int32_t *col, uint8_t *rho, const double *m, const double *fvol,
                     const uint8_t *flags, const double *bval, double A, double K, double G,
                     double rho_mass, double dt, double ramp_time, double s_c, int64_t step0,
                     int64_t nsteps, double *u, double *v, double *phi, double *e, double *xbar,
                     double *theta, double *f, double near_tol, int64_t *near_total) {
  int fracture = (s_c > 0.0) && isfinite(s_c);
  int64_t total = 0, near_sum = 0;
  for (int64_t s = 0; s < nsteps; ++s) {
    pdo_extension_geom(n, dim, coords, rowptr, col, rho, u, e, xbar);
    pdo_dilatation(n, V, rowptr, col, e, xbar, A, m, theta);
    pdo_force_density(n, dim, coords, V, rowptr, col, rho, e, xbar, theta, m, K, G, f);
    pdo_update(n, dim, f, flags, bval, rho_mass, dt, ramp_time, step0 + s, u, v);
    if (fracture) {
      int64_t nn = 0;
      total += pdo_break_geom(n, dim, coords, rowptr, col, flags, u, s_c, rho, near_tol, &nn);
      near_sum += nn;
    }
  }
  if (phi) pdo_damage(n, V, rowptr, col, rho, fvol, phi);
  if (near_total) *near_total = near_sum;
  return total;
}
