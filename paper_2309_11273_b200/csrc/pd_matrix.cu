// pd_matrix.cu -- the paper's OWN scheme on the B200, as the on-box comparison for the matrix-free path
// (SURVEY.md 8(f) #2): the four global sparse matrices of Eqs. 2.7-2.10 (assembled in
// pre-processing) and the solver body of App. B:
//
//     E = CE*U;  Theta = CTH*E;  PDF = KTH*Theta + KE*E;  RF = EXF + PDF;  ACC = RF./M;
//     VEL = VELold + ACC*Dt;  U(FreeDofs) = U(FreeDofs) + Dt*VEL(FreeDofs);  VELold = VEL;
//
// with hand-written FP64 CSR sparse matrix-vector products (the paper runs MATLAB's gpuArray SpMV).  No bond
// breaking: App. B elides the failure step, and the assembled matrices would have to be rebuilt when a bond breaks.
//
//   CE  (Nb x d Nn)  row b = bond (i < j):   -M_ij at the dofs of i, +M_ij at the dofs of j            (Eq. 2.7)
//   CTH (Nn x Nb)    row i: A xbar V_j / m_i at the bonds of i                                        (Eq. 2.10)
//   KTH (d Nn x Nn)  row (i,k): (K - G/3) xbar V_i V_j M_ij,k / m_j at column j, the sum over j of the
//                    same with 1 / m_i on the diagonal                                                 (Eq. 2.8)
//   KE  (d Nn x Nb)  row (i,k): G V_i V_j (1/m_i + 1/m_j) M_ij,k at the bonds of i                     (Eq. 2.9)
//   (w = 1; PDF is the nodal FORCE, M the lumped mass rho V_i, as in the paper)
//
// Everything is in USER node order (no reordering: the paper does none either).
#include <cub/device/device_scan.cuh>

#include <cmath>
#include <new>
#include <vector>

#include "pd_internal.cuh"

struct pd_matrix {
  int dim = 0;
  int64_t n = 0, nb = 0, Z = 0;
  double dt = 0, ramp_time = 0, rho = 0;
  int64_t step = 0;
  cudaStream_t stream = 0;
  std::vector<void *> allocs;
  size_t matrix_bytes = 0;
  // CSR matrices: rowptr (int64), col (int32), val (double)
  long long *rp[4] = {};
  int32_t *ci[4] = {};
  double *va[4] = {};
  int64_t rows[4] = {}, nnz[4] = {};
  int tpr[4] = {};
  double *U = nullptr, *VEL = nullptr, *E = nullptr, *Theta = nullptr, *PDF = nullptr, *EXF = nullptr, *Minv = nullptr;
  uint8_t *flags = nullptr;
  double *bval = nullptr;
};

namespace {

constexpr int TPB = 256;
inline unsigned nblk(int64_t n) { return (unsigned)((n + TPB - 1) / TPB); }

template <typename T>
T *mat_alloc(pd_matrix *pm, size_t count) {
  void *p = nullptr;
  if (cudaMalloc(&p, sizeof(T) * (count ? count : 1)) != cudaSuccess) { cudaGetLastError(); return nullptr; }
  pm->allocs.push_back(p);
  return (T *)p;
}

// bonds (i < j) that start at node i
__global__ void k_mat_count(int64_t n, const long long *__restrict__ rowptr, const int32_t *__restrict__ col, long long *cnt) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  long long c = 0;
  for (long long p = rowptr[i]; p < rowptr[i + 1]; ++p) c += col[p] > i;
  cnt[i] = c;
}

// id of the undirected bond {i, j}: the bonds of the lower end are numbered in the order of its row
__device__ long long bond_id(const long long *rowptr, const int32_t *col, const long long *bptr, int64_t i, int64_t j) {
  const int64_t lo = i < j ? i : j, hi = i < j ? j : i;
  long long r = 0;
  for (long long p = rowptr[lo]; p < rowptr[lo + 1]; ++p) {
    if (col[p] == hi) return bptr[lo] + r;
    r += col[p] > lo;
  }
  return -1;
}

// one thread per node i writes its rows of CTH, KTH, KE and the rows of CE of the bonds it starts
template <int DIM>
__global__ void k_mat_assemble(int64_t n, const double *__restrict__ x, const double *__restrict__ V, const double *__restrict__ m,
                               const long long *__restrict__ rowptr, const int32_t *__restrict__ col,
                               const long long *__restrict__ bptr, double A, double c1, double G,
                               long long *ce_rp, int32_t *ce_ci, double *ce_va, long long *cth_rp, int32_t *cth_ci, double *cth_va,
                               long long *kth_rp, int32_t *kth_ci, double *kth_va, long long *ke_rp, int32_t *ke_ci, double *ke_va) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const long long r0 = rowptr[i], r1 = rowptr[i + 1], len = r1 - r0;
  cth_rp[i] = r0;
  if (i == n - 1) cth_rp[n] = r1;
  double diag[DIM];
  for (int k = 0; k < DIM; ++k) {
    const int64_t row = i * DIM + k;
    kth_rp[row] = DIM * r0 + DIM * i + k * (len + 1);   // rows of node i: DIM rows of len + 1 entries
    ke_rp[row] = DIM * r0 + k * len;
    diag[k] = 0.0;
  }
  if (i == n - 1) { kth_rp[n * DIM] = DIM * r1 + DIM * n; ke_rp[n * DIM] = DIM * r1; }
  long long rank = 0;
  for (long long p = r0; p < r1; ++p) {
    const int64_t j = col[p];
    double xi[DIM], r2 = 0.0;
    for (int k = 0; k < DIM; ++k) { xi[k] = x[j * DIM + k] - x[i * DIM + k]; r2 += xi[k] * xi[k]; }
    const double xbar = sqrt(r2);
    const long long b = bond_id(rowptr, col, bptr, i, j);
    const long long q = p - r0;
    cth_ci[p] = (int32_t)b;
    cth_va[p] = A * xbar * V[j] / m[i];                                        // Eq. 2.10
    const double ck = c1 * xbar * V[i] * V[j], ce = G * V[i] * V[j] * (1.0 / m[i] + 1.0 / m[j]);
    for (int k = 0; k < DIM; ++k) {
      const double Mk = xi[k] / xbar;
      const long long pk = kth_rp[i * DIM + k] + 1 + q, pe = ke_rp[i * DIM + k] + q;
      kth_ci[pk] = (int32_t)j; kth_va[pk] = ck * Mk / m[j];                     // Eq. 2.8
      diag[k] += ck * Mk / m[i];
      ke_ci[pe] = (int32_t)b; ke_va[pe] = ce * Mk;                              // Eq. 2.9
    }
    if (j > i) {                                                                // Eq. 2.7: the bond's row of CE
      const long long bb = bptr[i] + rank;
      ++rank;
      ce_rp[bb] = 2 * DIM * bb;
      for (int k = 0; k < DIM; ++k) {
        const double Mk = xi[k] / xbar;
        ce_ci[2 * DIM * bb + k] = (int32_t)(i * DIM + k); ce_va[2 * DIM * bb + k] = -Mk;
        ce_ci[2 * DIM * bb + DIM + k] = (int32_t)(j * DIM + k); ce_va[2 * DIM * bb + DIM + k] = Mk;
      }
    }
  }
  for (int k = 0; k < DIM; ++k) {
    const long long pk = kth_rp[i * DIM + k];
    kth_ci[pk] = (int32_t)i; kth_va[pk] = diag[k];
  }
}
__global__ void k_mat_last(long long *ce_rp, int64_t nb, int dim) { ce_rp[nb] = 2 * dim * nb; }

// y = A x (+ y0): CSR, TPR threads per row (a power of two <= 32), FP64
template <int TPR>
__global__ void k_spmv_csr(int64_t nrows, const long long *__restrict__ rp, const int32_t *__restrict__ ci,
                           const double *__restrict__ va, const double *__restrict__ x, const double *__restrict__ y0, double *y) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t row = t / TPR;
  const int lane = (int)(t % TPR);
  double s = 0.0;
  if (row < nrows) {
    const long long a = rp[row], b = rp[row + 1];
    for (long long p = a + lane; p < b; p += TPR) s = fma(va[p], __ldg(x + ci[p]), s);
  }
#pragma unroll
  for (int o = TPR / 2; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o, TPR);
  if (row < nrows && lane == 0) y[row] = y0 ? y0[row] + s : s;
}

void spmv(const pd_matrix *pm, int which, const double *x, const double *y0, double *y) {
  const int64_t nr = pm->rows[which];
  const long long *rp = pm->rp[which];
  const int32_t *ci = pm->ci[which];
  const double *va = pm->va[which];
  switch (pm->tpr[which]) {
    case 2: k_spmv_csr<2><<<nblk(nr * 2), TPB, 0, pm->stream>>>(nr, rp, ci, va, x, y0, y); break;
    case 4: k_spmv_csr<4><<<nblk(nr * 4), TPB, 0, pm->stream>>>(nr, rp, ci, va, x, y0, y); break;
    case 8: k_spmv_csr<8><<<nblk(nr * 8), TPB, 0, pm->stream>>>(nr, rp, ci, va, x, y0, y); break;
    case 16: k_spmv_csr<16><<<nblk(nr * 16), TPB, 0, pm->stream>>>(nr, rp, ci, va, x, y0, y); break;
    default: k_spmv_csr<32><<<nblk(nr * 32), TPB, 0, pm->stream>>>(nr, rp, ci, va, x, y0, y); break;
  }
}

// RF = g EXF + PDF; ACC = RF./M; VEL += ACC Dt; U(Free) += Dt VEL(Free)   (App. B; boundary dofs as in pd_step: C-3, C-4)
__global__ void k_mat_update(int64_t ndof, int dim, const double *__restrict__ PDF, const double *__restrict__ EXF,
                             const double *__restrict__ Minv, const uint8_t *__restrict__ flags, const double *__restrict__ bval,
                             double gramp, double dt, double *VEL, double *U) {
  int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= ndof) return;
  const int64_t i = q / dim;
  const int k = (int)(q - i * dim);
  const unsigned fl = flags[i];
  double v = VEL[q], u = U[q];
  if (fl & (1u << k)) {
    v = 0.0;
  } else if (fl & (8u << k)) {
    v = bval[q];
    u += dt * v;
  } else {
    const double rf = gramp * EXF[q] + PDF[q];
    v += dt * (rf * Minv[q]);
    u += dt * v;
  }
  VEL[q] = v;
  U[q] = u;
}

__global__ void k_mat_init(int64_t n, int dim, const double *__restrict__ V, const uint8_t *__restrict__ flags,
                           const double *__restrict__ bval, const double *__restrict__ u0, const double *__restrict__ v0, double rho,
                           double *U, double *VEL, double *EXF, double *Minv) {
  int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= n * dim) return;
  const int64_t i = q / dim;
  const int k = (int)(q - i * dim);
  const unsigned fl = flags ? flags[i] : 0u;
  const bool clamped = fl & (1u << k);
  U[q] = (u0 && !clamped) ? u0[q] : 0.0;
  VEL[q] = (v0 && !clamped) ? v0[q] : 0.0;
  EXF[q] = (bval && (fl & PD_BODY_FORCE)) ? bval[q] * V[i] : 0.0;   // nodal external force b V_i
  Minv[q] = 1.0 / (rho * V[i]);
}

int pick_tpr(double mean) { return mean <= 3 ? 2 : mean <= 6 ? 4 : mean <= 12 ? 8 : mean <= 24 ? 16 : 32; }

}  // namespace

extern "C" {

int pd_matrix_destroy(pd_matrix *pm) {
  if (!pm) return PD_OK;
  cudaStreamSynchronize(pm->stream);
  for (void *p : pm->allocs) cudaFree(p);
  delete pm;
  return PD_OK;
}

int pd_matrix_create(pd_matrix **out, int64_t n, const double *coords, const double *volumes, const pd_material *mat,
                     const pd_boundary *bc, const int64_t *rowptr, const int32_t *col, const double *m, void *stream) {
  if (out) *out = nullptr;
  if (!out || !coords || !volumes || !mat || !rowptr || !col || !m || n <= 0) { pdi::set_error("null argument"); return PD_ERR_ARG; }
  if (!(mat->dim == 2 || mat->dim == 3)) { pdi::set_error("dim"); return PD_ERR_ARG; }
  pd_matrix *pm = new (std::nothrow) pd_matrix();
  if (!pm) return PD_ERR_ALLOC;
  const int dim = mat->dim;
  pm->dim = dim; pm->n = n; pm->dt = mat->dt; pm->ramp_time = mat->ramp_time; pm->rho = mat->rho;
  pm->stream = (cudaStream_t)stream;
  cudaStream_t st = pm->stream;
  auto fail = [&](int code, const char *msg) { pdi::set_error(msg); pd_matrix_destroy(pm); return code; };
  double A, K, G;
  {
    const double nu = mat->nu, kappa = mat->E / (3.0 * (1.0 - 2.0 * nu)), mu = mat->E / (2.0 * (1.0 + nu));
    if (mat->mode == PD_MODE_3D) { A = 3.0; K = 3.0 * kappa; G = 15.0 * mu; }
    else if (mat->mode == PD_MODE_PLANE_STRESS) {
      A = 2.0 * (1.0 - 2.0 * nu) / (1.0 - nu);
      K = 2.0 * kappa * (1.0 - 2.0 * nu) / (1.0 - nu) - (2.0 / 3.0) * mu * ((1.0 + nu) * (1.0 - 3.0 * nu)) / ((1.0 - nu) * (1.0 - 2.0 * nu));
      G = 8.0 * mu;
    } else { A = 2.0; K = 2.0 * kappa - (2.0 / 3.0) * mu; G = 8.0 * mu; }
  }
  // ---- stage the inputs (host or device pointers) ----
  long long hz = 0;
  double *d_x = mat_alloc<double>(pm, n * dim), *d_V = mat_alloc<double>(pm, n), *d_m = mat_alloc<double>(pm, n);
  long long *d_rp = mat_alloc<long long>(pm, n + 1);
  if (!d_x || !d_V || !d_m || !d_rp) return fail(PD_ERR_ALLOC, "device allocation failed");
  cudaMemcpyAsync(d_x, coords, sizeof(double) * n * dim, cudaMemcpyDefault, st);
  cudaMemcpyAsync(d_V, volumes, sizeof(double) * n, cudaMemcpyDefault, st);
  cudaMemcpyAsync(d_m, m, sizeof(double) * n, cudaMemcpyDefault, st);
  cudaMemcpyAsync(d_rp, rowptr, sizeof(long long) * (n + 1), cudaMemcpyDefault, st);
  cudaMemcpyAsync(&hz, d_rp + n, sizeof(long long), cudaMemcpyDeviceToHost, st);
  if (cudaStreamSynchronize(st) != cudaSuccess) return fail(PD_ERR_CUDA, "staging failed");
  pm->Z = hz; pm->nb = hz / 2;
  int32_t *d_col = mat_alloc<int32_t>(pm, hz);
  long long *d_cnt = mat_alloc<long long>(pm, n + 1), *d_bptr = mat_alloc<long long>(pm, n + 1);
  if (!d_col || !d_cnt || !d_bptr) return fail(PD_ERR_ALLOC, "device allocation failed");
  cudaMemcpyAsync(d_col, col, sizeof(int32_t) * hz, cudaMemcpyDefault, st);
  cudaMemsetAsync(d_cnt + n, 0, sizeof(long long), st);
  k_mat_count<<<nblk(n), TPB, 0, st>>>(n, d_rp, d_col, d_cnt);
  {
    size_t tb = 0;
    cub::DeviceScan::ExclusiveSum(nullptr, tb, d_cnt, d_bptr, (int)(n + 1), st);
    void *tmp = mat_alloc<char>(pm, tb);
    if (!tmp) return fail(PD_ERR_ALLOC, "device allocation failed");
    cub::DeviceScan::ExclusiveSum(tmp, tb, d_cnt, d_bptr, (int)(n + 1), st);
  }
  // ---- the four matrices ----
  const int64_t nb = pm->nb;
  const int64_t rows[4] = {nb, n, n * dim, n * dim};                       // CE, CTH, KTH, KE
  const int64_t nnz[4] = {2 * dim * nb, hz, dim * (hz + n), dim * hz};
  for (int q = 0; q < 4; ++q) {
    pm->rows[q] = rows[q]; pm->nnz[q] = nnz[q];
    if (nnz[q] >= (1ll << 40)) return fail(PD_ERR_LIMIT, "matrix too large");
    pm->rp[q] = mat_alloc<long long>(pm, rows[q] + 1);
    pm->ci[q] = mat_alloc<int32_t>(pm, nnz[q]);
    pm->va[q] = mat_alloc<double>(pm, nnz[q]);
    if (!pm->rp[q] || !pm->ci[q] || !pm->va[q]) return fail(PD_ERR_ALLOC, "device allocation failed for the sparse matrices");
    pm->matrix_bytes += sizeof(long long) * (rows[q] + 1) + 12 * (size_t)nnz[q];
    pm->tpr[q] = pick_tpr((double)nnz[q] / (double)rows[q]);
  }
  if (dim == 2)
    k_mat_assemble<2><<<nblk(n), TPB, 0, st>>>(n, d_x, d_V, d_m, d_rp, d_col, d_bptr, A, K - G / 3.0, G, pm->rp[0], pm->ci[0], pm->va[0],
                                               pm->rp[1], pm->ci[1], pm->va[1], pm->rp[2], pm->ci[2], pm->va[2], pm->rp[3], pm->ci[3], pm->va[3]);
  else
    k_mat_assemble<3><<<nblk(n), TPB, 0, st>>>(n, d_x, d_V, d_m, d_rp, d_col, d_bptr, A, K - G / 3.0, G, pm->rp[0], pm->ci[0], pm->va[0],
                                               pm->rp[1], pm->ci[1], pm->va[1], pm->rp[2], pm->ci[2], pm->va[2], pm->rp[3], pm->ci[3], pm->va[3]);
  k_mat_last<<<1, 1, 0, st>>>(pm->rp[0], nb, dim);
  // ---- solver vectors (App. A) ----
  const int64_t nd = n * dim;
  pm->U = mat_alloc<double>(pm, nd); pm->VEL = mat_alloc<double>(pm, nd); pm->PDF = mat_alloc<double>(pm, nd);
  pm->EXF = mat_alloc<double>(pm, nd); pm->Minv = mat_alloc<double>(pm, nd); pm->E = mat_alloc<double>(pm, nb);
  pm->Theta = mat_alloc<double>(pm, n); pm->flags = mat_alloc<uint8_t>(pm, n); pm->bval = mat_alloc<double>(pm, nd);
  double *d_u0 = mat_alloc<double>(pm, nd), *d_v0 = mat_alloc<double>(pm, nd);
  if (!pm->U || !pm->VEL || !pm->PDF || !pm->EXF || !pm->Minv || !pm->E || !pm->Theta || !pm->flags || !pm->bval || !d_u0 || !d_v0)
    return fail(PD_ERR_ALLOC, "device allocation failed");
  cudaMemsetAsync(pm->flags, 0, n, st);
  cudaMemsetAsync(pm->bval, 0, sizeof(double) * nd, st);
  cudaMemsetAsync(d_u0, 0, sizeof(double) * nd, st);
  cudaMemsetAsync(d_v0, 0, sizeof(double) * nd, st);
  if (bc) {
    if (bc->flags) cudaMemcpyAsync(pm->flags, bc->flags, n, cudaMemcpyDefault, st);
    if (bc->value) cudaMemcpyAsync(pm->bval, bc->value, sizeof(double) * nd, cudaMemcpyDefault, st);
    if (bc->u0) cudaMemcpyAsync(d_u0, bc->u0, sizeof(double) * nd, cudaMemcpyDefault, st);
    if (bc->v0) cudaMemcpyAsync(d_v0, bc->v0, sizeof(double) * nd, cudaMemcpyDefault, st);
  }
  k_mat_init<<<nblk(nd), TPB, 0, st>>>(n, dim, d_V, pm->flags, pm->bval, d_u0, d_v0, mat->rho, pm->U, pm->VEL, pm->EXF, pm->Minv);
  cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) { pdi::cuda_fail(e, "pd_matrix_create"); pd_matrix_destroy(pm); return PD_ERR_CUDA; }
  *out = pm;
  return PD_OK;
}

int pd_matrix_step(pd_matrix *pm, int64_t nsteps) {
  if (!pm || nsteps < 0) { pdi::set_error("bad argument"); return PD_ERR_ARG; }
  const int64_t nd = pm->n * pm->dim;
  for (int64_t it = 0; it < nsteps; ++it) {
    spmv(pm, 0, pm->U, nullptr, pm->E);              // E = CE*U
    spmv(pm, 1, pm->E, nullptr, pm->Theta);          // Theta = CTH*E
    spmv(pm, 2, pm->Theta, nullptr, pm->PDF);        // PDF = KTH*Theta
    spmv(pm, 3, pm->E, pm->PDF, pm->PDF);            //     + KE*E
    double g = 1.0;
    if (pm->ramp_time > 0.0) g = std::fmin(1.0, ((double)pm->step * pm->dt) / pm->ramp_time);
    k_mat_update<<<nblk(nd), TPB, 0, pm->stream>>>(nd, pm->dim, pm->PDF, pm->EXF, pm->Minv, pm->flags, pm->bval, g, pm->dt, pm->VEL, pm->U);
    pm->step += 1;
  }
  PD_CUDA(cudaGetLastError());
  return PD_OK;
}

int pd_matrix_get(pd_matrix *pm, double *u, double *v, int64_t info[8]) {
  if (!pm) { pdi::set_error("null argument"); return PD_ERR_ARG; }
  const size_t bytes = sizeof(double) * pm->n * pm->dim;
  if (u) PD_CUDA(cudaMemcpyAsync(u, pm->U, bytes, cudaMemcpyDefault, pm->stream));
  if (v) PD_CUDA(cudaMemcpyAsync(v, pm->VEL, bytes, cudaMemcpyDefault, pm->stream));
  PD_CUDA(cudaStreamSynchronize(pm->stream));
  if (info) {
    info[0] = pm->n; info[1] = pm->nb; info[2] = pm->nnz[0]; info[3] = pm->nnz[1]; info[4] = pm->nnz[2]; info[5] = pm->nnz[3];
    info[6] = (int64_t)pm->matrix_bytes; info[7] = pm->step;
  }
  return PD_OK;
}

}  // extern "C"
