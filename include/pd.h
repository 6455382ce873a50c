/*
 * pd.h -- C-ABI boundary of the B200-native explicit OSB-PD time stepper (libpd.so).
 *
 * One hot path: the per-time-step explicit dynamics of the linearized ordinary state-based
 * peridynamic model of arXiv 2309.11273, FP64, hand-written CUDA for sm_100a.
 * Every step of that path runs in the library's kernels; bindings above this header only
 * marshal arguments.  There is no CPU fallback: without a CUDA device every entry point
 * except pd_last_error / pd_version returns PD_ERR_CUDA.
 *
 * Conventions
 *  - Units SI, all floating point is IEEE binary64.
 *  - Node-indexed inputs/outputs are in USER node order (the order of `coords`); the library
 *    reorders internally for locality and hides it.
 *  - Vector fields are AoS: dim doubles per node (x0,y0[,z0],x1,...).
 *  - Every data pointer may be HOST or DEVICE memory (the library asks the driver which);
 *    inputs are copied during pd_create, the caller keeps ownership; outputs are written to
 *    caller-owned memory of the stated size.
 *  - All work is enqueued on the stream given in pd_runtime (default stream if none).
 *    pd_step never synchronises with the host.  pd_create and the pd_get_* calls return after
 *    the stream has drained (their results are complete on return).
 *  - Return value 0 = PD_OK, negative = error; pd_last_error() gives a message for the calling
 *    thread.  The library never throws, never aborts and never prints.
 */
#ifndef PD_H_
#define PD_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define PD_API __attribute__((visibility("default")))
#else
#define PD_API
#endif

#define PD_OK 0
#define PD_ERR_ARG (-1)      /* bad argument: n<=0, dim/mode mismatch, nu outside (-1,0.5), E/rho/dt/horizon<=0,
                                a pre-cut pair that is not a bond, null pointer                          */
#define PD_ERR_ISOLATED (-2) /* a node has an empty family (m_i = 0 would divide by zero, Eq. 1.6)     */
#define PD_ERR_ALLOC (-3)    /* device allocation failed                                               */
#define PD_ERR_CUDA (-4)     /* CUDA runtime error / no device                                         */
#define PD_ERR_LIMIT (-5)    /* problem exceeds an internal limit (2^31 directed bonds, cell table).
                                (SURVEY 8(b) sketched -5 as "non-finite state, debug builds"; there is no debug
                                build of this library, so the code is used for limits: DESIGN.md 1)      */

/* dimension modes: constants A, K, G of Eqs. 1.8, 1.15, 1.16 */
#define PD_MODE_3D 0
#define PD_MODE_PLANE_STRESS 1
#define PD_MODE_PLANE_STRAIN 2

/* bond extension (pd_material.extension) */
#define PD_EXT_LINEARIZED 0 /* e = M . (u_j - u_i)  (Eq. 2.7): the model of the paper */
#define PD_EXT_GEOMETRIC 1  /* e = ||xi + u_j - u_i|| - ||xi||  (App. C listing): variant */

/* per-node boundary flags (pd_boundary.flags) */
#define PD_CLAMP_X 0x01u /* bits 0-2: dof k clamped: u_k = 0 and v_k = 0 for all time (App. B "FreeDofs", */
#define PD_CLAMP_Y 0x02u /*           PAPER.md:878); u0/v0 on such dofs are overridden by 0              */
#define PD_CLAMP_Z 0x04u
#define PD_PRESC_X 0x08u /* bits 3-5: dof k has prescribed velocity value[dim*i+k] ("remains constant     */
#define PD_PRESC_Y 0x10u /*           during the simulation"): v_k = vbar, u_k += dt vbar */
#define PD_PRESC_Z 0x20u
#define PD_BODY_FORCE 0x40u /* bit 6: value[dim*i+k] is a body-force density b [N/m^3] (Eq. 1.1) on every
                                      dof of the node that is neither clamped nor prescribed             */
#define PD_NO_FAIL 0x80u    /* bit 7: bonds with this node at either end never break                    */
/* a clamped dof wins over a prescribed one if both bits are set */

typedef struct pd_sim pd_sim; /* opaque; owned by the library, released by pd_destroy */

typedef struct {
  int dim;          /* 2 or 3                                                                  */
  int mode;         /* PD_MODE_*; dim==3 <=> PD_MODE_3D                                         */
  double E;         /* Young modulus  > 0;  kappa = E/(3(1-2nu)), mu = E/(2(1+nu)) */
  double nu;        /* Poisson ratio in (-1, 0.5)                                               */
  double rho;       /* mass density > 0                                                         */
  double s_c;       /* critical stretch (Eqs. 1.26/1.28 give it); <= 0 or +inf disables fracture */
  double dt;        /* fixed time increment > 0 (Eq. 2.11)                                      */
  double ramp_time; /* body forces are scaled by g(t_n) = min(1, n*dt/ramp_time); <= 0 => g = 1 */
  int extension;    /* PD_EXT_LINEARIZED (0, the paper's model and the default) or PD_EXT_GEOMETRIC:
                       e = ||xi + eta|| - ||xi|| of the paper's loop code (App. C) in
                       the dilatation, the force and the failure stretch; direction M stays xi/||xi||   */
} pd_material;

typedef struct {
  const uint8_t *flags;  /* n bytes of PD_* flags, or NULL (= all free)                           */
  const double *value;   /* dim*n, meaning per the flags; may be NULL if no PRESC/BODY_FORCE flag */
  const int32_t *precut; /* 2*n_precut user indices: bonds broken from the start (either order,
                            each undirected bond once or twice); every pair must be a bond        */
  int64_t n_precut;
  const double *u0; /* dim*n initial displacement, or NULL (= 0)                                  */
  const double *v0; /* dim*n initial velocity, or NULL (= 0)                                      */
} pd_boundary;

/* device memory + stream come from the caller (PyTorch's caching allocator and current stream
 * in the Python binding).  alloc returns a device pointer aligned to >= 256 B or NULL. */
typedef struct {
  void *(*alloc)(size_t bytes, void *ctx);
  void (*free)(void *ptr, void *ctx);
  void *ctx;
  void *stream; /* cudaStream_t */
} pd_runtime;

/*
 * pd_create -- pre-processing, run once.  Builds on the GPU: the cell list, the
 * locality-sorted node order, the family H_i = { j != i : ||x_j - x_i|| <= horizon } (inclusive,
 * PAPER.md:121-125) with one intact/broken bit per directed bond (Eq. 1.30) -- as stencil bit masks
 * over a dense cell array when the body is a lattice, else as a sliced-ELL neighbour list --, the weighted volume m_i = sum_j ||xi_ij||^2 V_j (Eq. 1.9, w = 1)
 * and the family volume sum_j V_j (denominator of Eq. 1.31), both over the full geometric
 * family and never updated; clears the bits of the pre-cut pairs (both directions).
 *   coords  dim*n AoS reference positions; volumes n nodal volumes V_i (> 0)
 *   runtime may be NULL (cudaMallocAsync on the default stream)
 * Errors: PD_ERR_ARG, PD_ERR_ISOLATED, PD_ERR_ALLOC, PD_ERR_CUDA, PD_ERR_LIMIT.  *out is NULL on error.
 */
PD_API int pd_create(pd_sim **out, int64_t n, const double *coords, const double *volumes, double horizon,
              const pd_material *material, const pd_boundary *boundary, const pd_runtime *runtime);

/*
 * pd_step -- advance nsteps explicit steps.  Step n (t_n = n*dt), all on the device:
 *  (1) e_ij = M_ij . (u_j - u_i), M_ij = xi_ij/||xi_ij||, 0 if broken   (Eq. 2.7)
 *  (2) theta_i = (A/m_i) sum_j rho_ij xbar_ij e_ij V_j                   (Eq. 1.6 / 2.3)
 *  (3) f_i = sum_j rho_ij [(K-G/3)(theta_i/m_i + theta_j/m_j) xbar_ij
 *                          + G e_ij (1/m_i + 1/m_j)] M_ij V_j            (Eq. 2.1 / 2.2)
 *  (4) v_i += dt (f_i + g(t_n) b_i)/rho ; u_i += dt v_i ; boundary dofs  (Eq. 2.11; App. B)
 *  (5) every intact bond with s_ij = e_ij(u^{n+1})/xbar_ij >= s_c breaks, irreversibly
 *      (Eqs. 1.17, 1.30); damage phi_i = 1 - sum_j rho_ij V_j / sum_j V_j (Eq. 1.31)
 * Observable state at step boundaries is (u^n, v^n, rho^n, phi^n): forces at step n use rho^n
 * and u^n; rho^{n+1} is decided from u^{n+1}.  Asynchronous: no host synchronisation; in the steady
 * state (load ramp finished) the steps are replayed from a CUDA graph captured once per handle.
 * A launch that cannot be prepared returns its error code and leaves the step counter and the state
 * where they were; errors of the device work itself surface in the next synchronising call.
 */
PD_API int pd_step(pd_sim *sim, int64_t nsteps);

/*
 * pd_get_u / pd_get_v -- the state of the explicit scheme at the current step boundary: displacement u^n and
 * velocity v^n of Eq. 2.11 (`U`, `VEL` of App. A/B).
 *   dst  dim*n doubles, AoS, user node order, host or device, caller-owned.
 * pd_get_damage -- phi_i = 1 - sum_j rho_ij V_j / sum_j V_j (Eq. 1.31) with rho^n decided from u^n
 * (Eq. 1.30; a deferred failure pass is flushed first), denominator over the full geometric family.
 *   dst  n doubles, user node order, host or device, caller-owned.
 * All three synchronise with the stream.  Errors: PD_ERR_ARG (null), PD_ERR_ALLOC, PD_ERR_CUDA.
 */
PD_API int pd_get_u(pd_sim *sim, double *dst);
PD_API int pd_get_v(pd_sim *sim, double *dst);
PD_API int pd_get_damage(pd_sim *sim, double *dst);

/*
 * pd_get_u_static -- pd_get_u for callers that may not allocate device memory (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc): the same u^n of Eq. 2.11, the same dst
 * (dim*n doubles, AoS, user node order, host or device, caller-owned), bit for bit.  pd_get_u stages the reordered
 * field in a scratch buffer that it allocates and frees per call; this entry point stages it in a static device array of
 * PD_STATIC_MAX_DOUBLES doubles (8 MiB) that every GPU that loads the library holds until the process exits, and calls
 * no cudaMalloc / cudaFree, no pd_runtime callback and no allocating library routine: one kernel and one copy on the
 * handle's stream, then a synchronise.  The handle's device must be current (as for every call).
 * All calls, on all handles, share that one array per device: calls that overlap on the GPU (different streams or
 * host threads) race and must be serialised by the caller.  Nothing of an earlier call's contents is ever read.
 * Errors: PD_ERR_ARG (null), PD_ERR_LIMIT (dim*n > PD_STATIC_MAX_DOUBLES: use pd_get_u; nothing is launched),
 * PD_ERR_CUDA.
 */
#define PD_STATIC_MAX_DOUBLES (1 << 20)
PD_API int pd_get_u_static(pd_sim *sim, double *dst);

PD_API int pd_destroy(pd_sim *sim);

/* ---- extensions (not named by the north star; needed to check and report it) ---- */

/* device-side damage reduction.  Any pointer may be NULL.  n_broken_directed counts directed
 * bonds with rho = 0 (pre-cuts included). */
PD_API int pd_get_stats(pd_sim *sim, int64_t *n_directed_bonds, int64_t *n_broken_directed,
                 double *max_damage, int64_t *n_nodes_damage_ge_half, int64_t *step);

/* the family with its status, in user indices, for bond-by-bond parity of broken sets:
 * rowptr[n+1] (row i = user node i), col[Z] user index of the neighbour (order inside a row
 * unspecified), intact[Z] 1/0.  Pass col = intact = NULL to get rowptr only. */
PD_API int pd_get_bond_mask(pd_sim *sim, int64_t *rowptr, int32_t *col, uint8_t *intact);

/* per-node pre-processing results in user order (either may be NULL): m_i (Eq. 1.9) and the
 * dilatation theta_i of the current displacement (Eq. 1.6). */
PD_API int pd_get_node_fields(pd_sim *sim, double *m, double *theta);

/* layout/launch facts for the roofline report: counts[0]=n, [1]=n padded (array length incl. phantoms),
 * [2]=Z directed bonds, [3]=stored neighbour-index slots (0 in the lattice layout, which stores none),
 * [4]=kernel launches issued by pd_step so far, [5]=bytes of device memory held, [6]=1 if volumes are
 * uniform, [7]=layout: 0 = windowed sliced ELL (any point cloud), 1 = dense lattice, bond geometry per bond
 * (jittered lattices), 2 = dense UNIFORM lattice, bond geometry a constant per stencil offset (the paper's
 * uniform grids), 3 = the same with the stencil of horizon 3.015 dx compiled in (122 offsets in 3-D,
 * 28 in 2-D). */
PD_API int pd_get_layout(pd_sim *sim, int64_t counts[8]);

/* measurement aid for the roofline report: like pd_step, but brackets every kernel launch with
 * CUDA events on the sim's stream and returns the summed device time per kernel in milliseconds:
 * ms[0] = dilatation(+break) kernel, ms[1] = force+update kernel.  Synchronises. */
PD_API int pd_step_timed(pd_sim *sim, int64_t nsteps, double ms[2]);

/* ---- halo pack / unpack of the multi-GPU slab decomposition (paper_2309_11273_b200/slabs.py) ----
 * pd_gather_u copies the rows idx[0..count) (user node indices) of the current displacement u^n into dst (count*dim doubles,
 * AoS); pd_scatter_u overwrites those rows of u^n with src.  idx, dst, src are DEVICE pointers (the buffers that the
 * point-to-point exchange between slab neighbours sends and receives); both calls are asynchronous on the handle's
 * stream and do not touch v or the bond status.  Between two pd_step calls a rank gathers the owned nodes its
 * neighbours hold as halo, exchanges, and scatters the halo nodes it received: that is the whole exchange step. */
PD_API int pd_gather_u(pd_sim *sim, const int32_t *idx, int64_t count, double *dst);
PD_API int pd_scatter_u(pd_sim *sim, const int32_t *idx, int64_t count, const double *src);

/* ---- quasi-static driver: adaptive dynamic relaxation ----
 * The paper solves its Ex. 4 "by using an adaptive dynamic relaxation algorithm presented in [Underwood 1983; Kilic &
 * Madenci 2010]" and does not restate it; this is that algorithm with a uniform fictitious density
 * Lambda = lam I and pseudo time step 1, on top of the dilatation / force kernels of pd_step:
 *   R^n = f(U^n) + g b;  1K_ii = -(R_i^n - R_i^{n-1}) / (lam Ud_i^{n-1/2});  c^n = 2 sqrt((U.1K U)/(U.U)) over the free dofs
 *   Ud^{n+1/2} = ((2 - c^n) Ud^{n-1/2} + 2 R^n / lam) / (2 + c^n)   (first iteration: R^0 / (2 lam));  U^{n+1} = U^n + Ud^{n+1/2}
 * Clamped dofs keep U; dofs flagged PD_PRESC_* advance by value[dim*i+k] per iteration (a fixed displacement increment,
 * PAPER.md:813); PD_BODY_FORCE values are force densities as in pd_step; the failure check of pd_step runs on every
 * U^{n+1} when s_c > 0.  The handle must have been created with rho = 1 and dt = 1 (pseudo time; PD_ERR_ARG otherwise).
 * lam >= lambda_max(K)/4 for stability (K: f = -K u).  Asynchronous: c^n is formed on the device; pd_get_u returns U^n. */
PD_API int pd_adr_step(pd_sim *sim, int64_t niter, double lam);

/* ---- the paper's own scheme, as an on-box comparison for the matrix-free path ----
 * pd_matrix_create assembles, on the device, the four global sparse matrices CE (Nb x d n), CTH (n x Nb), KTH (d n x n),
 * KE (d n x Nb) of Eqs. 2.7-2.10 in CSR (int64 row pointers, int32 columns, FP64 values), user
 * node order, from the family of an existing handle:
 *   rowptr[n+1], col[Z]  the directed family as returned by pd_get_bond_mask; m[n] as returned by pd_get_node_fields
 *   coords, volumes, material, boundary  as for pd_create (pre-cuts and s_c are ignored: App. B has no failure step)
 *   stream  cudaStream_t or NULL.  All pointers host or device; inputs are copied.
 * pd_matrix_step runs the solver body of App. B: E = CE U; Theta = CTH E; PDF = KTH Theta + KE E;
 * RF = EXF + PDF; ACC = RF./M; VEL += ACC Dt; U(FreeDofs) += Dt VEL(FreeDofs) -- 4 hand-written CSR SpMVs + 1 vector
 * kernel per step, asynchronous.  pd_matrix_get copies U and VEL (dim*n each, may be NULL) and fills
 * info = {n, Nb, nnz(CE), nnz(CTH), nnz(KTH), nnz(KE), bytes of the four matrices, step}; synchronises. */
typedef struct pd_matrix pd_matrix;
PD_API int pd_matrix_create(pd_matrix **out, int64_t n, const double *coords, const double *volumes, const pd_material *material,
                            const pd_boundary *boundary, const int64_t *rowptr, const int32_t *col, const double *m, void *stream);
PD_API int pd_matrix_step(pd_matrix *pm, int64_t nsteps);
PD_API int pd_matrix_get(pd_matrix *pm, double *u, double *v, int64_t info[8]);
PD_API int pd_matrix_destroy(pd_matrix *pm);

/* ---- measured FP64 issue rate of the device (the denominator of the "alu" roofline that bench.py reports beside the HBM
 * one; DESIGN.md 5 derives the nominal figure 148 SM x 64 lanes x clock) ----
 * Runs `reps` timed launches of a kernel whose every thread advances 8 independent DFMA chains (32 resident warps per
 * SM, no memory traffic) and writes the best rate, in FP64 fused multiply-adds per second over all threads, to
 * *fma_per_s.  stream: cudaStream_t or NULL.  Synchronises.  Errors: PD_ERR_ARG, PD_ERR_ALLOC, PD_ERR_CUDA. */
PD_API int pd_measure_fp64_rate(int reps, void *stream, double *fma_per_s);

/* ---- measured issue rates behind DESIGN.md 5.1 "why every directed bond is evaluated from both ends" ----
 * t_ij = t_ji in Eq. 2.2: one end of a bond could compute the term and hand it to the other end, over
 * the lanes of a warp by a shuffle or between warps through shared memory.  Times four kernels at the launch shape of
 * pd_measure_fp64_rate and writes, over all threads, per second:
 *   per_s[0] FP64 fused multiply-adds alone; per_s[1] 64-bit lane shifts alone (2 SHFL.32 each); per_s[2] groups of
 *   {1 lane-shifted double + 5 dependent DFMA} (the trade of the force pass); per_s[3] doubles through shared memory
 *   (8-byte store + load of another lane's slot).
 * stream: cudaStream_t or NULL.  Allocates nothing.  Synchronises.  Errors: PD_ERR_ARG, PD_ERR_CUDA. */
PD_API int pd_measure_pair_exchange(int reps, void *stream, double per_s[4]);

PD_API const char *pd_last_error(void);
PD_API const char *pd_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PD_H_ */
