/*
 * numa_b200.h -- C ABI of libnuma_b200.so
 *
 * B200 (sm_100a) implementation of the data-parallel hot path of the xNUMA nonhydrostatic
 * atmospheric model of arXiv 2504.08157: the matrix-free continuous-Galerkin spectral-
 * element right-hand side of the compressible Euler equations in the paper's Section-2
 * form, q = (rho', u, v, w, theta') (Eq. 1a-1c; equation of state Eq. 3,
 * L76-L80; discretisation Eq. 4-12), its global assembly (DSS; Eq. 10-12,
 * Alg. 3) and the explicit Runge-Kutta stage update that consumes it
 * ("updating the state vector", L172).  FP64 throughout (L322).
 *
 * Conventions
 *   Nq = N+1 points per direction, Mn = Nq^3 nodes per element, Ne elements,
 *   NL = Ne*Mn local (element-duplicated) nodes, local node n = i + Nq*(j + Nq*k)
 *   (i along xi fastest), faces 0..5 = xi-, xi+, eta-, eta+, zeta-, zeta+.
 *   Every field is element-local structure-of-arrays:  f[m][e][n]  -- the paper's
 *   q_e(i,j,k,e,m) (Alg. 1); state variable order m = rho', u, v, w, theta'.
 *
 * Pointers
 *   Unless a function name ends in _host, every array pointer is a DEVICE pointer
 *   (>= 8-byte aligned; 16-byte alignment enables the vectorised paths) and stays
 *   caller-owned.  The library allocates no device memory: persistent tables live in the
 *   caller-provided workspace handed to numa_init_geometry.  `stream` is a cudaStream_t
 *   passed as void* (NULL = legacy default stream).  All calls except numa_init_geometry,
 *   the *_host calls and numa_copy_table(which >= 3) only enqueue work on `stream` and return
 *   without synchronising.  A context belongs to the device that was current when
 *   numa_init_geometry created it; calling it with another device current is NUMA_ERR_ARG.
 *
 * Errors
 *   Every call returns a numa_status; nothing throws.  Argument checks are synchronous and
 *   happen before any launch.  CUDA launch errors map to NUMA_ERR_CUDA; text in
 *   numa_last_error().  There is no CPU fallback: without a CUDA device every entry point
 *   that would launch returns NUMA_ERR_CUDA.
 */
#ifndef NUMA_B200_H
#define NUMA_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct numa_ctx numa_ctx; /* opaque; created by numa_init_geometry, freed by numa_destroy */

typedef enum {
    NUMA_OK = 0,
    NUMA_ERR_ARG = 1,          /* NULL pointer, N out of range, bad size                     */
    NUMA_ERR_UNSUPPORTED = 2,  /* method = DG / eqn_set = conservative (not built) */
    NUMA_ERR_CUDA = 3,         /* CUDA runtime or launch error, or no device                 */
    NUMA_ERR_NEG_JACOBIAN = 4, /* some node has det(dx/dxi) <= 0                             */
    NUMA_ERR_WORKSPACE = 5,    /* workspace too small or misaligned                          */
    NUMA_ERR_NOT_CONVERGED = 6 /* numa_step_ark2: GMRES above tol after the last restart     */
} numa_status;

typedef struct {
    int32_t N;       /* polynomial order, 2..8 (Eq. 4-5)                            */
    int32_t method;  /* 0 = CG + DSS (built); 1 = DG face flux -> NUMA_ERR_UNSUPPORTED       */
    int32_t eqn_set; /* 0 = Eq. 1 (rho',u,v,w,theta'); 1 = conservative -> UNSUPPORTED       */
    int32_t reserved;
    int64_t n_elem;   /* Ne                                                                  */
    int64_t n_global; /* number of unique CG nodes = max(intma_cg)+1 (N_p of Eq. 9)    */
    double g;         /* gravitational acceleration, Eq. 1b                                  */
    double p_a;       /* surface pressure of Eq. 3                                           */
    double R_gas;     /* specific gas constant of dry air, Eq. 3                             */
    double c_p, c_v;  /* gamma = c_p / c_v, Eq. 3                                            */
    double f_cor;     /* f-plane Coriolis parameter (BASELINE.json config 3; Q10)  */
} numa_params;

/* Bytes of device workspace numa_init_geometry needs for these parameters (0 on bad input). */
size_t numa_workspace_bytes(const numa_params *p);

/* Bytes of device scratch numa_step_rk3 needs: two state-sized buffers in the block-shell
 * layout (the state of the step and the stage state) PLUS one field for the heating.  Always
 * size scratch with this call; numa_step_rk3 has no size argument to check it against. */
size_t numa_step_scratch_bytes(const numa_params *p);

/*
 * A0 -- setup ("the simulation is set up ... all data is transferred").
 * Computes, into the workspace: the LGL derivative matrix D and weights (Eq. 5, Eq. 8);
 * metric terms grad xi_a and the Jacobian from the nodal coordinates (L92, L149); the
 * diagonal mass M = DSS(w J) (Eq. 10) and the assembly weight omega = wJ / M
 * (Eq. 11-12); the node -> copies lists of the deterministic DSS; the background pressure
 * p0 = p_a (rho0 R theta0 / p_a)^gamma (Eq. 3); copies of ref, sponge and face_bc.
 *
 *   xyz       [3][Ne][Mn]  nodal coordinates
 *   intma_cg  [Ne][Mn]     unique CG node id of every local node (Alg. 3)
 *   face_bc   [Ne][6]      0 = interior/periodic face, 1 = no-flux wall (L256)
 *   ref       [2][Ne][Mn]  rho0, theta0 (reference state, L66)
 *   sponge    [Ne][Mn]     Rayleigh coefficient beta [1/s], or NULL (Q9)
 *   workspace              >= numa_workspace_bytes(p) bytes, 256-byte aligned
 *
 * All inputs may be freed after the call returns (this call synchronises `stream`).
 * Returns NUMA_ERR_NEG_JACOBIAN if any node has J <= 0.
 */
numa_status numa_init_geometry(const numa_params *p, const double *xyz, const int32_t *intma_cg,
                               const uint8_t *face_bc, const double *ref, const double *sponge,
                               void *workspace, size_t workspace_bytes, void *stream,
                               numa_ctx **out);

/*
 * A2-A6 -- element-local volume term (Alg. 1 kernels 2-4, L207-L222; Alg. 2):
 * rhs[m][e][n] = omega * S_m(q), S the right-hand side of Eq. 1 with H = 0: tensor-product
 * LGL derivatives along xi, eta, zeta of p', u, v, w, theta (gradient) and of rho*u
 * (divergence), chain rule with the metric terms, gravity, times wJ/M (Eq. 11-12).
 * q, rhs: [5][Ne][Mn]; rhs must not alias q.
 */
numa_status numa_rhs(numa_ctx *ctx, const double *q, double *rhs, void *stream);

/*
 * A7 -- global assembly.  CG: direct stiffness summation (Eq. 10-11; Alg. 3 gather L263-L270
 * + scatter L283-L291) in place on rhs[5][Ne][Mn]: every local copy of a global node
 * receives the sum over all copies, accumulated in ascending local-index order (bitwise
 * reproducible; no floating-point atomics).  DG face flux: NUMA_ERR_UNSUPPORTED.
 */
numa_status numa_dss_or_flux(numa_ctx *ctx, double *rhs, void *stream);

/*
 * A8-A9 -- pointwise sources on the assembled tendency, then the no-flux walls, in place:
 *   rhs_theta += heating (S_theta of Eq. 1c; [Ne][Mn] K/s or NULL);
 *   rhs_u += f v, rhs_v -= f u (Coriolis);  rhs_m -= beta q_m, m = u,v,w,theta' (sponge);
 *   at nodes of wall faces: rhs_vel -= (rhs_vel . n) n per wall face, faces in order 0..5,
 *   n = outward unit normal -+ grad xi_a / |grad xi_a|  (L256; Q8).
 */
numa_status numa_apply_sources(numa_ctx *ctx, const double *q, const double *heating, double *rhs,
                               void *stream);

/*
 * A10 -- explicit Runge-Kutta stage update (L172): q_out = a0*q0 + a1*qs + b_dt*rhs over the
 * 5 fields.  q_out may alias q0 or qs.
 */
numa_status numa_rk_stage(numa_ctx *ctx, double a0, double a1, double b_dt, const double *q0,
                          const double *qs, const double *rhs, double *q_out, void *stream);

/*
 * A11 -- n_steps SSP-RK3 (Shu-Osher, Q11) steps of size dt, in place on
 * q[5][Ne][Mn], through the FUSED stage (two kernels per stage instead of four):
 *   q_out = a0*q0 + a1*qs + b_dt*L(qs),  L = walls(sources(DSS(omega*S)))  as defined by the
 * four calls above.  The volume kernel writes omega*(a0 q0 + a1 qs) + b_dt*P(omega*(S + src))
 * -- the stage update as DSS partial sums -- and the DSS kernel completes the shared nodes in
 * place; equal to the four-call route up to rounding because DSS is linear and
 * sum_copies(omega) = 1.  Both routes are parity-tested.
 * PRECONDITIONS of that identity (the four-call route needs none of them):
 *   (1) q, heating and sponge are single-valued at a global node: all local copies of a node
 *       hold bitwise the same value (true for any state this library produced and for nodal
 *       data sampled once per global node);
 *   (2) the no-flux projector is the same in every element sharing a wall node, i.e. the
 *       walls are planar (or the metric-derived normals agree across the copies);
 *   (3) every element that touches a wall node owns a wall face at that node.
 * Box meshes with planar walls (all BASELINE.json configurations) satisfy all three.  Where
 * (2) or (3) fails the fused route averages the projected tendencies of the copies with the
 * weights omega instead of projecting the assembled tendency: use the four-call route there.
 * numa_init_geometry checks (2) and (3) (projectors of all copies of a wall node compared to 1e-10);
 * on a mesh that fails the check numa_step_rk3 / _graph / _host return NUMA_ERR_UNSUPPORTED.
 *
 * Inside the call the state is kept in a block-shell layout in `scratch`; q is
 * converted on entry and written back (natural layout) before the call returns, so the cost
 * of the two conversions is amortised over n_steps.
 * heating may be NULL; it is held constant over the n_steps (the caller refreshes it between
 * calls: BASELINE.json config 3 "refreshed every 60 s").
 * scratch: >= numa_step_scratch_bytes(p) bytes (two states plus one field for the heating),
 * 256-byte aligned.
 *
 * numa_step_rk3_graph: the same steps with the three stages of a step captured once into a
 * CUDA graph (cached in the context, keyed by the pointer arguments, dt and stream) and
 * replayed n_steps times -- same kernels, same results bit for bit, one launch call per step
 * instead of six; meant for meshes so small that a stage is shorter than its launch overhead
 * (BASELINE.json configs 1-2).  Falls back to plain launches when `stream`
 * is itself being captured by the caller.
 */
numa_status numa_step_rk3(numa_ctx *ctx, double *q, void *scratch, const double *heating,
                          double dt, int32_t n_steps, void *stream);
numa_status numa_step_rk3_graph(numa_ctx *ctx, double *q, void *scratch, const double *heating,
                                double dt, int32_t n_steps, void *stream);

/*
 * numa_step_rk3 for callers that cannot allocate device memory.
 *
 * numa_step_rk3 wants `scratch` from the caller.  A caller may have none to give: code coupled
 * into a host model whose device memory all belongs to another runtime (OpenACC data regions, a
 * framework pool that took the whole GPU when it started, so that a plain cudaMalloc fails), or a
 * time loop in which cudaMalloc / cudaFree are off limits because they synchronise the device.
 * This variant keeps the step's scratch (two block-shell states and the heating field) in an
 * array compiled into the library, NUMA_STATIC_SCRATCH_BYTES long.  It calls no cudaMalloc,
 * cudaFree or allocating library routine; q and heating are still the caller's (device pointers,
 * as for numa_step_rk3), and the result is bit for bit that of numa_step_rk3.
 *
 *   - Limit: meshes with numa_step_scratch_bytes(p) <= NUMA_STATIC_SCRATCH_BYTES (64 MiB: about
 *     740,000 local nodes, e.g. BASELINE.json configs 1 and 2 at N = 4).  Anything larger returns
 *     NUMA_ERR_WORKSPACE with the two sizes in numa_last_error and runs nothing.
 *   - Cost: every GPU the library's code is loaded on holds those 64 MiB until the process exits.
 *   - First call on a device: looks up the array's device address (cudaGetSymbolAddress, with the
 *     context's device current) and keeps it.  Make that first call outside any stream capture.
 *   - One array per device, shared by every context and every call: two calls whose work overlaps
 *     on the GPU (different streams, no ordering between them) race on it.  Calls ordered on one
 *     stream, or separated by a synchronisation, are fine.  The array keeps the last call's
 *     contents; no part of it has to be cleared, because each call rewrites what it later reads.
 */
#define NUMA_STATIC_SCRATCH_BYTES (64u << 20)
size_t numa_static_scratch_bytes(void); /* = NUMA_STATIC_SCRATCH_BYTES of the loaded library */
numa_status numa_step_rk3_static(numa_ctx *ctx, double *q, const double *heating, double dt,
                                 int32_t n_steps, void *stream);

/*
 * End-to-end variant with HOST buffers: copies q (and heating, if non-NULL) host -> device
 * into caller-provided device staging buffers, runs n_steps of numa_step_rk3, copies q back
 * and synchronises.  q_host [5][Ne][Mn] (in/out), heating_host [Ne][Mn] or NULL; pinned host
 * memory gives the best copy rate.  d_q: device [5][Ne][Mn]; d_heating: device [Ne][Mn] or NULL.
 * heating_host != NULL: the field is uploaded into d_heating first (a refresh); heating_host == NULL
 * with d_heating != NULL: the heating already resident in d_heating is used (it only changes at a
 * refresh, BASELINE.json config 3 "refreshed every 60 s"); both NULL: no heating.
 */
numa_status numa_step_rk3_host(numa_ctx *ctx, double *q_host, const double *heating_host,
                               double *d_q, double *d_heating, void *scratch, double dt,
                               int32_t n_steps, void *stream);

/*
 * Copies one of the tables built by A0 out of the workspace (device -> device, enqueued on
 * `stream`), for parity tests of the setup: which = 0 met[9][NL] (d xi_a/d x_c, index
 * 3a+c), 1 omega[NL], 2 p0[NL], 3 D[Nq*Nq] (D[i*Nq+l] = h_l'(xi_i)), 4 w[Nq].
 */
numa_status numa_copy_table(const numa_ctx *ctx, int32_t which, double *out, void *stream);

/*
 * Tensor-based hyper-diffusion (Section 2.4, Eq. 14-16,
 * L139-L154): H_q = (-1)^(alpha+1) (div tau grad)^alpha q with alpha = 2 on u, v, w, theta'
 * (H_u, H_theta of Eq. 1b-1c; rho' has none).  Readings Q30-Q33 of DESIGN.md:
 *   - L f = div(tau grad f) element-locally in the strong chain-rule form of the rest of the
 *     path, assembled as every tendency: H = -DSS(omega L( DSS(omega L q) )), tau entering each
 *     application (L145);
 *   - Eq. 15-16 with the element size along the i-th principal axis dx_i = 2 lambda_i^(1/2):
 *     tau = 4 dt_ref^(-1/2) J E diag(c_i^(1/2)) E^T J^T, E = eigenvectors of G = J^-1 J^-T by
 *     ASCENDING eigenvalue (c_1 acts along the longest principal axis of the element, c_3 along
 *     the shortest).  Where two eigenvalues coincide (e.g. hx = hy) the matching c_i must be
 *     equal, otherwise tau depends on an arbitrary choice of eigenvectors;
 *   - H is added to the assembled velocity / theta' tendency before the no-flux projection.
 *
 * numa_hd_init (enqueue only): builds tau[6] at every node from the stored metric terms into
 *   hd_workspace (>= numa_hd_workspace_bytes, 256-byte aligned, caller-owned, must outlive its
 *   use) and switches hyper-diffusion on for this context (all c_i = 0 switches it off):
 *   numa_step_rk3 / _graph / _host then include H in every stage (three more launches and one
 *   more 4-field DSS per stage).  c3 = (c_1, c_2, c_3) >= 0 dimensionless, dt_ref = the dt of Eq. 16.
 * numa_hyperdiffusion (enqueue only): the four-call route's step, to be called between
 *   numa_dss_or_flux and numa_apply_sources: rhs[1..4] += H(q), q and rhs [5][Ne][Mn].
 */
size_t numa_hd_workspace_bytes(const numa_params *p);
numa_status numa_hd_init(numa_ctx *ctx, const double *c3, double dt_ref, void *hd_workspace,
                         size_t workspace_bytes, void *stream);
numa_status numa_hyperdiffusion(numa_ctx *ctx, const double *q, double *rhs, void *stream);

/*
 * IMEX time integration (Section 2.3, Eq. 13):
 * dq/dt = [S(q) - L(q)] + L(q) with the fast acoustic / gravity waves in the linear operator L,
 * integrated by the additive Runge-Kutta scheme ARK2 (L133) whose implicit stages are solved by
 * matrix-free GMRES (L135).  The paper prints neither L nor the tableau; readings Q34-Q36:
 *   - L = the Jacobian of the S of Eq. 1 at the reference state q = 0:
 *       L_rho = -div(rho0 u);   L_u = -grad p'_L / rho0 - (rho'/rho0) g k,
 *       p'_L = gamma p0 (rho'/rho0 + theta'/theta0);   L_theta = -u . grad theta0,
 *     assembled like S, L_h = P(DSS(omega L_loc)), P the no-flux projection; heating, Coriolis
 *     and the sponge stay in the explicit part;
 *   - ARK2 of Giraldo, Kelly & Constantinescu 2013: 3 stages, gamma = 1 - 1/sqrt(2), explicit
 *     a21 = 2 gamma, a32 = (3 + 2 sqrt(2))/6, a31 = 1 - a32; implicit rows (gamma, gamma, 0) and
 *     b = (1/(2 sqrt 2), 1/(2 sqrt 2), gamma) (stiffly accurate), b shared by both parts;
 *   - GMRES(m) of Saad & Schultz 1986: modified Gram-Schmidt, Givens rotations, no
 *     preconditioner, initial guess = the stage's right-hand side, stop at ||r|| <= tol ||b||,
 *     inner product = Euclidean over the unique global nodes.
 *
 * numa_imex_init (enqueue only): m = Krylov vectors per restart cycle (the paper: "fewer than 20");
 *   imex_workspace (>= numa_imex_workspace_bytes(p, m), 256-byte aligned, caller-owned) holds the
 *   (m + 13) state-sized work vectors.
 * numa_linear_operator (enqueue only): Lq = L_h(q), both [5][Ne][Mn]; Lq must not alias q.
 * numa_step_ark2 (SYNCHRONISES `stream`: every GMRES inner product is read back by the host):
 *   n_steps ARK2 steps of size dt in place on q[5][Ne][Mn]; S is evaluated through the four-call
 *   route, including the hyper-diffusion H_q when numa_hd_init switched it on (H stays in the
 *   explicit part: dt times its spectral radius must respect the explicit stability limit).
 *   gmres_iterations / max_rel_residual (host pointers, may be NULL) receive the total
 *   number of Krylov iterations and the largest final relative residual of the implicit solves
 *   (the Givens estimate of a converged solve; the recomputed ||b - A x|| / ||b|| of one that ran
 *   out of restarts).  If any solve ends above tol the call still completes its n_steps, q holds
 *   their result, and the return value is NUMA_ERR_NOT_CONVERGED (text in numa_last_error).
 */
size_t numa_imex_workspace_bytes(const numa_params *p, int32_t m);
numa_status numa_imex_init(numa_ctx *ctx, int32_t m, void *imex_workspace, size_t workspace_bytes,
                           void *stream);
numa_status numa_linear_operator(numa_ctx *ctx, const double *q, double *Lq, void *stream);
numa_status numa_step_ark2(numa_ctx *ctx, double *q, const double *heating, double dt, int32_t n_steps,
                           double tol, int32_t max_restarts, int64_t *gmres_iterations,
                           double *max_rel_residual, void *stream);

/*
 * RI-velocity diagnostic (Eq. 18-22) on the device;
 * the paper computes it on the CPU after copying the state back (L172).  Readings Q25-Q29 of
 * DESIGN.md:
 *   - "height z" = a horizontal node level: level[e][n] in [0, n_levels) names the level of
 *     every local node (index data, like intma_cg);
 *   - Eq. 22: centroid of a level x_c = sum a |u| x / sum a |u| over the level's local nodes,
 *     |u| = (u^2+v^2+w^2)^(1/2), a = w_i w_j |x_xi y_eta - x_eta y_xi| the horizontal LGL
 *     quadrature weight (column-preserving meshes, L162-L168); a level at rest has no
 *     centroid and takes no part;
 *   - Eq. 20-21: u_theta = |(I - e_r e_r - e_z e_z) u|, e_r = r/|r|, r = (x-x_c, y-y_c, 0);
 *   - L360-L366: arithmetic mean of u_theta over the POINTS (unique global nodes; the first
 *     local copy) with s eps <= r < (s+1) eps, eps = r_max / n_strips (the paper: 50 strips),
 *     r >= r_max left out, e_r := 0 at r = 0;  Eq. 18: u_RI = max over (level, strip) holding a point.
 * Results are bitwise reproducible run to run (fixed-order centroid sums; the strip sums are
 * accumulated in 64-bit fixed point, exact to 2^-56 m/s per point).
 *
 * numa_ri_init (synchronises `stream`): builds, in ri_workspace, the area weights from
 *   xyz [3][Ne][Mn] and the level-sorted node and point lists.  The context must outlive the
 *   numa_ri.  NUMA_ERR_ARG if a level entry is outside [0, n_levels) or n_strips > 1024.
 * numa_ri_velocity (enqueue only): q [5][Ne][Mn] ->
 *   ubar     [n_levels][n_strips]  strip means (0 where count = 0)
 *   count    [n_levels][n_strips]  points per strip (int32)
 *   centroid [3][..]: n_levels pairs (x_c, y_c), then n_levels flags 1.0 / 0.0 (has a centroid)
 *   scalars  [3]: u_RI, max over points of (u^2+v^2)^(1/2) (Fig. 9's "maximum horizontal
 *            velocity"), and 1.0 if some u_theta was NaN or >= 4096 m/s (left out), else 0.0
 */
typedef struct numa_ri numa_ri;
size_t numa_ri_workspace_bytes(const numa_params *p, int32_t n_levels, int32_t n_strips);
numa_status numa_ri_init(numa_ctx *ctx, const double *xyz, const int32_t *level, int32_t n_levels,
                         int32_t n_strips, double r_max, void *ri_workspace, size_t workspace_bytes,
                         void *stream, numa_ri **out);
numa_status numa_ri_velocity(numa_ri *ri, const double *q, double *ubar, int32_t *count,
                             double *centroid, double *scalars, void *stream);
numa_status numa_ri_destroy(numa_ri *ri);

numa_status numa_destroy(numa_ctx *ctx);

/* Text of the last error of this context ("" if none).  ctx may be NULL: returns the text
 * of the last error raised without a context (e.g. inside numa_init_geometry). */
const char *numa_last_error(const numa_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* NUMA_B200_H */
