// IMEX path (Section 2.3, Eq. 13): the linear operator
// L of the splitting dq/dt = [S(q) - L(q)] + L(q), the ARK2 additive Runge-Kutta step and the
// matrix-free restarted GMRES that solves its implicit stages ("the linearized operator is
// computed on the fly with no information precomputed or stored. The only memory required is to
// store the Krylov vectors", L135).  Readings Q34-Q36 of DESIGN.md:
//   Q34  L = the Jacobian of the S of Eq. 1 at the hydrostatic reference state q = 0:
//        L_rho = -div(rho0 u);  L_u = -grad p'_L / rho0 - (rho'/rho0) g k,
//        p'_L = gamma p0 (rho'/rho0 + theta'/theta0);  L_theta = -u . grad theta0;
//        assembled like S: L_h = P(DSS(omega L_loc)), P the no-flux projection;
//   Q35  ARK2 = the three-stage scheme of Giraldo, Kelly & Constantinescu 2013 (tableau below);
//   Q36  GMRES(m) of Saad & Schultz 1986: modified Gram-Schmidt, Givens rotations, no
//        preconditioner, initial guess = the stage's right-hand side, inner product = the
//        Euclidean one over the unique global nodes (local copies weighted 1/multiplicity).
// All vectors are natural-layout states [5][Ne][Mn]; the nonlinear S is the four-call route.
#include <cstdio>
#include <cmath>
#include <new>
#include <vector>

#include "numa_internal.cuh"

namespace {

struct ImMap { const int32_t *pos; int npb; int BS; int64_t FS; };
__device__ __forceinline__ int64_t im_shell_index(const ImMap &m, int64_t p)
{
    const int64_t b = p / m.npb;
    return b * m.BS + __ldg(m.pos + (int)(p - b * m.npb));
}

// omega * L_loc(q), one element per block (thread-per-node contractions as in k_rhs)
template <int Nq>
__global__ void __launch_bounds__(256)
k_linop(const double *__restrict__ q, double *__restrict__ out, int64_t NL,
        const double *__restrict__ ref3, const double *__restrict__ met,
        const double *__restrict__ omega, const __grid_constant__ LglTables tab, ImMap sm, double g,
        double gamma)
{
    constexpr int N2 = Nq * Nq, Mn = N2 * Nq;
    extern __shared__ double sh[];
    double *pl = sh, *th0 = sh + Mn, *Fx = sh + 2 * Mn, *Fy = sh + 3 * Mn, *Fz = sh + 4 * Mn, *sD = sh + 5 * Mn;
    const int64_t e = blockIdx.x;
    for (int t = threadIdx.x; t < Nq * Nq; t += blockDim.x) sD[t] = tab.D[t];
    const double th0e = ref3[sm.FS + im_shell_index(sm, e * Mn)];
    for (int n = threadIdx.x; n < Mn; n += blockDim.x) {
        const int64_t p = e * Mn + n, t = im_shell_index(sm, p);
        const double rho0 = ref3[t], theta0 = ref3[sm.FS + t], p0 = ref3[2 * sm.FS + t];
        pl[n] = gamma * p0 * (q[p] / rho0 + q[4 * NL + p] / theta0);
        th0[n] = theta0 - th0e;
        Fx[n] = rho0 * q[1 * NL + p];
        Fy[n] = rho0 * q[2 * NL + p];
        Fz[n] = rho0 * q[3 * NL + p];
    }
    __syncthreads();
    for (int n = threadIdx.x; n < Mn; n += blockDim.x) {
        const int k = n / N2, j = (n - k * N2) / Nq, i = n - Nq * (j + Nq * k);
        const int64_t p = e * Mn + n, t = im_shell_index(sm, p);
        double m[9];
#pragma unroll
        for (int c = 0; c < 9; ++c) m[c] = met[c * sm.FS + t];
        double d[5][3];
        double Di[Nq], Dj[Nq], Dk[Nq];
#pragma unroll
        for (int l = 0; l < Nq; ++l) { Di[l] = sD[i * Nq + l]; Dj[l] = sD[j * Nq + l]; Dk[l] = sD[k * Nq + l]; }
#pragma unroll
        for (int f = 0; f < 5; ++f) {
            const double *a = sh + f * Mn;
            double fx = 0.0, fe = 0.0, fz = 0.0;
#pragma unroll
            for (int l = 0; l < Nq; ++l) {
                fx = fma(Di[l], a[l + Nq * (j + Nq * k)], fx);
                fe = fma(Dj[l], a[i + Nq * (l + Nq * k)], fe);
                fz = fma(Dk[l], a[i + Nq * (j + Nq * l)], fz);
            }
            d[f][0] = fx; d[f][1] = fe; d[f][2] = fz;
        }
        const double rho0 = ref3[t], om = omega[t];
        const double u = q[1 * NL + p], v = q[2 * NL + p], w = q[3 * NL + p];
        double gp[3], gt[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            gp[c] = d[0][0] * m[0 + c] + d[0][1] * m[3 + c] + d[0][2] * m[6 + c];
            gt[c] = d[1][0] * m[0 + c] + d[1][1] * m[3 + c] + d[1][2] * m[6 + c];
        }
        double div = 0.0;
#pragma unroll
        for (int c = 0; c < 3; ++c) div += d[2 + c][0] * m[0 + c] + d[2 + c][1] * m[3 + c] + d[2 + c][2] * m[6 + c];
        out[0 * NL + p] = om * (-div);
        out[1 * NL + p] = om * (-gp[0] / rho0);
        out[2 * NL + p] = om * (-gp[1] / rho0);
        out[3 * NL + p] = om * (-gp[2] / rho0 - (q[p] / rho0) * g);
        out[4 * NL + p] = om * (-(u * gt[0] + v * gt[1] + w * gt[2]));
    }
}

// no-flux projection of the velocity part of r (natural layout), elements with wall faces only
template <int Nq>
__global__ void k_imex_walls(double *__restrict__ r, int64_t NL, const double *__restrict__ met,
                             const uint8_t *__restrict__ face_bc, ImMap sm)
{
    constexpr int N2 = Nq * Nq, Mn = N2 * Nq;
    const int64_t e = blockIdx.x;
    const uint2 bcw = *reinterpret_cast<const uint2 *>(face_bc + e * 8);
    if (!(bcw.x | bcw.y)) return;
    uint8_t bc[8];
    *reinterpret_cast<uint2 *>(bc) = bcw;
    for (int n = threadIdx.x; n < Mn; n += blockDim.x) {
        const int k = n / N2, j = (n - k * N2) / Nq, i = n - Nq * (j + Nq * k);
        const bool on_face = (i == 0) | (i == Nq - 1) | (j == 0) | (j == Nq - 1) | (k == 0) | (k == Nq - 1);
        if (!on_face) continue;
        const int64_t p = e * Mn + n, t = im_shell_index(sm, p);
        double m[9];
#pragma unroll
        for (int c = 0; c < 9; ++c) m[c] = met[c * sm.FS + t];
        double ru = r[1 * NL + p], rv = r[2 * NL + p], rw = r[3 * NL + p];
        wall_project<Nq>(bc, i, j, k, m, ru, rv, rw);
        r[1 * NL + p] = ru; r[2 * NL + p] = rv; r[3 * NL + p] = rw;
    }
}

__global__ void k_inv_mult(const int32_t *__restrict__ start, const int32_t *__restrict__ copies,
                           double *__restrict__ inv_mult, int64_t NG)
{
    const int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= NG) return;
    const int s = start[g], c = start[g + 1] - s;
    for (int a = 0; a < c; ++a) inv_mult[copies[s + a]] = 1.0 / (double)c;
}

// out = c0 x0 + c1 x1 + c2 x2 + c3 x3 (null pointers skipped); out may alias any x
__global__ void k_lincomb(double *out, int64_t n, double c0, const double *x0, double c1, const double *x1,
                          double c2, const double *x2, double c3, const double *x3)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        double s = 0.0;
        if (x0) s = c0 * x0[i];
        if (x1) s = fma(c1, x1[i], s);
        if (x2) s = fma(c2, x2[i], s);
        if (x3) s = fma(c3, x3[i], s);
        out[i] = s;
    }
}

// <a, b> = sum over fields and local nodes of inv_mult a b: fixed grid, fixed-order tree
constexpr int DOT_BLOCKS = 592, DOT_THREADS = 256;
__global__ void __launch_bounds__(DOT_THREADS)
k_dot_partial(const double *__restrict__ a, const double *__restrict__ b, const double *__restrict__ inv_mult,
              int64_t NL, double *__restrict__ partial)
{
    __shared__ double sh[DOT_THREADS];
    double s = 0.0;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < NL; p += stride) {
        double t = 0.0;
#pragma unroll
        for (int f = 0; f < 5; ++f) t = fma(a[f * NL + p], b[f * NL + p], t);
        s = fma(inv_mult[p], t, s);
    }
    sh[threadIdx.x] = s;
    __syncthreads();
    for (int w = DOT_THREADS / 2; w > 0; w >>= 1) {
        if (threadIdx.x < w) sh[threadIdx.x] += sh[threadIdx.x + w];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];
}
__global__ void __launch_bounds__(DOT_THREADS)
k_dot_final(const double *__restrict__ partial, int n, double *__restrict__ out)
{
    __shared__ double sh[DOT_THREADS];
    double s = 0.0;
    for (int i = threadIdx.x; i < n; i += DOT_THREADS) s += partial[i];
    sh[threadIdx.x] = s;
    __syncthreads();
    for (int w = DOT_THREADS / 2; w > 0; w >>= 1) {
        if (threadIdx.x < w) sh[threadIdx.x] += sh[threadIdx.x + w];
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = sh[0];
}

template <int Nq>
cudaError_t linop_launch(numa_ctx *c, const double *q, double *out, cudaStream_t s)
{
    constexpr size_t smem = sizeof(double) * (5 * Nq * Nq * Nq + Nq * Nq);
    cudaError_t e = cudaFuncSetAttribute(k_linop<Nq>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const ImMap sm{c->shell.pos, c->shell.epb * (int)c->Mn, (int)c->shell.BS, c->shell.FS};
    constexpr int threads = (Nq * Nq * Nq + 31) / 32 * 32 < 256 ? (Nq * Nq * Nq + 31) / 32 * 32 : 256;
    {
        LaunchScope ls(c, K_LINOP, s);
        k_linop<Nq><<<(unsigned)c->par.n_elem, threads, smem, s>>>(q, out, c->NL, c->ref3, c->met, c->omega, c->lgl, sm,
                                                              c->par.g, c->gamma);
    }
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    e = launch_dss_classes(c, c->dss_nat, out, c->NL, K_DSS, s);
    if (e != cudaSuccess) return e;
    if (c->has_walls) {
        LaunchScope ls(c, K_LINOP, s);
        k_imex_walls<Nq><<<(unsigned)c->par.n_elem, 128, 0, s>>>(out, c->NL, c->met, c->face_bc, sm);
        e = cudaGetLastError();
    }
    return e;
}

cudaError_t linop(numa_ctx *c, const double *q, double *out, cudaStream_t s)
{
    switch (c->par.N) {
        case 2: return linop_launch<3>(c, q, out, s);
        case 3: return linop_launch<4>(c, q, out, s);
        case 4: return linop_launch<5>(c, q, out, s);
        case 5: return linop_launch<6>(c, q, out, s);
        case 6: return linop_launch<7>(c, q, out, s);
        case 7: return linop_launch<8>(c, q, out, s);
        case 8: return linop_launch<9>(c, q, out, s);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace

// ---- host side ----------------------------------------------------------------------------------
// ARK2 (Q35): gamma = 1 - 1/sqrt(2); explicit A, implicit At (first stage explicit, then SDIRK), b shared
static const double kG = 1.0 - 1.0 / 1.4142135623730951;
static const double kA32 = (3.0 + 2.0 * 1.4142135623730951) / 6.0;
static const double kB12 = 1.0 / (2.0 * 1.4142135623730951);
static const double kArkA[3][3] = {{0, 0, 0}, {2.0 * kG, 0, 0}, {1.0 - kA32, kA32, 0}};
static const double kArkAt[3][3] = {{0, 0, 0}, {kG, kG, 0}, {kB12, kB12, kG}};
static const double kArkB[3] = {kB12, kB12, kG};

static inline size_t im_al(size_t x) { return (x + 255) & ~(size_t)255; }
static inline int imex_n_vec(int m) { return (m + 1) + 12; }   // Krylov basis + w, r, and the ARK work vectors

extern "C" size_t numa_imex_workspace_bytes(const numa_params *p, int32_t m)
{
    if (!p || p->N < 2 || p->N > 8 || p->n_elem <= 0 || m < 1 || m > 200) return 0;
    const int64_t Nq = p->N + 1, NL = p->n_elem * Nq * Nq * Nq;
    return im_al((size_t)NL * 8) + (size_t)imex_n_vec(m) * im_al((size_t)5 * NL * 8) + im_al((DOT_BLOCKS + 8) * 8);
}

extern "C" numa_status numa_imex_init(numa_ctx *ctx, int32_t m, void *workspace, size_t workspace_bytes, void *stream)
{
    if (!ctx) return NUMA_ERR_ARG;
    if (!workspace || m < 1 || m > 200) { ctx->err = "numa_imex_init: NULL workspace or m outside 1..200"; return NUMA_ERR_ARG; }
    if (workspace_bytes < numa_imex_workspace_bytes(&ctx->par, m) || ((uintptr_t)workspace & 255)) {
        ctx->err = "numa_imex_init: workspace too small or not 256-byte aligned";
        return NUMA_ERR_WORKSPACE;
    }
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != ctx->device) {
        ctx->err = "the current CUDA device is not the one this context was created on";
        cudaGetLastError();
        return NUMA_ERR_ARG;
    }
    ctx->imex_ws = (char *)workspace;
    ctx->imex_m = m;
    cudaStream_t s = (cudaStream_t)stream;
    const int64_t NG = ctx->par.n_global;
    k_inv_mult<<<(unsigned)((NG + 255) / 256), 256, 0, s>>>(ctx->dss_nat.start, ctx->dss_nat.copies,
                                                          (double *)ctx->imex_ws, NG);
    ctx->launches += 1;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { ctx->err = cudaGetErrorString(e); return NUMA_ERR_CUDA; }
    return NUMA_OK;
}

extern "C" numa_status numa_linear_operator(numa_ctx *ctx, const double *q, double *Lq, void *stream)
{
    if (!ctx || !q || !Lq || q == Lq) { if (ctx) ctx->err = "numa_linear_operator: NULL argument or Lq aliases q"; return NUMA_ERR_ARG; }
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != ctx->device) {
        ctx->err = "the current CUDA device is not the one this context was created on";
        cudaGetLastError();
        return NUMA_ERR_ARG;
    }
    cudaError_t e = linop(ctx, q, Lq, (cudaStream_t)stream);
    if (e != cudaSuccess) { ctx->err = cudaGetErrorString(e); cudaGetLastError(); return NUMA_ERR_CUDA; }
    return NUMA_OK;
}

namespace {

struct Imex {
    numa_ctx *c; cudaStream_t s; int64_t NL, n5; double *inv_mult, *partial, *d_scalar;
    cudaError_t err = cudaSuccess;
    void chk(cudaError_t e) { if (err == cudaSuccess && e != cudaSuccess) err = e; }
    void lincomb(double *out, double c0, const double *x0, double c1 = 0, const double *x1 = nullptr, double c2 = 0,
                 const double *x2 = nullptr, double c3 = 0, const double *x3 = nullptr)
    {
        {
            LaunchScope ls(c, K_VEC, s);
            k_lincomb<<<1184, 256, 0, s>>>(out, n5, c0, x0, c1, x1, c2, x2, c3, x3);
        }
        chk(cudaGetLastError());
    }
    double dot(const double *a, const double *b)
    {
        {
            LaunchScope ls(c, K_VEC, s);
            k_dot_partial<<<DOT_BLOCKS, DOT_THREADS, 0, s>>>(a, b, inv_mult, NL, partial);
            k_dot_final<<<1, DOT_THREADS, 0, s>>>(partial, DOT_BLOCKS, d_scalar);
            c->launches += 1;
        }
        chk(cudaGetLastError());
        double h = 0.0;
        chk(cudaMemcpyAsync(&h, d_scalar, 8, cudaMemcpyDeviceToHost, s));
        chk(cudaStreamSynchronize(s));
        return h;
    }
    void L(const double *q, double *out) { chk(linop(c, q, out, s)); }
    // S_h(q): the four-call route (volume, DSS, sources + walls)
    void S(const double *q, const double *heat, double *out)
    {
        chk(launch_rhs(c, q, out, s));
        chk(launch_dss_classes(c, c->dss_nat, out, NL, K_DSS, s));
        // H_q of Eq. 1 when numa_hd_init switched it on: added to the assembled tendency before the
        // sources and the no-flux projection, as in the four-call route; explicit part of the splitting
        if (c->hd_on && numa_hyperdiffusion(c, q, out, s) != NUMA_OK) chk(cudaErrorUnknown);
        chk(launch_sources(c, q, heat, out, s));
    }
};

// (I - a L) x = b by restarted GMRES(m) from x = b; returns inner iterations, *rel = last relative residual
int gmres_solve(Imex &I, double a, const double *b, double *x, double **V, double *w, double *r, int m, double tol,
                int max_restarts, double *rel_out)
{
    auto apply = [&](const double *v, double *out) { I.L(v, out); I.lincomb(out, 1.0, v, -a, out); };
    I.lincomb(x, 1.0, b);
    const double bnorm = std::sqrt(I.dot(b, b));
    int its = 0;
    double rel = 0.0;
    if (bnorm == 0.0) { *rel_out = 0.0; return 0; }
    std::vector<double> H((size_t)(m + 1) * m), cs(m), sn(m), g(m + 1), y(m);
    for (int restart = 0; restart <= max_restarts && I.err == cudaSuccess; ++restart) {
        apply(x, r);
        I.lincomb(r, 1.0, b, -1.0, r);
        const double beta = std::sqrt(I.dot(r, r));
        rel = beta / bnorm;
        if (rel <= tol) break;
        I.lincomb(V[0], 1.0 / beta, r);
        std::fill(H.begin(), H.end(), 0.0);
        std::fill(g.begin(), g.end(), 0.0);
        g[0] = beta;
        int k_used = 0;
        for (int k = 0; k < m && I.err == cudaSuccess; ++k) {
            apply(V[k], w);
            for (int i = 0; i <= k; ++i) {
                const double h = I.dot(w, V[i]);
                H[(size_t)i * m + k] = h;
                I.lincomb(w, 1.0, w, -h, V[i]);
            }
            const double hn = std::sqrt(I.dot(w, w));
            H[(size_t)(k + 1) * m + k] = hn;
            for (int i = 0; i < k; ++i) {
                const double t = cs[i] * H[(size_t)i * m + k] + sn[i] * H[(size_t)(i + 1) * m + k];
                H[(size_t)(i + 1) * m + k] = -sn[i] * H[(size_t)i * m + k] + cs[i] * H[(size_t)(i + 1) * m + k];
                H[(size_t)i * m + k] = t;
            }
            const double d = std::hypot(H[(size_t)k * m + k], H[(size_t)(k + 1) * m + k]);
            // breakdown: column k of the rotated Hessenberg matrix is zero, so V[k] adds nothing to
            // the span; the solution is taken from the first k columns (k_used stays k)
            if (d == 0.0) break;
            cs[k] = H[(size_t)k * m + k] / d; sn[k] = H[(size_t)(k + 1) * m + k] / d;
            H[(size_t)k * m + k] = d; H[(size_t)(k + 1) * m + k] = 0.0;
            g[k + 1] = -sn[k] * g[k]; g[k] = cs[k] * g[k];
            ++its;
            k_used = k + 1;
            rel = std::fabs(g[k + 1]) / bnorm;
            if (rel <= tol) break;
            if (k + 1 < m) I.lincomb(V[k + 1], 1.0 / hn, w);
        }
        for (int i = k_used - 1; i >= 0; --i) {
            double t = g[i];
            for (int j = i + 1; j < k_used; ++j) t -= H[(size_t)i * m + j] * y[j];
            y[i] = t / H[(size_t)i * m + i];
        }
        for (int i = 0; i < k_used; ++i) I.lincomb(x, 1.0, x, y[i], V[i]);
        if (rel <= tol) break;
    }
    if (rel > tol && I.err == cudaSuccess) {
        // restarts exhausted: report the true residual ||b - A x|| / ||b||, not the Givens estimate
        apply(x, r);
        I.lincomb(r, 1.0, b, -1.0, r);
        rel = std::sqrt(I.dot(r, r)) / bnorm;
    }
    *rel_out = rel;
    return its;
}

}  // namespace

extern "C" numa_status numa_step_ark2(numa_ctx *ctx, double *q, const double *heating, double dt, int32_t n_steps,
                                      double tol, int32_t max_restarts, int64_t *gmres_iterations,
                                      double *max_rel_residual, void *stream)
{
    if (!ctx || !q) { if (ctx) ctx->err = "numa_step_ark2: NULL argument"; return NUMA_ERR_ARG; }
    if (!ctx->imex_ws) { ctx->err = "numa_step_ark2: call numa_imex_init first"; return NUMA_ERR_ARG; }
    if (n_steps < 0 || !(tol > 0.0) || max_restarts < 0) { ctx->err = "numa_step_ark2: bad n_steps, tol or max_restarts"; return NUMA_ERR_ARG; }
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != ctx->device) {
        ctx->err = "the current CUDA device is not the one this context was created on";
        cudaGetLastError();
        return NUMA_ERR_ARG;
    }
    const int m = ctx->imex_m;
    const int64_t NL = ctx->NL;
    const size_t vb = im_al((size_t)5 * NL * 8);
    char *base = ctx->imex_ws + im_al((size_t)NL * 8);
    std::vector<double *> vec(imex_n_vec(m));
    for (size_t i = 0; i < vec.size(); ++i) vec[i] = (double *)(base + i * vb);
    double **V = vec.data();                       // V[0..m]
    double *w = vec[m + 1], *r = vec[m + 2], *R = vec[m + 3], *Q = vec[m + 4], *Sv = vec[m + 5], *Lv = vec[m + 6],
           *acc = vec[m + 7], *Nst[2] = {vec[m + 8], vec[m + 9]}, *Lst[2] = {vec[m + 10], vec[m + 11]};
    double *tail = (double *)(base + vec.size() * vb);
    Imex I{ctx, (cudaStream_t)stream, NL, 5 * NL, (double *)ctx->imex_ws, tail, tail + DOT_BLOCKS};
    int64_t its_total = 0;
    double rel_max = 0.0;
    for (int step = 0; step < n_steps && I.err == cudaSuccess; ++step) {
        I.lincomb(acc, 1.0, q);
        for (int i = 0; i < 3; ++i) {
            // R_i = q + dt sum_{j<i} (a_ij N_j + at_ij L_j)
            I.lincomb(R, 1.0, q);
            for (int j = 0; j < i; ++j) I.lincomb(R, 1.0, R, dt * kArkA[i][j], Nst[j], dt * kArkAt[i][j], Lst[j]);
            const double aii = kArkAt[i][i];
            const double *Qi = R;
            if (aii != 0.0) {
                double rel = 0.0;
                its_total += gmres_solve(I, dt * aii, R, Q, V, w, r, m, tol, max_restarts, &rel);
                rel_max = rel > rel_max ? rel : rel_max;
                Qi = Q;
            }
            I.S(Qi, heating, Sv);
            I.lincomb(acc, 1.0, acc, dt * kArkB[i], Sv);
            if (i < 2) {
                I.L(Qi, Lst[i]);
                I.lincomb(Nst[i], 1.0, Sv, -1.0, Lst[i]);
            }
        }
        I.lincomb(q, 1.0, acc);
    }
    (void)Lv;
    if (gmres_iterations) *gmres_iterations = its_total;
    if (max_rel_residual) *max_rel_residual = rel_max;
    if (I.err == cudaSuccess) I.chk(cudaStreamSynchronize(I.s));
    if (I.err != cudaSuccess) { ctx->err = cudaGetErrorString(I.err); cudaGetLastError(); return NUMA_ERR_CUDA; }
    if (!(rel_max <= tol)) {
        char buf[200];
        snprintf(buf, sizeof buf, "numa_step_ark2: GMRES left a relative residual of %.3e > tol = %.3e after %d restart(s) "
                 "of %d vectors; q holds the steps taken with those solves", rel_max, tol, (int)max_restarts, m);
        ctx->err = buf;
        return NUMA_ERR_NOT_CONVERGED;
    }
    return NUMA_OK;
}
