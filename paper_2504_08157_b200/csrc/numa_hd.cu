// Tensor-based hyper-diffusion (Section 2.4, Eq. 14-16,
// L139-L154):  H_q = -(div tau grad)^2 q on u, v, w, theta' (Eq. 1b-1c), alpha = 2 (L145).
// Readings Q30-Q33 of DESIGN.md:
//   - L f = div(tau grad f) element-locally in the strong, chain-rule form of the rest of the
//     path (Q2), assembled like every tendency: M^-1 DSS(wJ L f) = DSS(omega L f) (Eq. 11-12);
//     H = -DSS(omega L( DSS(omega L q) )): tau enters each application (L145);
//   - Eq. 16 with dx_i = 2 lambda_i^(1/2) makes nu_i / lambda_i = 4 (c_i / dt)^(1/2), so
//     tau = 4 dt^(-1/2) J E diag(c_i^(1/2)) E^T J^T  (Eq. 15), E = eigenvectors of
//     G = J^-1 J^-T by ascending eigenvalue (1/lambda_1 < 1/lambda_2 < 1/lambda_3);
//   - walls: H is part of the velocity tendency that the no-flux projection acts on (Q8).
#include <new>

#include "numa_internal.cuh"

namespace {

struct HdMap { const int32_t *pos; int npb; int BS; int64_t FS; };
__device__ __forceinline__ int64_t hd_shell_index(const HdMap &m, int64_t p)
{
    const int64_t b = p / m.npb;
    return b * m.BS + __ldg(m.pos + (int)(p - b * m.npb));
}

// ---- tau at every local node (block-shell order, like the metric terms it is made from) ----
// cyclic Jacobi on the symmetric 3x3 G; eigenvalues ascending, eigenvectors in the columns of V
__device__ void jacobi3(double A[3][3], double V[3][3], double ev[3])
{
    for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c) V[r][c] = (r == c) ? 1.0 : 0.0;
    for (int sweep = 0; sweep < 30; ++sweep) {
        const double off = fabs(A[0][1]) + fabs(A[0][2]) + fabs(A[1][2]);
        const double dia = fabs(A[0][0]) + fabs(A[1][1]) + fabs(A[2][2]);
        if (off <= 1e-300 + 1e-18 * dia) break;
        for (int p = 0; p < 2; ++p)
            for (int q = p + 1; q < 3; ++q) {
                if (A[p][q] == 0.0) continue;
                const double th = (A[q][q] - A[p][p]) / (2.0 * A[p][q]);
                const double t = ((th >= 0.0) ? 1.0 : -1.0) / (fabs(th) + sqrt(th * th + 1.0));
                const double c = 1.0 / sqrt(t * t + 1.0), s = t * c;
                for (int k = 0; k < 3; ++k) {   // A <- A R (columns p, q)
                    const double akp = A[k][p], akq = A[k][q];
                    A[k][p] = c * akp - s * akq; A[k][q] = s * akp + c * akq;
                }
                for (int k = 0; k < 3; ++k) {   // A <- R^T A (rows p, q)
                    const double apk = A[p][k], aqk = A[q][k];
                    A[p][k] = c * apk - s * aqk; A[q][k] = s * apk + c * aqk;
                }
                for (int k = 0; k < 3; ++k) {
                    const double vkp = V[k][p], vkq = V[k][q];
                    V[k][p] = c * vkp - s * vkq; V[k][q] = s * vkp + c * vkq;
                }
            }
    }
    for (int i = 0; i < 3; ++i) ev[i] = A[i][i];
    for (int a = 0; a < 2; ++a)          // sort ascending (columns of V follow)
        for (int b = 0; b < 2 - a; ++b)
            if (ev[b] > ev[b + 1]) {
                const double t = ev[b]; ev[b] = ev[b + 1]; ev[b + 1] = t;
                for (int k = 0; k < 3; ++k) { const double v = V[k][b]; V[k][b] = V[k][b + 1]; V[k][b + 1] = v; }
            }
}

__global__ void k_hd_tau(const double *__restrict__ met, double *__restrict__ tau, int64_t FS,
                         double s1, double s2, double s3)   // s_i = 4 (c_i / dt)^(1/2)
{
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= FS) return;
    double Ji[3][3];   // J^-1: row a = grad xi_a
    for (int a = 0; a < 3; ++a)
        for (int c = 0; c < 3; ++c) Ji[a][c] = met[(3 * a + c) * FS + t];
    const double det = Ji[0][0] * (Ji[1][1] * Ji[2][2] - Ji[1][2] * Ji[2][1]) -
                       Ji[0][1] * (Ji[1][0] * Ji[2][2] - Ji[1][2] * Ji[2][0]) +
                       Ji[0][2] * (Ji[1][0] * Ji[2][1] - Ji[1][1] * Ji[2][0]);
    if (!(det != 0.0)) {   // pad position of the block-shell tables
        for (int c = 0; c < 6; ++c) tau[c * FS + t] = 0.0;
        return;
    }
    // J = (J^-1)^-1: J[c][a] = d x_c / d xi_a  (adjugate / det)
    double J[3][3];
    const double id = 1.0 / det;
    J[0][0] = (Ji[1][1] * Ji[2][2] - Ji[1][2] * Ji[2][1]) * id;
    J[0][1] = (Ji[0][2] * Ji[2][1] - Ji[0][1] * Ji[2][2]) * id;
    J[0][2] = (Ji[0][1] * Ji[1][2] - Ji[0][2] * Ji[1][1]) * id;
    J[1][0] = (Ji[1][2] * Ji[2][0] - Ji[1][0] * Ji[2][2]) * id;
    J[1][1] = (Ji[0][0] * Ji[2][2] - Ji[0][2] * Ji[2][0]) * id;
    J[1][2] = (Ji[0][2] * Ji[1][0] - Ji[0][0] * Ji[1][2]) * id;
    J[2][0] = (Ji[1][0] * Ji[2][1] - Ji[1][1] * Ji[2][0]) * id;
    J[2][1] = (Ji[0][1] * Ji[2][0] - Ji[0][0] * Ji[2][1]) * id;
    J[2][2] = (Ji[0][0] * Ji[1][1] - Ji[0][1] * Ji[1][0]) * id;
    double T[3][3];
    if (s1 == s2 && s2 == s3) {
        // E diag(s) E^T = s I: tau = s J J^T, no eigenvectors needed
        for (int r = 0; r < 3; ++r)
            for (int c = 0; c < 3; ++c)
                T[r][c] = s1 * (J[r][0] * J[c][0] + J[r][1] * J[c][1] + J[r][2] * J[c][2]);
    } else {
        double G[3][3], V[3][3], ev[3];
        for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b)
                G[a][b] = Ji[a][0] * Ji[b][0] + Ji[a][1] * Ji[b][1] + Ji[a][2] * Ji[b][2];
        jacobi3(G, V, ev);
        const double sv[3] = {s1, s2, s3};
        double JE[3][3];
        for (int r = 0; r < 3; ++r)
            for (int i = 0; i < 3; ++i) JE[r][i] = J[r][0] * V[0][i] + J[r][1] * V[1][i] + J[r][2] * V[2][i];
        for (int r = 0; r < 3; ++r)
            for (int c = 0; c < 3; ++c)
                T[r][c] = sv[0] * JE[r][0] * JE[c][0] + sv[1] * JE[r][1] * JE[c][1] + sv[2] * JE[r][2] * JE[c][2];
    }
    tau[0 * FS + t] = T[0][0];
    tau[1 * FS + t] = 0.5 * (T[0][1] + T[1][0]);
    tau[2 * FS + t] = 0.5 * (T[0][2] + T[2][0]);
    tau[3 * FS + t] = T[1][1];
    tau[4 * FS + t] = 0.5 * (T[1][2] + T[2][1]);
    tau[5 * FS + t] = T[2][2];
}

// ---- omega * div(tau grad f) for 4 fields of one element per block ---------------------------
// f, out: natural [4][NL] (SHELL = false) or block-shell [4][FS] (SHELL = true); met, tau, omega:
// block-shell.  ACC: out += coef * P(omega L f) with the wall projection P on the first three
// fields (fused route); otherwise out = omega L f.
template <int Nq, bool SHELL, bool ACC>
__global__ void __launch_bounds__(256)
k_hd_lap(const double *__restrict__ f, double *out, int64_t fstride, const double *__restrict__ met,
         const double *__restrict__ tau, const double *__restrict__ omega,
         const uint8_t *__restrict__ face_bc, const __grid_constant__ LglTables tab, HdMap sm,
         double coef, int has_walls)
{
    constexpr int N2 = Nq * Nq, Mn = N2 * Nq;
    extern __shared__ double sh[];
    double *sf = sh;             // [4][Mn]
    double *sF = sh + 4 * Mn;    // [3][4][Mn]
    double *sD = sF + 12 * Mn;   // [Nq*Nq]
    const int64_t e = blockIdx.x;
    for (int t = threadIdx.x; t < Nq * Nq; t += blockDim.x) sD[t] = tab.D[t];
    for (int n = threadIdx.x; n < Mn; n += blockDim.x) {
        const int64_t p = e * Mn + n;
        const int64_t s = SHELL ? hd_shell_index(sm, p) : p;
#pragma unroll
        for (int m = 0; m < 4; ++m) sf[m * Mn + n] = f[m * fstride + s];
    }
    __syncthreads();
    for (int n = threadIdx.x; n < Mn; n += blockDim.x) {
        const int k = n / N2, j = (n - k * N2) / Nq, i = n - Nq * (j + Nq * k);
        const int64_t t = hd_shell_index(sm, e * Mn + n);
        double mt[9], tt[6];
#pragma unroll
        for (int c = 0; c < 9; ++c) mt[c] = met[c * sm.FS + t];
#pragma unroll
        for (int c = 0; c < 6; ++c) tt[c] = tau[c * sm.FS + t];
        double Di[Nq], Dj[Nq], Dk[Nq];   // this node's rows of D, reused by the 4 fields
#pragma unroll
        for (int l = 0; l < Nq; ++l) { Di[l] = sD[i * Nq + l]; Dj[l] = sD[j * Nq + l]; Dk[l] = sD[k * Nq + l]; }
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            const double *fm = sf + m * Mn;
            double fx = 0.0, fe = 0.0, fz = 0.0;
#pragma unroll
            for (int l = 0; l < Nq; ++l) {
                fx = fma(Di[l], fm[l + Nq * (j + Nq * k)], fx);
                fe = fma(Dj[l], fm[i + Nq * (l + Nq * k)], fe);
                fz = fma(Dk[l], fm[i + Nq * (j + Nq * l)], fz);
            }
            const double g0 = fx * mt[0] + fe * mt[3] + fz * mt[6];
            const double g1 = fx * mt[1] + fe * mt[4] + fz * mt[7];
            const double g2 = fx * mt[2] + fe * mt[5] + fz * mt[8];
            sF[(0 * 4 + m) * Mn + n] = tt[0] * g0 + tt[1] * g1 + tt[2] * g2;
            sF[(1 * 4 + m) * Mn + n] = tt[1] * g0 + tt[3] * g1 + tt[4] * g2;
            sF[(2 * 4 + m) * Mn + n] = tt[2] * g0 + tt[4] * g1 + tt[5] * g2;
        }
    }
    __syncthreads();
    for (int n = threadIdx.x; n < Mn; n += blockDim.x) {
        const int k = n / N2, j = (n - k * N2) / Nq, i = n - Nq * (j + Nq * k);
        const int64_t p = e * Mn + n;
        const int64_t t = hd_shell_index(sm, p);
        double mt[9];
#pragma unroll
        for (int c = 0; c < 9; ++c) mt[c] = met[c * sm.FS + t];
        const double om = omega[t];
        double r[4];
        double Di[Nq], Dj[Nq], Dk[Nq];
#pragma unroll
        for (int l = 0; l < Nq; ++l) { Di[l] = sD[i * Nq + l]; Dj[l] = sD[j * Nq + l]; Dk[l] = sD[k * Nq + l]; }
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            double div = 0.0;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const double *F = sF + (c * 4 + m) * Mn;
                double fx = 0.0, fe = 0.0, fz = 0.0;
#pragma unroll
                for (int l = 0; l < Nq; ++l) {
                    fx = fma(Di[l], F[l + Nq * (j + Nq * k)], fx);
                    fe = fma(Dj[l], F[i + Nq * (l + Nq * k)], fe);
                    fz = fma(Dk[l], F[i + Nq * (j + Nq * l)], fz);
                }
                div += fx * mt[0 + c] + fe * mt[3 + c] + fz * mt[6 + c];
            }
            r[m] = om * div;
        }
        const int64_t s = SHELL ? t : p;
        if (ACC) {
            if (has_walls) {
                const bool on_face = (i == 0) | (i == Nq - 1) | (j == 0) | (j == Nq - 1) | (k == 0) | (k == Nq - 1);
                if (on_face) {
                    const uint2 bcw = *reinterpret_cast<const uint2 *>(face_bc + e * 8);
                    if (bcw.x | bcw.y) {
                        uint8_t bc[8];
                        *reinterpret_cast<uint2 *>(bc) = bcw;
                        wall_project<Nq>(bc, i, j, k, mt, r[0], r[1], r[2]);
                    }
                }
            }
#pragma unroll
            for (int m = 0; m < 4; ++m) out[m * fstride + s] += coef * r[m];
        } else {
#pragma unroll
            for (int m = 0; m < 4; ++m) out[m * fstride + s] = r[m];
        }
    }
}

__global__ void k_hd_sub(double *__restrict__ r, const double *__restrict__ h, int64_t n)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) r[i] -= h[i];
}

template <int Nq, bool SHELL, bool ACC>
cudaError_t lap_launch(numa_ctx *c, const double *f, double *out, int64_t fstride, double coef, cudaStream_t s)
{
    constexpr size_t smem = sizeof(double) * (16 * Nq * Nq * Nq + Nq * Nq);
    cudaError_t e = cudaFuncSetAttribute(k_hd_lap<Nq, SHELL, ACC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const HdMap sm{c->shell.pos, c->shell.epb * (int)c->Mn, (int)c->shell.BS, c->shell.FS};
    constexpr int threads = (Nq * Nq * Nq + 31) / 32 * 32 < 256 ? (Nq * Nq * Nq + 31) / 32 * 32 : 256;
    k_hd_lap<Nq, SHELL, ACC><<<(unsigned)c->par.n_elem, threads, smem, s>>>(f, out, fstride, c->met, c->hd_tau, c->omega,
                                                                        c->face_bc, c->lgl, sm, coef, c->has_walls);
    return cudaGetLastError();
}

template <bool SHELL, bool ACC>
cudaError_t lap_dispatch(numa_ctx *c, const double *f, double *out, int64_t fstride, double coef, cudaStream_t s)
{
    switch (c->par.N) {
        case 2: return lap_launch<3, SHELL, ACC>(c, f, out, fstride, coef, s);
        case 3: return lap_launch<4, SHELL, ACC>(c, f, out, fstride, coef, s);
        case 4: return lap_launch<5, SHELL, ACC>(c, f, out, fstride, coef, s);
        case 5: return lap_launch<6, SHELL, ACC>(c, f, out, fstride, coef, s);
        case 6: return lap_launch<7, SHELL, ACC>(c, f, out, fstride, coef, s);
        case 7: return lap_launch<8, SHELL, ACC>(c, f, out, fstride, coef, s);
        case 8: return lap_launch<9, SHELL, ACC>(c, f, out, fstride, coef, s);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace

// fused route (numa_api.cu): h1 = DSS(omega L(qs[1..4])) into the context's buffer, block-shell
cudaError_t hd_stage_first(numa_ctx *c, const double *qs, cudaStream_t s)
{
    const int64_t FS = c->shell.FS;
    cudaError_t e;
    {
        LaunchScope ls(c, K_HD, s);
        e = lap_dispatch<true, false>(c, qs + FS, c->hd_buf, FS, 0.0, s);
    }
    if (e != cudaSuccess) return e;
    return launch_dss_classes(c, c->dss_int, c->hd_buf, FS, K_HD_DSS, s, 4);
}

// fused route: qout[1..4] += -b_dt P(omega L(h1)) (DSS partial sums; the stage's DSS completes them)
cudaError_t hd_stage_second(numa_ctx *c, double b_dt, double *qout, cudaStream_t s)
{
    const int64_t FS = c->shell.FS;
    LaunchScope ls(c, K_HD, s);
    return lap_dispatch<true, true>(c, c->hd_buf, qout + FS, FS, -b_dt, s);
}

extern "C" size_t numa_hd_workspace_bytes(const numa_params *p)
{
    if (!p || p->N < 2 || p->N > 8 || p->n_elem <= 0) return 0;
    const int64_t Nq = p->N + 1, Mn = Nq * Nq * Nq;
    const int epb = stage_epb(p->N);
    const int64_t BS = (epb * Mn + 31) / 32 * 32, FS = (p->n_elem + epb - 1) / epb * BS;
    const int64_t n = FS > p->n_elem * Mn ? FS : p->n_elem * Mn;
    return (size_t)(6 * FS + 8 * n) * sizeof(double) + 512;
}

extern "C" numa_status numa_hd_init(numa_ctx *ctx, const double *c3, double dt_ref, void *hd_workspace,
                                    size_t workspace_bytes, void *stream)
{
    if (!ctx) return NUMA_ERR_ARG;
    if (!c3 || !hd_workspace || !(dt_ref > 0.0) || !(c3[0] >= 0.0) || !(c3[1] >= 0.0) || !(c3[2] >= 0.0)) {
        ctx->err = "numa_hd_init: NULL argument, dt_ref <= 0 or a negative coefficient";
        return NUMA_ERR_ARG;
    }
    if (workspace_bytes < numa_hd_workspace_bytes(&ctx->par) || ((uintptr_t)hd_workspace & 255)) {
        ctx->err = "numa_hd_init: workspace too small or not 256-byte aligned";
        return NUMA_ERR_WORKSPACE;
    }
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != ctx->device) {
        ctx->err = "the current CUDA device is not the one this context was created on";
        cudaGetLastError();
        return NUMA_ERR_ARG;
    }
    cudaStream_t s = (cudaStream_t)stream;
    const int64_t FS = ctx->shell.FS;
    const int64_t n = FS > ctx->NL ? FS : ctx->NL;
    ctx->hd_tau = (double *)hd_workspace;
    ctx->hd_buf = ctx->hd_tau + 6 * FS;
    ctx->hd_buf2 = ctx->hd_buf + 4 * n;
    ctx->hd_on = (c3[0] > 0.0) || (c3[1] > 0.0) || (c3[2] > 0.0);
    if (ctx->graph) { cudaGraphExecDestroy(ctx->graph); ctx->graph = nullptr; }   // the step changes
    const double sc = 4.0 / sqrt(dt_ref);
    k_hd_tau<<<(unsigned)((FS + 127) / 128), 128, 0, s>>>(ctx->met, ctx->hd_tau, FS, sc * sqrt(c3[0]),
                                                          sc * sqrt(c3[1]), sc * sqrt(c3[2]));
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemsetAsync(ctx->hd_buf, 0, (size_t)8 * n * sizeof(double), s);
    ctx->launches += 1;
    if (e != cudaSuccess) { ctx->err = cudaGetErrorString(e); cudaGetLastError(); return NUMA_ERR_CUDA; }
    return NUMA_OK;
}

extern "C" numa_status numa_hyperdiffusion(numa_ctx *ctx, const double *q, double *rhs, void *stream)
{
    if (!ctx || !q || !rhs) { if (ctx) ctx->err = "numa_hyperdiffusion: NULL argument"; return NUMA_ERR_ARG; }
    if (!ctx->hd_tau) { ctx->err = "numa_hyperdiffusion: call numa_hd_init first"; return NUMA_ERR_ARG; }
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != ctx->device) {
        ctx->err = "the current CUDA device is not the one this context was created on";
        cudaGetLastError();
        return NUMA_ERR_ARG;
    }
    if (!ctx->hd_on) return NUMA_OK;
    cudaStream_t s = (cudaStream_t)stream;
    const int64_t NL = ctx->NL;
    cudaError_t e;
    {
        LaunchScope ls(ctx, K_HD, s);
        e = lap_dispatch<false, false>(ctx, q + NL, ctx->hd_buf, NL, 0.0, s);
    }
    if (e == cudaSuccess) e = launch_dss_classes(ctx, ctx->dss_nat, ctx->hd_buf, NL, K_HD_DSS, s, 4);
    if (e == cudaSuccess) {
        LaunchScope ls(ctx, K_HD, s);
        e = lap_dispatch<false, false>(ctx, ctx->hd_buf, ctx->hd_buf2, NL, 0.0, s);
    }
    if (e == cudaSuccess) e = launch_dss_classes(ctx, ctx->dss_nat, ctx->hd_buf2, NL, K_HD_DSS, s, 4);
    if (e == cudaSuccess) {
        // H = -DSS(omega L(h1)):  rhs[1..4] += H
        k_hd_sub<<<(unsigned)((4 * NL + 255) / 256), 256, 0, s>>>(rhs + NL, ctx->hd_buf2, 4 * NL);
        ctx->launches += 1;
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) { ctx->err = cudaGetErrorString(e); cudaGetLastError(); return NUMA_ERR_CUDA; }
    return NUMA_OK;
}
