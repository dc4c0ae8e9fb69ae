// CUDA kernels (sm_100a) of the hot path: element-local Euler tendency (Eq. 1-3,
// Alg. 1-2), deterministic DSS (Alg. 3), pointwise sources + no-flux walls, RK stage update,
// and the setup kernel for the metric terms.  FP64 everywhere.
//
// Layout of the API arrays: f[m][e][n], n = i + Nq*(j + Nq*k) (the paper's q_e(i,j,k,e,m), L205).
// The library's own tables (met, omega, ref3, sponge) are kept in the block-shell order of the
// fused route (ShellLayout); the kernels of this file reach them through shell_index().
#include "numa_internal.cuh"

namespace {

// position of natural local node p in a block-shell array (ShellLayout, numa_internal.cuh)
struct ShellMap { const int32_t *pos; int npb; int BS; int64_t FS; };
__device__ __forceinline__ int64_t shell_index(const ShellMap &m, int64_t p)
{
    const int64_t b = p / m.npb;
    return b * m.BS + __ldg(m.pos + (int)(p - b * m.npb));
}

template <int N>
struct Shape {
    static constexpr int Nq = N + 1;
    static constexpr int Mn = Nq * Nq * Nq;
    // elements per block so that a block has ~256 threads (one thread per node)
    static constexpr int EPB = (Mn >= 192) ? 1 : (256 / Mn);
    static constexpr int THREADS = ((EPB * Mn + 31) / 32) * 32;
};

// ---------------------------------------------------------------------------------------
// Alg. 2 (L227-L250): the three reference-space derivatives of one nodal field held in
// shared memory; Di/Dj/Dk are this thread's rows D[i][:], D[j][:], D[k][:] in registers.
// ---------------------------------------------------------------------------------------
template <int Nq>
__device__ __forceinline__ void ref_derivs(const double *__restrict__ f, int i, int j, int k,
                                           const double (&Di)[Nq], const double (&Dj)[Nq],
                                           const double (&Dk)[Nq], double &fx, double &fe,
                                           double &fz)
{
    const double *fi = f + Nq * (j + Nq * k);       // f(l, j, k), stride 1
    const double *fj = f + i + Nq * Nq * k;         // f(i, l, k), stride Nq
    const double *fk = f + i + Nq * j;              // f(i, j, l), stride Nq*Nq
    double a = 0.0, b = 0.0, c = 0.0;
#pragma unroll
    for (int l = 0; l < Nq; ++l) {
        a = fma(Di[l], fi[l], a);
        b = fma(Dj[l], fj[l * Nq], b);
        c = fma(Dk[l], fk[l * Nq * Nq], c);
    }
    fx = a; fe = b; fz = c;
}

// Difference form used for the geometry only: sum_{l != i} D[i][l] (f_l - f_i); exact zero
// for a coordinate that is constant along the direction (Q4).
template <int Nq>
__device__ __forceinline__ void ref_derivs_diff(const double *__restrict__ f, int i, int j, int k,
                                                const double (&Di)[Nq], const double (&Dj)[Nq],
                                                const double (&Dk)[Nq], double &fx, double &fe,
                                                double &fz)
{
    const double *fi = f + Nq * (j + Nq * k);
    const double *fj = f + i + Nq * Nq * k;
    const double *fk = f + i + Nq * j;
    const double f0 = f[i + Nq * (j + Nq * k)];
    double a = 0.0, b = 0.0, c = 0.0;
#pragma unroll
    for (int l = 0; l < Nq; ++l) {
        if (l != i) a = fma(Di[l], fi[l] - f0, a);
        if (l != j) b = fma(Dj[l], fj[l * Nq] - f0, b);
        if (l != k) c = fma(Dk[l], fk[l * Nq * Nq] - f0, c);
    }
    fx = a; fe = b; fz = c;
}

// Per-node tendency S(q) of Eq. 1 with H = 0, given the element's nodal work arrays in
// shared memory: sh[0..8] = p', u, v, w, theta', theta0, Fx, Fy, Fz (each Mn doubles).
// m[9] = d xi_a / d x_c at this node.  Uses the contravariant velocity U^a = u . grad xi_a so
// that u . grad f = sum_a U^a f_{xi_a} (same value as the chain-rule form up to rounding).
template <int N>
__device__ __forceinline__ void node_tendency(const double *__restrict__ sh, int i, int j, int k,
                                              const double (&Di)[N + 1], const double (&Dj)[N + 1],
                                              const double (&Dk)[N + 1], const double (&m)[9],
                                              double rhop, double rho0, double g, double (&S)[5])
{
    constexpr int Nq = N + 1, Mn = Nq * Nq * Nq;
    const int n = i + Nq * (j + Nq * k);
    const double u = sh[1 * Mn + n], v = sh[2 * Mn + n], w = sh[3 * Mn + n];
    const double Ux = u * m[0] + v * m[1] + w * m[2];
    const double Ue = u * m[3] + v * m[4] + w * m[5];
    const double Uz = u * m[6] + v * m[7] + w * m[8];
    const double rho = rho0 + rhop;
    const double irho = 1.0 / rho;
    double fx, fe, fz;
    // pressure gradient (chain rule, Q2)
    ref_derivs<Nq>(sh + 0 * Mn, i, j, k, Di, Dj, Dk, fx, fe, fz);
    const double px = fx * m[0] + fe * m[3] + fz * m[6];
    const double py = fx * m[1] + fe * m[4] + fz * m[7];
    const double pz = fx * m[2] + fe * m[5] + fz * m[8];
    // advection of u, v, w
    ref_derivs<Nq>(sh + 1 * Mn, i, j, k, Di, Dj, Dk, fx, fe, fz);
    S[1] = -(Ux * fx + Ue * fe + Uz * fz) - px * irho;
    ref_derivs<Nq>(sh + 2 * Mn, i, j, k, Di, Dj, Dk, fx, fe, fz);
    S[2] = -(Ux * fx + Ue * fe + Uz * fz) - py * irho;
    ref_derivs<Nq>(sh + 3 * Mn, i, j, k, Di, Dj, Dk, fx, fe, fz);
    S[3] = -(Ux * fx + Ue * fe + Uz * fz) - pz * irho - (rhop * irho) * g;
    // theta: theta' and theta0 differentiated separately (Q7)
    double gx, ge, gz;
    ref_derivs<Nq>(sh + 4 * Mn, i, j, k, Di, Dj, Dk, fx, fe, fz);
    ref_derivs<Nq>(sh + 5 * Mn, i, j, k, Di, Dj, Dk, gx, ge, gz);
    S[4] = -(Ux * (fx + gx) + Ue * (fe + ge) + Uz * (fz + gz));
    // divergence of F = rho u (9 reference derivatives, L424)
    double div;
    ref_derivs<Nq>(sh + 6 * Mn, i, j, k, Di, Dj, Dk, fx, fe, fz);
    div = fx * m[0] + fe * m[3] + fz * m[6];
    ref_derivs<Nq>(sh + 7 * Mn, i, j, k, Di, Dj, Dk, fx, fe, fz);
    div += fx * m[1] + fe * m[4] + fz * m[7];
    ref_derivs<Nq>(sh + 8 * Mn, i, j, k, Di, Dj, Dk, fx, fe, fz);
    div += fx * m[2] + fe * m[5] + fz * m[8];
    S[0] = -div;
}

// A2: pointwise pre-pass for one node -> the nine nodal work values.
__device__ __forceinline__ void node_prepass(double rhop, double u, double v, double w, double thp,
                                             double rho0, double theta0, double theta0_e0,
                                             double p0, double gamma, double *__restrict__ sh,
                                             int Mn, int n)
{
    // Eq. 3 in cancellation-free form: p' = p0 * expm1(gamma * log1p(x)),
    // 1 + x = (1 + rho'/rho0)(1 + theta'/theta0)   (Q6)
    const double a = rhop / rho0, b = thp / theta0;
    const double x = a + b + a * b;
    const double rho = rho0 + rhop;
    sh[0 * Mn + n] = p0 * expm1(gamma * log1p(x));
    sh[1 * Mn + n] = u;
    sh[2 * Mn + n] = v;
    sh[3 * Mn + n] = w;
    sh[4 * Mn + n] = thp;
    sh[5 * Mn + n] = theta0 - theta0_e0;  // relative to the element's first node (Q7)
    sh[6 * Mn + n] = rho * u;
    sh[7 * Mn + n] = rho * v;
    sh[8 * Mn + n] = rho * w;
}

template <int Nq>
__device__ __forceinline__ void load_D_rows(const LglTables &t, int i, int j, int k,
                                            double (&Di)[Nq], double (&Dj)[Nq], double (&Dk)[Nq],
                                            double *sD)
{
    // stage D in shared memory once per block, then each thread keeps its three rows
    for (int t_ = threadIdx.x; t_ < Nq * Nq; t_ += blockDim.x) sD[t_] = t.D[t_];
    __syncthreads();
#pragma unroll
    for (int l = 0; l < Nq; ++l) {
        Di[l] = sD[i * Nq + l];
        Dj[l] = sD[j * Nq + l];
        Dk[l] = sD[k * Nq + l];
    }
}

// ---------------------------------------------------------------------------------------
// numa_rhs: rhs = omega * S(q)   (A2-A6)
// ---------------------------------------------------------------------------------------
template <int N>
__global__ void __launch_bounds__(Shape<N>::THREADS)
k_rhs(const double *__restrict__ q, const double *__restrict__ ref3,
      const double *__restrict__ met, const double *__restrict__ omega, double *__restrict__ rhs,
      const __grid_constant__ LglTables tab, int64_t Ne, int64_t NL, double g, double gamma,
      const ShellMap sm)
{
    constexpr int Nq = Shape<N>::Nq, Mn = Shape<N>::Mn, EPB = Shape<N>::EPB;
    extern __shared__ double sh[];  // [EPB][9][Mn] + D[Nq*Nq]
    double *sD = sh + EPB * 9 * Mn;
    const int tid = threadIdx.x;
    const int le = tid / Mn, n = tid - le * Mn;
    const int64_t e = (int64_t)blockIdx.x * EPB + le;
    const bool valid = (le < EPB) && (e < Ne);
    const int k = n / (Nq * Nq), j = (n - k * Nq * Nq) / Nq, i = n - Nq * (j + Nq * k);
    double Di[Nq], Dj[Nq], Dk[Nq];
    load_D_rows<Nq>(tab, i, j, k, Di, Dj, Dk, sD);
    const int64_t p = e * Mn + n;
    const int64_t t = valid ? shell_index(sm, p) : 0;   // the library's tables are block-shell
    double rhop = 0.0, rho0 = 1.0;
    double *she = sh + (le < EPB ? le : 0) * 9 * Mn;
    if (valid) {
        rhop = q[0 * NL + p];
        rho0 = ref3[0 * sm.FS + t];
        node_prepass(rhop, q[1 * NL + p], q[2 * NL + p], q[3 * NL + p], q[4 * NL + p], rho0,
                     ref3[1 * sm.FS + t], ref3[1 * sm.FS + shell_index(sm, e * Mn)], ref3[2 * sm.FS + t],
                     gamma, she, Mn, n);
    }
    __syncthreads();
    if (!valid) return;
    double m[9];
#pragma unroll
    for (int c = 0; c < 9; ++c) m[c] = met[c * sm.FS + t];
    double S[5];
    node_tendency<N>(she, i, j, k, Di, Dj, Dk, m, rhop, rho0, g, S);
    const double om = omega[t];
#pragma unroll
    for (int c = 0; c < 5; ++c) rhs[c * NL + p] = om * S[c];
}

// mass: M = sum over copies of wJ (all global nodes), omega = wJ / M, in place on `om`
// (block-shell array; start/copies = the block-shell list set)
__global__ void k_mass(double *__restrict__ om, const int32_t *__restrict__ start,
                       const int32_t *__restrict__ copies, int64_t NG)
{
    const int64_t gI = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (gI >= NG) return;
    const int s = start[gI], c = start[gI + 1] - s;
    double M = 0.0;
    for (int a = 0; a < c; ++a) M += om[copies[s + a]];
    for (int a = 0; a < c; ++a) om[copies[s + a]] = om[copies[s + a]] / M;
}

// ---------------------------------------------------------------------------------------
// numa_apply_sources: A8 + A9, one thread per local node
// ---------------------------------------------------------------------------------------
template <int N>
__global__ void k_sources(const double *__restrict__ q, const double *__restrict__ heat,
                          const double *__restrict__ beta, const double *__restrict__ met,
                          const uint8_t *__restrict__ face_bc, double *__restrict__ r,
                          int64_t NL, double f_cor, const ShellMap sm)
{
    constexpr int Nq = N + 1, Mn = Nq * Nq * Nq;
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= NL) return;
    const int64_t e = p / Mn;
    const int n = (int)(p - e * Mn);
    const int k = n / (Nq * Nq), j = (n - k * Nq * Nq) / Nq, i = n - Nq * (j + Nq * k);
    const double u = q[1 * NL + p], v = q[2 * NL + p];
    double ru = r[1 * NL + p], rv = r[2 * NL + p], rw = r[3 * NL + p], rt = r[4 * NL + p];
    if (heat) rt += heat[p];
    ru += f_cor * v;
    rv -= f_cor * u;
    if (beta) {
        const double b = beta[shell_index(sm, p)];
        ru -= b * u; rv -= b * v; rw -= b * q[3 * NL + p]; rt -= b * q[4 * NL + p];
    }
    const uint2 bcw = *reinterpret_cast<const uint2 *>(face_bc + e * 8);
    const bool on_face = (i == 0) | (i == Nq - 1) | (j == 0) | (j == Nq - 1) | (k == 0) | (k == Nq - 1);
    if ((bcw.x | bcw.y) && on_face) {
        uint8_t bc[8];
        *reinterpret_cast<uint2 *>(bc) = bcw;
        double m[9];
        const int64_t t = shell_index(sm, p);
#pragma unroll
        for (int c = 0; c < 9; ++c) m[c] = met[c * sm.FS + t];
        wall_project<Nq>(bc, i, j, k, m, ru, rv, rw);
    }
    r[1 * NL + p] = ru; r[2 * NL + p] = rv; r[3 * NL + p] = rw; r[4 * NL + p] = rt;
}

// ---------------------------------------------------------------------------------------
// numa_rk_stage: q_out = a0 q0 + a1 qs + b_dt r
// ---------------------------------------------------------------------------------------
__global__ void k_rk(double a0, double a1, double b_dt, const double *q0, const double *qs,
                     const double *__restrict__ r, double *qout, int64_t n)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += stride)
        qout[p] = a0 * q0[p] + a1 * qs[p] + b_dt * r[p];
}

// ---------------------------------------------------------------------------------------
// A0: metric terms and wJ from nodal coordinates (L92, L149; Eq. 8)
// ---------------------------------------------------------------------------------------
template <int N>
__global__ void __launch_bounds__(Shape<N>::THREADS)
k_metrics(const double *__restrict__ xyz, double *__restrict__ met, double *__restrict__ wJ,
          const __grid_constant__ LglTables tab, int64_t Ne, int64_t NL, int32_t *flags,
          const ShellMap sm)
{
    constexpr int Nq = Shape<N>::Nq, Mn = Shape<N>::Mn, EPB = Shape<N>::EPB;
    __shared__ double sh[EPB * 3 * Mn];
    __shared__ double sD[Nq * Nq];
    const int tid = threadIdx.x;
    const int le = tid / Mn, n = tid - le * Mn;
    const int64_t e = (int64_t)blockIdx.x * EPB + le;
    const bool valid = (le < EPB) && (e < Ne);
    const int k = n / (Nq * Nq), j = (n - k * Nq * Nq) / Nq, i = n - Nq * (j + Nq * k);
    double Di[Nq], Dj[Nq], Dk[Nq];
    load_D_rows<Nq>(tab, i, j, k, Di, Dj, Dk, sD);
    const int64_t p = e * Mn + n;
    double *she = sh + (le < EPB ? le : 0) * 3 * Mn;
    if (valid) {
#pragma unroll
        for (int c = 0; c < 3; ++c) she[c * Mn + n] = xyz[c * NL + p];
    }
    __syncthreads();
    if (!valid) return;
    double xx, xe, xz, yx, ye, yz, zx, ze, zz;
    ref_derivs_diff<Nq>(she + 0 * Mn, i, j, k, Di, Dj, Dk, xx, xe, xz);
    ref_derivs_diff<Nq>(she + 1 * Mn, i, j, k, Di, Dj, Dk, yx, ye, yz);
    ref_derivs_diff<Nq>(she + 2 * Mn, i, j, k, Di, Dj, Dk, zx, ze, zz);
    const double c0 = ye * zz - yz * ze, c1 = xz * ze - xe * zz, c2 = xe * yz - xz * ye;
    const double J = xx * c0 + yx * c1 + zx * c2;
    if (!(J > 0.0)) atomicOr(flags, 1);
    const double iJ = 1.0 / J;
    const int64_t t = shell_index(sm, p), F = sm.FS;   // tables are written in block-shell order
    met[0 * F + t] = c0 * iJ;
    met[1 * F + t] = c1 * iJ;
    met[2 * F + t] = c2 * iJ;
    met[3 * F + t] = (yz * zx - yx * zz) * iJ;
    met[4 * F + t] = (xx * zz - xz * zx) * iJ;
    met[5 * F + t] = (xz * yx - xx * yz) * iJ;
    met[6 * F + t] = (yx * ze - ye * zx) * iJ;
    met[7 * F + t] = (xe * zx - xx * ze) * iJ;
    met[8 * F + t] = (xx * ye - xe * yx) * iJ;
    wJ[t] = tab.w[i] * tab.w[j] * tab.w[k] * J;
}

static ShellMap shell_map(const numa_ctx *c)
{
    return ShellMap{c->shell.pos, c->shell.epb * (int)c->Mn, (int)c->shell.BS, c->shell.FS};
}

template <int N>
cudaError_t rhs_N(numa_ctx *c, const double *q, double *rhs, cudaStream_t s)
{
    const int64_t blocks = (c->par.n_elem + Shape<N>::EPB - 1) / Shape<N>::EPB;
    constexpr size_t smem = sizeof(double) * (Shape<N>::EPB * 9 * Shape<N>::Mn + Shape<N>::Nq * Shape<N>::Nq);
    // the attribute is per device: set once per context (contexts are bound to one device)
    if (!c->attr_rhs) {
        cudaError_t e = cudaFuncSetAttribute(k_rhs<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        c->attr_rhs = true;
    }
    k_rhs<N><<<(unsigned)blocks, Shape<N>::THREADS, smem, s>>>(q, c->ref3, c->met, c->omega, rhs,
                                                               c->lgl, c->par.n_elem, c->NL,
                                                               c->par.g, c->gamma, shell_map(c));
    return cudaGetLastError();
}

template <int N>
cudaError_t metrics_N(numa_ctx *c, const double *xyz, double *wJ, cudaStream_t s)
{
    const int64_t blocks = (c->par.n_elem + Shape<N>::EPB - 1) / Shape<N>::EPB;
    k_metrics<N><<<(unsigned)blocks, Shape<N>::THREADS, 0, s>>>(xyz, c->met, wJ, c->lgl,
                                                                c->par.n_elem, c->NL, c->d_flags, shell_map(c));
    return cudaGetLastError();
}

template <int N>
cudaError_t sources_N(numa_ctx *c, const double *q, const double *heat, double *rhs,
                      cudaStream_t s)
{
    const int64_t blocks = (c->NL + 255) / 256;
    k_sources<N><<<(unsigned)blocks, 256, 0, s>>>(q, heat, c->sponge, c->met, c->face_bc, rhs,
                                                  c->NL, c->par.f_cor, shell_map(c));
    return cudaGetLastError();
}

}  // namespace

#define DISPATCH_N(fn, ...)                                  \
    switch (c->par.N) {                                      \
        case 2: return fn<2>(__VA_ARGS__);                   \
        case 3: return fn<3>(__VA_ARGS__);                   \
        case 4: return fn<4>(__VA_ARGS__);                   \
        case 5: return fn<5>(__VA_ARGS__);                   \
        case 6: return fn<6>(__VA_ARGS__);                   \
        case 7: return fn<7>(__VA_ARGS__);                   \
        case 8: return fn<8>(__VA_ARGS__);                   \
        default: return cudaErrorInvalidValue;               \
    }

cudaError_t launch_metrics(numa_ctx *c, const double *xyz, double *wJ_out, cudaStream_t s)
{
    c->launches++;
    DISPATCH_N(metrics_N, c, xyz, wJ_out, s);
}

cudaError_t launch_rhs(numa_ctx *c, const double *q, double *rhs, cudaStream_t s)
{
    LaunchScope ls(c, K_VOLUME, s);
    DISPATCH_N(rhs_N, c, q, rhs, s);
}

cudaError_t launch_mass(numa_ctx *c, cudaStream_t s)
{
    c->launches++;
    const int64_t blocks = (c->par.n_global + 255) / 256;
    k_mass<<<(unsigned)blocks, 256, 0, s>>>(c->omega, c->dss_int.start, c->dss_int.copies,
                                            c->par.n_global);
    return cudaGetLastError();
}

cudaError_t launch_sources(numa_ctx *c, const double *q, const double *heat, double *rhs,
                           cudaStream_t s)
{
    LaunchScope ls(c, K_SOURCES, s);
    DISPATCH_N(sources_N, c, q, heat, rhs, s);
}

cudaError_t launch_rk(numa_ctx *c, double a0, double a1, double b_dt, const double *q0,
                      const double *qs, const double *rhs, double *qout, cudaStream_t s)
{
    LaunchScope ls(c, K_RK, s);
    const int64_t n = 5 * c->NL;
    int64_t blocks = (n + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    k_rk<<<(unsigned)blocks, 256, 0, s>>>(a0, a1, b_dt, q0, qs, rhs, qout, n);
    return cudaGetLastError();
}
