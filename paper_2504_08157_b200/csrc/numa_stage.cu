// Fused RK-stage kernels (sm_100a): one pass over the mesh computes the element-local Euler
// tendency (Eq. 1-3, Alg. 1-2), adds the pointwise sources, projects the walls and
// writes the stage update as DSS partial sums; a second kernel sums the partial sums of the
// shared nodes in place (Alg. 3) in fixed order.  FP64 everywhere.
//
// Why this is the same result: with omega = wJ/M and DSS the sum over
// the copies of a global node,
//     q_out = a0 q0 + a1 qs + b_dt P( DSS(omega S) + src )
//           = DSS( omega (a0 q0 + a1 qs) + b_dt P( omega (S + src) ) )
// because q0, qs, src and the wall projector P are single-valued at a global node, DSS is
// linear and sum_copies(omega) = 1.  Interior nodes have omega == 1.0 exactly.
#include "numa_internal.cuh"

namespace {

// ---------------------------------------------------------------------------------------
// Column-marching layout: thread (le, i, j) owns the zeta-column k = 0..N of element le of the
// block.  zeta-derivatives are taken in registers with D as compile-time-indexed constant-bank
// operands; xi- and eta-derivatives are taken by the same threads re-indexed as line owners
// (one whole line of the contraction per thread, again with constant-bank D), exchanging
// through shared memory: 1 store + 2x(1 load + 1 store) + 2 loads per field and node instead
// of the 3(N+1) loads of a thread-per-node contraction.
// Shared-memory node index: i + SJ*j + SK*k with SJ odd (bank-conflict-free line access).
// ---------------------------------------------------------------------------------------
template <int N, int EPB_>
struct StageShape {
    static constexpr int Nq = N + 1, N2 = Nq * Nq, Mn = N2 * Nq;
    static constexpr int EPB = EPB_;
    static constexpr int SJ = (Nq & 1) ? Nq : Nq + 1;
    static constexpr int SK = SJ * Nq;
    static constexpr int ME = SK * Nq;  // padded nodes per element and field
    static constexpr int NF = 8;        // p', u, v, w, theta, Fx, Fy, Fz
    static constexpr int ACTIVE = EPB * N2;
    static constexpr int THREADS = (ACTIVE + 31) / 32 * 32;
    static constexpr size_t SMEM = sizeof(double) * 3 * NF * EPB * ME;
};

struct StageArgs {
    const double *qs, *q0;
    double *qout;
    const double *ref3, *met, *omega, *heat, *beta;
    const uint8_t *face_bc;
    int64_t Ne, NL;
    double g, gamma, f_cor, a0, a1, b_dt;
    int has_walls;
};

template <int N, int EPB>
__global__ void __launch_bounds__(StageShape<N, EPB>::THREADS)
k_stage_volume(const __grid_constant__ StageArgs A, const __grid_constant__ LglTables tab)
{
    using SH = StageShape<N, EPB>;
    constexpr int Nq = SH::Nq, N2 = SH::N2, Mn = SH::Mn, SJ = SH::SJ, SK = SH::SK, ME = SH::ME,
                  NF = SH::NF;
    extern __shared__ double smem[];
    double *sW = smem;                    // [NF][EPB][ME] nodal work fields
    double *sGx = sW + NF * EPB * ME;     // d/dxi
    double *sGe = sGx + NF * EPB * ME;    // d/deta

    const int tid = threadIdx.x;
    const int le = tid / N2, ij = tid - le * N2;
    const int j = ij / Nq, i = ij - j * Nq;
    const int64_t e = (int64_t)blockIdx.x * EPB + le;
    const bool active = (tid < SH::ACTIVE) && (e < A.Ne);
    const int64_t NL = A.NL;
    const int64_t pb = e * Mn + ij;            // global index of node (i, j, 0)
    const int sb = le * ME + i + SJ * j;       // shared index of node (i, j, 0)

    // ---- phase A: pointwise pre-pass (A2) down the column, zeta-derivatives in registers ----
    double Gz[NF][Nq];
    if (active) {
        const double *__restrict__ r0 = A.ref3, *__restrict__ r1 = A.ref3 + NL,
                                   *__restrict__ r2 = A.ref3 + 2 * NL;
        const double th0e = r1[e * Mn];  // theta0 relative to the element's first node (Q7)
        double W[NF][Nq];
#pragma unroll
        for (int k = 0; k < Nq; ++k) {
            const int64_t p = pb + (int64_t)k * N2;
            const double rhop = A.qs[p], u = A.qs[NL + p], v = A.qs[2 * NL + p],
                         w = A.qs[3 * NL + p], thp = A.qs[4 * NL + p];
            const double rho0 = r0[p], th0 = r1[p], p0 = r2[p];
            // Eq. 3, cancellation-free: p' = p0 expm1(gamma log1p(x)), 1+x = (1+a)(1+b)  (Q6)
            const double a = rhop / rho0, b = thp / th0;
            const double x = a + b + a * b;
            const double rho = rho0 + rhop;
            W[0][k] = p0 * expm1(A.gamma * log1p(x));
            W[1][k] = u;
            W[2][k] = v;
            W[3][k] = w;
            W[4][k] = thp + (th0 - th0e);
            W[5][k] = rho * u;
            W[6][k] = rho * v;
            W[7][k] = rho * w;
#pragma unroll
            for (int f = 0; f < NF; ++f) sW[f * EPB * ME + sb + SK * k] = W[f][k];
        }
#pragma unroll
        for (int f = 0; f < NF; ++f)
#pragma unroll
            for (int k = 0; k < Nq; ++k) {
                double acc = 0.0;
#pragma unroll
                for (int l = 0; l < Nq; ++l) acc = fma(tab.D[k * Nq + l], W[f][l], acc);
                Gz[f][k] = acc;
            }
    }
    __syncthreads();

    // ---- phase B: xi- and eta-lines (Alg. 2), one whole line per thread and field ----------
    if (active) {
        // this thread's xi-line: (le, j' = i_line, k' = j_line) -> nodes l + SJ*(jk)
        const int xb = le * ME + SJ * ij;                      // line index jk = ij
        // this thread's eta-line: (le, i' = i, k' = j)  -> nodes i + SJ*l + SK*j
        const int eb = le * ME + i + SK * j;
#pragma unroll
        for (int f = 0; f < NF; ++f) {
            const double *w = sW + f * EPB * ME;
            double x[Nq], y[Nq];
#pragma unroll
            for (int l = 0; l < Nq; ++l) { x[l] = w[xb + l]; y[l] = w[eb + SJ * l]; }
            double *gx = sGx + f * EPB * ME, *ge = sGe + f * EPB * ME;
#pragma unroll
            for (int m = 0; m < Nq; ++m) {
                double ax = 0.0, ay = 0.0;
#pragma unroll
                for (int l = 0; l < Nq; ++l) {
                    ax = fma(tab.D[m * Nq + l], x[l], ax);
                    ay = fma(tab.D[m * Nq + l], y[l], ay);
                }
                gx[xb + m] = ax;
                ge[eb + SJ * m] = ay;
            }
        }
    }
    __syncthreads();
    if (!active) return;

    // ---- phase C: chain rule, Eq. 1 tendencies, sources, walls, stage update (A5-A10) -------
    const uint2 bcw = *reinterpret_cast<const uint2 *>(A.face_bc + e * 8);
    uint8_t bc[8];
#pragma unroll
    for (int f = 0; f < 4; ++f) {
        bc[f] = (uint8_t)(bcw.x >> (8 * f));
        bc[4 + f] = (uint8_t)(bcw.y >> (8 * f));
    }
    const bool elem_walls = A.has_walls && ((bcw.x | bcw.y) != 0);
    const bool same = (A.q0 == A.qs);
#pragma unroll
    for (int k = 0; k < Nq; ++k) {
        const int64_t p = pb + (int64_t)k * N2;
        const int sp = sb + SK * k;
        double m[9];
#pragma unroll
        for (int c = 0; c < 9; ++c) m[c] = __ldg(A.met + c * NL + p);
        const double om = __ldg(A.omega + p);
        const double rho0 = __ldg(A.ref3 + p);
        double qv[5], q0v[5];
#pragma unroll
        for (int c = 0; c < 5; ++c) qv[c] = A.qs[c * NL + p];
        if (same) {
#pragma unroll
            for (int c = 0; c < 5; ++c) q0v[c] = qv[c];
        } else {
#pragma unroll
            for (int c = 0; c < 5; ++c) q0v[c] = A.q0[c * NL + p];
        }
        double fx[NF], fe[NF];
#pragma unroll
        for (int f = 0; f < NF; ++f) {
            fx[f] = sGx[f * EPB * ME + sp];
            fe[f] = sGe[f * EPB * ME + sp];
        }
        const double rhop = qv[0], u = qv[1], v = qv[2], w = qv[3];
        const double irho = 1.0 / (rho0 + rhop);
        // contravariant velocity: u . grad f = sum_a U^a f_{xi_a}
        const double Ux = u * m[0] + v * m[1] + w * m[2];
        const double Ue = u * m[3] + v * m[4] + w * m[5];
        const double Uz = u * m[6] + v * m[7] + w * m[8];
        const double px = fx[0] * m[0] + fe[0] * m[3] + Gz[0][k] * m[6];
        const double py = fx[0] * m[1] + fe[0] * m[4] + Gz[0][k] * m[7];
        const double pz = fx[0] * m[2] + fe[0] * m[5] + Gz[0][k] * m[8];
        double S[5];
        S[1] = -(Ux * fx[1] + Ue * fe[1] + Uz * Gz[1][k]) - px * irho;
        S[2] = -(Ux * fx[2] + Ue * fe[2] + Uz * Gz[2][k]) - py * irho;
        S[3] = -(Ux * fx[3] + Ue * fe[3] + Uz * Gz[3][k]) - pz * irho - (rhop * irho) * A.g;
        S[4] = -(Ux * fx[4] + Ue * fe[4] + Uz * Gz[4][k]);
        double div = fx[5] * m[0] + fe[5] * m[3] + Gz[5][k] * m[6];
        div += fx[6] * m[1] + fe[6] * m[4] + Gz[6][k] * m[7];
        div += fx[7] * m[2] + fe[7] * m[5] + Gz[7][k] * m[8];
        S[0] = -div;
        // A8: heating, Coriolis, sponge
        if (A.heat) S[4] += __ldg(A.heat + p);
        S[1] += A.f_cor * v;
        S[2] -= A.f_cor * u;
        if (A.beta) {
            const double b = __ldg(A.beta + p);
            S[1] -= b * u; S[2] -= b * v; S[3] -= b * w; S[4] -= b * qv[4];
        }
        // A6: weight; A9: walls on the weighted velocity tendency
        double r[5];
#pragma unroll
        for (int c = 0; c < 5; ++c) r[c] = om * S[c];
        if (elem_walls) wall_project<Nq>(bc, i, j, k, m, r[1], r[2], r[3]);
        // A10 as a DSS partial sum
#pragma unroll
        for (int c = 0; c < 5; ++c)
            A.qout[c * NL + p] = om * (A.a0 * q0v[c] + A.a1 * qv[c]) + A.b_dt * r[c];
    }
}

// ---------------------------------------------------------------------------------------
// DSS by multiplicity class (Alg. 3 gather + scatter, deterministic): one thread per shared
// global node; the copy lists of the nodes with C copies are stored transposed
// (idx[a*n + t]) so that the index loads coalesce and carry no dependent chain; all 5*C
// values are loaded before the first store.  Sum in ascending local index.
// ---------------------------------------------------------------------------------------
template <int C>
__device__ __forceinline__ void dss_node(double *r, const int32_t *__restrict__ idx, int64_t n,
                                         int64_t t, int64_t NL)
{
    int32_t id[C];
#pragma unroll
    for (int a = 0; a < C; ++a) id[a] = idx[a * n + t];
    double v[5][C];
#pragma unroll
    for (int m = 0; m < 5; ++m)
#pragma unroll
        for (int a = 0; a < C; ++a) v[m][a] = r[m * NL + id[a]];
#pragma unroll
    for (int m = 0; m < 5; ++m) {
        double s = v[m][0];
#pragma unroll
        for (int a = 1; a < C; ++a) s += v[m][a];
#pragma unroll
        for (int a = 0; a < C; ++a) r[m * NL + id[a]] = s;
    }
}

struct DssArgs {
    const int32_t *idx;        // class lists, transposed
    int64_t n[3], base[3];     // nodes and list offset of the classes C = 2, 4, 8
    int64_t blk[3];            // first block of the classes 4, 8 and of the generic tail
    const int32_t *gen_nodes;  // global ids with any other multiplicity >= 2
    int64_t n_gen;
    const int32_t *start, *copies;  // CSR lists (generic path)
    int64_t NL;
};

constexpr int kDssThreads = 128;

__global__ void __launch_bounds__(kDssThreads)
k_stage_dss(double *r, const __grid_constant__ DssArgs A)
{
    const int64_t b = blockIdx.x;
    if (b < A.blk[0]) {
        const int64_t t = b * kDssThreads + threadIdx.x;
        if (t < A.n[0]) dss_node<2>(r, A.idx + A.base[0], A.n[0], t, A.NL);
    } else if (b < A.blk[1]) {
        const int64_t t = (b - A.blk[0]) * kDssThreads + threadIdx.x;
        if (t < A.n[1]) dss_node<4>(r, A.idx + A.base[1], A.n[1], t, A.NL);
    } else if (b < A.blk[2]) {
        const int64_t t = (b - A.blk[1]) * kDssThreads + threadIdx.x;
        if (t < A.n[2]) dss_node<8>(r, A.idx + A.base[2], A.n[2], t, A.NL);
    } else {
        const int64_t t = (b - A.blk[2]) * kDssThreads + threadIdx.x;
        if (t >= A.n_gen) return;
        const int gI = A.gen_nodes[t];
        const int s = A.start[gI], c = A.start[gI + 1] - s;
        for (int m = 0; m < 5; ++m) {
            double *rm = r + (int64_t)m * A.NL;
            double sum = rm[A.copies[s]];
            for (int a = 1; a < c; ++a) sum += rm[A.copies[s + a]];
            for (int a = 0; a < c; ++a) rm[A.copies[s + a]] = sum;
        }
    }
}

template <int N, int EPB>
cudaError_t stage_launch(numa_ctx *c, const StageArgs &a, cudaStream_t s)
{
    using SH = StageShape<N, EPB>;
    static bool attr_done = false;
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(k_stage_volume<N, EPB>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SH::SMEM);
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    const int64_t blocks = (c->par.n_elem + EPB - 1) / EPB;
    k_stage_volume<N, EPB><<<(unsigned)blocks, SH::THREADS, SH::SMEM, s>>>(a, c->lgl);
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_stage_volume(numa_ctx *c, double a0, double a1, double b_dt, const double *q0,
                                const double *qs, const double *heat, double *qout, cudaStream_t s)
{
    LaunchScope ls(c, K_FUSED_VOLUME, s);
    StageArgs a;
    a.qs = qs; a.q0 = q0; a.qout = qout;
    a.ref3 = c->ref3; a.met = c->met; a.omega = c->omega; a.heat = heat; a.beta = c->sponge;
    a.face_bc = c->face_bc;
    a.Ne = c->par.n_elem; a.NL = c->NL;
    a.g = c->par.g; a.gamma = c->gamma; a.f_cor = c->par.f_cor;
    a.a0 = a0; a.a1 = a1; a.b_dt = b_dt;
    a.has_walls = c->has_walls;
    switch (c->par.N) {
        case 2: return stage_launch<2, 8>(c, a, s);
        case 3: return stage_launch<3, 4>(c, a, s);
        case 4: return stage_launch<4, 4>(c, a, s);
        case 5: return stage_launch<5, 2>(c, a, s);
        case 6: return stage_launch<6, 1>(c, a, s);
        case 7: return stage_launch<7, 1>(c, a, s);
        case 8: return stage_launch<8, 1>(c, a, s);
        default: return cudaErrorInvalidValue;
    }
}

cudaError_t launch_dss_classes(numa_ctx *c, double *r, int kernel_id, cudaStream_t s)
{
    if (c->n_shared == 0) return cudaSuccess;
    LaunchScope ls(c, kernel_id, s);
    DssArgs a;
    a.idx = c->dss_idx;
    int64_t blocks = 0;
    for (int k = 0; k < 3; ++k) {
        a.n[k] = c->cls_n[k];
        a.base[k] = c->cls_base[k];
        blocks += (c->cls_n[k] + kDssThreads - 1) / kDssThreads;
        a.blk[k] = blocks;
    }
    a.gen_nodes = c->gen_nodes;
    a.n_gen = c->n_gen;
    blocks += (c->n_gen + kDssThreads - 1) / kDssThreads;
    a.start = c->dss_start; a.copies = c->dss_copies;
    a.NL = c->NL;
    k_stage_dss<<<(unsigned)blocks, kDssThreads, 0, s>>>(r, a);
    return cudaGetLastError();
}
