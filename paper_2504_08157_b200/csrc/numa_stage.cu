// Fused RK-stage kernels (sm_100a): one pass over the mesh computes the element-local Euler
// tendency (Eq. 1-3, Alg. 1-2), adds the pointwise sources, projects the walls and
// writes the stage update as DSS partial sums; a second kernel sums the partial sums of the
// shared nodes in place (Alg. 3) in fixed order.  FP64 everywhere.
//
// Every per-node array of this route (state q0 / qs / q_out, metric terms, omega, reference
// state, sponge, heating) is stored in the BLOCK-SHELL layout (ShellLayout, numa_internal.cuh;
// DESIGN.md 6): the copies of shared nodes form long contiguous runs, so the DSS kernel touches
// whole 32-byte sectors, and the volume kernel runs its pointwise phases one thread per
// POSITION of a block record -- every global access is a coalesced, 256-byte-aligned stream.
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
// Volume kernel layout.  A block owns EPB consecutive elements (a contiguous chunk of
// EPB*Mn nodes of every field).  Pointwise work (A2 pre-pass; A5-A10 combine) is done one
// thread per node, so every global access is coalesced.  The 24 one-dimensional contractions
// of Alg. 2 are done as LINE TASKS: one thread takes one whole line of one field along one
// direction (N+1 shared loads), forms all N+1 derivatives of the line with D as
// compile-time-indexed constant-bank operands ((N+1)^2 FMAs, no further loads) and stores
// them (N+1 shared stores).  Per node and field that is 1 store + 3x(1 load + 1 store) + 3
// loads of shared memory instead of the 3(N+1) loads of a thread-per-node contraction.
// The zeta-derivatives overwrite the work fields in place (after a barrier), so a node needs
// 24 doubles of shared memory.  Shared node index: i + SJ*j + SK*k.  Line tasks are numbered
// field-fastest and the field stride is 2 (mod 4) doubles, which makes every line access of a
// half-warp hit 16 distinct banks (StageShape).
// ---------------------------------------------------------------------------------------
template <int N>
struct StageShape {
    static constexpr int Nq = N + 1, N2 = Nq * Nq, Mn = N2 * Nq;
#define STAGE_EPB4 1
#define STAGE_MINB4 6
#define STAGE_EPB3 2
#define STAGE_EPB5 1
    static constexpr int EPB = (N == 2) ? 9 : (N == 3) ? STAGE_EPB3 : (N == 4) ? STAGE_EPB4 : (N == 5) ? STAGE_EPB5 : 1;
    // shared node index i + SJ*j + SK*k; for even Nq the k-planes are padded by one double
    static constexpr int SJ = Nq;
    static constexpr int SK = (Nq & 1) ? N2 : N2 + 1;
    static constexpr int ME = SK * Nq;  // padded nodes per element and field
    static constexpr int NF = 8;        // p', u, v, w, theta, Fx, Fy, Fz
    static constexpr int NODES = EPB * Mn;
    // positions per block record (ShellLayout::BS): whole warps, so that every block record of
    // every field starts on a 256-byte line
    static constexpr int BS = (NODES + 31) / 32 * 32;
    // NPT nodes per thread in the pointwise phases: at high N a block of Mn threads would be
    // alone on its SM (registers, shared memory); half as many threads let two blocks overlap
    // their memory and compute phases.
#define STAGE_NPT_HI 2
#define STAGE_NPT_MINN 9  /* measured: no gain at N <= 8; kept for larger elements */
    // THR_OVR: explicit block size where the default (one thread per node) balances the line
    // tasks badly: 8*LINES tasks per direction should fill whole rounds of THREADS threads.
#define STAGE_THREADS5 0
#define STAGE_THREADS6 416  /* 392 line tasks per pass in one round (352 threads: 352 + 40) */
#define STAGE_THREADS8 0
    static constexpr int THR_OVR = (N == 5) ? STAGE_THREADS5 : (N == 6) ? STAGE_THREADS6 : (N == 8) ? STAGE_THREADS8 : 0;
    static constexpr int NPT = THR_OVR ? (NODES + THR_OVR - 1) / THR_OVR
                                       : (N >= STAGE_NPT_MINN) ? STAGE_NPT_HI : 1;
    static constexpr int THREADS = THR_OVR ? THR_OVR : ((BS / 32 + NPT - 1) / NPT) * 32;
    static constexpr int SLOTS = THREADS * NPT;  // >= BS
    static constexpr int LINES = EPB * N2;  // lines per field and direction
    // field stride in shared memory: = 2 (mod 4) doubles, so that with the FIELD-FASTEST task
    // enumeration (lane -> field = T mod 8, line = T / 8) the 16 lanes of a half-warp hit 16
    // different 8-byte banks in all three line directions (brute-forced).
    static constexpr int FS = EPB * ME + ((EPB * ME) % 4 == 2 ? 0 : (EPB * ME) % 4 == 1 ? 1
                            : (EPB * ME) % 4 == 0 ? 2 : 3);
    // POOLED: the zeta-derivatives get their own buffer, so the line tasks of all three
    // directions form one pool without a barrier in between (better balance at low N);
    // otherwise they overwrite the work fields in place after a barrier (less shared memory).
#define STAGE_POOLED_MASK 0x04  /* bit N set = pooled */
    static constexpr bool POOLED = (STAGE_POOLED_MASK >> N) & 1;
    static constexpr size_t SMEM_WORK = sizeof(double) * (POOLED ? 4 : 3) * NF * FS;
    // PREFETCH: request the phase-C inputs in phase A (17 doubles live across phase B); at high
    // N the registers are worth more as a second resident block.
#define STAGE_PREFETCH_MAXN 4  /* N=5: with the L2 prefetch, four blocks per SM without the register prefetch beat three with it (1.50 -> 1.39 ms per 32 M nodes) */
    static constexpr bool PREFETCH = (N <= STAGE_PREFETCH_MAXN) && NPT == 1;
    // (a cp.async staging of the same 17 inputs into shared memory was measured too: with the L2
    // prefetch it no longer pays, N = 8 1.92 -> 1.79 ms without; removed, in the history)
    static constexpr size_t SMEM = SMEM_WORK;
#define STAGE_MINB3 6
#define STAGE_MINB5 4
#define STAGE_MINB6 2
#define STAGE_MINB7 2
#define STAGE_MINB8 1
    static constexpr int MIN_BLOCKS = (N == 4) ? STAGE_MINB4 : (N == 3) ? STAGE_MINB3 : (N == 5) ? STAGE_MINB5
                                    : (N == 6) ? STAGE_MINB6 : (N == 7) ? STAGE_MINB7 : (N == 8) ? STAGE_MINB8 : 3;
};

struct StageArgs {
    // all per-node arrays are block-shell: [fields][GFS], GFS = n_blocks * BS
    const double *qs, *q0;
    double *qout;
    const double *ref3, *met, *omega, *heat, *beta;
    const uint32_t *tab;     // [BS] thread slot -> position and node (ShellLayout::tab)
    const uint8_t *face_bc;
    int64_t Ne, GFS;
    int first_pos[16];       // position of node 0 of the le-th element of a block (Q7)
    double g, gamma, f_cor, a0, a1, b_dt;
    double eos[14];  // binomial(gamma, n), n = 1..14: (1+x)^gamma - 1 = sum_n eos[n-1] x^n
    int has_walls;
    int pf_dist;     // blocks resident on the device: block b prefetches the phase-A inputs of block b + pf_dist
    int64_t blk0, n_blocks;   // first block of this launch (a launch may cover a sub-range) and blocks of the whole mesh
};

// Eq. 3 in cancellation-free form (Q6): p'/p0 = (1+x)^gamma - 1 with
// 1 + x = (1 + rho'/rho0)(1 + theta'/theta0).  For |x| <= 1/16 the binomial series to degree
// 14 is exact to double rounding (next term < 2e-20 |x|); otherwise expm1(gamma log1p(x)).
__device__ __forceinline__ double eos_ratio(double x, double gamma, const double (&c)[14])
{
    if (fabs(x) <= 0.0625) {
        double s = c[13];
#pragma unroll
        for (int n = 12; n >= 0; --n) s = fma(s, x, c[n]);
        return s * x;
    }
    return expm1(gamma * log1p(x));
}

// All Nq derivatives of one line.  D is centro-antisymmetric (D[N-m][N-l] = -D[m][l], enforced
// bitwise by numa_build_lgl), so rows m and N-m share their constants: only the upper half of
// D is touched -- on sm_100 constant operands travel through uniform registers, and the full
// (N+1)^2 table does not fit them at N >= 6 (the compiler then spills through vector registers
// to local memory).
template <int Nq>
__device__ __forceinline__ void line_derivs(const double *src, int sstride, double *dst,
                                            const LglTables &tab)
{
    double x[Nq];
#pragma unroll
    for (int l = 0; l < Nq; ++l) x[l] = src[sstride * l];
#define STAGE_ANTISYM_MINNQ 7  /* N >= 6; below that the full table fits and is faster */
    if constexpr (Nq < STAGE_ANTISYM_MINNQ) {
#pragma unroll
        for (int m = 0; m < Nq; ++m) {
            double acc = 0.0;
#pragma unroll
            for (int l = 0; l < Nq; ++l) acc = fma(tab.D[m * Nq + l], x[l], acc);
            dst[sstride * m] = acc;
        }
#define STAGE_EVEN_ODD 7  /* Nq from which the even-odd form is used (measured: pays at N >= 6) */
    } else if constexpr (Nq >= STAGE_EVEN_ODD) {
        // even-odd form: half the multiplications (A, B of LglTables)
        constexpr int H = Nq / 2;
        double e[H], o[H];
#pragma unroll
        for (int l = 0; l < H; ++l) { e[l] = x[l] + x[Nq - 1 - l]; o[l] = x[l] - x[Nq - 1 - l]; }
#pragma unroll
        for (int m = 0; m < H; ++m) {
            double P = (Nq & 1) ? tab.C[m] * x[H] : 0.0, Q = 0.0;
#pragma unroll
            for (int l = 0; l < H; ++l) { P = fma(tab.A[m * H + l], e[l], P); Q = fma(tab.B[m * H + l], o[l], Q); }
            dst[sstride * m] = P + Q;
            dst[sstride * (Nq - 1 - m)] = Q - P;
        }
        if constexpr (Nq & 1) {
            double a = 0.0;
#pragma unroll
            for (int l = 0; l < H; ++l) a = fma(tab.M[l], o[l], a);
            dst[sstride * H] = a;
        }
    } else {
#pragma unroll
        for (int m = 0; m < Nq / 2; ++m) {
            double a = 0.0, b = 0.0;
#pragma unroll
            for (int l = 0; l < Nq; ++l) {
                const double d = tab.D[m * Nq + l];
                a = fma(d, x[l], a);
                b = fma(d, x[Nq - 1 - l], b);
            }
            dst[sstride * m] = a;
            dst[sstride * (Nq - 1 - m)] = -b;
        }
        if constexpr (Nq & 1) {
            constexpr int m = Nq / 2;
            double a = 0.0;
#pragma unroll
            for (int l = 0; l < Nq; ++l) a = fma(tab.D[m * Nq + l], x[l], a);
            dst[sstride * m] = a;
        }
    }
}

// A9 for the few nodes that lie on a wall face: kept out of line so that its square roots
// and divisions do not weigh on the registers and code of the common path.
struct WallIO { double m[9]; double r[3]; };

template <int Nq>
__device__ __noinline__ void wall_project_cold(uint2 bcw, int i, int j, int k, WallIO *io)
{
    uint8_t bc[8];
#pragma unroll
    for (int f = 0; f < 4; ++f) {
        bc[f] = (uint8_t)(bcw.x >> (8 * f));
        bc[4 + f] = (uint8_t)(bcw.y >> (8 * f));
    }
    wall_project<Nq>(bc, i, j, k, io->m, io->r[0], io->r[1], io->r[2]);
}

// L2 prefetch of one contiguous run (bytes a multiple of 16, address 16-byte aligned): no
// registers, no shared memory; the later ld.global then pays the L2 latency instead of HBM's
__device__ __forceinline__ void l2_prefetch(const double *g, unsigned bytes)
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(g), "r"(bytes) : "memory");
}

// Pointwise role of a thread: slot -> position of the block record -> node, from the table
// (bits 0-9 shared-memory index sp, 10-13 i, 14-17 j, 18-21 k, 22-25 element of the block,
// 26-30 lane of the position inside its warp's 32 positions; all ones = no node).
struct NodeIx { bool has; int le, i, j, k, sp; int64_t p; };

template <class SH>
__device__ __forceinline__ NodeIx node_ix(const uint32_t *__restrict__ tab, int slot, int64_t rec,
                                          int n_elems)
{
    NodeIx x;
    const uint32_t w = (slot < SH::BS) ? __ldg(tab + slot) : 0xFFFFFFFFu;
    x.sp = (int)(w & 1023u);
    x.i = (int)((w >> 10) & 15u);
    x.j = (int)((w >> 14) & 15u);
    x.k = (int)((w >> 18) & 15u);
    x.le = (int)((w >> 22) & 15u);
    x.has = (w != 0xFFFFFFFFu) && (x.le < n_elems);
    x.p = rec + (slot & ~31) + (int)((w >> 26) & 31u);
    return x;
}

// Global accesses of the volume kernel: every value is used once per block, so nothing is
// gained by allocating it in L1: ld/st .cg (measured against ld.global.nc + default stores and against .cs)
#define VLD(p) __ldcg(p)
#define VST(p, v) __stcg(p, v)

template <int N>
__global__ void __launch_bounds__(StageShape<N>::THREADS, StageShape<N>::MIN_BLOCKS)
k_stage_volume(const __grid_constant__ StageArgs A, const __grid_constant__ LglTables tab)
{
    using SH = StageShape<N>;
    constexpr int Nq = SH::Nq, N2 = SH::N2, Mn = SH::Mn, SJ = SH::SJ, SK = SH::SK, ME = SH::ME,
                  NF = SH::NF, FS = SH::FS, LINES = SH::LINES;
    extern __shared__ double smem[];
    double *sW = smem;            // [NF][EPB][ME] nodal work fields, later d/dzeta
    double *sGx = sW + NF * FS;   // d/dxi
    double *sGe = sGx + NF * FS;  // d/deta

    const int tid = threadIdx.x;
    const int64_t NL = A.GFS;                                  // field stride of every array
    const int64_t bid = A.blk0 + blockIdx.x;                   // block of the mesh (a launch may cover a sub-range)
    const int64_t rec = bid * SH::BS;                          // this block's record
    const int64_t e0 = bid * SH::EPB;
    const int n_elems = (A.Ne - e0 < SH::EPB) ? (int)(A.Ne - e0) : SH::EPB;  // ragged last block
    const int n_lines = n_elems * N2;

#define STAGE_L2PF 3   /* bit 0: phase-C inputs of this block; bit 1: phase-A inputs of block b + pf_dist */
    if (STAGE_L2PF && tid == 0) {
        constexpr unsigned RB = SH::BS * sizeof(double);
        if (STAGE_L2PF & 1) {
#pragma unroll
            for (int c = 0; c < 9; ++c) l2_prefetch(A.met + c * NL + rec, RB);
            l2_prefetch(A.omega + rec, RB);
            if (A.q0 != A.qs) {
#pragma unroll
                for (int c = 0; c < 5; ++c) l2_prefetch(A.q0 + c * NL + rec, RB);
            }
            if (A.heat) l2_prefetch(A.heat + rec, RB);
            if (A.beta) l2_prefetch(A.beta + rec, RB);
        }
        if ((STAGE_L2PF & 2) && bid + A.pf_dist < A.n_blocks) {
            const int64_t rec2 = rec + (int64_t)A.pf_dist * SH::BS;
#pragma unroll
            for (int c = 0; c < 5; ++c) l2_prefetch(A.qs + c * NL + rec2, RB);
#pragma unroll
            for (int c = 0; c < 3; ++c) l2_prefetch(A.ref3 + c * NL + rec2, RB);
        }
    }

    constexpr int NPT = SH::NPT;
    static_assert(!SH::PREFETCH || NPT == 1, "register prefetch only with one node per thread");

    // ---- phase A: pointwise pre-pass (A2) ---------------------------------------------------
    double qv[NPT][5], rho0[NPT];
    // inputs of phase C, requested now so that they are in flight during phases A and B
    double m[9], q0v[5], om = 0.0, heat = 0.0, beta = 0.0;
    const bool same = (A.q0 == A.qs);
#pragma unroll
    for (int rr = 0; rr < NPT; ++rr) {
        const NodeIx x = node_ix<SH>(A.tab, tid + rr * SH::THREADS, rec, n_elems);
        const int64_t p = x.p;
        const int sp = x.sp;
        rho0[rr] = 1.0;
#pragma unroll
        for (int c = 0; c < 5; ++c) qv[rr][c] = 0.0;
        if (!x.has) continue;
#pragma unroll
        for (int c = 0; c < 5; ++c) qv[rr][c] = VLD(A.qs + c * NL + p);
        if constexpr (SH::PREFETCH) {
#pragma unroll
            for (int c = 0; c < 9; ++c) m[c] = VLD(A.met + c * NL + p);
            om = VLD(A.omega + p);
            if (!same) {
#pragma unroll
                for (int c = 0; c < 5; ++c) q0v[c] = VLD(A.q0 + c * NL + p);
            }
            if (A.heat) heat = VLD(A.heat + p);
            if (A.beta) beta = VLD(A.beta + p);
        }
        rho0[rr] = VLD(A.ref3 + p);
        const double th0 = VLD(A.ref3 + NL + p), p0 = VLD(A.ref3 + 2 * NL + p);
        const double th0e = VLD(A.ref3 + NL + rec + A.first_pos[x.le]);  // theta0 at the element's first node (Q7)
        const double xx = (qv[rr][0] * th0 + qv[rr][4] * rho0[rr] + qv[rr][0] * qv[rr][4]) / (rho0[rr] * th0);
        const double rho = rho0[rr] + qv[rr][0];
        sW[0 * FS + sp] = p0 * eos_ratio(xx, A.gamma, A.eos);
        sW[1 * FS + sp] = qv[rr][1];
        sW[2 * FS + sp] = qv[rr][2];
        sW[3 * FS + sp] = qv[rr][3];
        sW[4 * FS + sp] = qv[rr][4] + (th0 - th0e);
        sW[5 * FS + sp] = rho * qv[rr][1];
        sW[6 * FS + sp] = rho * qv[rr][2];
        sW[7 * FS + sp] = rho * qv[rr][3];
    }
    __syncthreads();

    // ---- phase B: line tasks (Alg. 2) ----------------------------------------------------------
    // Task t -> field f = t mod 8 (fastest), line = t / 8 = l2 + N2*element, l2 = lo + Nq*hi.
    //   xi-line:   odd Nq (j,k) = (lo,hi), even Nq (j,k) = (hi,lo);  points l + SJ*j + SK*k
    //   eta-line:  (i,k) = (lo,hi);  points i + SJ*l + SK*k
    //   zeta-line: (i,j) = (lo,hi);  points i + SJ*j + SK*l
    // buffers are laid out [sW | d/dxi | d/deta | d/dzeta], NF*FS each
    const double *sGz = sW;
    if constexpr (SH::POOLED) {
        sGz = sGe + NF * FS;
#pragma unroll 1
        for (int T = tid; T < 3 * NF * LINES; T += SH::THREADS) {
            const int dir = T / (NF * LINES), r = T - dir * (NF * LINES);
            const int f = r & 7, line = r >> 3;
            if (line >= n_lines) continue;
            const int el = (SH::EPB == 1) ? 0 : line / N2, l2 = line - el * N2;
            const int hi = l2 / Nq, lo = l2 - hi * Nq;
            const int bx = (Nq & 1) ? SJ * lo + SK * hi : SJ * hi + SK * lo;
            const int base = (dir == 0) ? bx : (dir == 1) ? lo + SK * hi : lo + SJ * hi;
            const int stride = (dir == 0) ? 1 : (dir == 1) ? SJ : SK;
            double *src = sW + f * FS + el * ME + base;
            line_derivs<Nq>(src, stride, src + (1 + dir) * NF * FS, tab);
        }
    } else {
        // xi and eta (both only read sW), barrier, then zeta in place
        for (int t = tid; t < NF * LINES; t += SH::THREADS) {
            const int f = t & 7, line = t >> 3;
            if (line >= n_lines) continue;
            const int el = (SH::EPB == 1) ? 0 : line / N2, l2 = line - el * N2;
            const int hi = l2 / Nq, lo = l2 - hi * Nq;
            const int base = f * FS + el * ME;
            const int bx = base + ((Nq & 1) ? SJ * lo + SK * hi : SJ * hi + SK * lo);
            line_derivs<Nq>(sW + bx, 1, sGx + bx, tab);
            line_derivs<Nq>(sW + base + lo + SK * hi, SJ, sGe + base + lo + SK * hi, tab);
        }
        __syncthreads();
        for (int t = tid; t < NF * LINES; t += SH::THREADS) {
            const int f = t & 7, line = t >> 3;
            if (line >= n_lines) continue;
            const int el = (SH::EPB == 1) ? 0 : line / N2, l2 = line - el * N2;
            const int hi = l2 / Nq, lo = l2 - hi * Nq;
            double *w = sW + f * FS + el * ME + lo + SJ * hi;
            line_derivs<Nq>(w, SK, w, tab);
        }
    }
    __syncthreads();

    // ---- phase C: chain rule, Eq. 1 tendencies, sources, walls, stage update (A5-A10) -------
#pragma unroll
    for (int rr = 0; rr < NPT; ++rr) {
    const NodeIx x = node_ix<SH>(A.tab, tid + rr * SH::THREADS, rec, n_elems);
    if (!x.has) continue;
    const int64_t p = x.p;
    const int sp = x.sp, i = x.i, j = x.j, k = x.k;
    if constexpr (!SH::PREFETCH) {
#pragma unroll
        for (int c = 0; c < 9; ++c) m[c] = VLD(A.met + c * NL + p);
        om = VLD(A.omega + p);
        if (!same) {
#pragma unroll
            for (int c = 0; c < 5; ++c) q0v[c] = VLD(A.q0 + c * NL + p);
        }
        heat = A.heat ? VLD(A.heat + p) : 0.0;
        beta = A.beta ? VLD(A.beta + p) : 0.0;
    }
    const double rhop = qv[rr][0], u = qv[rr][1], v = qv[rr][2], w = qv[rr][3];
    const double irho = 1.0 / (rho0[rr] + rhop);
    // contravariant velocity: u . grad f = sum_a U^a f_{xi_a}
    const double Ux = u * m[0] + v * m[1] + w * m[2];
    const double Ue = u * m[3] + v * m[4] + w * m[5];
    const double Uz = u * m[6] + v * m[7] + w * m[8];
    const double *gx = sGx + sp, *ge = sGe + sp, *gz = sGz + sp;
    double S[5];
    {   // pressure gradient and buoyancy (Eq. 1b)
        const double fx = gx[0], fe = ge[0], fz = gz[0];
        S[1] = -(fx * m[0] + fe * m[3] + fz * m[6]) * irho;
        S[2] = -(fx * m[1] + fe * m[4] + fz * m[7]) * irho;
        S[3] = -(fx * m[2] + fe * m[5] + fz * m[8]) * irho - (rhop * irho) * A.g;
    }
#pragma unroll
    for (int f = 1; f <= 4; ++f)  // advection of u, v, w, theta (Eq. 1b, 1c)
        S[f] = ((f == 4) ? 0.0 : S[f]) - (Ux * gx[f * FS] + Ue * ge[f * FS] + Uz * gz[f * FS]);
    {   // divergence of F = rho u (Eq. 1a)
        double div = gx[5 * FS] * m[0] + ge[5 * FS] * m[3] + gz[5 * FS] * m[6];
        div += gx[6 * FS] * m[1] + ge[6 * FS] * m[4] + gz[6 * FS] * m[7];
        div += gx[7 * FS] * m[2] + ge[7 * FS] * m[5] + gz[7 * FS] * m[8];
        S[0] = -div;
    }
    // A8: heating, Coriolis, sponge
    S[4] += heat;
    S[1] += A.f_cor * v;
    S[2] -= A.f_cor * u;
    S[1] -= beta * u; S[2] -= beta * v; S[3] -= beta * w; S[4] -= beta * qv[rr][4];
    // A6: weight; A9: walls on the weighted velocity tendency
    double r[5];
#pragma unroll
    for (int c = 0; c < 5; ++c) r[c] = om * S[c];
    if (A.has_walls) {
        const bool on_face = (i == 0) | (i == Nq - 1) | (j == 0) | (j == Nq - 1) | (k == 0) | (k == Nq - 1);
        if (on_face) {
            const int64_t e = e0 + x.le;
            const uint2 bcw = *reinterpret_cast<const uint2 *>(A.face_bc + e * 8);
            if (bcw.x | bcw.y) {
                // copies made only on this rare path: the out-of-line call needs its operands in
                // local memory, and m[] / r[] themselves must stay in registers for everyone else
                WallIO io;
#pragma unroll
                for (int c = 0; c < 9; ++c) io.m[c] = m[c];
                io.r[0] = r[1]; io.r[1] = r[2]; io.r[2] = r[3];
                wall_project_cold<Nq>(bcw, i, j, k, &io);
                r[1] = io.r[0]; r[2] = io.r[1]; r[3] = io.r[2];
            }
        }
    }
    // A10 as a DSS partial sum
    double *qop = A.qout + p;
    if (same) {
        const double a01 = A.a0 + A.a1;
#pragma unroll
        for (int c = 0; c < 5; ++c) VST(qop + c * NL, om * (a01 * qv[rr][c]) + A.b_dt * r[c]);
    } else {
#pragma unroll
        for (int c = 0; c < 5; ++c)
            VST(qop + c * NL, om * (A.a0 * q0v[c] + A.a1 * qv[rr][c]) + A.b_dt * r[c]);
    }
    }  // rr
}

// ---------------------------------------------------------------------------------------
// DSS by multiplicity class (Alg. 3 gather + scatter, deterministic): one thread per shared
// global node; the copy lists of the nodes with C copies are stored transposed
// (idx[a*n + t]) so that the index loads coalesce and carry no dependent chain; all 5*C
// values are loaded before the first store.  Sum in ascending local index.
// ---------------------------------------------------------------------------------------

// the copies are touched once per launch by this SM: keep them out of L1 (ld/st .cg)
#define DSS_LD(p) __ldcg(p)
#define DSS_ST(p, v) __stcg(p, v)

template <int C, int F>
__device__ __forceinline__ void dss_node(double *rm, const int32_t *__restrict__ idx, int64_t n,
                                         int64_t t, int64_t NL)
{
    int32_t id[C];
#pragma unroll
    for (int a = 0; a < C; ++a) id[a] = idx[a * n + t];
    double v[F][C];
#pragma unroll
    for (int m = 0; m < F; ++m)
#pragma unroll
        for (int a = 0; a < C; ++a) v[m][a] = DSS_LD(rm + m * NL + id[a]);
#pragma unroll
    for (int m = 0; m < F; ++m) {
        double s = v[m][0];
#pragma unroll
        for (int a = 1; a < C; ++a) s += v[m][a];
#pragma unroll
        for (int a = 0; a < C; ++a) DSS_ST(rm + m * NL + id[a], s);
    }
}

// block = NUMA_DSS_THREADS shared nodes, F fields per thread (5: the state; 4: hyper-diffusion)
#define NUMA_DSS_MINB 20  /* 32-thread blocks: 640 threads per SM, 96 registers; measured: neither more nor fewer is faster at N <= 5 */
#define NUMA_DSS_MINB_HI 32 /* (1024 threads per SM) N >= 6 on the compact layout (64 registers): N=7 0.394 / 0.366 / 0.359 ms at 10 / 14 / 16; N=4 prefers 10 */
template <int F, int MINB>
__global__ void __launch_bounds__(NUMA_DSS_THREADS, MINB)
k_stage_dss(double *r, const int32_t *__restrict__ idx, const DssSeg *__restrict__ segs,
            const int32_t *__restrict__ blkmap, const int32_t *__restrict__ nodes,
            const int32_t *__restrict__ start, const int32_t *__restrict__ copies, int64_t NL, int blk_off)
{
    const int bid = blk_off + (int)blockIdx.x;
    const DssSeg sg = segs[blkmap[bid]];
    const int t = (bid - sg.blk0) * NUMA_DSS_THREADS + threadIdx.x;
    if (t >= sg.n) return;
    double *rm = r;
    if (sg.cls == 0) {
        dss_node<2, F>(rm, idx + sg.idx_base, sg.n, t, NL);
    } else if (sg.cls == 1) {
        dss_node<4, F>(rm, idx + sg.idx_base, sg.n, t, NL);
    } else if (sg.cls == 2) {
        dss_node<8, F>(rm, idx + sg.idx_base, sg.n, t, NL);
    } else {
        const int gI = nodes[sg.node_off + t];
        const int s = start[gI], c = start[gI + 1] - s;
        for (int m = 0; m < F; ++m) {
            double *rf = rm + (int64_t)m * NL;
            double sum = rf[copies[s]];
            for (int a = 1; a < c; ++a) sum += rf[copies[s + a]];
            for (int a = 0; a < c; ++a) rf[copies[s + a]] = sum;
        }
    }
}

// natural [nf][NL] <-> block-shell [nf][GFS]; one thread per natural node, so the natural side
// is coalesced and the shell side is a gather / scatter inside the block's record (run once
// per numa_step_rk3 call, not per stage)
template <bool TO_SHELL>
__global__ void k_shell_layout(const double *__restrict__ src, double *__restrict__ dst,
                               const int32_t *__restrict__ pos, int64_t NL, int64_t GFS, int BS,
                               int nodes_per_block, int nf)
{
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= NL) return;
    const int64_t b = p / nodes_per_block;
    const int bn = (int)(p - b * nodes_per_block);
    const int64_t t = b * BS + __ldg(pos + bn);
    for (int c = 0; c < nf; ++c) {
        if (TO_SHELL) dst[c * GFS + t] = src[c * NL + p];
        else dst[c * NL + p] = src[c * GFS + t];
    }
}

template <int N>
cudaError_t stage_launch(numa_ctx *c, const StageArgs &a, cudaStream_t s)
{
    using SH = StageShape<N>;
    if (c->shell.BS != SH::BS || c->shell.epb != SH::EPB) return cudaErrorInvalidValue;  // layout of this context
    if (!c->attr_stage) {   // per device: a context is bound to one device
        cudaError_t e = cudaFuncSetAttribute(k_stage_volume<N>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SH::SMEM);
        if (e != cudaSuccess) return e;
        c->attr_stage = true;
    }
    const int64_t all_blocks = (c->par.n_elem + SH::EPB - 1) / SH::EPB;
    const int64_t blocks = (a.n_blocks >= 0) ? a.n_blocks : all_blocks - a.blk0;   // n_blocks carries the launch size here
    StageArgs a2 = a;
    a2.n_blocks = all_blocks;
#define STAGE_PF_MULT2 1   /* prefetch distance in half-waves of resident blocks (N=7: 1.605 / 1.626 / 1.732 ms at 1 / 2 / 4) */
    a2.pf_dist = c->n_sm * SH::MIN_BLOCKS * STAGE_PF_MULT2 / 2;
    k_stage_volume<N><<<(unsigned)blocks, SH::THREADS, SH::SMEM, s>>>(a2, c->lgl);
    return cudaGetLastError();
}

template <int N>
int epb_of() { return StageShape<N>::EPB; }

}  // namespace

int stage_epb(int N)
{
    switch (N) {
        case 2: return epb_of<2>();
        case 3: return epb_of<3>();
        case 4: return epb_of<4>();
        case 5: return epb_of<5>();
        case 6: return epb_of<6>();
        case 7: return epb_of<7>();
        case 8: return epb_of<8>();
        default: return 1;
    }
}

cudaError_t launch_stage_volume(numa_ctx *c, double a0, double a1, double b_dt, const double *q0,
                                const double *qs, const double *heat, double *qout, cudaStream_t s,
                                int64_t blk0, int64_t nblk)
{
    LaunchScope ls(c, K_FUSED_VOLUME, s);
    StageArgs a;
    a.qs = qs; a.q0 = q0; a.qout = qout;
    a.ref3 = c->ref3; a.met = c->met; a.omega = c->omega; a.heat = heat; a.beta = c->sponge;
    a.tab = c->shell.tab;
    for (int le = 0; le < 16; ++le) a.first_pos[le] = le < c->shell.epb ? c->shell.first_pos[le] : 0;
    a.face_bc = c->face_bc;
    a.Ne = c->par.n_elem; a.GFS = c->shell.FS;
    a.g = c->par.g; a.gamma = c->gamma; a.f_cor = c->par.f_cor;
    a.a0 = a0; a.a1 = a1; a.b_dt = b_dt;
    a.has_walls = c->has_walls;
    a.pf_dist = 0;
    a.blk0 = blk0; a.n_blocks = nblk;
    // binomial(gamma, n): c_1 = gamma, c_{n+1} = c_n (gamma - n) / (n + 1)
    {
        long double cn = (long double)c->gamma;
        for (int n = 1; n <= 14; ++n) {
            a.eos[n - 1] = (double)cn;
            cn = cn * ((long double)c->gamma - n) / (n + 1);
        }
    }
    switch (c->par.N) {
        case 2: return stage_launch<2>(c, a, s);
        case 3: return stage_launch<3>(c, a, s);
        case 4: return stage_launch<4>(c, a, s);
        case 5: return stage_launch<5>(c, a, s);
        case 6: return stage_launch<6>(c, a, s);
        case 7: return stage_launch<7>(c, a, s);
        case 8: return stage_launch<8>(c, a, s);
        default: return cudaErrorInvalidValue;
    }
}

cudaError_t launch_dss_classes(numa_ctx *c, const DssLists &L, double *r, int64_t stride,
                               int kernel_id, cudaStream_t s, int nf, int64_t blk0, int64_t nblk)
{
    if (nblk < 0) nblk = L.blocks - blk0;
    if (nblk <= 0) return cudaSuccess;
    LaunchScope ls(c, kernel_id, s);
    const bool hi = c->par.N >= 6;   // measured: N=5 0.52 (10) vs 0.56 (16); N=6 0.45 vs 0.44; N=7 0.39 vs 0.36; N=8 0.37 vs 0.34 ms
#define DSS_LAUNCH(F, MB) k_stage_dss<F, MB><<<(unsigned)nblk, NUMA_DSS_THREADS, 0, s>>>(r, L.idx, L.seg, L.blkmap, L.sh_nodes, L.start, L.copies, stride, (int)blk0)
    if (nf == 5) { if (hi) DSS_LAUNCH(5, NUMA_DSS_MINB_HI); else DSS_LAUNCH(5, NUMA_DSS_MINB); }
    else if (nf == 4) { if (hi) DSS_LAUNCH(4, NUMA_DSS_MINB_HI); else DSS_LAUNCH(4, NUMA_DSS_MINB); }
    else return cudaErrorInvalidValue;
#undef DSS_LAUNCH
    return cudaGetLastError();
}

cudaError_t launch_to_shell(numa_ctx *c, const double *q_nat, double *q_int, int nf, cudaStream_t s)
{
    LaunchScope ls(c, K_LAYOUT, s);
    const int npb = c->shell.epb * (int)c->Mn;
    k_shell_layout<true><<<(unsigned)((c->NL + 255) / 256), 256, 0, s>>>(q_nat, q_int, c->shell.pos, c->NL,
                                                                         c->shell.FS, (int)c->shell.BS, npb, nf);
    return cudaGetLastError();
}

cudaError_t launch_from_shell(numa_ctx *c, const double *q_int, double *q_nat, int nf, cudaStream_t s)
{
    LaunchScope ls(c, K_LAYOUT, s);
    const int npb = c->shell.epb * (int)c->Mn;
    k_shell_layout<false><<<(unsigned)((c->NL + 255) / 256), 256, 0, s>>>(q_int, q_nat, c->shell.pos, c->NL,
                                                                          c->shell.FS, (int)c->shell.BS, npb, nf);
    return cudaGetLastError();
}
