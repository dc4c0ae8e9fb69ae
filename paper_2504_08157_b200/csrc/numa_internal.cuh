// Internal declarations of libnuma_b200.so (not part of the C ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "../../include/numa_b200.h"
#include "../../include/numa_b200_measure.h"

#define NUMA_MAX_NQ 9

// LGL derivative matrix and weights, passed BY VALUE as a kernel parameter so that
// compile-time-indexed reads become constant-bank operands.
struct LglTables {
    double D[NUMA_MAX_NQ * NUMA_MAX_NQ];  // D[i*Nq + l] = h_l'(xi_i)  (Alg. 2)
    double w[NUMA_MAX_NQ];                // quadrature weights (Eq. 8)
    // even-odd split of D (H = Nq/2): A[m*H+l] = (D[m][l] + D[m][N-l])/2, B = (D[m][l] - D[m][N-l])/2,
    // C[m] = D[m][H] and M[l] = D[H][l] (odd Nq only); used by the line contraction at N >= 6
    double A[16], B[16], C[4], M[4];
};

// kernel ids of the optional per-kernel CUDA-event timing (numa_profile_*)
enum { K_VOLUME = 0, K_DSS = 1, K_SOURCES = 2, K_RK = 3, K_FUSED_VOLUME = 4, K_FUSED_DSS = 5, K_LAYOUT = 6, K_HD = 7, K_HD_DSS = 8, K_LINOP = 9, K_VEC = 10, K_COUNT = 11 };

#define NUMA_DSS_CHUNK 4096    // positions per DSS locality chunk at N <= 4 (compact layout: 0.605 / 0.515 / 0.497 / 0.504 ms at 1 K / 2 K / 4 K / 8 K on cfg3)
#define NUMA_DSS_CHUNK_HI 32768 // ... at N >= 5 (numa_api.cu, dss_chunk)
#define NUMA_DSS_THREADS 32    // shared nodes per thread block of the DSS kernel (cfg3: 0.492 / 0.515 / 0.536 ms at 32 / 64 / 128)

struct DssSeg {
    int64_t node_off;  // first node of the segment in sh_nodes
    int64_t idx_base;  // start of its transposed copy lists in dss_idx (classes 0..2)
    int32_t n;         // nodes in the segment
    int32_t cls;       // 0,1,2 = 2,4,8 copies; 3 = other
    int32_t blk0;      // first thread block of the segment
    int32_t pad;
};

struct ProfRec { int id; cudaEvent_t a, b; };

// One set of deterministic-DSS lists over an index space of `n_pos` local positions (the
// natural element-local order, or the block-shell order of the fused route).  CSR over global
// nodes (copies ascending within a node) plus the form the DSS kernel reads: the SHARED nodes
// (multiplicity >= 2) sorted by (chunk of NUMA_DSS_CHUNK positions holding their first copy,
// multiplicity class, first copy); a SEGMENT is a run of equal (chunk, class).  Classes 0,1,2
// = 2,4,8 copies keep their copy lists transposed in idx (copy a of node t of the segment at
// idx_base + a*n + t); class 3 = any other multiplicity goes through the CSR lists.
struct DssLists {
    int32_t *start = nullptr;    // [NG+1]
    int32_t *copies = nullptr;   // [NL]
    int32_t *sh_nodes = nullptr; // [n_shared] global ids of the shared nodes, in kernel order
    int32_t *idx = nullptr;      // [<= NL]
    DssSeg *seg = nullptr;       // [n_seg]
    int32_t *blkmap = nullptr;   // [blocks] segment of every thread block of the DSS kernel
    int64_t n_shared = 0, n_seg = 0, blocks = 0;
};

// Block-shell layout of every per-node device array the library keeps or works on
// internally (metric terms, omega, reference state, sponge; the state and heating of the fused
// route): elements are taken in blocks of `epb` consecutive elements; a block record of BS
// positions holds the block's nodes entity by entity (face interiors, edge interiors, corners
// each as contiguous runs, element by element; interior nodes fill the gaps), so the copies of
// shared nodes form long contiguous runs and the DSS touches whole 32-byte sectors.  The order
// is chosen (numa_shell.cpp) so that the volume kernel's thread-per-position shared-memory
// accesses are free of bank conflicts.
struct ShellLayout {
    int epb = 1;             // elements per block (= StageShape<N>::EPB)
    int64_t BS = 0;          // positions per block record (EPB*Mn rounded up to whole warps)
    int64_t n_blocks = 0;
    int64_t FS = 0;          // field stride = n_blocks * BS
    int32_t *pos = nullptr;  // device [epb*Mn]: (element of block, node) -> position
    uint32_t *tab = nullptr; // device [BS]: thread slot -> packed (position lane, node) (numa_stage.cu)
    int first_pos[16] = {0}; // position of node 0 of the le-th element of a block
};

struct GraphKey { const double *q = nullptr, *heat = nullptr; void *scratch = nullptr; double dt = 0.0; cudaStream_t s = nullptr; };

struct numa_ctx {
    numa_params par;
    int device = 0;
    int n_sm = 148;   // multiprocessors of `device` (grid of the persistent kernels)
    int Nq;
    int64_t Mn, NL;
    double gamma;
    LglTables lgl;
    // device tables, all inside the caller's workspace
    // (block-shell order, field stride shell.FS)
    double *met;     // [9][FS]   d xi_a / d x_c
    double *omega;   // [FS]      wJ / M
    double *ref3;    // [3][FS]   rho0, theta0, p0
    double *sponge;  // [FS] or nullptr
    DssLists dss_nat;     // natural element-local order (numa_dss_or_flux, mass)
    DssLists dss_int;     // block-shell order (fused stage)
    ShellLayout shell;
    uint8_t *face_bc;     // [Ne][8] (padded to 8 bytes per element)
    int32_t *d_flags;     // [4] device error flags
    int has_walls;
    bool fused_ok = true;   // the wall projector is single-valued at every wall node (k_check_walls)
    // tensor hyper-diffusion (numa_hd_init): tau[6][FS] block-shell and two 4-field work buffers
    double *hd_tau = nullptr, *hd_buf = nullptr, *hd_buf2 = nullptr;
    bool hd_on = false;
    // IMEX (numa_imex_init): inv_mult[NL] followed by the Krylov and ARK work vectors
    char *imex_ws = nullptr;
    int imex_m = 0;
    bool attr_rhs = false, attr_stage = false;  // dynamic-shared-memory attribute set on this device
    int64_t launches;
    std::string err;
    // CUDA graph of one SSP-RK3 step (numa_step_rk3_graph)
    cudaGraphExec_t graph = nullptr;
    int64_t graph_launches = 0;   // kernels in the captured step (counted by enqueue_step at capture)
    GraphKey graph_key;
    cudaStream_t gstream = nullptr;   // used when the caller's stream is the legacy default stream
    cudaEvent_t gev0 = nullptr, gev1 = nullptr;
    // per-kernel event timing
    bool prof = false;
    std::vector<ProfRec> recs;
    std::vector<cudaEvent_t> pool;
    double prof_ms[K_COUNT] = {0};
    int64_t prof_n[K_COUNT] = {0};
};

// RAII: counts the launch and, when profiling is on, brackets it with events on the stream
struct LaunchScope {
    numa_ctx *c; int id; cudaStream_t s; cudaEvent_t a = nullptr, b = nullptr;
    static cudaEvent_t get(numa_ctx *c)
    {
        cudaEvent_t e;
        if (!c->pool.empty()) { e = c->pool.back(); c->pool.pop_back(); return e; }
        cudaEventCreate(&e);
        return e;
    }
    LaunchScope(numa_ctx *c_, int id_, cudaStream_t s_) : c(c_), id(id_), s(s_)
    {
        c->launches++;
        if (c->prof) { a = get(c); b = get(c); cudaEventRecord(a, s); }
    }
    ~LaunchScope()
    {
        if (c->prof) { cudaEventRecord(b, s); c->recs.push_back({id, a, b}); }
    }
};

// host-side table construction (tables.cpp part of numa_api.cu)
void numa_build_lgl(int N, LglTables *t);

// kernel launchers (numa_kernels.cu); all return cudaError_t of the launch
cudaError_t launch_metrics(numa_ctx *c, const double *xyz, double *wJ_out, cudaStream_t s);
cudaError_t launch_mass(numa_ctx *c, cudaStream_t s);
cudaError_t launch_rhs(numa_ctx *c, const double *q, double *rhs, cudaStream_t s);
cudaError_t launch_sources(numa_ctx *c, const double *q, const double *heat, double *rhs,
                           cudaStream_t s);
cudaError_t launch_rk(numa_ctx *c, double a0, double a1, double b_dt, const double *q0,
                      const double *qs, const double *rhs, double *qout, cudaStream_t s);
// fused stage (numa_stage.cu): volume + sources + walls + RK written as DSS partial sums into
// the block-shell state, then the in-place DSS by multiplicity class.  q0, qs, qout are
// block-shell arrays [5][shell.FS]; heat is block-shell [shell.FS] or nullptr.
cudaError_t launch_stage_volume(numa_ctx *c, double a0, double a1, double b_dt, const double *q0,
                                const double *qs, const double *heat, double *qout,
                                cudaStream_t s, int64_t blk0 = 0, int64_t nblk = -1);
// in-place DSS of r[5][stride] over one list set (kernel_id = profiling slot)
cudaError_t launch_dss_classes(numa_ctx *c, const DssLists &L, double *r, int64_t stride,
                               int kernel_id, cudaStream_t s, int nf = 5, int64_t blk0 = 0, int64_t nblk = -1);
// hyper-diffusion inside a fused stage (numa_hd.cu): h1 = DSS(omega L(qs[1..4])) before the volume
// kernel; qout[1..4] += -b_dt P(omega L(h1)) after it (block-shell arrays)
cudaError_t hd_stage_first(numa_ctx *c, const double *qs, cudaStream_t s);
cudaError_t hd_stage_second(numa_ctx *c, double b_dt, double *qout, cudaStream_t s);
// natural [nf][NL] <-> block-shell [nf][shell.FS]
cudaError_t launch_to_shell(numa_ctx *c, const double *q_nat, double *q_int, int nf, cudaStream_t s);
cudaError_t launch_from_shell(numa_ctx *c, const double *q_int, double *q_nat, int nf, cudaStream_t s);
// elements per block of the fused volume kernel for order N (fixes the block-shell layout)
int stage_epb(int N);
// host (numa_shell.cpp): tables of the block-shell layout for (N, epb): pos[le*Mn + n] and the
// packed thread-slot table tab[BS]
void numa_build_shell_pos(int N, int epb, int64_t BS, std::vector<int32_t> &pos,
                          std::vector<uint32_t> &tab);

#ifdef __CUDACC__
// No-flux wall projection at one node (A9): faces in order 0..5; n = -+ grad xi_a/|grad xi_a|.
template <int Nq>
__device__ __forceinline__ void wall_project(const uint8_t *__restrict__ bc, int i, int j, int k,
                                             const double (&m)[9], double &ru, double &rv,
                                             double &rw)
{
    const int idx[3] = {i, j, k};
#pragma unroll
    for (int f = 0; f < 6; ++f) {
        const int a = f >> 1;
        const bool on = bc[f] && (idx[a] == ((f & 1) ? (Nq - 1) : 0));
        if (on) {
            const double gx = m[3 * a + 0], gy = m[3 * a + 1], gz = m[3 * a + 2];
            const double inv = 1.0 / sqrt(gx * gx + gy * gy + gz * gz);
            const double sgn = (f & 1) ? inv : -inv;
            const double nx = sgn * gx, ny = sgn * gy, nz = sgn * gz;
            const double rn = ru * nx + rv * ny + rw * nz;
            ru -= rn * nx; rv -= rn * ny; rw -= rn * nz;
        }
    }
}
#endif  // __CUDACC__
