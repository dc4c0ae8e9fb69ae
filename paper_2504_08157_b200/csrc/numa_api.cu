// C-ABI entry points of libnuma_b200.so (include/numa_b200.h) and the A0 setup.
#include <cub/cub.cuh>
#include <thrust/iterator/counting_iterator.h>

#include <cmath>
#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>
#include <new>

#include "numa_internal.cuh"

static thread_local std::string g_err;  // errors raised without a context

// ---------------------------------------------------------------------------------------
// Host tables.  LGL points as the roots of q(x) = P_{N+1}(x) - P_{N-1}(x) (which vanish at
// +-1 and at the roots of P'_N), Newton with q'(x) = (2N+1) P_N(x); derivative matrix from
// barycentric weights.  (Eq. 5; Eq. 8.)
// ---------------------------------------------------------------------------------------
static void legendre_q(int N, long double x, long double *q, long double *dq, long double *PN)
{
    long double pm1 = 1.0L, p = x;  // P_0, P_1
    for (int n = 1; n < N; ++n) {
        long double pn = ((2 * n + 1) * x * p - n * pm1) / (n + 1);
        pm1 = p; p = pn;
    }
    // now p = P_N, pm1 = P_{N-1};  P_{N+1} from the same recurrence
    long double pp1 = ((2 * N + 1) * x * p - N * pm1) / (N + 1);
    *q = pp1 - pm1;
    *dq = (2 * N + 1) * p;
    *PN = p;
}

void numa_build_lgl(int N, LglTables *t)
{
    const int Nq = N + 1;
    long double x[NUMA_MAX_NQ], PN[NUMA_MAX_NQ];
    const long double pi = 3.14159265358979323846264338327950288L;
    for (int i = 0; i < Nq; ++i) {
        long double xi = -cosl(pi * i / N);
        long double q, dq, p;
        if (i == 0) xi = -1.0L;
        else if (i == N) xi = 1.0L;
        else {
            // deflated Newton keeps distinct roots distinct
            for (int it = 0; it < 100; ++it) {
                legendre_q(N, xi, &q, &dq, &p);
                long double s = 0.0L;
                for (int m = 0; m < i; ++m) s += 1.0L / (xi - x[m]);
                long double dx = q / (dq - q * s);
                xi -= dx;
                if (fabsl(dx) < 1e-19L) break;
            }
        }
        x[i] = xi;
    }
    for (int i = 0; i < Nq / 2; ++i) {  // exact symmetry
        long double a = 0.5L * (x[N - i] - x[i]);
        x[i] = -a; x[N - i] = a;
    }
    if (N % 2 == 0) x[N / 2] = 0.0L;
    for (int i = 0; i < Nq; ++i) {
        long double q, dq;
        legendre_q(N, x[i], &q, &dq, &PN[i]);
        t->w[i] = (double)(2.0L / (N * (N + 1.0L) * PN[i] * PN[i]));
    }
    long double bw[NUMA_MAX_NQ];
    for (int j = 0; j < Nq; ++j) {
        long double prod = 1.0L;
        for (int k = 0; k < Nq; ++k)
            if (k != j) prod *= (x[j] - x[k]);
        bw[j] = 1.0L / prod;
    }
    for (int i = 0; i < NUMA_MAX_NQ * NUMA_MAX_NQ; ++i) t->D[i] = 0.0;
    for (int i = 0; i < Nq; ++i) {
        long double diag = 0.0L;
        for (int l = 0; l < Nq; ++l) {
            if (l == i) continue;
            long double d = (bw[l] / bw[i]) / (x[i] - x[l]);
            t->D[i * Nq + l] = (double)d;
            diag -= d;
        }
        t->D[i * Nq + i] = (double)diag;
    }
    {   // even-odd split, from the long double values
        const int H = Nq / 2;
        for (int k = 0; k < 16; ++k) t->A[k] = t->B[k] = 0.0;
        for (int k = 0; k < 4; ++k) t->C[k] = t->M[k] = 0.0;
        auto Dld = [&](int i, int l) -> long double {
            if (i == l) { long double d = 0.0L; for (int k = 0; k < Nq; ++k) if (k != i) d -= (bw[k] / bw[i]) / (x[i] - x[k]); return d; }
            return (bw[l] / bw[i]) / (x[i] - x[l]);
        };
        for (int m = 0; m < H; ++m) {
            for (int l = 0; l < H; ++l) {
                t->A[m * H + l] = (double)(0.5L * (Dld(m, l) + Dld(m, N - l)));
                t->B[m * H + l] = (double)(0.5L * (Dld(m, l) - Dld(m, N - l)));
            }
            if (Nq & 1) t->C[m] = (double)Dld(m, H);
        }
        if (Nq & 1) for (int l = 0; l < H; ++l) t->M[l] = (double)Dld(H, l);
    }
    // exact centro-antisymmetry D[N-i][N-l] = -D[i][l] (the kernels use only the upper half)
    for (int i = 0; i < Nq; ++i)
        for (int l = 0; l < Nq; ++l) {
            const int a = i * Nq + l, b = (N - i) * Nq + (N - l);
            if (a < b) t->D[b] = -t->D[a];
            else if (a == b) t->D[a] = 0.0;
        }
}

// ---------------------------------------------------------------------------------------
// workspace layout
// ---------------------------------------------------------------------------------------
static inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

static const size_t kSmallTmp = (size_t)4 << 20;  // CUB temp storage for small meshes
static const size_t kSmallScr = (size_t)2 << 20;  // list-building scratch for meshes too small to lend their `met` region

struct DssOff { size_t start, copies, sh_nodes, idx, seg, blkmap; };

struct WsLayout {
    size_t met, omega, ref3, sponge, face_bc, flags, small_tmp, shell_pos, shell_inv, shell_tab, total;
    DssOff nat, shl;
    ShellLayout shell;  // sizes only (pos = nullptr)
};

static inline size_t WsMaxSeg(size_t n_pos) { return 4 * (n_pos / NUMA_DSS_CHUNK + 2); }   // sized for the smaller chunk
// positions per DSS locality chunk: measured on the block-shell layout (cfg3 / cfg4, ms per launch)
//   N=4: 0.69 / 0.53 / 0.53 / 0.55 at 512 / 2048 / 8192 / 32768;  N=7: 0.70 / 0.55 / 0.50 / 0.48;  N=8: 0.67 / 0.54 / 0.49 / 0.46
static inline int64_t dss_chunk(int N) { return N <= 4 ? NUMA_DSS_CHUNK : NUMA_DSS_CHUNK_HI; }

static bool params_ok(const numa_params *p)
{
    return p && p->N >= 2 && p->N <= 8 && p->n_elem > 0 && p->n_global > 0 &&
           p->n_elem * (int64_t)((p->N + 1) * (p->N + 1) * (p->N + 1)) < (int64_t)2147483647 - 65536 &&
           p->n_global < (int64_t)2147483647 && p->c_v > 0 && p->c_p > 0 && p->p_a > 0 && p->R_gas > 0;
}

static ShellLayout shell_sizes(const numa_params *p)
{
    ShellLayout sh;
    const int64_t Nq = p->N + 1, Mn = Nq * Nq * Nq;
    sh.epb = stage_epb(p->N);
    sh.BS = (sh.epb * Mn + 31) / 32 * 32;   // whole warps: every block record starts on a 256-byte line
    sh.n_blocks = (p->n_elem + sh.epb - 1) / sh.epb;
    sh.FS = sh.n_blocks * sh.BS;
    return sh;
}

static size_t dss_layout(DssOff &d, size_t off, size_t n_pos, size_t NG)
{
    const size_t max_seg = WsMaxSeg(n_pos);
    d.start = off; off = align_up(off + (NG + 1) * 4);
    d.copies = off; off = align_up(off + n_pos * 4);
    d.sh_nodes = off; off = align_up(off + (NG + 1) * 4);
    d.idx = off; off = align_up(off + n_pos * 4);
    d.seg = off; off = align_up(off + max_seg * sizeof(DssSeg));
    d.blkmap = off; off = align_up(off + (NG / NUMA_DSS_THREADS + max_seg + 1) * 4);
    return off;
}

static WsLayout ws_layout(const numa_params *p)
{
    WsLayout L;
    const size_t Nq = p->N + 1, Mn = Nq * Nq * Nq, NL = (size_t)p->n_elem * Mn;
    L.shell = shell_sizes(p);
    size_t off = 0;
    const size_t FS = (size_t)L.shell.FS;   // the tables are block-shell arrays
    L.met = off; off = align_up(off + 9 * FS * 8);
    L.omega = off; off = align_up(off + FS * 8);
    L.ref3 = off; off = align_up(off + 3 * FS * 8);
    L.sponge = off; off = align_up(off + FS * 8);
    off = dss_layout(L.nat, off, NL, (size_t)p->n_global);
    off = dss_layout(L.shl, off, (size_t)L.shell.FS, (size_t)p->n_global);
    L.shell_pos = off; off = align_up(off + (size_t)L.shell.epb * Mn * 4);
    L.shell_inv = off; off = align_up(off + (size_t)L.shell.BS * 4);
    L.shell_tab = off; off = align_up(off + (size_t)L.shell.BS * 4);
    L.face_bc = off; off = align_up(off + (size_t)p->n_elem * 8);
    L.flags = off; off = align_up(off + 256);
    L.small_tmp = off; off = align_up(off + kSmallTmp + kSmallScr);
    L.total = off;
    return L;
}

extern "C" size_t numa_workspace_bytes(const numa_params *p)
{
    if (!params_ok(p)) return 0;
    return ws_layout(p).total;
}

// block-shell scratch of numa_step_rk3: the state of the step, the stage state, the heating
static inline size_t shell_state_bytes(const ShellLayout &sh) { return align_up((size_t)5 * sh.FS * 8); }
static inline size_t shell_field_bytes(const ShellLayout &sh) { return align_up((size_t)sh.FS * 8); }

extern "C" size_t numa_step_scratch_bytes(const numa_params *p)
{
    if (!params_ok(p)) return 0;
    const ShellLayout sh = shell_sizes(p);
    return 2 * shell_state_bytes(sh) + shell_field_bytes(sh);
}

// the layout tables depend on (N, epb) only: built once per process
struct ShellTables { std::vector<int32_t> pos; std::vector<uint32_t> tab; };
static const ShellTables &shell_tables(int N, int epb, int64_t BS)
{
    static std::mutex mu;
    static std::map<std::pair<int, int>, ShellTables> cache;
    std::lock_guard<std::mutex> lock(mu);
    auto key = std::make_pair(N, epb);
    auto it = cache.find(key);
    if (it == cache.end()) {
        ShellTables t;
        numa_build_shell_pos(N, epb, BS, t.pos, t.tab);
        it = cache.emplace(key, std::move(t)).first;
    }
    return it->second;
}

// ---------------------------------------------------------------------------------------
// setup kernels
// ---------------------------------------------------------------------------------------
// every intma_cg entry must lie in [0, NG): checked BEFORE anything is indexed with it
__global__ void k_check_ids(const int32_t *__restrict__ cg, int64_t n, int64_t NG, int32_t *flags)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    int bad = 0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const int32_t g = cg[i];
        bad |= (g < 0 || g >= NG);
    }
    if (bad) atomicOr(flags + 1, 1);
}

// sort input of one list set: position t of the index space -> (key = global id, value = t).
// Natural order: t = local node.  Block-shell order: t = b*BS + r, r -> (le, n) through the
// inverse table; holes of the layout (padding, elements past Ne) get the sentinel key NG.
__global__ void k_sort_input(int32_t *__restrict__ vals, int32_t *__restrict__ keys,
                             const int32_t *__restrict__ cg, int64_t n_pos, int64_t NG,
                             const int32_t *__restrict__ inv, int64_t BS, int epb, int64_t Mn,
                             int64_t Ne)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < n_pos; t += stride) {
        int32_t key;
        if (inv == nullptr) key = cg[t];
        else {
            const int64_t b = t / BS, r = t - b * BS;
            const int32_t ln = inv[r];  // le*Mn + n, or -1
            const int64_t e = b * epb + (ln >= 0 ? ln / Mn : 0);
            key = (ln >= 0 && e < Ne) ? cg[e * Mn + (ln % Mn)] : (int32_t)NG;
        }
        keys[t] = key;
        vals[t] = (int32_t)t;
    }
}

// start[g] = first position in the sorted key array whose key is >= g, g = 0..NG
// (keys are in [0, NG]; NG is the sentinel of layout holes and sorts last)
__global__ void k_find_starts(const int32_t *__restrict__ keys, int32_t *__restrict__ start,
                              int64_t n, int64_t NG)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const int32_t k1 = keys[i];
        const int32_t k0 = (i == 0) ? -1 : keys[i - 1];
        for (int32_t g = k0 + 1; g <= k1; ++g) start[g] = (int32_t)i;
        if (i == n - 1)
            for (int64_t g = (int64_t)k1 + 1; g <= NG; ++g) start[g] = (int32_t)n;
    }
}

struct SharedPred {
    const int32_t *start;
    __device__ bool operator()(int32_t g) const { return start[g + 1] - start[g] >= 2; }
};

// sort key of a shared node: (chunk of its first copy, multiplicity class, first copy);
// class 0,1,2 = 2,4,8 copies, 3 = anything else.
__global__ void k_class_keys(const int32_t *__restrict__ nodes, const int32_t *__restrict__ start,
                             const int32_t *__restrict__ copies, uint64_t *__restrict__ keys,
                             int64_t n, uint32_t chunk)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += stride) {
        const int32_t g = nodes[t];
        const int32_t s = start[g], c = start[g + 1] - s;
        const uint64_t cls = (c == 2) ? 0 : (c == 4) ? 1 : (c == 8) ? 2 : 3;
        const uint32_t first = (uint32_t)copies[s];
        keys[t] = ((uint64_t)(first / chunk) << 34) | (cls << 32) | first;
    }
}

struct SegHeadPred {
    const uint64_t *keys;
    __device__ bool operator()(int32_t t) const { return t == 0 || (keys[t] >> 32) != (keys[t - 1] >> 32); }
};

__global__ void k_gather_hi(const uint64_t *__restrict__ keys, const int32_t *__restrict__ heads,
                            int32_t *__restrict__ hi, int n)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t < n) hi[t] = (int32_t)(keys[heads[t]] >> 32);
}

// transposed copy lists: one thread per shared node, indexed exactly like the DSS kernel
__global__ void __launch_bounds__(NUMA_DSS_THREADS)
k_class_lists(const int32_t *__restrict__ nodes, const int32_t *__restrict__ start,
              const int32_t *__restrict__ copies, int32_t *__restrict__ idx,
              const DssSeg *__restrict__ segs, const int32_t *__restrict__ blkmap)
{
    const DssSeg sg = segs[blkmap[blockIdx.x]];
    const int t = (blockIdx.x - sg.blk0) * NUMA_DSS_THREADS + threadIdx.x;
    if (t >= sg.n || sg.cls > 2) return;
    const int C = 2 << sg.cls;
    const int32_t s = start[nodes[sg.node_off + t]];
    for (int a = 0; a < C; ++a) idx[sg.idx_base + (int64_t)a * sg.n + t] = copies[s + a];
}

// ref (natural) -> ref3 (block-shell): rho0, theta0, p0
__global__ void k_ref3(const double *__restrict__ ref, double *__restrict__ ref3, int64_t NL,
                       double p_a, double R, double gamma, const int32_t *__restrict__ pos, int npb,
                       int BS, int64_t FS)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < NL; p += stride) {
        const int64_t b = p / npb;
        const int64_t t = b * BS + pos[p - b * npb];
        const double rho0 = ref[p], th0 = ref[NL + p];
        ref3[t] = rho0;
        ref3[FS + t] = th0;
        ref3[2 * FS + t] = p_a * pow(rho0 * R * th0 / p_a, gamma);  // Eq. 3 at the background
    }
}

__global__ void k_face_bc(const uint8_t *__restrict__ in, uint8_t *__restrict__ out, int64_t Ne,
                          int32_t *flags)
{
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= Ne) return;
    int any = 0;
    for (int f = 0; f < 6; ++f) { out[e * 8 + f] = in[e * 6 + f] ? 1 : 0; any |= in[e * 6 + f]; }
    out[e * 8 + 6] = 0; out[e * 8 + 7] = 0;
    if (any) atomicOr(flags + 2, 1);
}

// Preconditions (2) and (3) of the fused route (include/numa_b200.h): the no-flux projector must be
// the same in every element that shares a wall node.  One thread per shared global node applies the
// projector of every copy (its element's wall faces, its own metric normals) to the three unit
// vectors and compares with the first copy; flags[3] is raised where they differ by more than 1e-10
// (curved or terrain-following walls; an element that touches a wall node without owning a wall face).
__global__ void k_check_walls(const int32_t *__restrict__ start, const int32_t *__restrict__ copies,
                              const double *__restrict__ met, const uint8_t *__restrict__ face_bc,
                              const int32_t *__restrict__ pos, int npb, int BS, int64_t FS, int Nq,
                              int64_t NG, int32_t *flags)
{
    const int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= NG) return;
    const int s0 = start[g], c = start[g + 1] - s0;
    if (c < 2) return;
    const int Mn = Nq * Nq * Nq;
    double P0[9];
    for (int a = 0; a < c; ++a) {
        const int64_t p = copies[s0 + a];
        const int64_t e = p / Mn;
        const int n = (int)(p - e * Mn);
        const int idx[3] = {n % Nq, (n / Nq) % Nq, n / (Nq * Nq)};
        const int64_t b = p / npb;
        const int64_t t = b * BS + pos[(int)(p - b * npb)];
        double P[9] = {1, 0, 0, 0, 1, 0, 0, 0, 1};   // columns = projected unit vectors
        for (int f = 0; f < 6; ++f) {
            const int d = f >> 1;
            if (!face_bc[e * 8 + f] || idx[d] != ((f & 1) ? Nq - 1 : 0)) continue;
            const double gx = met[(3 * d + 0) * FS + t], gy = met[(3 * d + 1) * FS + t], gz = met[(3 * d + 2) * FS + t];
            const double inv = 1.0 / sqrt(gx * gx + gy * gy + gz * gz);
            const double nx = gx * inv, ny = gy * inv, nz = gz * inv;   // the sign drops out of n n^T
            for (int col = 0; col < 3; ++col) {
                const double rn = P[col] * nx + P[3 + col] * ny + P[6 + col] * nz;
                P[col] -= rn * nx; P[3 + col] -= rn * ny; P[6 + col] -= rn * nz;
            }
        }
        if (a == 0) {
            for (int k = 0; k < 9; ++k) P0[k] = P[k];
        } else {
            double dmax = 0.0;
            for (int k = 0; k < 9; ++k) dmax = fmax(dmax, fabs(P[k] - P0[k]));
            if (dmax > 1e-10) atomicOr(flags + 3, 1);
        }
    }
}

#define CK(call)                                                                        \
    do {                                                                                \
        cudaError_t e_ = (call);                                                        \
        if (e_ != cudaSuccess) {                                                        \
            char buf[512];                                                              \
            snprintf(buf, sizeof buf, "%s:%d: %s: %s", __FILE__, __LINE__, #call,       \
                     cudaGetErrorString(e_));                                           \
            errstr = buf;                                                               \
            return false;                                                               \
        }                                                                               \
    } while (0)

static inline unsigned grid_for(int64_t n, int threads = 256, int64_t cap = 148 * 32)
{
    int64_t b = (n + threads - 1) / threads;
    if (b > cap) b = cap;
    if (b < 1) b = 1;
    return (unsigned)b;
}

// Builds one DssLists set over `n_pos` positions.  scr/scr_end: device scratch (the not yet
// written `met` region); small_tmp: fallback CUB temp storage of kSmallTmp bytes.
// inv == nullptr: natural order (position = local node).
static bool build_dss_lists(numa_ctx *c, DssLists &D, const int32_t *cg, int64_t n_pos,
                            const int32_t *inv, char *scr, char *scr_end, char *small_tmp,
                            cudaStream_t s, std::string &errstr)
{
    const int64_t NG = c->par.n_global;
    {   // tiny meshes: the `met` region is smaller than the lists' scratch; use the fixed one
        const size_t need_scr = 16 * (size_t)n_pos + 24 * (size_t)NG + 8 * 256;
        if ((size_t)(scr_end - scr) < need_scr) {
            if (need_scr > kSmallScr) { errstr = "internal: setup scratch does not fit"; return false; }
            scr = small_tmp + kSmallTmp;
            scr_end = scr + kSmallScr;
        }
    }
    int32_t *keysA = (int32_t *)scr;
    int32_t *keysB = keysA + n_pos;
    int32_t *valsA = keysB + n_pos;
    int32_t *valsB = valsA + n_pos;
    char *after = (char *)align_up((size_t)(valsB + n_pos));
    void *cub_tmp = (void *)after;
    size_t cub_avail = after < scr_end ? (size_t)(scr_end - after) : 0;
    if (cub_avail < kSmallTmp) { cub_tmp = small_tmp; cub_avail = kSmallTmp; }
    if (after > scr_end) { errstr = "internal: setup scratch does not fit"; return false; }
    k_sort_input<<<grid_for(n_pos), 256, 0, s>>>(valsA, keysA, cg, n_pos, NG, inv, c->shell.BS,
                                                 c->shell.epb, c->Mn, c->par.n_elem);
    CK(cudaGetLastError());
    int end_bit = 1;
    while (((int64_t)1 << end_bit) <= NG) ++end_bit;  // keys reach the sentinel NG
    cub::DoubleBuffer<int32_t> dk(keysA, keysB), dv(valsA, valsB);
    size_t need = 0;
    CK(cub::DeviceRadixSort::SortPairs(nullptr, need, dk, dv, (int)n_pos, 0, end_bit, s));
    if (need > cub_avail) { errstr = "internal: CUB scratch does not fit"; return false; }
    CK(cub::DeviceRadixSort::SortPairs(cub_tmp, need, dk, dv, (int)n_pos, 0, end_bit, s));
    k_find_starts<<<grid_for(n_pos), 256, 0, s>>>(dk.Current(), D.start, n_pos, NG);
    CK(cudaGetLastError());
    CK(cudaMemcpyAsync(D.copies, dv.Current(), (size_t)n_pos * 4, cudaMemcpyDeviceToDevice, s));
    c->launches += 4;
    // --- SHARED global nodes (multiplicity >= 2), sorted by (chunk, multiplicity class, first
    // copy), and the transposed per-class copy lists of the DSS kernel
    SharedPred pred{D.start};
    thrust::counting_iterator<int32_t> ids(0);
    int32_t *d_num = c->d_flags + 8;
    int32_t *nodesA = (int32_t *)after;                          // [NG]
    int32_t *nodesB = nodesA + NG;                               // [NG]
    uint64_t *kA = (uint64_t *)align_up((size_t)(nodesB + NG));  // [NG]
    uint64_t *kB = kA + NG;
    char *tmp2c = (char *)align_up((size_t)(kB + NG));
    void *tmp2 = tmp2c;
    if (tmp2c > scr_end) { errstr = "internal: setup scratch does not fit"; return false; }
    size_t avail2 = (size_t)(scr_end - tmp2c), need2 = 0;
    if (avail2 < kSmallTmp) { tmp2 = small_tmp; avail2 = kSmallTmp; }
    CK(cub::DeviceSelect::If(nullptr, need2, ids, nodesA, d_num, (int)NG, pred, s));
    if (need2 > avail2) { errstr = "internal: CUB scratch does not fit"; return false; }
    CK(cub::DeviceSelect::If(tmp2, need2, ids, nodesA, d_num, (int)NG, pred, s));
    int32_t h_num = 0;
    CK(cudaMemcpyAsync(&h_num, d_num, 4, cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    D.n_shared = h_num;
    D.n_seg = 0;
    D.blocks = 0;
    if (h_num == 0) return true;
    const uint32_t chunk = (uint32_t)dss_chunk(c->par.N);
    k_class_keys<<<grid_for(h_num), 256, 0, s>>>(nodesA, D.start, D.copies, kA, h_num, chunk);
    CK(cudaGetLastError());
    int end_bit2 = 35;
    while (((int64_t)chunk << (end_bit2 - 34)) < n_pos) ++end_bit2;
    cub::DoubleBuffer<uint64_t> dk2(kA, kB);
    cub::DoubleBuffer<int32_t> dv2(nodesA, nodesB);
    CK(cub::DeviceRadixSort::SortPairs(nullptr, need2, dk2, dv2, h_num, 0, end_bit2, s));
    if (need2 > avail2) { errstr = "internal: CUB scratch does not fit"; return false; }
    CK(cub::DeviceRadixSort::SortPairs(tmp2, need2, dk2, dv2, h_num, 0, end_bit2, s));
    CK(cudaMemcpyAsync(D.sh_nodes, dv2.Current(), (size_t)h_num * 4, cudaMemcpyDeviceToDevice, s));
    // segment heads (positions where (chunk, class) changes), ascending
    const size_t max_seg = WsMaxSeg((size_t)n_pos);
    int32_t *heads = dv2.Alternate();  // [<= h_num], free after the sort
    int32_t *hi = (int32_t *)dk2.Alternate();  // [<= h_num] ints inside a free [NG] uint64 buffer
    SegHeadPred hp{dk2.Current()};
    CK(cub::DeviceSelect::If(nullptr, need2, ids, heads, d_num, h_num, hp, s));
    if (need2 > avail2) { errstr = "internal: CUB scratch does not fit"; return false; }
    CK(cub::DeviceSelect::If(tmp2, need2, ids, heads, d_num, h_num, hp, s));
    int32_t n_seg = 0;
    CK(cudaMemcpyAsync(&n_seg, d_num, 4, cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    if ((size_t)n_seg > max_seg) { errstr = "internal: DSS segment table does not fit"; return false; }
    k_gather_hi<<<(n_seg + 255) / 256, 256, 0, s>>>(dk2.Current(), heads, hi, n_seg);
    CK(cudaGetLastError());
    std::vector<int32_t> h_heads(n_seg), h_hi(n_seg);
    CK(cudaMemcpyAsync(h_heads.data(), heads, (size_t)n_seg * 4, cudaMemcpyDeviceToHost, s));
    CK(cudaMemcpyAsync(h_hi.data(), hi, (size_t)n_seg * 4, cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    std::vector<DssSeg> h_seg(n_seg);
    std::vector<int32_t> h_map;
    int64_t idx_off = 0, blk = 0;
    for (int k = 0; k < n_seg; ++k) {
        DssSeg &sg = h_seg[k];
        sg.node_off = h_heads[k];
        sg.n = (k + 1 < n_seg ? h_heads[k + 1] : h_num) - h_heads[k];
        sg.cls = h_hi[k] & 3;
        sg.idx_base = idx_off;
        sg.blk0 = (int32_t)blk;
        sg.pad = 0;
        if (sg.cls < 3) idx_off += (int64_t)sg.n * (2 << sg.cls);
        const int nb = (sg.n + NUMA_DSS_THREADS - 1) / NUMA_DSS_THREADS;
        h_map.insert(h_map.end(), nb, k);
        blk += nb;
    }
    if ((size_t)blk > (size_t)NG / NUMA_DSS_THREADS + max_seg + 1 || idx_off > n_pos) {
        errstr = "internal: DSS tables do not fit";
        return false;
    }
    D.n_seg = n_seg;
    D.blocks = blk;
    CK(cudaMemcpyAsync(D.seg, h_seg.data(), (size_t)n_seg * sizeof(DssSeg), cudaMemcpyHostToDevice, s));
    CK(cudaMemcpyAsync(D.blkmap, h_map.data(), (size_t)blk * 4, cudaMemcpyHostToDevice, s));
    k_class_lists<<<(unsigned)blk, NUMA_DSS_THREADS, 0, s>>>(D.sh_nodes, D.start, D.copies, D.idx,
                                                            D.seg, D.blkmap);
    CK(cudaGetLastError());
    CK(cudaStreamSynchronize(s));  // h_seg / h_map are read by the copies above
    c->launches += 6;
    return true;
}

static void bind_lists(DssLists &D, char *ws, const DssOff &o)
{
    D.start = (int32_t *)(ws + o.start);
    D.copies = (int32_t *)(ws + o.copies);
    D.sh_nodes = (int32_t *)(ws + o.sh_nodes);
    D.idx = (int32_t *)(ws + o.idx);
    D.seg = (DssSeg *)(ws + o.seg);
    D.blkmap = (int32_t *)(ws + o.blkmap);
}

static bool init_device_tables(numa_ctx *c, const WsLayout &L, char *ws, const double *xyz,
                               const int32_t *intma_cg, const uint8_t *face_bc, const double *ref,
                               const double *sponge, cudaStream_t s, numa_status &result,
                               std::string &errstr)
{
    const numa_params *p = &c->par;
    const int64_t NL = c->NL, NG = p->n_global;
    int32_t h_flags[4] = {0, 0, 0, 0};
    CK(cudaMemsetAsync(c->d_flags, 0, 256, s));
    // ids are validated before any list is indexed with them
    k_check_ids<<<grid_for(NL), 256, 0, s>>>(intma_cg, NL, NG, c->d_flags);
    CK(cudaGetLastError());
    c->launches++;
    CK(cudaMemcpyAsync(h_flags, c->d_flags, 16, cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    if (h_flags[1]) {
        errstr = "numa_init_geometry: intma_cg entry outside [0, n_global)";
        result = NUMA_ERR_ARG;
        return false;
    }
    // block-shell tables (host-built once per (N, epb), tiny)
    {
        const ShellTables &T = shell_tables(p->N, c->shell.epb, c->shell.BS);
        std::vector<int32_t> inv((size_t)c->shell.BS, -1);
        for (size_t t = 0; t < T.pos.size(); ++t) inv[(size_t)T.pos[t]] = (int32_t)t;
        for (int le = 0; le < c->shell.epb && le < 16; ++le) c->shell.first_pos[le] = T.pos[(size_t)le * c->Mn];
        CK(cudaMemcpyAsync(c->shell.pos, T.pos.data(), T.pos.size() * 4, cudaMemcpyHostToDevice, s));
        CK(cudaMemcpyAsync(c->shell.tab, T.tab.data(), T.tab.size() * 4, cudaMemcpyHostToDevice, s));
        CK(cudaMemcpyAsync(ws + L.shell_inv, inv.data(), inv.size() * 4, cudaMemcpyHostToDevice, s));
        CK(cudaStreamSynchronize(s));
    }
    // DSS lists of both index spaces; scratch = the `met` region (written afterwards)
    char *scr = ws + L.met, *scr_end = ws + L.omega;
    if (!build_dss_lists(c, c->dss_nat, intma_cg, NL, nullptr, scr, scr_end, ws + L.small_tmp, s, errstr))
        return false;
    if (!build_dss_lists(c, c->dss_int, intma_cg, c->shell.FS, (const int32_t *)(ws + L.shell_inv), scr,
                         scr_end, ws + L.small_tmp, s, errstr))
        return false;
    // the holes of the block-shell tables (pad positions, elements past Ne) are never used, but
    // keep them finite; then metrics and wJ (wJ parked in `omega`), omega = wJ / M via the lists
    CK(cudaMemsetAsync(ws + L.met, 0, L.nat.start - L.met, s));
    CK(launch_metrics(c, xyz, c->omega, s));
    CK(launch_mass(c, s));
    k_ref3<<<grid_for(NL), 256, 0, s>>>(ref, c->ref3, NL, p->p_a, p->R_gas, c->gamma, c->shell.pos,
                                        c->shell.epb * (int)c->Mn, (int)c->shell.BS, c->shell.FS);
    CK(cudaGetLastError());
    if (sponge) CK(launch_to_shell(c, sponge, c->sponge, 1, s));
    k_face_bc<<<(unsigned)((p->n_elem + 255) / 256), 256, 0, s>>>(face_bc, c->face_bc, p->n_elem,
                                                                  c->d_flags);
    CK(cudaGetLastError());
    c->launches += 4;
    CK(cudaMemcpyAsync(h_flags, c->d_flags, 16, cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    c->has_walls = h_flags[2];
    c->fused_ok = true;
    if (c->has_walls) {
        k_check_walls<<<grid_for(NG), 256, 0, s>>>(c->dss_nat.start, c->dss_nat.copies, c->met, c->face_bc,
                                                   c->shell.pos, c->shell.epb * (int)c->Mn, (int)c->shell.BS,
                                                   c->shell.FS, c->Nq, NG, c->d_flags);
        CK(cudaGetLastError());
        c->launches++;
        CK(cudaMemcpyAsync(h_flags, c->d_flags, 16, cudaMemcpyDeviceToHost, s));
        CK(cudaStreamSynchronize(s));
        c->fused_ok = (h_flags[3] == 0);
    }
    if (h_flags[0]) {
        errstr = "numa_init_geometry: non-positive Jacobian determinant";
        result = NUMA_ERR_NEG_JACOBIAN;
        return false;
    }
    return true;
}

extern "C" numa_status numa_init_geometry(const numa_params *p, const double *xyz,
                                          const int32_t *intma_cg, const uint8_t *face_bc,
                                          const double *ref, const double *sponge, void *workspace,
                                          size_t workspace_bytes, void *stream, numa_ctx **out)
{
    g_err.clear();
    if (out) *out = nullptr;
    if (!p || !xyz || !intma_cg || !face_bc || !ref || !workspace || !out) {
        g_err = "numa_init_geometry: NULL argument";
        return NUMA_ERR_ARG;
    }
    if (p->method != 0 || p->eqn_set != 0) {
        g_err = "numa_init_geometry: only method=0 (CG/DSS) and eqn_set=0 (Eq. 1) are built";
        return NUMA_ERR_UNSUPPORTED;
    }
    if (!params_ok(p)) {
        g_err = "numa_init_geometry: parameters out of range (N in 2..8, sizes > 0, NL < 2^31)";
        return NUMA_ERR_ARG;
    }
    const WsLayout L = ws_layout(p);
    if (workspace_bytes < L.total || ((uintptr_t)workspace & 255)) {
        g_err = "numa_init_geometry: workspace too small or not 256-byte aligned";
        return NUMA_ERR_WORKSPACE;
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        g_err = "numa_init_geometry: no CUDA device (there is no CPU fallback)";
        cudaGetLastError();
        return NUMA_ERR_CUDA;
    }
    numa_ctx *c = new (std::nothrow) numa_ctx();
    if (!c) { g_err = "out of host memory"; return NUMA_ERR_ARG; }
    cudaStream_t s = (cudaStream_t)stream;
    char *ws = (char *)workspace;
    c->par = *p;
    cudaGetDevice(&c->device);
    if (cudaDeviceGetAttribute(&c->n_sm, cudaDevAttrMultiProcessorCount, c->device) != cudaSuccess || c->n_sm < 1) c->n_sm = 148;
    c->Nq = p->N + 1;
    c->Mn = (int64_t)c->Nq * c->Nq * c->Nq;
    c->NL = p->n_elem * c->Mn;
    c->gamma = p->c_p / p->c_v;
    c->launches = 0;
    numa_build_lgl(p->N, &c->lgl);
    c->met = (double *)(ws + L.met);
    c->omega = (double *)(ws + L.omega);
    c->ref3 = (double *)(ws + L.ref3);
    c->sponge = sponge ? (double *)(ws + L.sponge) : nullptr;
    bind_lists(c->dss_nat, ws, L.nat);
    bind_lists(c->dss_int, ws, L.shl);
    c->shell = L.shell;
    c->shell.pos = (int32_t *)(ws + L.shell_pos);
    c->shell.tab = (uint32_t *)(ws + L.shell_tab);
    c->face_bc = (uint8_t *)(ws + L.face_bc);
    c->d_flags = (int32_t *)(ws + L.flags);
    numa_status result = NUMA_ERR_CUDA;
    std::string errstr;
    if (!init_device_tables(c, L, ws, xyz, intma_cg, face_bc, ref, sponge, s, result, errstr)) {
        g_err = errstr;
        cudaGetLastError();
        delete c;
        return result;
    }
    *out = c;
    return NUMA_OK;
}

#undef CK
#define CKC(call)                                                                       \
    do {                                                                                \
        cudaError_t e_ = (call);                                                        \
        if (e_ != cudaSuccess) {                                                        \
            char buf[512];                                                              \
            snprintf(buf, sizeof buf, "%s: %s", #call, cudaGetErrorString(e_));         \
            ctx->err = buf;                                                             \
            cudaGetLastError();                                                         \
            return NUMA_ERR_CUDA;                                                       \
        }                                                                               \
    } while (0)

static numa_status arg_fail(numa_ctx *ctx, const char *msg)
{
    if (ctx) ctx->err = msg; else g_err = msg;
    return NUMA_ERR_ARG;
}

// a context is bound to the device that was current at numa_init_geometry
static bool wrong_device(numa_ctx *ctx)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != ctx->device) {
        ctx->err = "the current CUDA device is not the one this context was created on";
        cudaGetLastError();
        return true;
    }
    return false;
}

extern "C" numa_status numa_rhs(numa_ctx *ctx, const double *q, double *rhs, void *stream)
{
    if (!ctx || !q || !rhs) return arg_fail(ctx, "numa_rhs: NULL argument");
    if (q == rhs) return arg_fail(ctx, "numa_rhs: rhs must not alias q");
    if (wrong_device(ctx)) return NUMA_ERR_ARG;
    CKC(launch_rhs(ctx, q, rhs, (cudaStream_t)stream));
    return NUMA_OK;
}

extern "C" numa_status numa_dss_or_flux(numa_ctx *ctx, double *rhs, void *stream)
{
    if (!ctx || !rhs) return arg_fail(ctx, "numa_dss_or_flux: NULL argument");
    if (ctx->par.method != 0) { ctx->err = "DG face flux is not built"; return NUMA_ERR_UNSUPPORTED; }
    if (wrong_device(ctx)) return NUMA_ERR_ARG;
    CKC(launch_dss_classes(ctx, ctx->dss_nat, rhs, ctx->NL, K_DSS, (cudaStream_t)stream));
    return NUMA_OK;
}

extern "C" numa_status numa_apply_sources(numa_ctx *ctx, const double *q, const double *heating,
                                          double *rhs, void *stream)
{
    if (!ctx || !q || !rhs) return arg_fail(ctx, "numa_apply_sources: NULL argument");
    if (wrong_device(ctx)) return NUMA_ERR_ARG;
    CKC(launch_sources(ctx, q, heating, rhs, (cudaStream_t)stream));
    return NUMA_OK;
}

extern "C" numa_status numa_rk_stage(numa_ctx *ctx, double a0, double a1, double b_dt,
                                     const double *q0, const double *qs, const double *rhs,
                                     double *q_out, void *stream)
{
    if (!ctx || !q0 || !qs || !rhs || !q_out) return arg_fail(ctx, "numa_rk_stage: NULL argument");
    if (wrong_device(ctx)) return NUMA_ERR_ARG;
    CKC(launch_rk(ctx, a0, a1, b_dt, q0, qs, rhs, q_out, (cudaStream_t)stream));
    return NUMA_OK;
}

// SSP-RK3 (Shu-Osher; Q11): (a0, a1, b)
static const double kRK3[3][3] = {{1.0, 0.0, 1.0}, {0.75, 0.25, 0.25}, {1.0 / 3.0, 2.0 / 3.0, 2.0 / 3.0}};

// One SSP-RK3 step on the block-shell buffers A (state of the step, in/out) and B (stage state):
//   stage 1: B = A + dt L(A);  stage 2: B = 3/4 A + 1/4 B + 1/4 dt L(B);
//   stage 3: A = 1/3 A + 2/3 B + 2/3 dt L(B).
// Each stage: the volume kernel writes the update as DSS partial sums (a block reads its own
// records before it writes them, so q_out may alias qs or q0), then the DSS completes the
// shared nodes in place.
static cudaError_t enqueue_step(numa_ctx *ctx, double *A, double *B, const double *heating, double dt,
                                cudaStream_t s)
{
    for (int st = 0; st < 3; ++st) {
        const double *qs = (st == 0) ? A : B;
        double *qo = (st == 2) ? A : B;
        cudaError_t e = cudaSuccess;
        // hyper-diffusion (Eq. 14, alpha = 2): first application from qs before qo (which may alias
        // qs) is written; second application added to the partial sums before the stage's DSS
        if (ctx->hd_on) e = hd_stage_first(ctx, qs, s);
        if (e != cudaSuccess) return e;
        e = launch_stage_volume(ctx, kRK3[st][0], kRK3[st][1], kRK3[st][2] * dt, A, qs, heating, qo, s);
        if (e != cudaSuccess) return e;
        if (ctx->hd_on) e = hd_stage_second(ctx, kRK3[st][2] * dt, qo, s);
        if (e != cudaSuccess) return e;
        e = launch_dss_classes(ctx, ctx->dss_int, qo, ctx->shell.FS, K_FUSED_DSS, s);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

static numa_status step_rk3_impl(numa_ctx *ctx, double *q, void *scratch, const double *heating,
                                 double dt, int32_t n_steps, void *stream, bool use_graph)
{
    if (!ctx || !q || !scratch) return arg_fail(ctx, "numa_step_rk3: NULL argument");
    if (n_steps < 0 || ((uintptr_t)scratch & 255)) return arg_fail(ctx, "numa_step_rk3: bad n_steps or scratch alignment");
    if (wrong_device(ctx)) return NUMA_ERR_ARG;
    if (!ctx->fused_ok) {
        ctx->err = "numa_step_rk3: the wall projector differs between the copies of a wall node (curved walls, or an "
                   "element touching a wall node without a wall face): use the four-call route on this mesh";
        return NUMA_ERR_UNSUPPORTED;
    }
    if (n_steps == 0) return NUMA_OK;
    cudaStream_t s = (cudaStream_t)stream;
    double *A = (double *)scratch;
    double *B = (double *)((char *)scratch + shell_state_bytes(ctx->shell));
    double *H = nullptr;
    CKC(launch_to_shell(ctx, q, A, 5, s));
    if (heating) {
        H = (double *)((char *)scratch + 2 * shell_state_bytes(ctx->shell));
        CKC(launch_to_shell(ctx, heating, H, 1, s));
    }
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (use_graph) CKC(cudaStreamIsCapturing(s, &cap));
    if (use_graph && !ctx->prof && cap == cudaStreamCaptureStatusNone) {
        // the legacy default stream cannot be captured: the graph then runs on a stream of the
        // context, ordered after / before the caller's stream with events
        cudaStream_t cs = s;
        if (s == nullptr || s == cudaStreamLegacy) {
            if (!ctx->gstream) {
                CKC(cudaStreamCreateWithFlags(&ctx->gstream, cudaStreamNonBlocking));
                CKC(cudaEventCreateWithFlags(&ctx->gev0, cudaEventDisableTiming));
                CKC(cudaEventCreateWithFlags(&ctx->gev1, cudaEventDisableTiming));
            }
            cs = ctx->gstream;
            CKC(cudaEventRecord(ctx->gev0, s));
            CKC(cudaStreamWaitEvent(cs, ctx->gev0, 0));
        }
        GraphKey &k = ctx->graph_key;
        if (!ctx->graph || k.q != q || k.heat != heating || k.scratch != scratch || k.dt != dt || k.s != cs) {
            if (ctx->graph) { cudaGraphExecDestroy(ctx->graph); ctx->graph = nullptr; }
            cudaGraph_t g = nullptr;
            CKC(cudaStreamBeginCapture(cs, cudaStreamCaptureModeThreadLocal));
            const int64_t l0 = ctx->launches;
            cudaError_t e = enqueue_step(ctx, A, B, H, dt, cs);
            ctx->graph_launches = ctx->launches - l0;   // what one replay runs (same count as the plain route)
            ctx->launches = l0;  // capture enqueues nothing
            cudaError_t e2 = cudaStreamEndCapture(cs, &g);
            if (e != cudaSuccess || e2 != cudaSuccess) {
                if (g) cudaGraphDestroy(g);
                CKC(e != cudaSuccess ? e : e2);
            }
            e = cudaGraphInstantiate(&ctx->graph, g, 0);
            cudaGraphDestroy(g);
            CKC(e);
            k.q = q; k.heat = heating; k.scratch = scratch; k.dt = dt; k.s = cs;
        }
        for (int step = 0; step < n_steps; ++step) {
            CKC(cudaGraphLaunch(ctx->graph, cs));
            ctx->launches += ctx->graph_launches;  // kernels replayed per step
        }
        if (cs != s) {
            CKC(cudaEventRecord(ctx->gev1, cs));
            CKC(cudaStreamWaitEvent(s, ctx->gev1, 0));
        }
    } else {
        for (int step = 0; step < n_steps; ++step) CKC(enqueue_step(ctx, A, B, H, dt, s));
    }
    CKC(launch_from_shell(ctx, A, q, 5, s));
    return NUMA_OK;
}

extern "C" numa_status numa_step_rk3(numa_ctx *ctx, double *q, void *scratch, const double *heating,
                                     double dt, int32_t n_steps, void *stream)
{
    return step_rk3_impl(ctx, q, scratch, heating, dt, n_steps, stream, false);
}

extern "C" numa_status numa_step_rk3_graph(numa_ctx *ctx, double *q, void *scratch,
                                           const double *heating, double dt, int32_t n_steps,
                                           void *stream)
{
    return step_rk3_impl(ctx, q, scratch, heating, dt, n_steps, stream, true);
}

extern "C" numa_status numa_step_rk3_host(numa_ctx *ctx, double *q_host, const double *heating_host,
                                          double *d_q, double *d_heating, void *scratch, double dt,
                                          int32_t n_steps, void *stream)
{
    if (!ctx || !q_host || !d_q || !scratch) return arg_fail(ctx, "numa_step_rk3_host: NULL argument");
    if (heating_host != nullptr && d_heating == nullptr)
        return arg_fail(ctx, "numa_step_rk3_host: heating_host needs the device staging buffer d_heating");
    if (wrong_device(ctx)) return NUMA_ERR_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    const size_t nb = (size_t)ctx->NL * 8;
    CKC(cudaMemcpyAsync(d_q, q_host, 5 * nb, cudaMemcpyHostToDevice, s));
    if (heating_host) CKC(cudaMemcpyAsync(d_heating, heating_host, nb, cudaMemcpyHostToDevice, s));
    numa_status st = numa_step_rk3(ctx, d_q, scratch, d_heating, dt, n_steps, stream);
    if (st != NUMA_OK) return st;
    CKC(cudaMemcpyAsync(q_host, d_q, 5 * nb, cudaMemcpyDeviceToHost, s));
    CKC(cudaStreamSynchronize(s));
    return NUMA_OK;
}

extern "C" numa_status numa_copy_table(const numa_ctx *ctx, int32_t which, double *out, void *stream)
{
    if (!ctx || !out) return NUMA_ERR_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    cudaError_t e;
    numa_ctx *c = const_cast<numa_ctx *>(ctx);   // (launch counters only)
    switch (which) {   // the tables are kept block-shell; handed out in natural order
        case 0: e = launch_from_shell(c, ctx->met, out, 9, s); break;
        case 1: e = launch_from_shell(c, ctx->omega, out, 1, s); break;
        case 2: e = launch_from_shell(c, ctx->ref3 + 2 * ctx->shell.FS, out, 1, s); break;
        case 3: e = cudaMemcpyAsync(out, ctx->lgl.D, (size_t)ctx->Nq * ctx->Nq * 8, cudaMemcpyHostToDevice, s); break;
        case 4: e = cudaMemcpyAsync(out, ctx->lgl.w, (size_t)ctx->Nq * 8, cudaMemcpyHostToDevice, s); break;
        default: return NUMA_ERR_ARG;
    }
    if (e != cudaSuccess) { cudaGetLastError(); return NUMA_ERR_CUDA; }
    if (which >= 3) cudaStreamSynchronize(s);  // source is host memory of the context
    return NUMA_OK;
}

extern "C" numa_status numa_profile_enable(numa_ctx *ctx, int32_t enable)
{
    if (!ctx) return NUMA_ERR_ARG;
    for (auto &r : ctx->recs) { ctx->pool.push_back(r.a); ctx->pool.push_back(r.b); }
    ctx->recs.clear();
    for (int i = 0; i < K_COUNT; ++i) { ctx->prof_ms[i] = 0.0; ctx->prof_n[i] = 0; }
    ctx->prof = enable != 0;
    return NUMA_OK;
}

extern "C" numa_status numa_profile_read(numa_ctx *ctx, int32_t kernel_id, double *total_ms,
                                         int64_t *launches)
{
    if (!ctx || kernel_id < 0 || kernel_id >= K_COUNT || !total_ms || !launches) return NUMA_ERR_ARG;
    for (auto &r : ctx->recs) {
        float ms = 0.f;
        if (cudaEventSynchronize(r.b) != cudaSuccess || cudaEventElapsedTime(&ms, r.a, r.b) != cudaSuccess) {
            ctx->err = "numa_profile_read: event error";
            cudaGetLastError();
            return NUMA_ERR_CUDA;
        }
        ctx->prof_ms[r.id] += ms;
        ctx->prof_n[r.id] += 1;
        ctx->pool.push_back(r.a); ctx->pool.push_back(r.b);
    }
    ctx->recs.clear();
    *total_ms = ctx->prof_ms[kernel_id];
    *launches = ctx->prof_n[kernel_id];
    return NUMA_OK;
}

extern "C" const char *numa_kernel_name(int32_t kernel_id)
{
    static const char *names[K_COUNT] = {"k_rhs (volume)", "k_dss", "k_sources", "k_rk",
                                         "k_stage_volume (fused)", "k_stage_dss (fused)",
                                         "k_shell_layout (natural <-> block-shell)",
                                         "k_hd_lap (hyper-diffusion)", "k_hd_dss (hyper-diffusion)",
                                         "k_linop + k_imex_walls (IMEX linear operator)",
                                         "k_lincomb / k_dot (IMEX vector work)"};
    return (kernel_id >= 0 && kernel_id < K_COUNT) ? names[kernel_id] : "";
}

extern "C" int32_t numa_kernel_count(void) { return K_COUNT; }

extern "C" int64_t numa_launch_count(const numa_ctx *ctx) { return ctx ? ctx->launches : 0; }

extern "C" numa_status numa_destroy(numa_ctx *ctx)
{
    if (ctx) {
        if (ctx->graph) cudaGraphExecDestroy(ctx->graph);
        if (ctx->gstream) { cudaStreamDestroy(ctx->gstream); cudaEventDestroy(ctx->gev0); cudaEventDestroy(ctx->gev1); }
        for (auto &r : ctx->recs) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
        for (auto &e : ctx->pool) cudaEventDestroy(e);
    }
    delete ctx;
    return NUMA_OK;
}

extern "C" const char *numa_last_error(const numa_ctx *ctx)
{
    return ctx ? ctx->err.c_str() : g_err.c_str();
}
