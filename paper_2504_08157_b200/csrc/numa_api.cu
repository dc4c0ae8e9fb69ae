// C-ABI entry points of libnuma_b200.so (include/numa_b200.h) and the A0 setup.
#include <cub/cub.cuh>
#include <thrust/iterator/counting_iterator.h>

#include <cmath>
#include <cstdio>
#include <cstring>
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

struct WsLayout {
    size_t met, omega, ref3, sponge, start, copies, sh_nodes, dss_idx, dss_seg, dss_blkmap, face_bc, flags, small_tmp, total;
    size_t scratch_bytes;  // init-time scratch, aliased onto the (not yet written) met region
};

static inline size_t WsMaxSeg(size_t NL) { return 4 * (NL / NUMA_DSS_CHUNK + 2); }

static bool params_ok(const numa_params *p)
{
    return p && p->N >= 2 && p->N <= 8 && p->n_elem > 0 && p->n_global > 0 &&
           p->n_elem * (int64_t)((p->N + 1) * (p->N + 1) * (p->N + 1)) < (int64_t)2147483647 &&
           p->n_global < (int64_t)2147483647 && p->c_v > 0 && p->c_p > 0 && p->p_a > 0 && p->R_gas > 0;
}

static WsLayout ws_layout(const numa_params *p)
{
    WsLayout L;
    const size_t Nq = p->N + 1, Mn = Nq * Nq * Nq, NL = (size_t)p->n_elem * Mn;
    size_t off = 0;
    L.met = off; off = align_up(off + 9 * NL * 8);
    L.omega = off; off = align_up(off + NL * 8);
    L.ref3 = off; off = align_up(off + 3 * NL * 8);
    L.sponge = off; off = align_up(off + NL * 8);
    L.start = off; off = align_up(off + ((size_t)p->n_global + 1) * 4);
    L.copies = off; off = align_up(off + NL * 4);
    L.sh_nodes = off; off = align_up(off + ((size_t)p->n_global + 1) * 4);
    L.dss_idx = off; off = align_up(off + NL * 4);
    const size_t max_seg = WsMaxSeg(NL);
    L.dss_seg = off; off = align_up(off + max_seg * sizeof(DssSeg));
    L.dss_blkmap = off; off = align_up(off + ((size_t)p->n_global / NUMA_DSS_THREADS + max_seg + 1) * 4);
    L.face_bc = off; off = align_up(off + (size_t)p->n_elem * 8);
    L.flags = off; off = align_up(off + 256);
    L.small_tmp = off; off = align_up(off + kSmallTmp);
    L.total = off;
    return L;
}

extern "C" size_t numa_workspace_bytes(const numa_params *p)
{
    if (!params_ok(p)) return 0;
    return ws_layout(p).total;
}

extern "C" size_t numa_step_scratch_bytes(const numa_params *p)
{
    if (!params_ok(p)) return 0;
    const size_t Nq = p->N + 1, NL = (size_t)p->n_elem * Nq * Nq * Nq;
    return align_up(5 * NL * 8);
}

// ---------------------------------------------------------------------------------------
// setup kernels
// ---------------------------------------------------------------------------------------
__global__ void k_iota_check(int32_t *vals, const int32_t *keys_in, int32_t *keys, int64_t n,
                             int64_t NG, int32_t *flags)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const int32_t g = keys_in[i];
        if (g < 0 || g >= NG) atomicOr(flags + 1, 1);
        keys[i] = g;
        vals[i] = (int32_t)i;
    }
}

// start[g] = first position in the sorted key array whose key is >= g
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
                             int64_t n)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += stride) {
        const int32_t g = nodes[t];
        const int32_t s = start[g], c = start[g + 1] - s;
#ifdef NUMA_DSS_NOCLASS
        const uint64_t cls = 3;
#else
        const uint64_t cls = (c == 2) ? 0 : (c == 4) ? 1 : (c == 8) ? 2 : 3;
#endif
        const uint32_t first = (uint32_t)copies[s];
        keys[t] = ((uint64_t)(first / NUMA_DSS_CHUNK) << 34) | (cls << 32) | first;
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

__global__ void k_ref3(const double *__restrict__ ref, double *__restrict__ ref3, int64_t NL,
                       double p_a, double R, double gamma)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < NL; p += stride) {
        const double rho0 = ref[p], th0 = ref[NL + p];
        ref3[p] = rho0;
        ref3[NL + p] = th0;
        ref3[2 * NL + p] = p_a * pow(rho0 * R * th0 / p_a, gamma);  // Eq. 3 at the background
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

#define CK(call)                                                                        \
    do {                                                                                \
        cudaError_t e_ = (call);                                                        \
        if (e_ != cudaSuccess) {                                                        \
            char buf[512];                                                              \
            snprintf(buf, sizeof buf, "%s:%d: %s: %s", __FILE__, __LINE__, #call,       \
                     cudaGetErrorString(e_));                                           \
            errstr = buf;                                                               \
            goto cuda_fail;                                                             \
        }                                                                               \
    } while (0)

static inline unsigned grid_for(int64_t n, int threads = 256, int64_t cap = 148 * 32)
{
    int64_t b = (n + threads - 1) / threads;
    if (b > cap) b = cap;
    if (b < 1) b = 1;
    return (unsigned)b;
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
    std::string errstr;
    numa_status result = NUMA_OK;
    char *ws = (char *)workspace;
    c->par = *p;
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
    c->dss_start = (int32_t *)(ws + L.start);
    c->dss_copies = (int32_t *)(ws + L.copies);
    c->sh_nodes = (int32_t *)(ws + L.sh_nodes);
    c->dss_idx = (int32_t *)(ws + L.dss_idx);
    c->dss_seg = (DssSeg *)(ws + L.dss_seg);
    c->dss_blkmap = (int32_t *)(ws + L.dss_blkmap);
    c->face_bc = (uint8_t *)(ws + L.face_bc);
    c->d_flags = (int32_t *)(ws + L.flags);
    {
        const int64_t NL = c->NL, NG = p->n_global;
        int32_t h_flags[4] = {0, 0, 0, 0};
        // --- DSS lists: stable radix sort of (global id, local index); scratch aliases `met`
        char *scr = ws + L.met;
        int32_t *keysA = (int32_t *)scr;
        int32_t *keysB = keysA + NL;
        int32_t *valsA = keysB + NL;
        int32_t *valsB = valsA + NL;
        void *cub_tmp = (void *)align_up((size_t)(valsB + NL));
        size_t cub_avail = (char *)cub_tmp < ws + L.omega ? (size_t)((ws + L.omega) - (char *)cub_tmp) : 0;
        if (cub_avail < kSmallTmp) { cub_tmp = ws + L.small_tmp; cub_avail = kSmallTmp; }
        CK(cudaMemsetAsync(c->d_flags, 0, 256, s));
        k_iota_check<<<grid_for(NL), 256, 0, s>>>(valsA, intma_cg, keysA, NL, NG, c->d_flags);
        CK(cudaGetLastError());
        c->launches++;
        int end_bit = 1;
        while (((int64_t)1 << end_bit) < NG) ++end_bit;
        cub::DoubleBuffer<int32_t> dk(keysA, keysB), dv(valsA, valsB);
        size_t need = 0;
        CK(cub::DeviceRadixSort::SortPairs(nullptr, need, dk, dv, (int)NL, 0, end_bit, s));
        if (need > cub_avail) { errstr = "internal: CUB scratch does not fit"; goto cuda_fail; }
        CK(cub::DeviceRadixSort::SortPairs(cub_tmp, need, dk, dv, (int)NL, 0, end_bit, s));
        k_find_starts<<<grid_for(NL), 256, 0, s>>>(dk.Current(), c->dss_start, NL, NG);
        CK(cudaGetLastError());
        CK(cudaMemcpyAsync(c->dss_copies, dv.Current(), NL * 4, cudaMemcpyDeviceToDevice, s));
        // --- SHARED global nodes (multiplicity >= 2), sorted by (multiplicity class, first
        // copy), and the transposed per-class copy lists of the DSS kernel.  Scratch: the part
        // of the `met` region behind the first sort's buffers.
        {
            SharedPred pred{c->dss_start};
            thrust::counting_iterator<int32_t> ids(0);
            int32_t *d_num = c->d_flags + 8;
            char *scr2 = (char *)align_up((size_t)(valsB + NL));
            char *scr_end = ws + L.omega;
            int32_t *nodesA = (int32_t *)scr2;                         // [NG]
            int32_t *nodesB = nodesA + NG;                             // [NG]
            uint64_t *kA = (uint64_t *)align_up((size_t)(nodesB + NG));  // [NG]
            uint64_t *kB = kA + NG;
            void *tmp2 = (void *)align_up((size_t)(kB + NG));
            size_t avail2 = (char *)tmp2 < scr_end ? (size_t)(scr_end - (char *)tmp2) : 0, need2 = 0;
            if ((char *)tmp2 > scr_end) { errstr = "internal: setup scratch does not fit"; goto cuda_fail; }
            if (avail2 < kSmallTmp) { tmp2 = ws + L.small_tmp; avail2 = kSmallTmp; }
            CK(cub::DeviceSelect::If(nullptr, need2, ids, nodesA, d_num, (int)NG, pred, s));
            if (need2 > avail2) { errstr = "internal: CUB scratch does not fit"; goto cuda_fail; }
            CK(cub::DeviceSelect::If(tmp2, need2, ids, nodesA, d_num, (int)NG, pred, s));
            int32_t h_num = 0;
            CK(cudaMemcpyAsync(&h_num, d_num, 4, cudaMemcpyDeviceToHost, s));
            CK(cudaStreamSynchronize(s));
            c->n_shared = h_num;
            c->n_seg = 0;
            c->dss_blocks = 0;
            if (h_num > 0) {
                k_class_keys<<<grid_for(h_num), 256, 0, s>>>(nodesA, c->dss_start, c->dss_copies, kA, h_num);
                CK(cudaGetLastError());
                int end_bit2 = 35;
                while (((int64_t)NUMA_DSS_CHUNK << (end_bit2 - 34)) < NL) ++end_bit2;
                cub::DoubleBuffer<uint64_t> dk2(kA, kB);
                cub::DoubleBuffer<int32_t> dv2(nodesA, nodesB);
                CK(cub::DeviceRadixSort::SortPairs(nullptr, need2, dk2, dv2, h_num, 0, end_bit2, s));
                if (need2 > avail2) { errstr = "internal: CUB scratch does not fit"; goto cuda_fail; }
                CK(cub::DeviceRadixSort::SortPairs(tmp2, need2, dk2, dv2, h_num, 0, end_bit2, s));
                CK(cudaMemcpyAsync(c->sh_nodes, dv2.Current(), (size_t)h_num * 4, cudaMemcpyDeviceToDevice, s));
                // segment heads (positions where (chunk, class) changes), ascending
                int32_t *heads = dv2.Alternate();           // [<= h_num], free after the sort
                int32_t *hi = heads + WsMaxSeg(NL);
                SegHeadPred hp{dk2.Current()};
                CK(cub::DeviceSelect::If(nullptr, need2, ids, heads, d_num, h_num, hp, s));
                if (need2 > avail2) { errstr = "internal: CUB scratch does not fit"; goto cuda_fail; }
                CK(cub::DeviceSelect::If(tmp2, need2, ids, heads, d_num, h_num, hp, s));
                int32_t n_seg = 0;
                CK(cudaMemcpyAsync(&n_seg, d_num, 4, cudaMemcpyDeviceToHost, s));
                CK(cudaStreamSynchronize(s));
                if ((size_t)n_seg > WsMaxSeg(NL)) { errstr = "internal: DSS segment table does not fit"; goto cuda_fail; }
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
                if ((size_t)blk > (size_t)NG / NUMA_DSS_THREADS + WsMaxSeg(NL) + 1 || idx_off > NL) {
                    errstr = "internal: DSS tables do not fit"; goto cuda_fail;
                }
                c->n_seg = n_seg;
                c->dss_blocks = blk;
                CK(cudaMemcpyAsync(c->dss_seg, h_seg.data(), (size_t)n_seg * sizeof(DssSeg), cudaMemcpyHostToDevice, s));
                CK(cudaMemcpyAsync(c->dss_blkmap, h_map.data(), (size_t)blk * 4, cudaMemcpyHostToDevice, s));
                k_class_lists<<<(unsigned)blk, NUMA_DSS_THREADS, 0, s>>>(c->sh_nodes, c->dss_start, c->dss_copies,
                                                                        c->dss_idx, c->dss_seg, c->dss_blkmap);
                CK(cudaGetLastError());
                CK(cudaStreamSynchronize(s));  // h_seg / h_map are read by the copies above
                c->launches += 6;
            }
        }
        // --- metrics and wJ (wJ parked in `omega`), then omega = wJ / M via the CSR lists.
        // (the setup scratch aliased `met`; the stream order makes the reuse safe)
        CK(launch_metrics(c, xyz, c->omega, s));
        CK(launch_mass(c, s));
        k_ref3<<<grid_for(NL), 256, 0, s>>>(ref, c->ref3, NL, p->p_a, p->R_gas, c->gamma);
        CK(cudaGetLastError());
        if (sponge) CK(cudaMemcpyAsync(c->sponge, sponge, NL * 8, cudaMemcpyDeviceToDevice, s));
        k_face_bc<<<(unsigned)((p->n_elem + 255) / 256), 256, 0, s>>>(face_bc, c->face_bc, p->n_elem,
                                                                      c->d_flags);
        CK(cudaGetLastError());
        c->launches += 6;
        CK(cudaMemcpyAsync(h_flags, c->d_flags, 16, cudaMemcpyDeviceToHost, s));
        CK(cudaStreamSynchronize(s));
        c->has_walls = h_flags[2];
        if (h_flags[1]) {
            g_err = "numa_init_geometry: intma_cg entry outside [0, n_global)";
            result = NUMA_ERR_ARG;
        } else if (h_flags[0]) {
            g_err = "numa_init_geometry: non-positive Jacobian determinant";
            result = NUMA_ERR_NEG_JACOBIAN;
        }
    }
    if (result != NUMA_OK) { delete c; return result; }
    *out = c;
    return NUMA_OK;
cuda_fail:
    g_err = errstr;
    cudaGetLastError();
    delete c;
    return NUMA_ERR_CUDA;
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

extern "C" numa_status numa_rhs(numa_ctx *ctx, const double *q, double *rhs, void *stream)
{
    if (!ctx || !q || !rhs) return arg_fail(ctx, "numa_rhs: NULL argument");
    if (q == rhs) return arg_fail(ctx, "numa_rhs: rhs must not alias q");
    CKC(launch_rhs(ctx, q, rhs, (cudaStream_t)stream));
    return NUMA_OK;
}

extern "C" numa_status numa_dss_or_flux(numa_ctx *ctx, double *rhs, void *stream)
{
    if (!ctx || !rhs) return arg_fail(ctx, "numa_dss_or_flux: NULL argument");
    if (ctx->par.method != 0) { ctx->err = "DG face flux is not built"; return NUMA_ERR_UNSUPPORTED; }
    CKC(launch_dss_classes(ctx, rhs, K_DSS, (cudaStream_t)stream));
    return NUMA_OK;
}

extern "C" numa_status numa_apply_sources(numa_ctx *ctx, const double *q, const double *heating,
                                          double *rhs, void *stream)
{
    if (!ctx || !q || !rhs) return arg_fail(ctx, "numa_apply_sources: NULL argument");
    CKC(launch_sources(ctx, q, heating, rhs, (cudaStream_t)stream));
    return NUMA_OK;
}

extern "C" numa_status numa_rk_stage(numa_ctx *ctx, double a0, double a1, double b_dt,
                                     const double *q0, const double *qs, const double *rhs,
                                     double *q_out, void *stream)
{
    if (!ctx || !q0 || !qs || !rhs || !q_out) return arg_fail(ctx, "numa_rk_stage: NULL argument");
    CKC(launch_rk(ctx, a0, a1, b_dt, q0, qs, rhs, q_out, (cudaStream_t)stream));
    return NUMA_OK;
}

// SSP-RK3 (Shu-Osher; Q11): (a0, a1, b)
static const double kRK3[3][3] = {{1.0, 0.0, 1.0}, {0.75, 0.25, 0.25}, {1.0 / 3.0, 2.0 / 3.0, 2.0 / 3.0}};

extern "C" numa_status numa_step_rk3(numa_ctx *ctx, double *q, void *scratch, const double *heating,
                                     double dt, int32_t n_steps, void *stream)
{
    if (!ctx || !q || !scratch) return arg_fail(ctx, "numa_step_rk3: NULL argument");
    if (n_steps < 0 || ((uintptr_t)scratch & 255)) return arg_fail(ctx, "numa_step_rk3: bad n_steps or scratch alignment");
    cudaStream_t s = (cudaStream_t)stream;
    double *q1 = (double *)scratch;
    for (int step = 0; step < n_steps; ++step) {
        // stage 1: q1 = q + dt L(q);  stage 2: q1 = 3/4 q + 1/4 q1 + 1/4 dt L(q1);
        // stage 3: q  = 1/3 q + 2/3 q1 + 2/3 dt L(q1).  Each stage: the volume kernel writes the
        // update as DSS partial sums (element-local, so q_out may alias qs or q0), then the DSS
        // completes the shared nodes in place.
        for (int st = 0; st < 3; ++st) {
            const double *qs = (st == 0) ? q : q1;
            double *qo = (st == 2) ? q : q1;
            CKC(launch_stage_volume(ctx, kRK3[st][0], kRK3[st][1], kRK3[st][2] * dt, q, qs, heating, qo, s));
            CKC(launch_dss_classes(ctx, qo, K_FUSED_DSS, s));
        }
    }
    return NUMA_OK;
}

extern "C" numa_status numa_step_rk3_host(numa_ctx *ctx, double *q_host, const double *heating_host,
                                          double *d_q, double *d_heating, void *scratch, double dt,
                                          int32_t n_steps, void *stream)
{
    if (!ctx || !q_host || !d_q || !scratch) return arg_fail(ctx, "numa_step_rk3_host: NULL argument");
    if ((heating_host == nullptr) != (d_heating == nullptr))
        return arg_fail(ctx, "numa_step_rk3_host: heating_host and d_heating must both be given or both NULL");
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
    const size_t NL = (size_t)ctx->NL;
    cudaError_t e;
    switch (which) {
        case 0: e = cudaMemcpyAsync(out, ctx->met, 9 * NL * 8, cudaMemcpyDeviceToDevice, s); break;
        case 1: e = cudaMemcpyAsync(out, ctx->omega, NL * 8, cudaMemcpyDeviceToDevice, s); break;
        case 2: e = cudaMemcpyAsync(out, ctx->ref3 + 2 * NL, NL * 8, cudaMemcpyDeviceToDevice, s); break;
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
                                         "k_stage_volume (fused)", "k_stage_dss (fused)"};
    return (kernel_id >= 0 && kernel_id < K_COUNT) ? names[kernel_id] : "";
}

extern "C" int64_t numa_launch_count(const numa_ctx *ctx) { return ctx ? ctx->launches : 0; }

extern "C" numa_status numa_destroy(numa_ctx *ctx)
{
    if (ctx) {
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
