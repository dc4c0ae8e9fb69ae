// RI-velocity diagnostic on the device (Eq. 18-22; the paper computes it
// on the CPU after a device -> host copy, L172).  DESIGN.md readings Q25-Q29:
//   centroid x_c(level) = sum a |u| x / sum a |u| over the LOCAL nodes of a level, a = the
//     horizontal LGL quadrature weight w_i w_j |x_xi y_eta - x_eta y_xi|           (Eq. 22)
//   u_theta = |(I - e_r e_r - e_z e_z) u| at every POINT = unique global node      (Eq. 20-21)
//   strip means: arithmetic mean over the points of strip s eps <= r < (s+1) eps   (L360-L364)
//   u_RI = max over (level, strip) with at least one point                         (Eq. 18)
// Everything is bitwise reproducible run to run: the centroid sums are fixed-order chunk
// reductions over level-sorted node lists (built once), the strip sums are accumulated in
// 64-bit fixed point (integer atomics are exact, hence order-independent).
#include <cub/cub.cuh>

#include <new>

#include "numa_internal.cuh"

namespace {

constexpr int RI_CH = 2048;        // list entries per chunk (one thread block)
constexpr int RI_THREADS = 256;
constexpr size_t RI_CUB_TMP = (size_t)32 << 20;

inline size_t al(size_t x) { return (x + 255) & ~(size_t)255; }

struct RiLayout {
    size_t xy, area, lidx, uidx, bins, umax, flag, partial, chunks, sort, total;
    size_t max_chunks;
};

RiLayout ri_layout(int64_t NL, int64_t NG, int n_lev, int n_strip)
{
    RiLayout L;
    size_t o = 0;
    L.max_chunks = (size_t)(NL / RI_CH + n_lev + 2) + (size_t)(NG / RI_CH + n_lev + 2);
    L.xy = o; o = al(o + (size_t)NL * 16);
    L.area = o; o = al(o + (size_t)NL * 8);
    L.lidx = o; o = al(o + (size_t)NL * 4);
    L.uidx = o; o = al(o + (size_t)NG * 4);
    L.bins = o; o = al(o + (size_t)n_lev * n_strip * 16);
    L.umax = o; o = al(o + 8);
    L.flag = o; o = al(o + 16);
    L.partial = o; o = al(o + L.max_chunks * 3 * 8);
    L.chunks = o; o = al(o + L.max_chunks * 3 * 4 + ((size_t)n_lev + 1) * 4 * 2);
    L.sort = o; o = al(o + (size_t)NL * 16 + ((size_t)n_lev + 2) * 4 + RI_CUB_TMP);
    L.total = o;
    return L;
}

}  // namespace

struct numa_ri {
    numa_ctx *ctx = nullptr;
    int n_lev = 0, n_strip = 0;
    double r_max = 0.0;
    int64_t NL = 0, NG = 0;
    double *xy = nullptr, *area = nullptr, *partial = nullptr;
    int32_t *lidx = nullptr, *uidx = nullptr;
    int32_t *lchunk = nullptr, *uchunk = nullptr;   // [n][3]: level, begin, end
    int32_t *lvl_chunk0 = nullptr;                  // [n_lev+1]: first L-chunk of a level
    unsigned long long *bins = nullptr, *umax = nullptr;
    int32_t *flag = nullptr;
    int n_lchunk = 0, n_uchunk = 0;
    std::string err;
};

namespace {

// ---- setup kernels -------------------------------------------------------------------------
// horizontal quadrature weight of every local node (Q26); natural element-local order
template <int Nq>
__global__ void k_ri_area(const double *__restrict__ xyz, double *__restrict__ xy,
                          double *__restrict__ area, const __grid_constant__ LglTables tab,
                          int64_t NL)
{
    constexpr int Mn = Nq * Nq * Nq;
    __shared__ double sx[Mn], sy[Mn];
    const int64_t e = blockIdx.x;
    for (int n = threadIdx.x; n < Mn; n += blockDim.x) {
        sx[n] = xyz[e * Mn + n];
        sy[n] = xyz[NL + e * Mn + n];
    }
    __syncthreads();
    for (int n = threadIdx.x; n < Mn; n += blockDim.x) {
        const int k = n / (Nq * Nq), j = (n - k * Nq * Nq) / Nq, i = n - Nq * (j + Nq * k);
        const double x0 = sx[n], y0 = sy[n];
        double xx = 0.0, xe = 0.0, yx = 0.0, ye = 0.0;   // difference form, as the metric terms (Q4)
        for (int l = 0; l < Nq; ++l) {
            if (l != i) {
                const double d = tab.D[i * Nq + l];
                const int m = l + Nq * (j + Nq * k);
                xx = fma(d, sx[m] - x0, xx); yx = fma(d, sy[m] - y0, yx);
            }
            if (l != j) {
                const double d = tab.D[j * Nq + l];
                const int m = i + Nq * (l + Nq * k);
                xe = fma(d, sx[m] - x0, xe); ye = fma(d, sy[m] - y0, ye);
            }
        }
        const int64_t p = e * Mn + n;
        area[p] = tab.w[i] * tab.w[j] * fabs(xx * ye - xe * yx);
        xy[p] = x0;
        xy[NL + p] = y0;
    }
}

__global__ void k_ri_keys_local(const int32_t *__restrict__ level, int32_t *keys, int32_t *vals,
                                int64_t NL, int n_lev, int32_t *flag)
{
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= NL) return;
    int l = level[p];
    if (l < 0 || l >= n_lev) { atomicOr(flag, 1); l = n_lev; }
    keys[p] = l;
    vals[p] = (int32_t)p;
}

// a POINT = the first local copy of a global node (Q28); unused global ids get the sentinel key
__global__ void k_ri_keys_unique(const int32_t *__restrict__ level, const int32_t *__restrict__ start,
                                 const int32_t *__restrict__ copies, int32_t *keys, int32_t *vals,
                                 int64_t NG, int n_lev)
{
    const int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= NG) return;
    const int s = start[g];
    if (start[g + 1] == s) { keys[g] = n_lev; vals[g] = 0; return; }
    const int p = copies[s];
    const int l = level[p];
    keys[g] = (l < 0 || l >= n_lev) ? n_lev : l;
    vals[g] = p;
}

// start[l] = first position of the sorted key array with key >= l, l = 0..n_lev
__global__ void k_ri_starts(const int32_t *__restrict__ keys, int32_t *start, int64_t n, int n_lev)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i > n) return;
    const int k0 = (i == 0) ? -1 : keys[i - 1];
    const int k1 = (i == n) ? n_lev : min(keys[i], n_lev);
    for (int l = k0 + 1; l <= k1; ++l) start[l] = (int32_t)i;
}

// ---- per-call kernels ----------------------------------------------------------------------
__global__ void k_ri_clear(unsigned long long *bins, int32_t *count, int64_t n, unsigned long long *umax,
                           int32_t *flag)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { bins[2 * i] = 0ull; bins[2 * i + 1] = 0ull; count[i] = 0; }
    if (i == 0) { *umax = 0ull; flag[1] = 0; }
}

// Eq. 22, first pass: fixed-order partial sums of (a|u|x, a|u|y, a|u|) over one chunk of a level
__global__ void __launch_bounds__(RI_THREADS)
k_ri_centroid_partial(const int32_t *__restrict__ chunk, const int32_t *__restrict__ lidx,
                      const double *__restrict__ xy, const double *__restrict__ area,
                      const double *__restrict__ q, int64_t NL, double *__restrict__ partial)
{
    __shared__ double sh[3][RI_THREADS];
    const int b = chunk[3 * blockIdx.x + 1], e = chunk[3 * blockIdx.x + 2];
    double sx = 0.0, sy = 0.0, sm = 0.0;
    for (int t = b + threadIdx.x; t < e; t += RI_THREADS) {
        const int64_t p = lidx[t];
        const double u = q[1 * NL + p], v = q[2 * NL + p], w = q[3 * NL + p];
        const double am = area[p] * sqrt(u * u + v * v + w * w);
        sx += am * xy[p];
        sy += am * xy[NL + p];
        sm += am;
    }
    sh[0][threadIdx.x] = sx; sh[1][threadIdx.x] = sy; sh[2][threadIdx.x] = sm;
    __syncthreads();
    for (int s = RI_THREADS / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s) {
#pragma unroll
            for (int c = 0; c < 3; ++c) sh[c][threadIdx.x] += sh[c][threadIdx.x + s];
        }
        __syncthreads();
    }
    if (threadIdx.x < 3) partial[3 * (int64_t)blockIdx.x + threadIdx.x] = sh[threadIdx.x][0];
}

// Eq. 22, second pass: chunk partials of a level in ascending order; centroid[l] = (x_c, y_c),
// NaN when the level is at rest (no centroid: the level takes no part)
__global__ void k_ri_centroid_final(const int32_t *__restrict__ lvl_chunk0, const double *__restrict__ partial,
                                    double *__restrict__ centroid, int n_lev)
{
    const int l = blockIdx.x * blockDim.x + threadIdx.x;
    if (l >= n_lev) return;
    double sx = 0.0, sy = 0.0, sm = 0.0;
    for (int c = lvl_chunk0[l]; c < lvl_chunk0[l + 1]; ++c) {
        sx += partial[3 * c + 0]; sy += partial[3 * c + 1]; sm += partial[3 * c + 2];
    }
    const bool ok = sm > 0.0;
    centroid[2 * l + 0] = ok ? sx / sm : 0.0;
    centroid[2 * l + 1] = ok ? sy / sm : 0.0;
    centroid[2 * n_lev + l] = ok ? 1.0 : 0.0;   // validity, kept behind the centroids
}

// Eq. 20-21 and the strip sums.  u_theta < 2^12 m/s is split into hi = floor(u_theta 2^24)
// and lo = floor(frac 2^32): integer sums, exact to 2^-56 m/s per point.
__global__ void __launch_bounds__(RI_THREADS)
k_ri_bins(const int32_t *__restrict__ chunk, const int32_t *__restrict__ uidx,
          const double *__restrict__ xy, const double *__restrict__ q, int64_t NL,
          const double *__restrict__ centroid, int n_lev, int n_strip, double r_max,
          unsigned long long *__restrict__ bins, int32_t *__restrict__ count,
          unsigned long long *__restrict__ umax, int32_t *__restrict__ flag)
{
    extern __shared__ unsigned long long sbin[];   // [n_strip][2] then counts
    unsigned int *scnt = reinterpret_cast<unsigned int *>(sbin + 2 * n_strip);
    __shared__ unsigned long long smax;
    const int l = chunk[3 * blockIdx.x + 0], b = chunk[3 * blockIdx.x + 1], e = chunk[3 * blockIdx.x + 2];
    for (int s = threadIdx.x; s < n_strip; s += RI_THREADS) { sbin[2 * s] = 0ull; sbin[2 * s + 1] = 0ull; scnt[s] = 0u; }
    if (threadIdx.x == 0) smax = 0ull;
    __syncthreads();
    const bool valid = centroid[2 * n_lev + l] != 0.0;
    const double xc = centroid[2 * l], yc = centroid[2 * l + 1];
    const double eps = r_max / n_strip;
    unsigned long long mymax = 0ull;
    for (int t = b + threadIdx.x; t < e; t += RI_THREADS) {
        const int64_t p = uidx[t];
        const double u = q[1 * NL + p], v = q[2 * NL + p];
        const double uh = sqrt(u * u + v * v);
        const unsigned long long uhb = (unsigned long long)__double_as_longlong(uh);   // uh >= 0: bit order = value order
        if (uh == uh && uhb > mymax) mymax = uhb;
        if (!valid) continue;
        const double rx = xy[p] - xc, ry = xy[NL + p] - yc;
        const double r = sqrt(rx * rx + ry * ry);
        if (!(r < r_max)) continue;
        const double erx = (r > 0.0) ? rx / r : 0.0, ery = (r > 0.0) ? ry / r : 0.0;   // r = 0: no radial direction (Q29)
        const double ur = u * erx + v * ery;               // u . e_r (e_r has no z-component)
        const double t0 = u - ur * erx, t1 = v - ur * ery;   // w - (u . e_z) = 0: e_z removes the vertical part
        const double ut = sqrt(t0 * t0 + t1 * t1);
        const int s = (int)floor(r / eps);
        if (s >= n_strip) continue;
        if (!(ut < 4096.0)) { atomicOr(flag + 1, 1); continue; }   // NaN or absurd: reported, not binned
        const double sc = ut * 16777216.0;                 // 2^24, exact
        const double hi = floor(sc);
        const unsigned long long lo = (unsigned long long)floor((sc - hi) * 4294967296.0);
        atomicAdd(&sbin[2 * s], (unsigned long long)hi);
        atomicAdd(&sbin[2 * s + 1], lo);
        atomicAdd(&scnt[s], 1u);
    }
    atomicMax(&smax, mymax);
    __syncthreads();
    for (int s = threadIdx.x; s < n_strip; s += RI_THREADS) {
        if (scnt[s]) {
            const int64_t g = (int64_t)l * n_strip + s;
            atomicAdd(&bins[2 * g], sbin[2 * s]);
            atomicAdd(&bins[2 * g + 1], sbin[2 * s + 1]);
            atomicAdd(&count[g], (int)scnt[s]);
        }
    }
    if (threadIdx.x == 0 && smax) atomicMax(umax, smax);
}

// strip means and Eq. 18 (one block): scalars = (u_RI, max horizontal speed, error flag)
__global__ void __launch_bounds__(RI_THREADS)
k_ri_final(const unsigned long long *__restrict__ bins, const int32_t *__restrict__ count, int64_t n,
           const unsigned long long *__restrict__ umax, const int32_t *__restrict__ flag,
           double *__restrict__ ubar, double *__restrict__ scalars)
{
    __shared__ double sh[RI_THREADS];
    double best = 0.0;
    for (int64_t i = threadIdx.x; i < n; i += RI_THREADS) {
        const int c = count[i];
        double m = 0.0;
        if (c > 0) {
            m = ((double)bins[2 * i] + (double)bins[2 * i + 1] * (1.0 / 4294967296.0)) * (1.0 / 16777216.0) / (double)c;
            best = fmax(best, m);
        }
        ubar[i] = m;
    }
    sh[threadIdx.x] = best;
    __syncthreads();
    for (int s = RI_THREADS / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s) sh[threadIdx.x] = fmax(sh[threadIdx.x], sh[threadIdx.x + s]);
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        scalars[0] = sh[0];
        scalars[1] = __longlong_as_double((long long)*umax);
        scalars[2] = (double)flag[1];
    }
}

template <int Nq>
cudaError_t area_launch(numa_ri *r, const double *xyz, cudaStream_t s)
{
    k_ri_area<Nq><<<(unsigned)r->ctx->par.n_elem, 256, 0, s>>>(xyz, r->xy, r->area, r->ctx->lgl, r->NL);
    return cudaGetLastError();
}

}  // namespace

#define RCK(call)                                                                        \
    do {                                                                                \
        cudaError_t e_ = (call);                                                        \
        if (e_ != cudaSuccess) {                                                        \
            char buf[512];                                                              \
            snprintf(buf, sizeof buf, "%s: %s", #call, cudaGetErrorString(e_));         \
            if (ri) ri->err = buf;                                                      \
            ctx->err = buf;                                                             \
            cudaGetLastError();                                                         \
            fail = NUMA_ERR_CUDA;                                                       \
            goto done;                                                                  \
        }                                                                               \
    } while (0)

extern "C" size_t numa_ri_workspace_bytes(const numa_params *p, int32_t n_levels, int32_t n_strips)
{
    if (!p || p->N < 2 || p->N > 8 || p->n_elem <= 0 || p->n_global <= 0 || n_levels < 1 || n_strips < 1 ||
        n_strips > 1024)
        return 0;
    const int64_t Nq = p->N + 1;
    return ri_layout(p->n_elem * Nq * Nq * Nq, p->n_global, n_levels, n_strips).total;
}

extern "C" numa_status numa_ri_init(numa_ctx *ctx, const double *xyz, const int32_t *level,
                                    int32_t n_levels, int32_t n_strips, double r_max,
                                    void *ri_workspace, size_t workspace_bytes, void *stream,
                                    numa_ri **out)
{
    if (out) *out = nullptr;
    if (!ctx) return NUMA_ERR_ARG;
    if (!xyz || !level || !ri_workspace || !out || n_levels < 1 || n_strips < 1 || n_strips > 1024 ||
        !(r_max > 0.0)) {
        ctx->err = "numa_ri_init: NULL argument, n_levels < 1, n_strips outside 1..1024 or r_max <= 0";
        return NUMA_ERR_ARG;
    }
    const RiLayout L = ri_layout(ctx->NL, ctx->par.n_global, n_levels, n_strips);
    if (workspace_bytes < L.total || ((uintptr_t)ri_workspace & 255)) {
        ctx->err = "numa_ri_init: workspace too small or not 256-byte aligned";
        return NUMA_ERR_WORKSPACE;
    }
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != ctx->device) {
        ctx->err = "the current CUDA device is not the one this context was created on";
        cudaGetLastError();
        return NUMA_ERR_ARG;
    }
    numa_ri *ri = new (std::nothrow) numa_ri();
    if (!ri) { ctx->err = "out of host memory"; return NUMA_ERR_ARG; }
    numa_status fail = NUMA_OK;
    cudaStream_t s = (cudaStream_t)stream;
    char *ws = (char *)ri_workspace;
    const int64_t NL = ctx->NL, NG = ctx->par.n_global;
    ri->ctx = ctx; ri->n_lev = n_levels; ri->n_strip = n_strips; ri->r_max = r_max; ri->NL = NL; ri->NG = NG;
    ri->xy = (double *)(ws + L.xy); ri->area = (double *)(ws + L.area);
    ri->lidx = (int32_t *)(ws + L.lidx); ri->uidx = (int32_t *)(ws + L.uidx);
    ri->bins = (unsigned long long *)(ws + L.bins); ri->umax = (unsigned long long *)(ws + L.umax);
    ri->flag = (int32_t *)(ws + L.flag); ri->partial = (double *)(ws + L.partial);
    int32_t *chunks = (int32_t *)(ws + L.chunks);
    char *scr = ws + L.sort;
    int32_t *d_start = (int32_t *)(scr + (size_t)NL * 16);   // [n_lev+1], in front of the CUB scratch
    std::vector<int32_t> hl(n_levels + 1), hu(n_levels + 1), h_chunks, h_c0(n_levels + 1);
    int32_t h_flag[4] = {0, 0, 0, 0};
    {
        RCK(cudaMemsetAsync(ri->flag, 0, 16, s));
        cudaError_t e;
        switch (ctx->par.N) {
            case 2: e = area_launch<3>(ri, xyz, s); break;
            case 3: e = area_launch<4>(ri, xyz, s); break;
            case 4: e = area_launch<5>(ri, xyz, s); break;
            case 5: e = area_launch<6>(ri, xyz, s); break;
            case 6: e = area_launch<7>(ri, xyz, s); break;
            case 7: e = area_launch<8>(ri, xyz, s); break;
            default: e = area_launch<9>(ri, xyz, s); break;
        }
        RCK(e);
        // local nodes by level (ascending local index inside a level: the radix sort is stable)
        int32_t *kA = (int32_t *)scr, *vA = kA + 2 * NL;
        k_ri_keys_local<<<(unsigned)((NL + 255) / 256), 256, 0, s>>>(level, kA, vA, NL, n_levels, ri->flag);
        RCK(cudaGetLastError());
        // (the CUB scratch sits behind the four key/value buffers and the start table)
        {
            cub::DoubleBuffer<int32_t> dk(kA, kA + NL), dv(vA, vA + NL);
            int end_bit = 1;
            while ((1 << end_bit) <= n_levels) ++end_bit;
            size_t need = 0;
            RCK(cub::DeviceRadixSort::SortPairs(nullptr, need, dk, dv, (int)NL, 0, end_bit, s));
            if (need > RI_CUB_TMP) { ri->err = ctx->err = "numa_ri_init: CUB scratch does not fit"; fail = NUMA_ERR_WORKSPACE; goto done; }
            void *tmp = (void *)(scr + al((size_t)NL * 16 + ((size_t)n_levels + 2) * 4));
            RCK(cub::DeviceRadixSort::SortPairs(tmp, need, dk, dv, (int)NL, 0, end_bit, s));
            k_ri_starts<<<(unsigned)((NL + 1 + 255) / 256), 256, 0, s>>>(dk.Current(), d_start, NL, n_levels);
            RCK(cudaGetLastError());
            RCK(cudaMemcpyAsync(ri->lidx, dv.Current(), (size_t)NL * 4, cudaMemcpyDeviceToDevice, s));
            RCK(cudaMemcpyAsync(hl.data(), d_start, ((size_t)n_levels + 1) * 4, cudaMemcpyDeviceToHost, s));
            RCK(cudaMemcpyAsync(h_flag, ri->flag, 16, cudaMemcpyDeviceToHost, s));
            RCK(cudaStreamSynchronize(s));
        }
        if (h_flag[0]) { ri->err = ctx->err = "numa_ri_init: level entry outside [0, n_levels)"; fail = NUMA_ERR_ARG; goto done; }
        // points (unique global nodes) by level
        k_ri_keys_unique<<<(unsigned)((NG + 255) / 256), 256, 0, s>>>(level, ctx->dss_nat.start, ctx->dss_nat.copies,
                                                                     kA, vA, NG, n_levels);
        RCK(cudaGetLastError());
        {
            cub::DoubleBuffer<int32_t> dk(kA, kA + NL), dv(vA, vA + NL);
            int end_bit = 1;
            while ((1 << end_bit) <= n_levels) ++end_bit;
            size_t need = 0;
            RCK(cub::DeviceRadixSort::SortPairs(nullptr, need, dk, dv, (int)NG, 0, end_bit, s));
            if (need > RI_CUB_TMP) { ri->err = ctx->err = "numa_ri_init: CUB scratch does not fit"; fail = NUMA_ERR_WORKSPACE; goto done; }
            void *tmp = (void *)(scr + al((size_t)NL * 16 + ((size_t)n_levels + 2) * 4));
            RCK(cub::DeviceRadixSort::SortPairs(tmp, need, dk, dv, (int)NG, 0, end_bit, s));
            k_ri_starts<<<(unsigned)((NG + 1 + 255) / 256), 256, 0, s>>>(dk.Current(), d_start, NG, n_levels);
            RCK(cudaGetLastError());
            RCK(cudaMemcpyAsync(ri->uidx, dv.Current(), (size_t)NG * 4, cudaMemcpyDeviceToDevice, s));
            RCK(cudaMemcpyAsync(hu.data(), d_start, ((size_t)n_levels + 1) * 4, cudaMemcpyDeviceToHost, s));
            RCK(cudaStreamSynchronize(s));
        }
        // chunk tables: (level, begin, end) per thread block; a chunk never straddles a level
        auto add_chunks = [&](const std::vector<int32_t> &st, std::vector<int32_t> *c0) {
            int n = 0;
            for (int l = 0; l < n_levels; ++l) {
                if (c0) (*c0)[l] = n;
                for (int32_t b = st[l]; b < st[l + 1]; b += RI_CH) {
                    h_chunks.push_back(l); h_chunks.push_back(b);
                    h_chunks.push_back(std::min<int32_t>(b + RI_CH, st[l + 1]));
                    ++n;
                }
            }
            if (c0) (*c0)[n_levels] = n;
            return n;
        };
        ri->n_lchunk = add_chunks(hl, &h_c0);
        ri->n_uchunk = add_chunks(hu, nullptr);
        if ((size_t)(ri->n_lchunk + ri->n_uchunk) > L.max_chunks) { ri->err = ctx->err = "numa_ri_init: chunk table does not fit"; fail = NUMA_ERR_WORKSPACE; goto done; }
        ri->lchunk = chunks;
        ri->uchunk = chunks + 3 * (size_t)ri->n_lchunk;
        ri->lvl_chunk0 = chunks + 3 * L.max_chunks;
        RCK(cudaMemcpyAsync(chunks, h_chunks.data(), h_chunks.size() * 4, cudaMemcpyHostToDevice, s));
        RCK(cudaMemcpyAsync(ri->lvl_chunk0, h_c0.data(), h_c0.size() * 4, cudaMemcpyHostToDevice, s));
        RCK(cudaStreamSynchronize(s));
        ctx->launches += 7;
    }
done:
    if (fail != NUMA_OK) { delete ri; return fail; }
    *out = ri;
    return NUMA_OK;
}
#undef RCK

extern "C" numa_status numa_ri_velocity(numa_ri *ri, const double *q, double *ubar, int32_t *count,
                                        double *centroid, double *scalars, void *stream)
{
    if (!ri) return NUMA_ERR_ARG;
    numa_ctx *ctx = ri->ctx;
    if (!q || !ubar || !count || !centroid || !scalars) { ri->err = ctx->err = "numa_ri_velocity: NULL argument"; return NUMA_ERR_ARG; }
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != ctx->device) {
        ri->err = ctx->err = "the current CUDA device is not the one this context was created on";
        cudaGetLastError();
        return NUMA_ERR_ARG;
    }
    cudaStream_t s = (cudaStream_t)stream;
    const int64_t nb = (int64_t)ri->n_lev * ri->n_strip;
    k_ri_clear<<<(unsigned)((nb + 255) / 256), 256, 0, s>>>(ri->bins, count, nb, ri->umax, ri->flag);
    if (ri->n_lchunk)
        k_ri_centroid_partial<<<ri->n_lchunk, RI_THREADS, 0, s>>>(ri->lchunk, ri->lidx, ri->xy, ri->area, q, ri->NL, ri->partial);
    k_ri_centroid_final<<<(ri->n_lev + 127) / 128, 128, 0, s>>>(ri->lvl_chunk0, ri->partial, centroid, ri->n_lev);
    if (ri->n_uchunk)
        k_ri_bins<<<ri->n_uchunk, RI_THREADS, (size_t)ri->n_strip * 20, s>>>(ri->uchunk, ri->uidx, ri->xy, q, ri->NL, centroid,
                                                                            ri->n_lev, ri->n_strip, ri->r_max, ri->bins, count,
                                                                            ri->umax, ri->flag);
    k_ri_final<<<1, RI_THREADS, 0, s>>>(ri->bins, count, nb, ri->umax, ri->flag, ubar, scalars);
    ctx->launches += 5;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { ri->err = ctx->err = cudaGetErrorString(e); return NUMA_ERR_CUDA; }
    return NUMA_OK;
}

extern "C" numa_status numa_ri_destroy(numa_ri *ri)
{
    delete ri;
    return NUMA_OK;
}
