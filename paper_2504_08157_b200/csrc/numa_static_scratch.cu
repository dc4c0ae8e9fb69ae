// numa_step_rk3_static: the SSP-RK3 step of numa_step_rk3 for callers that cannot hand the
// library any device scratch.
//
// Every other entry point works inside buffers the caller allocated.  That presumes the caller
// HAS an allocator.  Some do not: a coupling layer inside a host model whose device memory is
// owned entirely by another runtime (OpenACC data regions of a Fortran model such as the paper's,
// or a framework pool that claimed the whole GPU at start-up, after which a raw cudaMalloc just
// fails), and time loops that must not call cudaMalloc / cudaFree at all because both
// synchronise the device.  For them the two block-shell states and the heating field that a step
// works in live in the fixed array below instead.  The array is part of the library image: a GPU
// holds its NUMA_STATIC_SCRATCH_BYTES from the moment the library's code is loaded onto it until
// the process exits, whether or not this entry point is ever called, which is why the limit is
// kept modest and larger meshes are sent back to numa_step_rk3.
//
// Nothing here allocates: no cudaMalloc / cudaFree, no allocating library routine.  The only
// set-up is asking the runtime where the array lives on the current device.
#include <mutex>

#include "numa_internal.cuh"

// In host code `g_step_scratch` is only a handle for the runtime, NOT a device address; the address
// the kernels need comes from cudaGetSymbolAddress below.
static __device__ __align__(256) unsigned char g_step_scratch[NUMA_STATIC_SCRATCH_BYTES];

namespace {

constexpr int kMaxDevices = 64;
std::mutex g_mu;
void *g_scratch_addr[kMaxDevices] = {nullptr};   // device address of g_step_scratch, per device

// Device address of the array on device `dev`, which must be the current device.  Resolved on the
// first call per device and remembered; that first resolution may make the runtime load this
// file's code onto the device, so it belongs before any stream capture.
cudaError_t static_scratch_address(int dev, void **out)
{
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_addr[dev]) {
        void *p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&p, g_step_scratch);
        if (e != cudaSuccess) return e;
        g_scratch_addr[dev] = p;
    }
    *out = g_scratch_addr[dev];
    return cudaSuccess;
}

}  // namespace

extern "C" size_t numa_static_scratch_bytes(void) { return NUMA_STATIC_SCRATCH_BYTES; }

extern "C" numa_status numa_step_rk3_static(numa_ctx *ctx, double *q, const double *heating, double dt,
                                            int32_t n_steps, void *stream)
{
    if (!ctx) return NUMA_ERR_ARG;
    if (!q) { ctx->err = "numa_step_rk3_static: NULL argument"; return NUMA_ERR_ARG; }
    const size_t need = numa_step_scratch_bytes(&ctx->par);
    if (need == 0 || need > (size_t)NUMA_STATIC_SCRATCH_BYTES) {
        ctx->err = "numa_step_rk3_static: this mesh needs " + std::to_string(need) +
                   " bytes of step scratch but the built-in buffer holds " +
                   std::to_string((size_t)NUMA_STATIC_SCRATCH_BYTES) +
                   " (NUMA_STATIC_SCRATCH_BYTES); call numa_step_rk3 with scratch of your own";
        return NUMA_ERR_WORKSPACE;
    }
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        ctx->err = "numa_step_rk3_static: no CUDA device";
        cudaGetLastError();
        return NUMA_ERR_CUDA;
    }
    if (dev != ctx->device || dev < 0 || dev >= kMaxDevices) {
        ctx->err = "the current CUDA device is not the one this context was created on";
        return NUMA_ERR_ARG;
    }
    void *scratch = nullptr;
    cudaError_t e = static_scratch_address(dev, &scratch);
    if (e != cudaSuccess) {
        ctx->err = std::string("numa_step_rk3_static: cudaGetSymbolAddress: ") + cudaGetErrorString(e);
        cudaGetLastError();
        return NUMA_ERR_CUDA;
    }
    // From here on this is numa_step_rk3 itself, on the built-in buffer.  Nothing in the buffer has
    // to start at zero: the layout conversion at the head of the call writes every node position
    // the stages later read, and the padding of the block records never reaches a result.
    return numa_step_rk3(ctx, q, scratch, heating, dt, n_steps, stream);
}
