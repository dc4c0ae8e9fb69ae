// Internal declarations of libnuma_b200.so (not part of the C ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>

#include "../../include/numa_b200.h"

#define NUMA_MAX_NQ 9

// LGL derivative matrix and weights, passed BY VALUE as a kernel parameter so that
// compile-time-indexed reads become constant-bank operands.
struct LglTables {
    double D[NUMA_MAX_NQ * NUMA_MAX_NQ];  // D[i*Nq + l] = h_l'(xi_i)  (Alg. 2)
    double w[NUMA_MAX_NQ];                // quadrature weights (Eq. 8)
};

struct numa_ctx {
    numa_params par;
    int Nq;
    int64_t Mn, NL;
    double gamma;
    LglTables lgl;
    // device tables, all inside the caller's workspace
    double *met;     // [9][NL]   d xi_a / d x_c
    double *omega;   // [NL]      wJ / M
    double *ref3;    // [3][NL]   rho0, theta0, p0
    double *sponge;  // [NL] or nullptr
    int32_t *dss_start;   // [NG+1]  CSR over global nodes
    int32_t *dss_copies;  // [NL]    local indices, ascending within a node
    int32_t *sh_nodes;    // [n_shared] global ids of SHARED nodes (multiplicity >= 2), ascending
    int64_t n_shared;
    uint8_t *face_bc;     // [Ne][8] (padded to 8 bytes per element)
    int32_t *d_flags;     // [4] device error flags
    int has_walls;
    int64_t launches;
    std::string err;
};

// host-side table construction (tables.cpp part of numa_api.cu)
void numa_build_lgl(int N, LglTables *t);

// kernel launchers (numa_kernels.cu); all return cudaError_t of the launch
cudaError_t launch_metrics(numa_ctx *c, const double *xyz, double *wJ_out, cudaStream_t s);
cudaError_t launch_mass(numa_ctx *c, cudaStream_t s);
cudaError_t launch_rhs(numa_ctx *c, const double *q, double *rhs, cudaStream_t s);
cudaError_t launch_dss(numa_ctx *c, double *r, int nfields, cudaStream_t s);
cudaError_t launch_sources(numa_ctx *c, const double *q, const double *heat, double *rhs,
                           cudaStream_t s);
cudaError_t launch_rk(numa_ctx *c, double a0, double a1, double b_dt, const double *q0,
                      const double *qs, const double *rhs, double *qout, cudaStream_t s);
// fused stage: volume + sources + walls + RK written as partial sums, then in-place DSS
cudaError_t launch_stage_fused(numa_ctx *c, double a0, double a1, double b_dt, const double *q0,
                               const double *qs, const double *heat, double *qout,
                               cudaStream_t s);
