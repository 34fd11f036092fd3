// Internal declarations shared by the CUDA translation units of libppm_b200.so.
// (Nothing here is shared with oracle/.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "ppm.h"

#define PPM_TINY 1e-30f

// Per-launch parameters of one directional sweep (passed by value as a kernel argument).
struct SweepParams {
    const float* __restrict__ in;   // 15 fields, SoA, perturbation form
    float* __restrict__ out;
    long long ncell;                // nx*ny*nz (field stride)
    int n;                          // cells along the sweep axis
    int na, nb;                     // transverse extents: a is mapped to threads, b to blockIdx.y
    long long sd, sa, sb;           // element strides of the sweep / transverse axes
    int bc_lo, bc_hi;
    int chunk;                      // cells marched per thread (pencil split along the sweep axis)
    float dt, dx, dtdx, inv_dx;
    float gamma, rho_floor, p_floor;
    // gravity / base state
    int tab_n;
    float s0, inv_ds;
    float cen_d, cen_a, cen_b;      // RADIAL centre along (sweep, a, b) axes
    const float4* __restrict__ tab; // node k: {g, rho0, p0, 0}
    int* flag;                      // sticky state flag (bit 0: floor hit, bit 1: NaN)
};

struct ppm_ctx {
    ppm_params prm;
    float* buf[2];
    int cur;                        // buf[cur] holds the state
    cudaStream_t stream;
    float4* tab;                    // device gravity table (fp32 nodes)
    double* tab64;                  // device gravity table as doubles {g, rho0, p0} x n (set/get/reductions)
    int* flag;                      // device sticky flag
    unsigned int* cflmax;           // device: ordered-uint encoded max
    double* partial;                // device: conserved partial sums [6][nblocks]
    double* result;                 // device: final 6 sums
    int nblocks_red;
    int chunk;
    long long launches;
    char err[512];
};

// launchers (defined in the .cu files)
cudaError_t ppm_launch_sweep(ppm_ctx* c, int axis, double dt);
cudaError_t ppm_launch_to_perturbation(ppm_ctx* c, float* state, int z0, int nzs);
cudaError_t ppm_launch_to_full(ppm_ctx* c, const float* state, float* dst, int z0, int nzs);
cudaError_t ppm_launch_cfl(ppm_ctx* c);
cudaError_t ppm_launch_conserved(ppm_ctx* c);
