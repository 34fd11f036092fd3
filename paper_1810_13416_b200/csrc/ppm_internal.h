// Internal declarations shared by the CUDA translation units of libppm_b200.so.
// (Nothing here is shared with oracle/.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "ppm.h"

#define PPM_TINY 1e-30f

// Per-launch parameters of one directional sweep (passed by value as a kernel argument).
struct SweepParams {
    const float* inf[PPM_NFIELDS];  // 15 field planes, SoA, perturbation form
    float* outf[PPM_NFIELDS];
    long long ncell;                // nx*ny*nz (field stride)
    int n;                          // cells along the sweep axis
    int na, nb;                     // transverse extents: a is mapped to threads, b to blockIdx.y
    // element offset of cell (j along the sweep axis, a, b) inside a field plane set:
    //   (j>>2)*SBd + (j&3)*SId + (a>>2)*SBa + (a&3)*SIa + (b>>2)*SBb + (b&3)*SIb
    // brick layout: SB = stride between 4x4x4 bricks (256 B each), SI = stride inside a brick;
    // plane layout: SB = 4*stride, SI = stride.
    long long SBd, SBa, SBb;
    int SId, SIa, SIb;
    int brick;                      // 1: threads map to in-brick coordinates (4 a x 4 b per 16 lanes)
    int nbrick_d;                   // bricks along the sweep axis (brick layout)
    int bc_lo, bc_hi;
    int chunk;                      // cells marched per thread (pencil split along the sweep axis)
    float dt, dx, dtdx, inv_dx;
    float gamma, rho_floor, p_floor;
    // gravity / base state
    int tab_n;
    float s0, inv_ds;
    float cen_d, cen_a, cen_b;      // RADIAL centre along (sweep, a, b) axes
    const float4* __restrict__ tab; // node k: {rho0, p0, g, 0}
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
    int layout;                     // 0 = SoA planes [f][z][y][x]; 1 = SoA bricks [f][bz][by][bx][4z][4y][4x]
    int layout_locked;              // set once a state has been loaded
    int tma_ok;                     // tensor maps for the x-sweep TMA path are valid
    int force_direct;               // option: take the direct-global x path even when TMA is available
    long long launches;
    char err[512];
    alignas(64) unsigned char xmap[2][128];   // CUtensorMap of buf[0], buf[1]: 5-D {64, nbx, nby, nbz, 15}, box {64,1,2,1,5}
};

// launchers (defined in the .cu files)
cudaError_t ppm_launch_sweep(ppm_ctx* c, int axis, double dt);
bool ppm_make_xmaps(ppm_ctx* c);
cudaError_t ppm_launch_to_perturbation(ppm_ctx* c, const float* dense_slab, float* state, int z0, int nzs);
cudaError_t ppm_launch_to_full(ppm_ctx* c, const float* state, float* dst, int z0, int nzs);
cudaError_t ppm_launch_cfl(ppm_ctx* c);
cudaError_t ppm_launch_conserved(ppm_ctx* c);
