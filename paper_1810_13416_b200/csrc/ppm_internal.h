// Internal declarations shared by the CUDA translation units of libppm_b200.so.
// (Nothing here is shared with oracle/.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "ppm.h"

#define PPM_TINY 1e-30f

// State layout inside each borrowed buffer ("brick records"): the grid is cut into bricks of 4x4x4 cells
// (extents rounded up to multiples of 4; pad cells are never read or written by the sweeps) and a brick
// holds all 15 fields of its 64 cells, field-major:   [bz][by][bx][field 15][4z][4y][4x]   (3840 B per brick).
// A cell's 15 values are 256 B apart, so one 64-bit pointer plus compile-time offsets addresses all of them,
// and every sweep direction reads and writes whole 64-byte brick layers.
#define PPM_BRICK_FLOATS (PPM_NFIELDS * 64)

// Per-launch parameters of one directional sweep (passed by value as a kernel argument).
struct SweepParams {
    const float* in;                // state, perturbation form
    float* out;
    int n;                          // cells along the sweep axis
    int na, nb;                     // transverse extents: a and b index the 4x4 pencils of a brick column
    // float offset of cell (j along the sweep axis, a, b), field f:
    //   (j>>2)*SBd + ((j&3) << 2*axis_d) + (a>>2)*SBa + ((a&3) << 2*axis_a) + (b>>2)*SBb + ((b&3) << 2*axis_b) + 64*f
    // SB = stride between bricks along that axis (960, 960*nbx, 960*nbx*nby floats)
    long long SBd, SBa, SBb;
    int nbrick_d;                   // bricks along the sweep axis
    int ntiles;                     // bulk path: CTA tiles (8 x 1 brick columns) in the transverse plane
    int tiles_a, chunk_b;           // bulk path: tiles [0, tiles_a) march segments of `chunk` cells, the rest of `chunk_b` cells
    int bc_lo, bc_hi;
    int chunk;                      // cells marched per thread (pencil split along the sweep axis)
    float dt, dx, dtdx, inv_dx;
    float gamma, rho_floor, p_floor;
    float gp, gmg, g_gm1, hdt;      // (gamma+1)/2, (gamma-1)/(2 gamma), gamma/(gamma-1), dt/2: kernel-argument constants cost no registers
    // gravity / base state
    int tab_n;
    float s0, inv_ds;
    float cen_d, cen_a, cen_b;      // RADIAL centre along (sweep, a, b) axes
    const float4* __restrict__ tab; // node k: {rho0, p0, g, 0}
    // the same table as interval records, so that a lookup is one load per quantity: interval k (nodes k, k+1):
    const float4* __restrict__ tabp; // {rho0_k, p0_k, rho0_k+1 - rho0_k, p0_k+1 - p0_k}
    const float2* __restrict__ tabg; // {g_k, g_k+1 - g_k}
    int* flag;                      // sticky state flag (bit 0: floor hit, bit 1: NaN)
    unsigned int* cflmax;           // non-NULL: fold max_d |u_d| + c of every finished cell into it (bit pattern of a float >= 0)
    // brick decomposition (NEXT-4): global index of cell 0 along the (sweep, a, b) axes, and the brick layers received
    // from the two neighbours along the sweep axis (PPM_BC_HALO faces): [bricks along b][bricks along a] records, strides HBa, HBb
    int org_d, org_a, org_b;
    const float* halo_lo;
    const float* halo_hi;
    long long HBa, HBb;
    unsigned long long k10;         // the packed f32x2 constant (1.0f, 0.0f)
    int fv_shortcut;                // PPM_OPT_FV_SHORTCUT: skip the PPB remap where FV is uniform under a whole warp (same values)
    // two-fluid EOS (NEXT-4, reading R25): beta(f) = beta2 + f dbeta, beta2 = 1/(gamma_rest - 1), dbeta = 1/(gamma_tracked - 1) - beta2
    int twof;
    float beta2, dbeta;
    // confining sphere (NEXT-3): centre along the (sweep, a, b) axes, radius^2, cell size — fp64, the oracle's criterion
    int sphere;
    double sph_dx, sph_r2, sph_cd, sph_ca, sph_cb;
    // 3-D flattening mode: F~ of every cell, [brick][4z][4y][4x] (a brick is 64 floats: strides = SB / 15); else NULL
    const float* flat;
    long long FBd, FBa, FBb;
    // PPB-only sweeps, bulk-staged path: the brick records at in + hdelta hold the hydro fields (the other state buffer, or 0)
    long long hdelta;
};

struct ppm_ctx {
    ppm_params prm;
    float* buf[2];
    int cur;                        // buf[cur] holds the state ...
    int hyd;                        // ... except, after PPB-only sweeps, the hydro part of the records: that is in buf[hyd] (ppm_make_whole)
    cudaStream_t stream;
    int device;                     // the device that owns buf[0], buf[1]; every entry point switches to it
    float4* tab;                    // device gravity table (fp32 nodes)
    float4* tabp;                   // device: interval records {rho0, p0, d rho0, d p0} (the sweeps' lookups)
    float2* tabg;                   // device: interval records {g, d g}
    double* tab64;                  // device gravity table as doubles {g, rho0, p0} x n (set/get/reductions)
    int* flag;                      // device sticky flag
    unsigned int* cflmax;           // device: ordered-uint encoded max
    double* partial;                // device: conserved partial sums [6][nblocks]
    double* result;                 // device: final 6 sums
    int nblocks_red;
    int chunk;
    int nbx, nby, nbz;              // bricks per axis (extents rounded up to multiples of 4)
    int flat3d;                     // PPM_OPT_FLATTEN3D
    int sphere;                     // ppm_set_sphere: confining sphere on (NEXT-3)
    double sph_r, sph_c[3];         // its radius and centre
    int org[3];                     // ppm_set_origin: global index of cell (0,0,0) (a sub-domain of a brick decomposition; else 0)
    const float* halo[3][2];        // ppm_set_halo: per axis, low / high side: the neighbour's brick layer (borrowed device memory)
    int twof;                       // ppm_set_two_fluid: two-fluid equation of state on (NEXT-4)
    double gam_tracked, gam_rest;   // adiabatic index of the tracked fluid (FV) and of the rest
    float* R0c;                     // device: rho0 / p0 at every cell centre (3-D flattening mode with RADIAL gravity; library-owned), else NULL
    float* P0c;
    float* F3;                      // device: 3-D shock detector field (library-owned, allocated when the option is set)
    int sms;                        // multiprocessors of the device
    int cfl_fused;                  // PPM_OPT_CFL_FUSED (default 1): the last sweep of ppm_step also reduces the CFL maximum of the new state
    int cfl_valid;                  // cflmax holds the maximum of the CURRENT state (set by a fused step, cleared by anything else that changes the state)
    int io_path;                    // PPM_OPT_IO_PATH: 0 = bulk-staged where the sweep-axis extent is whole bricks, 1 = direct everywhere
    int fv_shortcut;                // PPM_OPT_FV_SHORTCUT (default 1)
    int pert_io;                    // PPM_OPT_STATE_FORM: 1 = ppm_set_state / ppm_get_state exchange rho', p' (perturbation form, as stored)
    long long launches;
    char err[512];
};

// launchers (defined in the .cu files)
cudaError_t ppm_launch_sweep(ppm_ctx* c, int axis, double dt, bool advect = false, bool fuse_cfl = false);   // advect: PPB-only sweep (NEXT-2); fuse_cfl: S10 folded into this sweep (bulk path only)
bool ppm_axis_is_bulk(const ppm_ctx* c, int axis);
int ppm_tail_chunk(int ntail, int slots, int n);   // segment length for the pencils of the ragged last wave
cudaError_t ppm_launch_to_perturbation(ppm_ctx* c, const float* dense_slab, float* state, int z0, int nzs);
cudaError_t ppm_launch_to_full(ppm_ctx* c, const float* state, float* dst, int z0, int nzs);
cudaError_t ppm_make_whole(ppm_ctx* c);          // hyd != cur: copies the hydro part of every record into buf[cur]; every reader of the state calls it
cudaError_t ppm_launch_cfl(ppm_ctx* c);
cudaError_t ppm_launch_flatten3d(ppm_ctx* c);
cudaError_t ppm_launch_base_fill(ppm_ctx* c);    // fills R0c, P0c
cudaError_t ppm_launch_conserved(ppm_ctx* c);
void ppm_static_scratch_prepare();                 // looks the array's address up for the current device (never fails the caller)
cudaError_t ppm_launch_conserved_static(ppm_ctx* c, int nblocks, double* dev_out);   // partial sums in a file-scope device array
cudaError_t ppm_run_fma_peak(ppm_ctx* c, double* tflops);
cudaError_t ppm_launch_spin_up(ppm_ctx* c, double domega);
cudaError_t ppm_launch_pack_halo(ppm_ctx* c, int axis, int side, float* dst);
