// ppm_aux.cu — state conversion (full <-> perturbation form), the CFL max-reduction
// (C6, "the algorithm is explicit") and the conserved sums (C7).  sm_100a.
#include "ppm_internal.h"

namespace {

struct AuxParams {
    int nx, ny, nz;
    long long nslots;                   // storage slots = bricks * 64 (pad cells included)
    double dx, gamma;
    int grav_kind, tab_n;
    double s0, ds, cx, cy, cz;
    const double* __restrict__ tab64;   // node k: g, rho0, p0 (3 doubles)
    int nbx, nby;                       // bricks along x, y
    int bc[6];
    const float4* __restrict__ tab32;   // node k: {rho0, p0, g, 0} (the sweeps' fp32 table)
    float dxf, cxf, cyf, czf, s0f, inv_dsf, gamf;   // fp32 copies for the fp32 kernels (no fp64 conversions in their loops)
    int sphere;                         // NEXT-3: confining sphere on
    const float* __restrict__ R0c;      // 3-D flattening mode with RADIAL gravity: rho0, p0 at every cell centre as the sweeps evaluate them
    const float* __restrict__ P0c;      // ([brick][4z][4y][4x], filled once when the option is set), else NULL
    int ox, oy, oz;                     // ppm_set_origin: global index of cell (0,0,0) (brick decomposition), else 0
    int twof;                           // NEXT-4: two-fluid EOS, beta(f) = beta2 + f dbeta (reading R25)
    double beta2, dbeta;
    float beta2f, dbetaf;
    int pert_io;                        // PPM_OPT_STATE_FORM = 1: the boundary arrays carry rho', p' as stored (no base state added / removed)
    double sph_r2, sph_cx, sph_cy, sph_cz;
};

// NEXT-3 (reading R23): a cell is solid when its centre lies outside the sphere — the oracle's criterion, operation by
// operation in fp64 with no contraction: ((X-cx)^2 + (Y-cy)^2) + (Z-cz)^2 > R^2
__device__ __forceinline__ bool aux_is_solid(const AuxParams& A, int i, int j, int k) {
    if (!A.sphere) return false;
    const double x = __dsub_rn(__dmul_rn((double)i + 0.5, A.dx), A.sph_cx), y = __dsub_rn(__dmul_rn((double)j + 0.5, A.dx), A.sph_cy),
                 z = __dsub_rn(__dmul_rn((double)k + 0.5, A.dx), A.sph_cz);
    return __dadd_rn(__dadd_rn(__dmul_rn(x, x), __dmul_rn(y, y)), __dmul_rn(z, z)) > A.sph_r2;
}

// float offset of field 0 of cell (i,j,k): brick record [bz][by][bx][15][4z][4y][4x]; field f is 64*f further
__device__ __forceinline__ long long cell_offset(const AuxParams& A, int i, int j, int k) {
    return (long long)(((k >> 2) * A.nby + (j >> 2)) * A.nbx + (i >> 2)) * PPM_BRICK_FLOATS + ((k & 3) << 4 | (j & 3) << 2 | (i & 3));   // (brick index < 2^25: ppm_create caps the cells at 2^31)
}
// storage slot t (brick * 64 + cell in brick) -> (i,j,k) and the offset of field 0; false for a pad cell
__device__ __forceinline__ bool cell_of(const AuxParams& A, long long t, int& i, int& j, int& k, long long& off) {
    const int c = (int)(t & 63);
    const unsigned B = (unsigned)(t >> 6);                 // brick index < 2^25 (ppm_create caps the cells at 2^31): 32-bit divisions
    off = (long long)B * PPM_BRICK_FLOATS + c;
    const unsigned q = B / (unsigned)A.nbx;
    const int bx = (int)(B - q * (unsigned)A.nbx);
    const int bz = (int)(q / (unsigned)A.nby);
    const int by = (int)(q - (unsigned)bz * (unsigned)A.nby);
    i = bx * 4 + (c & 3); j = by * 4 + ((c >> 2) & 3); k = bz * 4 + (c >> 4);
    return i < A.nx && j < A.ny && k < A.nz;
}

// fp64 base state at a cell centre (same definition as the sweep's, evaluated in double: the
// conversion full <-> perturbation must not add fp32 error of the size of the base state)
__device__ __forceinline__ void base64(const AuxParams& A, int i, int j, int k, double& r0, double& p0) {
    r0 = 0.0; p0 = 0.0;
    if (A.grav_kind == PPM_GRAV_CONST_Z) {
        const double* t = A.tab64 + 3 * (2 * k + 2 * PPM_NGHOST + 1);
        r0 = t[1]; p0 = t[2];
    } else if (A.grav_kind == PPM_GRAV_RADIAL) {
        const double x = (i + A.ox + 0.5) * A.dx - A.cx, y = (j + A.oy + 0.5) * A.dx - A.cy, z = (k + A.oz + 0.5) * A.dx - A.cz;
        const double r = sqrt(x * x + y * y + z * z);
        double t = (r - A.s0) / A.ds;
        int kk = (int)floor(t);
        kk = min(max(kk, 0), A.tab_n - 2);
        const double w = t - (double)kk;
        const double* a = A.tab64 + 3 * kk;
        r0 = (1.0 - w) * a[1] + w * a[4];
        p0 = (1.0 - w) * a[2] + w * a[5];
    }
}

// state (layout order, perturbation form) <- dense slab [15][nzs][ny][nx] of full values, z-planes [z0, z0+nzs)
__global__ void __launch_bounds__(256) to_perturbation_kernel(AuxParams A, const float* __restrict__ src, float* __restrict__ st, int z0, int nzs) {
    const long long plane = (long long)A.nx * A.ny, tot = plane * nzs;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < tot; t += (long long)gridDim.x * blockDim.x) {
        const int k = z0 + (int)(t / plane);
        const long long rem = t % plane;
        const int j = (int)(rem / A.nx), i = (int)(rem % A.nx);
        const long long id = cell_offset(A, i, j, k);
        double r0, p0;
        base64(A, i, j, k, r0, p0);
#pragma unroll
        for (int f = 0; f < PPM_NFIELDS; ++f) {
            float v = src[f * tot + t];
            if (f == 0 && !A.pert_io) v = (float)((double)v - r0);
            if (f == 4 && !A.pert_io) v = (float)((double)v - p0);
            st[id + 64 * f] = v;
        }
    }
}

// dst (dense slab [15][nzs][ny][nx]) <- full state of z-planes [z0, z0+nzs)
__global__ void __launch_bounds__(256) to_full_kernel(AuxParams A, const float* __restrict__ st, float* __restrict__ dst, int z0, int nzs) {
    const long long plane = (long long)A.nx * A.ny, tot = plane * nzs;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < tot; t += (long long)gridDim.x * blockDim.x) {
        const int k = z0 + (int)(t / plane);
        const long long rem = t % plane;
        const int j = (int)(rem / A.nx), i = (int)(rem % A.nx);
        const long long id = cell_offset(A, i, j, k);
        double r0, p0;
        base64(A, i, j, k, r0, p0);
#pragma unroll
        for (int f = 0; f < PPM_NFIELDS; ++f) {
            float v = st[id + 64 * f];
            if (f == 0 && !A.pert_io) v = (float)((double)v + r0);
            if (f == 4 && !A.pert_io) v = (float)((double)v + p0);
            dst[f * tot + t] = v;
        }
    }
}

// The same two conversions for grids whose x extent is a multiple of 4 (every bulk-staged grid): pure permutes moved as float4.
// A warp takes one field of two x-adjacent bricks: lane = (brick of the pair, z layer, y row) reads the 4 x-cells of its row from
// the dense slab (the two bricks' rows are 32 contiguous bytes: whole sectors) and writes them into the brick record, where the
// 16 rows of a field are 256 contiguous bytes.  TO_PERT: dense full values -> brick records in perturbation form; else the reverse.
template <bool TO_PERT>
__global__ void __launch_bounds__(256) convert4_kernel(AuxParams A, const float* __restrict__ from, float* __restrict__ to, int z0, int nzs) {
    // one CTA per row of bricks along x (blockIdx.x = by, blockIdx.y = brick layer of the slab); its 8 warps share out the brick pairs
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, sub = lane >> 4, zz = (lane >> 2) & 3, yy = lane & 3;
    const int nbxp = (A.nbx + 1) >> 1;
    const int by = blockIdx.x, bz = (z0 >> 2) + blockIdx.y;
    const int y = by * 4 + yy, z = bz * 4 + zz;
    if (y >= A.ny || z < z0 || z >= z0 + nzs) return;
    const long long plane = (long long)nzs * A.ny * A.nx;                              // one field of the dense slab
    const long long drow = ((long long)(z - z0) * A.ny + y) * A.nx;                    // this lane's row in it
    const long long brow = (long long)(bz * A.nby + by) * A.nbx * PPM_BRICK_FLOATS + zz * 16 + yy * 4;
    const bool based = !A.pert_io && A.grav_kind != PPM_GRAV_NONE;
    for (int bxp = warp; bxp < nbxp; bxp += 8) {
        const int bx = 2 * bxp + sub;
        if (bx >= A.nbx) continue;
        const float* fd = from + (TO_PERT ? drow + bx * 4 : brow + (long long)bx * PPM_BRICK_FLOATS);
        float* td = to + (TO_PERT ? brow + (long long)bx * PPM_BRICK_FLOATS : drow + bx * 4);
        float4 v[PPM_NFIELDS];
#pragma unroll
        for (int f = 0; f < PPM_NFIELDS; ++f) v[f] = *reinterpret_cast<const float4*>(fd + (TO_PERT ? f * plane : (long long)f * 64));
        if (based) {
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                double r0, p0;
                base64(A, bx * 4 + e, y, z, r0, p0);
                float* c0 = &v[0].x; float* c4 = &v[4].x;
                c0[e] = TO_PERT ? (float)((double)c0[e] - r0) : (float)((double)c0[e] + r0);
                c4[e] = TO_PERT ? (float)((double)c4[e] - p0) : (float)((double)c4[e] + p0);
            }
        }
#pragma unroll
        for (int f = 0; f < PPM_NFIELDS; ++f) *reinterpret_cast<float4*>(td + (TO_PERT ? (long long)f * 64 : f * plane)) = v[f];
    }
}

// fp32 base state (rho0, p0) at a cell centre, as the sweeps evaluate it
__device__ __forceinline__ float2 base32(const AuxParams& A, int i, int j, int k) {
    if (A.grav_kind == PPM_GRAV_CONST_Z) {
        const float4 v = __ldg(A.tab32 + 2 * k + 2 * PPM_NGHOST + 1);
        return make_float2(v.x, v.y);
    }
    if (A.grav_kind == PPM_GRAV_RADIAL) {
        const float dx = A.dxf;
        const float x = ((float)(i + A.ox) + 0.5f) * dx - A.cxf, y = ((float)(j + A.oy) + 0.5f) * dx - A.cyf, z = ((float)(k + A.oz) + 0.5f) * dx - A.czf;
        const float r2 = fmaf(x, x, fmaf(y, y, z * z));
        const float r = r2 * rsqrtf(fmaxf(r2, 1e-30f));
        const float t = (r - A.s0f) * A.inv_dsf;
        int kk = (int)floorf(t);
        kk = min(max(kk, 0), A.tab_n - 2);
        const float w = t - (float)kk;
        const float4 a = __ldg(A.tab32 + kk), b = __ldg(A.tab32 + kk + 1);
        return make_float2(fmaf(w, b.x - a.x, a.x), fmaf(w, b.y - a.y, a.y));
    }
    return make_float2(0.f, 0.f);
}

// streaming read: touched once, keep it out of L1
__device__ __forceinline__ float ld_stream(const float* p) { float v; asm volatile("ld.global.nc.L1::no_allocate.f32 %0, [%1];" : "=f"(v) : "l"(p)); return v; }

// One warp per brick record: a lane takes cells `lane` and `lane + 32` of the brick, i.e. the hydro part of the record
// (5 fields x 256 B, contiguous) is read as ten fully coalesced 128-byte rows that are all in flight before the first
// one is used.  c = x rsqrt(x), x = gamma p / rho — the formula of the reduction fused into the sweeps (ppm_sweep.cu).
__global__ void __launch_bounds__(256) cfl_kernel(const AuxParams A, const float* __restrict__ st, unsigned int* __restrict__ out, int* flag) {
    const int lane = threadIdx.x & 31;
    const long long nbricks = A.nslots >> 6;
    const long long nwarps = (long long)gridDim.x * (blockDim.x >> 5);
    const float gam = A.gamf;
    float vmax = 0.f;
    bool bad = false;
    for (long long B = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5; B < nbricks; B += nwarps) {
        const float* p = st + B * PPM_BRICK_FLOATS + lane;
        float v[2][5], fv[2] = {0.f, 0.f};
#pragma unroll
        for (int h = 0; h < 2; ++h)
#pragma unroll
            for (int f = 0; f < 5; ++f) v[h][f] = ld_stream(p + 32 * h + 64 * f);
        if (A.twof) { fv[0] = ld_stream(p + 64 * 5); fv[1] = ld_stream(p + 32 + 64 * 5); }      // m000: the mixture's Gamma
        const unsigned q = (unsigned)B / (unsigned)A.nbx;
        const int bx = (int)((unsigned)B - q * (unsigned)A.nbx);
        const int bz = (int)(q / (unsigned)A.nby);
        const int by = (int)(q - (unsigned)bz * (unsigned)A.nby);
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int c = lane + 32 * h;
            const int i = bx * 4 + (c & 3), j = by * 4 + ((c >> 2) & 3), k = bz * 4 + (c >> 4);
            if (i >= A.nx || j >= A.ny || k >= A.nz) continue;             // pad cell of a ragged grid
            if (aux_is_solid(A, i, j, k)) continue;                        // outside the confining sphere: not part of the flow
            const float2 b0 = base32(A, i, j, k);                          // fp32 base state, as the sweeps evaluate it
            const float rho = b0.x + v[h][0], pr = b0.y + v[h][4];
            const float gk = A.twof ? 1.0f + __fdividef(1.0f, fmaf(__saturatef(fv[h]), A.dbetaf, A.beta2f)) : gam;
            const float xs = gk * pr * __fdividef(1.0f, rho);
            const float cs = xs * rsqrtf(fmaxf(xs, 1e-37f));
            const float sp = fmaxf(fabsf(v[h][1]), fmaxf(fabsf(v[h][2]), fabsf(v[h][3]))) + cs;
            bad |= !(sp == sp) || !(rho > 0.f) || !(pr > 0.f);
            vmax = fmaxf(vmax, sp);
        }
    }
    if (bad) atomicOr(flag, 2);
    const unsigned m = __reduce_max_sync(0xffffffffu, __float_as_uint(fmaxf(vmax, 0.f)));
    __shared__ unsigned sm[8];
    if (lane == 0) sm[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x < 32) {
        const unsigned w = __reduce_max_sync(0xffffffffu, threadIdx.x < (blockDim.x >> 5) ? sm[threadIdx.x] : 0u);
        if (threadIdx.x == 0) atomicMax(out, w);
    }
}

// conserved sums: fp64 accumulation, fixed assignment of cells to threads, fixed reduction trees
__global__ void __launch_bounds__(256) conserved_kernel(AuxParams A, const float* __restrict__ st, double* __restrict__ partial) {
    double acc[6] = {0, 0, 0, 0, 0, 0};
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < A.nslots; t += (long long)gridDim.x * blockDim.x) {
        int i, j, k;
        long long o;
        if (!cell_of(A, t, i, j, k, o)) continue;
        if (aux_is_solid(A, i, j, k)) continue;            // NEXT-3: the sums run over the fluid cells
        double r0, p0;
        base64(A, i, j, k, r0, p0);
        const double rho = r0 + (double)st[o], p = p0 + (double)st[o + 4 * 64];
        const double u = st[o + 64], v = st[o + 2 * 64], w = st[o + 3 * 64];
        acc[0] += rho; acc[1] += rho * u; acc[2] += rho * v; acc[3] += rho * w;
        const double f000 = st[o + 5 * 64];
        const double beta = A.twof ? A.beta2 + fmin(fmax(f000, 0.0), 1.0) * A.dbeta : 1.0 / (A.gamma - 1.0);     // e = p beta(f)
        acc[4] += (A.twof ? p * beta : p / (A.gamma - 1.0)) + 0.5 * rho * (u * u + v * v + w * w);
        acc[5] += rho * (double)st[o + 5 * 64];
    }
    __shared__ double sm[6][256];
#pragma unroll
    for (int q = 0; q < 6; ++q) sm[q][threadIdx.x] = acc[q];
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if (threadIdx.x < s) {
#pragma unroll
            for (int q = 0; q < 6; ++q) sm[q][threadIdx.x] += sm[q][threadIdx.x + s];
        }
        __syncthreads();
    }
    if (threadIdx.x < 6) partial[threadIdx.x * gridDim.x + blockIdx.x] = sm[threadIdx.x][0];
}

__global__ void conserved_final_kernel(const double* __restrict__ partial, int nb, double dv, double* __restrict__ out) {
    // one warp per quantity would do; a single thread per quantity keeps the order fixed and trivial
    if (threadIdx.x < 6) {
        double s = 0.0;
        for (int b = 0; b < nb; ++b) s += partial[threadIdx.x * nb + b];
        out[threadIdx.x] = s * dv;
    }
}


// ---- NEXT-1 ("a fully 3-D treatment of the shock dissipation"): the 3-D shock detector
// F~_i = max over the three directions d of the H4 coefficient f~^d_i = steep * jump * conv, each evaluated along d
// (full p at i-2..i+2, u_d at i-1, i+1, c_i) on the state the step starts from; ghost cells by the boundary images
// (periodic wrap / mirror with the normal velocity negated).  One value per cell, [brick][4z][4y][4x].
__device__ __forceinline__ int aux_image(int i, int n, int bc_lo, int bc_hi, float& sgn) {
    sgn = 1.0f;
    if ((unsigned)i < (unsigned)n) return i;
    const int bcx = (i < 0) ? bc_lo : bc_hi;
    if (bcx == PPM_BC_PERIODIC) return ((i % n) + n) % n;
    sgn = -1.0f;
    const int s = (i < 0) ? (-1 - i) : (2 * n - 1 - i);
    return min(max(s, 0), n - 1);
}

// CTA = a tile of 2x2x2 bricks (8x8x8 cells), one thread per cell; shared memory holds the full pressure of the tile and
// of its two-cell arms along the three axes (the detector needs no corners): 2.5 staged points per cell instead of 13.
constexpr int F3_T = 8, F3_H = 2, F3_W = F3_T + 2 * F3_H, F3_N = F3_W * F3_W * F3_W;
__device__ __forceinline__ int f3_idx(int lx, int ly, int lz) { return ((lz + F3_H) * F3_W + (ly + F3_H)) * F3_W + (lx + F3_H); }

// Full pressure of one point of a BOUNDARY tile (the tile itself: d < 0; its arms: d = axis of the arm) -> shared memory,
// with the boundary images of the grid faces.
__device__ __forceinline__ void f3_point_edge(const AuxParams& A, const float* __restrict__ st, float* sP,
                                              int ox0, int oy0, int oz0, int lx, int ly, int lz, int d) {
    int gx = ox0 + lx, gy = oy0 + ly, gz = oz0 + lz;
    const int si = f3_idx(lx, ly, lz);
    float sgn;
    // A point outside the grid along ONE axis is the boundary image of a cell along that axis (an arm point
    // by construction, a tile point when the tile overhangs a ragged grid); outside along two axes it is
    // never anybody's neighbour.
    const bool ox = (unsigned)gx >= (unsigned)A.nx, oy = (unsigned)gy >= (unsigned)A.ny, oz = (unsigned)gz >= (unsigned)A.nz;
    const int nout = (int)ox + (int)oy + (int)oz;
    const int dout = ox ? 0 : (oy ? 1 : (oz ? 2 : d));
    if (nout > 1 || (d >= 0 && nout == 1 && dout != d)) { sP[si] = 1.f; return; }
    if (ox) gx = aux_image(gx, A.nx, A.bc[0], A.bc[1], sgn);
    if (oy) gy = aux_image(gy, A.ny, A.bc[2], A.bc[3], sgn);
    if (oz) gz = aux_image(gz, A.nz, A.bc[4], A.bc[5], sgn);
    const int br = ((gz >> 2) * A.nby + (gy >> 2)) * A.nbx + (gx >> 2), cb = (gz & 3) << 4 | (gy & 3) << 2 | (gx & 3);
    const float p0 = A.P0c ? __ldg(A.P0c + br * 64LL + cb) : base32(A, gx, gy, gz).y;
    sP[si] = p0 + st[(long long)br * PPM_BRICK_FLOATS + 4 * 64 + cb];
}

// One slab of the arms of an INTERIOR tile: face (D, SIDE), the 2 x 4 x 4 cells of neighbour brick (ta, tb) that touch the
// tile — one warp, lane = (depth e, transverse cell a, bq).  Axis and side are compile-time, the brick is warp-uniform: no
// index decoding per point.
template <int D, int SIDE>
__device__ __forceinline__ void f3_arm(const AuxParams& A, const float* __restrict__ st, float* sP, int B0, int ox0, int oy0, int oz0,
                                       int ta, int tb, int lane) {
    constexpr int DA = (D == 0) ? 1 : 0, DB = (D == 2) ? 1 : 2;           // the two transverse axes, in increasing order
    const int e = lane & 1, a = (lane >> 1) & 3, bq = lane >> 3;
    const int sB[3] = {1, A.nbx, A.nbx * A.nby};
    const int br = B0 + (SIDE ? 2 : -1) * sB[D] + ta * sB[DA] + tb * sB[DB];
    const int ca = SIDE ? e : 2 + e;                                      // cell along D inside that brick
    const int cb = (ca << (2 * D)) | (a << (2 * DA)) | (bq << (2 * DB));
    int l[3];
    l[D] = SIDE ? F3_T + e : e - F3_H; l[DA] = 4 * ta + a; l[DB] = 4 * tb + bq;
    float p0;
    if (A.P0c) p0 = __ldg(A.P0c + br * 64LL + cb);
    else p0 = base32(A, ox0 + l[0], oy0 + l[1], oz0 + l[2]).y;
    sP[f3_idx(l[0], l[1], l[2])] = p0 + st[(long long)br * PPM_BRICK_FLOATS + 4 * 64 + cb];
}

// CTA = a tile of 2x2x2 bricks, 128 threads, FOUR cells per thread (the same cell of the four bricks of a y-z square: four
// times the loads in flight per warp, the per-thread set-up paid once; 2 and 8 cells per thread measured slower).  Phase 1
// stages the full pressure of the tile and of its arms; phase 2 evaluates the three 1-D detectors from shared memory.  The
// velocities and the density enter only where a pressure jump is near (conv, c): those few warps read them from the state.
#ifndef PPM_F3_CPT
#define PPM_F3_CPT 4
#endif
#ifndef PPM_F3_MINB
#define PPM_F3_MINB (4 * PPM_F3_CPT)
#endif
constexpr int F3_CPT = PPM_F3_CPT, F3_THREADS = 512 / F3_CPT;      // cells per thread (2: bricks adjacent in z; 4: in y and z; 8: all of the tile's)
__global__ void __launch_bounds__(F3_THREADS, PPM_F3_MINB) flatten3d_kernel(const AuxParams A, const float* __restrict__ st, float* __restrict__ F3) {
    __shared__ float sP[F3_N];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int org[3] = {(int)blockIdx.x * F3_T, (int)blockIdx.y * F3_T, (int)blockIdx.z * F3_T};
    const float gam = A.gamf;
    const bool inside = org[0] >= F3_H && org[1] >= F3_H && org[2] >= F3_H &&
                        org[0] + F3_T + F3_H <= A.nx && org[1] + F3_T + F3_H <= A.ny && org[2] + F3_T + F3_H <= A.nz;
    const int b = tid >> 6, c = tid & 63;                                  // thread = (first of its bricks, cell in brick)
    const int lx = (b & 1) * 4 + (c & 3), ly = (b >> 1) * 4 + ((c >> 2) & 3), lz = c >> 4;       // first cell; cell h: see hy, hz
    const int gx = org[0] + lx, gy = org[1] + ly;
    const int s0 = f3_idx(lx, ly, lz);
    const int B0 = ((org[2] >> 2) * A.nby + (org[1] >> 2)) * A.nbx + (org[0] >> 2);
    const int bz = A.nbx * A.nby;
    const int brick0 = B0 + (b & 1) + (b >> 1) * A.nbx;                    // (meaningful where valid)
    // cell h of a thread: the same cell of the brick shifted by (hx, hy, hz) bricks
    auto hx = [](int h) { return F3_CPT == 8 ? (h & 1) : 0; };
    auto hy = [](int h) { return F3_CPT == 8 ? ((h >> 1) & 1) : (F3_CPT == 4 ? (h & 1) : 0); };
    auto hz = [](int h) { return F3_CPT == 8 ? (h >> 2) : (F3_CPT == 4 ? (h >> 1) : h); };
    if (inside) {
        {   // the tile itself: coalesced brick reads
            float p0[F3_CPT], pq[F3_CPT];
#pragma unroll
            for (int h = 0; h < F3_CPT; ++h) {
                const int br = brick0 + hx(h) + hy(h) * A.nbx + hz(h) * bz;
                p0[h] = A.P0c ? __ldg(A.P0c + br * 64LL + c) : base32(A, gx + 4 * hx(h), gy + 4 * hy(h), org[2] + lz + 4 * hz(h)).y;
                pq[h] = st[(long long)br * PPM_BRICK_FLOATS + 4 * 64 + c];
            }
#pragma unroll
            for (int h = 0; h < F3_CPT; ++h) sP[s0 + 4 * hx(h) + 4 * hy(h) * F3_W + 4 * hz(h) * F3_W * F3_W] = p0[h] + pq[h];
        }
        // the arms: 6 faces x 4 neighbour bricks = 24 slabs of 32 points, dealt to the warps by (neighbour brick, side)
        constexpr int NW = F3_THREADS / 32;
#pragma unroll
        for (int i = 0; i < 8 / NW; ++i) {
            const int k = warp + i * NW, ta = k & 1, tb = (k >> 1) & 1;
            if ((k >> 2) == 0) {
                f3_arm<0, 0>(A, st, sP, B0, org[0], org[1], org[2], ta, tb, lane);
                f3_arm<1, 0>(A, st, sP, B0, org[0], org[1], org[2], ta, tb, lane);
                f3_arm<2, 0>(A, st, sP, B0, org[0], org[1], org[2], ta, tb, lane);
            } else {
                f3_arm<0, 1>(A, st, sP, B0, org[0], org[1], org[2], ta, tb, lane);
                f3_arm<1, 1>(A, st, sP, B0, org[0], org[1], org[2], ta, tb, lane);
                f3_arm<2, 1>(A, st, sP, B0, org[0], org[1], org[2], ta, tb, lane);
            }
        }
    } else {
#pragma unroll
        for (int h = 0; h < F3_CPT; ++h) f3_point_edge(A, st, sP, org[0], org[1], org[2], lx + 4 * hx(h), ly + 4 * hy(h), lz + 4 * hz(h), -1);
        // 6 faces x 2 depths x 64 points = 768 arm points; a warp works on one (face, depth) slab half
        for (int r = tid; r < 6 * 2 * 64; r += F3_THREADS) {
            const int f = r >> 7, w = r & 127, h = w >> 6, a = w & 7, bb = (w >> 3) & 7;
            const int d = f >> 1;
            const int along = (f & 1) ? F3_T + h : -1 - h;
            const int ax = (d == 0) ? along : (d == 1 ? bb : a);
            const int ay = (d == 1) ? along : (d == 2 ? bb : a);
            const int az = (d == 2) ? along : (d == 0 ? bb : a);
            f3_point_edge(A, st, sP, org[0], org[1], org[2], ax, ay, az, d);
        }
    }
    __syncthreads();
    const int stride[3] = {1, F3_W, F3_W * F3_W};
    const int nd[3] = {A.nx, A.ny, A.nz};
#pragma unroll
    for (int h = 0; h < F3_CPT; ++h) {
        const int g[3] = {gx + 4 * hx(h), gy + 4 * hy(h), org[2] + lz + 4 * hz(h)};
        const int sc = s0 + 4 * hx(h) + 4 * hy(h) * F3_W + 4 * hz(h) * F3_W * F3_W;
        const int brick = brick0 + hx(h) + hy(h) * A.nbx + hz(h) * bz;
        const bool valid = g[0] < A.nx && g[1] < A.ny && g[2] < A.nz;          // (a tile may overhang a ragged grid)
        float F = 0.f;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const int sd = stride[d];
            const float pp = sP[sc + sd], pm = sP[sc - sd];
            const float d1 = pp - pm, pmin = fminf(pp, pm);
            // the jump ramp clamp(3|d1|/min(p) - 1) is zero unless the pressure changes by a third over two cells: when no cell of
            // the warp is that near a shock along d the coefficient is the same zero without the three divisions
            if (__any_sync(0xffffffffu, valid && 3.0f * fabsf(d1) > pmin)) {
                if (valid) {
                    // u_d of the two neighbours along d (boundary image: the normal velocity changes sign in a mirror) and the
                    // density of the cell, from the state
                    float um = 0.f, up = 0.f;
#pragma unroll
                    for (int sgi = 0; sgi < 2; ++sgi) {
                        int q[3] = {g[0], g[1], g[2]};
                        float sgn = 1.f;
                        q[d] += sgi ? 1 : -1;
                        if ((unsigned)q[d] >= (unsigned)nd[d]) q[d] = aux_image(q[d], nd[d], A.bc[2 * d], A.bc[2 * d + 1], sgn);
                        const float u = sgn * st[cell_offset(A, q[0], q[1], q[2]) + (1 + d) * 64];
                        if (sgi) up = u; else um = u;
                    }
                    const float r0 = A.P0c ? __ldg(A.R0c + brick * 64LL + c) : base32(A, g[0], g[1], g[2]).x;
                    const float rc = r0 + st[(long long)brick * PPM_BRICK_FLOATS + c];
                    const float d2 = sP[sc + 2 * sd] - sP[sc - 2 * sd];
                    const float ics = rsqrtf(gam * __fdividef(sP[sc], rc)) * 20.0f;        // 1 / (0.05 c)
                    const float steep = __saturatef(10.0f * (__fdividef(fabsf(d1), fmaxf(fabsf(d2), PPM_TINY)) - 0.75f));
                    const float jump = __saturatef(__fdividef(3.0f * fabsf(d1), pmin) - 1.0f);
                    const float conv = __saturatef((um - up) * ics);
                    F = fmaxf(F, steep * jump * conv);
                }
            }
        }
        if (valid) F3[brick * 64LL + c] = F;
    }
}

// rho0, p0 of every storage slot (pad cells included: harmless values), fp32 exactly as base32 gives them
__global__ void __launch_bounds__(256) base_fill_kernel(const AuxParams A, float* __restrict__ R0c, float* __restrict__ P0c) {
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < A.nslots; t += (long long)gridDim.x * blockDim.x) {
        int i, j, k;
        long long o;
        cell_of(A, t, i, j, k, o);
        const float2 b = base32(A, i, j, k);
        R0c[t] = b.x; P0c[t] = b.y;
    }
}

// NEXT-3 ("adding a solid body rotational flow component ... gradually over the first several thousand
// time steps"; reading R24): one increment of the ramp, du = domega e_z x (X - centre) on every fluid cell.
__global__ void __launch_bounds__(256) spin_up_kernel(const AuxParams A, float* __restrict__ st, double domega, double cx, double cy) {
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < A.nslots; t += (long long)gridDim.x * blockDim.x) {
        int i, j, k;
        long long o;
        if (!cell_of(A, t, i, j, k, o) || aux_is_solid(A, i, j, k)) continue;
        const double x = ((double)(i + A.ox) + 0.5) * A.dx - cx, y = ((double)(j + A.oy) + 0.5) * A.dx - cy;
        st[o + 64] = (float)((double)st[o + 64] - domega * y);
        st[o + 2 * 64] = (float)((double)st[o + 2 * 64] + domega * x);
    }
}

// NEXT-4 (bricks with a halo one briquette thick): one brick layer of the state — the bricks
// with index kb along `axis` — gathered into a contiguous buffer [bricks along b][bricks along a] of whole brick records (a < b the
// two other axes), the layout the sweeps read a PPM_BC_HALO ghost brick from.  Pure copy: one float4 per thread and trip.
__global__ void __launch_bounds__(256) pack_halo_kernel(const float4* __restrict__ st, float4* __restrict__ dst, int nbx, int nby, int nbz, int axis, int kb) {
    constexpr int R4 = PPM_BRICK_FLOATS / 4;                       // float4 per brick record
    const int na = (axis == 0) ? nby : nbx, nb = (axis == 2) ? nby : nbz;
    const long long tot = (long long)na * nb * R4;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < tot; t += (long long)gridDim.x * blockDim.x) {
        const int e = (int)(t % R4);
        const long long br = t / R4;
        const int a = (int)(br % na), b = (int)(br / na);
        const int bx = (axis == 0) ? kb : a, by = (axis == 1) ? kb : (axis == 0 ? a : b), bz = (axis == 2) ? kb : b;
        dst[t] = st[((long long)(bz * nby + by) * nbx + bx) * R4 + e];
    }
}

// FP32 pipe micro-benchmark (the denominator of bench.py's roofline.alu; "must be measured with an FMA
// micro-benchmark at the clock the sweep actually runs at"): 16 independent FFMA chains per thread, 8 resident warps
// per scheduler; 2 flop per lane per FFMA.
__global__ void __launch_bounds__(256) fma_peak_kernel(float* out, int iters, float a, float b) {
    float x[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) x[k] = (float)(threadIdx.x + k) * 1e-3f;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 16; ++k) x[k] = fmaf(x[k], a, b);
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < 16; ++k) s += x[k];
    if (s == 123.456f) out[0] = s;          // never true: keeps the chains alive
}

AuxParams make_aux(const ppm_ctx* c) {
    AuxParams A;
    const ppm_params& p = c->prm;
    A.nx = p.nx; A.ny = p.ny; A.nz = p.nz;
    A.nslots = (long long)c->nbx * c->nby * c->nbz * 64;
    A.dx = p.dx; A.gamma = p.gamma;
    A.grav_kind = p.grav.kind; A.tab_n = p.grav.n;
    A.s0 = p.grav.s0; A.ds = p.grav.ds;
    A.cx = p.grav.center[0]; A.cy = p.grav.center[1]; A.cz = p.grav.center[2];
    A.tab64 = c->tab64;
    A.nbx = c->nbx; A.nby = c->nby;
    for (int k = 0; k < 6; ++k) A.bc[k] = p.bc[k];
    A.tab32 = c->tab;
    A.dxf = (float)A.dx; A.cxf = (float)A.cx; A.cyf = (float)A.cy; A.czf = (float)A.cz;
    A.s0f = (float)A.s0; A.inv_dsf = (float)(A.grav_kind != PPM_GRAV_NONE ? 1.0 / A.ds : 0.0); A.gamf = (float)A.gamma;
    A.pert_io = c->pert_io;
    A.R0c = c->R0c; A.P0c = c->P0c;
    A.ox = c->org[0]; A.oy = c->org[1]; A.oz = c->org[2];
    A.twof = c->twof;
    A.beta2 = c->twof ? 1.0 / (c->gam_rest - 1.0) : 0.0;
    A.dbeta = c->twof ? 1.0 / (c->gam_tracked - 1.0) - A.beta2 : 0.0;
    A.beta2f = (float)A.beta2; A.dbetaf = (float)A.dbeta;
    A.sphere = c->sphere; A.sph_r2 = c->sph_r * c->sph_r; A.sph_cx = c->sph_c[0]; A.sph_cy = c->sph_c[1]; A.sph_cz = c->sph_c[2];
    return A;
}

int grid_for(long long n, int cap) {
    long long g = (n + 255) / 256;
    if (g > cap) g = cap;
    if (g < 1) g = 1;
    return (int)g;
}

}  // namespace

// float4 path: x extent a multiple of 4 (rows and brick rows are then 16-byte aligned: the slab sits at the start of a buffer)
static bool convert4_ok(const ppm_ctx* c) { return (c->prm.nx & 3) == 0; }
static dim3 convert4_grid(const ppm_ctx* c, int z0, int nzs) { return dim3(c->nby, ((z0 + nzs - 1) >> 2) - (z0 >> 2) + 1, 1); }

cudaError_t ppm_launch_to_perturbation(ppm_ctx* c, const float* dense_slab, float* state, int z0, int nzs) {
    if (convert4_ok(c)) {
        convert4_kernel<true><<<convert4_grid(c, z0, nzs), 256, 0, c->stream>>>(make_aux(c), dense_slab, state, z0, nzs);
        c->launches += 1;
        return cudaGetLastError();
    }
    const long long tot = (long long)c->prm.nx * c->prm.ny * nzs;
    to_perturbation_kernel<<<grid_for(tot, 148 * 16), 256, 0, c->stream>>>(make_aux(c), dense_slab, state, z0, nzs);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t ppm_launch_to_full(ppm_ctx* c, const float* state, float* dst, int z0, int nzs) {
    if (convert4_ok(c)) {
        convert4_kernel<false><<<convert4_grid(c, z0, nzs), 256, 0, c->stream>>>(make_aux(c), state, dst, z0, nzs);
        c->launches += 1;
        return cudaGetLastError();
    }
    const long long tot = (long long)c->prm.nx * c->prm.ny * nzs;
    to_full_kernel<<<grid_for(tot, 148 * 16), 256, 0, c->stream>>>(make_aux(c), state, dst, z0, nzs);
    c->launches += 1;
    return cudaGetLastError();
}

// hydro part (the first 5 of the 15 fields: 320 floats) of every brick record, src -> dst
__global__ void __launch_bounds__(256) hydro_part_copy_kernel(const float4* __restrict__ src, float4* __restrict__ dst, long long nbricks) {
    constexpr int H4 = 5 * 64 / 4, R4 = PPM_BRICK_FLOATS / 4;
    const long long tot = nbricks * H4;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < tot; t += (long long)gridDim.x * blockDim.x) {
        const long long b = t / H4;
        const int e = (int)(t - b * H4);
        dst[b * R4 + e] = src[b * R4 + e];
    }
}

// After PPB-only sweeps through the bulk-staged path the PPB coefficients are in buf[cur] and the hydro fields still in
// buf[hyd]: this brings them together in buf[cur] (one copy of 20 B per cell, only when something other than another
// PPB-only sweep looks at the state).
cudaError_t ppm_make_whole(ppm_ctx* c) {
    if (c->hyd == c->cur) return cudaSuccess;
    const long long nbricks = (long long)c->nbx * c->nby * c->nbz;
    hydro_part_copy_kernel<<<grid_for(nbricks * 80, c->sms * 8), 256, 0, c->stream>>>(reinterpret_cast<const float4*>(c->buf[c->hyd]),
                                                                                  reinterpret_cast<float4*>(c->buf[c->cur]), nbricks);
    c->hyd = c->cur;
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t ppm_launch_flatten3d(ppm_ctx* c) {
    { cudaError_t ew = ppm_make_whole(c); if (ew != cudaSuccess) return ew; }
    const dim3 grid((c->nbx + 1) / 2, (c->nby + 1) / 2, (c->nbz + 1) / 2);
    flatten3d_kernel<<<grid, F3_THREADS, 0, c->stream>>>(make_aux(c), c->buf[c->cur], c->F3);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t ppm_launch_base_fill(ppm_ctx* c) {
    AuxParams A = make_aux(c);
    A.R0c = A.P0c = nullptr;
    base_fill_kernel<<<grid_for(A.nslots, c->sms * 16), 256, 0, c->stream>>>(A, c->R0c, c->P0c);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t ppm_launch_cfl(ppm_ctx* c) {
    { cudaError_t ew = ppm_make_whole(c); if (ew != cudaSuccess) return ew; }
    cudaError_t e = cudaMemsetAsync(c->cflmax, 0, sizeof(unsigned int), c->stream);
    if (e != cudaSuccess) return e;
    const long long n = (long long)c->nbx * c->nby * c->nbz * 64;
    cfl_kernel<<<grid_for(n / 2, c->sms * 8), 256, 0, c->stream>>>(make_aux(c), c->buf[c->cur], c->cflmax, c->flag);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t ppm_launch_spin_up(ppm_ctx* c, double domega) {
    { cudaError_t ew = ppm_make_whole(c); if (ew != cudaSuccess) return ew; }
    const long long n = (long long)c->nbx * c->nby * c->nbz * 64;
    const double cx = c->sphere ? c->sph_c[0] : c->prm.grav.center[0], cy = c->sphere ? c->sph_c[1] : c->prm.grav.center[1];
    spin_up_kernel<<<grid_for(n, c->sms * 16), 256, 0, c->stream>>>(make_aux(c), c->buf[c->cur], domega, cx, cy);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t ppm_launch_pack_halo(ppm_ctx* c, int axis, int side, float* dst) {
    { cudaError_t ew = ppm_make_whole(c); if (ew != cudaSuccess) return ew; }
    const int nbd = (axis == 0) ? c->nbx : (axis == 1 ? c->nby : c->nbz);
    const int na = (axis == 0) ? c->nby : c->nbx, nb = (axis == 2) ? c->nby : c->nbz;
    const long long tot = (long long)na * nb * (PPM_BRICK_FLOATS / 4);
    pack_halo_kernel<<<grid_for(tot, c->sms * 8), 256, 0, c->stream>>>(reinterpret_cast<const float4*>(c->buf[c->cur]), reinterpret_cast<float4*>(dst),
                                                                     c->nbx, c->nby, c->nbz, axis, side ? nbd - 1 : 0);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t ppm_run_fma_peak(ppm_ctx* c, double* tflops) {
    const int iters = 4096, blocks = c->sms * 8, reps = 5;
    cudaEvent_t e0, e1;
    cudaError_t e = cudaEventCreate(&e0);
    if (e != cudaSuccess) return e;
    e = cudaEventCreate(&e1);
    if (e != cudaSuccess) { cudaEventDestroy(e0); return e; }
    double best = 0.0;
    for (int r = 0; r < reps + 1 && e == cudaSuccess; ++r) {          // first pass is a warm-up
        cudaEventRecord(e0, c->stream);
        fma_peak_kernel<<<blocks, 256, 0, c->stream>>>(reinterpret_cast<float*>(c->result), iters, 0.999f, 1e-3f);
        cudaEventRecord(e1, c->stream);
        e = cudaEventSynchronize(e1);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        const double tf = 2.0 * 16.0 * iters * 256.0 * blocks / (ms * 1e-3) / 1e12;
        if (r > 0 && tf > best) best = tf;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    c->launches += reps + 1;
    *tflops = best;
    return e == cudaSuccess ? cudaGetLastError() : e;
}

cudaError_t ppm_launch_conserved(ppm_ctx* c) {
    { cudaError_t ew = ppm_make_whole(c); if (ew != cudaSuccess) return ew; }
    const int nb = c->nblocks_red;
    conserved_kernel<<<nb, 256, 0, c->stream>>>(make_aux(c), c->buf[c->cur], c->partial);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    const double dv = c->prm.dx * c->prm.dx * c->prm.dx;
    conserved_final_kernel<<<1, 32, 0, c->stream>>>(c->partial, nb, dv, c->result);
    c->launches += 2;
    return cudaGetLastError();
}

// ---- conserved sums without any allocation (ppm_reduce_conserved_static) ---------------------------------------------
// The first pass of the reduction needs 6 partial sums per CTA.  ppm_reduce_conserved keeps them in an array ppm_create
// allocated; this variant keeps them in a file-scope device array, so the call works where cudaMalloc cannot be called
// (graph capture, serving loops).  Every GPU that loads the library holds the 48 KB until the process exits; every call
// on a device shares them.  Each first-pass CTA b < nb overwrites its six slots [q * nb + b] before the second pass reads
// exactly those, so nothing has to start at zero and a previous call's contents (another nb, another grid) are never read.
// In host code `g_static_partial` is a host-side stand-in, not a device address: the launch below gets the address
// cudaGetSymbolAddress reports, looked up once per device with that device current.
static __device__ __align__(256) double g_static_partial[6 * PPM_STATIC_RED_BLOCKS];

static double* g_static_partial_dev[64] = {};      // device ordinal -> address of g_static_partial on that device

// address of the array on the current device (no allocation; the first call per device asks the runtime)
static cudaError_t static_partial_ptr(double** out) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    double* p = g_static_partial_dev[dev];
    if (!p) {
        e = cudaGetSymbolAddress((void**)&p, g_static_partial);
        if (e != cudaSuccess) return e;
        g_static_partial_dev[dev] = p;             // (two threads racing here store the same value)
    }
    *out = p;
    return cudaSuccess;
}

// called by ppm_create with the context's device current: the look-up happens at set-up, outside any capture; should it fail
// there, ppm_reduce_conserved_static tries again and reports the error
void ppm_static_scratch_prepare() {
    double* p = nullptr;
    if (static_partial_ptr(&p) != cudaSuccess) cudaGetLastError();
}

// same two kernels, same assignment of cells to threads and the same reduction trees as ppm_launch_conserved: with
// nb = c->nblocks_red the six sums come out bit for bit the same.  The caller made c's device current.
cudaError_t ppm_launch_conserved_static(ppm_ctx* c, int nb, double* dev_out) {
    { cudaError_t ew = ppm_make_whole(c); if (ew != cudaSuccess) return ew; }
    double* partial = nullptr;
    cudaError_t e = static_partial_ptr(&partial);
    if (e != cudaSuccess) return e;
    conserved_kernel<<<nb, 256, 0, c->stream>>>(make_aux(c), c->buf[c->cur], partial);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    const double dv = c->prm.dx * c->prm.dx * c->prm.dx;
    conserved_final_kernel<<<1, 32, 0, c->stream>>>(partial, nb, dv, dev_out);
    c->launches += 2;
    return cudaGetLastError();
}
