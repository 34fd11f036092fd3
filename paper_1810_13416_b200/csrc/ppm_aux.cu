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
};

// float offset of field 0 of cell (i,j,k): brick record [bz][by][bx][15][4z][4y][4x]; field f is 64*f further
__device__ __forceinline__ long long cell_offset(const AuxParams& A, int i, int j, int k) {
    return (((long long)(k >> 2) * A.nby + (j >> 2)) * A.nbx + (i >> 2)) * PPM_BRICK_FLOATS + ((k & 3) << 4 | (j & 3) << 2 | (i & 3));
}
// storage slot t (brick * 64 + cell in brick) -> (i,j,k) and the offset of field 0; false for a pad cell
__device__ __forceinline__ bool cell_of(const AuxParams& A, long long t, int& i, int& j, int& k, long long& off) {
    const int c = (int)(t & 63);
    long long B = t >> 6;
    off = B * PPM_BRICK_FLOATS + c;
    const int bx = (int)(B % A.nbx); B /= A.nbx;
    const int by = (int)(B % A.nby);
    const int bz = (int)(B / A.nby);
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
        const double x = (i + 0.5) * A.dx - A.cx, y = (j + 0.5) * A.dx - A.cy, z = (k + 0.5) * A.dx - A.cz;
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
            if (f == 0) v = (float)((double)v - r0);
            if (f == 4) v = (float)((double)v - p0);
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
            if (f == 0) v = (float)((double)v + r0);
            if (f == 4) v = (float)((double)v + p0);
            dst[f * tot + t] = v;
        }
    }
}

// order-preserving float -> uint encoding for atomicMax (all values here are >= 0)
__device__ __forceinline__ unsigned int enc(float x) { return __float_as_uint(fmaxf(x, 0.f)); }

__global__ void __launch_bounds__(256) cfl_kernel(AuxParams A, const float* __restrict__ st, unsigned int* __restrict__ out, int* flag) {
    float vmax = 0.f;
    const float gam = (float)A.gamma;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < A.nslots; t += (long long)gridDim.x * blockDim.x) {
        int i, j, k;
        long long o;
        if (!cell_of(A, t, i, j, k, o)) continue;
        double r0, p0;
        base64(A, i, j, k, r0, p0);
        const float rho = (float)(r0 + (double)st[o]), p = (float)(p0 + (double)st[o + 4 * 64]);
        const float c = sqrtf(gam * p / rho);
        const float um = fmaxf(fabsf(st[o + 64]), fmaxf(fabsf(st[o + 2 * 64]), fabsf(st[o + 3 * 64])));
        const float v = um + c;
        if (!(v == v) || !(rho > 0.f) || !(p > 0.f)) atomicOr(flag, 2);
        vmax = fmaxf(vmax, v);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) vmax = fmaxf(vmax, __shfl_xor_sync(0xffffffffu, vmax, o));
    __shared__ float sm[8];
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = vmax;
    __syncthreads();
    if (threadIdx.x < 32) {
        float v = (threadIdx.x < (blockDim.x >> 5)) ? sm[threadIdx.x] : 0.f;
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
        if (threadIdx.x == 0) atomicMax(out, enc(v));
    }
}

// conserved sums: fp64 accumulation, fixed assignment of cells to threads, fixed reduction trees
__global__ void __launch_bounds__(256) conserved_kernel(AuxParams A, const float* __restrict__ st, double* __restrict__ partial) {
    double acc[6] = {0, 0, 0, 0, 0, 0};
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < A.nslots; t += (long long)gridDim.x * blockDim.x) {
        int i, j, k;
        long long o;
        if (!cell_of(A, t, i, j, k, o)) continue;
        double r0, p0;
        base64(A, i, j, k, r0, p0);
        const double rho = r0 + (double)st[o], p = p0 + (double)st[o + 4 * 64];
        const double u = st[o + 64], v = st[o + 2 * 64], w = st[o + 3 * 64];
        acc[0] += rho; acc[1] += rho * u; acc[2] += rho * v; acc[3] += rho * w;
        acc[4] += p / (A.gamma - 1.0) + 0.5 * rho * (u * u + v * v + w * w);
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
    return A;
}

int grid_for(long long n, int cap) {
    long long g = (n + 255) / 256;
    if (g > cap) g = cap;
    if (g < 1) g = 1;
    return (int)g;
}

}  // namespace

cudaError_t ppm_launch_to_perturbation(ppm_ctx* c, const float* dense_slab, float* state, int z0, int nzs) {
    const long long tot = (long long)c->prm.nx * c->prm.ny * nzs;
    to_perturbation_kernel<<<grid_for(tot, 148 * 16), 256, 0, c->stream>>>(make_aux(c), dense_slab, state, z0, nzs);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t ppm_launch_to_full(ppm_ctx* c, const float* state, float* dst, int z0, int nzs) {
    const long long tot = (long long)c->prm.nx * c->prm.ny * nzs;
    to_full_kernel<<<grid_for(tot, 148 * 16), 256, 0, c->stream>>>(make_aux(c), state, dst, z0, nzs);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t ppm_launch_cfl(ppm_ctx* c) {
    cudaError_t e = cudaMemsetAsync(c->cflmax, 0, sizeof(unsigned int), c->stream);
    if (e != cudaSuccess) return e;
    const long long n = (long long)c->nbx * c->nby * c->nbz * 64;
    cfl_kernel<<<grid_for(n, 148 * 8), 256, 0, c->stream>>>(make_aux(c), c->buf[c->cur], c->cflmax, c->flag);
    c->launches += 1;
    return cudaGetLastError();
}

cudaError_t ppm_launch_conserved(ppm_ctx* c) {
    const int nb = c->nblocks_red;
    conserved_kernel<<<nb, 256, 0, c->stream>>>(make_aux(c), c->buf[c->cur], c->partial);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    const double dv = c->prm.dx * c->prm.dx * c->prm.dx;
    conserved_final_kernel<<<1, 32, 0, c->stream>>>(c->partial, nb, dv, c->result);
    c->launches += 2;
    return cudaGetLastError();
}
