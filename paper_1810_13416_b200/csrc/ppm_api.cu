// ppm_api.cu — the C ABI declared in include/ppm.h (host driver; argument validation, launches).
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <vector>

#include "ppm_internal.h"

static char g_err[512] = "";

static void set_err(ppm_ctx* c, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(c ? c->err : g_err, 512, fmt, ap);
    va_end(ap);
}

#define CU(call)                                                                            \
    do {                                                                                    \
        cudaError_t e_ = (call);                                                            \
        if (e_ != cudaSuccess) {                                                            \
            set_err(c, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
            return PPM_ECUDA;                                                               \
        }                                                                                   \
    } while (0)

// Every entry point runs on the device that owns the state buffers, whatever device is current in the caller.
struct DevGuard {
    int old = -1, dev;
    explicit DevGuard(const ppm_ctx* c) : dev(c ? c->device : -1) {
        if (dev >= 0 && cudaGetDevice(&old) == cudaSuccess && old != dev) cudaSetDevice(dev); else old = -1;
    }
    ~DevGuard() { if (old >= 0) cudaSetDevice(old); }
};

static const int ORDERS[6][3] = {{0, 1, 2}, {0, 2, 1}, {1, 0, 2}, {1, 2, 0}, {2, 0, 1}, {2, 1, 0}};

extern "C" const char* ppm_last_error(const ppm_ctx* c) { return c ? c->err : g_err; }

extern "C" size_t ppm_state_floats(int nx, int ny, int nz) {
    if (nx < 1 || ny < 1 || nz < 1) return 0;
    return (size_t)((nx + 3) / 4) * (size_t)((ny + 3) / 4) * (size_t)((nz + 3) / 4) * PPM_BRICK_FLOATS;
}

extern "C" int ppm_create(ppm_ctx** out, const ppm_params* prm, float* dev_buf_a, float* dev_buf_b) {
    ppm_ctx* c = nullptr;
    if (!out) { set_err(c, "ppm_create: out is NULL"); return PPM_EINVAL; }
    *out = nullptr;
    if (!prm || !dev_buf_a || !dev_buf_b || dev_buf_a == dev_buf_b) { set_err(c, "ppm_create: NULL or aliased argument"); return PPM_EINVAL; }
    if (prm->struct_size != sizeof(ppm_params)) { set_err(c, "ppm_create: struct_size %zu != %zu", prm->struct_size, sizeof(ppm_params)); return PPM_EINVAL; }
    if (prm->nx < 1 || prm->ny < 1 || prm->nz < 1) { set_err(c, "ppm_create: grid dims must be >= 1"); return PPM_EINVAL; }
    if ((long long)prm->nx * prm->ny * prm->nz >= (1LL << 31)) { set_err(c, "ppm_create: more than 2^31 - 1 cells (2 x 15 such fields would not fit one GPU anyway)"); return PPM_EINVAL; }
    if (!(prm->dx > 0.0) || !(prm->gamma > 1.0) || !((float)prm->rho_floor > PPM_TINY) || !(prm->p_floor > 0.0)) {     // (rho_floor > 1e-30: the PPB remap divides by the new mass)
        set_err(c, "ppm_create: need dx > 0, gamma > 1, floors > 0"); return PPM_EINVAL;
    }
    if (((uintptr_t)dev_buf_a | (uintptr_t)dev_buf_b) & 127) { set_err(c, "ppm_create: device buffers must be 128-byte aligned"); return PPM_EINVAL; }
    const int ext[3] = {prm->nx, prm->ny, prm->nz};
    for (int d = 0; d < 3; ++d) {
        const int lo = prm->bc[2 * d], hi = prm->bc[2 * d + 1];
        if ((lo != PPM_BC_PERIODIC && lo != PPM_BC_REFLECT && lo != PPM_BC_HALO) || (hi != PPM_BC_PERIODIC && hi != PPM_BC_REFLECT && hi != PPM_BC_HALO)) {
            set_err(c, "ppm_create: unknown boundary type on axis %d", d); return PPM_EINVAL;
        }
        if ((lo == PPM_BC_PERIODIC) != (hi == PPM_BC_PERIODIC)) { set_err(c, "ppm_create: periodic faces must pair up (axis %d)", d); return PPM_EINVAL; }
        if ((lo == PPM_BC_HALO || hi == PPM_BC_HALO) && (ext[d] % 4 != 0 || ext[d] < 8)) {
            set_err(c, "ppm_create: an axis with a PPM_BC_HALO face needs an extent that is a multiple of 4 and >= 8 (axis %d)", d); return PPM_EINVAL;
        }
        if (lo == PPM_BC_REFLECT && ext[d] < PPM_NGHOST) { set_err(c, "ppm_create: reflecting axis %d needs >= %d cells", d, PPM_NGHOST); return PPM_EINVAL; }
    }
    const ppm_gravity& g = prm->grav;
    if (g.kind != PPM_GRAV_NONE && g.kind != PPM_GRAV_CONST_Z && g.kind != PPM_GRAV_RADIAL) { set_err(c, "ppm_create: unknown gravity kind"); return PPM_EINVAL; }
    if (g.kind != PPM_GRAV_NONE) {
        if (g.n < 2 || !g.g || !g.rho0 || !g.p0 || !(g.ds > 0.0)) { set_err(c, "ppm_create: gravity table missing"); return PPM_EINVAL; }
        if (g.kind == PPM_GRAV_CONST_Z) {
            const double tol = 1e-9 * prm->dx;
            if (g.n != 2 * (prm->nz + 2 * PPM_NGHOST) + 1 || fabs(g.s0 + PPM_NGHOST * prm->dx) > tol || fabs(g.ds - 0.5 * prm->dx) > tol) {
                set_err(c, "ppm_create: CONST_Z table must have n = 2*(nz+8)+1 nodes, s0 = -4 dx, ds = dx/2"); return PPM_EINVAL;
            }
        }
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { set_err(c, "ppm_create: no CUDA device (this library has no CPU fallback)"); return PPM_ECUDA; }

    void* mem = nullptr;
    if (posix_memalign(&mem, 64, sizeof(ppm_ctx)) != 0 || !mem) { set_err(nullptr, "ppm_create: out of host memory"); return PPM_ENOMEM; }
    memset(mem, 0, sizeof(ppm_ctx));
    c = (ppm_ctx*)mem;
    c->prm = *prm;
    c->prm.grav.g = c->prm.grav.rho0 = c->prm.grav.p0 = nullptr;   // host arrays are not kept
    c->buf[0] = dev_buf_a; c->buf[1] = dev_buf_b; c->cur = 0; c->hyd = 0;
    {   // the device that owns the buffers (falls back to the current one for memory the runtime does not know)
        cudaPointerAttributes pa;
        int cur = 0;
        cudaGetDevice(&cur);
        c->device = (cudaPointerGetAttributes(&pa, dev_buf_a) == cudaSuccess && pa.type == cudaMemoryTypeDevice) ? pa.device : cur;
        cudaGetLastError();
    }
    DevGuard guard(c);
    c->stream = (cudaStream_t)prm->stream;
    c->nblocks_red = 148 * 4;
    if (cudaDeviceGetAttribute(&c->sms, cudaDevAttrMultiProcessorCount, c->device) != cudaSuccess || c->sms < 1) c->sms = 148;
    c->chunk = 0;
    c->cfl_fused = 1; c->cfl_valid = 0;
    c->fv_shortcut = 1;
    c->err[0] = 0;
    // brick records of 4x4x4 cells x 15 fields; extents are rounded up to whole bricks (ppm_state_floats)
    c->nbx = (prm->nx + 3) / 4; c->nby = (prm->ny + 3) / 4; c->nbz = (prm->nz + 3) / 4;
    cudaError_t e;
#define CUC(call) do { e = (call); if (e != cudaSuccess) { set_err(nullptr, "%s failed: %s", #call, cudaGetErrorString(e)); ppm_destroy(c); return e == cudaErrorMemoryAllocation ? PPM_ENOMEM : PPM_ECUDA; } } while (0)
    CUC(cudaMalloc(&c->flag, sizeof(int)));
    CUC(cudaMemsetAsync(c->flag, 0, sizeof(int), c->stream));
    CUC(cudaMalloc(&c->cflmax, sizeof(unsigned int)));
    CUC(cudaMalloc(&c->partial, sizeof(double) * 6 * c->nblocks_red));
    CUC(cudaMalloc(&c->result, sizeof(double) * 6));
    ppm_static_scratch_prepare();     // set-up, this device current: the address of the static scratch array of ppm_reduce_conserved_static
    if (g.kind != PPM_GRAV_NONE) {
        std::vector<float4> t32(g.n);
        std::vector<double> t64(3 * (size_t)g.n);
        for (int k = 0; k < g.n; ++k) {
            t32[k] = make_float4(g.rho0[k], g.p0[k], g.g[k], 0.f);   // (rho0, p0) is an aligned pair for the packed lerp
            t64[3 * k] = g.g[k]; t64[3 * k + 1] = g.rho0[k]; t64[3 * k + 2] = g.p0[k];
        }
        // interval records for the sweeps: the differences are taken in fp32, as the kernel's own subtraction would
        std::vector<float4> tp(g.n);
        std::vector<float2> tg(g.n);
        auto ftz = [](float x) { return fabsf(x) < 1.17549435e-38f ? 0.0f : x; };
        for (int k = 0; k < g.n; ++k) {
            const int k1 = k + 1 < g.n ? k + 1 : k;
            tp[k] = make_float4(g.rho0[k], g.p0[k], ftz(g.rho0[k1] - g.rho0[k]), ftz(g.p0[k1] - g.p0[k]));
            tg[k] = make_float2(g.g[k], ftz(g.g[k1] - g.g[k]));
        }
        CUC(cudaMalloc(&c->tabp, sizeof(float4) * g.n));
        CUC(cudaMalloc(&c->tabg, sizeof(float2) * g.n));
        CUC(cudaMemcpy(c->tabp, tp.data(), sizeof(float4) * g.n, cudaMemcpyHostToDevice));
        CUC(cudaMemcpy(c->tabg, tg.data(), sizeof(float2) * g.n, cudaMemcpyHostToDevice));
        CUC(cudaMalloc(&c->tab, sizeof(float4) * g.n));
        CUC(cudaMalloc(&c->tab64, sizeof(double) * 3 * g.n));
        CUC(cudaMemcpy(c->tab, t32.data(), sizeof(float4) * g.n, cudaMemcpyHostToDevice));
        CUC(cudaMemcpy(c->tab64, t64.data(), sizeof(double) * 3 * g.n, cudaMemcpyHostToDevice));
    }
#undef CUC
    *out = c;
    return PPM_OK;
}

extern "C" void ppm_destroy(ppm_ctx* c) {
    if (!c) return;
    DevGuard guard(c);
    cudaFree(c->flag); cudaFree(c->cflmax); cudaFree(c->partial); cudaFree(c->result);
    cudaFree(c->tab); cudaFree(c->tabp); cudaFree(c->tabg); cudaFree(c->tab64); cudaFree(c->F3); cudaFree(c->R0c); cudaFree(c->P0c);
    free(c);
}

static int check_slab(ppm_ctx* c, const void* fields, int z0, int nzs, const char* who) {
    if (!c) { set_err(nullptr, "%s: ctx is NULL", who); return PPM_EINVAL; }
    if (!fields) { set_err(c, "%s: fields is NULL", who); return PPM_EINVAL; }
    if (z0 < 0 || nzs < 1 || z0 + nzs > c->prm.nz) { set_err(c, "%s: slab [%d,%d) outside [0,%d)", who, z0, z0 + nzs, c->prm.nz); return PPM_EINVAL; }
    return PPM_OK;
}

static int read_flag(ppm_ctx* c) {
    int f = 0;
    CU(cudaMemcpyAsync(&f, c->flag, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    if (f) { set_err(c, "state flag %d: %s", f, (f & 2) ? "NaN or non-positive density/pressure" : "density/pressure floor hit"); return PPM_ESTATE; }
    return PPM_OK;
}

extern "C" int ppm_set_state(ppm_ctx* c, const float* const fields[PPM_NFIELDS], int z0, int nzs, int src_is_device) {
    int rc = check_slab(c, fields, z0, nzs, "ppm_set_state");
    if (rc) return rc;
    DevGuard guard(c);
    for (int f = 0; f < PPM_NFIELDS; ++f) if (!fields[f]) { set_err(c, "ppm_set_state: fields[%d] is NULL", f); return PPM_EINVAL; }
    const long long plane = (long long)c->prm.nx * c->prm.ny;
    CU(ppm_make_whole(c));                  // (the scratch buffer may hold the hydro fields after PPB-only sweeps)
    float* st = c->buf[c->cur];
    float* scratch = c->buf[c->cur ^ 1];    // free between steps: stages the dense slab
    const long long tot = plane * nzs;
    const cudaMemcpyKind kind = src_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    for (int f = 0; f < PPM_NFIELDS; ++f)
        CU(cudaMemcpyAsync(scratch + f * tot, fields[f], sizeof(float) * tot, kind, c->stream));
    CU(ppm_launch_to_perturbation(c, scratch, st, z0, nzs));
    c->cfl_valid = 0;
    CU(cudaMemsetAsync(c->flag, 0, sizeof(int), c->stream));
    return PPM_OK;
}

extern "C" int ppm_get_state(ppm_ctx* c, float* const fields[PPM_NFIELDS], int z0, int nzs, int dst_is_device) {
    int rc = check_slab(c, fields, z0, nzs, "ppm_get_state");
    if (rc) return rc;
    DevGuard guard(c);
    for (int f = 0; f < PPM_NFIELDS; ++f) if (!fields[f]) { set_err(c, "ppm_get_state: fields[%d] is NULL", f); return PPM_EINVAL; }
    const long long plane = (long long)c->prm.nx * c->prm.ny, tot = plane * nzs;
    CU(ppm_make_whole(c));
    float* scratch = c->buf[c->cur ^ 1];    // free between steps
    CU(ppm_launch_to_full(c, c->buf[c->cur], scratch, z0, nzs));
    const cudaMemcpyKind kind = dst_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    for (int f = 0; f < PPM_NFIELDS; ++f)
        CU(cudaMemcpyAsync(fields[f], scratch + f * tot, sizeof(float) * tot, kind, c->stream));
    // host destinations: wait and report the state flag.  Device destinations are stream-ordered like everything else
    // the library enqueues, so the call stays asynchronous (slab pipelines: PPM.step_host_pipelined in binding.py)
    return dst_is_device ? PPM_OK : read_flag(c);
}

// PPM_BC_HALO faces: the sweep along `axis` reads the neighbour's brick layer — it must have been handed over, and only the
// bulk-staged sweeps of the plain scheme know how to
static int halo_ready(ppm_ctx* c, int axis, const char* who) {
    const bool lo = c->prm.bc[2 * axis] == PPM_BC_HALO, hi = c->prm.bc[2 * axis + 1] == PPM_BC_HALO;
    if (!lo && !hi) return PPM_OK;
    if ((lo && !c->halo[axis][0]) || (hi && !c->halo[axis][1])) { set_err(c, "%s: axis %d has a PPM_BC_HALO face without a halo layer (ppm_set_halo)", who, axis); return PPM_EINVAL; }
    if (!ppm_axis_is_bulk(c, axis)) { set_err(c, "%s: PPM_BC_HALO faces need the bulk-staged path (PPM_OPT_IO_PATH = 0)", who); return PPM_EINVAL; }
    if (c->flat3d || c->twof || c->sphere) { set_err(c, "%s: PPM_BC_HALO faces are not combined with PPM_OPT_FLATTEN3D, the two-fluid EOS or the sphere", who); return PPM_EINVAL; }
    return PPM_OK;
}
static bool has_halo(const ppm_ctx* c) {
    for (int k = 0; k < 6; ++k) if (c->prm.bc[k] == PPM_BC_HALO) return true;
    return false;
}

static int sweep_impl(ppm_ctx* c, double dt, int axis, bool with_cfl, const char* who) {
    if (!c) { set_err(nullptr, "%s: ctx is NULL", who); return PPM_EINVAL; }
    DevGuard guard(c);
    if (!(dt > 0.0) || !isfinite(dt) || axis < 0 || axis > 2) { set_err(c, "%s: need finite dt > 0 and axis in 0..2", who); return PPM_EINVAL; }
    int rc = halo_ready(c, axis, who);
    if (rc) return rc;
    if (c->flat3d) CU(ppm_launch_flatten3d(c));     // the detector field of the state this sweep starts from
    c->cfl_valid = 0;
    const bool fuse = with_cfl && c->cfl_fused && ppm_axis_is_bulk(c, axis);
    if (fuse) CU(cudaMemsetAsync(c->cflmax, 0, sizeof(unsigned int), c->stream));
    CU(ppm_launch_sweep(c, axis, dt, false, fuse));
    if (fuse) c->cfl_valid = 1;
    return PPM_OK;
}

extern "C" int ppm_sweep(ppm_ctx* c, double dt, int axis) { return sweep_impl(c, dt, axis, false, "ppm_sweep"); }
extern "C" int ppm_sweep_cfl(ppm_ctx* c, double dt, int axis) { return sweep_impl(c, dt, axis, true, "ppm_sweep_cfl"); }

extern "C" int ppm_step(ppm_ctx* c, double dt, int sweep_order) {
    if (!c) { set_err(nullptr, "ppm_step: ctx is NULL"); return PPM_EINVAL; }
    DevGuard guard(c);
    if (!(dt > 0.0) || !isfinite(dt) || sweep_order < 0 || sweep_order > 5) { set_err(c, "ppm_step: need finite dt > 0 and sweep_order in 0..5"); return PPM_EINVAL; }
    if (has_halo(c)) { set_err(c, "ppm_step: a grid with PPM_BC_HALO faces advances sweep by sweep (ppm_sweep / ppm_sweep_cfl), the halo layers exchanged before each"); return PPM_EINVAL; }
    if (c->flat3d) CU(ppm_launch_flatten3d(c));     // once per step, on the step's starting state
    c->cfl_valid = 0;
    for (int s = 0; s < 3; ++s) {
        const int axis = ORDERS[sweep_order][s];
        // S10 fused: the step's last sweep also leaves max_d |u_d| + c of the NEW state in cflmax (bulk-staged sweeps only)
        const bool fuse = s == 2 && c->cfl_fused && ppm_axis_is_bulk(c, axis);
        if (fuse) CU(cudaMemsetAsync(c->cflmax, 0, sizeof(unsigned int), c->stream));
        CU(ppm_launch_sweep(c, axis, dt, false, fuse));
        if (fuse) c->cfl_valid = 1;
    }
    return PPM_OK;
}

extern "C" int ppm_advect(ppm_ctx* c, double dt, int sweep_order) {
    if (!c) { set_err(nullptr, "ppm_advect: ctx is NULL"); return PPM_EINVAL; }
    DevGuard guard(c);
    if (!(dt > 0.0) || !isfinite(dt) || sweep_order < 0 || sweep_order > 5) { set_err(c, "ppm_advect: need finite dt > 0 and sweep_order in 0..5"); return PPM_EINVAL; }
    if (c->sphere) { set_err(c, "ppm_advect: the PPB-only mode has no confining sphere"); return PPM_EINVAL; }
    if (has_halo(c)) { set_err(c, "ppm_advect: not on a grid with PPM_BC_HALO faces"); return PPM_EINVAL; }
    if (c->twof) c->cfl_valid = 0;      // two-fluid EOS: the sound speed depends on FV, which these sweeps move
    for (int s = 0; s < 3; ++s) CU(ppm_launch_sweep(c, ORDERS[sweep_order][s], dt, true));
    return PPM_OK;
}

extern "C" int ppm_cfl_dt(ppm_ctx* c, double cfl, double* dt_out) {
    if (!c) { set_err(nullptr, "ppm_cfl_dt: ctx is NULL"); return PPM_EINVAL; }
    DevGuard guard(c);
    if (!dt_out || !(cfl > 0.0)) { set_err(c, "ppm_cfl_dt: need cfl > 0 and dt_out"); return PPM_EINVAL; }
    if (!c->cfl_valid) CU(ppm_launch_cfl(c));       // else: the last ppm_step already reduced the maximum of this state
    unsigned int enc = 0;
    CU(cudaMemcpyAsync(&enc, c->cflmax, sizeof(enc), cudaMemcpyDeviceToHost, c->stream));
    int rc = read_flag(c);
    if (rc) return rc;
    float vmax;
    memcpy(&vmax, &enc, sizeof(float));
    if (!(vmax > 0.f)) { c->cfl_valid = 0; set_err(c, "ppm_cfl_dt: max signal speed is not positive or not a number"); return PPM_ESTATE; }
    c->cfl_valid = 1;                               // cflmax now holds the maximum of the current state
    *dt_out = cfl * c->prm.dx / (double)vmax;
    return PPM_OK;
}

extern "C" int ppm_reduce_conserved(ppm_ctx* c, double out[6]) {
    if (!c) { set_err(nullptr, "ppm_reduce_conserved: ctx is NULL"); return PPM_EINVAL; }
    DevGuard guard(c);
    if (!out) { set_err(c, "ppm_reduce_conserved: out is NULL"); return PPM_EINVAL; }
    CU(ppm_launch_conserved(c));
    CU(cudaMemcpyAsync(out, c->result, sizeof(double) * 6, cudaMemcpyDeviceToHost, c->stream));
    return read_flag(c);
}

extern "C" int ppm_reduce_conserved_static(ppm_ctx* c, int nblocks, double* dev_out) {
    if (!c) { set_err(nullptr, "ppm_reduce_conserved_static: ctx is NULL"); return PPM_EINVAL; }
    if (!dev_out) { set_err(c, "ppm_reduce_conserved_static: dev_out is NULL"); return PPM_EINVAL; }
    if (nblocks < 0) { set_err(c, "ppm_reduce_conserved_static: nblocks must be >= 0"); return PPM_EINVAL; }
    const int nb = nblocks ? nblocks : c->nblocks_red;
    if (nb > PPM_STATIC_RED_BLOCKS) {
        set_err(c, "ppm_reduce_conserved_static: %d first-pass blocks need %zu bytes of partial sums; the static scratch array holds %d blocks (%zu bytes)",
                nb, sizeof(double) * 6 * (size_t)nb, PPM_STATIC_RED_BLOCKS, sizeof(double) * 6 * (size_t)PPM_STATIC_RED_BLOCKS);
        return PPM_EINVAL;
    }
    DevGuard guard(c);
    CU(ppm_launch_conserved_static(c, nb, dev_out));
    return PPM_OK;
}

extern "C" int ppm_sync(ppm_ctx* c) {
    if (!c) { set_err(nullptr, "ppm_sync: ctx is NULL"); return PPM_EINVAL; }
    DevGuard guard(c);
    return read_flag(c);
}

extern "C" int ppm_set_chunk(ppm_ctx* c, int chunk_cells) {
    if (!c) { set_err(nullptr, "ppm_set_chunk: ctx is NULL"); return PPM_EINVAL; }
    if (chunk_cells < 0) { set_err(c, "ppm_set_chunk: chunk_cells must be >= 0"); return PPM_EINVAL; }
    c->chunk = chunk_cells;
    return PPM_OK;
}

extern "C" int ppm_set_option(ppm_ctx* c, int option, int value) {
    if (!c) { set_err(nullptr, "ppm_set_option: ctx is NULL"); return PPM_EINVAL; }
    DevGuard guard(c);
    if (c->sphere && ((option == PPM_OPT_IO_PATH && value == 1) || (option == PPM_OPT_FLATTEN3D && value == 1))) {
        set_err(c, "ppm_set_option: not together with the confining sphere"); return PPM_EINVAL;
    }
    if (c->twof && option == PPM_OPT_FLATTEN3D && value == 1) { set_err(c, "ppm_set_option: PPM_OPT_FLATTEN3D not together with the two-fluid equation of state"); return PPM_EINVAL; }
    if (option == PPM_OPT_IO_PATH && (value == 0 || value == 1)) { c->io_path = value; return PPM_OK; }
    if (option == PPM_OPT_STATE_FORM && (value == 0 || value == 1)) { c->pert_io = value; return PPM_OK; }
    if (option == PPM_OPT_FV_SHORTCUT && (value == 0 || value == 1)) { c->fv_shortcut = value; return PPM_OK; }
    if (option == PPM_OPT_CFL_FUSED && (value == 0 || value == 1)) { c->cfl_fused = value; c->cfl_valid = 0; return PPM_OK; }
    if (option == PPM_OPT_FLATTEN3D && (value == 0 || value == 1)) {
        if (value && !c->F3) {
            const size_t n = (size_t)c->nbx * c->nby * c->nbz * 64;
            cudaError_t e = cudaMalloc(&c->F3, n * sizeof(float));
            if (e != cudaSuccess) { c->F3 = nullptr; cudaGetLastError(); set_err(c, "ppm_set_option: cannot allocate the %zu-byte detector field", n * sizeof(float)); return PPM_ENOMEM; }
        }
        if (value && c->prm.grav.kind == PPM_GRAV_RADIAL && !c->P0c) {
            // the detector kernel stages 2.5 points per cell: with a radial profile their base state comes from two per-cell
            // arrays (8 more bytes per cell, filled once) instead of a table lookup each
            const size_t n = (size_t)c->nbx * c->nby * c->nbz * 64;
            if (cudaMalloc(&c->R0c, n * sizeof(float)) != cudaSuccess || cudaMalloc(&c->P0c, n * sizeof(float)) != cudaSuccess) {
                cudaGetLastError(); cudaFree(c->R0c); c->R0c = c->P0c = nullptr;      // fall back to the lookups
            } else CU(ppm_launch_base_fill(c));
        }
        c->flat3d = value;
        return PPM_OK;
    }
    set_err(c, "ppm_set_option: unknown option %d or value %d", option, value);
    return PPM_EINVAL;
}

extern "C" int ppm_set_sphere(ppm_ctx* c, double radius, const double center[3]) {
    if (!c) { set_err(nullptr, "ppm_set_sphere: ctx is NULL"); return PPM_EINVAL; }
    if (!(radius > 0.0)) { c->sphere = 0; c->cfl_valid = 0; return PPM_OK; }
    if (!center) { set_err(c, "ppm_set_sphere: center is NULL"); return PPM_EINVAL; }
    for (int k = 0; k < 6; ++k)
        if (c->prm.bc[k] != PPM_BC_REFLECT) { set_err(c, "ppm_set_sphere: the confining sphere needs reflecting walls on all six faces"); return PPM_EINVAL; }
    if ((c->prm.nx | c->prm.ny | c->prm.nz) & 3) { set_err(c, "ppm_set_sphere: grid extents must be multiples of 4 (the sphere runs on the bulk-staged sweeps)"); return PPM_EINVAL; }
    if (c->prm.grav.kind == PPM_GRAV_CONST_Z) { set_err(c, "ppm_set_sphere: not with plane-parallel (CONST_Z) gravity"); return PPM_EINVAL; }
    if (c->flat3d) { set_err(c, "ppm_set_sphere: not together with PPM_OPT_FLATTEN3D"); return PPM_EINVAL; }
    if (c->org[0] | c->org[1] | c->org[2]) { set_err(c, "ppm_set_sphere: not on a sub-domain (ppm_set_origin)"); return PPM_EINVAL; }
    if (c->twof) { set_err(c, "ppm_set_sphere: not together with the two-fluid equation of state"); return PPM_EINVAL; }
    if (c->io_path != 0) { set_err(c, "ppm_set_sphere: not together with PPM_OPT_IO_PATH = 1"); return PPM_EINVAL; }
    c->sphere = 1; c->sph_r = radius;
    for (int d = 0; d < 3; ++d) c->sph_c[d] = center[d];
    c->cfl_valid = 0;
    return PPM_OK;
}

// ---- NEXT-4: brick decomposition -----------------------------------------------------
extern "C" size_t ppm_halo_floats(int nx, int ny, int nz, int axis) {
    if (nx < 1 || ny < 1 || nz < 1 || axis < 0 || axis > 2) return 0;
    const size_t nb[3] = {(size_t)(nx + 3) / 4, (size_t)(ny + 3) / 4, (size_t)(nz + 3) / 4};
    return (size_t)PPM_BRICK_FLOATS * nb[(axis + 1) % 3] * nb[(axis + 2) % 3];
}

static int halo_args(ppm_ctx* c, int axis, int side, const void* p, const char* who) {
    if (!c) { set_err(nullptr, "%s: ctx is NULL", who); return PPM_EINVAL; }
    if (axis < 0 || axis > 2 || side < 0 || side > 1 || !p) { set_err(c, "%s: need axis in 0..2, side in 0..1 and a device buffer", who); return PPM_EINVAL; }
    if (((uintptr_t)p & 15) != 0) { set_err(c, "%s: the buffer must be 16-byte aligned", who); return PPM_EINVAL; }
    return PPM_OK;
}

extern "C" int ppm_pack_halo(ppm_ctx* c, int axis, int side, float* dev_dst) {
    int rc = halo_args(c, axis, side, dev_dst, "ppm_pack_halo");
    if (rc) return rc;
    DevGuard guard(c);
    CU(ppm_launch_pack_halo(c, axis, side, dev_dst));
    return PPM_OK;
}

extern "C" int ppm_set_halo(ppm_ctx* c, int axis, int side, const float* dev_layer) {
    int rc = halo_args(c, axis, side, dev_layer, "ppm_set_halo");
    if (rc) return rc;
    if (c->prm.bc[2 * axis + side] != PPM_BC_HALO) { set_err(c, "ppm_set_halo: face %d of axis %d is not PPM_BC_HALO", side, axis); return PPM_EINVAL; }
    c->halo[axis][side] = dev_layer;
    return PPM_OK;
}

extern "C" int ppm_set_origin(ppm_ctx* c, const int org[3]) {
    if (!c) { set_err(nullptr, "ppm_set_origin: ctx is NULL"); return PPM_EINVAL; }
    if (!org || org[0] < 0 || org[1] < 0 || org[2] < 0) { set_err(c, "ppm_set_origin: need three non-negative cell indices"); return PPM_EINVAL; }
    if (c->prm.grav.kind == PPM_GRAV_CONST_Z && org[2] != 0) { set_err(c, "ppm_set_origin: a grid with plane-parallel (CONST_Z) gravity cannot be cut along z"); return PPM_EINVAL; }
    if (c->sphere) { set_err(c, "ppm_set_origin: not together with the confining sphere"); return PPM_EINVAL; }
    for (int d = 0; d < 3; ++d) c->org[d] = org[d];
    c->cfl_valid = 0;
    return PPM_OK;
}

extern "C" int ppm_set_two_fluid(ppm_ctx* c, double gamma_tracked, double gamma_rest) {
    if (!c) { set_err(nullptr, "ppm_set_two_fluid: ctx is NULL"); return PPM_EINVAL; }
    if (!(gamma_tracked > 0.0)) { c->twof = 0; c->cfl_valid = 0; return PPM_OK; }
    if (!(gamma_tracked > 1.0) || !(gamma_rest > 1.0) || !isfinite(gamma_tracked) || !isfinite(gamma_rest)) { set_err(c, "ppm_set_two_fluid: both adiabatic indices must be finite and > 1"); return PPM_EINVAL; }
    if (c->sphere) { set_err(c, "ppm_set_two_fluid: not together with the confining sphere"); return PPM_EINVAL; }
    if (c->flat3d) { set_err(c, "ppm_set_two_fluid: not together with PPM_OPT_FLATTEN3D"); return PPM_EINVAL; }
    c->twof = 1; c->gam_tracked = gamma_tracked; c->gam_rest = gamma_rest;
    c->cfl_valid = 0;
    return PPM_OK;
}

extern "C" int ppm_spin_up(ppm_ctx* c, double domega) {
    if (!c) { set_err(nullptr, "ppm_spin_up: ctx is NULL"); return PPM_EINVAL; }
    DevGuard guard(c);
    if (!isfinite(domega)) { set_err(c, "ppm_spin_up: domega is not finite"); return PPM_EINVAL; }
    c->cfl_valid = 0;
    CU(ppm_launch_spin_up(c, domega));
    return PPM_OK;
}

extern "C" int ppm_axis_path(const ppm_ctx* c, int axis) { return (c && axis >= 0 && axis <= 2 && ppm_axis_is_bulk(c, axis)) ? 1 : 0; }

extern "C" int ppm_plan_tail_chunk(int tail_tiles, int resident_ctas, int n) {
    if (tail_tiles < 1 || resident_ctas < 1 || n < 1) return 0;
    return ppm_tail_chunk(tail_tiles, resident_ctas, n);
}

extern "C" long long ppm_launch_count(const ppm_ctx* c) { return c ? c->launches : 0; }

extern "C" int ppm_measure_fp32_peak(ppm_ctx* c, double* tflops_out) {
    if (!c) { set_err(nullptr, "ppm_measure_fp32_peak: ctx is NULL"); return PPM_EINVAL; }
    DevGuard guard(c);
    if (!tflops_out) { set_err(c, "ppm_measure_fp32_peak: tflops_out is NULL"); return PPM_EINVAL; }
    CU(ppm_run_fma_peak(c, tflops_out));
    return PPM_OK;
}
