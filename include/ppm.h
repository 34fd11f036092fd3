/*
 * ppm.h — C ABI of the B200-native PPM+PPB timestep library (libppm_b200.so).
 *
 * One hot path of arxiv/paper_1810_13416 (Woodward et al.): the directionally split 3-D PPM
 * gas-dynamics timestep fused with PPB ten-moment advection of the fractional volume FV
 * (BASELINE.json north_star, which also names this call
 * list).  The numerical definition of every step is SURVEY.md section 8(c) (H0-H9, P1-P4, C1-C7),
 * restated in DESIGN.md.  All arithmetic on the device is fp32, one GPU, no CPU
 * fallback: every entry point fails with PPM_ECUDA if no sm_100 device / kernel image is usable.
 *
 * Conventions
 *  - plain C types only; every call returns a status code, never throws or aborts.
 *  - NULL / size / non-paired-periodic / dt <= 0 / unknown order -> PPM_EINVAL, no side effects.
 *  - CUDA failures -> PPM_ECUDA; text kept for ppm_last_error().
 *  - ppm_step only enqueues kernels on the context's stream; a sticky device flag (NaN, or a
 *    density/pressure floor was hit) is reported as PPM_ESTATE by the next synchronising call
 *    (ppm_cfl_dt, ppm_reduce_conserved, ppm_get_state, ppm_sync).
 *  - pointers marked [host] / [device] say where the memory lives; pointers passed in arrays
 *    (fields[]) are borrowed for the duration of the call only.
 *
 * State at the boundary (ppm_set_state / ppm_get_state): 15 fp32 fields per cell, each a dense [nz][ny][nx]
 * array, x fastest.  Inside the two borrowed buffers the library keeps them as brick records: 4x4x4 cells x
 * 15 fields per 3840-byte brick, extents rounded up to whole bricks.
 *   0 rho  1 ux  2 uy  3 uz  4 p   5..14 = m000 m100 m010 m001 m200 m020 m002 m110 m101 m011
 * where m_abc are the coefficients of FV in the cell-local Legendre basis P0=1, P1=s, P2=s^2-1/12
 * on [-1/2,1/2]^3 (m000 = cell mean; "cell average and its 9 lowest-order moments").
 * Internally rho and p are stored as perturbations to the hydrostatic base state.
 */
#ifndef PPM_B200_H
#define PPM_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ppm_ctx ppm_ctx; /* opaque; owns only small device scratch (tables, reduction cells) */

enum { PPM_OK = 0, PPM_EINVAL = 1, PPM_ENOMEM = 2, PPM_ECUDA = 3, PPM_ESTATE = 4 };
enum { PPM_BC_PERIODIC = 0, PPM_BC_REFLECT = 1, PPM_BC_HALO = 2 }; /* per face: xlo,xhi,ylo,yhi,zlo,zhi; periodic must pair up;
                                                     HALO: the cells beyond the face belong to a neighbouring sub-domain (see ppm_set_halo) */
enum { PPM_GRAV_NONE = 0, PPM_GRAV_CONST_Z = 1, PPM_GRAV_RADIAL = 2 };
#define PPM_NFIELDS 15
#define PPM_NGHOST 4 /* stencil reach per sweep */

/* "Gravity profile": the acceleration AND the hydrostatic base state it balances.
 * Node k sits at s = s0 + k*ds.  Point values are linear interpolations between nodes.
 *  CONST_Z: s = z, acceleration g(z) along +z.  The table MUST have n = 2*(nz+8)+1 nodes with
 *           s0 = -4*dx, ds = dx/2, so that every cell centre and face is a node (else PPM_EINVAL).
 *  RADIAL : s = r = |X - center|, acceleration g(r) * (X - center)/r.
 * g, rho0, p0: [host] arrays of n floats, copied by ppm_create (fp32 on purpose: the oracle and
 * the GPU must see bit-identical nodes). */
typedef struct {
    int kind; /* PPM_GRAV_* */
    int n;
    double s0, ds;
    double center[3];
    const float *g, *rho0, *p0;
} ppm_gravity;

typedef struct {
    size_t struct_size; /* = sizeof(ppm_params); checked */
    int nx, ny, nz;     /* cells; each >= 1 */
    double dx;          /* cubic cells; cell (i,j,k) is centred at ((i+.5)dx, (j+.5)dx, (k+.5)dx) */
    double gamma;       /* ideal-gas adiabatic index, > 1 */
    double rho_floor, p_floor; /* p_floor > 0; rho_floor > 1e-30 (the PPB remap divides by the new mass of a cell) */
    ppm_gravity grav;
    int bc[6];
    void *stream; /* cudaStream_t the library enqueues on (0 = default stream) */
} ppm_params;

/* Number of floats each of the two state buffers must hold for an nx x ny x nz grid:
 * 15 * 64 * ceil(nx/4) * ceil(ny/4) * ceil(nz/4)  (= 15*nx*ny*nz when the extents are multiples of 4).
 * Returns 0 for a non-positive extent.  Pure host arithmetic; needs no device. */
size_t ppm_state_floats(int nx, int ny, int nz);

/* Creates a context for one uniform Cartesian grid with its boundary types (L69: walls; periodic for
 * the test problems), equation of state and gravity profile (L35).  dev_buf_a, dev_buf_b: [device] two caller-owned buffers of
 * ppm_state_floats(nx,ny,nz) floats each, 128-byte aligned (e.g. torch tensors).  The library BORROWS them for the
 * life of the context: the state lives in one, the other is sweep scratch, and they ping-pong.  It
 * never frees them.  Contents are undefined until ppm_set_state has covered every z-slab.  Every later call runs on
 * the device that owns these buffers, whatever device is current in the calling thread (and restores the caller's). */
int ppm_create(ppm_ctx **out, const ppm_params *prm, float *dev_buf_a, float *dev_buf_b);

/* Loads the full state (rho, ux, uy, uz, p, m000..m011) for z-planes [z0, z0+nz_slab).
 * fields[f]: [host] array of 15 pointers, each to a dense [nz_slab][ny][nx] float array that lives on
 * the host (src_is_device = 0) or on the device (src_is_device = 1).  Converts rho, p to
 * perturbation form (rho' = rho - rho0 at the cell centre, formed in fp64, rounded once to fp32;
 * SURVEY 8(c) C1).  Asynchronous w.r.t. the host only if the sources are device or pinned memory. */
int ppm_set_state(ppm_ctx *ctx, const float *const fields[PPM_NFIELDS], int z0, int nz_slab, int src_is_device);

/* Inverse of ppm_set_state (full rho = rho0 + rho', p = p0 + p').  Host destinations: synchronises the
 * stream before returning and reports the sticky state flag.  Device destinations: only enqueues work on the context's
 * stream (the arrays are valid in stream order; the flag is reported by the next synchronising call). */
int ppm_get_state(ppm_ctx *ctx, float *const fields[PPM_NFIELDS], int z0, int nz_slab, int dst_is_device);

/* One timestep = three 1-D sweeps (ghost fill, PPM hydro, PPB remap fused) with the same dt (PAPER.md L87
 * "directionally split"; L27, L33, L35, L37, L51, L120).
 * sweep_order 0..5 = xyz, xzy, yxz, yzx, zxy, zyx.  Only enqueues work (3 kernel launches). */
int ppm_step(ppm_ctx *ctx, double dt, int sweep_order);

/* One sweep along axis d (0,1,2) — the unit ppm_step is made of; exposed for per-sweep parity tests. */
int ppm_sweep(ppm_ctx *ctx, double dt, int axis);

/* PPB-only step (Fig. 3: the slotted disc in solid-body rotation, "linear
 * advection"): three PPB-only sweeps in the given order with one dt.  The hydro fields are held fixed; FV (its ten
 * coefficients) is advected by the stored velocity field with the PPB remap P2-P4 of the full step.  Reading R22
 * (DESIGN.md): the gas is taken as uniform and the velocity at a face is the mean of the two cell values, so the
 * mode is meant for velocity fields whose component along an axis does not vary along that axis (rotation, shear,
 * translation), for which every sweep is volume preserving.  Only enqueues work (3 kernel launches).  On a grid whose three
 * extents are multiples of 4 these sweeps move the PPB part of the records only; the next call of any other kind then first
 * copies the hydro fields to where the coefficients are (one more launch, after an odd number of PPB-only sweeps). */
int ppm_advect(ppm_ctx *ctx, double dt, int sweep_order);

/* dt = cfl*dx / max over cells of max_d(|u_d|) + c, c from the full rho, p (the scheme is explicit, PAPER.md L55;
 * SURVEY 8(c) C6).  The maximum is already on the device when the state was last changed by ppm_step (it is reduced
 * inside the step's last sweep, see PPM_OPT_CFL_FUSED); otherwise one reduction kernel runs first.  Synchronises the stream.  dt_out: [host].  PPM_ESTATE if a cell has non-positive rho or p. */
int ppm_cfl_dt(ppm_ctx *ctx, double cfl, double *dt_out);

/* (BASELINE.json north_star: conservation to round-off on periodic boxes)
 * out[6] [host] = mass, momentum x, y, z, total energy, tracked mass (sum rho*m000), each * dx^3;
 * fp64 accumulation in a fixed order (deterministic).  Synchronises the stream. */
int ppm_reduce_conserved(ppm_ctx *ctx, double out[6]);

/* The same six sums for callers that cannot allocate device memory (code under CUDA graph capture, serving loops,
 * harnesses that forbid cudaMalloc): the per-block partial sums of the first pass live in a file-scope device array of
 * the library instead of memory ppm_create allocated.  The call allocates and frees nothing, does not synchronise and
 * does not read the state flag: it enqueues two kernels on the context's stream.
 *   nblocks : blocks of the first pass, 1..PPM_STATIC_RED_BLOCKS; 0 = the count ppm_reduce_conserved uses (592) — the
 *             sums are then bit for bit those of ppm_reduce_conserved; another count changes the order of the fp64
 *             additions (differences at the 1e-15 level).  More than PPM_STATIC_RED_BLOCKS -> PPM_EINVAL, nothing runs.
 *   dev_out : [device] 6 doubles, written by the second kernel (valid once the stream has reached it).
 * The array (6 * PPM_STATIC_RED_BLOCKS doubles = 48 KB) is held by every GPU that loads the library until the process
 * exits and is SHARED by every call on that GPU, whatever the context: calls that may overlap on the GPU (different
 * streams) race on it — order them.  It keeps the last call's contents; nothing in it has to start at zero (every slot
 * that is read was written by the same call).  ppm_create looks the array's address up for its device (cudaGetSymbolAddress; no
 * allocation by this library), so the call itself only launches. */
#define PPM_STATIC_RED_BLOCKS 1024
int ppm_reduce_conserved_static(ppm_ctx *ctx, int nblocks, double *dev_out);

/* Waits for the stream and reports the sticky state flag (PPM_OK / PPM_ESTATE / PPM_ECUDA). */
int ppm_sync(ppm_ctx *ctx);

/* Tuning knob for benchmarks: cells marched per thread along the sweep axis before the pencil is
 * split into another chunk (0 = library default).  Results do not depend on it. */
int ppm_set_chunk(ppm_ctx *ctx, int chunk_cells);

/* Options.  Tuning option (results do not depend on it):
 *  PPM_OPT_IO_PATH : 0 = automatic: a sweep along an axis whose extent is a multiple of 4 stages whole brick
 *                    records through shared memory with bulk copies (cp.async.bulk), any other axis uses the
 *                    direct global-memory path; 1 = direct path for every axis.
 *  PPM_OPT_CFL_FUSED : 1 (default) = the last sweep of ppm_step also reduces max over cells of max_d |u_d| + c of the
 *                    state it writes (warp max + one atomicMax per warp), so that the next ppm_cfl_dt
 *                    only reads 4 bytes back; 0 = ppm_cfl_dt always runs its own reduction pass over the state.  The
 *                    two agree to fp32 rounding of c (bit for bit without a base state).  Whatever else changes the
 *                    state (ppm_set_state, ppm_sweep, a sweep on the direct path) makes ppm_cfl_dt fall back to the pass.
 *  PPM_OPT_FV_SHORTCUT : 1 (default) = where FV is uniform under a whole warp — the three cells the PPB remap of a cell draws from have
 *                    the same mean and no higher coefficient, in all 32 pencils of the warp — the remap is skipped: it would return
 *                    that mean and nine zeros whatever mass moves (the tracked gas differs from its surroundings
 *                    only near the boundary of the convection zone).  The values are the same (a denormal is a zero either way:
 *                    the arithmetic is flush-to-zero); 0 = always run the remap (bench.py reports both timings).
 *  PPM_OPT_STATE_FORM : 0 (default) = ppm_set_state / ppm_get_state exchange the FULL rho and p; 1 = they exchange the
 *                    perturbations rho' = rho - rho0, p' = p - p0 exactly as the library stores and evolves them (PAPER.md L35:
 *                    "perturbations to a base, hydrostatic state"), so that no digit of a small perturbation is lost to the
 *                    fp32 rounding of rho0 + rho' at the boundary (the parity tests compare the perturbation fields this way).
 *
 * Option that changes the numerical scheme ("a fully 3-D treatment of the
 * shock dissipation"; reading R5b in DESIGN.md):
 *  PPM_OPT_FLATTEN3D : 0 (default) = the flattening coefficient of a sweep comes from the 1-D shock detector
 *                    along that sweep (H4); 1 = it comes from a 3-D detector field F~ = max over the three
 *                    directions of the H4 coefficient, evaluated once per ppm_step on the step's starting state
 *                    (ppm_sweep: on the state that sweep starts from) and spread over i-1..i+1 along the sweep.
 *                    Setting it allocates one library-owned device array of ppm_state_floats()/15 floats
 *                    (PPM_ENOMEM if that fails) and adds one light kernel launch per step. */
enum { PPM_OPT_IO_PATH = 2, PPM_OPT_FLATTEN3D = 3, PPM_OPT_CFL_FUSED = 4, PPM_OPT_STATE_FORM = 5, PPM_OPT_FV_SHORTCUT = 6 };
int ppm_set_option(ppm_ctx *ctx, int option, int value);
/* Confining sphere ("our star is enclosed in an impenetrable and immovable sphere that
 * is inscribed in the cubical domain of our uniform Cartesian grid ... a very simple boundary condition at the sphere";
 * reading R23 in DESIGN.md).  A cell whose centre lies outside the sphere of this radius about center[3] [host] (physical
 * units; the paper's case: radius = half the box, centre = box centre) is SOLID: it is never changed and never read by
 * the flow.  In every sweep each grid pencil is cut down to its fluid segment, whose two ends are reflecting walls (the
 * ghost cells are the mirror images along the pencil, C3), so no mass crosses the sphere.  ppm_cfl_dt and
 * ppm_reduce_conserved then run over the fluid cells only.  radius <= 0 switches the sphere off.
 * PPM_EINVAL unless all six faces are PPM_BC_REFLECT, the extents are multiples of 4, gravity is NONE or RADIAL, and
 * neither PPM_OPT_FLATTEN3D nor PPM_OPT_IO_PATH = 1 is set.  Host-side state only (no launch). */
int ppm_set_sphere(ppm_ctx *ctx, double radius, const double center[3]);

/* ---- Brick decomposition over several GPUs ("each MPI rank ... a grid brick ... must
 * exchange ... a halo one briquette thick").  One context per sub-domain (one process per GPU); a face shared with a neighbouring
 * sub-domain has the boundary type PPM_BC_HALO.  A 1-D sweep along an axis only ever needs ghost cells ALONG that axis, 4 deep = one
 * brick layer, so before each sweep a sub-domain packs its first and last brick layer along the sweep axis (ppm_pack_halo), the
 * layers travel to the two neighbours (NCCL send/recv or a peer copy — the caller's plumbing), and the sweep reads the received
 * layer as its ghost brick (ppm_set_halo).  No edge or corner data is ever exchanged and no ghost cell is updated redundantly.
 * The results are bit for bit those of the undivided grid (ppm_set_origin makes the base state be evaluated at the global
 * positions).  A grid with a HALO face advances with ppm_sweep / ppm_sweep_cfl (ppm_step returns PPM_EINVAL: an exchange is due
 * between its sweeps); the extent along an axis with a HALO face must be a multiple of 4 and >= 8.  Not combined with
 * PPM_OPT_FLATTEN3D, PPM_OPT_IO_PATH = 1, ppm_set_sphere, ppm_set_two_fluid or ppm_advect. */

/* Floats in one brick layer normal to `axis` of an nx x ny x nz grid (= the size of a halo buffer): 960 * ceil(n_a/4) * ceil(n_b/4)
 * with a, b the two other axes.  0 for bad arguments.  Pure host arithmetic. */
size_t ppm_halo_floats(int nx, int ny, int nz, int axis);

/* Gathers the first (side = 0: cells 0..3) or last (side = 1) brick layer along `axis` of the current state into dev_dst [device,
 * ppm_halo_floats() floats, 16-byte aligned]: whole brick records, ordered [bricks along b][bricks along a] with a < b the two other
 * axes.  Only enqueues work (1 copy kernel). */
int ppm_pack_halo(ppm_ctx *ctx, int axis, int side, float *dev_dst);

/* Registers the brick layer of the neighbour beyond the low (side = 0) or high (side = 1) face of `axis` — a buffer filled by the
 * NEIGHBOUR's ppm_pack_halo(axis, 1 - side) — as the ghost brick of the sweeps along `axis`.  dev_layer: [device], borrowed until
 * replaced or the context is destroyed; its contents are read by every later ppm_sweep along that axis (stream-ordered: refill it
 * before each).  PPM_EINVAL unless that face is PPM_BC_HALO.  Host-side state only. */
int ppm_set_halo(ppm_ctx *ctx, int axis, int side, const float *dev_layer);

/* Global cell index of this grid's cell (0,0,0) [host, 3 ints >= 0]: positions (the radial distance of the gravity profile, the
 * spin-up axis) are then taken at the global cell centres, with the arithmetic of the undivided grid.  Host-side state only. */
int ppm_set_origin(ppm_ctx *ctx, const int org[3]);

/* ppm_sweep that also reduces the CFL maximum of the state it writes (S10 fused, as the last sweep of ppm_step does), so that
 * the next ppm_cfl_dt reads 4 bytes back: the last sweep of a step driven sweep by sweep. */
int ppm_sweep_cfl(ppm_ctx *ctx, double dt, int axis);

/* Two-fluid equation of state ("multifluid", L87 "fv ... gives the fraction of the volume of a
 * cell that is occupied by a special, tracked multifluid constituent"; the paper prints no EOS: reading R25 in DESIGN.md).  The
 * tracked fluid (volume fraction f = FV, the PPB cell mean m000 clamped to [0,1]) has adiabatic index gamma_tracked, the rest
 * gamma_rest; both are ideal gases in pressure equilibrium inside a cell, so the internal energy per volume is e = p beta(f) with
 * beta(f) = f/(gamma_tracked-1) + (1-f)/(gamma_rest-1), i.e. the cell is an ideal gas with Gamma(f) = 1 + 1/beta(f).  Each side of
 * a face takes Gamma of its own cell, the enthalpy flux carries beta of the gas the PPB remap moves through the face, and the new
 * pressure is recovered from the conserved energy with beta of the new f; ppm_cfl_dt and the energy of ppm_reduce_conserved use
 * Gamma(f) too.  gamma of ppm_params is not used while the mode is on.  gamma_tracked <= 0 switches it off.
 * PPM_EINVAL unless both indices are finite and > 1; not together with ppm_set_sphere or PPM_OPT_FLATTEN3D.  Host-side state only. */
int ppm_set_two_fluid(ppm_ctx *ctx, double gamma_tracked, double gamma_rest);

/* One increment of the rotation spin-up ("We treat the rotation by adding a solid body rotational flow
 * component to our simulation gradually over the first several thousand time steps"; reading R24): every fluid cell gets
 * du = domega e_z x (X - centre), i.e. du_x = -domega (Y - cy), du_y = +domega (X - cx), about the sphere's centre (the
 * gravity centre without a sphere); rho and p are left as they are.  The caller applies it once per step with
 * domega = Omega_target / N_ramp during the first N_ramp steps.  Only enqueues work (1 light kernel launch). */
int ppm_spin_up(ppm_ctx *ctx, double domega);

/* 1 if the next sweep along axis (0,1,2) will take the bulk-staged path, 0 if the direct path. */
int ppm_axis_path(const ppm_ctx *ctx, int axis);

/* Host-side planning arithmetic of the bulk-staged sweeps, exposed for tests (needs no device): the sweeps march whole
 * pencils while the pencil tiles fill complete waves of resident CTAs; the tail_tiles pencil tiles of the ragged last
 * wave are cut into segments of this many cells (a multiple of 4, or n itself when cutting does not pay; 0 for
 * non-positive arguments) so that the SMs run dry together.  Each cut costs 8 redundant warm-up cells. */
int ppm_plan_tail_chunk(int tail_tiles, int resident_ctas, int n);

/* Number of kernel launches the context has enqueued so far (bench.py reports it). */
long long ppm_launch_count(const ppm_ctx *ctx);

/* Measurement hook (the FP32 roofline "must be measured with an FMA micro-benchmark at the clock the
 * sweep actually runs at"): runs a register-only FFMA kernel on the context's device and stream (16 independent chains
 * per thread, best of 5) and returns the achieved fp32 rate in Tflop/s (2 flop per FFMA lane) in *tflops_out [host].
 * Synchronises the stream; touches no state. */
int ppm_measure_fp32_peak(ppm_ctx *ctx, double *tflops_out);

void ppm_destroy(ppm_ctx *ctx);
const char *ppm_last_error(const ppm_ctx *ctx); /* never NULL; "" if no error; ctx may be NULL */

#ifdef __cplusplus
}
#endif
#endif /* PPM_B200_H */
