/*
 * sldg.h -- C-ABI boundary of libsldg: the data-parallel hot path of the drift-kinetic solver of
 * arxiv 2212.03036 (Einkemmer & Moriggl), i.e. the split semi-Lagrangian discontinuous Galerkin (SLDG)
 * advection of the 4d distribution f(x,y,z,v) in fp64, as hand-written CUDA for sm_100a (B200).
 * Citations are PAPER.md:LINE (the paper's text) and SURVEY.md section 8 (the readings taken where the
 * paper is silent; they are listed in DESIGN.md).
 *
 * Conventions
 *   axes            0:x 1:y 2:z 3:v.  n[d] cells, order[d] Gauss-Legendre nodes per cell,
 *                   N[d] = n[d]*order[d] degrees of freedom; DOF index = cell*order + node; node
 *                   coordinate = lo + (cell + xi_node) * h,  h = (hi-lo)/n.  DOFs are point values.
 *   canonical f     double [Nz][Nv][Ny][Nx]   (x fastest)        -- the layout of import/export
 *   Ez              double [Nz][Ny][Nx]       speed of the v-advection, Ez = -d(phi)/dz (eq. 5)
 *   a, b            double [Nz][ny+1][nx+1]   poloidal velocity at the cell vertices (eq. 12)
 *   rho             double [Nz][Ny][Nx]
 *   boundary        f is periodic along all four axes (PAPER.md:55 for theta, z, v; SURVEY.md 8(c) A15
 *                   for the Cartesian x, y).
 *   memory          every pointer named *_dev is DEVICE memory, *_host is HOST memory.  All device buffers
 *                   are allocated by the caller and BORROWED: the context owns no device memory except
 *                   what lives inside `workspace`.  f_a, f_b, workspace must stay valid until
 *                   sldg_destroy and must be 256-byte aligned.
 *   state           the library keeps f in an INTERNAL layout (v fastest) inside f_a/f_b and
 *                   ping-pongs between them; sldg_import_state / sldg_export_state convert.
 *   stream          every call enqueues on the cudaStream_t given at sldg_create and returns without
 *                   synchronising, unless stated otherwise.
 *   errors          return value 0 = success, negative = SLDG_E* below.  Errors detected on the device
 *                   (geometry) are sticky and reported by sldg_check.  There is no CPU fallback: without
 *                   a CUDA device every compute call returns SLDG_ECUDA.
 */
#ifndef SLDG_H
#define SLDG_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sldg_ctx sldg_ctx; /* opaque */

typedef struct {
    int32_t n[4];        /* cells in x, y, z, v                                                     */
    int32_t order[4];    /* nodes per cell per axis, each 1, 2 or 3; order[0] == order[1]
                            (per-axis degree is in the paper: PAPER.md:396; the paper runs 2)       */
    double lo[4], hi[4]; /* box                                                                     */
    int32_t max_stencil; /* largest block of source cells one upstream cell may touch per direction;
                            must be 3 (the paper's 3x3 assumption)                    */
    int32_t layout;      /* internal line order: 0 = library default, 1 = z,y,x  2 = y,x,z  3 = y,z,x
                            (v is always fastest; a tuning knob, results do not depend on it)       */
} sldg_params;

enum {
    SLDG_OK = 0,
    SLDG_EINVAL = -1,   /* bad parameter, null pointer, misaligned or too small buffer               */
    SLDG_ECUDA = -2,    /* CUDA runtime / launch error, or no device                                  */
    SLDG_ESTENCIL = -3, /* an upstream cell's bounding box exceeds max_stencil   */
    SLDG_EGEOM = -4,    /* upstream cell not convex / not positively oriented (crossed characteristics,
                           PAPER.md:190) or a singular Vandermonde system              */
    SLDG_ELIMIT = -5    /* the problem exceeds the fixed scratch of sldg_mass_static                  */
};

/* Sizes (bytes) of each ping-pong state buffer and of the workspace for these parameters; 0 on
 * invalid parameters.  Host-only, no device needed. */
size_t sldg_state_bytes(const sldg_params *p);
size_t sldg_workspace_bytes(const sldg_params *p);

/* Create a context.  f_a_dev / f_b_dev: the two state buffers (sldg_state_bytes each); workspace_dev:
 * sldg_workspace_bytes; cuda_stream: a cudaStream_t (NULL = legacy default stream).  The state is
 * undefined until sldg_import_state.  Fields default to Ez = 0, a = b = 0, trace order 2. */
int sldg_create(const sldg_params *p, double *f_a_dev, double *f_b_dev, void *workspace_dev,
                size_t workspace_bytes, void *cuda_stream, sldg_ctx **out);
int sldg_destroy(sldg_ctx *ctx);

/* State in/out, canonical layout [Nz][Nv][Ny][Nx].  The *_dev calls are asynchronous device-to-device
 * transposes.  The *_host calls copy through the idle ping-pong buffer and synchronise the stream. */
int sldg_import_state(sldg_ctx *ctx, const double *f_canonical_dev);
int sldg_export_state(sldg_ctx *ctx, double *f_canonical_dev);
int sldg_import_state_host(sldg_ctx *ctx, const double *f_canonical_host);
int sldg_export_state_host(sldg_ctx *ctx, double *f_canonical_host);
/* Which of f_a / f_b currently holds the state (internal layout). */
double *sldg_current(sldg_ctx *ctx);

/* Fields; copied into the workspace, the caller's buffers are free afterwards.
 * sldg_set_vxy: `periodic` != 0 declares a, b bitwise periodic (a[.., ny, :] == a[.., 0, :] and
 * a[.., :, nx] == a[.., :, 0]); the half-step point of the second-order tracing (eq. 15) is
 * then looked up modulo the box so that the upstream mesh tiles across the periodic seam; with
 * periodic == 0 the cell index is clamped to the box (reading A15); periodic == 2: periodic
 * along y only, clamped along x -- the polar plane with x = r, y = theta, where the radial velocity is zero at r_min and
 * r_max and no upstream cell leaves the box through those edges. */
int sldg_set_Ez(sldg_ctx *ctx, const double *Ez_dev);
int sldg_set_vxy(sldg_ctx *ctx, const double *a_dev, const double *b_dev, int periodic);

/* 1d SLDG sweep along z with speed v (eq. 4; eq. 11): for each v node q,
 * delta = v_q tau / h_z, s = floor(-delta), alpha = -delta - s, and for every z cell i, node j
 *   f'[i,j] = sum_m A_jm(alpha) f[(i+s) mod nz, m] + B_jm(alpha) f[(i+s+1) mod nz, m]
 * with A, B the overlap matrices of eq. (10).  Any tau, any Courant number. */
int sldg_advect_z(sldg_ctx *ctx, double tau);
/* 1d SLDG sweep along v with speed Ez(x,y,z) (eq. 5), periodic in v. */
int sldg_advect_v(sldg_ctx *ctx, double tau);
/* 2d SLDG step in the poloidal plane (eq. 6, 12-18; Algorithm 3):
 * per z node the upstream quadrilaterals, adjoint polynomials and Green's-theorem integrals C (18) are
 * computed once and applied to every v node (17).  trace_order 1: eq. (14); 2: eq. (15) as explicit
 * midpoint with the one field set by sldg_set_vxy.  Geometry failures are reported
 * by sldg_check (SLDG_ESTENCIL, SLDG_EGEOM); the state is then unspecified. */
int sldg_advect_xy(sldg_ctx *ctx, double tau, int trace_order);
/* rho[z,y,x] = int f dv = h_v sum_{l,q} w_q f[z,(l,q),y,x].  rho_dev: [Nz][Ny][Nx]. */
int sldg_charge_density(sldg_ctx *ctx, double *rho_dev);
/* Total mass sum f w_x w_y w_z w_v h_x h_y h_z h_v into one device double. */
int sldg_mass(sldg_ctx *ctx, double *mass_dev);
/* One Strang step with the fields currently set (Algorithm 1 steps 3,4,6,7,8; the
 * source terms vanish for the Cartesian full-f formulation):
 *   advect_z(dt/2), advect_v(dt/2), advect_xy(dt), advect_v(dt/2), advect_z(dt/2).
 * The result is bit-identical to those five calls.  Where the (z,v) plane of one (x,y) node fits in shared
 * memory, each pair of adjacent sweeps runs as ONE kernel that reads and writes f once (3 passes over f per
 * step instead of 5); environment variable SLDG_NO_FUSE at sldg_create time disables that. */
int sldg_strang_step(sldg_ctx *ctx, double dt);
int sldg_set_trace_order(sldg_ctx *ctx, int trace_order); /* used by sldg_strang_step; default 2 */

/* The same step driven from HOST buffers (what a host-side field solver sees): copies Ez, a, b from
 * host to device, runs sldg_strang_step, then the charge density and the mass, copies rho and mass back
 * to the host, and synchronises the stream.  Pinned host buffers make the copies asynchronous.
 * Any of Ez_host / a_host+b_host / rho_host / mass_host may be NULL to skip that transfer.
 * The transfers overlap the kernels where the data dependences allow: E_z goes up in chunks of y rows, each chunk's
 * (z,v) planes swept as soon as it has arrived (when the z,v pair runs fused), or in one piece under the z sweep, which
 * does not read it (when the pair is certain to run as two kernels); a, b go up under the first sweeps.  rho:
 * where the v,z pair runs fused at o = 2 with unpadded v lines of whole warps (Nv a multiple of 32), that kernel forms the
 * charge density from its own results -- no further pass over f -- and is launched in chunks of y rows, the rows of a
 * chunk coming down under the next chunk; otherwise a reduction over f in slabs of z, each slab coming down under the
 * reduction of the next.  The two sum over v in a different order: rho_host agrees with sldg_charge_density to
 * round-off (1e-14 relative), not bit for bit; the state is the same bit for bit.  The host buffers must stay valid
 * until the call returns (it synchronises). */
int sldg_strang_step_host(sldg_ctx *ctx, double dt, const double *Ez_host, const double *a_host,
                          const double *b_host, int periodic, double *rho_host, double *mass_host);

/* Synchronises the stream and returns the sticky device error word (0, SLDG_ESTENCIL, SLDG_EGEOM) or
 * SLDG_ECUDA; clears it. */
int sldg_check(sldg_ctx *ctx);
/* Device times (CUDA events) of the last sldg_strang_step, in ms:
 * ms[0] z  ms[1] v  ms[3] the WHOLE xy substep (geometry + apply, first launch to last)  ms[4] v  ms[5] z
 * ms[7] total; ms[2] = duration of the geometry kernel alone (it is part of ms[3], not in addition to it);
 * ms[6] = flags: +2 if the first pair of adjacent sweeps (z,v before the 2d step) ran fused in one pass over f
 * -- then ms[0] holds the time of the pair and ms[1] = 0 --, +4 if the second pair (v,z after it) did -- then
 * ms[4] holds the time of the pair and ms[5] = 0.
 * After a single sldg_advect_* call only that entry (and ms[7]) is set.  Synchronises. */
int sldg_last_timing_ms(sldg_ctx *ctx, float ms[8]);
/* The same eight numbers for each of the last n sldg_strang_step calls (n <= 64, oldest first; ms: n x 8 floats): the
 * library keeps the events of the last 64 steps, so a timed loop needs no synchronisation inside it.  Synchronises. */
int sldg_timing_history(sldg_ctx *ctx, int n, float *ms);
/* Number of kernels the library launched on behalf of this context since creation. */
long long sldg_launch_count(sldg_ctx *ctx);
/* Debug / test access to the geometry of the last sldg_advect_xy: for z node `z` copies, per target
 * cell t = j*nx + i, anchor[2t..2t+1] = offset (in cells, unwrapped) of the source cell of slot (0,0)
 * relative to the target cell, mask[t] = bitmask over the
 * 3x3 slots (bit dx + 3 dy), and W[t][slot][m][k] = C^{ij,m}_{rs,k} / W_m (dense, 9*o^4 doubles per cell,
 * entries of empty slots are unspecified).  Device buffers; asynchronous. */
int sldg_debug_geometry(sldg_ctx *ctx, int z, int32_t *anchor_dev, int32_t *mask_dev, double *W_dev);
/* Diagnostic counter `which` since creation, into *value_host; synchronises the stream.
 *   0: blocks (strip x segment x z node) of the 2d apply whose source window does not fit the streaming kernel's
 *      shared-memory ring (anchors varying by many cells inside the block, more than 3 source rows per target
 *      row) and were handed to the direct kernel instead. */
/*   1: non-empty weight blocks (target cell, source cell) of the last sldg_advect_xy, summed over all z nodes: the 2d
 *      apply does 2 o^4 flops per block and v node (eq. 17; PAPER.md:378-382 counts the dense 3x3 case). */
int sldg_debug_counter(sldg_ctx *ctx, int which, long long *value_host);
/* Measures the device's fp64 FMA throughput (independent FMA chains, every SM busy), best of `repeats` launches, in
 * TFLOP/s: the roof of the ALU-bound kernels (the paper's intensity argument).
 * Synchronises. */
int sldg_debug_fp64_peak(sldg_ctx *ctx, int repeats, double *tflops_host);

/* ---- Field step, invariants and the two time-stepping algorithms ----------------
 * Outside the timed hot path (1/Nv of the volume).  Field grid: the nx x ny cell vertices (periodic) x Nz equidistant
 * z points at (m + 1/2) h_z / o_z ("inside the cell"); arrays on it are double [Nz][ny][nx].
 *
 * sldg_set_profiles: n0 and T_e of the quasi-neutrality equation (eq. 2) at the vertices, [ny][nx], and
 * the magnetic field strength B of the drift (eq. 1); copied into the workspace. */
int sldg_set_profiles(sldg_ctx *ctx, const double *n0_dev, const double *Te_dev, double B);
/* Algorithm 1 step 1 / 5 (section 3.6): charge density of the current state ->
 * resampled to the field grid (vertex value = mean of the four adjacent cells' polynomials) ->
 *   -(1/n0) div(n0 grad phi) + (phi - <phi>)/Te = rho/n0 - 1,  <phi> = z average (R20-R22),
 * second-order differences, Jacobi-preconditioned conjugate gradients to |r| <= tol |b| or max_iter iterations ->
 * a = -d_y phi/B, b = d_x phi/B, E_z = -d_z phi by centred differences, interpolated to where the advection steps
 * read them (as after sldg_set_vxy(.., periodic = 1) and sldg_set_Ez).  SLDG_EINVAL before sldg_set_profiles. */
int sldg_field_step(sldg_ctx *ctx, double tol, int max_iter);
/* Largest iteration count and relative residual over the systems of the last field step.  Synchronises. */
int sldg_field_info(sldg_ctx *ctx, int *max_iters_host, double *max_relres_host);
/* Copies of the last field step's results: phi on the field grid; E_z [Nz][Ny][Nx], a, b [Nz][ny+1][nx+1] as the
 * advection steps see them (any pointer may be NULL).  Asynchronous. */
int sldg_get_phi(sldg_ctx *ctx, double *phi_dev);
int sldg_get_fields(sldg_ctx *ctx, double *Ez_dev, double *a_dev, double *b_dev);
/* The quantities of PAPER.md:332-346 for the current state and the potential of the last field step:
 * out[0] electric energy sqrt(int phi^2(r_p, theta, z) dtheta dz) on the circle of radius r_p around the box centre
 * (bilinear samples at 4 max(nx, ny) angles), out[1] mass, out[2] L2 norm, out[3] kinetic energy int v^2/2 f,
 * out[4] potential energy int phi f (total energy = out[3] + out[4]).  Synchronises. */
int sldg_diagnostics(sldg_ctx *ctx, double r_p, double out_host[5]);
/* One time step of Algorithm 1 (the source terms vanish for the Cartesian full-f formulation):
 * field step, z(dt/2), v(dt/2), field step, xy(dt), v(dt/2), z(dt/2). */
int sldg_step_algorithm1(sldg_ctx *ctx, double dt, double tol, int max_iter);
/* A third state buffer (sldg_state_bytes, 256-byte aligned, borrowed until sldg_destroy) for Algorithm 2, which
 * restarts its corrector from the state of time level n ("three copies"). */
int sldg_set_third_buffer(sldg_ctx *ctx, double *f_c_dev);
/* One time step of Algorithm 2: field step; predictor z(dt/2), v(dt/2), xy(dt/2) with first-order
 * tracing (eq. 14); field step on the predicted state; corrector from the state of level n: z(dt/2), v(dt/2), xy(dt)
 * with second-order tracing (eq. 15), v(dt/2), z(dt/2).  No state is copied: the three buffers rotate. */
int sldg_step_algorithm2(sldg_ctx *ctx, double dt, double tol, int max_iter);

/* ---- Source term of the delta-g formulation in polar coordinates ------------------------
 * The paper advects dg = g - g_eq, g = r f, in (r, theta, z, v) (eq. 3): axis 0 is r, axis 1 theta; the
 * three advections are the calls above with the drift (-d_theta phi / r, d_r phi / r) at the vertices -- radial
 * component zero at r_min and r_max, sldg_set_vxy(.., periodic = 2) -- and the equilibrium enters through
 *     dg += tau ( d_z phi * d_v g_eq + d_theta phi * d_r(g_eq / r) )          (section 3.5)
 * sldg_set_equilibrium: d_v g_eq and d_r(g_eq/r) as double [Nv][Nr] (r fastest).  sldg_set_source_fields: d_z phi and
 * d_theta phi at the nodes, double [Nz][Ntheta][Nr].  Both are copied into the workspace. */
int sldg_set_equilibrium(sldg_ctx *ctx, const double *dv_geq_dev, const double *dr_geq_dev);
int sldg_set_source_fields(sldg_ctx *ctx, const double *dz_phi_dev, const double *dtheta_phi_dev);
/* Forward-Euler source step of size tau, in place (one pass over f).  SLDG_EINVAL before the two setters.
 * sldg_last_timing_ms()[7] holds its device time afterwards. */
int sldg_source_step(sldg_ctx *ctx, double tau);
/* Algorithm 1 steps 2-4, 6-9 with the fields currently set: source(dt/2), z(dt/2), v(dt/2), 2d(dt),
 * v(dt/2), z(dt/2), source(dt/2). */
int sldg_strang_step_sources(sldg_ctx *ctx, double dt);
/* The paper's quasi-neutrality solver in polar coordinates (eq. 2; Neumann at r_min, Dirichlet at r_max,
 * PAPER.md:43; Fourier transform in theta and z, second-order differences and a tridiagonal solve in r):
 * sldg_set_polar_profiles: r n0(r), n0'/n0 (r), T_e(r) at the nr + 1 radial vertices (device doubles, copied).
 * sldg_polar_field_step: charge density of the current delta-g -> rhs = rho~/(r n0) on the field grid (nr + 1 radial
 * vertices x ntheta x Nz equidistant z points) -> phi -> drift (-d_theta phi/r, d_r phi/r) at the vertices with zero
 * radial ends, E_z, d_z phi and d_theta phi at the nodes, written where sldg_set_vxy(.., 2), sldg_set_Ez and
 * sldg_set_source_fields put them.  <phi> = z average (R21). */
int sldg_set_polar_profiles(sldg_ctx *ctx, const double *r_n0_dev, const double *dln_n0_dev, const double *Te_dev);
int sldg_polar_field_step(sldg_ctx *ctx);
int sldg_get_polar_phi(sldg_ctx *ctx, double *phi_dev);                 /* [Nz][ntheta][nr+1] */
int sldg_get_source_fields(sldg_ctx *ctx, double *dz_phi_dev, double *dtheta_phi_dev); /* [Nz][Ntheta][Nr], either may be NULL */
/* Algorithm 1 with all nine steps in the delta-g formulation: field, source(dt/2), z(dt/2), v(dt/2),
 * field, 2d(dt), v(dt/2), z(dt/2), source(dt/2).  Needs sldg_set_polar_profiles and sldg_set_equilibrium. */
int sldg_step_algorithm1_polar(sldg_ctx *ctx, double dt);
/* Algorithm 2 with all thirteen steps in the delta-g formulation; needs sldg_set_third_buffer too. */
int sldg_step_algorithm2_polar(sldg_ctx *ctx, double dt);
const char *sldg_strerror(int code);

/* ---- allocation-free entry point (sldg_static.cu) -------------------------------------------------------------
 * Total mass (the v integral is the charge density of PAPER.md:57) of a distribution given in the
 * canonical layout [Nz][Nv][Ny][Nx], WITHOUT a context, a workspace or any allocation: for callers that may not call
 * cudaMalloc (CUDA graph capture, serving loops).  The intermediate charge density and partial sums live in a file-scope
 * static __device__ array of SLDG_STATIC_MAX_NODES + 1024 doubles (8 MiB + 8 KiB per GPU that loads the library).
 *   p               only n, order, lo, hi are read (order[d] in 1..3)
 *   f_canonical_dev DEVICE, borrowed, read only, 8-byte aligned
 *   mass_dev        DEVICE, one double, written
 *   cuda_stream     a cudaStream_t of the CURRENT device (NULL = legacy default stream); asynchronous
 * Returns SLDG_ELIMIT when Nx*Ny*Nz > SLDG_STATIC_MAX_NODES (nothing is launched), SLDG_EINVAL on bad arguments,
 * SLDG_ECUDA on a launch error or without a device.  Every call on a device shares the one array: calls ordered on a
 * stream are safe, calls that overlap on the GPU race.  Nothing in the array needs clearing between calls.
 * sldg_mass_static_setup looks up the array's device address for the current device (cudaGetSymbolAddress, once per
 * device; the first sldg_mass_static does it otherwise -- call it beforehand when the first call is under capture). */
#define SLDG_STATIC_MAX_NODES (1 << 20)
long long sldg_mass_static_max_nodes(void);
int sldg_mass_static_setup(void);
int sldg_mass_static(const sldg_params *p, const double *f_canonical_dev, double *mass_dev, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* SLDG_H */
