// sldg_internal.cuh -- shared declarations of the CUDA SLDG library (sm_100a).  Product code: shares
// nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "sldg.h"

#define SLDG_MAXO 3
#define SLDG_MAXO2 9
#define SLDG_MAXQ 5       // quadrature points per edge for the Green's-theorem line integrals (2o-1)
#define SLDG_HIST 64      // Strang steps whose per-kernel event times are kept (sldg_timing_history)
#ifndef SLDG_EZ_CHUNKS
#define SLDG_EZ_CHUNKS 8   // y chunks of the E_z upload of sldg_strang_step_host
#endif
#ifndef SLDG_RHO_CHUNKS
#define SLDG_RHO_CHUNKS 8  // y chunks of its rho download (the v,z pair forming the charge density)
#endif
#define SLDG_PV_ALIGN 16  // internal v-line pitch is a multiple of 16 doubles (128 B)

// Doubles between two weight blocks of the 2d geometry in memory: o^4, at o = 3 padded to an even number (bulk
// copies move multiples of 16 bytes).
__host__ __device__ constexpr int sldg_w_block_doubles(int O) { return O == 3 ? 82 : O * O * O * O; }

// Grid description passed by value to kernels (lives in the constant bank).
struct GridDev {
    int n[4];   // cells x,y,z,v
    int o[4];   // nodes per cell
    int N[4];   // DOFs
    double lo[4], h[4];
    // internal layout: element (z,Y,X,v) at  z*sZ + Y*sY + X*sX + v   (doubles), v contiguous, pitch Pv
    long long sX, sY, sZ;
    int Pv;
    int contig;       // 1: lines are stored in canonical (z,Y,X) enumeration order, base = line*Pv
    long long lines;  // Nz*Ny*Nx
};

// Gauss-Legendre tables on (0,1) per axis order, Lagrange monomial coefficients, edge quadrature.
struct Basis {
    double xi[SLDG_MAXO + 1][SLDG_MAXO];              // xi[o][node]
    double w[SLDG_MAXO + 1][SLDG_MAXO];               // w[o][node], sums to 1
    double L[SLDG_MAXO + 1][SLDG_MAXO][SLDG_MAXO];    // l_j(x) = sum_a L[o][j][a] x^a
    double qx[SLDG_MAXQ], qw[SLDG_MAXQ];              // (2*oxy-1)-point rule for edge integrals
    int nq;
};

// A_jm(alpha) = sum_d a[j][m][d] alpha^d,  B likewise; degree 2o-1 (eq. 10-11).
struct ShiftPoly {
    double a[SLDG_MAXO][SLDG_MAXO][2 * SLDG_MAXO];
    double b[SLDG_MAXO][SLDG_MAXO][2 * SLDG_MAXO];
    double w[SLDG_MAXO], iw[SLDG_MAXO];  // Gauss-Legendre weights of this order and their reciprocals
    int o;
};

// Workspace of the field step (sldg_field.cu): profiles, the potential on the field grid [Nz][ny][nx], vectors of the
// conjugate-gradient solves, the potential at the nodes (potential energy), scalars and per-system solver records.
struct FieldWs {
    double *n0, *Te, *phi, *rhs, *r, *p, *q, *bar[5], *phin, *scal, *relres;
    int *iters;
    double invB;
    int have_profiles, have_phi;
};

// Workspace of the polar quasi-neutrality solver (sldg_polar_field.cu): profiles at the r vertices, two complex arrays on
// the field grid [Nz][nth][nr+1], the potential, the Thomas scratch, the twiddle tables.
struct PolarWs {
    double *rn0, *dln, *Te, *phi, *cp;
    double2 *ca, *cb, *tw_th, *tw_z;
    int ready, have_phi;
};

struct sldg_ctx {
    sldg_params p;
    GridDev g;
    Basis basis;
    ShiftPoly sp_z, sp_v;
    cudaStream_t stream;
    double *f[2];
    int cur;
    // workspace carve-up
    double *Ez, *va, *vb;   // fields
    int4 *hdr;              // [Nz][ncell] {anchor x, anchor y, slot mask, number of blocks}
    double *W;              // [Nz][ncell][9][o2*o2]  (k-major: W[k*o2+m]), `count` blocks packed from 0
    double *partials;       // reduction scratch
    double *rho_ws;         // [Nz][Ny][Nx] scratch charge density (mass, host entry point)
    double *scalar_ws;      // one double
    int32_t *err;           // sticky device error word
    int32_t *stage_ok;      // [Nz][strips*segments] 1: that block of the streaming 2d apply can stage its rows
    cudaEvent_t gev[2];     // start / end of the geometry kernel of the last 2d step
    cudaStream_t cstream;   // copy stream: sldg_strang_step_host uploads a, b under the first sweeps
    cudaEvent_t cev[2];     // fork / join of that upload
    int ab_pending;         // an upload of a, b is in flight on cstream: the next 2d step waits for it
    // sldg_strang_step_host: E_z uploaded on cstream in ez_chunks chunks of y rows, chunk k complete at ezev[k]; the fused
    // z,v pair that follows is launched per chunk behind its event (0: no such upload in flight)
    int ez_chunks;
    int ez_pending;         // ... or in one piece, complete at ezev[0]: the v sweep of an unfused z,v pair waits for it
    cudaEvent_t ezev[SLDG_EZ_CHUNKS];
    // sldg_strang_step_host: the v,z pair launched in rho_chunks chunks of y rows, each writing the charge density of its
    // planes (fused RHO kernel) and followed by the download of those rows to rho_host on cstream (0: off)
    int rho_chunks;
    double *rho_host;
    cudaEvent_t rhoev[SLDG_RHO_CHUNKS];
    int tile;               // z-tiled pair kernel: 1 when the whole plane does not fit, 2 first (SLDG_FORCE_TILE), 0 never (SLDG_NO_TILE)
    int fuse, last_fused;   // fuse: sldg_strang_step runs each pair of adjacent sweeps in one pass
    size_t n_partials;
    int trace_order, vel_periodic;
    cudaEvent_t ev[8];      // events of the call in progress: handles of the history slot in use (owned by hev)
    cudaEvent_t hev[SLDG_HIST][8];  // per Strang step: ev[0..5] and the two geometry events; ring of the last SLDG_HIST steps
    int hist_fused[SLDG_HIST];
    int hpos;               // slot the next Strang step records into
    long long hcount;       // Strang steps recorded since creation
    int last_slot;
    int ev_kind;            // 0 none, 1 strang, 2 z, 3 v, 4 xy
    long long launches;
    int sm_count;
    FieldWs fld;
    PolarWs pol;
    double *src_dz, *src_dth;  // d_z phi, d_theta phi at the nodes [Nz][Ny][Nx] (source term of the delta-g formulation)
    double *src_gv, *src_gr;   // d_v g_eq, d_r(g_eq/r) as [Nx][Pv] tables
    int src_ready;             // bit 0: profiles set, bit 1: fields set
    double *f_c;            // optional third state buffer (Algorithm 2 keeps the state of time level n)
};

// ---- kernel launchers (each returns cudaGetLastError()) ------------------------------------------
cudaError_t launch_pack(sldg_ctx *c, const double *canon, double *internal);
cudaError_t launch_unpack(sldg_ctx *c, const double *internal, double *canon);
cudaError_t launch_advect_z(sldg_ctx *c, const double *fin, double *fout, double tau);
cudaError_t launch_advect_v(sldg_ctx *c, const double *fin, double *fout, double tau);
cudaError_t launch_charge_density(sldg_ctx *c, const double *fin, double *rho, long long line0 = 0, long long line1 = -1);  // lines [line0, line1)
cudaError_t launch_mass(sldg_ctx *c, const double *fin, double *mass_out);
cudaError_t launch_mass_from_rho(sldg_ctx *c, const double *rho, double *mass_out);
cudaError_t launch_xy_geometry(sldg_ctx *c, double tau, int trace_order);
size_t xy_apply_stage_flags(const sldg_params *p);  // number of stage_ok entries
cudaError_t launch_geometry_expand(sldg_ctx *c, int z, int32_t *anchor, int32_t *mask, double *Wd);
cudaError_t launch_xy_apply(sldg_ctx *c, const double *fin, double *fout);
cudaError_t count_weight_blocks(sldg_ctx *c, long long *total_host);
// planes (Y,X) with index Y * Nx + X in [col0, col1); col1 < 0: all from col0 on
cudaError_t launch_fused_sweeps(sldg_ctx *c, const double *fin, double *fout, double tau_z, double tau_v, bool z_first,
                                bool z_only = false, int col0 = 0, int col1 = -1, double *rho = nullptr);
// launch_fused_sweeps would not return cudaErrorNotSupported (rho: with the charge density from the v,z pair)
bool fused_sweeps_supported(const sldg_ctx *c, bool z_first, bool rho = false);
cudaError_t launch_tiled_sweeps(sldg_ctx *c, const double *fin, double *fout, double tau_z, double tau_v, bool z_first);
size_t field_workspace_bytes(const sldg_params *p);
void field_carve(sldg_ctx *c, char *base);
cudaError_t launch_field_step(sldg_ctx *c, const double *fin, double tol, int max_iter);
cudaError_t launch_diagnostics(sldg_ctx *c, const double *fin, double r_p, double *out_host);
size_t source_workspace_bytes(const sldg_params *p);
void source_carve(sldg_ctx *c, char *base);
cudaError_t launch_source_profiles(sldg_ctx *c, const double *dv_geq, const double *dr_geq);
cudaError_t launch_source_step(sldg_ctx *c, double *f, double tau, const double *fin = nullptr);  // fin: out of place
size_t polar_workspace_bytes(const sldg_params *p);
void polar_carve(sldg_ctx *c, char *base);
cudaError_t launch_polar_profiles(sldg_ctx *c, const double *rn0, const double *dln, const double *Te);
cudaError_t launch_polar_field_step(sldg_ctx *c, const double *fin);
