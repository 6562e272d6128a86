// sldg_api.cu -- the C-ABI of libsldg (include/sldg.h): context, host-side tables, orchestration.
// Product code for sm_100a; no CPU fallback, nothing from oracle/.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>
#include <vector>

#include "sldg_internal.cuh"

namespace {

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

bool params_ok(const sldg_params *p)
{
    if (!p) return false;
    for (int d = 0; d < 4; ++d) {
        if (p->n[d] < 1 || p->order[d] < 1 || p->order[d] > SLDG_MAXO) return false;
        if (!(p->hi[d] > p->lo[d])) return false;
    }
    if (p->order[0] != p->order[1]) return false;
    if (p->max_stencil != 3) return false;
    if (p->layout < 0 || p->layout > 3) return false;
    return true;
}

void fill_grid(const sldg_params *p, GridDev *g)
{
    for (int d = 0; d < 4; ++d) {
        g->n[d] = p->n[d];
        g->o[d] = p->order[d];
        g->N[d] = p->n[d] * p->order[d];
        g->lo[d] = p->lo[d];
        g->h[d] = (p->hi[d] - p->lo[d]) / p->n[d];
    }
    g->Pv = (int)align_up((size_t)g->N[3], SLDG_PV_ALIGN);
    const long long Nx = g->N[0], Ny = g->N[1], Nz = g->N[2], Pv = g->Pv;
    int layout = p->layout == 0 ? 1 : p->layout;
    if (layout == 1) {  // z, y, x, v
        g->sX = Pv; g->sY = Nx * Pv; g->sZ = Ny * Nx * Pv;
    } else if (layout == 2) {  // y, x, z, v
        g->sZ = Pv; g->sX = Nz * Pv; g->sY = Nx * Nz * Pv;
    } else {  // y, z, x, v
        g->sX = Pv; g->sZ = Nx * Pv; g->sY = Nz * Nx * Pv;
    }
    g->lines = Nz * Ny * Nx;
    g->contig = (layout == 1) ? 1 : 0;
}

struct WorkspaceMap {
    size_t Ez, va, vb, hdr, W, partials, rho, scalar, err, stage_ok, field, source, polar, total;
    size_t n_partials;
};

WorkspaceMap map_workspace(const sldg_params *p)
{
    GridDev g;
    fill_grid(p, &g);
    WorkspaceMap m;
    const size_t ncell = (size_t)g.n[0] * g.n[1], Nz = (size_t)g.N[2];
    const size_t vplane = (size_t)(g.n[0] + 1) * (g.n[1] + 1);
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t at = off; off = align_up(off + bytes, 256); return at; };
    m.Ez = take((size_t)g.lines * 8);
    m.va = take(Nz * vplane * 8);
    m.vb = take(Nz * vplane * 8);
    m.hdr = take(Nz * ncell * 16);
    m.W = take(Nz * ncell * 9 * (size_t)sldg_w_block_doubles(g.o[0]) * 8);
    m.n_partials = 8192;
    m.partials = take(m.n_partials * 8);
    m.rho = take((size_t)g.lines * 8);
    m.scalar = take(256);
    m.err = take(256);
    m.stage_ok = take(xy_apply_stage_flags(p) * 4);
    m.field = take(field_workspace_bytes(p));
    m.source = take(source_workspace_bytes(p));
    m.polar = take(polar_workspace_bytes(p));
    m.total = off;
    return m;
}

// ---- host-side tables (long double) ---------------------------------------------------------------
typedef std::vector<long double> Poly;

Poly pmul(const Poly &a, const Poly &b)
{
    Poly r(a.size() + b.size() - 1, 0.0L);
    for (size_t i = 0; i < a.size(); ++i)
        for (size_t j = 0; j < b.size(); ++j) r[i + j] += a[i] * b[j];
    return r;
}

long double binom(int n, int k)
{
    long double r = 1.0L;
    for (int i = 1; i <= k; ++i) r = r * (n - k + i) / i;
    return r;
}

void gl_nodes(int o, long double *x, long double *w)
{
    if (o == 1) {
        x[0] = 0.5L; w[0] = 1.0L;
    } else if (o == 2) {
        long double d = sqrtl(3.0L) / 6.0L;
        x[0] = 0.5L - d; x[1] = 0.5L + d;
        w[0] = w[1] = 0.5L;
    } else if (o == 3) {
        long double d = sqrtl(15.0L) / 10.0L;
        x[0] = 0.5L - d; x[1] = 0.5L; x[2] = 0.5L + d;
        w[0] = w[2] = 5.0L / 18.0L; w[1] = 4.0L / 9.0L;
    } else {  // o == 5 (edge quadrature only)
        long double s = sqrtl(10.0L / 7.0L);
        long double t1 = sqrtl(5.0L - 2.0L * s) / 3.0L, t2 = sqrtl(5.0L + 2.0L * s) / 3.0L;
        long double w1 = (322.0L + 13.0L * sqrtl(70.0L)) / 900.0L, w2 = (322.0L - 13.0L * sqrtl(70.0L)) / 900.0L;
        x[0] = 0.5L - 0.5L * t2; x[1] = 0.5L - 0.5L * t1; x[2] = 0.5L; x[3] = 0.5L + 0.5L * t1; x[4] = 0.5L + 0.5L * t2;
        w[0] = w[4] = 0.5L * w2; w[1] = w[3] = 0.5L * w1; w[2] = 0.5L * 128.0L / 225.0L;
    }
}

// monomial coefficients of the Lagrange basis on the o GL nodes
void lagrange_monomials(int o, const long double *x, long double L[SLDG_MAXO][SLDG_MAXO])
{
    for (int j = 0; j < o; ++j) {
        Poly p(1, 1.0L);
        for (int i = 0; i < o; ++i)
            if (i != j) {
                Poly f(2);
                f[0] = -x[i] / (x[j] - x[i]);
                f[1] = 1.0L / (x[j] - x[i]);
                p = pmul(p, f);
            }
        for (int a = 0; a < SLDG_MAXO; ++a) L[j][a] = a < (int)p.size() ? p[a] : 0.0L;
    }
}

void fill_basis(const sldg_params *p, Basis *bs)
{
    memset(bs, 0, sizeof(*bs));
    for (int o = 1; o <= SLDG_MAXO; ++o) {
        long double x[5], w[5], L[SLDG_MAXO][SLDG_MAXO];
        gl_nodes(o, x, w);
        lagrange_monomials(o, x, L);
        for (int j = 0; j < o; ++j) {
            bs->xi[o][j] = (double)x[j];
            bs->w[o][j] = (double)w[j];
            for (int a = 0; a < o; ++a) bs->L[o][j][a] = (double)L[j][a];
        }
    }
    const int nq = 2 * p->order[0] - 1;  // exact for the edge integrand of degree 4o-3
    long double x[5], w[5];
    gl_nodes(nq, x, w);
    bs->nq = nq;
    for (int k = 0; k < nq; ++k) {
        bs->qx[k] = (double)x[k];
        bs->qw[k] = (double)w[k];
    }
}

// Polynomial coefficients in alpha of the overlap matrices of eq. (10)-(11):
//   A_jm(alpha) = (1/w_j) int_0^{1-alpha} l_j(xi) l_m(xi+alpha) dxi
//   B_jm(alpha) = (1/w_j) int_0^{alpha}   l_j(eta+1-alpha) l_m(eta) deta
// obtained by expanding the integrals symbolically (binomial theorem), long double arithmetic.
void fill_shift_poly(int o, ShiftPoly *sp)
{
    memset(sp, 0, sizeof(*sp));
    sp->o = o;
    long double x[5], w[5], L[SLDG_MAXO][SLDG_MAXO];
    gl_nodes(o, x, w);
    lagrange_monomials(o, x, L);
    for (int j = 0; j < o; ++j) {
        sp->w[j] = (double)w[j];
        sp->iw[j] = 1.0 / sp->w[j];
    }
    const int deg = 2 * o;  // number of coefficients (degree 2o-1)
    auto one_minus_alpha_pow = [&](int n) {
        Poly r(n + 1);
        for (int e = 0; e <= n; ++e) r[e] = binom(n, e) * ((e & 1) ? -1.0L : 1.0L);
        return r;
    };
    auto alpha_pow = [&](int n) {
        Poly r(n + 1, 0.0L);
        r[n] = 1.0L;
        return r;
    };
    for (int j = 0; j < o; ++j)
        for (int m = 0; m < o; ++m) {
            Poly pa(deg, 0.0L), pb(deg, 0.0L);
            for (int a = 0; a < o; ++a)
                for (int b = 0; b < o; ++b) {
                    // A: l_m(xi+alpha) = sum_b L_m[b] sum_c C(b,c) xi^c alpha^(b-c)
                    for (int c = 0; c <= b; ++c) {
                        Poly t = pmul(alpha_pow(b - c), one_minus_alpha_pow(a + c + 1));
                        long double k = L[j][a] * L[m][b] * binom(b, c) / (a + c + 1);
                        for (size_t d = 0; d < t.size(); ++d) pa[d] += k * t[d];
                    }
                    // B: l_j(eta+1-alpha) = sum_a L_j[a] sum_c C(a,c) eta^c (1-alpha)^(a-c)
                    for (int c = 0; c <= a; ++c) {
                        Poly t = pmul(one_minus_alpha_pow(a - c), alpha_pow(b + c + 1));
                        long double k = L[j][a] * L[m][b] * binom(a, c) / (b + c + 1);
                        for (size_t d = 0; d < t.size(); ++d) pb[d] += k * t[d];
                    }
                }
            for (int d = 0; d < deg; ++d) {
                sp->a[j][m][d] = (double)(pa[d] / w[j]);
                sp->b[j][m][d] = (double)(pb[d] / w[j]);
            }
            // A(0) = I and B(0) = 0 hold exactly (orthogonality of the basis): integer Courant numbers
            // must be bit-exact copies, so the constant terms are set to their exact values.
            sp->a[j][m][0] = (j == m) ? 1.0 : 0.0;
            sp->b[j][m][0] = 0.0;
        }
}

int cuda_fail(cudaError_t e) { return e == cudaSuccess ? SLDG_OK : SLDG_ECUDA; }

// the events a call records are those of one slot of the history ring (ev[0..5]: the substeps, ev[6..7] = gev: the
// geometry kernel); a Strang step moves on to the next slot when it is done, so that the per-kernel times of the last
// SLDG_HIST steps can be read after a timed loop without a synchronisation inside it (sldg_timing_history)
void use_history_slot(sldg_ctx *c, int h)
{
    for (int k = 0; k < 8; ++k) c->ev[k] = c->hev[h][k];
    c->gev[0] = c->hev[h][6];
    c->gev[1] = c->hev[h][7];
}

void swap_state(sldg_ctx *c) { c->cur ^= 1; }

}  // namespace

extern "C" {

size_t sldg_state_bytes(const sldg_params *p)
{
    if (!params_ok(p)) return 0;
    GridDev g;
    fill_grid(p, &g);
    return (size_t)g.lines * g.Pv * 8;
}

size_t sldg_workspace_bytes(const sldg_params *p)
{
    if (!params_ok(p)) return 0;
    return map_workspace(p).total;
}

int sldg_create(const sldg_params *p, double *f_a_dev, double *f_b_dev, void *workspace_dev,
                size_t workspace_bytes, void *cuda_stream, sldg_ctx **out)
{
    if (!out) return SLDG_EINVAL;
    *out = nullptr;
    if (!params_ok(p) || !f_a_dev || !f_b_dev || !workspace_dev) return SLDG_EINVAL;
    if (((uintptr_t)f_a_dev | (uintptr_t)f_b_dev | (uintptr_t)workspace_dev) & 255) return SLDG_EINVAL;
    WorkspaceMap m = map_workspace(p);
    if (workspace_bytes < m.total) return SLDG_EINVAL;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return SLDG_ECUDA;
    sldg_ctx *c = new (std::nothrow) sldg_ctx();
    if (!c) return SLDG_EINVAL;
    memset(c, 0, sizeof(*c));
    c->p = *p;
    fill_grid(p, &c->g);
    fill_basis(p, &c->basis);
    fill_shift_poly(p->order[2], &c->sp_z);
    fill_shift_poly(p->order[3], &c->sp_v);
    c->stream = (cudaStream_t)cuda_stream;
    c->f[0] = f_a_dev;
    c->f[1] = f_b_dev;
    c->cur = 0;
    char *ws = (char *)workspace_dev;
    c->Ez = (double *)(ws + m.Ez);
    c->va = (double *)(ws + m.va);
    c->vb = (double *)(ws + m.vb);
    c->hdr = (int4 *)(ws + m.hdr);
    c->W = (double *)(ws + m.W);
    c->partials = (double *)(ws + m.partials);
    c->n_partials = m.n_partials;
    c->rho_ws = (double *)(ws + m.rho);
    c->scalar_ws = (double *)(ws + m.scalar);
    c->err = (int32_t *)(ws + m.err);
    c->stage_ok = (int32_t *)(ws + m.stage_ok);
    field_carve(c, ws + m.field);
    source_carve(c, ws + m.source);
    polar_carve(c, ws + m.polar);
    c->fuse = getenv("SLDG_NO_FUSE") ? 0 : 1;
    c->tile = getenv("SLDG_NO_TILE") ? 0 : (getenv("SLDG_FORCE_TILE") ? 2 : 1);
    c->trace_order = 2;
    c->vel_periodic = 0;
    if (cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        delete c;
        return SLDG_ECUDA;
    }
    for (int h = 0; h < SLDG_HIST; ++h)
        for (int k = 0; k < 8; ++k)
            if (cudaEventCreate(&c->hev[h][k]) != cudaSuccess) {
                sldg_destroy(c);
                return SLDG_ECUDA;
            }
    use_history_slot(c, 0);
    for (int k = 0; k < 2; ++k)
        if (cudaEventCreate(&c->cev[k]) != cudaSuccess) {
            sldg_destroy(c);
            return SLDG_ECUDA;
        }
    if (cudaStreamCreateWithFlags(&c->cstream, cudaStreamNonBlocking) != cudaSuccess) {
        sldg_destroy(c);
        return SLDG_ECUDA;
    }
    for (int k = 0; k < SLDG_EZ_CHUNKS; ++k)
        if (cudaEventCreateWithFlags(&c->ezev[k], cudaEventDisableTiming) != cudaSuccess) {
            sldg_destroy(c);
            return SLDG_ECUDA;
        }
    for (int k = 0; k < SLDG_RHO_CHUNKS; ++k)
        if (cudaEventCreateWithFlags(&c->rhoev[k], cudaEventDisableTiming) != cudaSuccess) {
            sldg_destroy(c);
            return SLDG_ECUDA;
        }
    // fields default to zero, error word cleared
    cudaError_t e = cudaMemsetAsync(ws + m.Ez, 0, m.hdr - m.Ez, c->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(c->err, 0, 256, c->stream);
    if (e != cudaSuccess) {
        sldg_destroy(c);
        return SLDG_ECUDA;
    }
    *out = c;
    return SLDG_OK;
}

int sldg_destroy(sldg_ctx *c)
{
    if (!c) return SLDG_EINVAL;
    for (int h = 0; h < SLDG_HIST; ++h)
        for (int k = 0; k < 8; ++k)
            if (c->hev[h][k]) cudaEventDestroy(c->hev[h][k]);
    if (c->cstream) {
        cudaStreamSynchronize(c->cstream);
        cudaStreamDestroy(c->cstream);
    }
    for (int k = 0; k < 2; ++k) {
        if (c->cev[k]) cudaEventDestroy(c->cev[k]);
    }
    for (int k = 0; k < SLDG_EZ_CHUNKS; ++k)
        if (c->ezev[k]) cudaEventDestroy(c->ezev[k]);
    for (int k = 0; k < SLDG_RHO_CHUNKS; ++k)
        if (c->rhoev[k]) cudaEventDestroy(c->rhoev[k]);
    delete c;
    return SLDG_OK;
}

double *sldg_current(sldg_ctx *c) { return c ? c->f[c->cur] : nullptr; }

int sldg_import_state(sldg_ctx *c, const double *f_canonical_dev)
{
    if (!c || !f_canonical_dev) return SLDG_EINVAL;
    return cuda_fail(launch_pack(c, f_canonical_dev, c->f[c->cur]));
}

int sldg_export_state(sldg_ctx *c, double *f_canonical_dev)
{
    if (!c || !f_canonical_dev) return SLDG_EINVAL;
    return cuda_fail(launch_unpack(c, c->f[c->cur], f_canonical_dev));
}

int sldg_import_state_host(sldg_ctx *c, const double *f_host)
{
    if (!c || !f_host) return SLDG_EINVAL;
    const GridDev &g = c->g;
    size_t bytes = (size_t)g.lines * g.N[3] * 8;
    double *stage = c->f[c->cur ^ 1];
    if (cudaMemcpyAsync(stage, f_host, bytes, cudaMemcpyHostToDevice, c->stream) != cudaSuccess) return SLDG_ECUDA;
    if (launch_pack(c, stage, c->f[c->cur]) != cudaSuccess) return SLDG_ECUDA;
    return cuda_fail(cudaStreamSynchronize(c->stream));
}

int sldg_export_state_host(sldg_ctx *c, double *f_host)
{
    if (!c || !f_host) return SLDG_EINVAL;
    const GridDev &g = c->g;
    size_t bytes = (size_t)g.lines * g.N[3] * 8;
    double *stage = c->f[c->cur ^ 1];
    if (launch_unpack(c, c->f[c->cur], stage) != cudaSuccess) return SLDG_ECUDA;
    if (cudaMemcpyAsync(f_host, stage, bytes, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess) return SLDG_ECUDA;
    return cuda_fail(cudaStreamSynchronize(c->stream));
}

int sldg_set_Ez(sldg_ctx *c, const double *Ez_dev)
{
    if (!c || !Ez_dev) return SLDG_EINVAL;
    return cuda_fail(cudaMemcpyAsync(c->Ez, Ez_dev, (size_t)c->g.lines * 8, cudaMemcpyDeviceToDevice, c->stream));
}

int sldg_set_vxy(sldg_ctx *c, const double *a_dev, const double *b_dev, int periodic)
{
    if (!c || !a_dev || !b_dev) return SLDG_EINVAL;
    const GridDev &g = c->g;
    size_t bytes = (size_t)g.N[2] * (g.n[0] + 1) * (g.n[1] + 1) * 8;
    c->vel_periodic = periodic == 2 ? 2 : (periodic ? 1 : 0);
    if (cudaMemcpyAsync(c->va, a_dev, bytes, cudaMemcpyDeviceToDevice, c->stream) != cudaSuccess) return SLDG_ECUDA;
    return cuda_fail(cudaMemcpyAsync(c->vb, b_dev, bytes, cudaMemcpyDeviceToDevice, c->stream));
}

int sldg_set_trace_order(sldg_ctx *c, int trace_order)
{
    if (!c || (trace_order != 1 && trace_order != 2)) return SLDG_EINVAL;
    c->trace_order = trace_order;
    return SLDG_OK;
}

static int do_z(sldg_ctx *c, double tau)
{
    cudaError_t e = launch_advect_z(c, c->f[c->cur], c->f[c->cur ^ 1], tau);
    if (e != cudaSuccess) return e == cudaErrorInvalidValue ? SLDG_EINVAL : SLDG_ECUDA;
    swap_state(c);
    return SLDG_OK;
}

static int do_v(sldg_ctx *c, double tau)
{
    cudaError_t e = launch_advect_v(c, c->f[c->cur], c->f[c->cur ^ 1], tau);
    if (e != cudaSuccess) return e == cudaErrorInvalidValue ? SLDG_EINVAL : SLDG_ECUDA;
    swap_state(c);
    return SLDG_OK;
}

// One pass over f for a pair of adjacent sweeps: the whole (z,v) plane in shared memory if it fits (fastest: 5.3-5.6
// TB/s at 128 KB planes), else z tiles with a halo when the Courant numbers of the z sweep are small (the paper's grid,
// 256 KB planes: 5.7 TB/s against 3.3 for the two separate kernels); cudaErrorNotSupported if neither applies.
// SLDG_FORCE_TILE (read at sldg_create) tries the tiles first: the tests use it to reach that kernel at small sizes.
static cudaError_t launch_pair(sldg_ctx *c, double tau, bool z_first)
{
    const double *fin = c->f[c->cur];
    double *fout = c->f[c->cur ^ 1];
    cudaError_t e = cudaErrorNotSupported;
    if (c->ez_chunks > 0 && z_first) {
        // sldg_strang_step_host: E_z is arriving on the copy stream in chunks of y rows; the planes of a chunk are
        // swept as soon as its rows are there (the caller checked that the whole-plane kernel takes this pair)
        const int nch = c->ez_chunks, Ny = c->g.N[1], Nx = c->g.N[0];
        c->ez_chunks = 0;
        for (int k = 0; k < nch; ++k) {
            const int y0 = (int)((long long)Ny * k / nch), y1 = (int)((long long)Ny * (k + 1) / nch);
            cudaStreamWaitEvent(c->stream, c->ezev[k], 0);
            e = launch_fused_sweeps(c, fin, fout, tau, tau, true, false, y0 * Nx, y1 * Nx);
            if (e != cudaSuccess) return e;
        }
        return e;
    }
    if (c->rho_chunks > 0 && !z_first) {
        // sldg_strang_step_host: the v,z pair in chunks of y rows; each launch also writes the charge density of its planes
        // (the caller checked that the kernel takes this pair), whose rows go down to the host on the copy stream -- strided
        // copies, rho is [Nz][Ny][Nx] -- under the next chunk's sweep
        const int nch = c->rho_chunks, Ny = c->g.N[1], Nx = c->g.N[0];
        const size_t pitch = (size_t)Ny * Nx * 8;
        c->rho_chunks = 0;
        for (int k = 0; k < nch; ++k) {
            const long long y0 = (long long)Ny * k / nch, y1 = (long long)Ny * (k + 1) / nch;
            e = launch_fused_sweeps(c, fin, fout, tau, tau, false, false, (int)(y0 * Nx), (int)(y1 * Nx), c->rho_ws);
            if (e != cudaSuccess) return e;
            cudaEventRecord(c->rhoev[k], c->stream);
            cudaStreamWaitEvent(c->cstream, c->rhoev[k], 0);
            e = cudaMemcpy2DAsync(c->rho_host + y0 * Nx, pitch, c->rho_ws + y0 * Nx, pitch, (size_t)(y1 - y0) * Nx * 8,
                                  (size_t)c->g.N[2], cudaMemcpyDeviceToHost, c->cstream);
            if (e != cudaSuccess) return e;
        }
        return e;
    }
    if (c->tile == 2) e = launch_tiled_sweeps(c, fin, fout, tau, tau, z_first);
    if (e == cudaErrorNotSupported) {
        cudaGetLastError();
        e = launch_fused_sweeps(c, fin, fout, tau, tau, z_first);
    }
    if (e == cudaErrorNotSupported && c->tile == 1) {
        cudaGetLastError();
        e = launch_tiled_sweeps(c, fin, fout, tau, tau, z_first);
    }
    return e;
}

// The two adjacent sweeps of a Strang step (Algorithm 1 steps 3,4 or 7,8) in one pass over f when the (z,v)
// plane of an (x,y) node fits in shared memory; *fused = 0 and the two separate kernels otherwise.
static int do_pair(sldg_ctx *c, double tau, bool z_first, cudaEvent_t mid, int *fused)
{
    *fused = 0;
    if (c->fuse) {
        cudaError_t e = launch_pair(c, tau, z_first);
        if (e == cudaSuccess) {
            swap_state(c);
            cudaEventRecord(mid, c->stream);
            *fused = 1;
            return SLDG_OK;
        }
        if (e != cudaErrorNotSupported) return SLDG_ECUDA;
        cudaGetLastError();
    }
    if (c->ez_pending && !z_first) {  // (not reached: the upload is only deferred ahead of a z,v pair)
        cudaStreamWaitEvent(c->stream, c->ezev[0], 0);
        c->ez_pending = 0;
    }
    int rc = z_first ? do_z(c, tau) : do_v(c, tau);
    if (rc) return rc;
    cudaEventRecord(mid, c->stream);
    if (c->ez_pending) {  // sldg_strang_step_host: E_z went up on the copy stream under the z sweep, which does not read it
        cudaStreamWaitEvent(c->stream, c->ezev[0], 0);
        c->ez_pending = 0;
    }
    return z_first ? do_v(c, tau) : do_z(c, tau);
}

// The geometry (once per z node) and the apply (every v) of one 2d step, back to back on the
// caller's stream.  (Running the ALU-bound geometry concurrently with the bandwidth-bound apply -- on a second
// stream with per-z counters, or as a prologue of every apply block -- was built and measured slower: DESIGN.md 6.3.)
static int do_xy(sldg_ctx *c, double tau, int trace_order)
{
    if (c->ab_pending) {  // a, b uploaded on the copy stream by sldg_strang_step_host
        cudaStreamWaitEvent(c->stream, c->cev[1], 0);
        c->ab_pending = 0;
    }
    cudaEventRecord(c->gev[0], c->stream);
    if (launch_xy_geometry(c, tau, trace_order) != cudaSuccess) return SLDG_ECUDA;
    cudaEventRecord(c->gev[1], c->stream);
    if (launch_xy_apply(c, c->f[c->cur], c->f[c->cur ^ 1]) != cudaSuccess) return SLDG_ECUDA;
    swap_state(c);
    return SLDG_OK;
}

int sldg_advect_z(sldg_ctx *c, double tau)
{
    if (!c) return SLDG_EINVAL;
    cudaEventRecord(c->ev[0], c->stream);
    int rc = do_z(c, tau);
    cudaEventRecord(c->ev[1], c->stream);
    c->ev_kind = 2;
    return rc;
}

int sldg_advect_v(sldg_ctx *c, double tau)
{
    if (!c) return SLDG_EINVAL;
    cudaEventRecord(c->ev[0], c->stream);
    int rc = do_v(c, tau);
    cudaEventRecord(c->ev[1], c->stream);
    c->ev_kind = 3;
    return rc;
}

int sldg_advect_xy(sldg_ctx *c, double tau, int trace_order)
{
    if (!c || (trace_order != 1 && trace_order != 2)) return SLDG_EINVAL;
    cudaEventRecord(c->ev[0], c->stream);
    int rc = do_xy(c, tau, trace_order);
    cudaEventRecord(c->ev[1], c->stream);
    c->ev_kind = 4;
    return rc;
}

int sldg_charge_density(sldg_ctx *c, double *rho_dev)
{
    if (!c || !rho_dev) return SLDG_EINVAL;
    return cuda_fail(launch_charge_density(c, c->f[c->cur], rho_dev));
}

int sldg_mass(sldg_ctx *c, double *mass_dev)
{
    if (!c || !mass_dev) return SLDG_EINVAL;
    return cuda_fail(launch_mass(c, c->f[c->cur], mass_dev));
}

int sldg_strang_step(sldg_ctx *c, double dt)
{
    if (!c) return SLDG_EINVAL;
    int rc;
    int fused0 = 0, fused1 = 0;
    use_history_slot(c, c->hpos);
    cudaEventRecord(c->ev[0], c->stream);
    if ((rc = do_pair(c, 0.5 * dt, true, c->ev[1], &fused0))) return rc;
    cudaEventRecord(c->ev[2], c->stream);
    if ((rc = do_xy(c, dt, c->trace_order))) return rc;
    cudaEventRecord(c->ev[3], c->stream);
    if ((rc = do_pair(c, 0.5 * dt, false, c->ev[4], &fused1))) return rc;
    cudaEventRecord(c->ev[5], c->stream);
    c->last_fused = (fused0 ? 2 : 0) + (fused1 ? 4 : 0);
    c->ev_kind = 1;
    c->hist_fused[c->hpos] = c->last_fused;
    c->hpos = (c->hpos + 1) % SLDG_HIST;
    c->hcount++;
    c->last_slot = (c->hpos + SLDG_HIST - 1) % SLDG_HIST;
    use_history_slot(c, c->hpos);  // single substep calls that follow record into the next slot, not over this step's
    return SLDG_OK;
}

int sldg_strang_step_host(sldg_ctx *c, double dt, const double *Ez_host, const double *a_host,
                          const double *b_host, int periodic, double *rho_host, double *mass_host)
{
    if (!c) return SLDG_EINVAL;
    if ((a_host == nullptr) != (b_host == nullptr)) return SLDG_EINVAL;
    const GridDev &g = c->g;
    double *rho_dev = c->rho_ws;
    double *mass_dev = c->scalar_ws;
    // E_z is first needed by the v sweep of the z,v pair.  Where that pair runs as the whole-plane kernel (one pass over the
    // (z,v) planes in the order of (y,x)), E_z goes up on the copy stream in chunks of y rows -- strided copies, E_z is
    // [Nz][Ny][Nx] -- and the planes of a chunk are swept as soon as its rows have arrived (launch_pair): only the first
    // chunk's upload is exposed.  Otherwise one copy on the caller's stream ahead of the step.
    const bool ez_chunked = Ez_host && c->fuse && c->tile != 2 && g.N[1] >= SLDG_EZ_CHUNKS && fused_sweeps_supported(c, true);
    // Where the z,v pair is certain to run as two kernels (no fused pairs, or the plane does not fit and the z-tiled kernel
    // does not take this order), the z sweep does not read E_z: one copy on the copy stream under it, the v sweep waits.
    static const bool force_tile = getenv("SLDG_FORCE_TILE") != nullptr;
    const bool ez_deferred = Ez_host && !ez_chunked &&
                             (!c->fuse || (!fused_sweeps_supported(c, true) && (c->tile == 0 || (g.o[2] == 3 && !force_tile))));
    if (Ez_host && !ez_chunked && !ez_deferred &&
        cudaMemcpyAsync(c->Ez, Ez_host, (size_t)g.lines * 8, cudaMemcpyHostToDevice, c->stream) != cudaSuccess)
        return SLDG_ECUDA;
    if (ez_chunked || ez_deferred || a_host) {
        cudaEventRecord(c->cev[0], c->stream);
        cudaStreamWaitEvent(c->cstream, c->cev[0], 0);
    }
    if (ez_deferred) {
        if (cudaMemcpyAsync(c->Ez, Ez_host, (size_t)g.lines * 8, cudaMemcpyHostToDevice, c->cstream) != cudaSuccess)
            return SLDG_ECUDA;
        cudaEventRecord(c->ezev[0], c->cstream);
        c->ez_pending = 1;
    }
    if (ez_chunked) {
        const size_t pitch = (size_t)g.N[1] * g.N[0] * 8;
        for (int k = 0; k < SLDG_EZ_CHUNKS; ++k) {
            const long long y0 = (long long)g.N[1] * k / SLDG_EZ_CHUNKS, y1 = (long long)g.N[1] * (k + 1) / SLDG_EZ_CHUNKS;
            if (cudaMemcpy2DAsync(c->Ez + y0 * g.N[0], pitch, Ez_host + y0 * g.N[0], pitch, (size_t)(y1 - y0) * g.N[0] * 8,
                                  (size_t)g.N[2], cudaMemcpyHostToDevice, c->cstream) != cudaSuccess)
                return SLDG_ECUDA;
            cudaEventRecord(c->ezev[k], c->cstream);
        }
        c->ez_chunks = SLDG_EZ_CHUNKS;
    }
    if (a_host) {
        size_t bytes = (size_t)g.N[2] * (g.n[0] + 1) * (g.n[1] + 1) * 8;
        c->vel_periodic = periodic == 2 ? 2 : (periodic ? 1 : 0);
        // a, b are first needed by the 2d step: their upload runs on the copy stream under the z and v sweeps
        if (cudaMemcpyAsync(c->va, a_host, bytes, cudaMemcpyHostToDevice, c->cstream) != cudaSuccess) return SLDG_ECUDA;
        if (cudaMemcpyAsync(c->vb, b_host, bytes, cudaMemcpyHostToDevice, c->cstream) != cudaSuccess) return SLDG_ECUDA;
        cudaEventRecord(c->cev[1], c->cstream);
        c->ab_pending = 1;
    }
    // rho: where the v,z pair runs as the whole-plane kernel at o = 2, that kernel forms the charge density from its own
    // results (no further pass over f) and is launched in chunks of y rows, the download of a chunk's rows under the next
    // chunk (launch_pair); otherwise a reduction over f in slabs of z after the step, downloads under the next slab.  The
    // two differ in the order of the v sum (last bits).
    const bool rho_fused = rho_host && c->fuse && c->tile != 2 && g.N[1] >= SLDG_RHO_CHUNKS && fused_sweeps_supported(c, false, true);
    if (rho_fused) {
        c->rho_chunks = SLDG_RHO_CHUNKS;
        c->rho_host = rho_host;
    }
    int rc = sldg_strang_step(c, dt);
    c->rho_chunks = 0;
    c->ez_pending = 0;
    if (rc) return rc;
    if (rho_fused) {
        cudaEventRecord(c->cev[0], c->cstream);
        cudaStreamWaitEvent(c->stream, c->cev[0], 0);  // the caller's stream sees the downloads complete
    } else if (rho_host) {
        // rho in slabs of z: the download of a slab (copy stream) runs under the reduction of the next one
        const int nslab = g.N[2] < 8 ? g.N[2] : 8;
        const long long per_z = (long long)g.N[1] * g.N[0];
        for (int k = 0; k < nslab; ++k) {
            const long long l0 = (long long)g.N[2] * k / nslab * per_z, l1 = (long long)g.N[2] * (k + 1) / nslab * per_z;
            if (launch_charge_density(c, c->f[c->cur], rho_dev, l0, l1) != cudaSuccess) return SLDG_ECUDA;
            cudaEventRecord(c->cev[0], c->stream);
            cudaStreamWaitEvent(c->cstream, c->cev[0], 0);
            if (cudaMemcpyAsync(rho_host + l0, rho_dev + l0, (size_t)(l1 - l0) * 8, cudaMemcpyDeviceToHost, c->cstream) != cudaSuccess)
                return SLDG_ECUDA;
        }
        cudaEventRecord(c->cev[0], c->cstream);
        cudaStreamWaitEvent(c->stream, c->cev[0], 0);  // the caller's stream sees the downloads complete
    } else if (mass_host) {
        if (launch_charge_density(c, c->f[c->cur], rho_dev) != cudaSuccess) return SLDG_ECUDA;
    }
    if (mass_host) {
        if (launch_mass_from_rho(c, rho_dev, mass_dev) != cudaSuccess) return SLDG_ECUDA;
        if (cudaMemcpyAsync(mass_host, mass_dev, 8, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess) return SLDG_ECUDA;
    }
    return cuda_fail(cudaStreamSynchronize(c->stream));
}

int sldg_check(sldg_ctx *c)
{
    if (!c) return SLDG_EINVAL;
    int32_t word = 0;
    if (cudaMemcpyAsync(&word, c->err, 4, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess) return SLDG_ECUDA;
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return SLDG_ECUDA;
    if (cudaGetLastError() != cudaSuccess) return SLDG_ECUDA;
    if (word != 0) cudaMemsetAsync(c->err, 0, 4, c->stream);
    return (int)word;
}

int sldg_last_timing_ms(sldg_ctx *c, float ms[8])
{
    if (!c || !ms) return SLDG_EINVAL;
    for (int k = 0; k < 8; ++k) ms[k] = 0.0f;
    if (c->ev_kind == 0) return SLDG_OK;
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return SLDG_ECUDA;
    cudaEvent_t *E = c->ev_kind == 1 ? c->hev[c->last_slot] : c->ev;  // a Strang step's events sit in its history slot
    auto el = [&](int a, int b) {
        float t = 0.0f;
        cudaEventElapsedTime(&t, E[a], E[b]);
        return t;
    };
    auto geom = [&]() { return el(6, 7); };
    if (c->ev_kind == 1) {
        ms[0] = el(0, 1); ms[1] = el(1, 2); ms[3] = el(2, 3); ms[4] = el(3, 4); ms[5] = el(4, 5);
        ms[2] = geom();
        ms[6] = (float)c->last_fused;
        ms[7] = el(0, 5);
    } else if (c->ev_kind == 2) {
        ms[0] = ms[7] = el(0, 1);
    } else if (c->ev_kind == 3) {
        ms[1] = ms[7] = el(0, 1);
    } else if (c->ev_kind == 4) {
        ms[2] = geom();
        ms[3] = ms[7] = el(0, 1);
    } else if (c->ev_kind == 5) {
        ms[7] = el(0, 1);
    }
    return SLDG_OK;
}

int sldg_timing_history(sldg_ctx *c, int n, float *ms)
{
    if (!c || !ms || n < 1 || n > SLDG_HIST || n > c->hcount) return SLDG_EINVAL;
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return SLDG_ECUDA;
    for (int i = 0; i < n; ++i) {
        const int h = (c->hpos + SLDG_HIST - n + i) % SLDG_HIST;  // oldest first
        cudaEvent_t *e = c->hev[h];
        float *o = ms + 8 * i, t = 0.0f;
        auto el = [&](int a, int b) {
            cudaEventElapsedTime(&t, e[a], e[b]);
            return t;
        };
        o[0] = el(0, 1); o[1] = el(1, 2); o[2] = el(6, 7); o[3] = el(2, 3); o[4] = el(3, 4); o[5] = el(4, 5);
        o[6] = (float)c->hist_fused[h];
        o[7] = el(0, 5);
    }
    return SLDG_OK;
}

long long sldg_launch_count(sldg_ctx *c) { return c ? c->launches : 0; }

// ---- field step, invariants, Algorithms 1 and 2 --------------------------------------------------------------

int sldg_set_profiles(sldg_ctx *c, const double *n0_dev, const double *Te_dev, double B)
{
    if (!c || !n0_dev || !Te_dev || !(B != 0.0)) return SLDG_EINVAL;
    const size_t bytes = (size_t)c->g.n[0] * c->g.n[1] * 8;
    if (cudaMemcpyAsync(c->fld.n0, n0_dev, bytes, cudaMemcpyDeviceToDevice, c->stream) != cudaSuccess) return SLDG_ECUDA;
    if (cudaMemcpyAsync(c->fld.Te, Te_dev, bytes, cudaMemcpyDeviceToDevice, c->stream) != cudaSuccess) return SLDG_ECUDA;
    c->fld.invB = 1.0 / B;
    c->fld.have_profiles = 1;
    return SLDG_OK;
}

int sldg_field_step(sldg_ctx *c, double tol, int max_iter)
{
    if (!c || !c->fld.have_profiles || !(tol > 0.0) || max_iter < 1) return SLDG_EINVAL;
    return cuda_fail(launch_field_step(c, c->f[c->cur], tol, max_iter));
}

int sldg_field_info(sldg_ctx *c, int *max_iters_host, double *max_relres_host)
{
    if (!c || !c->fld.have_phi) return SLDG_EINVAL;
    const int n = c->g.N[2] + 1;
    std::vector<int> it(n);
    std::vector<double> rr(n);
    if (cudaMemcpyAsync(it.data(), c->fld.iters, n * 4, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess) return SLDG_ECUDA;
    if (cudaMemcpyAsync(rr.data(), c->fld.relres, n * 8, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess) return SLDG_ECUDA;
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return SLDG_ECUDA;
    int mi = 0;
    double mr = 0.0;
    for (int k = 0; k < n; ++k) {
        mi = it[k] > mi ? it[k] : mi;
        mr = rr[k] > mr ? rr[k] : mr;
    }
    if (max_iters_host) *max_iters_host = mi;
    if (max_relres_host) *max_relres_host = mr;
    return SLDG_OK;
}

int sldg_get_phi(sldg_ctx *c, double *phi_dev)
{
    if (!c || !phi_dev || !c->fld.have_phi) return SLDG_EINVAL;
    const size_t bytes = (size_t)c->g.N[2] * c->g.n[0] * c->g.n[1] * 8;
    return cuda_fail(cudaMemcpyAsync(phi_dev, c->fld.phi, bytes, cudaMemcpyDeviceToDevice, c->stream));
}

int sldg_get_fields(sldg_ctx *c, double *Ez_dev, double *a_dev, double *b_dev)
{
    if (!c) return SLDG_EINVAL;
    const GridDev &g = c->g;
    const size_t vb = (size_t)g.N[2] * (g.n[0] + 1) * (g.n[1] + 1) * 8;
    if (Ez_dev && cudaMemcpyAsync(Ez_dev, c->Ez, (size_t)g.lines * 8, cudaMemcpyDeviceToDevice, c->stream) != cudaSuccess)
        return SLDG_ECUDA;
    if (a_dev && cudaMemcpyAsync(a_dev, c->va, vb, cudaMemcpyDeviceToDevice, c->stream) != cudaSuccess) return SLDG_ECUDA;
    if (b_dev && cudaMemcpyAsync(b_dev, c->vb, vb, cudaMemcpyDeviceToDevice, c->stream) != cudaSuccess) return SLDG_ECUDA;
    return SLDG_OK;
}

int sldg_diagnostics(sldg_ctx *c, double r_p, double out_host[5])
{
    if (!c || !out_host || !c->fld.have_phi) return SLDG_EINVAL;
    return cuda_fail(launch_diagnostics(c, c->f[c->cur], r_p, out_host));
}

int sldg_step_algorithm1(sldg_ctx *c, double dt, double tol, int max_iter)
{
    int rc, fused;
    if ((rc = sldg_field_step(c, tol, max_iter))) return rc;
    if ((rc = do_pair(c, 0.5 * dt, true, c->ev[1], &fused))) return rc;
    if ((rc = sldg_field_step(c, tol, max_iter))) return rc;
    if ((rc = do_xy(c, dt, 2))) return rc;
    if ((rc = do_pair(c, 0.5 * dt, false, c->ev[4], &fused))) return rc;
    c->ev_kind = 0;
    return SLDG_OK;
}

// ---- source term of the delta-g formulation ----------------------------------------

int sldg_set_equilibrium(sldg_ctx *c, const double *dv_geq_dev, const double *dr_geq_dev)
{
    if (!c || !dv_geq_dev || !dr_geq_dev) return SLDG_EINVAL;
    c->src_ready |= 1;
    return cuda_fail(launch_source_profiles(c, dv_geq_dev, dr_geq_dev));
}

int sldg_set_source_fields(sldg_ctx *c, const double *dz_phi_dev, const double *dtheta_phi_dev)
{
    if (!c || !dz_phi_dev || !dtheta_phi_dev) return SLDG_EINVAL;
    const size_t bytes = (size_t)c->g.lines * 8;
    if (cudaMemcpyAsync(c->src_dz, dz_phi_dev, bytes, cudaMemcpyDeviceToDevice, c->stream) != cudaSuccess) return SLDG_ECUDA;
    if (cudaMemcpyAsync(c->src_dth, dtheta_phi_dev, bytes, cudaMemcpyDeviceToDevice, c->stream) != cudaSuccess) return SLDG_ECUDA;
    c->src_ready |= 2;
    return SLDG_OK;
}

int sldg_source_step(sldg_ctx *c, double tau)
{
    if (!c || c->src_ready != 3) return SLDG_EINVAL;
    cudaEventRecord(c->ev[0], c->stream);
    cudaError_t e = launch_source_step(c, c->f[c->cur], tau);
    cudaEventRecord(c->ev[1], c->stream);
    c->ev_kind = 5;
    return cuda_fail(e);
}

int sldg_strang_step_sources(sldg_ctx *c, double dt)
{
    if (!c || c->src_ready != 3) return SLDG_EINVAL;
    int rc;
    if (launch_source_step(c, c->f[c->cur], 0.5 * dt) != cudaSuccess) return SLDG_ECUDA;
    if ((rc = sldg_strang_step(c, dt))) return rc;
    return cuda_fail(launch_source_step(c, c->f[c->cur], 0.5 * dt));
}

int sldg_set_polar_profiles(sldg_ctx *c, const double *r_n0_dev, const double *dln_n0_dev, const double *Te_dev)
{
    if (!c || !r_n0_dev || !dln_n0_dev || !Te_dev || c->g.n[0] < 3) return SLDG_EINVAL;
    return cuda_fail(launch_polar_profiles(c, r_n0_dev, dln_n0_dev, Te_dev));
}

int sldg_polar_field_step(sldg_ctx *c)
{
    if (!c || !c->pol.ready) return SLDG_EINVAL;
    return cuda_fail(launch_polar_field_step(c, c->f[c->cur]));
}

int sldg_get_polar_phi(sldg_ctx *c, double *phi_dev)
{
    if (!c || !phi_dev || !c->pol.have_phi) return SLDG_EINVAL;
    const size_t bytes = (size_t)c->g.N[2] * c->g.n[1] * (c->g.n[0] + 1) * 8;
    return cuda_fail(cudaMemcpyAsync(phi_dev, c->pol.phi, bytes, cudaMemcpyDeviceToDevice, c->stream));
}

int sldg_get_source_fields(sldg_ctx *c, double *dz_phi_dev, double *dtheta_phi_dev)
{
    if (!c || !(c->src_ready & 2)) return SLDG_EINVAL;
    const size_t bytes = (size_t)c->g.lines * 8;
    if (dz_phi_dev && cudaMemcpyAsync(dz_phi_dev, c->src_dz, bytes, cudaMemcpyDeviceToDevice, c->stream) != cudaSuccess) return SLDG_ECUDA;
    if (dtheta_phi_dev && cudaMemcpyAsync(dtheta_phi_dev, c->src_dth, bytes, cudaMemcpyDeviceToDevice, c->stream) != cudaSuccess) return SLDG_ECUDA;
    return SLDG_OK;
}

int sldg_step_algorithm1_polar(sldg_ctx *c, double dt)
{
    if (!c || !c->pol.ready || !(c->src_ready & 1)) return SLDG_EINVAL;
    int rc, fused;
    if ((rc = sldg_polar_field_step(c))) return rc;                                          // 1
    if (launch_source_step(c, c->f[c->cur], 0.5 * dt) != cudaSuccess) return SLDG_ECUDA;     // 2
    if ((rc = do_pair(c, 0.5 * dt, true, c->ev[1], &fused))) return rc;                       // 3, 4
    if ((rc = sldg_polar_field_step(c))) return rc;                                          // 5
    if ((rc = do_xy(c, dt, 2))) return rc;                                                    // 6
    if ((rc = do_pair(c, 0.5 * dt, false, c->ev[4], &fused))) return rc;                      // 7, 8
    if (launch_source_step(c, c->f[c->cur], 0.5 * dt) != cudaSuccess) return SLDG_ECUDA;     // 9
    c->ev_kind = 0;
    return SLDG_OK;
}

int sldg_set_third_buffer(sldg_ctx *c, double *f_c_dev)
{
    if (!c || !f_c_dev || ((uintptr_t)f_c_dev & 255) || f_c_dev == c->f[0] || f_c_dev == c->f[1]) return SLDG_EINVAL;
    c->f_c = f_c_dev;
    return SLDG_OK;
}

// Algorithm 2 writes every substep into a buffer that is neither its source nor `keep` (the state of level n while the
// corrector still needs it): the spare buffer takes the place of the context's idle ping-pong buffer when necessary.
static void aim_away_from(sldg_ctx *c, const double *keep)
{
    if (c->f[c->cur ^ 1] == keep) {
        double *t = c->f[c->cur ^ 1];
        c->f[c->cur ^ 1] = c->f_c;
        c->f_c = t;
    }
}

static int pair_keeping(sldg_ctx *c, double tau, bool z_first, const double *keep)
{
    aim_away_from(c, keep);
    if (c->fuse) {
        cudaError_t e = launch_pair(c, tau, z_first);
        if (e == cudaSuccess) {
            swap_state(c);
            return SLDG_OK;
        }
        if (e != cudaErrorNotSupported) return SLDG_ECUDA;
        cudaGetLastError();
    }
    int rc = z_first ? do_z(c, tau) : do_v(c, tau);
    if (rc) return rc;
    aim_away_from(c, keep);
    return z_first ? do_v(c, tau) : do_z(c, tau);
}

int sldg_step_algorithm2(sldg_ctx *c, double dt, double tol, int max_iter)
{
    if (!c || !c->f_c) return SLDG_EINVAL;
    int rc;
    double *fn = c->f[c->cur];  // the state of time level n
    if ((rc = sldg_field_step(c, tol, max_iter))) return rc;
    // predictor with phi^n: first-order tracing over dt/2
    if ((rc = pair_keeping(c, 0.5 * dt, true, fn))) return rc;
    aim_away_from(c, fn);
    if ((rc = do_xy(c, 0.5 * dt, 1))) return rc;
    if ((rc = sldg_field_step(c, tol, max_iter))) return rc;  // phi^{n+1/2}
    // corrector: start again from level n; the predicted state is dead, level n after its first read
    if (c->f[0] == fn) c->cur = 0;
    else if (c->f[1] == fn) c->cur = 1;
    else {  // level n sits in the spare slot: exchange it with the predicted state
        c->f_c = c->f[c->cur];
        c->f[c->cur] = fn;
    }
    if ((rc = pair_keeping(c, 0.5 * dt, true, nullptr))) return rc;
    if ((rc = do_xy(c, dt, 2))) return rc;
    if ((rc = pair_keeping(c, 0.5 * dt, false, nullptr))) return rc;
    c->ev_kind = 0;
    return SLDG_OK;
}

int sldg_step_algorithm2_polar(sldg_ctx *c, double dt)
{
    if (!c || !c->f_c || !c->pol.ready || !(c->src_ready & 1)) return SLDG_EINVAL;
    int rc;
    double *fn = c->f[c->cur];  // delta g of time level n
    if ((rc = sldg_polar_field_step(c))) return rc;                                                    // 1  phi^n
    // predictor: the source step writes into another buffer, level n stays untouched
    aim_away_from(c, fn);
    if (launch_source_step(c, c->f[c->cur ^ 1], 0.5 * dt, fn) != cudaSuccess) return SLDG_ECUDA;       // 2
    swap_state(c);
    if ((rc = pair_keeping(c, 0.5 * dt, true, fn))) return rc;                                         // 3, 4
    aim_away_from(c, fn);
    if ((rc = do_xy(c, 0.5 * dt, 1))) return rc;                                                       // 5  eq. (14)
    if ((rc = sldg_polar_field_step(c))) return rc;                                                    // 6  phi^{n+1/2}
    // corrector from level n
    if (c->f[0] == fn) c->cur = 0;
    else if (c->f[1] == fn) c->cur = 1;
    else {
        c->f_c = c->f[c->cur];
        c->f[c->cur] = fn;
    }
    if (launch_source_step(c, c->f[c->cur], 0.5 * dt) != cudaSuccess) return SLDG_ECUDA;               // 7
    if ((rc = pair_keeping(c, 0.5 * dt, true, nullptr))) return rc;                                    // 8, 9
    if ((rc = do_xy(c, dt, 2))) return rc;                                                             // 10 eq. (15)
    if ((rc = pair_keeping(c, 0.5 * dt, false, nullptr))) return rc;                                   // 11, 12
    if (launch_source_step(c, c->f[c->cur], 0.5 * dt) != cudaSuccess) return SLDG_ECUDA;               // 13
    c->ev_kind = 0;
    return SLDG_OK;
}

int sldg_debug_geometry(sldg_ctx *c, int z, int32_t *anchor_dev, int32_t *mask_dev, double *W_dev)
{
    if (!c || z < 0 || z >= c->g.N[2]) return SLDG_EINVAL;
    return cuda_fail(launch_geometry_expand(c, z, anchor_dev, mask_dev, W_dev));
}

int sldg_debug_counter(sldg_ctx *c, int which, long long *value_host)
{
    if (!c || !value_host || which < 0 || which > 1) return SLDG_EINVAL;
    if (which == 1) return cuda_fail(count_weight_blocks(c, value_host));
    int32_t word = 0;
    if (cudaMemcpyAsync(&word, c->err + 1 + which, 4, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess) return SLDG_ECUDA;
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return SLDG_ECUDA;
    *value_host = word;
    return SLDG_OK;
}

const char *sldg_strerror(int code)
{
    switch (code) {
        case SLDG_OK: return "ok";
        case SLDG_EINVAL: return "invalid argument";
        case SLDG_ECUDA: return "CUDA error or no device";
        case SLDG_ESTENCIL: return "upstream cell exceeds the 3x3 stencil";
        case SLDG_EGEOM: return "degenerate upstream geometry (crossed characteristics or singular Vandermonde)";
        default: return "unknown error";
    }
}

}  // extern "C"
