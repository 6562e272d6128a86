/*
 * sldg_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct CPU implementation (fp64) of what the SLDG hot path computes,
 * written from the paper (arxiv 2212.03036, Einkemmer & Moriggl; cited below as PAPER.md:LINE) and from
 * the readings listed in DESIGN.md / SURVEY.md section 8(c).  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code, header, table or
 * constant generator with the CUDA library under paper_2212_03036_b200/csrc/.
 *
 * Every substep is implemented as its DEFINITION ("exact transport of the piecewise polynomial by the
 * flow map, followed by the cell-wise L2 projection"), in the paper's order, with no blocking, fusion
 * or reordering:
 *   1d (eq. 10-11): A(alpha), B(alpha) are the overlap integrals of the shifted
 *       Lagrange basis, evaluated with an o-point Gauss rule on each of the two sub-intervals (exact).
 *   2d (eq. 13, 16-18): corner feet -> upstream quadrilateral; node feet -> Vandermonde
 *       solve for phi*; Sutherland-Hodgman clip of the quadrilateral against each Eulerian cell; the
 *       integral (18) over each piece by fan triangulation and a collapsed tensor Gauss rule (exact).
 *       The paper evaluates the same integral through Green's theorem; the integral
 *       is unique, so the oracle deliberately uses area quadrature instead.
 *   charge density and mass: Gauss-Legendre weighted sums.
 *
 * Parity pins (tests/test_oracle_*.py): every function below is pinned; see DESIGN.md "Oracle pins".
 *
 * Canonical layouts: f[Nz][Nv][Ny][Nx], Ez[Nz][Ny][Nx], a,b[Nz][ny+1][nx+1]; N. = n. * order.
 * DOF index along an axis = cell*order + node; node coordinate = lo + (cell + xi_node) * h.
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define MAXO 4            /* nodes per cell per axis supported by the oracle (paper uses 2) */
#define MAXO2 (MAXO * MAXO)
#define MAXGL 16

typedef struct {
    int32_t n[4];      /* cells in x, y, z, v */
    int32_t order[4];  /* nodes per cell per axis */
    double lo[4], hi[4];
} sldg_oracle_grid;

enum { ORACLE_OK = 0, ORACLE_EINVAL = -1, ORACLE_EGEOM = -4, ORACLE_ENOMEM = -5 };

/* ------------------------------------------------------------------------------------------------
 * Gauss-Legendre rule on (0,1), weights sum to 1 (the DG nodes).
 * Newton iteration on the Legendre three-term recurrence.
 * ---------------------------------------------------------------------------------------------- */
void sldg_oracle_gl(int n, double *x, double *w)
{
    for (int k = 0; k < n; ++k) {
        double t = cos(M_PI * (k + 0.75) / (n + 0.5));
        double dp = 1.0;
        for (int it = 0; it < 100; ++it) {
            double p0 = 1.0, p1 = t;
            for (int j = 2; j <= n; ++j) {
                double p2 = ((2.0 * j - 1.0) * t * p1 - (j - 1.0) * p0) / j;
                p0 = p1;
                p1 = p2;
            }
            if (n == 0) p1 = 1.0;
            dp = n * (t * p1 - p0) / (t * t - 1.0);
            double dt = p1 / dp;
            t -= dt;
            if (fabs(dt) < 1e-17) break;
        }
        /* recompute derivative at the converged root */
        {
            double p0 = 1.0, p1 = t;
            for (int j = 2; j <= n; ++j) {
                double p2 = ((2.0 * j - 1.0) * t * p1 - (j - 1.0) * p0) / j;
                p0 = p1;
                p1 = p2;
            }
            dp = n * (t * p1 - p0) / (t * t - 1.0);
        }
        /* roots come out descending in t; store ascending on (0,1) */
        x[n - 1 - k] = 0.5 * (t + 1.0);
        w[n - 1 - k] = 1.0 / ((1.0 - t * t) * dp * dp); /* = (2/((1-t^2) P'^2)) / 2 */
    }
    if (n == 1) { x[0] = 0.5; w[0] = 1.0; }
}

/* Lagrange basis function j on the nodes x[0..o-1], evaluated at xi. */
static double lagrange(int o, const double *x, int j, double xi)
{
    double v = 1.0;
    for (int i = 0; i < o; ++i)
        if (i != j) v *= (xi - x[i]) / (x[j] - x[i]);
    return v;
}

/* ------------------------------------------------------------------------------------------------
 * 1d SLDG overlap matrices (eq. 10-11; reading A1 of SURVEY.md 8(c)-1):
 *   A_jm(alpha) = (1/w_j) int_0^{1-alpha} l_j(xi) l_m(xi+alpha)   dxi
 *   B_jm(alpha) = (1/w_j) int_{1-alpha}^1 l_j(xi) l_m(xi+alpha-1) dxi
 * Integrands have degree 2o-2: the o-point Gauss rule mapped to each sub-interval is exact.
 * Row-major o x o.
 * ---------------------------------------------------------------------------------------------- */
void sldg_oracle_shift_matrices(int o, double alpha, double *A, double *B)
{
    double x[MAXGL], w[MAXGL];
    sldg_oracle_gl(o, x, w);
    for (int j = 0; j < o; ++j)
        for (int m = 0; m < o; ++m) {
            double sa = 0.0, sb = 0.0;
            for (int q = 0; q < o; ++q) {
                double xi = (1.0 - alpha) * x[q];
                sa += (1.0 - alpha) * w[q] * lagrange(o, x, j, xi) * lagrange(o, x, m, xi + alpha);
            }
            for (int q = 0; q < o; ++q) {
                double xi = (1.0 - alpha) + alpha * x[q];
                sb += alpha * w[q] * lagrange(o, x, j, xi) * lagrange(o, x, m, xi + alpha - 1.0);
            }
            A[j * o + m] = sa / w[j];
            B[j * o + m] = sb / w[j];
        }
}

static int wrap(int i, int n)
{
    int r = i % n;
    return r < 0 ? r + n : r;
}

/* Courant number delta = speed*tau/h  ->  s = floor(-delta), alpha = -delta - s in [0,1):
 * the foot of the left edge of cell i lies in cell i+s at offset alpha. */
static void shift_of(double speed, double tau, double h, int *s, double *alpha)
{
    double delta = speed * tau / h;
    double fl = floor(-delta);
    *s = (int)fl;
    *alpha = -delta - fl;
}

/* One periodic line: u+[i,j] = sum_m A_jm u[(i+s) mod n, m] + B_jm u[(i+s+1) mod n, m]  (eq. 11).
 * `stride` is the distance (in doubles) between consecutive DOFs of the line. */
static void shift_line(int n, int o, int s, const double *A, const double *B,
                       const double *in, double *out, ptrdiff_t stride)
{
    for (int i = 0; i < n; ++i) {
        int c0 = wrap(i + s, n), c1 = wrap(i + s + 1, n);
        for (int j = 0; j < o; ++j) {
            double acc = 0.0;
            for (int m = 0; m < o; ++m)
                acc += A[j * o + m] * in[(ptrdiff_t)(c0 * o + m) * stride] +
                       B[j * o + m] * in[(ptrdiff_t)(c1 * o + m) * stride];
            out[(ptrdiff_t)(i * o + j) * stride] = acc;
        }
    }
}

/* Stand-alone periodic line shift (used by the pins): delta = Courant number a*tau/h. */
void sldg_oracle_shift_line(int n, int o, double delta, const double *in, double *out)
{
    double A[MAXO2], B[MAXO2];
    int s;
    double alpha;
    shift_of(delta, 1.0, 1.0, &s, &alpha);
    sldg_oracle_shift_matrices(o, alpha, A, B);
    shift_line(n, o, s, A, B, in, out, 1);
}

/* ------------------------------------------------------------------------------------------------
 * z-advection (eq. 4): speed = the v NODE value (reading A2), periodic in z.
 * ---------------------------------------------------------------------------------------------- */
int sldg_oracle_advect_z(const sldg_oracle_grid *g, const double *fin, double *fout, double tau)
{
    const int ox = g->order[0], oy = g->order[1], oz = g->order[2], ov = g->order[3];
    const int Nx = g->n[0] * ox, Ny = g->n[1] * oy, Nv = g->n[3] * ov;
    const int nz = g->n[2];
    if (oz > MAXO || ov > MAXO) return ORACLE_EINVAL;
    const double hz = (g->hi[2] - g->lo[2]) / g->n[2];
    const double hv = (g->hi[3] - g->lo[3]) / g->n[3];
    double xv[MAXGL], wv[MAXGL];
    sldg_oracle_gl(ov, xv, wv);
    const ptrdiff_t plane = (ptrdiff_t)Ny * Nx;
    const ptrdiff_t zstride = (ptrdiff_t)Nv * plane;
#pragma omp parallel for schedule(static)
    for (int V = 0; V < Nv; ++V) {
        int l = V / ov, q = V % ov;
        double vq = g->lo[3] + (l + xv[q]) * hv;
        int s;
        double alpha, A[MAXO2], B[MAXO2];
        shift_of(vq, tau, hz, &s, &alpha);
        sldg_oracle_shift_matrices(oz, alpha, A, B);
        for (ptrdiff_t yx = 0; yx < plane; ++yx)
            shift_line(nz, oz, s, A, B, fin + V * plane + yx, fout + V * plane + yx, zstride);
    }
    return ORACLE_OK;
}

/* ------------------------------------------------------------------------------------------------
 * v-advection (eq. 5): speed = Ez = -d(phi)/dz at each (x,y,z) node (reading A3),
 * periodic in v (reading A4).
 * ---------------------------------------------------------------------------------------------- */
int sldg_oracle_advect_v(const sldg_oracle_grid *g, const double *fin, const double *Ez, double *fout,
                         double tau)
{
    const int ox = g->order[0], oy = g->order[1], oz = g->order[2], ov = g->order[3];
    const int Nx = g->n[0] * ox, Ny = g->n[1] * oy, Nz = g->n[2] * oz, Nv = g->n[3] * ov;
    const int nv = g->n[3];
    if (ov > MAXO) return ORACLE_EINVAL;
    const double hv = (g->hi[3] - g->lo[3]) / g->n[3];
    const ptrdiff_t plane = (ptrdiff_t)Ny * Nx;
#pragma omp parallel for schedule(static)
    for (int Z = 0; Z < Nz; ++Z)
        for (ptrdiff_t yx = 0; yx < plane; ++yx) {
            int s;
            double alpha, A[MAXO2], B[MAXO2];
            shift_of(Ez[Z * plane + yx], tau, hv, &s, &alpha);
            sldg_oracle_shift_matrices(ov, alpha, A, B);
            shift_line(nv, ov, s, A, B, fin + (ptrdiff_t)Z * Nv * plane + yx,
                       fout + (ptrdiff_t)Z * Nv * plane + yx, plane);
        }
    return ORACLE_OK;
}

/* ------------------------------------------------------------------------------------------------
 * Charge density rho[z,y,x] = int f dv = h_v sum_{l,q} w_q f[z,(l,q),y,x].
 * ---------------------------------------------------------------------------------------------- */
int sldg_oracle_charge_density(const sldg_oracle_grid *g, const double *f, double *rho)
{
    const int Nx = g->n[0] * g->order[0], Ny = g->n[1] * g->order[1], Nz = g->n[2] * g->order[2];
    const int ov = g->order[3], Nv = g->n[3] * ov;
    const double hv = (g->hi[3] - g->lo[3]) / g->n[3];
    double xv[MAXGL], wv[MAXGL];
    sldg_oracle_gl(ov, xv, wv);
    const ptrdiff_t plane = (ptrdiff_t)Ny * Nx;
#pragma omp parallel for schedule(static)
    for (int Z = 0; Z < Nz; ++Z)
        for (ptrdiff_t yx = 0; yx < plane; ++yx) {
            double acc = 0.0;
            for (int V = 0; V < Nv; ++V) acc += wv[V % ov] * f[((ptrdiff_t)Z * Nv + V) * plane + yx];
            rho[Z * plane + yx] = hv * acc;
        }
    return ORACLE_OK;
}

/* ------------------------------------------------------------------------------------------------
 * Total mass = sum f w_x w_y w_z w_v h_x h_y h_z h_v  (Cartesian: Jacobian 1).
 * Accumulated in long double, one partial sum per (z,v) plane.
 * ---------------------------------------------------------------------------------------------- */
double sldg_oracle_mass(const sldg_oracle_grid *g, const double *f)
{
    int N[4];
    double h[4], x[4][MAXGL], w[4][MAXGL];
    for (int d = 0; d < 4; ++d) {
        N[d] = g->n[d] * g->order[d];
        h[d] = (g->hi[d] - g->lo[d]) / g->n[d];
        sldg_oracle_gl(g->order[d], x[d], w[d]);
    }
    const ptrdiff_t plane = (ptrdiff_t)N[1] * N[0];
    long double total = 0.0L;
    for (int Z = 0; Z < N[2]; ++Z)
        for (int V = 0; V < N[3]; ++V) {
            long double acc = 0.0L;
            const double *p = f + ((ptrdiff_t)Z * N[3] + V) * plane;
            for (int Y = 0; Y < N[1]; ++Y) {
                long double row = 0.0L;
                for (int X = 0; X < N[0]; ++X) row += (long double)w[0][X % g->order[0]] * p[(ptrdiff_t)Y * N[0] + X];
                acc += (long double)w[1][Y % g->order[1]] * row;
            }
            total += (long double)w[2][Z % g->order[2]] * (long double)w[3][V % g->order[3]] * acc;
        }
    return (double)(total * (long double)h[0] * h[1] * h[2] * h[3]);
}

/* ================================================================================================
 * 2d SLDG.  All geometry is done in coordinates scaled by (h_x, h_y) and taken
 * RELATIVE TO THE TARGET CELL (i,j): the target cell is [0,1]^2, source cell (i+r, j+s) is
 * [r,r+1] x [s,s+1].  The integral (18) for source cell (r,s) is evaluated in that cell's own local
 * coordinates (reading A11).
 * ============================================================================================== */

typedef struct { double x, y; } pt;

/* piecewise-bilinear velocity ("bilinear interpolation is applied") in cell (ci,cj) at
 * local (xi,eta); a,b are one z-plane [(ny+1)][(nx+1)] */
static void bilinear(const double *a, const double *b, int nx, int ci, int cj, double xi, double eta,
                     double *ua, double *ub)
{
    const ptrdiff_t p = nx + 1;
    const double w00 = (1.0 - xi) * (1.0 - eta), w10 = xi * (1.0 - eta), w01 = (1.0 - xi) * eta,
                 w11 = xi * eta;
    const double *a0 = a + (ptrdiff_t)cj * p + ci, *b0 = b + (ptrdiff_t)cj * p + ci;
    *ua = w00 * a0[0] + w10 * a0[1] + w01 * a0[p] + w11 * a0[p + 1];
    *ub = w00 * b0[0] + w10 * b0[1] + w01 * b0[p] + w11 * b0[p + 1];
}

static int clampi(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }

/* Foot of the characteristic through the point at local (xi,eta) of cell (i,j), relative to cell (i,j),
 * in cell units.  trace_order 1: eq. (14); 2: eq. (15) as explicit midpoint
 * with the one frozen field (reading A9); the half-step point is located in the grid with the cell
 * index clamped to the box. */
static pt trace_point(const double *a, const double *b, int nx, int ny, double hx, double hy, int i,
                      int j, double xi, double eta, double tau, int trace_order, int vel_periodic)
{
    double ua, ub;
    pt f;
    /* a vertex with xi==1 or eta==1 is evaluated in this same cell: bilinear weights pick it exactly */
    bilinear(a, b, nx, i, j, xi, eta, &ua, &ub);
    if (trace_order == 1) {
        f.x = xi - tau * ua / hx;
        f.y = eta - tau * ub / hy;
        return f;
    }
    double mx = xi - 0.5 * tau * ua / hx, my = eta - 0.5 * tau * ub / hy;
    {
        /* Per axis: a bitwise-periodic field is looked up modulo the box, so that the two periodic images of a vertex get
         * the same foot and the upstream mesh tiles (reading A15); otherwise the cell index is clamped to the box.
         * vel_periodic 1: both axes periodic; 0: both clamped; 2: x clamped, y periodic -- the polar plane, x = r
         * (bounded, radial velocity zero at r_min and r_max), y = theta (periodic). */
        const int px = vel_periodic == 1, py = vel_periodic == 1 || vel_periodic == 2;
        int fi = (int)floor(mx), fj = (int)floor(my);
        const int ci = px ? wrap(i + fi, nx) : clampi(i + fi, 0, nx - 1);
        const int cj = py ? wrap(j + fj, ny) : clampi(j + fj, 0, ny - 1);
        if (!px) fi = ci - i;
        if (!py) fj = cj - j;
        bilinear(a, b, nx, ci, cj, mx - fi, my - fj, &ua, &ub);
    }
    f.x = xi - tau * ua / hx;
    f.y = eta - tau * ub / hy;
    return f;
}

/* Exported for the pins: foot (relative to cell (i,j), cell units) of the point at local (xi,eta). */
void sldg_oracle_trace(const sldg_oracle_grid *g, const double *a, const double *b, int i, int j,
                       double xi, double eta, double tau, int trace_order, int vel_periodic,
                       double *foot)
{
    const int nx = g->n[0], ny = g->n[1];
    const double hx = (g->hi[0] - g->lo[0]) / nx, hy = (g->hi[1] - g->lo[1]) / ny;
    pt f = trace_point(a, b, nx, ny, hx, hy, i, j, xi, eta, tau, trace_order, vel_periodic);
    foot[0] = f.x;
    foot[1] = f.y;
}

/* Sutherland-Hodgman: clip polygon against the half-plane  sgn*(coord - bound) >= 0. */
static int clip_halfplane(const pt *in, int n, pt *out, int axis, double bound, double sgn)
{
    int m = 0;
    for (int k = 0; k < n; ++k) {
        pt p = in[k], q = in[(k + 1) % n];
        double dp = sgn * ((axis ? p.y : p.x) - bound), dq = sgn * ((axis ? q.y : q.x) - bound);
        int pin = dp >= 0.0, qin = dq >= 0.0;
        if (pin) out[m++] = p;
        if (pin != qin) {
            double t = dp / (dp - dq);
            pt r;
            r.x = p.x + t * (q.x - p.x);
            r.y = p.y + t * (q.y - p.y);
            if (axis) r.y = bound; else r.x = bound;
            out[m++] = r;
        }
    }
    return m;
}

static int clip_to_unit_square(const pt *quad, pt *poly)
{
    pt b1[16], b2[16];
    int n = 4;
    memcpy(b1, quad, 4 * sizeof(pt));
    n = clip_halfplane(b1, n, b2, 0, 0.0, 1.0);
    if (n < 3) return 0;
    n = clip_halfplane(b2, n, b1, 0, 1.0, -1.0);
    if (n < 3) return 0;
    n = clip_halfplane(b1, n, b2, 1, 0.0, 1.0);
    if (n < 3) return 0;
    n = clip_halfplane(b2, n, b1, 1, 1.0, -1.0);
    if (n < 3) return 0;
    memcpy(poly, b1, n * sizeof(pt));
    return n;
}

/* Solve V X = I (n x n) by Gaussian elimination with partial pivoting; X row-major, X[b*n+m] =
 * coefficient of basis function b in phi*_m.  Returns the smallest pivot magnitude. */
static double invert(int n, double *V, double *X)
{
    double minpiv = 1e300;
    for (int i = 0; i < n * n; ++i) X[i] = 0.0;
    for (int i = 0; i < n; ++i) X[i * n + i] = 1.0;
    for (int c = 0; c < n; ++c) {
        int p = c;
        for (int r = c + 1; r < n; ++r)
            if (fabs(V[r * n + c]) > fabs(V[p * n + c])) p = r;
        if (p != c)
            for (int k = 0; k < n; ++k) {
                double t = V[c * n + k]; V[c * n + k] = V[p * n + k]; V[p * n + k] = t;
                t = X[c * n + k]; X[c * n + k] = X[p * n + k]; X[p * n + k] = t;
            }
        double piv = V[c * n + c];
        if (fabs(piv) < minpiv) minpiv = fabs(piv);
        if (piv == 0.0) return 0.0;
        for (int r = 0; r < n; ++r) {
            if (r == c) continue;
            double fct = V[r * n + c] / piv;
            if (fct == 0.0) continue;
            for (int k = 0; k < n; ++k) {
                V[r * n + k] -= fct * V[c * n + k];
                X[r * n + k] -= fct * X[c * n + k];
            }
        }
    }
    for (int r = 0; r < n; ++r) {
        double piv = V[r * n + r];
        for (int k = 0; k < n; ++k) X[r * n + k] /= piv;
    }
    return minpiv;
}

/* ------------------------------------------------------------------------------------------------
 * Coefficients (18) for ONE target cell and ONE source cell:
 *   C[m*o2 + k] = int_{A*_ij  cap  A_rs} phi_{rs,k}(x,y) phi*_{ij,m}(x,y) dx dy      (cell units)
 * corner[4]: back-traced corners, counter-clockwise from lower-left, relative to the target cell.
 * node[o2]:  back-traced GL nodes, index m = p + o*q (p along x), same frame.
 * (r,s):     source cell offset relative to the target cell.
 * phi*_m is the unique Q^{o-1} polynomial with phi*_m(node[m']) = delta_mm'; the
 * Vandermonde system is set up in the source cell's local coordinates with monomials centred at the
 * centroid of the feet (any basis of Q^{o-1} gives the same polynomial).
 * Returns 1 if the intersection is a polygon (>= 3 vertices), 0 if empty (C zeroed), <0 on error.
 * ---------------------------------------------------------------------------------------------- */
int sldg_oracle_cell_coefficients(int o, const double *corner_xy, const double *node_xy, int r, int s,
                                  double *C)
{
    const int o2 = o * o;
    if (o > MAXO) return ORACLE_EINVAL;
    double xg[MAXGL], wg[MAXGL], xq[MAXGL], wq[MAXGL];
    sldg_oracle_gl(o, xg, wg);
    const int nq = 2 * o; /* >= 2o-1 needed for the collapsed rule */
    sldg_oracle_gl(nq, xq, wq);
    for (int i = 0; i < o2 * o2; ++i) C[i] = 0.0;

    pt quad[4], poly[16];
    for (int c = 0; c < 4; ++c) {
        quad[c].x = corner_xy[2 * c] - r;
        quad[c].y = corner_xy[2 * c + 1] - s;
    }
    int np = clip_to_unit_square(quad, poly);
    if (np < 3) return 0;

    /* adjoint polynomial: Vandermonde at the node feet, source-cell-local, centred monomials */
    double fx[MAXO2], fy[MAXO2], xc = 0.0, yc = 0.0;
    for (int m = 0; m < o2; ++m) {
        fx[m] = node_xy[2 * m] - r;
        fy[m] = node_xy[2 * m + 1] - s;
        xc += fx[m];
        yc += fy[m];
    }
    xc /= o2;
    yc /= o2;
    double V[MAXO2 * MAXO2], coef[MAXO2 * MAXO2];
    for (int mp = 0; mp < o2; ++mp)
        for (int bq = 0; bq < o; ++bq)
            for (int bp = 0; bp < o; ++bp)
                V[mp * o2 + (bp + o * bq)] = pow(fx[mp] - xc, bp) * pow(fy[mp] - yc, bq);
    double minpiv = invert(o2, V, coef);
    if (!(minpiv > 1e-10)) return ORACLE_EGEOM;

    /* fan triangulation + collapsed (Duffy) tensor Gauss rule: exact for the polynomial integrand */
    for (int t = 1; t + 1 < np; ++t) {
        pt P0 = poly[0], P1 = poly[t], P2 = poly[t + 1];
        double e1x = P1.x - P0.x, e1y = P1.y - P0.y, e2x = P2.x - P1.x, e2y = P2.y - P1.y;
        double cross = e1x * e2y - e1y * e2x; /* 2 * signed area */
        for (int iu = 0; iu < nq; ++iu)
            for (int iv = 0; iv < nq; ++iv) {
                double u = xq[iu], v = xq[iv];
                double x = P0.x + u * (e1x + v * e2x), y = P0.y + u * (e1y + v * e2y);
                double wgt = wq[iu] * wq[iv] * u * cross;
                double lx[MAXO], ly[MAXO];
                for (int p = 0; p < o; ++p) {
                    lx[p] = lagrange(o, xg, p, x);
                    ly[p] = lagrange(o, xg, p, y);
                }
                for (int m = 0; m < o2; ++m) {
                    double ps = 0.0;
                    for (int bq = 0; bq < o; ++bq)
                        for (int bp = 0; bp < o; ++bp)
                            ps += coef[(bp + o * bq) * o2 + m] * pow(x - xc, bp) * pow(y - yc, bq);
                    for (int kq = 0; kq < o; ++kq)
                        for (int kp = 0; kp < o; ++kp)
                            C[m * o2 + (kp + o * kq)] += wgt * lx[kp] * ly[kq] * ps;
                }
            }
    }
    return 1;
}

/* ------------------------------------------------------------------------------------------------
 * Geometry of one z-plane (Algorithm 3 / Table 4 steps 1-5).
 * Two-pass interface: call with entries==NULL to get the number of (target, source) entries, then
 * with caller-allocated arrays.  For target cell t = j*nx+i the entries are offs[t]..offs[t+1]-1.
 *   ent_r, ent_s : UNWRAPPED absolute source cell indices (i+r, j+s)
 *   ent_C        : o2*o2 doubles per entry, C[m*o2+k], in physical units / (h_x h_y)  (cell units)
 * No stencil-size limit (reading A10).  Returns number of entries, or <0 on error.
 * ---------------------------------------------------------------------------------------------- */
long sldg_oracle_xy_plane_geometry(const sldg_oracle_grid *g, const double *a, const double *b,
                                   double tau, int trace_order, int vel_periodic, long *offs,
                                   int32_t *ent_r, int32_t *ent_s, double *ent_C)
{
    const int o = g->order[0], o2 = o * o;
    const int nx = g->n[0], ny = g->n[1];
    if (g->order[1] != o || o > MAXO) return ORACLE_EINVAL;
    const double hx = (g->hi[0] - g->lo[0]) / nx, hy = (g->hi[1] - g->lo[1]) / ny;
    double xg[MAXGL], wg[MAXGL];
    sldg_oracle_gl(o, xg, wg);
    const int ncell = nx * ny;
    long *cnt = (long *)malloc(sizeof(long) * (size_t)(ncell + 1));
    int32_t *box = (int32_t *)malloc(sizeof(int32_t) * 4 * (size_t)ncell);
    if (!cnt || !box) { free(cnt); free(box); return ORACLE_ENOMEM; }
    int err = 0;

    /* pass 1: corner feet -> bounding box of candidate source cells (step 3, half-open) */
#pragma omp parallel for schedule(static)
    for (int t = 0; t < ncell; ++t) {
        int i = t % nx, j = t / nx;
        static const double cxi[4] = {0, 1, 1, 0}, ceta[4] = {0, 0, 1, 1};
        pt c[4];
        double xmin = 1e300, xmax = -1e300, ymin = 1e300, ymax = -1e300;
        for (int k = 0; k < 4; ++k) {
            c[k] = trace_point(a, b, nx, ny, hx, hy, i, j, cxi[k], ceta[k], tau, trace_order, vel_periodic);
            xmin = fmin(xmin, c[k].x); xmax = fmax(xmax, c[k].x);
            ymin = fmin(ymin, c[k].y); ymax = fmax(ymax, c[k].y);
        }
        double area = 0.0;
        for (int k = 0; k < 4; ++k) area += c[k].x * c[(k + 1) % 4].y - c[(k + 1) % 4].x * c[k].y;
        if (!(area > 0.0)) {
#pragma omp atomic write
            err = 1;
        }
        int r0 = (int)floor(xmin), r1 = (int)ceil(xmax) - 1, s0 = (int)floor(ymin), s1 = (int)ceil(ymax) - 1;
        if (r1 < r0) r1 = r0;
        if (s1 < s0) s1 = s0;
        box[4 * t + 0] = r0; box[4 * t + 1] = r1; box[4 * t + 2] = s0; box[4 * t + 3] = s1;
        cnt[t] = (long)(r1 - r0 + 1) * (s1 - s0 + 1);
    }
    if (err) { free(cnt); free(box); return ORACLE_EGEOM; }
    long total = 0;
    for (int t = 0; t < ncell; ++t) { long c = cnt[t]; cnt[t] = total; total += c; }
    cnt[ncell] = total;
    if (!ent_C) { free(cnt); free(box); return total; }
    memcpy(offs, cnt, sizeof(long) * (size_t)(ncell + 1));

    /* pass 2: node feet, adjoint polynomial, clip, integrate (steps 2, 4-6) */
#pragma omp parallel for schedule(dynamic, 16)
    for (int t = 0; t < ncell; ++t) {
        int i = t % nx, j = t / nx;
        static const double cxi[4] = {0, 1, 1, 0}, ceta[4] = {0, 0, 1, 1};
        double corner[8], node[2 * MAXO2];
        for (int k = 0; k < 4; ++k) {
            pt c = trace_point(a, b, nx, ny, hx, hy, i, j, cxi[k], ceta[k], tau, trace_order, vel_periodic);
            corner[2 * k] = c.x; corner[2 * k + 1] = c.y;
        }
        for (int q = 0; q < o; ++q)
            for (int p = 0; p < o; ++p) {
                pt c = trace_point(a, b, nx, ny, hx, hy, i, j, xg[p], xg[q], tau, trace_order, vel_periodic);
                node[2 * (p + o * q)] = c.x; node[2 * (p + o * q) + 1] = c.y;
            }
        long e = cnt[t];
        for (int s = box[4 * t + 2]; s <= box[4 * t + 3]; ++s)
            for (int r = box[4 * t + 0]; r <= box[4 * t + 1]; ++r, ++e) {
                ent_r[e] = i + r;
                ent_s[e] = j + s;
                int rc = sldg_oracle_cell_coefficients(o, corner, node, r, s, ent_C + (size_t)e * o2 * o2);
                if (rc < 0) {
#pragma omp atomic write
                    err = 1;
                }
            }
    }
    free(cnt);
    free(box);
    return err ? ORACLE_EGEOM : total;
}

/* ------------------------------------------------------------------------------------------------
 * 2d advection of the whole 4d array (eq. 17; Algorithm 3):
 * geometry once per z-node, then  u+_{ij,m} = (1/W_m) sum_{rs} sum_k C^{ij,m}_{rs,k} u_{rs,k}  for
 * every v-node, W_m = w_p w_q (cell units; reading A12).  f periodic in x and y (reading A15).
 * ---------------------------------------------------------------------------------------------- */
int sldg_oracle_advect_xy(const sldg_oracle_grid *g, const double *fin, const double *a,
                          const double *b, double *fout, double tau, int trace_order, int vel_periodic)
{
    const int o = g->order[0], o2 = o * o;
    const int nx = g->n[0], ny = g->n[1];
    const int Nx = nx * o, Ny = ny * o, Nz = g->n[2] * g->order[2], Nv = g->n[3] * g->order[3];
    if (g->order[1] != o || o > MAXO) return ORACLE_EINVAL;
    double xg[MAXGL], wg[MAXGL];
    sldg_oracle_gl(o, xg, wg);
    const ptrdiff_t plane = (ptrdiff_t)Ny * Nx, vplane = (ptrdiff_t)(ny + 1) * (nx + 1);
    const int ncell = nx * ny;
    long *offs = (long *)malloc(sizeof(long) * (size_t)(ncell + 1));
    if (!offs) return ORACLE_ENOMEM;
    int rc = ORACLE_OK;
    for (int Z = 0; Z < Nz && rc == ORACLE_OK; ++Z) {
        const double *az = a + Z * vplane, *bz = b + Z * vplane;
        long ne = sldg_oracle_xy_plane_geometry(g, az, bz, tau, trace_order, vel_periodic, NULL, NULL, NULL, NULL);
        if (ne < 0) { rc = (int)ne; break; }
        int32_t *er = (int32_t *)malloc(sizeof(int32_t) * (size_t)(ne + 1));
        int32_t *es = (int32_t *)malloc(sizeof(int32_t) * (size_t)(ne + 1));
        double *eC = (double *)malloc(sizeof(double) * (size_t)(ne + 1) * o2 * o2);
        if (!er || !es || !eC) { free(er); free(es); free(eC); rc = ORACLE_ENOMEM; break; }
        long ne2 = sldg_oracle_xy_plane_geometry(g, az, bz, tau, trace_order, vel_periodic, offs, er, es, eC);
        if (ne2 < 0) { free(er); free(es); free(eC); rc = (int)ne2; break; }
#pragma omp parallel for schedule(static)
        for (int V = 0; V < Nv; ++V) {
            const double *pin = fin + ((ptrdiff_t)Z * Nv + V) * plane;
            double *pout = fout + ((ptrdiff_t)Z * Nv + V) * plane;
            for (int t = 0; t < ncell; ++t) {
                int i = t % nx, j = t / nx;
                for (int mq = 0; mq < o; ++mq)
                    for (int mp = 0; mp < o; ++mp) {
                        int m = mp + o * mq;
                        double acc = 0.0;
                        for (long e = offs[t]; e < offs[t + 1]; ++e) {
                            int rr = wrap(er[e], nx), ss = wrap(es[e], ny);
                            const double *Cm = eC + (size_t)e * o2 * o2 + (size_t)m * o2;
                            for (int kq = 0; kq < o; ++kq)
                                for (int kp = 0; kp < o; ++kp)
                                    acc += Cm[kp + o * kq] * pin[(ptrdiff_t)(ss * o + kq) * Nx + rr * o + kp];
                        }
                        pout[(ptrdiff_t)(j * o + mq) * Nx + i * o + mp] = acc / (wg[mp] * wg[mq]);
                    }
            }
        }
        free(er); free(es); free(eC);
    }
    free(offs);
    return rc;
}

/* ------------------------------------------------------------------------------------------------
 * One Strang step with frozen fields (Algorithm 1 steps 3,4,6,7,8; the source terms
 * vanish for the Cartesian full-f formulation):
 *   z(dt/2) -> v(dt/2) -> xy(dt) -> v(dt/2) -> z(dt/2).   f is updated in place; tmp is scratch.
 * ---------------------------------------------------------------------------------------------- */
int sldg_oracle_strang_step(const sldg_oracle_grid *g, double *f, double *tmp, const double *Ez,
                            const double *a, const double *b, double dt, int trace_order,
                            int vel_periodic)
{
    int rc;
    if ((rc = sldg_oracle_advect_z(g, f, tmp, 0.5 * dt))) return rc;
    if ((rc = sldg_oracle_advect_v(g, tmp, Ez, f, 0.5 * dt))) return rc;
    if ((rc = sldg_oracle_advect_xy(g, f, a, b, tmp, dt, trace_order, vel_periodic))) return rc;
    if ((rc = sldg_oracle_advect_v(g, tmp, Ez, f, 0.5 * dt))) return rc;
    if ((rc = sldg_oracle_advect_z(g, f, tmp, 0.5 * dt))) return rc;
    memcpy(f, tmp, sizeof(double) * (size_t)g->n[0] * g->order[0] * g->n[1] * g->order[1] *
                       g->n[2] * g->order[2] * g->n[3] * g->order[3]);
    return ORACLE_OK;
}

int sldg_oracle_num_threads(void)
{
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}
