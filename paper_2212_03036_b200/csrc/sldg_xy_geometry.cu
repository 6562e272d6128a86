// sldg_xy_geometry.cu -- 2d SLDG step in the poloidal plane (Algorithm 3).
//
//   xy_geometry : per (z node, target cell, 3x3 slot): back-trace corners and GL nodes (eq. 14/15,
//                 PAPER.md:206-218), adjoint polynomial phi* from a Vandermonde solve,
//                 monomial moments of  A*_ij cap A_rs  by Green's theorem along the clipped upstream edges
//                 ("outer segments") and the grid-line pieces inside the upstream cell ("inner
//                 segments", Table 4), coefficients C of eq. (18), scaled by 1/W_m.
//   (the apply kernels, eq. (17), live in sldg_xy_apply.cu)
//
// Green's theorem with P = 0, Q^{(p,q)} = x^{p+1} y^q / (p+1)  (reproduces the paper's
// Q^{(2,1)}, Q^{(2,2)}): in the source cell's local coordinates horizontal segments and
// segments on the cell's left edge x=0 contribute nothing; only the upstream edges and the pieces of the
// cell's right edge x=1 inside the upstream cell do.
//
// All geometry is done in cell units relative to the target cell (the target is [0,1]^2), the integrals
// in the source cell's own local coordinates.
#include "sldg_internal.cuh"

__device__ __forceinline__ int wrap_idx(int i, int n)
{
    int r = i % n;
    return r < 0 ? r + n : r;
}

// piecewise-bilinear velocity of cell (ci,cj) at local (xi,eta), scaled to Courant units
__device__ __forceinline__ void bilinear_vel(const double *__restrict__ a, const double *__restrict__ b,
                                             int pitch, int ci, int cj, double xi, double eta,
                                             double &ua, double &ub)
{
    const double *a0 = a + (long long)cj * pitch + ci;
    const double *b0 = b + (long long)cj * pitch + ci;
    const double w00 = (1.0 - xi) * (1.0 - eta), w10 = xi * (1.0 - eta), w01 = (1.0 - xi) * eta,
                 w11 = xi * eta;
    ua = w00 * __ldg(a0) + w10 * __ldg(a0 + 1) + w01 * __ldg(a0 + pitch) + w11 * __ldg(a0 + pitch + 1);
    ub = w00 * __ldg(b0) + w10 * __ldg(b0 + 1) + w01 * __ldg(b0 + pitch) + w11 * __ldg(b0 + pitch + 1);
}

// foot of the characteristic through local (xi,eta) of cell (i,j), relative to that cell, cell units
__device__ __forceinline__ void trace_point(const double *__restrict__ a, const double *__restrict__ b,
                                            int nx, int ny, double tx, double ty, int i, int j,
                                            double xi, double eta, int order, int periodic, double &fx,
                                            double &fy)
{
    double ua, ub;
    bilinear_vel(a, b, nx + 1, i, j, xi, eta, ua, ub);
    if (order != 1) {
        double mx = xi - 0.5 * tx * ua, my = eta - 0.5 * ty * ub;
        int fi = (int)floor(mx), fj = (int)floor(my);
        int ci, cj;
        if (periodic) {
            ci = wrap_idx(i + fi, nx);
            cj = wrap_idx(j + fj, ny);
        } else {
            ci = min(max(i + fi, 0), nx - 1);
            cj = min(max(j + fj, 0), ny - 1);
            fi = ci - i;
            fj = cj - j;
        }
        bilinear_vel(a, b, nx + 1, ci, cj, mx - fi, my - fj, ua, ub);
    }
    fx = xi - tx * ua;
    fy = eta - ty * ub;
}

// Gauss-Jordan with partial pivoting on [V | X], fully unrolled so that everything stays in registers.
// On exit X = V^{-1}.  Returns the smallest pivot magnitude.
template <int N>
__device__ __forceinline__ double gauss_jordan(double (&V)[N][N], double (&X)[N][N])
{
    double minpiv = 1e300;
#pragma unroll
    for (int c = 0; c < N; ++c) {
        int p = c;
        double best = fabs(V[c][c]);
#pragma unroll
        for (int r = c + 1; r < N; ++r) {
            double v = fabs(V[r][c]);
            if (v > best) {
                best = v;
                p = r;
            }
        }
#pragma unroll
        for (int r = c + 1; r < N; ++r) {
            if (p == r) {
#pragma unroll
                for (int k = 0; k < N; ++k) {
                    double t = V[c][k]; V[c][k] = V[r][k]; V[r][k] = t;
                    t = X[c][k]; X[c][k] = X[r][k]; X[r][k] = t;
                }
            }
        }
        minpiv = fmin(minpiv, best);
        const double inv = 1.0 / V[c][c];
#pragma unroll
        for (int k = 0; k < N; ++k) {
            V[c][k] *= inv;
            X[c][k] *= inv;
        }
#pragma unroll
        for (int r = 0; r < N; ++r) {
            if (r != c) {
                const double fct = V[r][c];
#pragma unroll
                for (int k = 0; k < N; ++k) {
                    V[r][k] = fma(-fct, V[c][k], V[r][k]);
                    X[r][k] = fma(-fct, X[c][k], X[r][k]);
                }
            }
        }
    }
    return minpiv;
}

// Monomial moments M[p][q] = int x^p y^q over (upstream quadrilateral) cap (unit cell), by Green's theorem.
// (X,Y): quadrilateral corners counter-clockwise in the source cell's local coordinates.
// inner_right: the grid line x_local = 1 lies strictly inside the quadrilateral's x-extent.
template <int O>
__device__ __forceinline__ void piece_moments(const double (&X)[4], const double (&Y)[4],
                                              bool inner_right, const Basis &bs,
                                              double (&M)[2 * O - 1][2 * O - 1])
{
    constexpr int NM = 2 * O - 1;
#pragma unroll
    for (int p = 0; p < NM; ++p)
#pragma unroll
        for (int q = 0; q < NM; ++q) M[p][q] = 0.0;
    double ylo = 1e300, yhi = -1e300;
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const double x0 = X[e], y0 = Y[e], x1 = X[(e + 1) & 3], y1 = Y[(e + 1) & 3];
        const double dx = x1 - x0, dy = y1 - y0;
        // crossing with the line x = 1 (for the inner segment)
        if (inner_right && dx != 0.0 && (x0 - 1.0) * (x1 - 1.0) <= 0.0) {
            double yc = fma((1.0 - x0) / dx, dy, y0);
            ylo = fmin(ylo, yc);
            yhi = fmax(yhi, yc);
        }
        // outer segment: Liang-Barsky clip of the edge against the closed unit square
        double t0 = 0.0, t1 = 1.0;
        bool ok = true;
        {
            const double pp[4] = {-dx, dx, -dy, dy};
            const double qq[4] = {x0, 1.0 - x0, y0, 1.0 - y0};
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                if (pp[k] == 0.0) {
                    if (qq[k] < 0.0) ok = false;
                } else {
                    double r = qq[k] / pp[k];
                    if (pp[k] < 0.0)
                        t0 = fmax(t0, r);
                    else
                        t1 = fmin(t1, r);
                }
            }
        }
        if (ok && t1 > t0 && dy != 0.0) {
            const double xa = fmin(fmax(fma(t0, dx, x0), 0.0), 1.0), ya = fmin(fmax(fma(t0, dy, y0), 0.0), 1.0);
            const double xb = fmin(fmax(fma(t1, dx, x0), 0.0), 1.0), yb = fmin(fmax(fma(t1, dy, y0), 0.0), 1.0);
            const double ex = xb - xa, ey = yb - ya;
            for (int gq = 0; gq < bs.nq; ++gq) {
                const double t = bs.qx[gq];
                const double x = fma(t, ex, xa), y = fma(t, ey, ya);
                const double wgt = bs.qw[gq] * ey;
                double xp = x;  // x^{p+1}
#pragma unroll
                for (int p = 0; p < NM; ++p) {
                    double term = wgt * xp * (1.0 / (p + 1));
#pragma unroll
                    for (int q = 0; q < NM; ++q) {
                        M[p][q] += term;
                        term *= y;
                    }
                    xp *= x;
                }
            }
        }
    }
    if (inner_right) {
        const double ya = fmax(ylo, 0.0), yb = fmin(yhi, 1.0);
        if (yb > ya) {
            double pa = ya, pb = yb;  // y^{q+1}
#pragma unroll
            for (int q = 0; q < NM; ++q) {
                const double seg = (pb - pa) * (1.0 / (q + 1));
#pragma unroll
                for (int p = 0; p < NM; ++p) M[p][q] += seg * (1.0 / (p + 1));
                pa *= ya;
                pb *= yb;
            }
        }
    }
}

template <int O>
__global__ void __launch_bounds__(128) xy_geometry_kernel(const double *__restrict__ va,
                                                          const double *__restrict__ vb,
                                                          int32_t *__restrict__ anchor,
                                                          int32_t *__restrict__ mask,
                                                          double *__restrict__ W, int32_t *err,
                                                          GridDev g, Basis bs, double tau, int order,
                                                          int periodic)
{
    constexpr int O2 = O * O, NM = 2 * O - 1;
    const int nx = g.n[0], ny = g.n[1];
    const long long ncell = (long long)nx * ny;
    const long long total = (long long)g.N[2] * ncell * 9;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= total) return;
    const int slot = (int)(gid % 9);
    const long long cellid = gid / 9;
    const int z = (int)(cellid / ncell);
    const int t = (int)(cellid % ncell);
    const int i = t % nx, j = t / nx;
    const long long vplane = (long long)(ny + 1) * (nx + 1);
    const double *a = va + z * vplane, *b = vb + z * vplane;
    const double tx = tau / g.h[0], ty = tau / g.h[1];

    // step 1: corner feet -> upstream quadrilateral (counter-clockwise from lower-left)
    double cx[4], cy[4];
    trace_point(a, b, nx, ny, tx, ty, i, j, 0.0, 0.0, order, periodic, cx[0], cy[0]);
    trace_point(a, b, nx, ny, tx, ty, i, j, 1.0, 0.0, order, periodic, cx[1], cy[1]);
    trace_point(a, b, nx, ny, tx, ty, i, j, 1.0, 1.0, order, periodic, cx[2], cy[2]);
    trace_point(a, b, nx, ny, tx, ty, i, j, 0.0, 1.0, order, periodic, cx[3], cy[3]);
    const double xmin = fmin(fmin(cx[0], cx[1]), fmin(cx[2], cx[3]));
    const double xmax = fmax(fmax(cx[0], cx[1]), fmax(cx[2], cx[3]));
    const double ymin = fmin(fmin(cy[0], cy[1]), fmin(cy[2], cy[3]));
    const double ymax = fmax(fmax(cy[0], cy[1]), fmax(cy[2], cy[3]));
    const int r0 = (int)floor(xmin), s0 = (int)floor(ymin);
    const int r1 = max((int)ceil(xmax) - 1, r0), s1 = max((int)ceil(ymax) - 1, s0);
    if (slot == 0) {
        anchor[2 * cellid] = r0;      // relative to the target cell, unwrapped
        anchor[2 * cellid + 1] = s0;
        bool convex = true;
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            double e1x = cx[(e + 1) & 3] - cx[e], e1y = cy[(e + 1) & 3] - cy[e];
            double e2x = cx[(e + 2) & 3] - cx[(e + 1) & 3], e2y = cy[(e + 2) & 3] - cy[(e + 1) & 3];
            if (!(e1x * e2y - e1y * e2x > 0.0)) convex = false;
        }
        if (!convex) atomicMin(err, SLDG_EGEOM);
        if (r1 - r0 > 2 || s1 - s0 > 2) atomicMin(err, SLDG_ESTENCIL);
    }
    const int dr = slot % 3, ds = slot / 3;
    if (dr > r1 - r0 || ds > s1 - s0) return;
    const int r = r0 + dr, s = s0 + ds;

    // moments of the piece in the source cell's local coordinates
    double X[4], Y[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        X[k] = cx[k] - r;
        Y[k] = cy[k] - s;
    }
    double M[NM][NM];
    piece_moments<O>(X, Y, r < r1, bs, M);
    if (!(M[0][0] > 0.0)) return;  // empty intersection

    // step 2: node feet and adjoint polynomial (centred monomials, then shifted to local monomials)
    double fx[O2], fy[O2], xc = 0.0, yc = 0.0;
#pragma unroll
    for (int q = 0; q < O; ++q)
#pragma unroll
        for (int p = 0; p < O; ++p) {
            double px, py;
            trace_point(a, b, nx, ny, tx, ty, i, j, bs.xi[O][p], bs.xi[O][q], order, periodic, px, py);
            fx[p + O * q] = px - r;
            fy[p + O * q] = py - s;
            xc += px - r;
            yc += py - s;
        }
    xc *= 1.0 / O2;
    yc *= 1.0 / O2;
    double V[O2][O2], Vi[O2][O2];
#pragma unroll
    for (int m = 0; m < O2; ++m) {
        double py = 1.0;
#pragma unroll
        for (int bq = 0; bq < O; ++bq) {
            double px = 1.0;
#pragma unroll
            for (int bp = 0; bp < O; ++bp) {
                V[m][bp + O * bq] = px * py;
                px *= fx[m] - xc;
            }
            py *= fy[m] - yc;
        }
#pragma unroll
        for (int k = 0; k < O2; ++k) Vi[m][k] = (m == k) ? 1.0 : 0.0;
    }
    const double minpiv = gauss_jordan<O2>(V, Vi);  // Vi[ab][m]: phi*_m = sum_ab Vi[ab][m] (x-xc)^a (y-yc)^b
    if (!(minpiv > 1e-10)) atomicMin(err, SLDG_EGEOM);
    // shift to monomials x^a y^b of the source cell: (x-xc)^a = sum_a' binom(a,a') (-xc)^(a-a') x^a'
    double cf[O2][O2];  // cf[a'+O b'][m]
    {
        double sxp[O][O], syp[O][O];  // sxp[a][a'] = binom(a,a') (-xc)^(a-a')
#pragma unroll
        for (int aa = 0; aa < O; ++aa)
#pragma unroll
            for (int ap = 0; ap < O; ++ap) {
                double bin = (ap > aa) ? 0.0 : ((aa == 2 && ap == 1) ? 2.0 : 1.0);
                double px = 1.0, py = 1.0;
                for (int e = 0; e < aa - ap; ++e) {
                    px *= -xc;
                    py *= -yc;
                }
                sxp[aa][ap] = bin * px;
                syp[aa][ap] = bin * py;
            }
#pragma unroll
        for (int m = 0; m < O2; ++m)
#pragma unroll
            for (int bp_ = 0; bp_ < O; ++bp_)
#pragma unroll
                for (int ap = 0; ap < O; ++ap) {
                    double acc = 0.0;
#pragma unroll
                    for (int bb = bp_; bb < O; ++bb)
#pragma unroll
                        for (int aa = ap; aa < O; ++aa) acc = fma(Vi[aa + O * bb][m], sxp[aa][ap] * syp[bb][bp_], acc);
                    cf[ap + O * bp_][m] = acc;
                }
    }
    // G[k][a'+O b'] = int phi_k x^a' y^b' = sum_{p',q'} L[kp][p'] L[kq][q'] M[p'+a'][q'+b']  (separable)
    double T[O][O][NM];  // T[kp][a'][q] = sum_p' L[kp][p'] M[p'+a'][q]
#pragma unroll
    for (int kp = 0; kp < O; ++kp)
#pragma unroll
        for (int ap = 0; ap < O; ++ap)
#pragma unroll
            for (int q = 0; q < NM; ++q) {
                double acc = 0.0;
#pragma unroll
                for (int pp = 0; pp < O; ++pp) acc = fma(bs.L[O][kp][pp], M[pp + ap][q], acc);
                T[kp][ap][q] = acc;
            }
    double *Wout = W + ((size_t)cellid * 9 + slot) * (O2 * O2);
#pragma unroll
    for (int kq = 0; kq < O; ++kq)
#pragma unroll
        for (int kp = 0; kp < O; ++kp) {
            double G[O2];
#pragma unroll
            for (int bp_ = 0; bp_ < O; ++bp_)
#pragma unroll
                for (int ap = 0; ap < O; ++ap) {
                    double acc = 0.0;
#pragma unroll
                    for (int qq = 0; qq < O; ++qq) acc = fma(bs.L[O][kq][qq], T[kp][ap][qq + bp_], acc);
                    G[ap + O * bp_] = acc;
                }
            const int k = kp + O * kq;
#pragma unroll
            for (int m = 0; m < O2; ++m) {
                double acc = 0.0;
#pragma unroll
                for (int ab = 0; ab < O2; ++ab) acc = fma(cf[ab][m], G[ab], acc);
                Wout[k * O2 + m] = acc / (bs.w[O][m % O] * bs.w[O][m / O]);
            }
        }
    atomicOr(&mask[cellid], 1 << slot);
}

cudaError_t launch_xy_geometry(sldg_ctx *c, double tau, int trace_order)
{
    const GridDev &g = c->g;
    const long long ncell = (long long)g.n[0] * g.n[1];
    const long long total = (long long)g.N[2] * ncell * 9;
    cudaError_t e = cudaMemsetAsync(c->mask, 0, sizeof(int32_t) * (size_t)g.N[2] * ncell, c->stream);
    if (e != cudaSuccess) return e;
    const int threads = 128;
    const unsigned grid = (unsigned)((total + threads - 1) / threads);
    const int O = g.o[0];
#define LAUNCH_G(OO)                                                                                 \
    xy_geometry_kernel<OO><<<grid, threads, 0, c->stream>>>(c->va, c->vb, c->anchor, c->mask, c->W, \
                                                            c->err, g, c->basis, tau, trace_order,  \
                                                            c->vel_periodic)
    if (O == 1) LAUNCH_G(1); else if (O == 2) LAUNCH_G(2); else LAUNCH_G(3);
#undef LAUNCH_G
    c->launches++;
    return cudaGetLastError();
}

