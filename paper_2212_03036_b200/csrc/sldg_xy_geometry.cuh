// sldg_xy_geometry.cuh -- device code of the 2d geometry (eq. 14-18) used by the geometry kernel
// of sldg_xy_geometry.cu: tracing, adjoint polynomials, clipping, Green's-theorem moments, contraction.
#pragma once
#include "sldg_internal.cuh"

namespace sldg_geom {

// i modulo n in [0, n); the division (some 25 instructions) only when i is outside the box
__device__ __forceinline__ int wrap_idx(int i, int n)
{
    if ((unsigned)i < (unsigned)n) return i;
    int r = i % n;
    return r < 0 ? r + n : r;
}

// min / max as one compare + select.  fmin()/fmax() cost ~8 instructions each in fp64 on sm_100a (NaN
// handling); nothing here can be NaN.
__device__ __forceinline__ double dmin(double a, double b) { return a < b ? a : b; }
__device__ __forceinline__ double dmax(double a, double b) { return a > b ? a : b; }

// piecewise-bilinear velocity at local (xi,eta) of a cell, from the cell's four vertex values (lower-left,
// lower-right, upper-left, upper-right)
__device__ __forceinline__ void bilinear_val(const double (&va)[4], const double (&vb)[4], double xi, double eta,
                                             double &ua, double &ub)
{
    const double w00 = (1.0 - xi) * (1.0 - eta), w10 = xi * (1.0 - eta), w01 = (1.0 - xi) * eta,
                 w11 = xi * eta;
    ua = w00 * va[0] + w10 * va[1] + w01 * va[2] + w11 * va[3];
    ub = w00 * vb[0] + w10 * vb[1] + w01 * vb[2] + w11 * vb[3];
}

// Gauss-Jordan with partial pivoting on [V | X], fully unrolled so that everything stays in registers (o <= 2).
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
        minpiv = dmin(minpiv, best);
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

// In-place Gauss-Jordan inversion with partial pivoting of the N x N matrix whose element (r, k) lives at
// a[(r * N + k) * stride] (one thread's column of a shared-memory array: conflict-free).  For o = 3 (N = 9): two
// 9 x 9 matrices in registers are 324 registers' worth and spill; in local memory they thrash L1 (measured: 2x
// slower).  Returns the smallest pivot magnitude.
template <int N>
__device__ __forceinline__ double invert_in_place(double *a, int stride)
{
    double minpiv = 1e300;
    unsigned long long perm = 0;  // 4 bits per column: the row it was swapped with
#pragma unroll 1
    for (int c = 0; c < N; ++c) {
        int p = c;
        double best = fabs(a[(c * N + c) * stride]);
#pragma unroll 1
        for (int r = c + 1; r < N; ++r) {
            const double v = fabs(a[(r * N + c) * stride]);
            if (v > best) {
                best = v;
                p = r;
            }
        }
        perm |= (unsigned long long)p << (4 * c);
        if (p != c) {
#pragma unroll
            for (int k = 0; k < N; ++k) {
                const double t = a[(c * N + k) * stride];
                a[(c * N + k) * stride] = a[(p * N + k) * stride];
                a[(p * N + k) * stride] = t;
            }
        }
        minpiv = dmin(minpiv, best);
        const double inv = 1.0 / a[(c * N + c) * stride];
        a[(c * N + c) * stride] = 1.0;
        double rowc[N];
#pragma unroll
        for (int k = 0; k < N; ++k) {
            rowc[k] = a[(c * N + k) * stride] * inv;
            a[(c * N + k) * stride] = rowc[k];
        }
#pragma unroll 1
        for (int r = 0; r < N; ++r) {
            if (r == c) continue;
            const double fct = a[(r * N + c) * stride];
            a[(r * N + c) * stride] = 0.0;
#pragma unroll
            for (int k = 0; k < N; ++k) a[(r * N + k) * stride] = fma(-fct, rowc[k], a[(r * N + k) * stride]);
        }
    }
    // the row swaps of the elimination become column swaps of the inverse, undone in reverse order
#pragma unroll 1
    for (int c = N - 1; c >= 0; --c) {
        const int p = (int)((perm >> (4 * c)) & 15);
        if (p != c) {
#pragma unroll 1
            for (int r = 0; r < N; ++r) {
                const double t = a[(r * N + c) * stride];
                a[(r * N + c) * stride] = a[(r * N + p) * stride];
                a[(r * N + p) * stride] = t;
            }
        }
    }
    return minpiv;
}

// Monomial moments M[p][q] = int x^p y^q over (upstream quadrilateral) cap (source cell (r,s)), in that
// cell's local coordinates, by Green's theorem.  The quadrilateral of the block's cell c comes from shared memory
// (corners counter-clockwise in anchor-cell units sh.cx/sh.cy, reciprocals of the edge direction components sh.idx/
// sh.idy, 0 when the component is 0); the loop over its four edges stays rolled (code size).  inner_right: the grid line
// x_local = 1 lies inside the quadrilateral's bounding box (r < r1).
template <int O, class SH>
__device__ __forceinline__ void piece_moments(const SH &sh, int c, double offx, double offy, bool inner_right,
                                              const Basis &bs, double (&M)[2 * O - 1][2 * O - 1])
{
    constexpr int NM = 2 * O - 1;
#pragma unroll
    for (int p = 0; p < NM; ++p)
#pragma unroll
        for (int qq = 0; qq < NM; ++qq) M[p][qq] = 0.0;
    double ylo = 1e300, yhi = -1e300;
    double xn = sh.cx[0][c], yn = sh.cy[0][c];  // start of the next edge
#pragma unroll 1
    for (int e = 0; e < 4; ++e) {
        const double xs = xn, ys = yn;
        xn = sh.cx[(e + 1) & 3][c];
        yn = sh.cy[(e + 1) & 3][c];
        const double x0 = xs - offx, y0 = ys - offy;
        const double dx = xn - xs, dy = yn - ys;
        const double idx = sh.idx[e][c], idy = sh.idy[e][c];
        // crossing with the line x = 1 (for the inner segment); decided from the actual end points
        const double x1 = xn - offx;
        if (inner_right && dx != 0.0 && (x0 - 1.0) * (x1 - 1.0) <= 0.0) {
            const double yc = fma(dmin(dmax((1.0 - x0) * idx, 0.0), 1.0), dy, y0);
            ylo = dmin(ylo, yc);
            yhi = dmax(yhi, yc);
        }
        // outer segment: Liang-Barsky clip of the edge against the closed unit square.  Which of the two crossings of an
        // axis is the entry is the sign of the direction component (one integer test on the reciprocal's sign bit and two
        // selects instead of a min and a max: fp64 min/max are compare + 2 selects each and were 30 % of this kernel's
        // instructions together with the clamps of the end points, which only moved them by round-off and are gone).
        double t0 = 0.0, t1 = 1.0;
        bool ok = dy != 0.0;  // horizontal edges contribute nothing (dy = 0 in the line integral)
        if (dx == 0.0) {
            ok = ok && x0 >= 0.0 && x0 <= 1.0;
        } else {
            const double ta = -x0 * idx, tb = (1.0 - x0) * idx;
            const bool neg = __double2hiint(idx) < 0;
            t0 = dmax(t0, neg ? tb : ta);
            t1 = dmin(t1, neg ? ta : tb);
        }
        {
            const double ta = -y0 * idy, tb = (1.0 - y0) * idy;
            const bool neg = __double2hiint(idy) < 0;
            t0 = dmax(t0, neg ? tb : ta);
            t1 = dmin(t1, neg ? ta : tb);
        }
        if (ok && t1 > t0) {
            const double xa = fma(t0, dx, x0), ya = fma(t0, dy, y0);
            const double ex = (t1 - t0) * dx, ey = (t1 - t0) * dy;
#pragma unroll
            for (int gq = 0; gq < NM; ++gq) {  // (2o-1)-point Gauss rule: exact for degree 4o-3
                const double t = bs.qx[gq];
                const double x = fma(t, ex, xa), y = fma(t, ey, ya);
                const double wgt = bs.qw[gq] * ey;
                double xw[NM], yp[NM];  // wgt x^{p+1} / (p+1),  y^q
                double xpow = x;
                yp[0] = 1.0;
#pragma unroll
                for (int p = 0; p < NM; ++p) {
                    xw[p] = (wgt * (1.0 / (p + 1))) * xpow;
                    xpow *= x;
                    if (p + 1 < NM) yp[p + 1] = yp[p] * y;
                }
#pragma unroll
                for (int p = 0; p < NM; ++p)
#pragma unroll
                    for (int qq = 0; qq < NM; ++qq) M[p][qq] = fma(xw[p], yp[qq], M[p][qq]);
            }
        }
    }
    if (inner_right) {
        const double ya = dmax(ylo, 0.0), yb = dmin(yhi, 1.0);
        if (yb > ya) {
            double pa = ya, pb = yb;  // y^{q+1}
#pragma unroll
            for (int qq = 0; qq < NM; ++qq) {
                const double seg = (pb - pa) * (1.0 / (qq + 1));
#pragma unroll
                for (int p = 0; p < NM; ++p) M[p][qq] += seg * (1.0 / (p + 1));
                pa *= ya;
                pb *= yb;
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------
// Two phases per block of GEOM_CELLS target cells of one z node, handing over through shared memory:
//   phase 1, thread <-> target cell: steps 1 and 4 (corner feet, bounding box, node feet, inverse Vandermonde);
//   phase 2, thread <-> work item = (target cell, candidate source cell of its bounding box): steps 2, 3, 5
//            (clipped edges, moments, contraction) for ONE piece.  The items of the block are enumerated
//            densely (prefix sum of the per-cell candidate counts), so a warp never idles on a cell with fewer
//            candidates than its neighbours', and each phase keeps only its own state in registers.
// The non-empty pieces of a cell are stored packed in slot order, W[cell][0 .. count); the header's mask says
// which slots they are.
// ---------------------------------------------------------------------------------------------------------
template <int O, int NCELLS = (O == 3 ? 64 : 128)>
struct GeomShared {
    static constexpr int O2 = O * O;
    static constexpr int CELLS = NCELLS;
    // structure of arrays, [field][cell]: phase 1 writes with consecutive lanes on consecutive words
    double cx[4][CELLS], cy[4][CELLS];     // corner feet relative to the anchor cell, cell units
    double idx[4][CELLS], idy[4][CELLS];   // reciprocals of the edge direction components (0 if the component is 0)
    // inverse Vandermonde, Vi[ab * O2 + m]; phase 1 first parks the 4 + O2 traced feet (x, then y) here
    static constexpr int NVI = O2 * O2 > 2 * (4 + O2) ? O2 * O2 : 2 * (4 + O2);
    double Vi[NVI][CELLS];
    double xc[CELLS], yc[CELLS];           // centre of the node feet
    int r0[CELLS], s0[CELLS], nr[CELLS], ns[CELLS], mask[CELLS];
    unsigned short item[CELLS * 11];       // work item -> cell | candidate index << 7 | dr << 11 | ds << 13, 0xffff = padding
    int warp_tot[CELLS / 32];
};

template <int O, class SH>
__device__ __forceinline__ int geometry_setup(const double *__restrict__ va, const double *__restrict__ vb, int32_t *err,
                                              const GridDev &g, const Basis &bs, double tau, int order, int periodic,
                                              int t, int z, SH &sh, int c)
{
    constexpr int O2 = O * O;
    const int nx = g.n[0], ny = g.n[1];
    const int i = t % nx, j = t / nx;
    const long long vplane = (long long)(ny + 1) * (nx + 1);
    const double *a = va + z * vplane, *b = vb + z * vplane;
    const double tx = tau / g.h[0], ty = tau / g.h[1];

    // steps 1 and 4, tracing: the four corners (counter-clockwise from lower-left) and the O2 Gauss-Legendre nodes, feet
    // parked in this cell's column of sh.Vi (x at [pt], y at [4 + O2 + pt]).  Every point starts in the target cell, so
    // the first velocity look-up of eq. (15) uses the same four vertex values for all of them: loaded once.  The points
    // are traced in groups of TG, the second look-ups of a group (one cell each, wherever the half-step points fell)
    // requested together: a thread waits for global memory 1 + NPT / TG times instead of 2 NPT times (these waits were
    // 14 % of the kernel's stall samples).  The group loop stays rolled (code size).
    constexpr int NPT = 4 + O2;
    constexpr int TG = O == 3 ? 2 : 2;
    const int pitch = nx + 1;
    double av[4], bv[4];
    {
        const double *a0 = a + (long long)j * pitch + i, *b0 = b + (long long)j * pitch + i;
        av[0] = __ldg(a0); av[1] = __ldg(a0 + 1); av[2] = __ldg(a0 + pitch); av[3] = __ldg(a0 + pitch + 1);
        bv[0] = __ldg(b0); bv[1] = __ldg(b0 + 1); bv[2] = __ldg(b0 + pitch); bv[3] = __ldg(b0 + pitch + 1);
    }
    // foot of the characteristic through local (xi,eta) of cell (i,j), relative to that cell, cell units: eq. (14), or
    // eq. (15) as an explicit midpoint step whose half-step point is looked up, per axis, modulo the box (bitwise-periodic
    // field) or clamped; periodic 1: both axes, 0: none, 2: y only (polar plane: x = r bounded with zero radial velocity
    // at both ends, y = theta)
    const bool perx = periodic == 1, pery = periodic == 1 || periodic == 2;
#pragma unroll 1
    for (int p0 = 0; p0 < NPT; p0 += TG) {
        double xi[TG], eta[TG], ua[TG], ub[TG];
#pragma unroll
        for (int q = 0; q < TG; ++q) {
            const int pt = p0 + q < NPT ? p0 + q : NPT - 1;  // a last group may repeat the last point
            if (pt < 4) {
                xi[q] = (pt == 1 || pt == 2) ? 1.0 : 0.0;
                eta[q] = pt >= 2 ? 1.0 : 0.0;
            } else {
                xi[q] = bs.xi[O][(pt - 4) % O];
                eta[q] = bs.xi[O][(pt - 4) / O];
            }
            bilinear_val(av, bv, xi[q], eta[q], ua[q], ub[q]);
        }
        if (order != 1) {
            double lx[TG], ly[TG], wa[TG][4], wb[TG][4];
#pragma unroll
            for (int q = 0; q < TG; ++q) {
                const double mx = xi[q] - 0.5 * tx * ua[q], my = eta[q] - 0.5 * ty * ub[q];
                int fi = (int)floor(mx), fj = (int)floor(my);
                const int ci = perx ? wrap_idx(i + fi, nx) : min(max(i + fi, 0), nx - 1);
                const int cj = pery ? wrap_idx(j + fj, ny) : min(max(j + fj, 0), ny - 1);
                if (!perx) fi = ci - i;
                if (!pery) fj = cj - j;
                lx[q] = mx - fi;
                ly[q] = my - fj;
                const double *a0 = a + (long long)cj * pitch + ci, *b0 = b + (long long)cj * pitch + ci;
                wa[q][0] = __ldg(a0); wa[q][1] = __ldg(a0 + 1); wa[q][2] = __ldg(a0 + pitch); wa[q][3] = __ldg(a0 + pitch + 1);
                wb[q][0] = __ldg(b0); wb[q][1] = __ldg(b0 + 1); wb[q][2] = __ldg(b0 + pitch); wb[q][3] = __ldg(b0 + pitch + 1);
            }
#pragma unroll
            for (int q = 0; q < TG; ++q) bilinear_val(wa[q], wb[q], lx[q], ly[q], ua[q], ub[q]);
        }
#pragma unroll
        for (int q = 0; q < TG; ++q) {
            const int pt = p0 + q < NPT ? p0 + q : NPT - 1;
            sh.Vi[pt][c] = xi[q] - tx * ua[q];
            sh.Vi[NPT + pt][c] = eta[q] - ty * ub[q];
        }
    }
    // step 1: upstream quadrilateral
    double cx[4], cy[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        cx[e] = sh.Vi[e][c];
        cy[e] = sh.Vi[NPT + e][c];
    }
    const double xmin = dmin(dmin(cx[0], cx[1]), dmin(cx[2], cx[3]));
    const double ymin = dmin(dmin(cy[0], cy[1]), dmin(cy[2], cy[3]));
    const int r0 = (int)floor(xmin), s0 = (int)floor(ymin);
    int nr, ns;  // the bounding box covers source cells r0 .. r0+nr, s0 .. s0+ns
    {
        // Corners relative to the anchor cell (keeps |coordinates| <= 4).  Everything below -- edge
        // directions, clip parameters, crossings -- is derived from these rounded coordinates only, so
        // that the clipped pieces of neighbouring source cells fit together exactly.
        double qx[4], qy[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            qx[e] = cx[e] - r0;
            qy[e] = cy[e] - s0;
            sh.cx[e][c] = qx[e];
            sh.cy[e][c] = qy[e];
        }
        bool convex = true;
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const double e1x = qx[(e + 1) & 3] - qx[e], e1y = qy[(e + 1) & 3] - qy[e];
            const double e2x = qx[(e + 2) & 3] - qx[(e + 1) & 3], e2y = qy[(e + 2) & 3] - qy[(e + 1) & 3];
            if (!(e1x * e2y - e1y * e2x > 0.0)) convex = false;
            sh.idx[e][c] = e1x != 0.0 ? 1.0 / e1x : 0.0;
            sh.idy[e][c] = e1y != 0.0 ? 1.0 / e1y : 0.0;
        }
        if (!convex) atomicMin(err, SLDG_EGEOM);
        // half-open bounding box, taken from the same rounded coordinates (a foot exactly on a grid line
        // does not add a zero-area column, R12)
        const double xmax = dmax(dmax(qx[0], qx[1]), dmax(qx[2], qx[3]));
        const double ymax = dmax(dmax(qy[0], qy[1]), dmax(qy[2], qy[3]));
        nr = max((int)ceil(xmax) - 1, 0);
        ns = max((int)ceil(ymax) - 1, 0);
        if (nr > 2 || ns > 2) {
            atomicMin(err, SLDG_ESTENCIL);
            nr = min(nr, 2);
            ns = min(ns, 2);
        }
    }
    sh.r0[c] = r0;
    sh.s0[c] = s0;
    sh.nr[c] = nr;
    sh.ns[c] = ns;
    sh.mask[c] = 0;

    // step 4: node feet and adjoint polynomials in centred coordinates (relative to the anchor cell)
    double xc = 0.0, yc = 0.0;
    {
        double fx[O2], fy[O2];
#pragma unroll
        for (int m = 0; m < O2; ++m) {  // node m = p + O * qn
            const double px = sh.Vi[4 + m][c], py = sh.Vi[NPT + 4 + m][c];
            fx[m] = px - r0;
            fy[m] = py - s0;
            xc += px - r0;
            yc += py - s0;
        }
        xc *= 1.0 / O2;
        yc *= 1.0 / O2;
        if constexpr (O == 3) {
            // Vandermonde matrix straight into this cell's column of sh.Vi, inverted there in place
#pragma unroll
            for (int m = 0; m < O2; ++m) {
                double py = 1.0;
#pragma unroll
                for (int bq = 0; bq < O; ++bq) {
                    double px = 1.0;
#pragma unroll
                    for (int bp = 0; bp < O; ++bp) {
                        sh.Vi[m * O2 + bp + O * bq][c] = px * py;
                        px *= fx[m] - xc;
                    }
                    py *= fy[m] - yc;
                }
            }
            const double minpiv = invert_in_place<O2>(&sh.Vi[0][c], SH::CELLS);  // Vi[ab][m] = (V^-1)[ab][m]
            if (!(minpiv > 1e-10)) atomicMin(err, SLDG_EGEOM);
        } else {
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
        const double minpiv = gauss_jordan<O2>(V, Vi);  // phi*_m = sum_ab Vi[ab][m] (x-xc)^a (y-yc)^b
        if (!(minpiv > 1e-10)) atomicMin(err, SLDG_EGEOM);
#pragma unroll
        for (int ab = 0; ab < O2; ++ab)
#pragma unroll
            for (int m = 0; m < O2; ++m) sh.Vi[ab * O2 + m][c] = Vi[ab][m];
        }
    }
    sh.xc[c] = xc;
    sh.yc[c] = yc;
    return (nr + 1) * (ns + 1);
}

// steps 2, 3, 5 for one piece: target cell c of the block, candidate source cell (dr, ds) of its bounding box
// The pieces of one target cell sit on consecutive lanes of one warp, in slot order (k = candidate index of the
// lane): the non-empty ones are stored packed, W[cell][rank], rank from a warp ballot.  `valid` is false on padding
// lanes, which only take part in the ballot.
template <int O, class SH>
__device__ __forceinline__ void geometry_piece(const SH &sh, bool valid, int c, int k, int dr, int ds,
                                               const Basis &bs, double *__restrict__ Wcell, int *mask_out)
{
    constexpr int O2 = O * O, NM = 2 * O - 1;
    const int lane = threadIdx.x & 31;
    if (!valid) c = 0;
    double M[NM][NM];
    piece_moments<O>(sh, c, (double)dr, (double)ds, dr < sh.nr[c], bs, M);
    const bool nonempty = valid && M[0][0] > 0.0;
    const unsigned ballot = __ballot_sync(0xffffffffu, nonempty);
    if (!nonempty) return;  // empty intersection
    const int rank = __popc((ballot >> (lane - k)) & ((1u << k) - 1u));
    // phi*_m in the source cell's monomials: (x-xc)^a = sum_a' binom(a,a') (-xc)^(a-a') x^a'
    const double lxc = sh.xc[c] - dr, lyc = sh.yc[c] - ds;
    double cf[O2][O2];  // cf[a'+O b'][m]
    {
        double sxp[O][O], syp[O][O];  // sxp[a][a'] = binom(a,a') (-lxc)^(a-a')
#pragma unroll
        for (int aa = 0; aa < O; ++aa)
#pragma unroll
            for (int ap = 0; ap < O; ++ap) {
                const double bin = (ap > aa) ? 0.0 : ((aa == 2 && ap == 1) ? 2.0 : 1.0);
                double px = 1.0, py = 1.0;
#pragma unroll
                for (int e = 0; e < O; ++e)
                    if (e < aa - ap) {
                        px *= -lxc;
                        py *= -lyc;
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
                        for (int aa = ap; aa < O; ++aa)
                            acc = fma(sh.Vi[(aa + O * bb) * O2 + m][c], sxp[aa][ap] * syp[bb][bp_], acc);
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
            for (int qq = 0; qq < NM; ++qq) {
                double acc = 0.0;
#pragma unroll
                for (int pp = 0; pp < O; ++pp) acc = fma(bs.L[O][kp][pp], M[pp + ap][qq], acc);
                T[kp][ap][qq] = acc;
            }
    double iw[O2];
#pragma unroll
    for (int m = 0; m < O2; ++m) iw[m] = 1.0 / (bs.w[O][m % O] * bs.w[O][m / O]);
    const int slot = dr + 3 * ds;
    double *Wout = Wcell + (size_t)rank * sldg_w_block_doubles(O);
    // o = 3: the two loops over the source node stay rolled -- unrolled, the kernel's code no longer fits the
    // instruction cache (`no_instruction` was its largest stall) and T, cf spill anyway
#pragma unroll(O == 3 ? 1 : O)
    for (int kq = 0; kq < O; ++kq)
#pragma unroll(O == 3 ? 1 : O)
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
            double out[O2];
#pragma unroll
            for (int m = 0; m < O2; ++m) {
                double acc = 0.0;
#pragma unroll
                for (int ab = 0; ab < O2; ++ab) acc = fma(cf[ab][m], G[ab], acc);
                out[m] = acc * iw[m];
            }
            if (O == 2) {
                reinterpret_cast<double2 *>(Wout + k * O2)[0] = make_double2(out[0], out[1]);
                reinterpret_cast<double2 *>(Wout + k * O2)[1] = make_double2(out[O2 - 2], out[O2 - 1]);
            } else {
#pragma unroll
                for (int m = 0; m < O2; ++m) Wout[k * O2 + m] = out[m];
            }
        }
    atomicOr(mask_out, 1 << slot);
}

// The geometry of up to CELLS target cells of one z node by one thread block (see the two phases above).
// cell_of(c) -> index t = j * nx + i of the block's c-th cell, or -1.  Threads 0 .. CELLS-1 do phase 1, all
// `nthreads` (a multiple of 32, >= CELLS) phase 2.  Every thread of the block must call this (block barriers).
// WARP: the "block" is ONE warp (CELLS = nthreads = 32, tid = lane) that synchronises with __syncwarp only -- the
// geometry warps of the persistent 2d kernel (sldg_xy_apply.cu), which must not touch the block-wide barrier.
template <int O, int CELLS, bool WARP = false, class CellOf>
__device__ __forceinline__ void geometry_block(GeomShared<O, CELLS> &sh, int tid, int nthreads, CellOf cell_of, int z,
                                               const double *__restrict__ va, const double *__restrict__ vb,
                                               int4 *hdr, double *W, int32_t *err, const GridDev &g, const Basis &bs,
                                               double tau, int order, int periodic)
{
    static_assert(!WARP || CELLS == 32, "a geometry warp does 32 cells at a time");
    auto sync = [] {
        if constexpr (WARP) __syncwarp(); else __syncthreads();
    };
    const int lane = tid & 31, warp = tid >> 5;
    const int ncell = g.n[0] * g.n[1];
    const int t = tid < CELLS ? cell_of(tid) : -1;

    // phase 1: per-cell set-up, number of candidate source cells
    const int n = t >= 0 ? geometry_setup<O>(va, vb, err, g, bs, tau, order, periodic, t, z, sh, tid) : 0;
    // Enumerate the work items: the cells of a warp in order, a cell's items on consecutive lanes of ONE warp
    // (padded to the next multiple of 32 where they would straddle), each warp's list rounded up to 32.
    int first = 0, pos = 0;
    if (tid < CELLS) {
        // exclusive prefix of the counts over the warp; then, boundary by boundary, the first cell whose items would
        // straddle a multiple of 32 moves up to it, and every later cell with it (at most 9 boundaries; a loop over
        // the 32 lanes in turn was 3 % of the kernel's instructions)
        int S = n;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int u = __shfl_up_sync(0xffffffffu, S, d);
            if (lane >= d) S += u;
        }
        first = S - n;
        for (;;) {
            const unsigned strad = __ballot_sync(0xffffffffu, (first & 31) + n > 32);
            if (!strad) break;
            const int l0 = __ffs(strad) - 1;
            const int s0 = __shfl_sync(0xffffffffu, first, l0);
            if (lane >= l0) first += 32 - (s0 & 31);
        }
        pos = (__shfl_sync(0xffffffffu, first + n, 31) + 31) & ~31;
        if (lane == 0) sh.warp_tot[warp] = pos;
    }
    sync();
    int base = 0, total = 0;
    for (int w = 0; w < CELLS / 32; ++w) {
        if (w < warp) base += sh.warp_tot[w];
        total += sh.warp_tot[w];
    }
    for (int it = tid; it < total; it += nthreads) sh.item[it] = 0xffff;
    sync();
    {
        // item code: cell | candidate index k << 7 | dr << 11 | ds << 13 (k = dr + ds (nr + 1)): 15 bits, never 0xffff
        const int w = n > 0 ? sh.nr[tid < CELLS ? tid : 0] + 1 : 1;
        int dr = 0, ds = 0;
        for (int k = 0; k < n; ++k) {
            sh.item[base + first + k] = (unsigned short)(tid | (k << 7) | (dr << 11) | (ds << 13));
            if (++dr == w) {
                dr = 0;
                ++ds;
            }
        }
    }
    sync();

    // phase 2: one piece per thread and pass (whole warps: total is a multiple of 32)
    for (int it = tid; it < total; it += nthreads) {
        const int code = sh.item[it];
        const bool valid = code != 0xffff;
        const int cc = valid ? (code & 0x7f) : 0, k = valid ? ((code >> 7) & 15) : 0;
        const int dr = valid ? ((code >> 11) & 3) : 0, ds = valid ? ((code >> 13) & 3) : 0;
        const long long cellid = (long long)z * ncell + cell_of(cc);
        geometry_piece<O>(sh, valid, cc, k, dr, ds, bs, W + (size_t)cellid * 9 * sldg_w_block_doubles(O), &sh.mask[cc]);
    }
    sync();
    if (t >= 0) {
        const int m = sh.mask[tid];
        hdr[(long long)z * ncell + t] = make_int4(sh.r0[tid], sh.s0[tid], m, __popc(m));
    }
    sync();
}

}  // namespace sldg_geom
