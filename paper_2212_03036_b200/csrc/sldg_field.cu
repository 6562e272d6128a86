// sldg_field.cu -- the 3d field step of the drift-kinetic solver (Algorithm 1 steps 1 and 5; section
// 3.6; eq. (2)) and the invariants of PAPER.md:332-346.  OUTSIDE the timed hot path:
// 1/Nv of the volume.  Readings for BASELINE.json's Cartesian periodic box: DESIGN.md R19-R26.
//
//   rho (Gauss-Legendre nodes) --resample--> field grid: the nx x ny cell vertices (mean of the four adjacent cells'
//       polynomials at the corner, "since the function is discontinuous") x Nz equidistant z points inside
//       the cells, at (m + 1/2) h_z / o_z
//   -(1/n0) div(n0 grad phi) + (phi - <phi>)/Te = rho/n0 - 1,  <phi> = z average: second-order conservative differences;
//       the z average decouples the problem exactly (what the paper's FFT in z does mode by mode): one singular system
//       A <phi> = <rhs> (compatibility defect projected out, zero-mean solution), then (A + 1/Te) phi_m = rhs_m + <phi>/Te
//       for every z point.  All systems are symmetric positive (semi-)definite after multiplication by n0 and are solved
//       by Jacobi-preconditioned conjugate gradients, ONE THREAD BLOCK PER SYSTEM (no grid-wide reductions; the Nz
//       systems run side by side, the vectors stay in L2).
//   a = -d_y phi / B, b = d_x phi / B, E_z = -d_z phi by centred differences on the field grid, linear interpolation in
//       z to the Gauss-Legendre z nodes, bilinear interpolation in (x,y) to the nodes for E_z; written
//       where sldg_set_vxy / sldg_set_Ez would put them.
#include <math.h>
#include <stdlib.h>

#include "sldg_internal.cuh"

namespace {

__device__ __forceinline__ int wrapf(int i, int n) { return i < 0 ? i + n : (i >= n ? i - n : i); }

// l_j(x) of order o from the monomial coefficients of the basis tables
__device__ __forceinline__ double lagr(const Basis &bs, int o, int j, double x)
{
    double v = bs.L[o][j][o - 1];
    for (int a = o - 2; a >= 0; --a) v = fma(v, x, bs.L[o][j][a]);
    return v;
}

// rhs[m][j][i] = rho~ / n0 - 1 on the field grid
__global__ void __launch_bounds__(256) field_resample_kernel(const double *__restrict__ rho,
                                                             const double *__restrict__ n0,
                                                             double *__restrict__ rhs, GridDev g, Basis bs)
{
    const int nx = g.n[0], ny = g.n[1], Nz = g.N[2];
    const int ox = g.o[0], oy = g.o[1], oz = g.o[2];
    const long long total = (long long)Nz * ny * nx;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(t % nx), j = (int)((t / nx) % ny), m = (int)(t / ((long long)nx * ny));
        const int iz = m / oz, mp = m - iz * oz;
        const double zeta = (mp + 0.5) / oz;
        double acc = 0.0;
        for (int q = 0; q < oz; ++q) {
            const double lz = lagr(bs, oz, q, zeta);
            const double *plane = rho + (long long)(iz * oz + q) * g.N[1] * g.N[0];
            double sy = 0.0;
            for (int side_y = 0; side_y < 2; ++side_y) {          // 0: cell j-1 at its upper end, 1: cell j at its lower end
                const int cj = wrapf(j - 1 + side_y, ny);
                for (int bq = 0; bq < oy; ++bq) {
                    const double ly = lagr(bs, oy, bq, side_y ? 0.0 : 1.0);
                    const double *row = plane + (long long)(cj * oy + bq) * g.N[0];
                    double sx = 0.0;
                    for (int side_x = 0; side_x < 2; ++side_x) {
                        const int ci = wrapf(i - 1 + side_x, nx);
                        for (int ap = 0; ap < ox; ++ap) sx = fma(lagr(bs, ox, ap, side_x ? 0.0 : 1.0), row[ci * ox + ap], sx);
                    }
                    sy = fma(ly, 0.5 * sx, sy);
                }
            }
            acc = fma(lz, 0.5 * sy, acc);
        }
        rhs[t] = acc / n0[j * nx + i] - 1.0;
    }
}

// rbar[j][i] = mean over m of rhs
__global__ void __launch_bounds__(256) field_zmean_kernel(const double *__restrict__ rhs, double *__restrict__ rbar,
                                                          int ncell, int Nz)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= ncell) return;
    double s = 0.0;
    for (int m = 0; m < Nz; ++m) s += rhs[(long long)m * ncell + k];
    rbar[k] = s / Nz;
}

template <int T>
__device__ __forceinline__ void block_sum2(double &a, double &b, double *red)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        a += __shfl_xor_sync(0xffffffffu, a, off);
        b += __shfl_xor_sync(0xffffffffu, b, off);
    }
    __syncthreads();  // red may still be read from the previous call
    if (lane == 0) {
        red[2 * wid] = a;
        red[2 * wid + 1] = b;
    }
    __syncthreads();
    a = 0.0;
    b = 0.0;
    for (int w = 0; w < T / 32; ++w) {  // every thread sums in the same order: identical values everywhere
        a += red[2 * w];
        b += red[2 * w + 1];
    }
}

// c = sum n0 rbar / sum n0 (one block), then rbar -= c; the same c is later taken from every rhs_m
template <int T>
__global__ void __launch_bounds__(T) field_defect_kernel(const double *__restrict__ n0, double *__restrict__ rbar,
                                                         int ncell, double *__restrict__ c_out)
{
    __shared__ double red[2 * T / 32];
    double a = 0.0, b = 0.0;
    for (int k = threadIdx.x; k < ncell; k += T) {
        a = fma(n0[k], rbar[k], a);
        b += n0[k];
    }
    block_sum2<T>(a, b, red);
    const double c = a / b;
    for (int k = threadIdx.x; k < ncell; k += T) rbar[k] -= c;
    if (threadIdx.x == 0) *c_out = c;
}

// rhs_m += pbar / Te - c   (right-hand sides of the Nz systems with A + 1/Te)
__global__ void __launch_bounds__(256) field_rhs_shift_kernel(double *__restrict__ rhs, const double *__restrict__ pbar,
                                                              const double *__restrict__ Te, const double *__restrict__ c,
                                                              int ncell, long long total)
{
    const double cc = *c;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const int k = (int)(t % ncell);
        rhs[t] = rhs[t] - cc + pbar[k] / Te[k];
    }
}

// Jacobi-preconditioned conjugate gradients for  n0 (A + shift/Te) x = n0 b,  one block per system (blockIdx.x), all
// vectors of a system contiguous (ncell doubles).  A: conservative 5-point differences, face coefficient = mean of the two
// vertex values of n0, periodic.  Stops when |r| <= tol |n0 b| or after max_iter iterations.  zero_mean: the system is
// singular (shift = 0, constants); the mean of x is removed at the end.
template <int T>
__global__ void __launch_bounds__(T) field_cg_kernel(double *__restrict__ x_all, const double *__restrict__ b_all,
                                                     double *__restrict__ r_all, double *__restrict__ p_all,
                                                     double *__restrict__ q_all, const double *__restrict__ n0,
                                                     const double *__restrict__ Te, int nx, int ny, double ihx2,
                                                     double ihy2, double shift, double tol, int max_iter, int zero_mean,
                                                     int warm, int *__restrict__ iters, double *__restrict__ relres)
{
    __shared__ double red[2 * T / 32];
    const int N = nx * ny;
    const long long off = (long long)blockIdx.x * N;
    double *x = x_all + off, *r = r_all + off, *p = p_all + off, *q = q_all + off;
    const double *b = b_all + off;

    auto faces = [&](int k, double &nE, double &nW, double &nN, double &nS) {
        const int i = k % nx, j = k / nx;
        const double nc = n0[k];
        nE = 0.5 * (nc + n0[j * nx + wrapf(i + 1, nx)]);
        nW = 0.5 * (nc + n0[j * nx + wrapf(i - 1, nx)]);
        nN = 0.5 * (nc + n0[wrapf(j + 1, ny) * nx + i]);
        nS = 0.5 * (nc + n0[wrapf(j - 1, ny) * nx + i]);
    };
    auto diag = [&](int k) {
        double nE, nW, nN, nS;
        faces(k, nE, nW, nN, nS);
        return (nE + nW) * ihx2 + (nN + nS) * ihy2 + shift * n0[k] / Te[k];
    };

    // stencil of the symmetrised operator n0 (A + shift / Te) at vertex k
    auto apply = [&](const double *u, int k) {
        const int i = k % nx, j = k / nx;
        double nE, nW, nN, nS;
        faces(k, nE, nW, nN, nS);
        const double uc = u[k];
        return -(nE * (u[j * nx + wrapf(i + 1, nx)] - uc) - nW * (uc - u[j * nx + wrapf(i - 1, nx)])) * ihx2 -
               (nN * (u[wrapf(j + 1, ny) * nx + i] - uc) - nS * (uc - u[wrapf(j - 1, ny) * nx + i])) * ihy2 +
               shift * n0[k] / Te[k] * uc;
    };
    // start: x0 = 0, or (warm) the solution of the previous field step left in x -- in a time-stepping run the potential
    // changes little from one solve to the next and most of the iterations go away
    double rz = 0.0, bb = 0.0, r0 = 0.0;
    for (int k = threadIdx.x; k < N; k += T) {
        const double bk = n0[k] * b[k];
        double rk = bk;
        if (warm) rk -= apply(x, k);
        else x[k] = 0.0;
        const double zk = rk / diag(k);
        r[k] = rk;
        p[k] = zk;
        rz = fma(rk, zk, rz);
        bb = fma(bk, bk, bb);
        r0 = fma(rk, rk, r0);
    }
    {
        double dummy = 0.0;
        block_sum2<T>(r0, dummy, red);
    }
    block_sum2<T>(rz, bb, red);
    double rr = r0;
    int it = 0;
    if (!(bb > 0.0)) {
        for (int k = threadIdx.x; k < N; k += T) x[k] = 0.0;  // zero source: zero potential, whatever the initial guess
        rr = 0.0;
    }
    if (bb > 0.0) {
        for (; it < max_iter && rr > tol * tol * bb; ++it) {
            double pq = 0.0, dummy = 0.0;
            for (int k = threadIdx.x; k < N; k += T) {
                const double qk = apply(p, k);
                q[k] = qk;
                pq = fma(p[k], qk, pq);
            }
            block_sum2<T>(pq, dummy, red);
            const double alpha = rz / pq;
            double rz_new = 0.0;
            rr = 0.0;
            for (int k = threadIdx.x; k < N; k += T) {
                x[k] = fma(alpha, p[k], x[k]);
                const double rk = fma(-alpha, q[k], r[k]);
                r[k] = rk;
                const double zk = rk / diag(k);
                q[k] = zk;  // z parked in q until p is updated
                rz_new = fma(rk, zk, rz_new);
                rr = fma(rk, rk, rr);
            }
            block_sum2<T>(rz_new, rr, red);
            const double beta = rz_new / rz;
            rz = rz_new;
            for (int k = threadIdx.x; k < N; k += T) p[k] = fma(beta, p[k], q[k]);
            __syncthreads();  // p complete before the next stencil pass
        }
    }
    if (zero_mean) {
        double s = 0.0, dummy = 0.0;
        for (int k = threadIdx.x; k < N; k += T) s += x[k];
        block_sum2<T>(s, dummy, red);
        const double mean = s / N;
        for (int k = threadIdx.x; k < N; k += T) x[k] -= mean;
    }
    if (threadIdx.x == 0) {
        iters[blockIdx.x] = it;
        relres[blockIdx.x] = bb > 0.0 ? sqrt(rr / bb) : 0.0;
    }
}

}  // namespace

namespace {

// linear interpolation in z: GL z node Z (cell iz, node q) lies at s = (iz + xi_q) o_z - 1/2 in field-grid index units
__device__ __forceinline__ void z_stencil(const GridDev &g, const Basis &bs, int Z, int &m0, int &m1, double &w)
{
    const int oz = g.o[2], Nz = g.N[2];
    const int iz = Z / oz, q = Z - iz * oz;
    const double s = (iz + bs.xi[oz][q]) * oz - 0.5;
    const double fl = floor(s);
    w = s - fl;
    m0 = (int)fl;
    m1 = m0 + 1;
    m0 = m0 < 0 ? m0 + Nz : (m0 >= Nz ? m0 - Nz : m0);
    m1 = m1 < 0 ? m1 + Nz : (m1 >= Nz ? m1 - Nz : m1);
}

// a, b [Nz][ny+1][nx+1] at the cell vertices per GL z node (wrap row and column are copies: bitwise periodic)
__global__ void __launch_bounds__(256) field_drift_kernel(const double *__restrict__ phi, double *__restrict__ va,
                                                          double *__restrict__ vb, GridDev g, Basis bs, double invB)
{
    const int nx = g.n[0], ny = g.n[1], Nz = g.N[2];
    const long long ncell = (long long)nx * ny;
    const long long total = (long long)Nz * (ny + 1) * (nx + 1);
    const double i2hx = 1.0 / (2.0 * g.h[0]), i2hy = 1.0 / (2.0 * g.h[1]);
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const int iw = (int)(t % (nx + 1)), jw = (int)((t / (nx + 1)) % (ny + 1)), Z = (int)(t / ((long long)(nx + 1) * (ny + 1)));
        const int i = iw == nx ? 0 : iw, j = jw == ny ? 0 : jw;
        int m0, m1;
        double w;
        z_stencil(g, bs, Z, m0, m1, w);
        const int ip = wrapf(i + 1, nx), im = wrapf(i - 1, nx), jp = wrapf(j + 1, ny), jm = wrapf(j - 1, ny);
        double a[2], b[2];
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const double *pl = phi + (long long)(e ? m1 : m0) * ncell;
            a[e] = -(pl[jp * nx + i] - pl[jm * nx + i]) * i2hy * invB;
            b[e] = (pl[j * nx + ip] - pl[j * nx + im]) * i2hx * invB;
        }
        va[t] = (1.0 - w) * a[0] + w * a[1];
        vb[t] = (1.0 - w) * b[0] + w * b[1];
    }
}

// E_z = -d_z phi and phi itself at the (x,y,z) GL nodes: centred difference in z on the field grid, bilinear in the
// cell, linear in z
__global__ void __launch_bounds__(256) field_nodes_kernel(const double *__restrict__ phi, double *__restrict__ Ez,
                                                          double *__restrict__ phin, GridDev g, Basis bs)
{
    const int nx = g.n[0], ny = g.n[1], Nz = g.N[2], Nx = g.N[0], Ny = g.N[1];
    const int ox = g.o[0], oy = g.o[1];
    const long long ncell = (long long)nx * ny;
    const long long total = (long long)Nz * Ny * Nx;
    const double i2hz = 1.0 / (2.0 * (g.h[2] / g.o[2]));
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const int X = (int)(t % Nx), Y = (int)((t / Nx) % Ny), Z = (int)(t / ((long long)Nx * Ny));
        const int i = X / ox, j = Y / oy;
        const double xi = bs.xi[ox][X - i * ox], eta = bs.xi[oy][Y - j * oy];
        const int ip = wrapf(i + 1, nx), jp = wrapf(j + 1, ny);
        const double w00 = (1.0 - xi) * (1.0 - eta), w10 = xi * (1.0 - eta), w01 = (1.0 - xi) * eta, w11 = xi * eta;
        const int k00 = j * nx + i, k10 = j * nx + ip, k01 = jp * nx + i, k11 = jp * nx + ip;
        int m0, m1;
        double w;
        z_stencil(g, bs, Z, m0, m1, w);
        double e[2], p[2];
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            const int m = s ? m1 : m0;
            const double *pc = phi + (long long)m * ncell;
            const double *pu = phi + (long long)wrapf(m + 1, Nz) * ncell, *pd = phi + (long long)wrapf(m - 1, Nz) * ncell;
            e[s] = w00 * (-(pu[k00] - pd[k00]) * i2hz) + w10 * (-(pu[k10] - pd[k10]) * i2hz) +
                   w01 * (-(pu[k01] - pd[k01]) * i2hz) + w11 * (-(pu[k11] - pd[k11]) * i2hz);
            p[s] = w00 * pc[k00] + w10 * pc[k10] + w01 * pc[k01] + w11 * pc[k11];
        }
        Ez[t] = (1.0 - w) * e[0] + w * e[1];
        phin[t] = (1.0 - w) * p[0] + w * p[1];
    }
}

// Per line (z,Y,X): Gauss sums over v of f, f^2 and v^2/2 f, times the line's (x,y,z) Gauss weight; block partials of
// mass, L2^2, kinetic and potential energy.  One warp per line.
__global__ void __launch_bounds__(256) field_moments_kernel(const double *__restrict__ f, const double *__restrict__ phin,
                                                            double *__restrict__ partials, GridDev g, Basis bs)
{
    __shared__ double red[8][4];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const unsigned warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarp = (gridDim.x * blockDim.x) >> 5;
    const int Nv = g.N[3], ov = g.o[3];
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    for (unsigned line = warp; line < (unsigned)g.lines; line += nwarp) {
        const unsigned X = line % (unsigned)g.N[0], t = line / (unsigned)g.N[0];
        const unsigned Y = t % (unsigned)g.N[1], Z = t / (unsigned)g.N[1];
        const double *u = f + (long long)Z * g.sZ + (long long)Y * g.sY + (long long)X * g.sX;
        double s1 = 0.0, s2 = 0.0, s3 = 0.0;
        for (int v = lane; v < Nv; v += 32) {
            const int cell = v / ov, q = v - cell * ov;
            const double vv = g.lo[3] + (cell + bs.xi[ov][q]) * g.h[3];
            const double wq = bs.w[ov][q], fv = u[v];
            s1 = fma(wq, fv, s1);
            s2 = fma(wq * fv, fv, s2);
            s3 = fma(wq * 0.5 * vv * vv, fv, s3);
        }
        const double wl = bs.w[g.o[0]][X % g.o[0]] * bs.w[g.o[1]][Y % g.o[1]] * bs.w[g.o[2]][Z % g.o[2]];
        acc[0] = fma(wl, s1, acc[0]);
        acc[1] = fma(wl, s2, acc[1]);
        acc[2] = fma(wl, s3, acc[2]);
        acc[3] = fma(wl * phin[line], s1, acc[3]);
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) {
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) acc[k] += __shfl_xor_sync(0xffffffffu, acc[k], off);
        if (lane == 0) red[wid][k] = acc[k];
    }
    __syncthreads();
    if (threadIdx.x < 4) {
        double s = 0.0;
        for (int w = 0; w < 8; ++w) s += red[w][threadIdx.x];
        partials[4 * blockIdx.x + threadIdx.x] = s;
    }
}

// Electric energy: phi sampled bilinearly on the circle of radius r_p around the box centre at nth angles, all z points
// of the field grid; one block; out[4] = sum phi^2
template <int T>
__global__ void __launch_bounds__(T) field_circle_kernel(const double *__restrict__ phi, GridDev g, double r_p, int nth,
                                                         const double *__restrict__ partials, int nblk,
                                                         double *__restrict__ out)
{
    __shared__ double red[2 * T / 32];
    const int nx = g.n[0], ny = g.n[1], Nz = g.N[2];
    const double cx = g.lo[0] + 0.5 * nx * g.h[0], cy = g.lo[1] + 0.5 * ny * g.h[1];
    double acc = 0.0, dummy = 0.0;
    for (long long t = threadIdx.x; t < (long long)nth * Nz; t += T) {
        const int a = (int)(t % nth), m = (int)(t / nth);
        const double th = 2.0 * 3.14159265358979323846 * (a + 0.5) / nth;
        const double sx = (cx + r_p * cos(th) - g.lo[0]) / g.h[0], sy = (cy + r_p * sin(th) - g.lo[1]) / g.h[1];
        const double fx = floor(sx), fy = floor(sy);
        const double wx = sx - fx, wy = sy - fy;
        int i0 = (int)fx % nx, j0 = (int)fy % ny;
        if (i0 < 0) i0 += nx;
        if (j0 < 0) j0 += ny;
        const int i1 = wrapf(i0 + 1, nx), j1 = wrapf(j0 + 1, ny);
        const double *pl = phi + (long long)m * nx * ny;
        const double v = (1 - wx) * (1 - wy) * pl[j0 * nx + i0] + wx * (1 - wy) * pl[j0 * nx + i1] +
                         (1 - wx) * wy * pl[j1 * nx + i0] + wx * wy * pl[j1 * nx + i1];
        acc = fma(v, v, acc);
    }
    block_sum2<T>(acc, dummy, red);
    // the four volume sums: reduce the block partials of field_moments_kernel here as well
    double s[4] = {0.0, 0.0, 0.0, 0.0};
    for (int k = threadIdx.x; k < nblk; k += T)
        for (int e = 0; e < 4; ++e) s[e] += partials[4 * k + e];
    block_sum2<T>(s[0], s[1], red);
    block_sum2<T>(s[2], s[3], red);
    if (threadIdx.x == 0) {
        out[0] = s[0];
        out[1] = s[1];
        out[2] = s[2];
        out[3] = s[3];
        out[4] = acc;
    }
}

}  // namespace

// ---- host side --------------------------------------------------------------------------------------------

size_t field_workspace_bytes(const sldg_params *p)
{
    const size_t ncell = (size_t)p->n[0] * p->n[1], Nz = (size_t)p->n[2] * p->order[2];
    const size_t lines = Nz * (size_t)p->n[0] * p->order[0] * p->n[1] * p->order[1];
    auto al = [](size_t b) { return (b + 255) & ~(size_t)255; };
    // n0, Te | phi, rhs, r, p, q (field grid) | 5 vectors of the <phi> system | phi at the nodes | scalars | per-system info
    return 2 * al(ncell * 8) + 5 * al(Nz * ncell * 8) + 5 * al(ncell * 8) + al(lines * 8) + al(256) + al((Nz + 1) * 4) +
           al((Nz + 1) * 8);
}

void field_carve(sldg_ctx *c, char *base)
{
    const GridDev &g = c->g;
    const size_t ncell = (size_t)g.n[0] * g.n[1], Nz = (size_t)g.N[2];
    auto al = [](size_t b) { return (b + 255) & ~(size_t)255; };
    size_t off = 0;
    auto take = [&](size_t bytes) { char *at = base + off; off += al(bytes); return at; };
    FieldWs &f = c->fld;
    f.n0 = (double *)take(ncell * 8);
    f.Te = (double *)take(ncell * 8);
    f.phi = (double *)take(Nz * ncell * 8);
    f.rhs = (double *)take(Nz * ncell * 8);
    f.r = (double *)take(Nz * ncell * 8);
    f.p = (double *)take(Nz * ncell * 8);
    f.q = (double *)take(Nz * ncell * 8);
    for (int k = 0; k < 5; ++k) f.bar[k] = (double *)take(ncell * 8);
    f.phin = (double *)take((size_t)g.lines * 8);
    f.scal = (double *)take(256);
    f.iters = (int *)take((Nz + 1) * 4);
    f.relres = (double *)take((Nz + 1) * 8);
    f.invB = 1.0;
    f.have_profiles = 0;
    f.have_phi = 0;
}

static int field_grid_blocks(const sldg_ctx *c, long long total)
{
    long long nblk = (total + 255) / 256, cap = (long long)c->sm_count * 16;
    return (int)(nblk < cap ? nblk : cap);
}

cudaError_t launch_field_step(sldg_ctx *c, const double *fin, double tol, int max_iter)
{
    const GridDev &g = c->g;
    FieldWs &f = c->fld;
    const int nx = g.n[0], ny = g.n[1], Nz = g.N[2];
    const int ncell = nx * ny;
    const long long total = (long long)Nz * ncell;
    constexpr int T = 1024;
    cudaStream_t st = c->stream;
    const int warm = f.have_phi && !getenv("SLDG_FIELD_COLD") ? 1 : 0;  // previous potential as the initial guess
    cudaError_t e = launch_charge_density(c, fin, c->rho_ws);
    if (e != cudaSuccess) return e;
    field_resample_kernel<<<field_grid_blocks(c, total), 256, 0, st>>>(c->rho_ws, f.n0, f.rhs, g, c->basis);
    // <phi>: bar[0] = x, bar[1] = b, bar[2..4] = r, p, q
    field_zmean_kernel<<<(ncell + 255) / 256, 256, 0, st>>>(f.rhs, f.bar[1], ncell, Nz);
    field_defect_kernel<T><<<1, T, 0, st>>>(f.n0, f.bar[1], ncell, f.scal);
    const double ihx2 = 1.0 / (g.h[0] * g.h[0]), ihy2 = 1.0 / (g.h[1] * g.h[1]);
    field_cg_kernel<T><<<1, T, 0, st>>>(f.bar[0], f.bar[1], f.bar[2], f.bar[3], f.bar[4], f.n0, f.Te, nx, ny, ihx2, ihy2, 0.0,
                                        tol, max_iter, 1, warm, f.iters + Nz, f.relres + Nz);
    field_rhs_shift_kernel<<<field_grid_blocks(c, total), 256, 0, st>>>(f.rhs, f.bar[0], f.Te, f.scal, ncell, total);
    field_cg_kernel<T><<<Nz, T, 0, st>>>(f.phi, f.rhs, f.r, f.p, f.q, f.n0, f.Te, nx, ny, ihx2, ihy2, 1.0, tol, max_iter, 0,
                                         warm, f.iters, f.relres);
    field_drift_kernel<<<field_grid_blocks(c, (long long)Nz * (ny + 1) * (nx + 1)), 256, 0, st>>>(f.phi, c->va, c->vb, g,
                                                                                                 c->basis, f.invB);
    field_nodes_kernel<<<field_grid_blocks(c, g.lines), 256, 0, st>>>(f.phi, c->Ez, f.phin, g, c->basis);
    c->vel_periodic = 1;
    f.have_phi = 1;
    c->launches += 9;
    return cudaGetLastError();
}

// out_host[5]: electric energy, mass, L2 norm, kinetic energy, potential energy.  Synchronises.
cudaError_t launch_diagnostics(sldg_ctx *c, const double *fin, double r_p, double *out_host)
{
    const GridDev &g = c->g;
    FieldWs &f = c->fld;
    long long nb = (g.lines + 7) / 8;
    const long long cap = (long long)(c->n_partials / 4);
    const int grid = (int)(nb < cap ? nb : cap);
    field_moments_kernel<<<grid, 256, 0, c->stream>>>(fin, f.phin, c->partials, g, c->basis);
    const int nth = 4 * (g.n[0] > g.n[1] ? g.n[0] : g.n[1]);
    field_circle_kernel<1024><<<1, 1024, 0, c->stream>>>(f.phi, g, r_p, nth, c->partials, grid, f.scal + 8);
    c->launches += 2;
    double s[5];
    cudaError_t e = cudaMemcpyAsync(s, f.scal + 8, sizeof(s), cudaMemcpyDeviceToHost, c->stream);
    if (e != cudaSuccess) return e;
    e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return e;
    const double vol = g.h[0] * g.h[1] * g.h[2] * g.h[3];
    out_host[0] = sqrt(s[4] * (2.0 * 3.14159265358979323846 / nth) * (g.h[2] / g.o[2]));
    out_host[1] = s[0] * vol;
    out_host[2] = sqrt(s[1] * vol);
    out_host[3] = s[2] * vol;
    out_host[4] = s[3] * vol;
    return cudaGetLastError();
}
