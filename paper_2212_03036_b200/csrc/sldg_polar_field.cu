// sldg_polar_field.cu -- the paper's own quasi-neutrality solver, polar coordinates (eq. (2); boundary
// conditions PAPER.md:43; section 3.6).  Axis 0 of the grid is r, axis 1 theta.  Outside the timed path.
//
//   rho = int dg dv at the nodes --resample--> field grid: r vertices i = 0..nr, theta vertices j < nth (periodic), Nz
//       equidistant z points; a vertex takes the mean of the adjacent cells' polynomials at that corner (two cells at the
//       radial ends); rhs = rho~ / (r n0)
//   Fourier transform in theta and z ("we can use FFT in the (theta, z) plane"): discrete Fourier sums written out as
//       one kernel per axis (n <= a few hundred per axis and 1/Nv of the volume: a matrix-vector product per line is
//       micro-seconds; no cuFFT plan, no extra library to load)
//   per mode (kz, m): -[phi'' + (1/r + n0'/n0) phi' - m^2 phi / r^2] + [kz != 0] phi / Te = rhs, second-order centred
//       differences, phi'(r_min) = 0 (ghost value phi_{-1} = phi_1), phi(r_max) = 0: a tridiagonal system, Thomas
//       algorithm, one thread per mode ("for each degree of freedom in the theta and z direction, a tridiagonal linear
//       system has to be solved"); <phi> = z average (R21) removes the 1/Te term from the kz = 0 modes
//   back-transform; a = -d_theta phi / r, b = d_r phi / r at the vertices (a exactly zero at r_min and r_max),
//       E_z = -d_z phi, d_z phi, d_theta phi at the nodes: second-order differences, (bi)linear interpolation -- written where
//       sldg_set_vxy(.., 2), sldg_set_Ez and sldg_set_source_fields would put them.
#include <math.h>

#include "sldg_internal.cuh"

namespace {

__device__ __forceinline__ int wrapp(int i, int n) { return i < 0 ? i + n : (i >= n ? i - n : i); }

__device__ __forceinline__ double lagr1(const Basis &bs, int o, int j, double x)
{
    double v = bs.L[o][j][o - 1];
    for (int a = o - 2; a >= 0; --a) v = fma(v, x, bs.L[o][j][a]);
    return v;
}

// rhs[m][j][i] (complex, imaginary part 0) = rho~ / (r n0) on the field grid
__global__ void __launch_bounds__(256) polar_resample_kernel(const double *__restrict__ rho, const double *__restrict__ rn0,
                                                             double2 *__restrict__ rhs, GridDev g, Basis bs)
{
    const int nr = g.n[0], nth = g.n[1], Nz = g.N[2], nr1 = nr + 1;
    const int orr = g.o[0], oth = g.o[1], oz = g.o[2];
    const long long total = (long long)Nz * nth * nr1;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(t % nr1), j = (int)((t / nr1) % nth), m = (int)(t / ((long long)nr1 * nth));
        const int iz = m / oz, mp = m - iz * oz;
        double acc = 0.0;
        for (int q = 0; q < oz; ++q) {
            const double lz = lagr1(bs, oz, q, (mp + 0.5) / oz);
            const double *plane = rho + (long long)(iz * oz + q) * g.N[1] * g.N[0];
            double sy = 0.0;
            for (int side_y = 0; side_y < 2; ++side_y) {
                const int cj = wrapp(j - 1 + side_y, nth);
                for (int bq = 0; bq < oth; ++bq) {
                    const double *row = plane + (long long)(cj * oth + bq) * g.N[0];
                    double sx = 0.0;
                    int cnt = 0;
                    for (int side_x = 0; side_x < 2; ++side_x) {
                        const int ci = i - 1 + side_x;  // cell i-1 at its outer end, cell i at its inner end
                        if (ci < 0 || ci >= nr) continue;
                        ++cnt;
                        for (int ap = 0; ap < orr; ++ap) sx = fma(lagr1(bs, orr, ap, side_x ? 0.0 : 1.0), row[ci * orr + ap], sx);
                    }
                    sy = fma(lagr1(bs, oth, bq, side_y ? 0.0 : 1.0), cnt == 2 ? 0.5 * sx : sx, sy);
                }
            }
            acc = fma(lz, 0.5 * sy, acc);
        }
        rhs[t] = make_double2(acc / rn0[i], 0.0);
    }
}

// One axis of a discrete Fourier transform: data [outer][n][inner] complex, out[o][k][x] = sum_a in[o][a][x] w^(a k),
// w = exp(sign 2 pi i / n) from the table tw[n] (forward table; the inverse uses the conjugate); scale on output
__global__ void __launch_bounds__(256) dft_axis_kernel(const double2 *__restrict__ in, double2 *__restrict__ out, int outer,
                                                       int n, int inner, const double2 *__restrict__ tw, int inverse,
                                                       double scale)
{
    const long long total = (long long)outer * n * inner;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const int x = (int)(t % inner), k = (int)((t / inner) % n);
        const long long o = t / ((long long)inner * n);
        const double2 *src = in + o * n * inner + x;
        double re = 0.0, im = 0.0;
        int idx = 0;  // (a k) mod n
        for (int a = 0; a < n; ++a) {
            const double2 v = src[(long long)a * inner];
            double2 w = __ldg(tw + idx);
            if (inverse) w.y = -w.y;
            re = fma(v.x, w.x, re);
            re = fma(-v.y, w.y, re);
            im = fma(v.x, w.y, im);
            im = fma(v.y, w.x, im);
            idx += k;
            if (idx >= n) idx -= n;
        }
        out[t] = make_double2(re * scale, im * scale);
    }
}

__global__ void twiddle_kernel(double2 *tw, int n)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    double s, c;
    sincospi(-2.0 * k / n, &s, &c);
    tw[k] = make_double2(c, s);
}

// Thomas algorithm per mode (kz, kth); spectrum [Nz][nth][nr1] complex, solved in place; cp: scratch [modes][nr]
__global__ void __launch_bounds__(128) polar_tridiag_kernel(double2 *__restrict__ spec, double *__restrict__ cp,
                                                            const double *__restrict__ dln, const double *__restrict__ Te,
                                                            int Nz, int nth, int nr, double rmin, double h)
{
    const int mode = blockIdx.x * blockDim.x + threadIdx.x;
    if (mode >= Nz * nth) return;
    const int kz = mode / nth, j = mode - kz * nth;
    const int mth = j <= nth / 2 ? j : j - nth;  // integer mode number of d/dtheta (the Nyquist mode counts as +nth/2)
    const double m2 = (double)mth * mth, ih2 = 1.0 / (h * h);
    double2 *d = spec + (long long)mode * (nr + 1);
    double *c = cp + (long long)mode * nr;
    double cprev = 0.0;
    double2 dprev = make_double2(0.0, 0.0);
    for (int i = 0; i < nr; ++i) {
        const double r = rmin + i * h;
        const double adv = (1.0 / r + dln[i]) / (2.0 * h);
        const double diag = 2.0 * ih2 + m2 / (r * r) + (kz != 0 ? 1.0 / Te[i] : 0.0);
        double lo = -ih2 + adv, hi = -ih2 - adv;
        if (i == 0) {
            hi += lo;  // phi_{-1} = phi_1
            lo = 0.0;
        }
        const double den = diag - lo * cprev;
        cprev = hi / den;
        c[i] = cprev;
        const double2 di = d[i];
        dprev = make_double2((di.x - lo * dprev.x) / den, (di.y - lo * dprev.y) / den);
        d[i] = dprev;
    }
    d[nr] = make_double2(0.0, 0.0);
    double2 x = d[nr - 1];
    for (int i = nr - 2; i >= 0; --i) {
        const double2 di = d[i];
        x = make_double2(di.x - c[i] * x.x, di.y - c[i] * x.y);
        d[i] = x;
    }
}

__global__ void __launch_bounds__(256) real_part_kernel(const double2 *__restrict__ in, double *__restrict__ out, long long n)
{
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x)
        out[t] = in[t].x;
}

__device__ __forceinline__ void z_stencil_p(const GridDev &g, const Basis &bs, int Z, int &m0, int &m1, double &w)
{
    const int oz = g.o[2], Nz = g.N[2];
    const int iz = Z / oz, q = Z - iz * oz;
    const double s = (iz + bs.xi[oz][q]) * oz - 0.5;
    const double fl = floor(s);
    w = s - fl;
    m0 = wrapp((int)fl, Nz);
    m1 = wrapp((int)fl + 1, Nz);
}

// a, b [Nz][nth+1][nr+1] at the vertices per GL z node (theta wrap row copied)
__global__ void __launch_bounds__(256) polar_drift_kernel(const double *__restrict__ phi, double *__restrict__ va,
                                                          double *__restrict__ vb, GridDev g, Basis bs)
{
    const int nr = g.n[0], nth = g.n[1], Nz = g.N[2], nr1 = nr + 1;
    const long long plane = (long long)nth * nr1;
    const long long total = (long long)Nz * (nth + 1) * nr1;
    const double h = g.h[0], hth = g.h[1];
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(t % nr1), jw = (int)((t / nr1) % (nth + 1)), Z = (int)(t / ((long long)nr1 * (nth + 1)));
        const int j = jw == nth ? 0 : jw;
        const double r = g.lo[0] + i * h;
        int m0, m1;
        double w;
        z_stencil_p(g, bs, Z, m0, m1, w);
        double a[2], b[2];
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const double *pl = phi + (long long)(e ? m1 : m0) * plane;
            const double dth = (pl[wrapp(j + 1, nth) * nr1 + i] - pl[wrapp(j - 1, nth) * nr1 + i]) / (2.0 * hth);
            double dr;
            if (i == 0) dr = 0.0;
            else if (i == nr) dr = (3.0 * pl[j * nr1 + nr] - 4.0 * pl[j * nr1 + nr - 1] + pl[j * nr1 + nr - 2]) / (2.0 * h);
            else dr = (pl[j * nr1 + i + 1] - pl[j * nr1 + i - 1]) / (2.0 * h);
            a[e] = (i == 0 || i == nr) ? 0.0 : -dth / r;
            b[e] = dr / r;
        }
        va[t] = (1.0 - w) * a[0] + w * a[1];
        vb[t] = (1.0 - w) * b[0] + w * b[1];
    }
}

// E_z = -d_z phi, d_z phi and d_theta phi at the (r, theta, z) GL nodes
__global__ void __launch_bounds__(256) polar_nodes_kernel(const double *__restrict__ phi, double *__restrict__ Ez,
                                                          double *__restrict__ dzp, double *__restrict__ dthp, GridDev g,
                                                          Basis bs)
{
    const int nr = g.n[0], nth = g.n[1], Nz = g.N[2], nr1 = nr + 1, Nr = g.N[0], Nth = g.N[1];
    const int orr = g.o[0], oth = g.o[1];
    const long long plane = (long long)nth * nr1;
    const long long total = (long long)Nz * Nth * Nr;
    const double i2hz = 1.0 / (2.0 * (g.h[2] / g.o[2])), i2hth = 1.0 / (2.0 * g.h[1]);
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const int X = (int)(t % Nr), Y = (int)((t / Nr) % Nth), Z = (int)(t / ((long long)Nr * Nth));
        const int i = X / orr, j = Y / oth;
        const double xi = bs.xi[orr][X - i * orr], eta = bs.xi[oth][Y - j * oth];
        const int jp = wrapp(j + 1, nth);
        const double w00 = (1.0 - xi) * (1.0 - eta), w10 = xi * (1.0 - eta), w01 = (1.0 - xi) * eta, w11 = xi * eta;
        int m0, m1;
        double w;
        z_stencil_p(g, bs, Z, m0, m1, w);
        double e[2], d[2];
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            const int m = s ? m1 : m0;
            const double *pc = phi + (long long)m * plane;
            const double *pu = phi + (long long)wrapp(m + 1, Nz) * plane, *pd = phi + (long long)wrapp(m - 1, Nz) * plane;
            auto ez = [&](int jj, int ii) { return -(pu[jj * nr1 + ii] - pd[jj * nr1 + ii]) * i2hz; };
            auto dt = [&](int jj, int ii) { return (pc[wrapp(jj + 1, nth) * nr1 + ii] - pc[wrapp(jj - 1, nth) * nr1 + ii]) * i2hth; };
            e[s] = w00 * ez(j, i) + w10 * ez(j, i + 1) + w01 * ez(jp, i) + w11 * ez(jp, i + 1);
            d[s] = w00 * dt(j, i) + w10 * dt(j, i + 1) + w01 * dt(jp, i) + w11 * dt(jp, i + 1);
        }
        const double ezv = (1.0 - w) * e[0] + w * e[1];
        Ez[t] = ezv;
        dzp[t] = -ezv;
        dthp[t] = (1.0 - w) * d[0] + w * d[1];
    }
}

}  // namespace

// ---- host side --------------------------------------------------------------------------------------------
size_t polar_workspace_bytes(const sldg_params *p)
{
    const size_t nr1 = (size_t)p->n[0] + 1, nth = p->n[1], Nz = (size_t)p->n[2] * p->order[2];
    auto al = [](size_t b) { return (b + 255) & ~(size_t)255; };
    const size_t grid = Nz * nth * nr1;
    return 3 * al(nr1 * 8) + 2 * al(grid * 16) + al(grid * 8) + al(Nz * nth * nr1 * 8) + al((nth + Nz) * 16);
}

void polar_carve(sldg_ctx *c, char *base)
{
    const GridDev &g = c->g;
    const size_t nr1 = (size_t)g.n[0] + 1, nth = g.n[1], Nz = g.N[2];
    auto al = [](size_t b) { return (b + 255) & ~(size_t)255; };
    const size_t grid = Nz * nth * nr1;
    size_t off = 0;
    auto take = [&](size_t bytes) { char *at = base + off; off += al(bytes); return at; };
    PolarWs &w = c->pol;
    w.rn0 = (double *)take(nr1 * 8);
    w.dln = (double *)take(nr1 * 8);
    w.Te = (double *)take(nr1 * 8);
    w.ca = (double2 *)take(grid * 16);
    w.cb = (double2 *)take(grid * 16);
    w.phi = (double *)take(grid * 8);
    w.cp = (double *)take(Nz * nth * nr1 * 8);
    w.tw_th = (double2 *)take((nth + Nz) * 16);
    w.tw_z = w.tw_th + nth;
    w.ready = 0;
    w.have_phi = 0;
}

cudaError_t launch_polar_profiles(sldg_ctx *c, const double *rn0, const double *dln, const double *Te)
{
    const GridDev &g = c->g;
    PolarWs &w = c->pol;
    const size_t b = ((size_t)g.n[0] + 1) * 8;
    cudaError_t e;
    if ((e = cudaMemcpyAsync(w.rn0, rn0, b, cudaMemcpyDeviceToDevice, c->stream)) != cudaSuccess) return e;
    if ((e = cudaMemcpyAsync(w.dln, dln, b, cudaMemcpyDeviceToDevice, c->stream)) != cudaSuccess) return e;
    if ((e = cudaMemcpyAsync(w.Te, Te, b, cudaMemcpyDeviceToDevice, c->stream)) != cudaSuccess) return e;
    twiddle_kernel<<<(g.n[1] + 127) / 128, 128, 0, c->stream>>>(w.tw_th, g.n[1]);
    twiddle_kernel<<<(g.N[2] + 127) / 128, 128, 0, c->stream>>>(w.tw_z, g.N[2]);
    c->launches += 2;
    w.ready = 1;
    return cudaGetLastError();
}

cudaError_t launch_polar_field_step(sldg_ctx *c, const double *fin)
{
    const GridDev &g = c->g;
    PolarWs &w = c->pol;
    const int nr = g.n[0], nth = g.n[1], Nz = g.N[2], nr1 = nr + 1;
    const long long grid = (long long)Nz * nth * nr1;
    auto blocks = [&](long long total) {
        long long nb = (total + 255) / 256, cap = (long long)c->sm_count * 16;
        return (unsigned)(nb < cap ? nb : cap);
    };
    cudaStream_t st = c->stream;
    cudaError_t e = launch_charge_density(c, fin, c->rho_ws);
    if (e != cudaSuccess) return e;
    polar_resample_kernel<<<blocks(grid), 256, 0, st>>>(c->rho_ws, w.rn0, w.ca, g, c->basis);
    // forward: theta ([Nz][nth][nr1]: outer Nz, inner nr1), then z (outer 1, inner nth nr1)
    dft_axis_kernel<<<blocks(grid), 256, 0, st>>>(w.ca, w.cb, Nz, nth, nr1, w.tw_th, 0, 1.0);
    dft_axis_kernel<<<blocks(grid), 256, 0, st>>>(w.cb, w.ca, 1, Nz, nth * nr1, w.tw_z, 0, 1.0);
    polar_tridiag_kernel<<<(Nz * nth + 127) / 128, 128, 0, st>>>(w.ca, w.cp, w.dln, w.Te, Nz, nth, nr, g.lo[0], g.h[0]);
    dft_axis_kernel<<<blocks(grid), 256, 0, st>>>(w.ca, w.cb, 1, Nz, nth * nr1, w.tw_z, 1, 1.0 / Nz);
    dft_axis_kernel<<<blocks(grid), 256, 0, st>>>(w.cb, w.ca, Nz, nth, nr1, w.tw_th, 1, 1.0 / nth);
    real_part_kernel<<<blocks(grid), 256, 0, st>>>(w.ca, w.phi, grid);
    polar_drift_kernel<<<blocks((long long)Nz * (nth + 1) * nr1), 256, 0, st>>>(w.phi, c->va, c->vb, g, c->basis);
    polar_nodes_kernel<<<blocks(g.lines), 256, 0, st>>>(w.phi, c->Ez, c->src_dz, c->src_dth, g, c->basis);
    c->vel_periodic = 2;
    c->src_ready |= 2;
    w.have_phi = 1;
    c->launches += 10;
    return cudaGetLastError();
}
