// sldg_sweeps.cu -- 1d SLDG sweeps along z and v (eq. 11), charge density,
// mass and the canonical <-> internal layout transposes.  sm_100a.
//
// Internal layout: v fastest.  Element (z,Y,X,v) lives at z*sZ + Y*sY + X*sX + v; every (z,Y,X) "line"
// of Nv doubles is contiguous and starts on a 128-byte boundary (pitch Pv).
#include "sldg_internal.cuh"

// --------------------------------------------------------------------------------------------------
// small helpers
// --------------------------------------------------------------------------------------------------
__device__ __forceinline__ long long line_base(const GridDev &g, long long line)
{
    // line = (z*Ny + Y)*Nx + X  (canonical enumeration of the (x,y,z) nodes)
    int X = (int)(line % g.N[0]);
    long long t = line / g.N[0];
    int Y = (int)(t % g.N[1]);
    int z = (int)(t / g.N[1]);
    return z * g.sZ + Y * g.sY + X * g.sX;
}

// Courant number -> (s, alpha): the foot of the left edge of cell i lies in cell i+s at offset alpha
// (PAPER.md:164-168).  Uncontracted multiply/divide so that the branch of floor() is taken from the
// same IEEE value a plain C implementation computes.
__device__ __forceinline__ void shift_of(double speed, double tau, double h, int &s, double &alpha)
{
    double delta = __ddiv_rn(__dmul_rn(speed, tau), h);
    double fl = floor(-delta);
    s = (int)fl;
    alpha = -delta - fl;
}

template <int O>
__device__ __forceinline__ void eval_shift(const ShiftPoly &sp, double alpha, double (&A)[O][O],
                                           double (&B)[O][O])
{
#pragma unroll
    for (int j = 0; j < O; ++j)
#pragma unroll
        for (int m = 0; m < O; ++m) {
            double pa = sp.a[j][m][2 * O - 1], pb = sp.b[j][m][2 * O - 1];
#pragma unroll
            for (int d = 2 * O - 2; d >= 0; --d) {
                pa = fma(pa, alpha, sp.a[j][m][d]);
                pb = fma(pb, alpha, sp.b[j][m][d]);
            }
            A[j][m] = pa;
            B[j][m] = pb;
        }
}

__device__ __forceinline__ int wrapi(int i, int n)
{
    int r = i % n;
    return r < 0 ? r + n : r;
}

// --------------------------------------------------------------------------------------------------
// canonical [Nz][Nv][Ny][Nx]  <->  internal (v fastest): tiled transposes through shared memory
// --------------------------------------------------------------------------------------------------
template <bool PACK>
__global__ void __launch_bounds__(256) transpose_kernel(const double *__restrict__ src,
                                                        double *__restrict__ dst, GridDev g)
{
    __shared__ double tile[32][33];
    const long long plane = (long long)g.N[1] * g.N[0];
    const int z = blockIdx.z;
    const long long yx0 = (long long)blockIdx.x * 32;
    const int v0 = blockIdx.y * 32;
    const int tx = threadIdx.x, ty = threadIdx.y;
    const int Nv = g.N[3];
    if (PACK) {
        // read canonical rows (fixed v) along yx, write internal lines (fixed yx) along v
        for (int k = ty; k < 32; k += 8) {
            int v = v0 + k;
            long long yx = yx0 + tx;
            if (v < Nv && yx < plane) tile[k][tx] = src[((long long)z * Nv + v) * plane + yx];
        }
        __syncthreads();
        for (int k = ty; k < 32; k += 8) {
            long long yx = yx0 + k;
            int v = v0 + tx;
            if (yx < plane && v < Nv) dst[line_base(g, (long long)z * plane + yx) + v] = tile[tx][k];
        }
    } else {
        for (int k = ty; k < 32; k += 8) {
            long long yx = yx0 + k;
            int v = v0 + tx;
            if (yx < plane && v < Nv) tile[k][tx] = src[line_base(g, (long long)z * plane + yx) + v];
        }
        __syncthreads();
        for (int k = ty; k < 32; k += 8) {
            int v = v0 + k;
            long long yx = yx0 + tx;
            if (v < Nv && yx < plane) dst[((long long)z * Nv + v) * plane + yx] = tile[tx][k];
        }
    }
}

static cudaError_t launch_transpose(sldg_ctx *c, const double *src, double *dst, bool pack)
{
    const GridDev &g = c->g;
    long long plane = (long long)g.N[1] * g.N[0];
    dim3 grid((unsigned)((plane + 31) / 32), (unsigned)((g.N[3] + 31) / 32), (unsigned)g.N[2]);
    dim3 block(32, 8);
    if (pack)
        transpose_kernel<true><<<grid, block, 0, c->stream>>>(src, dst, g);
    else
        transpose_kernel<false><<<grid, block, 0, c->stream>>>(src, dst, g);
    c->launches++;
    return cudaGetLastError();
}
cudaError_t launch_pack(sldg_ctx *c, const double *canon, double *internal)
{
    return launch_transpose(c, canon, internal, true);
}
cudaError_t launch_unpack(sldg_ctx *c, const double *internal, double *canon)
{
    return launch_transpose(c, internal, canon, false);
}

// --------------------------------------------------------------------------------------------------
// advect_v: every (z,Y,X) line is a contiguous periodic line of nv cells; one Courant number per line.
// A block stages LPB consecutive-in-enumeration lines in shared memory, one thread per (line, cell).
// --------------------------------------------------------------------------------------------------
template <int O>
__global__ void __launch_bounds__(256) advect_v_kernel(const double *__restrict__ fin,
                                                       double *__restrict__ fout,
                                                       const double *__restrict__ Ez, GridDev g,
                                                       ShiftPoly sp, double tau, int lpb)
{
    extern __shared__ double smem[];
    const int Pv = g.Pv, Nv = g.N[3], nv = g.n[3];
    double *sin_ = smem;                                   // [lpb][Pv]
    double *sAB = smem + (size_t)lpb * Pv;                 // [lpb][2*O*O]
    int *sS = (int *)(sAB + (size_t)lpb * 2 * O * O);      // [lpb]
    long long *sBase = (long long *)(sS + ((lpb + 1) & ~1)); // [lpb]

    for (long long l0 = (long long)blockIdx.x * lpb; l0 < g.lines; l0 += (long long)gridDim.x * lpb) {
        const int nl = (int)min((long long)lpb, g.lines - l0);
        // per-line shift data
        for (int l = threadIdx.x; l < nl; l += blockDim.x) {
            int s;
            double alpha, A[O][O], B[O][O];
            shift_of(Ez[l0 + l], tau, g.h[3], s, alpha);
            eval_shift<O>(sp, alpha, A, B);
#pragma unroll
            for (int j = 0; j < O; ++j)
#pragma unroll
                for (int m = 0; m < O; ++m) {
                    sAB[(size_t)l * 2 * O * O + j * O + m] = A[j][m];
                    sAB[(size_t)l * 2 * O * O + O * O + j * O + m] = B[j][m];
                }
            sS[l] = wrapi(s, nv);
            sBase[l] = line_base(g, l0 + l);
        }
        __syncthreads();
        // stage the lines (16-byte vector loads; Pv is even and lines are 128-byte aligned)
        const int vec_per_line = Pv / 2;
        for (int idx = threadIdx.x; idx < nl * vec_per_line; idx += blockDim.x) {
            int l = idx / vec_per_line, k = idx - l * vec_per_line;
            double2 val = *reinterpret_cast<const double2 *>(fin + sBase[l] + 2 * k);
            *reinterpret_cast<double2 *>(sin_ + (size_t)l * Pv + 2 * k) = val;
        }
        __syncthreads();
        for (int idx = threadIdx.x; idx < nl * nv; idx += blockDim.x) {
            int l = idx / nv, cell = idx - l * nv;
            const double *A = sAB + (size_t)l * 2 * O * O, *B = A + O * O;
            const double *u = sin_ + (size_t)l * Pv;
            int c0 = cell + sS[l];
            if (c0 >= nv) c0 -= nv;
            int c1 = c0 + 1;
            if (c1 >= nv) c1 -= nv;
            double u0[O], u1[O], r[O];
#pragma unroll
            for (int m = 0; m < O; ++m) {
                u0[m] = u[c0 * O + m];
                u1[m] = u[c1 * O + m];
            }
#pragma unroll
            for (int j = 0; j < O; ++j) {
                double acc = 0.0;
#pragma unroll
                for (int m = 0; m < O; ++m) acc = fma(A[j * O + m], u0[m], acc);
#pragma unroll
                for (int m = 0; m < O; ++m) acc = fma(B[j * O + m], u1[m], acc);
                r[j] = acc;
            }
            double *dst = fout + sBase[l] + cell * O;
            if (O == 2) {
                *reinterpret_cast<double2 *>(dst) = make_double2(r[0], r[O - 1]);
            } else {
#pragma unroll
                for (int j = 0; j < O; ++j) dst[j] = r[j];
            }
        }
        __syncthreads();
    }
    (void)Nv;
}

cudaError_t launch_advect_v(sldg_ctx *c, const double *fin, double *fout, double tau)
{
    const GridDev &g = c->g;
    const int O = g.o[3];
    int lpb = (1024 + g.n[3] - 1) / g.n[3];  // about 1024 cells per block iteration
    if (lpb < 1) lpb = 1;
    auto smem_for = [&](int l) {
        return (size_t)l * g.Pv * 8 + (size_t)l * 2 * O * O * 8 + (size_t)((l + 1) & ~1) * 4 + (size_t)l * 8;
    };
    while (lpb > 1 && smem_for(lpb) > 64 * 1024) lpb--;
    size_t smem = smem_for(lpb);
    if (smem > 227 * 1024) return cudaErrorInvalidValue;
    long long nblk = (g.lines + lpb - 1) / lpb;
    long long cap = (long long)c->sm_count * 32;
    int grid = (int)(nblk < cap ? nblk : cap);
#define LAUNCH_V(OO)                                                                                 \
    {                                                                                                \
        cudaFuncSetAttribute(advect_v_kernel<OO>, cudaFuncAttributeMaxDynamicSharedMemorySize,       \
                             (int)smem);                                                             \
        advect_v_kernel<OO><<<grid, 256, smem, c->stream>>>(fin, fout, c->Ez, g, c->sp_v, tau, lpb); \
    }
    if (O == 1) LAUNCH_V(1) else if (O == 2) LAUNCH_V(2) else LAUNCH_V(3)
#undef LAUNCH_V
    c->launches++;
    return cudaGetLastError();
}

// --------------------------------------------------------------------------------------------------
// advect_z: the z axis is strided.  A block owns one (Y,X) position and a chunk of VC consecutive v
// values, stages the [Nz][VC] slab in shared memory (rows of VC*8 contiguous bytes, no transpose), and
// shifts every v column along z by its own (s, alpha): lane <-> v, so shared-memory reads are
// conflict-free whatever the per-lane row offsets are.
// --------------------------------------------------------------------------------------------------
template <int O, int VC>
__global__ void __launch_bounds__(256) advect_z_kernel(const double *__restrict__ fin,
                                                       double *__restrict__ fout, GridDev g,
                                                       ShiftPoly sp, Basis bs, double tau)
{
    extern __shared__ double slab[];  // [Nz][VC]
    const int Nz = g.N[2], nz = g.n[2], Nv = g.N[3], ov = g.o[3];
    const int nchunk = (Nv + VC - 1) / VC;
    const long long nyx = (long long)g.N[1] * g.N[0];
    const long long ntask = nyx * nchunk;
    const int lane = threadIdx.x % VC, grp = threadIdx.x / VC, ngrp = blockDim.x / VC;

    for (long long task = blockIdx.x; task < ntask; task += gridDim.x) {
        const int chunk = (int)(task % nchunk);
        const long long yx = task / nchunk;
        const int X = (int)(yx % g.N[0]), Y = (int)(yx / g.N[0]);
        const long long base = Y * g.sY + X * g.sX + (long long)chunk * VC;
        const int v = chunk * VC + lane;
        const bool live = v < Nv;
        // stage rows
        constexpr int VEC = VC / 2;
        for (int idx = threadIdx.x; idx < Nz * VEC; idx += blockDim.x) {
            int row = idx / VEC, k = idx - row * VEC;
            if (chunk * VC + 2 * k < g.Pv) {
                double2 val = *reinterpret_cast<const double2 *>(fin + base + row * g.sZ + 2 * k);
                *reinterpret_cast<double2 *>(slab + row * VC + 2 * k) = val;
            }
        }
        // per-lane shift
        int s = 0;
        double A[O][O], B[O][O];
        {
            int l = v / ov, q = v - l * ov;
            double vq = __dadd_rn(g.lo[3], __dmul_rn(__dadd_rn((double)l, bs.xi[ov][q]), g.h[3]));
            double alpha;
            if (!live) vq = 0.0;
            shift_of(vq, tau, g.h[2], s, alpha);
            eval_shift<O>(sp, alpha, A, B);
            s = wrapi(s, nz);
        }
        __syncthreads();
        for (int cell = grp; cell < nz; cell += ngrp) {
            int c0 = cell + s;
            if (c0 >= nz) c0 -= nz;
            int c1 = c0 + 1;
            if (c1 >= nz) c1 -= nz;
            double u0[O], u1[O];
#pragma unroll
            for (int m = 0; m < O; ++m) {
                u0[m] = slab[(c0 * O + m) * VC + lane];
                u1[m] = slab[(c1 * O + m) * VC + lane];
            }
#pragma unroll
            for (int j = 0; j < O; ++j) {
                double acc = 0.0;
#pragma unroll
                for (int m = 0; m < O; ++m) acc = fma(A[j][m], u0[m], acc);
#pragma unroll
                for (int m = 0; m < O; ++m) acc = fma(B[j][m], u1[m], acc);
                if (live) fout[base + (long long)(cell * O + j) * g.sZ + lane] = acc;
            }
        }
        __syncthreads();
    }
}

cudaError_t launch_advect_z(sldg_ctx *c, const double *fin, double *fout, double tau)
{
    const GridDev &g = c->g;
    const int O = g.o[2];
    constexpr int VC = 32;
    size_t smem = (size_t)g.N[2] * VC * 8;
    if (smem > 227 * 1024) return cudaErrorInvalidValue;
    long long ntask = (long long)g.N[1] * g.N[0] * ((g.N[3] + VC - 1) / VC);
    long long cap = (long long)c->sm_count * 64;
    int grid = (int)(ntask < cap ? ntask : cap);
#define LAUNCH_Z(OO)                                                                                   \
    {                                                                                                  \
        cudaFuncSetAttribute(advect_z_kernel<OO, VC>, cudaFuncAttributeMaxDynamicSharedMemorySize,     \
                             (int)smem);                                                               \
        advect_z_kernel<OO, VC><<<grid, 256, smem, c->stream>>>(fin, fout, g, c->sp_z, c->basis, tau); \
    }
    if (O == 1) LAUNCH_Z(1) else if (O == 2) LAUNCH_Z(2) else LAUNCH_Z(3)
#undef LAUNCH_Z
    c->launches++;
    return cudaGetLastError();
}

// --------------------------------------------------------------------------------------------------
// charge density: one warp per line, Gauss-weighted sum over v with a shuffle reduction.
// --------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) charge_density_kernel(const double *__restrict__ fin,
                                                             double *__restrict__ rho, GridDev g,
                                                             Basis bs)
{
    const int lane = threadIdx.x & 31;
    const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long long nwarp = ((long long)gridDim.x * blockDim.x) >> 5;
    const int Nv = g.N[3], ov = g.o[3];
    for (long long line = warp; line < g.lines; line += nwarp) {
        const double *u = fin + line_base(g, line);
        double acc = 0.0;
        for (int v = lane; v < Nv; v += 32) acc = fma(bs.w[ov][v % ov], u[v], acc);
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
        if (lane == 0) rho[line] = g.h[3] * acc;
    }
}

cudaError_t launch_charge_density(sldg_ctx *c, const double *fin, double *rho)
{
    const GridDev &g = c->g;
    long long nblk = (g.lines + 7) / 8;
    long long cap = (long long)c->sm_count * 32;
    int grid = (int)(nblk < cap ? nblk : cap);
    charge_density_kernel<<<grid, 256, 0, c->stream>>>(fin, rho, g, c->basis);
    c->launches++;
    return cudaGetLastError();
}

// --------------------------------------------------------------------------------------------------
// mass: two-pass deterministic reduction (per-block partial sums, then one block).
// --------------------------------------------------------------------------------------------------
__device__ __forceinline__ double block_sum(double v)
{
    __shared__ double red[32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    if (lane == 0) red[wid] = v;
    __syncthreads();
    double t = 0.0;
    if (wid == 0) {
        t = lane < (int)(blockDim.x >> 5) ? red[lane] : 0.0;
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) t += __shfl_xor_sync(0xffffffffu, t, off);
    }
    __syncthreads();
    return t;
}

__global__ void __launch_bounds__(256) mass_partial_kernel(const double *__restrict__ fin,
                                                           double *__restrict__ partials, GridDev g,
                                                           Basis bs)
{
    const int lane = threadIdx.x & 31;
    const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long long nwarp = ((long long)gridDim.x * blockDim.x) >> 5;
    const int Nv = g.N[3], ov = g.o[3];
    double total = 0.0, comp = 0.0;  // Kahan over the lines of this lane
    for (long long line = warp; line < g.lines; line += nwarp) {
        int X = (int)(line % g.N[0]);
        long long t = line / g.N[0];
        int Y = (int)(t % g.N[1]);
        int z = (int)(t / g.N[1]);
        const double wl = bs.w[g.o[0]][X % g.o[0]] * bs.w[g.o[1]][Y % g.o[1]] * bs.w[g.o[2]][z % g.o[2]];
        const double *u = fin + z * g.sZ + Y * g.sY + X * g.sX;
        double acc = 0.0;
        for (int v = lane; v < Nv; v += 32) acc = fma(bs.w[ov][v % ov], u[v], acc);
        double yk = wl * acc - comp;
        double tk = total + yk;
        comp = (tk - total) - yk;
        total = tk;
    }
    double s = block_sum(total);
    if (threadIdx.x == 0) partials[blockIdx.x] = s;
}

__global__ void __launch_bounds__(256) mass_final_kernel(const double *__restrict__ partials, int n,
                                                         double scale, double *__restrict__ out)
{
    double acc = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) acc += partials[i];
    double s = block_sum(acc);
    if (threadIdx.x == 0) *out = s * scale;
}

cudaError_t launch_mass(sldg_ctx *c, const double *fin, double *mass_out)
{
    const GridDev &g = c->g;
    long long nblk = (g.lines + 7) / 8;
    long long cap = (long long)c->n_partials;
    int grid = (int)(nblk < cap ? nblk : cap);
    mass_partial_kernel<<<grid, 256, 0, c->stream>>>(fin, c->partials, g, c->basis);
    double scale = g.h[0] * g.h[1] * g.h[2] * g.h[3];
    mass_final_kernel<<<1, 256, 0, c->stream>>>(c->partials, grid, scale, mass_out);
    c->launches += 2;
    return cudaGetLastError();
}
