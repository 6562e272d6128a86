// sldg_sweeps.cu -- 1d SLDG sweeps along z and v (eq. 11), charge density,
// mass and the canonical <-> internal layout transposes.  sm_100a.
//
// Internal layout: v fastest.  Element (z,Y,X,v) lives at z*sZ + Y*sY + X*sX + v; every (z,Y,X) "line"
// of Nv doubles is contiguous and starts on a 128-byte boundary (pitch Pv).
#include <math.h>
#include <stdlib.h>

#include "sldg_internal.cuh"
#include "sldg_sweep_common.cuh"

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
// advect_v: every (z,Y,X) line is a contiguous periodic line of nv cells with one Courant number.
// warp <-> line, lane <-> target cell (lane, lane+32, ...).  A target cell reads its two source cells
// (i+s, i+s+1) straight from global memory: neighbouring lanes overlap by one cell, the overlap is served
// by L1 (each 128-byte line is fetched from L2 once), so there is no shared-memory staging and no
// block-level synchronisation; every byte of f crosses HBM once in each direction.
// --------------------------------------------------------------------------------------------------
__device__ __forceinline__ long long line_base_fast(const GridDev &g, unsigned line)
{
    if (g.contig) return (long long)line * g.Pv;
    unsigned X = line % (unsigned)g.N[0], t = line / (unsigned)g.N[0];
    unsigned Y = t % (unsigned)g.N[1], z = t / (unsigned)g.N[1];
    return z * g.sZ + Y * g.sY + X * g.sX;
}

// LPL lanes share one line (32/LPL lines per warp); CU target cells per lane are in flight at once.
template <int O, int LPL, int CU>
__global__ void __launch_bounds__(256) advect_v_kernel(const double *__restrict__ fin,
                                                       double *__restrict__ fout,
                                                       const double *__restrict__ Ez, GridDev g,
                                                       ShiftPoly sp, double tau)
{
    constexpr int LPW = 32 / LPL;  // lines per warp
    const int nv = g.n[3];
    const int lane = threadIdx.x & 31, sub = lane % LPL, grp = lane / LPL;
    const unsigned warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const unsigned nwarp = (gridDim.x * blockDim.x) >> 5;
    const unsigned lines = (unsigned)g.lines;
    unsigned line = warp * LPW + grp;
    double e_next = line < lines ? __ldg(Ez + line) : 0.0;
    for (; line < lines; line += nwarp * LPW) {
        const double e = e_next;
        const unsigned nline = line + nwarp * LPW;
        if (nline < lines) e_next = __ldg(Ez + nline);  // prefetch: takes the Ez latency off the critical path
        int s;
        double alpha, A[O][O], B[O][O];
        shift_of(e, tau, g.h[3], s, alpha);
        eval_shift<O>(sp, alpha, A, B);
        s = wrapi(s, nv);
        const long long base = line_base_fast(g, line);
        const double *u = fin + base;
        double *w = fout + base;
        for (int cell0 = sub; cell0 < nv; cell0 += LPL * CU) {
            double u0[CU][O], u1[CU][O];
#pragma unroll
            for (int k = 0; k < CU; ++k) {
                const int cell = cell0 + k * LPL;
                if (cell < nv) {
                    int c0 = cell + s;
                    if (c0 >= nv) c0 -= nv;
                    int c1 = c0 + 1;
                    if (c1 >= nv) c1 -= nv;
                    if (O == 2) {
                        const double2 t0 = __ldg(reinterpret_cast<const double2 *>(u + 2 * c0));
                        const double2 t1 = __ldg(reinterpret_cast<const double2 *>(u + 2 * c1));
                        u0[k][0] = t0.x; u0[k][O - 1] = t0.y;
                        u1[k][0] = t1.x; u1[k][O - 1] = t1.y;
                    } else {
#pragma unroll
                        for (int m = 0; m < O; ++m) {
                            u0[k][m] = __ldg(u + c0 * O + m);
                            u1[k][m] = __ldg(u + c1 * O + m);
                        }
                    }
                }
            }
#pragma unroll
            for (int k = 0; k < CU; ++k) {
                const int cell = cell0 + k * LPL;
                if (cell < nv) {
                    double r[O];
#pragma unroll
                    for (int j = 0; j < O; ++j) {
                        double acc = 0.0;
#pragma unroll
                        for (int m = 0; m < O; ++m) acc = fma(A[j][m], u0[k][m], acc);
#pragma unroll
                        for (int m = 0; m < O; ++m) acc = fma(B[j][m], u1[k][m], acc);
                        r[j] = acc;
                    }
                    if (O == 2) {
                        __stcs(reinterpret_cast<double2 *>(w + 2 * cell), make_double2(r[0], r[O - 1]));
                    } else {
#pragma unroll
                        for (int j = 0; j < O; ++j) __stcs(w + cell * O + j, r[j]);
                    }
                }
            }
        }
    }
}

cudaError_t launch_advect_v(sldg_ctx *c, const double *fin, double *fout, double tau)
{
    const GridDev &g = c->g;
    const int O = g.o[3];
    if (g.lines >= (1ll << 31)) return cudaErrorInvalidValue;
    constexpr int LPL = 8, CU = 4;
    long long nblk = (g.lines + 8 * (32 / LPL) - 1) / (8 * (32 / LPL));  // 8 warps per block
    long long cap = (long long)c->sm_count * 8 * 8;
    int grid = (int)(nblk < cap ? nblk : cap);
#define LAUNCH_V(OO) \
    advect_v_kernel<OO, LPL, CU><<<grid, 256, 0, c->stream>>>(fin, fout, c->Ez, g, c->sp_v, tau)
    if (O == 1) LAUNCH_V(1); else if (O == 2) LAUNCH_V(2); else LAUNCH_V(3);
#undef LAUNCH_V
    c->launches++;
    return cudaGetLastError();
}

// --------------------------------------------------------------------------------------------------
// advect_z: the z axis is strided, v is contiguous.  thread <-> one (Y,X,v) column, lanes along v
// (coalesced), walking z with a rolling register window: the two source cells of target cell i are
// cells i+s and i+s+1, so every step loads one new cell and stores one -- each input is read exactly
// once, no shared memory, no transpose.  (s, A, B) depend on the v node only and live in registers.
// U target cells are processed per iteration so that U*O independent loads are in flight per thread.
// --------------------------------------------------------------------------------------------------
template <int O, int U>
__global__ void __launch_bounds__(256) advect_z_kernel(const double *__restrict__ fin,
                                                       double *__restrict__ fout, GridDev g,
                                                       ShiftPoly sp, Basis bs, double tau)
{
    const int nz = g.n[2], Nv = g.N[3], ov = g.o[3];
    const unsigned Pv = (unsigned)g.Pv;
    const unsigned long long tid = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    const unsigned yx = (unsigned)(tid / Pv);
    const int v = (int)(tid - (unsigned long long)yx * Pv);
    if (yx >= (unsigned)(g.N[1] * g.N[0]) || v >= Nv) return;
    const unsigned X = yx % (unsigned)g.N[0], Y = yx / (unsigned)g.N[0];
    const long long base = Y * g.sY + X * g.sX + v;
    int s;
    double A[O][O], B[O][O];
    {
        const int l = v / ov, q = v - l * ov;
        const double vq = __dadd_rn(g.lo[3], __dmul_rn(__dadd_rn((double)l, bs.xi[ov][q]), g.h[3]));
        double alpha;
        shift_of(vq, tau, g.h[2], s, alpha);
        eval_shift<O>(sp, alpha, A, B);
        s = wrapi(s, nz);
    }
    const long long sZ = g.sZ;
    const double *src = fin + base;
    double *dst = fout + base;
    int c = s;  // source cell of the window's left half
    double up[O];
#pragma unroll
    for (int m = 0; m < O; ++m) up[m] = __ldcs(src + (long long)(c * O + m) * sZ);
    for (int i0 = 0; i0 < nz; i0 += U) {
        double un[U][O];
#pragma unroll
        for (int k = 0; k < U; ++k) {
            if (i0 + k < nz) {
                c = (c + 1 == nz) ? 0 : c + 1;
#pragma unroll
                for (int m = 0; m < O; ++m) un[k][m] = __ldcs(src + (long long)(c * O + m) * sZ);
            }
        }
#pragma unroll
        for (int k = 0; k < U; ++k) {
            if (i0 + k < nz) {
#pragma unroll
                for (int j = 0; j < O; ++j) {
                    double acc = 0.0;
#pragma unroll
                    for (int m = 0; m < O; ++m) acc = fma(A[j][m], k == 0 ? up[m] : un[k == 0 ? 0 : k - 1][m], acc);
#pragma unroll
                    for (int m = 0; m < O; ++m) acc = fma(B[j][m], un[k][m], acc);
                    __stcs(dst + (long long)((i0 + k) * O + j) * sZ, acc);
                }
            }
        }
#pragma unroll
        for (int m = 0; m < O; ++m) up[m] = un[U - 1][m];
    }
}

cudaError_t launch_advect_z(sldg_ctx *c, const double *fin, double *fout, double tau)
{
    const GridDev &g = c->g;
    const int O = g.o[2];
    {
        // The Courant number grows linearly with the v node.  When it changes by more than ~2 cells across the 32 v
        // nodes of a warp, the lanes of the column walk below read different z rows (scattered 8-24 byte runs:
        // measured 7.1 ms instead of 2.6 ms at |CFL| = 20, configs[2]): the plane-tiled kernel of sldg_fused_sweeps.cu
        // does the same sweep (same arithmetic, bit-identical) with every row read whole.
        const double dv_warp = 32.0 * g.h[3] / g.o[3];
        const double spread = fabs(dv_warp * tau / g.h[2]);
        if (spread > 2.0 && !getenv("SLDG_ADVECT_Z_COLUMNS")) {
            cudaError_t e = launch_fused_sweeps(c, fin, fout, tau, 0.0, false, true);
            if (e != cudaErrorNotSupported) return e;
            cudaGetLastError();
        }
    }
    const long long nthreads = (long long)g.N[1] * g.N[0] * g.Pv;
    const long long nblk = (nthreads + 255) / 256;
    if (nblk >= (1ll << 31)) return cudaErrorInvalidValue;
    const unsigned grid = (unsigned)nblk;
#define LAUNCH_Z(OO, UU) advect_z_kernel<OO, UU><<<grid, 256, 0, c->stream>>>(fin, fout, g, c->sp_z, c->basis, tau)
    if (O == 1) LAUNCH_Z(1, 8); else if (O == 2) LAUNCH_Z(2, 4); else LAUNCH_Z(3, 2);
#undef LAUNCH_Z
    c->launches++;
    return cudaGetLastError();
}

// --------------------------------------------------------------------------------------------------
// charge density: one warp per line, Gauss-weighted sum over v with a shuffle reduction.
// --------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) charge_density_kernel(const double *__restrict__ fin,
                                                             double *__restrict__ rho, GridDev g,
                                                             Basis bs, unsigned line0, unsigned line1)
{
    const int lane = threadIdx.x & 31;
    const unsigned warp = line0 + ((blockIdx.x * blockDim.x + threadIdx.x) >> 5);
    const unsigned nwarp = (gridDim.x * blockDim.x) >> 5;
    const unsigned lines = line1;  // this launch does the lines [line0, line1)
    const int Nv = g.N[3], ov = g.o[3];
    for (unsigned line = warp; line < lines; line += nwarp) {
        const double *u = fin + line_base_fast(g, line);
        double acc = 0.0;
        // pairs (2 lane, 2 lane + 1) + 64 k; Nv is even unless ov * nv is odd (tail handled below)
        int v = 2 * lane;
        for (; v + 1 < Nv; v += 64) {
            const double2 t = __ldcs(reinterpret_cast<const double2 *>(u + v));
            acc = fma(bs.w[ov][v % ov], t.x, acc);
            acc = fma(bs.w[ov][(v + 1) % ov], t.y, acc);
        }
        if (v < Nv) acc = fma(bs.w[ov][v % ov], u[v], acc);
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
        if (lane == 0) rho[line] = g.h[3] * acc;
    }
}

cudaError_t launch_charge_density(sldg_ctx *c, const double *fin, double *rho, long long line0, long long line1)
{
    const GridDev &g = c->g;
    if (g.lines >= (1ll << 31)) return cudaErrorInvalidValue;
    if (line1 < 0) line1 = g.lines;
    long long nblk = (line1 - line0 + 7) / 8;
    long long cap = (long long)c->sm_count * 8 * 16;
    int grid = (int)(nblk < cap ? nblk : cap);
    if (grid < 1) return cudaSuccess;
    charge_density_kernel<<<grid, 256, 0, c->stream>>>(fin, rho, g, c->basis, (unsigned)line0, (unsigned)line1);
    c->launches++;
    return cudaGetLastError();
}

// --------------------------------------------------------------------------------------------------
// mass: the v integral is the charge density; the remaining (x,y,z) Gauss sum is a
// two-pass deterministic reduction over rho (per-block Kahan partial sums, then one block).
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

__global__ void __launch_bounds__(256) mass_partial_kernel(const double *__restrict__ rho,
                                                           double *__restrict__ partials, GridDev g,
                                                           Basis bs)
{
    const unsigned lines = (unsigned)g.lines;
    double total = 0.0, comp = 0.0;  // Kahan over the lines of this thread
    for (unsigned line = blockIdx.x * blockDim.x + threadIdx.x; line < lines; line += gridDim.x * blockDim.x) {
        const unsigned X = line % (unsigned)g.N[0], t = line / (unsigned)g.N[0];
        const unsigned Y = t % (unsigned)g.N[1], z = t / (unsigned)g.N[1];
        const double wl = bs.w[g.o[0]][X % g.o[0]] * bs.w[g.o[1]][Y % g.o[1]] * bs.w[g.o[2]][z % g.o[2]];
        double yk = wl * rho[line] - comp;
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

cudaError_t launch_mass_from_rho(sldg_ctx *c, const double *rho, double *mass_out)
{
    const GridDev &g = c->g;
    long long nblk = (g.lines + 255) / 256;
    long long cap = 1024;
    int grid = (int)(nblk < cap ? nblk : cap);
    mass_partial_kernel<<<grid, 256, 0, c->stream>>>(rho, c->partials, g, c->basis);
    double scale = g.h[0] * g.h[1] * g.h[2];
    mass_final_kernel<<<1, 256, 0, c->stream>>>(c->partials, grid, scale, mass_out);
    c->launches += 2;
    return cudaGetLastError();
}

cudaError_t launch_mass(sldg_ctx *c, const double *fin, double *mass_out)
{
    cudaError_t e = launch_charge_density(c, fin, c->rho_ws);
    if (e != cudaSuccess) return e;
    return launch_mass_from_rho(c, c->rho_ws, mass_out);
}
