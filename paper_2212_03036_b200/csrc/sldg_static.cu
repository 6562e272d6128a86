// sldg_static.cu -- sldg_mass_static: the total mass of a distribution in the canonical layout, for
// callers that may not allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).
//
// sldg_mass works on a context, whose workspace the caller had to allocate: the charge density goes to the workspace
// (one double per (x,y,z) node), the per-block partial sums next to it.  This variant needs no context and no buffer
// from the caller except its input and its output: the same two intermediate arrays live in ONE file-scope
// `static __device__` array of a fixed size, SLDG_STATIC_MAX_NODES doubles for the charge density plus 1024 partial
// sums (8 MiB + 8 KiB; every GPU that loads libsldg.so holds it until the process exits).
//
//   * In host code the array's name is a host-side stand-in, not a device address.  The address the kernels get is
//     asked for once per device, with that device current, by cudaGetSymbolAddress (scratch_of_current_device below);
//     device code never needs it, only the launches do (they receive it as an ordinary pointer argument so that the
//     kernels stay free of hidden state).
//   * Every call shares the array.  Nothing in it has to start at zero: the first kernel writes rho[0, nodes), the second
//     reads exactly those and writes partials[0, grid), the third reads exactly those -- stale contents of an earlier,
//     larger call are never read.  Two calls that overlap on the GPU (different streams, or the same device from two
//     threads without ordering) RACE on it; calls on one stream are ordered and safe.
//   * No cudaMalloc, cudaFree or allocating library routine anywhere in this file; three kernel launches per call.
//
// The arithmetic is that of sldg_sweeps.cu's charge density and mass kernels (Gauss-weighted v sum per node, Kahan sum of
// the weighted nodes per thread, fixed-order block sums: deterministic), on the canonical layout [Nz][Nv][Ny][Nx] instead
// of the internal one; the summation order over v differs, so the result agrees with sldg_mass to rounding (1e-13
// relative in tests/test_zz_no_alloc.py), not bitwise.  This file shares no code path with the rest of the library.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include <mutex>

#include "sldg.h"

namespace {

constexpr long long MAX_NODES = SLDG_STATIC_MAX_NODES;
constexpr int MAX_PARTIALS = 1024;
constexpr int MAX_DEVICES = 64;

static __device__ __align__(256) double sldg_static_scratch[MAX_NODES + MAX_PARTIALS];

struct StaticGrid {
    int N[4];        // degrees of freedom per axis (x, y, z, v)
    int o[4];        // nodes per cell per axis
    double w[4][3];  // Gauss-Legendre weights on [0,1] of each axis' order
    double hv;       // cell width in v
    double scale;    // h_x h_y h_z
    long long nodes; // Nx Ny Nz
};

// Gauss-Legendre weights on [0,1] (the DOFs are point values at these nodes)
void gl_weights(int o, double *w)
{
    if (o == 1) {
        w[0] = 1.0;
    } else if (o == 2) {
        w[0] = w[1] = 0.5;
    } else {
        w[0] = w[2] = (double)(5.0L / 18.0L);
        w[1] = (double)(4.0L / 9.0L);
    }
}

// rho[z][Y][X] = h_v sum_v w_v f[z][v][Y][X]; thread <-> node, x fastest: coalesced for every v
__global__ void __launch_bounds__(256) static_rho_kernel(const double *__restrict__ f, double *__restrict__ rho,
                                                         StaticGrid g)
{
    const long long plane = (long long)g.N[1] * g.N[0];
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < g.nodes;
         k += (long long)gridDim.x * blockDim.x) {
        const long long z = k / plane, yx = k - z * plane;
        const double *u = f + z * g.N[3] * plane + yx;
        double acc = 0.0;
        int q = 0;
        for (int v = 0; v < g.N[3]; ++v) {
            acc = fma(g.w[3][q], __ldcs(u + (long long)v * plane), acc);
            if (++q == g.o[3]) q = 0;
        }
        rho[k] = g.hv * acc;
    }
}

// fixed-order sum over the block; valid in thread 0
__device__ __forceinline__ double static_block_sum(double v)
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

// partials[block] = sum over this block's nodes of w_x w_y w_z rho (Kahan per thread)
__global__ void __launch_bounds__(256) static_partial_kernel(const double *__restrict__ rho,
                                                             double *__restrict__ partials, StaticGrid g)
{
    double total = 0.0, comp = 0.0;
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < g.nodes;
         k += (long long)gridDim.x * blockDim.x) {
        const int X = (int)(k % g.N[0]);
        const long long t = k / g.N[0];
        const int Y = (int)(t % g.N[1]), z = (int)(t / g.N[1]);
        const double wl = g.w[0][X % g.o[0]] * g.w[1][Y % g.o[1]] * g.w[2][z % g.o[2]];
        const double yk = wl * rho[k] - comp;
        const double tk = total + yk;
        comp = (tk - total) - yk;
        total = tk;
    }
    const double s = static_block_sum(total);
    if (threadIdx.x == 0) partials[blockIdx.x] = s;
}

__global__ void __launch_bounds__(256) static_final_kernel(const double *__restrict__ partials, int n, double scale,
                                                           double *__restrict__ out)
{
    double acc = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) acc += partials[i];
    const double s = static_block_sum(acc);
    if (threadIdx.x == 0) *out = s * scale;
}

// Device address of the scratch array on the CURRENT device, asked for once per device.
std::mutex scratch_mutex;
double *scratch_addr[MAX_DEVICES];
bool scratch_known[MAX_DEVICES];

int scratch_of_current_device(double **out)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAX_DEVICES) {
        cudaGetLastError();
        return SLDG_ECUDA;
    }
    std::lock_guard<std::mutex> lock(scratch_mutex);
    if (!scratch_known[dev]) {
        void *p = nullptr;
        if (cudaGetSymbolAddress(&p, sldg_static_scratch) != cudaSuccess || p == nullptr) {
            cudaGetLastError();
            return SLDG_ECUDA;
        }
        scratch_addr[dev] = static_cast<double *>(p);
        scratch_known[dev] = true;
    }
    *out = scratch_addr[dev];
    return SLDG_OK;
}

}  // namespace

extern "C" {

long long sldg_mass_static_max_nodes(void) { return MAX_NODES; }

int sldg_mass_static_setup(void)
{
    double *p = nullptr;
    return scratch_of_current_device(&p);
}

int sldg_mass_static(const sldg_params *p, const double *f_canonical_dev, double *mass_dev, void *cuda_stream)
{
    if (!p || !f_canonical_dev || !mass_dev) return SLDG_EINVAL;
    if (((uintptr_t)f_canonical_dev & 7) || ((uintptr_t)mass_dev & 7)) return SLDG_EINVAL;
    StaticGrid g;
    double h[4];
    for (int d = 0; d < 4; ++d) {
        if (p->n[d] < 1 || p->order[d] < 1 || p->order[d] > 3 || !(p->hi[d] > p->lo[d])) return SLDG_EINVAL;
        if ((long long)p->n[d] * p->order[d] >= (1ll << 31)) return SLDG_EINVAL;
        g.N[d] = p->n[d] * p->order[d];
        g.o[d] = p->order[d];
        g.w[d][0] = g.w[d][1] = g.w[d][2] = 0.0;
        gl_weights(p->order[d], g.w[d]);
        h[d] = (p->hi[d] - p->lo[d]) / p->n[d];
    }
    // the limit first: a product of three 31-bit numbers can overflow 64 bits
    if ((long long)g.N[0] * g.N[1] > MAX_NODES) return SLDG_ELIMIT;
    g.nodes = (long long)g.N[0] * g.N[1] * g.N[2];
    if (g.nodes > MAX_NODES) return SLDG_ELIMIT;
    g.hv = h[3];
    g.scale = h[0] * h[1] * h[2];

    double *scratch = nullptr;
    const int rc = scratch_of_current_device(&scratch);
    if (rc != SLDG_OK) return rc;
    double *rho = scratch, *partials = scratch + MAX_NODES;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);

    const long long nblk = (g.nodes + 255) / 256;
    const int grid_rho = (int)(nblk < 148 * 16 ? nblk : 148 * 16);
    const int grid_par = (int)(nblk < MAX_PARTIALS ? nblk : MAX_PARTIALS);
    static_rho_kernel<<<grid_rho, 256, 0, st>>>(f_canonical_dev, rho, g);
    static_partial_kernel<<<grid_par, 256, 0, st>>>(rho, partials, g);
    static_final_kernel<<<1, 256, 0, st>>>(partials, grid_par, g.scale, mass_dev);
    return cudaGetLastError() == cudaSuccess ? SLDG_OK : SLDG_ECUDA;
}

}  // extern "C"
