// sldg_xy_geometry.cu -- geometry of the 2d SLDG step in the poloidal plane (Algorithm 3
// PAPER.md:287-293): everything of eq. (14)-(18) that does not depend on v.
//
//   Per (z node, target cell), once:
//     step 1  back-trace the four corners (eq. 14/15) -> upstream quadrilateral, its
//             bounding box -> anchor (r0,s0) and the candidate source cells (Table 4 step 1);
//     step 4  back-trace the o^2 Gauss-Legendre nodes, invert the Vandermonde matrix in centred
//             coordinates -> adjoint polynomials phi*_m (Table 4 step 4);
//   then per candidate source cell (<= 3x3):
//     steps 2,3,5  monomial moments of  A*_ij cap A_rs  by Green's theorem along the clipped upstream
//             edges ("outer segments") and the piece of the cell's right edge inside the upstream cell
//             ("inner segments", Table 4 steps 2,3,5), contracted with the Lagrange basis
//             and phi* into the coefficients C of eq. (18), stored as W = C / W_m.
//   (the apply kernels, eq. (17), live in sldg_xy_apply.cu)
//
// Green's theorem with P = 0, Q^{(p,q)} = x^{p+1} y^q / (p+1)  (R7; reproduces the paper's
// Q^{(2,1)}, Q^{(2,2)}): in the source cell's local coordinates horizontal segments and
// segments on the cell's left edge x=0 contribute nothing; only the upstream edges and the pieces of the
// cell's right edge x=1 inside the upstream cell do.
//
// All geometry is done in cell units relative to the target cell (the target is [0,1]^2), the integrals
// in the source cell's own local coordinates (R10).
//
// Output per (z node, cell): header int4 {ax, ay, mask, count} (anchor = offset of slot (0,0) relative to
// the target cell, unwrapped; mask over the 3x3 slots, bit dx + 3 dy) and `count` weight blocks of o^4
// doubles, k-major (W[k*o2+m]), packed in increasing slot order at W[cell][0..count).
#include "sldg_internal.cuh"
#include "sldg_xy_geometry.cuh"

using namespace sldg_geom;

namespace {

#ifndef SLDG_GEOM_WARPS
#define SLDG_GEOM_WARPS 1  // 1: the warps of a block work independently (32 cells each); 0: block-wide phases
#endif
#ifndef SLDG_GEOM_MINB2
#define SLDG_GEOM_MINB2 5  // resident blocks per SM the o = 2 kernel is compiled for (102 registers)
#endif
template <int O>
__global__ void __launch_bounds__(GeomShared<O>::CELLS, (O == 2 ? SLDG_GEOM_MINB2 : 1)) xy_geometry_kernel(const double *__restrict__ va,
                                                                           const double *__restrict__ vb,
                                                                           int4 *__restrict__ hdr, double *__restrict__ W,
                                                                           int32_t *err,
                                                                           GridDev g, Basis bs, double tau, int order,
                                                                           int periodic)
{
    constexpr int CELLS = GeomShared<O>::CELLS;
    extern __shared__ __align__(16) unsigned char geom_smem[];
    const int ncell = g.n[0] * g.n[1];
    const int t0 = blockIdx.x * CELLS, z = blockIdx.y;
#if SLDG_GEOM_WARPS
    // every warp does its own 32 cells -- set-up, enumeration of their pieces, the pieces -- on its own slice of shared
    // memory and synchronises with __syncwarp only: no block-wide barrier (their stalls were 9 % of the kernel's samples;
    // the warps of a block drift apart and hide each other's latencies)
    GeomShared<O, 32> &sh = reinterpret_cast<GeomShared<O, 32> *>(geom_smem)[threadIdx.x >> 5];
    const int w0 = t0 + (threadIdx.x & ~31);
    geometry_block<O, 32, true>(sh, threadIdx.x & 31, 32, [&](int c) { return w0 + c < ncell ? w0 + c : -1; }, z, va, vb,
                                hdr, W, err, g, bs, tau, order, periodic);
#else
    GeomShared<O> &sh = *reinterpret_cast<GeomShared<O> *>(geom_smem);
    geometry_block<O, CELLS>(sh, threadIdx.x, CELLS, [&](int c) { return t0 + c < ncell ? t0 + c : -1; }, z, va, vb,
                             hdr, W, err, g, bs, tau, order, periodic);
#endif
}

// debug/test helper: expand the packed weight blocks of one z plane to the dense [cell][slot] form
__global__ void geometry_expand_kernel(const int4 *__restrict__ hdr, const double *__restrict__ W, int ncell, int o4,
                                       int wbs,
                                       int32_t *__restrict__ anchor, int32_t *__restrict__ mask,
                                       double *__restrict__ Wd)
{
    const int t = blockIdx.x;
    const int4 h = hdr[t];
    if (threadIdx.x == 0) {
        if (anchor) {
            anchor[2 * t] = h.x;
            anchor[2 * t + 1] = h.y;
        }
        if (mask) mask[t] = h.z;
    }
    if (!Wd) return;
    int n = 0;
    for (int slot = 0; slot < 9; ++slot) {
        if (!((h.z >> slot) & 1)) continue;
        for (int e = threadIdx.x; e < o4; e += blockDim.x)
            Wd[((size_t)t * 9 + slot) * o4 + e] = W[((size_t)t * 9 + n) * wbs + e];
        ++n;
    }
}

}  // namespace

static int xy_geometry_blocks_per_z(const sldg_ctx *c)
{
    const int ncell = c->g.n[0] * c->g.n[1];
    const int threads = c->g.o[0] == 3 ? GeomShared<3>::CELLS : GeomShared<2>::CELLS;
    return (ncell + threads - 1) / threads;
}

cudaError_t launch_xy_geometry(sldg_ctx *c, double tau, int trace_order)
{
    cudaStream_t stream = c->stream;
    const GridDev &g = c->g;
    const int O = g.o[0];
    dim3 grid((unsigned)xy_geometry_blocks_per_z(c), (unsigned)g.N[2]);
#define LAUNCH_G(OO)                                                                                              \
    do {                                                                                                          \
        auto kern = xy_geometry_kernel<OO>;                                                                       \
        const size_t smem = SLDG_GEOM_WARPS ? (GeomShared<OO>::CELLS / 32) * sizeof(GeomShared<OO, 32>)            \
                                            : sizeof(GeomShared<OO>);                                             \
        cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);                       \
        kern<<<grid, GeomShared<OO>::CELLS, smem, stream>>>(                                                      \
            c->va, c->vb, c->hdr, c->W, c->err, g, c->basis, tau, trace_order, c->vel_periodic);        \
    } while (0)
    if (O == 1) LAUNCH_G(1); else if (O == 2) LAUNCH_G(2); else LAUNCH_G(3);
#undef LAUNCH_G
    c->launches++;
    return cudaGetLastError();
}

cudaError_t launch_geometry_expand(sldg_ctx *c, int z, int32_t *anchor, int32_t *mask, double *Wd)
{
    const GridDev &g = c->g;
    const int ncell = g.n[0] * g.n[1];
    const int o4 = g.o[0] * g.o[0] * g.o[0] * g.o[0];
    const int wbs = sldg_w_block_doubles(g.o[0]);
    geometry_expand_kernel<<<ncell, 32, 0, c->stream>>>(c->hdr + (size_t)z * ncell, c->W + (size_t)z * ncell * 9 * wbs,
                                                        ncell, o4, wbs, anchor, mask, Wd);
    c->launches++;
    return cudaGetLastError();
}
