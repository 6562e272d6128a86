// sldg_source.cu -- the source-term substep of the delta-g formulation (eq. (3); section 3.5, PAPER.md:269-279;
// Algorithm 1 steps 2 and 9):
//     dg[z,v,y,x] += tau * ( d_z phi[z,y,x] * d_v g_eq[v,x]  +  d_theta phi[z,y,x] * d_r(g_eq / r)[v,x] )
// with x = r, y = theta.  Forward Euler, as printed at PAPER.md:279; it conserves mass when the two derivatives of phi
// have zero Gauss sums along z and theta (centred differences of a periodic potential) -- and the v sum of d_v g_eq is
// zero by symmetry.  One pass over f, in place: 16 B per DOF, HBM-bound (the paper: 1290 GB/s on an A100).
// Lanes along v (contiguous): the two field values of a line are warp-uniform, the two equilibrium profiles are rows of
// an [X][Pv] table that stays in L1/L2.
#include "sldg_internal.cuh"

namespace {

// [Nv][Nx] (canonical, x fastest) -> [Nx][Pv] (v fastest, zero padded): the layout the kernel streams
__global__ void __launch_bounds__(256) source_profile_kernel(const double *__restrict__ in, double *__restrict__ out,
                                                             int Nx, int Nv, int Pv)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= Nx * Pv) return;
    const int X = t / Pv, v = t - X * Pv;
    out[t] = v < Nv ? in[(long long)v * Nx + X] : 0.0;
}

// Block <-> rows (z, Y) of Nx lines; warp <-> U lines of the row at a time, lane <-> the v pairs lane + 32 k: no
// divisions in the inner loops, all loads of the U lines issued before the first store.
template <int U>
__global__ void __launch_bounds__(256) source_step_kernel(const double *fin, double *f, const double *__restrict__ dz,
                                                          const double *__restrict__ dth, const double *__restrict__ gv,
                                                          const double *__restrict__ gr, GridDev g, double tau)
{
    constexpr int MAXP = 4;  // v pairs per lane held in registers (Pv <= 256); longer lines take more passes
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int Nx = g.N[0], Ny = g.N[1], P2 = g.Pv / 2;
    const int rows = g.N[2] * Ny;
    for (int row = blockIdx.x; row < rows; row += gridDim.x) {
        const int Z = row / Ny, Y = row - Z * Ny;
        double *frow = f + Z * g.sZ + Y * g.sY;
        const double *irow = fin + Z * g.sZ + Y * g.sY;  // fin == f: in place
        const double *dzr = dz + (long long)row * Nx, *dtr = dth + (long long)row * Nx;
        for (int X0 = warp * U; X0 < Nx; X0 += 8 * U) {
            for (int v0 = lane; v0 < P2; v0 += 32 * MAXP) {
                double2 u[U][MAXP];
#pragma unroll
                for (int k = 0; k < U; ++k)
#pragma unroll
                    for (int p = 0; p < MAXP; ++p) {
                        const int X = X0 + k, v2 = v0 + 32 * p;
                        if (X < Nx && v2 < P2) u[k][p] = __ldcs(reinterpret_cast<const double2 *>(irow + X * g.sX + 2 * v2));
                    }
#pragma unroll
                for (int k = 0; k < U; ++k) {
                    const int X = X0 + k;
                    if (X >= Nx) continue;
                    const double a = tau * __ldg(dzr + X), b = tau * __ldg(dtr + X);
#pragma unroll
                    for (int p = 0; p < MAXP; ++p) {
                        const int v2 = v0 + 32 * p;
                        if (v2 >= P2) continue;
                        const double2 pv = __ldg(reinterpret_cast<const double2 *>(gv + (long long)X * g.Pv + 2 * v2));
                        const double2 pr = __ldg(reinterpret_cast<const double2 *>(gr + (long long)X * g.Pv + 2 * v2));
                        u[k][p].x += a * pv.x + b * pr.x;
                        u[k][p].y += a * pv.y + b * pr.y;
                        __stcs(reinterpret_cast<double2 *>(frow + X * g.sX + 2 * v2), u[k][p]);
                    }
                }
            }
        }
    }
}

}  // namespace

size_t source_workspace_bytes(const sldg_params *p)
{
    const size_t Nx = (size_t)p->n[0] * p->order[0], Ny = (size_t)p->n[1] * p->order[1], Nz = (size_t)p->n[2] * p->order[2];
    const size_t Pv = (((size_t)p->n[3] * p->order[3]) + SLDG_PV_ALIGN - 1) / SLDG_PV_ALIGN * SLDG_PV_ALIGN;
    auto al = [](size_t b) { return (b + 255) & ~(size_t)255; };
    return 2 * al(Nz * Ny * Nx * 8) + 2 * al(Nx * Pv * 8);
}

void source_carve(sldg_ctx *c, char *base)
{
    const GridDev &g = c->g;
    auto al = [](size_t b) { return (b + 255) & ~(size_t)255; };
    c->src_dz = (double *)base;
    c->src_dth = (double *)(base + al((size_t)g.lines * 8));
    c->src_gv = (double *)(base + 2 * al((size_t)g.lines * 8));
    c->src_gr = (double *)(base + 2 * al((size_t)g.lines * 8) + al((size_t)g.N[0] * g.Pv * 8));
    c->src_ready = 0;
}

// canon_dev: [Nv][Nx]; staged through the (idle) partial-sum scratch is not possible (size): the caller's buffer is read directly
cudaError_t launch_source_profiles(sldg_ctx *c, const double *dv_geq, const double *dr_geq)
{
    const GridDev &g = c->g;
    const int n = g.N[0] * g.Pv;
    source_profile_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(dv_geq, c->src_gv, g.N[0], g.N[3], g.Pv);
    source_profile_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(dr_geq, c->src_gr, g.N[0], g.N[3], g.Pv);
    c->launches += 2;
    return cudaGetLastError();
}

cudaError_t launch_source_step(sldg_ctx *c, double *f, double tau, const double *fin)
{
    if (!fin) fin = f;
    const GridDev &g = c->g;
    const long long rows = (long long)g.N[2] * g.N[1];
    const long long cap = (long long)c->sm_count * 8;
    source_step_kernel<2><<<(unsigned)(rows < cap ? rows : cap), 256, 0, c->stream>>>(fin, f, c->src_dz, c->src_dth, c->src_gv,
                                                                                   c->src_gr, g, tau);
    c->launches++;
    return cudaGetLastError();
}
