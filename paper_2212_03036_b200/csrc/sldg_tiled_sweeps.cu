// sldg_tiled_sweeps.cu -- the two adjacent 1d SLDG sweeps of a Strang step in one pass over f, z-TILED (sm_100a).
//
// sldg_fused_sweeps.cu keeps the whole (z,v) plane of an (x,y) node in shared memory: one block per SM, every phase
// of a plane ends at a block-wide barrier and nothing else runs on the SM meanwhile (ncu, round 2: `barrier` 0.8-1.7
// and `long_scoreboard` 1.7-2.2 stalls per issue, 80-85 % of the copy rate), and a plane of more than 227 KB (the
// paper's grid, Nv = 256) does not fit at all.  When the Courant numbers of the z sweep are small -- the drift-kinetic
// regime: |v| dt / (2 h_z) = 0.6 at BASELINE.json's configs -- a target z cell only needs the source cells
// [i + s_min, i + s_max + 1] (eq. 11), so the plane is cut into tiles of T target z cells plus a halo of
// hl = ceil(max |v| tau / h_z) cells below and hl + 1 above.  A tile is 20-40 KB: several independent blocks share an
// SM and one block's barrier and load waits hide under the others' arithmetic; no producer warp, no double buffering
// inside a block.  The halo lines are read twice, from L2 (neighbouring tiles are in flight at the same time).
//
//   ZV  phase A  z sweep in place, thread <-> (v, slice of the tile's targets): the result of target cell i is written
//                over its left source cell, dead by then -- column v ends up shifted by s(v) cells (no wrap: the halo);
//       phase B  v sweep of the tile's target lines, warp <-> line, lane <-> source cells, results to global memory.
//   VZ  phase A  v sweep in place of every loaded line (the halo lines are done by both neighbours);
//       phase B  z sweep, thread <-> (v, slice), results to global memory.
// The arithmetic of each sweep is that of sldg_sweeps.cu / sldg_fused_sweeps.cu, operation by operation: the result is
// bit-identical to the two separate kernels.  Large Courant numbers (configs[2]) keep the other kernels.
#include <math.h>
#include <stdlib.h>

#include "sldg_async.cuh"
#include "sldg_sweep_common.cuh"

namespace {

constexpr int TILE_THREADS = 256;
constexpr int TILE_WARPS = TILE_THREADS / 32;
constexpr int TILE_MAXCPL = 4;  // v cells per lane in the line-wise phases (nv <= 128)

// dynamic shared memory: lines [NLmax][Pv] | per line A, B of its v shift [NLmax][2 O^2] | per column A, B of its z
// shift [2 O^2][Pv] | per line s_v [NLmax] | per column s_z + hl [Pv] | barrier
__host__ __device__ inline size_t tile_smem_bytes(int NLmax, int Pv, int O)
{
    return (size_t)NLmax * Pv * 8 + (size_t)NLmax * 2 * O * O * 8 + (size_t)Pv * 2 * O * O * 8 + (size_t)NLmax * 4 +
           (size_t)Pv * 4 + 32;
}

template <int O, int CPL, bool ZFIRST>
__global__ void __launch_bounds__(TILE_THREADS) tiled_sweep_kernel(const double *__restrict__ fin,
                                                                   double *__restrict__ fout,
                                                                   const double *__restrict__ Ez, GridDev g,
                                                                   ShiftPoly spz, ShiftPoly spv, Basis bs,
                                                                   double tau_z, double tau_v, int T, int hl, int hr)
{
    extern __shared__ __align__(128) unsigned char tile_smem[];
    const int Nz = g.N[2], nz = g.n[2], Nv = g.N[3], nv = g.n[3], Pv = g.Pv;
    const int NLmax = (T + hl + hr) * O;
    double *buf = reinterpret_cast<double *>(tile_smem);
    double *vAB = buf + (size_t)NLmax * Pv;               // [NLmax][2][O][O]
    double *zAB = vAB + (size_t)NLmax * 2 * O * O;        // [2 O O][Pv]
    int *vs = reinterpret_cast<int *>(zAB + (size_t)Pv * 2 * O * O);  // [NLmax]
    int *zsh = vs + NLmax;                                // [Pv]: s_z(v) + hl = buffer cell of target 0's left source
    uint64_t *bar = reinterpret_cast<uint64_t *>((reinterpret_cast<uintptr_t>(zsh + Pv) + 7) & ~(uintptr_t)7);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const long long plane_nodes = (long long)g.N[1] * g.N[0];

    // per column: (s, A, B) of the z shift, once per block
    for (int c = tid; c < Pv; c += TILE_THREADS) {
        const int ov = g.o[3];
        const int vv = c < Nv ? c : 0;
        const int l = vv / ov, q = vv - l * ov;
        const double vq = __dadd_rn(g.lo[3], __dmul_rn(__dadd_rn((double)l, bs.xi[ov][q]), g.h[3]));
        int s0;
        double alpha, A0[O][O], B0[O][O];
        shift_of(vq, tau_z, g.h[2], s0, alpha);
        eval_shift<O>(spz, alpha, A0, B0);
        zsh[c] = c < Nv ? s0 + hl : 0;  // the host chose hl, hr such that 0 <= s + hl and s + hl + 1 < hl + hr
#pragma unroll
        for (int j = 0; j < O; ++j)
#pragma unroll
            for (int m = 0; m < O; ++m) {
                zAB[(j * O + m) * Pv + c] = A0[j][m];
                zAB[(O * O + j * O + m) * Pv + c] = B0[j][m];
            }
    }
    if (tid == 0) {
        mbar_init(bar, 1);
        mbar_fence_init();
    }
    __syncthreads();

    // z sweep: thread <-> (v, slice qd of the tile's target cells)
    const int v = tid % Pv, qd = tid / Pv;
    const int nqmax = TILE_THREADS / Pv > 0 ? TILE_THREADS / Pv : 1;
    // line-wise phase of the z,v pair: byte offsets of row 0 of this lane's columns (left source cell c0 of its target
    // and the next cell), shifted by s_z(v) cells; o = 2: lanes 8-15 / 24-31 take the two DOFs in the opposite order so
    // that a half warp covers all banks (sldg_fused_sweeps.cu)
    const int msw = (O == 2) ? ((lane >> 3) & 1) : 0;
    uint32_t off0[CPL][O], off1[CPL][O];
#pragma unroll
    for (int k = 0; k < CPL; ++k)
#pragma unroll
        for (int m = 0; m < O; ++m) {
            const int cell = lane + 32 * k;
            const int c0 = (ZFIRST && cell < nv) ? cell : 0;
            const int c1 = (c0 + 1 == nv) ? 0 : c0 + 1;
            const int md = m ^ msw;
            off0[k][m] = ZFIRST ? (uint32_t)(zsh[c0 * O + md] * O * Pv + c0 * O + md) * 8u : 0u;
            off1[k][m] = ZFIRST ? (uint32_t)(zsh[c1 * O + md] * O * Pv + c1 * O + md) * 8u : 0u;
        }

    const int ntiles = (nz + T - 1) / T;
    const long long nitems = plane_nodes * ntiles;
    uint32_t ph = 0;
    const uint32_t line_bytes = (uint32_t)Pv * 8;
    for (long long item = blockIdx.x; item < nitems; item += gridDim.x) {
        const int col = (int)(item / ntiles), t = (int)(item - (long long)col * ntiles);
        const int i0 = t * T, Tt = min(T, nz - i0);
        const int NLt = (Tt + hl + hr) * O;
        const int X = col % g.N[0], Y = col / g.N[0];
        const double *src = fin + Y * g.sY + X * g.sX;
        double *dst = fout + Y * g.sY + X * g.sX;
        const int zfirst = (i0 - hl) * O;  // global z line of buffer line 0 (before wrapping)
        // ---- stage the tile: one bulk copy per line, all completing on one barrier ------------------------------
        if (warp == 0) {
            if (lane == 0) mbar_arrive_expect_tx(bar, (uint32_t)NLt * line_bytes);
            __syncwarp();
            for (int l = lane; l < NLt; l += 32) bulk_g2s(buf + (size_t)l * Pv, src + (long long)wrapi(zfirst + l, Nz) * g.sZ, line_bytes, bar);
        }
        // ---- per line the (s, A, B) of its v shift (under the copies): the target lines (ZV) or every line (VZ) ---
        for (int l = tid; l < (ZFIRST ? Tt * O : NLt); l += TILE_THREADS) {
            const int zg = ZFIRST ? i0 * O + l : wrapi(zfirst + l, Nz);
            int s;
            double alpha, A[O][O], B[O][O];
            shift_of(__ldg(Ez + zg * plane_nodes + col), tau_v, g.h[3], s, alpha);
            eval_shift<O>(spv, alpha, A, B);
            vs[l] = wrapi(s, nv);
#pragma unroll
            for (int j = 0; j < O; ++j)
#pragma unroll
                for (int m = 0; m < O; ++m) {
                    vAB[(l * 2) * O * O + j * O + m] = A[j][m];
                    vAB[(l * 2 + 1) * O * O + j * O + m] = B[j][m];
                }
        }
        mbar_wait(bar, ph);
        ph ^= 1;
        __syncthreads();

        const int nq = min(nqmax, Tt);
        const bool zact = qd < nq && v < Nv;
        const int zi0 = (int)((long long)qd * Tt / nq), zi1 = (int)((long long)(qd + 1) * Tt / nq);
        if (ZFIRST) {
            // ---- phase A: z sweep in place; the result of target cell i lands on buffer cell i + s + hl ------------
            int c = 0;
            double up[O], last[O], Az[O][O], Bz[O][O];
            if (zact) {
#pragma unroll
                for (int j = 0; j < O; ++j)
#pragma unroll
                    for (int m = 0; m < O; ++m) {
                        Az[j][m] = zAB[(j * O + m) * Pv + v];
                        Bz[j][m] = zAB[(O * O + j * O + m) * Pv + v];
                    }
                c = zi0 + zsh[v];
                const int cl = zi1 + zsh[v];
#pragma unroll
                for (int m = 0; m < O; ++m) {
                    up[m] = buf[(size_t)(c * O + m) * Pv + v];
                    last[m] = buf[(size_t)(cl * O + m) * Pv + v];  // first slot of the next slice: it is overwritten
                }
            }
            __syncthreads();
            if (zact) {
                const int cstep = O * Pv;
                int off = c * cstep + v;
                auto step = [&](const double (&un)[O]) {
#pragma unroll
                    for (int j = 0; j < O; ++j) {
                        double acc = 0.0;
#pragma unroll
                        for (int m = 0; m < O; ++m) acc = fma(Az[j][m], up[m], acc);
#pragma unroll
                        for (int m = 0; m < O; ++m) acc = fma(Bz[j][m], un[m], acc);
                        buf[off + j * Pv] = acc;
                    }
#pragma unroll
                    for (int m = 0; m < O; ++m) up[m] = un[m];
                };
#pragma unroll 2
                for (int i = zi0; i + 1 < zi1; ++i) {
                    const int offn = off + cstep;
                    double un[O];
#pragma unroll
                    for (int m = 0; m < O; ++m) un[m] = buf[offn + m * Pv];
                    step(un);
                    off = offn;
                }
                step(last);
            }
            __syncthreads();
            // ---- phase B: v sweep of the target lines, to global memory -------------------------------------------
            const uint32_t buf_b = smem_u32(buf), vab_b = smem_u32(vAB), vs_b = smem_u32(vs);
            const uint32_t row_b = (uint32_t)Pv * 8u;
#pragma unroll 1
            for (int r = warp; r < Tt * O; r += TILE_WARPS) {
                const int s = lds_s32(vs_b + 4u * r);
                double A[O][O], B[O][O];
                {
                    double ab[2 * O * O];
                    const uint32_t at = vab_b + (uint32_t)r * (2 * O * O * 8);
#pragma unroll
                    for (int e = 0; e < O * O; ++e) {
                        const double2 tt = lds_v2f64(at + 16u * e);
                        ab[2 * e] = tt.x;
                        ab[2 * e + 1] = tt.y;
                    }
#pragma unroll
                    for (int j = 0; j < O; ++j)
#pragma unroll
                        for (int m = 0; m < O; ++m) {
                            A[j][m] = ab[j * O + m];
                            B[j][m] = ab[O * O + j * O + m];
                        }
                }
                double *w = dst + (long long)(i0 * O + r) * g.sZ;
                const uint32_t zb = buf_b + (uint32_t)r * row_b;
#pragma unroll
                for (int k = 0; k < CPL; ++k) {
                    const int cell = lane + 32 * k;
                    if (cell < nv) {
                        double u0[O], u1[O];
#pragma unroll
                        for (int m = 0; m < O; ++m) {
                            u0[m] = lds_f64(zb + off0[k][m]);
                            u1[m] = lds_f64(zb + off1[k][m]);
                        }
                        if (O == 2 && msw) {
                            double tt = u0[0]; u0[0] = u0[O - 1]; u0[O - 1] = tt;
                            tt = u1[0]; u1[0] = u1[O - 1]; u1[O - 1] = tt;
                        }
                        int c = cell - s;  // the target whose left source cell this is
                        if (c < 0) c += nv;
                        double rr[O];
#pragma unroll
                        for (int j = 0; j < O; ++j) {
                            double acc = 0.0;
#pragma unroll
                            for (int m = 0; m < O; ++m) acc = fma(A[j][m], u0[m], acc);
#pragma unroll
                            for (int m = 0; m < O; ++m) acc = fma(B[j][m], u1[m], acc);
                            rr[j] = acc;
                        }
                        if (O == 2) {
                            __stcs(reinterpret_cast<double2 *>(w + 2 * c), make_double2(rr[0], rr[O - 1]));
                        } else {
#pragma unroll
                            for (int j = 0; j < O; ++j) __stcs(w + c * O + j, rr[j]);
                        }
                    }
                }
            }
        } else {
            // ---- phase A: v sweep in place of every loaded line, warp <-> line ------------------------------------
#pragma unroll 1
            for (int l = warp; l < NLt; l += TILE_WARPS) {
                const int s = vs[l];
                double A[O][O], B[O][O];
#pragma unroll
                for (int j = 0; j < O; ++j)
#pragma unroll
                    for (int m = 0; m < O; ++m) {
                        A[j][m] = vAB[(l * 2) * O * O + j * O + m];
                        B[j][m] = vAB[(l * 2 + 1) * O * O + j * O + m];
                    }
                double *u = buf + (size_t)l * Pv;
                double u0[CPL][O], u1[CPL][O];
#pragma unroll
                for (int k = 0; k < CPL; ++k) {
                    const int cell = lane + 32 * k;
                    if (cell < nv) {
                        int c0 = cell + s;
                        if (c0 >= nv) c0 -= nv;
                        int c1 = c0 + 1;
                        if (c1 >= nv) c1 -= nv;
                        if (O == 2) {
                            const double2 t0 = *reinterpret_cast<const double2 *>(u + 2 * c0);
                            const double2 t1 = *reinterpret_cast<const double2 *>(u + 2 * c1);
                            u0[k][0] = t0.x; u0[k][O - 1] = t0.y;
                            u1[k][0] = t1.x; u1[k][O - 1] = t1.y;
                        } else {
#pragma unroll
                            for (int m = 0; m < O; ++m) {
                                u0[k][m] = u[c0 * O + m];
                                u1[k][m] = u[c1 * O + m];
                            }
                        }
                    }
                }
                __syncwarp();  // every source of this line is in registers: the line may be overwritten
#pragma unroll
                for (int k = 0; k < CPL; ++k) {
                    const int cell = lane + 32 * k;
                    if (cell < nv) {
                        double rr[O];
#pragma unroll
                        for (int j = 0; j < O; ++j) {
                            double acc = 0.0;
#pragma unroll
                            for (int m = 0; m < O; ++m) acc = fma(A[j][m], u0[k][m], acc);
#pragma unroll
                            for (int m = 0; m < O; ++m) acc = fma(B[j][m], u1[k][m], acc);
                            rr[j] = acc;
                        }
                        if (O == 2) {
                            *reinterpret_cast<double2 *>(u + 2 * cell) = make_double2(rr[0], rr[O - 1]);
                        } else {
#pragma unroll
                            for (int j = 0; j < O; ++j) u[cell * O + j] = rr[j];
                        }
                    }
                }
            }
            __syncthreads();
            // ---- phase B: z sweep, thread <-> (v, slice of the targets), to global memory -------------------------
            if (zact) {
                double Az[O][O], Bz[O][O];
#pragma unroll
                for (int j = 0; j < O; ++j)
#pragma unroll
                    for (int m = 0; m < O; ++m) {
                        Az[j][m] = zAB[(j * O + m) * Pv + v];
                        Bz[j][m] = zAB[(O * O + j * O + m) * Pv + v];
                    }
                const int cstep = O * Pv;
                int off = (zi0 + zsh[v]) * cstep + v;
                double up[O];
#pragma unroll
                for (int m = 0; m < O; ++m) up[m] = buf[off + m * Pv];
                double *w = dst + v + (long long)((i0 + zi0) * O) * g.sZ;
#pragma unroll 2
                for (int i = zi0; i < zi1; ++i) {
                    off += cstep;
                    double un[O];
#pragma unroll
                    for (int m = 0; m < O; ++m) un[m] = buf[off + m * Pv];
#pragma unroll
                    for (int j = 0; j < O; ++j) {
                        double acc = 0.0;
#pragma unroll
                        for (int m = 0; m < O; ++m) acc = fma(Az[j][m], up[m], acc);
#pragma unroll
                        for (int m = 0; m < O; ++m) acc = fma(Bz[j][m], un[m], acc);
                        __stcs(w, acc);
                        w += g.sZ;
                    }
#pragma unroll
                    for (int m = 0; m < O; ++m) up[m] = un[m];
                }
            }
        }
        fence_proxy_async();  // generic reads and writes of the tile before the next item's bulk copies
        __syncthreads();
    }
}

}  // namespace

// The pair (z then v, or v then z) in one z-tiled pass; cudaErrorNotSupported when the Courant numbers of the z sweep
// are too large for a halo (the caller falls back to the whole-plane kernel or the two separate kernels).
cudaError_t launch_tiled_sweeps(sldg_ctx *c, const double *fin, double *fout, double tau_z, double tau_v, bool z_first)
{
    const GridDev &g = c->g;
    const int O = g.o[2];
    if (g.o[3] != O || g.Pv > TILE_THREADS || g.n[3] > 32 * TILE_MAXCPL) return cudaErrorNotSupported;
    // o = 3: ~200 registers, one block per SM -- measured no faster than the two separate kernels (c4o3: 10.6 vs 10.4 ms)
    if (O == 3 && !getenv("SLDG_FORCE_TILE")) return cudaErrorNotSupported;
    // |s| <= ceil(max |v| |tau| / h_z): sources of target i lie in cells [i - hl, i + hl + 1]
    const double vabs = fmax(fabs(g.lo[3]), fabs(g.lo[3] + g.n[3] * g.h[3]));
    const double dmax = vabs * fabs(tau_z) / g.h[2];
    if (!(dmax < 1e6)) return cudaErrorNotSupported;
    const int hl = (int)ceil(dmax), hr = hl + 1;
    const int nz = g.n[2];
    static const int t_env = getenv("SLDG_TILE_T") ? atoi(getenv("SLDG_TILE_T")) : 16;
    int T = nz < t_env ? nz : t_env;
    if (hl + hr > T) return cudaErrorNotSupported;  // halo larger than the tile: not the regime this kernel is for
    const size_t budget = 227 * 1024;
    const int NLmax = (T + hl + hr) * O;
    const size_t smem = tile_smem_bytes(NLmax, g.Pv, O);
    if (smem + 1024 > budget) return cudaErrorNotSupported;
    const int cpl = (g.n[3] + 31) / 32;
#define PICK_T(OO, CC) (z_first ? (const void *)tiled_sweep_kernel<OO, CC, true> : (const void *)tiled_sweep_kernel<OO, CC, false>)
#define PICK_C(OO) (cpl <= 1 ? PICK_T(OO, 1) : cpl == 2 ? PICK_T(OO, 2) : cpl == 3 ? PICK_T(OO, 3) : PICK_T(OO, 4))
    const void *kern = O == 1 ? PICK_C(1) : (O == 2 ? PICK_C(2) : PICK_C(3));
#undef PICK_C
#undef PICK_T
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, TILE_THREADS, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorNotSupported;
    const long long nitems = (long long)g.N[0] * g.N[1] * ((nz + T - 1) / T);
    const long long cap = (long long)c->sm_count * per_sm;
    const unsigned grid = (unsigned)(nitems < cap ? nitems : cap);
    GridDev gg = g;
    ShiftPoly spz = c->sp_z, spv = c->sp_v;
    Basis bs = c->basis;
    const double *Ez = c->Ez;
    void *args[] = {&fin, &fout, &Ez, &gg, &spz, &spv, &bs, &tau_z, &tau_v, &T, (void *)&hl, (void *)&hr};
    e = cudaLaunchKernel(kern, dim3(grid), dim3(TILE_THREADS), args, smem, c->stream);
    if (e != cudaSuccess) return e;
    c->launches++;
    return cudaGetLastError();
}
