// sldg_fused_sweeps.cu -- the two adjacent 1d SLDG sweeps of a Strang step in ONE pass over f (sm_100a).
//
// Algorithm 1 runs z(dt/2) v(dt/2) before the 2d step and v(dt/2) z(dt/2) after it, with
// nothing in between the two sweeps of a pair.  Each sweep alone reads and writes all of f (16 B per DOF); the
// pair fused moves the same 16 B per DOF once.  Both sweeps act inside one (x,y) node's (z,v) plane (the z sweep
// mixes z cells at fixed v, the v sweep v cells at fixed z), and that plane -- Nz lines of Pv doubles, 128 KiB at
// 128 x 128 -- fits in shared memory.  The arithmetic of each sweep is that of sldg_sweeps.cu, operation by
// operation, so the fused pair is bit-identical to the two separate kernels.
//
// One persistent block (16 compute warps + 1 producer warp) per SM walks over the (Y,X) planes:
//   stage   a dedicated producer warp fetches the planes with bulk copies (one per line, completing on mbarriers).
//           Shared memory holds [L_a: NL lines | H: NH lines | L_b: NL lines], NL + NH = Nz: even planes live in
//           [L_a | H], odd planes in [H | L_b], so a plane is always one contiguous tile [Nz][Pv] and the other L
//           is free: NL lines of the NEXT plane are fetched under the compute phases of the current one, the
//           remaining NH lines as soon as the current plane is done (NL = 80 of 128 at 128 x 128, o = 2);
//   ZV      phase A  z sweep in place, thread <-> (v, slice of z): the result for target cell i is written over
//                    its left source cell (i+s) mod nz, which is dead by then -- column v ends up rotated by s(v);
//           phase B  v sweep line by line, warp <-> line, lane <-> source cells (the rotation offsets of a lane's
//                    columns sit in registers; the other source cell of a target comes from the next lane by
//                    shuffle), results straight to global memory;
//   VZ      phase A  v sweep in place, warp <-> line (all sources of a warp's line are in registers before the
//                    first write);
//           phase B  z sweep, thread <-> (v, slice of z), results straight to global memory.
#include "sldg_async.cuh"
#include "sldg_sweep_common.cuh"

namespace {

constexpr int FUSED_THREADS = 512;          // compute threads (16 warps)
constexpr int FUSED_BLOCK = FUSED_THREADS + 32;  // + one producer warp
constexpr int FUSED_MAXCPL = 4;  // v cells per lane in the line-wise phases (nv <= 128)

// dynamic shared memory: planes [2 NL + NH][Pv] doubles | per line: A, B of its v shift [Nz][2 O^2] doubles |
// per column: A, B of its z shift [2 O^2][Pv] doubles | per line: s [Nz] ints | per column: rotation offset
// [Pv] ints, z shift [Pv] ints | barriers | z,v pair: line order per plane parity [2][Nz] shorts, marks [2][Nz] bytes
__host__ __device__ inline size_t fused_table_bytes(int Nz, int Pv, int O, bool rho = false)
{
    // o <= 2: A, B of the column's z shift stay in the registers of the column's threads (every KB of tables is a line
    // less fetched ahead: 0.02 ms per KB and z,v pair at 128 x 128)
    return (size_t)Nz * 2 * O * O * 8 + (O <= 2 ? 0 : (size_t)Pv * 2 * O * O * 8) + (size_t)Nz * 4 + (size_t)Pv * 8 + 64 +
           (size_t)Nz * 6 + 16 +  // + line order of the z,v pair's line-wise phase [2][Nz] shorts, marks [2][Nz] bytes
           (rho ? (size_t)(Pv / 32) * Nz * 8 + 8 : 0);  // RHO: per warp of a z slice, the partial v sums of the plane's rows
}

// ZONLY (with ZFIRST = false): the z sweep alone through the same planes -- for Courant numbers so different from
// one v node to the next that the column walk of advect_z_kernel reads a different z row in almost every lane.
// RHO (v,z pair only; o <= 2, Pv a multiple of 32, Nv = Pv): the charge density of the NEW state, rho = h_v sum_v w f
// (PAPER.md:57), is formed from the results of the z sweep as they leave for global memory -- sldg_strang_step_host then
// needs no further pass over f.
template <int O, int CPL, bool ZFIRST, bool ZONLY, bool FULLV, bool RHO = false>
__global__ void __launch_bounds__(FUSED_BLOCK, 1) fused_sweep_kernel(const double *__restrict__ fin,
                                                                       double *__restrict__ fout,
                                                                       const double *__restrict__ Ez, GridDev g,
                                                                       ShiftPoly spz, ShiftPoly spv, Basis bs,
                                                                       double tau_z, double tau_v, int NL, int col0,
                                                                       int col1, double *__restrict__ rho)
{
    extern __shared__ __align__(16) unsigned char fused_smem[];
    const int Nz = g.N[2], nz = g.n[2], Nv = g.N[3], nv = g.n[3], Pv = g.Pv;
    const int NH = Nz - NL;
    double *buf = reinterpret_cast<double *>(fused_smem);  // [L_a | H | L_b]
    double *vAB = buf + (size_t)(2 * NL + NH) * Pv;        // [Nz][2][O][O]: A then B of the line's v shift
    double *zAB = vAB + (size_t)Nz * 2 * O * O;            // [2 O O][Pv]: A then B of the column's z shift
    constexpr bool ZREG = O <= 2;                          // zAB in registers instead (fused_table_bytes)
    int *vs = reinterpret_cast<int *>(zAB + (ZREG ? 0 : (size_t)Pv * 2 * O * O));  // [Nz]: the line's integer v shift, wrapped
    int *rotoff = vs + Nz;                                 // [Pv]: s_z(v) * O * Pv, the column's rotation in doubles
    int *zs = rotoff + Pv;                                 // [Pv]: s_z(v), wrapped
    const int NzPv = Nz * Pv;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int ncol = col1;  // this launch does the planes (Y,X) with index Y * Nx + X in [col0, col1)
    const long long plane_nodes = (long long)g.N[1] * g.N[0];

    // z sweep: thread <-> (v, slice qd of the target z cells); (s, A, B) depend on the v node only
    const int nq = min(FUSED_THREADS / Pv, nz);  // slices of z
    const int v = tid % Pv, qd = tid / Pv;
    const bool zact = qd < nq && v < Nv;
    double Azr[ZREG ? O : 1][ZREG ? O : 1], Bzr[ZREG ? O : 1][ZREG ? O : 1];  // ZREG: A, B of this thread's column
    if (tid < Pv || ZREG) {
        // (s, A, B) of the z shift depend on the v node only: once per block, into shared memory (o = 3) or into the
        // registers of every thread of the column
        const int ov = g.o[3];
        const int vv = v < Nv ? v : 0;
        const int l = vv / ov, q = vv - l * ov;
        const double vq = __dadd_rn(g.lo[3], __dmul_rn(__dadd_rn((double)l, bs.xi[ov][q]), g.h[3]));
        int s0;
        double alpha, A0[O][O], B0[O][O];
        shift_of(vq, tau_z, g.h[2], s0, alpha);
        eval_shift<O>(spz, alpha, A0, B0);
        s0 = wrapi(s0, nz);
        if (tid < Pv) {
            zs[tid] = s0;
            rotoff[tid] = tid < Nv ? s0 * O * Pv : 0;
        }
#pragma unroll
        for (int j = 0; j < O; ++j)
#pragma unroll
            for (int m = 0; m < O; ++m) {
                if (ZREG) {
                    Azr[ZREG ? j : 0][ZREG ? m : 0] = A0[j][m];
                    Bzr[ZREG ? j : 0][ZREG ? m : 0] = B0[j][m];
                } else if (tid < Pv) {
                    zAB[(j * O + m) * Pv + tid] = A0[j][m];
                    zAB[(O * O + j * O + m) * Pv + tid] = B0[j][m];
                }
            }
    }
    const int zi0 = (int)((long long)qd * nz / nq), zi1 = (int)((long long)(qd + 1) * nz / nq);

    // staging by bulk copies (TMA), issued by the producer warp, completing on mbarriers: line l of a plane ->
    // tile + l * Pv.  bars: full_L[2], full_H, done (all compute warps are through with a plane)
    uint64_t *bars = reinterpret_cast<uint64_t *>((reinterpret_cast<uintptr_t>(zs + Pv) + 7) & ~(uintptr_t)7);  // 8-byte aligned (Nz, Pv may be odd)
    if (tid == 0) {
        for (int k = 0; k < 3; ++k) mbar_init(&bars[k], 1);
        mbar_init(&bars[3], FUSED_THREADS / 32);
        mbar_init(&bars[4], FUSED_THREADS / 32);  // z,v pair: the H rows of the current plane are no longer read
        mbar_fence_init();
    }
    __syncthreads();
    // z,v pair: the line-wise phase reads line zr of column v from physical row (zr + s_z(v) O) mod Nz.  The lines that
    // touch the H rows (the part of the tile the NEXT plane's late lines go to) are done first; once they are through,
    // the producer fetches those late lines under the rest of the phase instead of after the plane.  order[p] = the
    // lines of a plane of parity p in that order, n_early[p] = how many of them touch H.
    short *order = reinterpret_cast<short *>(bars + 6);
    unsigned char *mark = reinterpret_cast<unsigned char *>(order + 2 * Nz);
    int *n_early = reinterpret_cast<int *>(bars + 5);
    double *rho_part = reinterpret_cast<double *>((reinterpret_cast<uintptr_t>(mark + 2 * Nz) + 7) & ~(uintptr_t)7);  // RHO: [Pv / 32][Nz]
    if (ZFIRST) {
        for (int i = tid; i < 2 * Nz; i += FUSED_BLOCK) mark[i] = 0;
        __syncthreads();
        if (tid < Nv) {
            const int rot = zs[tid] * O;
            for (int r = 0; r < NH; ++r) {  // physical rows of H: NL + r in an even plane's tile, r in an odd plane's
                int l0 = NL + r - rot, l1 = r - rot;
                if (l0 < 0) l0 += Nz;
                if (l1 < 0) l1 += Nz;
                mark[l0] = 1;
                mark[Nz + l1] = 1;
            }
        }
        __syncthreads();
        if (tid < 2) {
            int n = 0;
            for (int zr = 0; zr < Nz; ++zr)
                if (mark[tid * Nz + zr]) order[tid * Nz + n++] = (short)zr;
            n_early[tid] = n;
            for (int zr = 0; zr < Nz; ++zr)
                if (!mark[tid * Nz + zr]) order[tid * Nz + n++] = (short)zr;
        }
        __syncthreads();
    }
    auto compute_sync = [&]() { asm volatile("bar.sync 1, %0;" ::"n"(FUSED_THREADS) : "memory"); };
    const uint32_t line_bytes = (uint32_t)Pv * 8;
    auto issue_lines = [&](int col, double *tl, int first, int count, uint64_t *bar) {  // producer warp only
        if (count <= 0) return;
        const int X = col % g.N[0], Y = col / g.N[0];
        const double *src = fin + Y * g.sY + X * g.sX;
        if (lane == 0) mbar_arrive_expect_tx(bar, (uint32_t)count * line_bytes);
        __syncwarp();
        for (int l = first + lane; l < first + count; l += 32) bulk_g2s(tl + l * Pv, src + l * g.sZ, line_bytes, bar);
    };
    if (warp == FUSED_THREADS / 32) {
        // ---------------- producer warp ------------------------------------------------------------------------
        uint32_t phD = 0, phF = 0;
        int col = col0 + blockIdx.x, par = 0;
        if (col < ncol) issue_lines(col, buf, 0, NL, &bars[0]);  // L lines of the first (even) plane
        if (ZFIRST && col < ncol) issue_lines(col, buf, NL, NH, &bars[2]);  // z,v: and its H lines
        for (bool first = true; col < ncol; col += gridDim.x, par ^= 1, first = false) {
            if (!first) {
                mbar_wait(&bars[3], phD);  // the previous plane is done: (H and) the other L are free
                phD ^= 1;
            }
            double *tile = buf + (par ? NL * Pv : 0);
            const int ncolx = col + (int)gridDim.x;
            // H lines of this plane: [NL,Nz) of an even plane, [0,NH) of an odd one
            if (!ZFIRST) issue_lines(col, tile, par ? 0 : NL, NH, &bars[2]);
            // L lines of the next plane into the other L: [0,NL) of an even plane, [NH,Nz) of an odd one
            if (ncolx < ncol) issue_lines(ncolx, buf + (par ? 0 : NL * Pv), par ? 0 : NH, NL, &bars[par ^ 1]);
            if (ZFIRST && NH > 0 && ncolx < ncol) {
                // z,v: the H lines of the NEXT plane as soon as this plane's line-wise phase is through with the H rows
                mbar_wait(&bars[4], phF);
                issue_lines(ncolx, buf + (par ? 0 : NL * Pv), par ? NL : 0, NH, &bars[2]);
            }
            phF ^= 1;
        }
        return;
    }

    // z,v pair, line-wise phase: byte offset inside the plane tile of row 0 of this lane's columns after the in-place z
    // sweep (column v ends up rotated by s_z(v) cells), for the lane's own source cell (left source of its target)
    // and for the next cell (right source); the columns of a cell rotate independently (s_z depends on the v NODE)
    const int msw = (O == 2) ? ((lane >> 3) & 1) : 0;
    uint32_t off0[CPL][O], off1[CPL][O];
#pragma unroll
    for (int k = 0; k < CPL; ++k)
#pragma unroll
        for (int m = 0; m < O; ++m) {
            const int cell = lane + 32 * k;
            const int c0 = (ZFIRST && cell < nv) ? cell : 0;
            const int c1 = (c0 + 1 == nv) ? 0 : c0 + 1;
            // o = 2: a lane's cell is two adjacent columns, so one 8-byte load per lane at a fixed DOF m strides by 16
            // bytes and the 16 lanes of a half warp cover only half of the banks (2-way conflict: 36 % of the kernel's
            // shared-memory wavefronts).  Lanes 8-15 and 24-31 therefore take the DOFs in the opposite order: slot m of
            // such a lane holds DOF m ^ 1 until two selects put the pair back in order (the sums keep their order of
            // operations: bit-identical to the separate sweeps), and a half warp reads 16 distinct columns modulo 16.
            const int md = m ^ msw;
            off0[k][m] = ZFIRST ? (uint32_t)(rotoff[c0 * O + md] + c0 * O + md) * 8u : 0u;
            off1[k][m] = ZFIRST ? (uint32_t)(rotoff[c1 * O + md] + c1 * O + md) * 8u : 0u;
        }
    double ez_next = 0.0;
    int col = col0 + blockIdx.x, par = 0;
    uint32_t phL[2] = {0, 0}, phH = 0;
    if (!ZONLY && col < ncol && tid < Nz) ez_next = __ldg(Ez + tid * plane_nodes + col);
    // RHO: the previous plane's partial sums (one per warp of a z slice, written in its z sweep) -> rho, in a fixed order
    auto flush_rho = [&](int pcol) {
        if (tid < Nz) {
            double sum = 0.0;
            for (int q = 0; q < Pv / 32; ++q) sum += rho_part[q * Nz + tid];
            rho[tid * plane_nodes + pcol] = g.h[3] * sum;
        }
    };
    int prev_col = -1;
    for (; col < ncol; col += gridDim.x, par ^= 1) {
        double *tile = buf + (par ? NL * Pv : 0);
        const int ncolx = col + (int)gridDim.x;
        const double ez_cur = ez_next;
        if (RHO && prev_col >= 0) flush_rho(prev_col);
        prev_col = col;
        if (!ZONLY && ncolx < ncol && tid < Nz) ez_next = __ldg(Ez + tid * plane_nodes + ncolx);
        // ---- per line the (s, A, B) of its v shift (under the copies) ------------------------------------------
        if (!ZONLY && tid < Nz) {
            int s;
            double alpha, A[O][O], B[O][O];
            shift_of(ez_cur, tau_v, g.h[3], s, alpha);
            eval_shift<O>(spv, alpha, A, B);
            vs[tid] = wrapi(s, nv);
#pragma unroll
            for (int j = 0; j < O; ++j)
#pragma unroll
                for (int m = 0; m < O; ++m) {
                    vAB[(tid * 2) * O * O + j * O + m] = A[j][m];
                    vAB[(tid * 2 + 1) * O * O + j * O + m] = B[j][m];
                }
        }
        if (NL > 0) {
            mbar_wait(&bars[par], phL[par]);
            phL[par] ^= 1;
        }
        if ((ZFIRST || ZONLY) && NH > 0) {  // the z sweep needs every line; the v sweep (VZ) starts on the L lines
            mbar_wait(&bars[2], phH);
            phH ^= 1;
        }
        compute_sync();
        const int X = col % g.N[0], Y = col / g.N[0];
        double *dst = fout + Y * g.sY + X * g.sX;

        if (ZFIRST) {
            // ---- phase A: z sweep in place; the result of target cell i lands on slot (i + s) mod nz ------
            int c = 0;
            double up[O], last[O], Az[O][O], Bz[O][O];
            if (zact) {
                const int sz = zs[v];
#pragma unroll
                for (int j = 0; j < O; ++j)
#pragma unroll
                    for (int m = 0; m < O; ++m) {
                        Az[j][m] = ZREG ? Azr[ZREG ? j : 0][ZREG ? m : 0] : zAB[(j * O + m) * Pv + v];
                        Bz[j][m] = ZREG ? Bzr[ZREG ? j : 0][ZREG ? m : 0] : zAB[(O * O + j * O + m) * Pv + v];
                    }
                c = zi0 + sz;
                if (c >= nz) c -= nz;
                int cl = zi1 + sz;
                if (cl >= nz) cl -= nz;
#pragma unroll
                for (int m = 0; m < O; ++m) {
                    up[m] = tile[(size_t)(c * O + m) * Pv + v];
                    last[m] = tile[(size_t)(cl * O + m) * Pv + v];  // first slot of the next slice: it is overwritten
                }
            }
            compute_sync();
            if (zact) {
                // running offset of cell c's first row in column v; it wraps at the end of the plane
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
                        tile[off + j * Pv] = acc;
                    }
#pragma unroll
                    for (int m = 0; m < O; ++m) up[m] = un[m];
                };
#pragma unroll 2
                for (int i = zi0; i + 1 < zi1; ++i) {
                    int offn = off + cstep;
                    if (offn >= NzPv) offn -= NzPv;
                    double un[O];
#pragma unroll
                    for (int m = 0; m < O; ++m) un[m] = tile[offn + m * Pv];
                    step(un);
                    off = offn;
                }
                step(last);  // the last target of the slice: its right source cell was read before the sweep
            }
            compute_sync();
            // ---- phase B: v sweep of every line, to global memory.  warp <-> line, lane <-> SOURCE cell c0 of the
            //      target cell (c0 - s): its two source cells c0, c0 + 1 are read straight from the rotated columns
            //      (explicit 32-bit shared addresses; the wrap of a rotated column is one unsigned min), no shuffles,
            //      so lanes beyond nv simply skip ---------------------------------------------------------------------
            const uint32_t tile_b = smem_u32(tile), vab_b = smem_u32(vAB), vs_b = smem_u32(vs);
            const uint32_t plane_b = (uint32_t)NzPv * 8u, row_b = (uint32_t)Pv * 8u;
            const uint32_t ord_b = smem_u32(order + par * Nz);
            const int ne = n_early[par];
            bool told = false;
#pragma unroll 1
            for (int idx = warp; idx < Nz; idx += FUSED_THREADS / 32) {
                if (!told && idx >= ne) {  // this warp has read its last line that touches the H rows
                    told = true;
                    fence_proxy_async();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&bars[4]);
                }
                const int zr = lds_s16(ord_b + 2u * idx);
                const int s = lds_s32(vs_b + 4u * zr);
                double A[O][O], B[O][O];
                {
                    double ab[2 * O * O];
                    const uint32_t at = vab_b + (uint32_t)zr * (2 * O * O * 8);
#pragma unroll
                    for (int e = 0; e < O * O; ++e) {
                        const double2 t = lds_v2f64(at + 16u * e);
                        ab[2 * e] = t.x;
                        ab[2 * e + 1] = t.y;
                    }
#pragma unroll
                    for (int j = 0; j < O; ++j)
#pragma unroll
                        for (int m = 0; m < O; ++m) {
                            A[j][m] = ab[j * O + m];
                            B[j][m] = ab[O * O + j * O + m];
                        }
                }
                double *w = dst + zr * g.sZ;
                const uint32_t zb = (uint32_t)zr * row_b;
#pragma unroll
                for (int k = 0; k < CPL; ++k) {
                    const int cell = lane + 32 * k;
                    if (FULLV || cell < nv) {
                        double u0[O], u1[O];
#pragma unroll
                        for (int m = 0; m < O; ++m) {
                            uint32_t t0 = off0[k][m] + zb, t1 = off1[k][m] + zb;
                            t0 = min(t0, t0 - plane_b);  // unsigned: subtracts the plane size exactly when t >= it
                            t1 = min(t1, t1 - plane_b);
                            u0[m] = lds_f64(tile_b + t0);
                            u1[m] = lds_f64(tile_b + t1);
                        }
                        if (O == 2 && msw) {
                            double t = u0[0]; u0[0] = u0[O - 1]; u0[O - 1] = t;
                            t = u1[0]; u1[0] = u1[O - 1]; u1[O - 1] = t;
                        }
                        int c = cell - s;  // the target whose left source cell this is
                        if (c < 0) c += nv;
                        double r[O];
#pragma unroll
                        for (int j = 0; j < O; ++j) {
                            double acc = 0.0;
#pragma unroll
                            for (int m = 0; m < O; ++m) acc = fma(A[j][m], u0[m], acc);
#pragma unroll
                            for (int m = 0; m < O; ++m) acc = fma(B[j][m], u1[m], acc);
                            r[j] = acc;
                        }
                        if (O == 2) {
                            __stcs(reinterpret_cast<double2 *>(w + 2 * c), make_double2(r[0], r[O - 1]));
                        } else {
#pragma unroll
                            for (int j = 0; j < O; ++j) __stcs(w + c * O + j, r[j]);
                        }
                    }
                }
            }
            if (!told) {
                fence_proxy_async();
                __syncwarp();
                if (lane == 0) mbar_arrive(&bars[4]);
            }
        } else {
            // ---- phase A: v sweep in place, warp <-> line; first the L lines (fetched one plane ahead), then,
            //      once they have arrived, the H lines ---------------------------------------------------------
#pragma unroll 1
            for (int pass = 0; pass < (ZONLY ? 0 : 2); ++pass) {
            const int cnt = pass ? NH : NL;
            const int base = pass ? (par ? 0 : NL) : (par ? NH : 0);
            if (pass && NH > 0) {
                mbar_wait(&bars[2], phH);
                phH ^= 1;
            }
#pragma unroll 1
            for (int k = warp; k < cnt; k += FUSED_THREADS / 32) {
                const int zr = base + k;
                const int s = vs[zr];
                double A[O][O], B[O][O];
#pragma unroll
                for (int j = 0; j < O; ++j)
#pragma unroll
                    for (int m = 0; m < O; ++m) {
                        A[j][m] = vAB[(zr * 2) * O * O + j * O + m];
                        B[j][m] = vAB[(zr * 2 + 1) * O * O + j * O + m];
                    }
                double *u = tile + (size_t)zr * Pv;
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
                            *reinterpret_cast<double2 *>(u + 2 * cell) = make_double2(r[0], r[O - 1]);
                        } else {
#pragma unroll
                            for (int j = 0; j < O; ++j) u[cell * O + j] = r[j];
                        }
                    }
                }
            }
            }
            compute_sync();
            // ---- phase B: z sweep, thread <-> (v, slice of z), to global memory -------------------------------
            if (zact) {
                double Az[O][O], Bz[O][O];
#pragma unroll
                for (int j = 0; j < O; ++j)
#pragma unroll
                    for (int m = 0; m < O; ++m) {
                        Az[j][m] = ZREG ? Azr[ZREG ? j : 0][ZREG ? m : 0] : zAB[(j * O + m) * Pv + v];
                        Bz[j][m] = ZREG ? Bzr[ZREG ? j : 0][ZREG ? m : 0] : zAB[(O * O + j * O + m) * Pv + v];
                    }
                int c = zi0 + zs[v];
                if (c >= nz) c -= nz;
                const int cstep = O * Pv;
                int off = c * cstep + v;
                double up[O];
#pragma unroll
                for (int m = 0; m < O; ++m) up[m] = tile[off + m * Pv];
                double *w = dst + v + (long long)(zi0 * O) * g.sZ;
                if constexpr (RHO && O <= 2) {
                    // the same sweep in batches of 8 rows (8 / O cells); the weighted results of a batch are summed over the
                    // warp's 32 v nodes by a butterfly that halves the values a lane holds at every exchange (9 exchanges
                    // per 8 rows), lane l < 8 ending with the sum of row l of the batch
                    constexpr int U = 8 / O;
                    const double wv = bs.w[O][v % O];
                    double *part = rho_part + (v >> 5) * Nz;
#pragma unroll 1
                    for (int i = zi0; i < zi1; i += U) {
                        double x[8];
#pragma unroll
                        for (int u = 0; u < U; ++u) {
                            if (i + u < zi1) {
                                off += cstep;
                                if (off >= NzPv) off -= NzPv;
                                double un[O];
#pragma unroll
                                for (int m = 0; m < O; ++m) un[m] = tile[off + m * Pv];
#pragma unroll
                                for (int j = 0; j < O; ++j) {
                                    double acc = 0.0;
#pragma unroll
                                    for (int m = 0; m < O; ++m) acc = fma(Az[j][m], up[m], acc);
#pragma unroll
                                    for (int m = 0; m < O; ++m) acc = fma(Bz[j][m], un[m], acc);
                                    __stcs(w, acc);
                                    w += g.sZ;
                                    x[u * O + j] = wv * acc;
                                }
#pragma unroll
                                for (int m = 0; m < O; ++m) up[m] = un[m];
                            } else {
#pragma unroll
                                for (int j = 0; j < O; ++j) x[u * O + j] = 0.0;
                            }
                        }
#pragma unroll
                        for (int d = 4; d >= 1; d >>= 1) {
                            const bool hi = (lane & d) != 0;
#pragma unroll
                            for (int k = 0; k < d; ++k) {
                                const double send = hi ? x[k] : x[k + d], keep = hi ? x[k + d] : x[k];
                                x[k] = keep + __shfl_xor_sync(0xffffffffu, send, d);
                            }
                        }
                        x[0] += __shfl_xor_sync(0xffffffffu, x[0], 8);
                        x[0] += __shfl_xor_sync(0xffffffffu, x[0], 16);
                        if (lane < 8 && i + lane / O < zi1) part[(i + lane / O) * O + lane % O] = x[0];
                    }
                } else {
#pragma unroll 2
                for (int i = zi0; i < zi1; ++i) {
                    off += cstep;
                    if (off >= NzPv) off -= NzPv;
                    double un[O];
#pragma unroll
                    for (int m = 0; m < O; ++m) un[m] = tile[off + m * Pv];
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
        }
        fence_proxy_async();  // generic writes before the next bulk copies
        __syncwarp();
        if (lane == 0) mbar_arrive(&bars[3]);
        compute_sync();  // the per-line tables are free for the next plane
    }
    if (RHO && prev_col >= 0) flush_rho(prev_col);
}

}  // namespace

// Whether the pair can run in this kernel (see launch_fused_sweeps); *NL_out = lines fetched one plane ahead.
static bool fused_pair_fits(const sldg_ctx *c, bool z_first, bool z_only, int *NL_out, size_t *smem_out, bool rho = false)
{
    if (z_only) z_first = false;
    const GridDev &g = c->g;
    const int O = g.o[2];
    if (!z_only && g.o[3] != O) return false;
    if (g.Pv > FUSED_THREADS || (!z_only && g.n[3] > 32 * FUSED_MAXCPL)) return false;
    const int Nz = g.N[2];
    // the per-line tables of the v shift (vs, vAB, the E_z prefetch) are filled by thread <-> line
    if (!z_only && Nz > FUSED_THREADS) return false;
    // the charge density from the z sweep of the v,z pair (RHO): o = 2, whole warps of v nodes, no padding of the v lines
    if (rho && (z_first || z_only || O != 2 || g.Pv % 32 != 0 || g.N[3] != g.Pv)) return false;
    const size_t tables = fused_table_bytes(Nz, g.Pv, O, rho), row = (size_t)g.Pv * 8;
    static const int budget_kb = getenv("SLDG_FUSED_KB") ? atoi(getenv("SLDG_FUSED_KB")) : 227;  // KB of dynamic shared memory the kernel may take (sm_100: 227 per block)
    const size_t budget = (size_t)budget_kb * 1024;
    if (tables + row * Nz > budget) return false;
    long long NLl = (long long)((budget - tables) / row) - Nz;  // spare lines = lines fetched one plane ahead
    const int NL = (int)(NLl > Nz ? Nz : (NLl < 0 ? 0 : NLl));
    // z first: the z sweep cannot start before the whole plane is there, so the lines that do not fit beside the
    // current plane (NH = Nz - NL, fetched only when it is done) are fully exposed; measured at 144 x 144 (o = 3,
    // NL = 0.28 Nz) the pair is then slower than the two separate kernels.  v first hides them under its L lines.
    if ((z_first || z_only) && 2 * NL < Nz) return false;
    *NL_out = NL;
    *smem_out = tables + row * (size_t)(2 * NL + (Nz - NL));
    return true;
}

bool fused_sweeps_supported(const sldg_ctx *c, bool z_first, bool rho)
{
    int NL;
    size_t smem;
    return fused_pair_fits(c, z_first, false, &NL, &smem, rho);
}

// The pair (z then v, or v then z) in one pass over the planes (Y,X) with index Y * Nx + X in [col0, col1) (col1 < 0:
// all from col0 on); returns cudaErrorNotSupported when the (z,v) plane does not fit (the caller then runs the two
// separate kernels).
// rho != nullptr (v,z pair only): the kernel also writes the charge density of its planes, rho[Nz][Ny][Nx].
cudaError_t launch_fused_sweeps(sldg_ctx *c, const double *fin, double *fout, double tau_z, double tau_v, bool z_first,
                                bool z_only, int col0, int col1, double *rho)
{
    if (z_only) z_first = false;
    const GridDev &g = c->g;
    const int O = g.o[2];
    int NL;
    size_t smem;
    if (!fused_pair_fits(c, z_first, z_only, &NL, &smem, rho != nullptr)) return cudaErrorNotSupported;
    const bool cpl2 = g.n[3] <= 64;
    const bool fullv = g.n[3] == (cpl2 ? 64 : 128);  // every lane of the line-wise phase has all its cells
    if (col1 < 0) col1 = g.N[0] * g.N[1];
    const int ncol = col1 - col0;
    if (ncol <= 0) return cudaSuccess;
    const int grid = ncol < c->sm_count ? ncol : c->sm_count;
    if (rho) {
        auto kern = cpl2 ? fused_sweep_kernel<2, 2, false, false, false, true> : fused_sweep_kernel<2, 4, false, false, false, true>;
        cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        kern<<<grid, FUSED_BLOCK, smem, c->stream>>>(fin, fout, c->Ez, g, c->sp_z, c->sp_v, c->basis, tau_z, tau_v, NL, col0, col1,
                                                       rho);
        c->launches++;
        return cudaGetLastError();
    }
#define LAUNCH_F(OO)                                                                                              \
    do {                                                                                                          \
        auto kern = z_only ? fused_sweep_kernel<OO, 2, false, true, false>                                        \
                  : z_first ? (cpl2 ? (fullv ? fused_sweep_kernel<OO, 2, true, false, true>                       \
                                             : fused_sweep_kernel<OO, 2, true, false, false>)                     \
                                    : (fullv ? fused_sweep_kernel<OO, 4, true, false, true>                       \
                                             : fused_sweep_kernel<OO, 4, true, false, false>))                    \
                            : (cpl2 ? fused_sweep_kernel<OO, 2, false, false, false>                              \
                                    : fused_sweep_kernel<OO, 4, false, false, false>);                            \
        cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);                       \
        kern<<<grid, FUSED_BLOCK, smem, c->stream>>>(fin, fout, c->Ez, g, c->sp_z, c->sp_v, c->basis, tau_z,    \
                                                       tau_v, NL, col0, col1, nullptr);                           \
    } while (0)
    if (O == 1) LAUNCH_F(1); else if (O == 2) LAUNCH_F(2); else LAUNCH_F(3);
#undef LAUNCH_F
    c->launches++;
    return cudaGetLastError();
}
