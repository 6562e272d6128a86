// sldg_xy_apply.cu -- eq. (17):  out[ij,m] = sum_{rs} sum_k (C^{ij,m}_{rs,k} / W_m) in[rs,k]
// for every (z, v), with the weights the geometry kernel left in the workspace (Algorithm 3, PAPER.md:287-293:
// coefficients once per z node, reused for every v).
//
// Thread mapping everywhere: lane <-> v (contiguous in memory), so the weights of a target cell are
// warp-uniform, the control flow over the (up to 3x3) non-empty source cells is warp-uniform, and empty
// source cells cost nothing.
//
//   xy_apply_stream_kernel (o = 2 and 3; the numbers below are o = 2): a streaming stencil in SOURCE-row order.
//     A block owns a strip of TX = 8 target cells in x (o = 3: 4), a segment of up to 128 target rows in y, one z node and one chunk
//     of <= 128 v values.  The prologue reads the segment's headers and takes the bounds of the anchors;
//     they fix a static schedule: target row j uses source rows j+aymin .. j+aymin+2 and the x window
//     [axmin, TX-1+axmax].  A producer warp streams the source rows (each row = the window's lines, all v
//     of the chunk, 40 KB) and each target row's packed weight blocks into shared-memory rings with
//     cp.async.bulk copies completing on mbarriers.  Eight consumer warps (one per target cell, four v values
//     per lane) wait for ONE source row at a time, add its contributions to the (up to three) target rows that
//     use it -- their partial sums live in registers -- release the row at once, and store a target row
//     when its last source row has been applied.  Because a source row is never held while others arrive,
//     all but one ring slot are in flight.  Every input line is fetched once per strip (x halo:
//     window/TX = 10/8), weights once.
//   xy_stageable_kernel: decides per block (strip, segment, z node) whether its anchors allow that schedule.
//   xy_apply_direct_kernel (any o): warp <-> target cell, inputs through L1; does the blocks that cannot stream.
#include <stdlib.h>

#include "sldg_async.cuh"
#include "sldg_internal.cuh"

__device__ __forceinline__ int wrap_idx(int i, int n)
{
    int r = i % n;
    return r < 0 ? r + n : r;
}

// One source cell's contribution for NP v pairs per lane (pair p at v = 64 p + 2 lane): o^2 inputs (k), o^4
// weights W[k][m].  The weights are warp-uniform shared-memory broadcasts.
template <int O, int NP>
__device__ __forceinline__ void fma_block(double (&acc)[O * O][2 * NP], const double *__restrict__ src,
                                          size_t kq_stride, int VL, const double *__restrict__ Wp)
{
    constexpr int O2 = O * O;
    // all input loads of the block first (o^2 NP in flight), weights k by k (broadcast loads, short latency)
    double2 in[O2][NP];
#pragma unroll
    for (int k = 0; k < O2; ++k)
#pragma unroll
        for (int p = 0; p < NP; ++p)
            in[k][p] = *reinterpret_cast<const double2 *>(src + (k / O) * kq_stride + (k % O) * VL + 64 * p);
#pragma unroll
    for (int k = 0; k < O2; ++k) {
        double w[O2];
        if (O == 2) {
            const double2 w01 = *reinterpret_cast<const double2 *>(Wp + k * 4);
            const double2 w23 = *reinterpret_cast<const double2 *>(Wp + k * 4 + 2);
            w[0] = w01.x; w[1] = w01.y; w[2] = w23.x; w[O2 - 1] = w23.y;
        } else {
#pragma unroll
            for (int m = 0; m < O2; ++m) w[m] = Wp[k * O2 + m];
        }
#pragma unroll
        for (int m = 0; m < O2; ++m)
#pragma unroll
            for (int p = 0; p < NP; ++p) {
                acc[m][2 * p] = fma(w[m], in[k][p].x, acc[m][2 * p]);
                acc[m][2 * p + 1] = fma(w[m], in[k][p].y, acc[m][2 * p + 1]);
            }
    }
}

// Per order: target cells per strip, weight stages (target rows), weight blocks per stage (TX cells x <= 9 blocks),
// doubles per weight block in memory (o = 3: 81 padded to 82, bulk copies move multiples of 16 bytes), ring bytes.
template <int O> struct StreamCfg;
#ifndef SLDG_RING2_KB
#define SLDG_RING2_KB 160
#endif
#ifndef SLDG_NW2
#define SLDG_NW2 5
#endif
template <> struct StreamCfg<2> {
    static constexpr int TX = 8, NW = SLDG_NW2, WROW = 72, WB = 16;
    static constexpr size_t RING = SLDG_RING2_KB * 1024;
};
template <> struct StreamCfg<3> {
    static constexpr int TX = 4, NW = 4, WROW = 36, WB = 82;
    static constexpr size_t RING = 126 * 1024;
};
constexpr int STREAM_LMAX = 128;    // target rows per segment
constexpr int STREAM_VMAX = 128;    // v values per chunk
// consumer warps: VSPLIT per target cell of the strip (VSPLIT = 1: one warp, 4 v values per lane; 2: two warps, one
// half of the v chunk each, 2 v values per lane); + 1 producer warp
constexpr int STREAM_NRMAX = 8;     // ring slots (barrier arrays)
constexpr int STREAM_NACC = 3;      // source rows per target row handled by the register accumulators
template <int O> __host__ __device__ constexpr size_t stream_wring_bytes() { return (size_t)StreamCfg<O>::NW * StreamCfg<O>::WROW * StreamCfg<O>::WB * 8; }
template <int O> __host__ __device__ constexpr size_t stream_hdr_bytes() { return (size_t)STREAM_LMAX * StreamCfg<O>::TX * 16; }
template <int O> __host__ __device__ constexpr size_t stream_smem_bytes() { return StreamCfg<O>::RING + stream_wring_bytes<O>() + stream_hdr_bytes<O>() + 512; }
static int stream_tx(int O) { return O == 3 ? StreamCfg<3>::TX : StreamCfg<2>::TX; }

// Whether the block (strip, segment, z node) of the streaming kernel can stage its rows: the x window of the
// strip over the whole segment must leave at least two ring slots, and a target row may use at most NACC source rows.
// One criterion, evaluated by the scan kernel below and relied upon by the streaming kernel.
__device__ __forceinline__ bool stream_block_stageable(int axmin, int axmax, int aymin, int aymax, int VL, int O,
                                                       int TX, size_t ring_bytes)
{
    const int RW = TX + axmax - axmin;
    const size_t stage_bytes = (size_t)O * O * RW * VL * 8;
    return ring_bytes / stage_bytes >= 2 && aymax - aymin + 1 <= STREAM_NACC;
}

// grid (strips * segments, Nz): bounds of the anchors of one streaming block -> stage_ok[z][block]
__global__ void __launch_bounds__(128) xy_stageable_kernel(const int4 *__restrict__ hdrg, GridDev g, int L, int VL,
                                                           int TX, size_t ring_bytes,
                                                           int32_t *__restrict__ stage_ok, int32_t *err)
{
    __shared__ int bnd[4];
    const int nx = g.n[0], ny = g.n[1];
    const int strips = (nx + TX - 1) / TX;
    const int strip = blockIdx.x % strips, seg = blockIdx.x / strips;
    const int i0 = strip * TX, j0 = seg * L;
    const int rows = min(L, ny - j0);
    const long long zc = (long long)blockIdx.y * nx * ny;
    if (threadIdx.x == 0) { bnd[0] = 1 << 30; bnd[1] = -(1 << 30); bnd[2] = 1 << 30; bnd[3] = -(1 << 30); }
    __syncthreads();
    int lo_x = 1 << 30, hi_x = -(1 << 30), lo_y = 1 << 30, hi_y = -(1 << 30);
    for (int c = threadIdx.x; c < rows * TX; c += blockDim.x) {
        const int jr = c / TX, ci = c - jr * TX;
        if (i0 + ci >= nx) continue;
        const int4 h = __ldcg(hdrg + zc + (long long)(j0 + jr) * nx + i0 + ci);
        if (!h.z) continue;
        const int wx = (h.z & 0x124) ? 3 : ((h.z & 0x092) ? 2 : 1);
        const int wy = (h.z & 0x1c0) ? 3 : ((h.z & 0x038) ? 2 : 1);
        lo_x = min(lo_x, h.x); hi_x = max(hi_x, h.x + wx - 1);
        lo_y = min(lo_y, h.y); hi_y = max(hi_y, h.y + wy - 1);
    }
    atomicMin(&bnd[0], lo_x); atomicMax(&bnd[1], hi_x); atomicMin(&bnd[2], lo_y); atomicMax(&bnd[3], hi_y);
    __syncthreads();
    if (threadIdx.x == 0) {
        const bool ok = bnd[1] < bnd[0] || stream_block_stageable(bnd[0], bnd[1], bnd[2], bnd[3], VL, g.o[0], TX, ring_bytes);
        stage_ok[blockIdx.y * gridDim.x + blockIdx.x] = ok ? 1 : 0;
        if (!ok) atomicAdd(err + 1, 1);  // diagnostic counter 0 (sldg_debug_counter)
    }
}

template <int O, int VSPLIT>
__global__ void __launch_bounds__(32 * (StreamCfg<O>::TX * VSPLIT + 1), 1) xy_apply_stream_kernel(
    const double *__restrict__ fin, double *__restrict__ fout, const int4 *__restrict__ hdrg,
    const double *__restrict__ W, GridDev g, int L, const int32_t *__restrict__ stage_ok, int vend)
{
    if (!stage_ok[blockIdx.z * gridDim.x + blockIdx.x]) return;  // the direct kernel handles this block
    using Cfg = StreamCfg<O>;
    constexpr int TX = Cfg::TX, NW = Cfg::NW, NACC = STREAM_NACC, O2 = O * O, WB = Cfg::WB, STREAM_WROW = Cfg::WROW;
    constexpr int STREAM_CWARPS = TX * VSPLIT, STREAM_THREADS = 32 * (STREAM_CWARPS + 1), NP = 2 / VSPLIT;
    constexpr size_t STREAM_RING_BYTES = Cfg::RING, STREAM_WRING_BYTES = stream_wring_bytes<O>(),
                     STREAM_HDR_BYTES = stream_hdr_bytes<O>();
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double *ring = reinterpret_cast<double *>(smem_raw);                                  // [NR][O kq][O*RW][VL]
    double *wring = reinterpret_cast<double *>(smem_raw + STREAM_RING_BYTES);             // [NW][WROW][WB]
    int4 *hdr = reinterpret_cast<int4 *>(smem_raw + STREAM_RING_BYTES + STREAM_WRING_BYTES);  // [L][TX]
    int *bnd = reinterpret_cast<int *>(smem_raw + STREAM_RING_BYTES + STREAM_WRING_BYTES + STREAM_HDR_BYTES);
    uint64_t *full = reinterpret_cast<uint64_t *>(bnd + 16);
    uint64_t *empty = full + STREAM_NRMAX, *wfull = empty + STREAM_NRMAX, *wempty = wfull + NW;

    const int nx = g.n[0], ny = g.n[1];
    const int strips = (nx + TX - 1) / TX;
    const int strip = blockIdx.x % strips, seg = blockIdx.x / strips;
    const int i0 = strip * TX, j0 = seg * L;
    const int rows = min(L, ny - j0);
    const int z = blockIdx.z;
    const int v0 = blockIdx.y * STREAM_VMAX;
    const int VL = min(STREAM_VMAX, vend - v0);  // multiple of 16; this kernel covers the v values [0, vend)
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const long long ncell = (long long)nx * ny;
    const long long zc = (long long)z * ncell;

    // ---- prologue: headers of the segment, anchor bounds, per-row packing of the weight blocks -----------
    if (tid == 0) {
        bnd[0] = 1 << 30; bnd[1] = -(1 << 30); bnd[2] = 1 << 30; bnd[3] = -(1 << 30); bnd[4] = 0;
        for (int s = 0; s < STREAM_NRMAX; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], STREAM_CWARPS); }
        for (int s = 0; s < NW; ++s) { mbar_init(&wfull[s], 1); mbar_init(&wempty[s], STREAM_CWARPS); }
        mbar_fence_init();
    }
    __syncthreads();
    for (int c = tid; c < rows * TX; c += STREAM_THREADS) {
        const int jr = c / TX, ci = c % TX;
        int4 h = make_int4(0, 0, 0, 0);
        if (i0 + ci < nx) h = __ldcg(hdrg + zc + (long long)(j0 + jr) * nx + i0 + ci);
        hdr[c] = h;
        if (h.z) {
            const int wx = (h.z & 0x124) ? 3 : ((h.z & 0x092) ? 2 : 1);
            const int wy = (h.z & 0x1c0) ? 3 : ((h.z & 0x038) ? 2 : 1);
            atomicMin(&bnd[0], h.x);
            atomicMax(&bnd[1], h.x + wx - 1);
            atomicMin(&bnd[2], h.y);
            atomicMax(&bnd[3], h.y + wy - 1);
        }
    }
    __syncthreads();
    // per target row: exclusive prefix of the block counts -> hdr.w = offset of the cell's first block
    for (int jr = tid; jr < rows; jr += STREAM_THREADS) {
        int off = 0;
#pragma unroll
        for (int ci = 0; ci < TX; ++ci) {
            const int n = hdr[jr * TX + ci].w;
            hdr[jr * TX + ci].w = off;
            off += n;
        }
        atomicMax(&bnd[4], off);
    }
    __syncthreads();
    if (bnd[4] == 0) return;                 // nothing to do (no valid cell)
    const int axmin = bnd[0], aymin = bnd[2];
    const int RW = TX + bnd[1] - axmin;      // window width in cells
    const int S = bnd[3] - aymin + 1;        // source rows per target row
    const size_t stage_doubles = (size_t)O * O * RW * VL;
    int NR = (int)(STREAM_RING_BYTES / (stage_doubles * 8));
    NR = NR > STREAM_NRMAX ? STREAM_NRMAX : NR;
    const double *fz = fin + z * g.sZ + v0;
    double *oz = fout + z * g.sZ + v0;

    // Headers -> per-target-row descriptors, in place.  A target row jr is touched by the source rows
    // jr + d, d = 0..2 (relative to aymin); descriptor d = {bits 0-2: mask of the 3 source cells of that row,
    // bits 3-11: index of its first weight block inside the row's weight stage, bits 12..: first source cell's
    // position in the x window}; .w = {bits 0-7: offset of the cell's blocks in the stage, bits 8-16: slot mask}.
    for (int c = tid; c < rows * TX; c += STREAM_THREADS) {
        const int4 h = hdr[c];
        int dsc[3] = {0, 0, 0};
        const int bx = (c % TX) + h.x - axmin;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const int dy = d - (h.y - aymin);
            if (h.z && dy >= 0 && dy <= 2) {
                const int mrow = (h.z >> (3 * dy)) & 7;
                if (mrow) dsc[d] = mrow | ((h.w + __popc(h.z & ((1 << (3 * dy)) - 1))) << 3) | (bx << 12);
            }
        }
        hdr[c] = make_int4(dsc[0], dsc[1], dsc[2], h.w | (h.z << 8));
    }
    __syncthreads();

    const int nsrc = rows + S - 1;  // source rows y' = 0 .. nsrc-1, Y = j0 + aymin + y'

    if (warp == STREAM_CWARPS) {
        // ---------------- producer warp -------------------------------------------------------------------
        const int wx0 = wrap_idx(i0 + axmin, nx);       // first cell of the x window (wrapped)
        const int n1 = min(RW, nx - wx0);               // cells before the periodic seam
        const bool runs = (g.sX == (long long)VL) && RW <= nx;  // window lines contiguous in memory (z,y,x order)
        const uint32_t row_bytes = (uint32_t)(stage_doubles * 8);
        int st = 0, ph = 1, ws = 0, wph = 1;  // ring slot / parity of the `empty` barriers to wait for
        for (int k = 0; k < nsrc; ++k) {
            if (k >= NR) mbar_wait(&empty[st], ph);
            if (lane == 0) mbar_arrive_expect_tx(&full[st], row_bytes);
            __syncwarp();
            const int sY = wrap_idx(j0 + aymin + k, ny);
            double *dst = ring + (size_t)st * stage_doubles;
            if (runs) {
                // per kq: one copy up to the seam, one after it
                if (lane < 2 * O) {
                    const int kq = lane % O, part = lane / O;
                    const int c0 = part ? 0 : wx0, nc = part ? RW - n1 : n1, off = part ? n1 : 0;
                    if (nc > 0)
                        bulk_g2s(dst + ((size_t)kq * O * RW + O * off) * VL,
                                 fz + (long long)(O * sY + kq) * g.sY + (long long)(O * c0) * g.sX,
                                 (uint32_t)(O * nc * VL * 8), &full[st]);
                }
            } else {
                for (int l = lane; l < O * O * RW; l += 32) {
                    const int kq = l / (O * RW), xd = l - kq * O * RW;
                    const int r = (wx0 + xd / O) % nx;  // the window may be wider than the periodic box
                    bulk_g2s(dst + ((size_t)kq * O * RW + xd) * VL,
                             fz + (long long)(O * sY + kq) * g.sY + (long long)(O * r + xd % O) * g.sX,
                             (uint32_t)(VL * 8), &full[st]);
                }
            }
            if (++st == NR) { st = 0; ph ^= 1; }
            // weights of target row k (first used with source row k)
            if (k < rows) {
                if (k >= NW) mbar_wait(&wempty[ws], wph);
                int cnt = 0, off = 0;                     // one packed run of weight blocks per cell
                if (lane < TX) {
                    const int w = hdr[k * TX + lane].w;
                    cnt = __popc(w >> 8);
                    off = w & 0xff;
                }
                int tot = cnt;
#pragma unroll
                for (int o = 1; o < TX; o <<= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
                if (lane == 0) mbar_arrive_expect_tx(&wfull[ws], (uint32_t)(tot * WB * 8));
                __syncwarp();
                if (cnt > 0) {
                    const long long cellid = zc + (long long)(j0 + k) * nx + i0 + lane;
                    bulk_g2s(wring + ((size_t)ws * STREAM_WROW + off) * WB, W + (size_t)cellid * 9 * WB,
                             (uint32_t)(cnt * WB * 8), &wfull[ws]);
                }
                if (++ws == NW) { ws = 0; wph ^= 1; }
            }
        }
        return;
    }

    // ---------------- consumer warps: one per target cell of the strip ---------------------------------------
    // lane <-> the v pairs (2 lane, 2 lane + 1) and/or (64 + 2 lane, 64 + 2 lane + 1): every shared-memory load of a
    // warp is a contiguous 512-byte run.  Lanes whose pair lies beyond VL compute on stale ring contents and
    // never store.
    const int ci = warp / VSPLIT, vbase = (warp % VSPLIT) * 64 + 2 * lane;
    const size_t kq_stride = (size_t)O * RW * VL;
    const bool wlive = VSPLIT == 1 || (warp % VSPLIT) * 64 < VL;  // this warp's half of the chunk holds data
    double acc[NACC][O2][2 * NP];
    int4 dsc[NACC];
#pragma unroll
    for (int a = 0; a < NACC; ++a) {
        dsc[a] = make_int4(0, 0, 0, 0);
#pragma unroll
        for (int m = 0; m < O2; ++m)
#pragma unroll
            for (int e = 0; e < 2 * NP; ++e) acc[a][m][e] = 0.0;
    }
    int st = 0, ph = 0, ws = 0, wph = 0;  // source ring slot / parity, weight stage / parity (of the `full` barriers)
    int wsd = 0;                          // weight stage of the target row that is stored next
    double *orow = oz + (long long)(O * j0) * g.sY + (long long)(O * (i0 + ci)) * g.sX + vbase;

    // one step: source row k; target rows k, k-1, k-2 (accumulator sets are indexed by row mod 3, static
    // because the step loop is unrolled by 3)
    for (int kb = 0; kb < rows + NACC - 1; kb += NACC) {
#pragma unroll
        for (int u = 0; u < NACC; ++u) {
            const int k = kb + u;
            if (k >= rows + NACC - 1) break;
            if (k < rows) {
                // target row k enters: its descriptor and weight stage
                mbar_wait(&wfull[ws], wph);
                dsc[u] = hdr[k * TX + ci];
                const int wb = (ws * STREAM_WROW) << 3;  // block indices become absolute in the weight ring
                dsc[u].x += wb;
                dsc[u].y += wb;
                dsc[u].z += wb;
                if (++ws == NW) { ws = 0; wph ^= 1; }
            }
            if (k < nsrc) {
                mbar_wait(&full[st], ph);
                const double *srow = ring + (size_t)st * stage_doubles + vbase;
#pragma unroll
                for (int d = 0; d < NACC; ++d) {
                    const int set = (u - d + NACC) % NACC;
                    if (k - d < 0 || k - d >= rows) continue;
                    const int desc = d == 0 ? dsc[set].x : (d == 1 ? dsc[set].y : dsc[set].z);
                    if (!(desc & 7) || !wlive) continue;
                    const double *Wp = wring + ((desc >> 3) & 0x1ff) * WB;
                    const double *src = srow + (size_t)(O * (desc >> 12)) * VL;
                    if (O == 2) {
#pragma unroll
                        for (int dx = 0; dx < 3; ++dx) {
                            if ((desc >> dx) & 1) {
                                fma_block<O, NP>(acc[set], src + (size_t)(O * dx) * VL, kq_stride, VL, Wp);
                                Wp += WB;
                            }
                        }
                    } else {
                        // o = 3: one copy of the 162-FMA block per (set, d), or the code outgrows the I-cache
#pragma unroll 1
                        for (int dx = 0; dx < 3; ++dx) {
                            if ((desc >> dx) & 1) {
                                fma_block<O, NP>(acc[set], src + (size_t)(O * dx) * VL, kq_stride, VL, Wp);
                                Wp += WB;
                            }
                        }
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[st]);
                if (++st == NR) { st = 0; ph ^= 1; }
            }
            // target row k - 2 has seen all its source rows
            const int jd = k - (NACC - 1);
            if (jd >= 0 && jd < rows) {
                const int set = (u + 1) % NACC;  // (u - 2 + 3) % 3
                if (dsc[set].w >> 8) {
                    double *o = orow;
#pragma unroll
                    for (int m = 0; m < O2; ++m) {
                        double *om = o + (m / O) * g.sY + (m % O) * g.sX;
#pragma unroll
                        for (int p = 0; p < NP; ++p)
                            if (vbase + 64 * p < VL)
                                __stcs(reinterpret_cast<double2 *>(om + 64 * p),
                                       make_double2(acc[set][m][2 * p], acc[set][m][2 * p + 1]));
                    }
                }
                orow += O * g.sY;
#pragma unroll
                for (int m = 0; m < O2; ++m)
#pragma unroll
                    for (int e = 0; e < 2 * NP; ++e) acc[set][m][e] = 0.0;
                __syncwarp();
                if (lane == 0) mbar_arrive(&wempty[wsd]);
                if (++wsd == NW) wsd = 0;
            }
        }
    }
}

// --------------------------------------------------------------------------------------------------
// direct apply (any o): block = 8 warps, a tile of 8x4 target cells at one z node and one chunk of 32*NV v
// values; warp <-> target cell (4 cells per warp), lane <-> the v values lane + 32 e, e < NV (coalesced 256-byte
// loads).  Per source cell and source node k: NV inputs per lane, then o^2 weights W[k][m] (warp-uniform loads,
// contiguous in m) each feeding NV FMAs -- o^2 NV accumulators per lane, o^2 + NV loads per o^2 NV FMAs.
// Inputs and weights through L1/L2.  At o = 3 the step is bound by the fp64 pipe (2*9*c FMA per DOF).
// --------------------------------------------------------------------------------------------------
// stage_ok != nullptr (filtered): the grid is that of the streaming kernel, a block does the cells of one streaming
// block (strip of stx columns, segment of L rows, z node) if that block is NOT stageable, and nothing otherwise.
// CPW > 1 (a remainder of at most 16 v values): CPW cells per warp, 32 / CPW lanes per cell, the lane's values at
// stride 32 / CPW.
template <int O, int NV, int CPW = 1>
__global__ void __launch_bounds__(256, 2) xy_apply_direct_kernel(const double *__restrict__ fin,
                                                              double *__restrict__ fout,
                                                              const int4 *__restrict__ hdrg,
                                                              const double *__restrict__ W, GridDev g,
                                                              const int32_t *__restrict__ stage_ok, int L, int stx,
                                                              int vbeg, int vend)
{
    constexpr int O2 = O * O, TX = 8, TY = 4;
    const int nx = g.n[0], ny = g.n[1];
    const int z = blockIdx.z;
    // the block's cells: a tile of 8 x 4, or -- filtered -- one whole block of the streaming kernel (strip x segment)
    int ri0, rj0, rw, rh;
    if (stage_ok) {
        if (stage_ok[z * gridDim.x + blockIdx.x]) return;  // streamed
        const int strips = (nx + stx - 1) / stx;
        ri0 = (blockIdx.x % strips) * stx;
        rj0 = (blockIdx.x / strips) * L;
        rw = min(stx, nx - ri0);
        rh = min(L, ny - rj0);
    } else {
        const int tiles_x = (nx + TX - 1) / TX;
        ri0 = (blockIdx.x % tiles_x) * TX;
        rj0 = (blockIdx.x / tiles_x) * TY;
        rw = min(TX, nx - ri0);
        rh = min(TY, ny - rj0);
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    constexpr int LPC = 32 / CPW;  // lanes per cell
    const int v = vbeg + blockIdx.y * LPC * NV + lane % LPC;  // this launch covers [vbeg, vend)
    if (v >= vend) return;
    int nve = 0;  // values of this lane inside the line
#pragma unroll
    for (int e = 0; e < NV; ++e) nve += (v + LPC * e < vend) ? 1 : 0;
    const long long ncell = (long long)nx * ny;
    const double *fz = fin + z * g.sZ + v;
    double *oz = fout + z * g.sZ + v;

    for (int c = CPW * warp + lane / LPC; c < rw * rh; c += 8 * CPW) {
        const int i = ri0 + (c % rw), j = rj0 + (c / rw);
        const long long cellid = (long long)z * ncell + (long long)j * nx + i;
        const int4 h = __ldcg(hdrg + cellid);
        const int ax = wrap_idx(i + h.x, nx);
        const int ay = wrap_idx(j + h.y, ny);
        const int msk = h.z;
        int nb = 0;
        double acc[O2][NV];
#pragma unroll
        for (int m = 0; m < O2; ++m)
#pragma unroll
            for (int e = 0; e < NV; ++e) acc[m][e] = 0.0;
        // the non-empty source cells in ascending slot order (with CPW > 1 the cells of a warp have different masks: the
        // warp runs as many rounds as its fullest cell has blocks, not one per slot that any of them uses)
        int rem = msk;
#pragma unroll 1
        for (int it = 0; it < 9; ++it) {
            int slot = it;
            if (CPW == 1) {
                if (!((msk >> slot) & 1)) continue;
            } else {
                if (!rem) break;
                slot = __ffs(rem) - 1;
                rem &= rem - 1;
            }
            const int r = wrap_idx(ax + slot % 3, nx), s = wrap_idx(ay + slot / 3, ny);  // nx, ny may be < 3
            const double *Wp = W + ((size_t)cellid * 9 + nb++) * sldg_w_block_doubles(O);
#pragma unroll
            for (int kq = 0; kq < O; ++kq)
#pragma unroll
                for (int kp = 0; kp < O; ++kp) {
                    const double *src = fz + (long long)(s * O + kq) * g.sY + (long long)(r * O + kp) * g.sX;
                    double in[NV];
#pragma unroll
                    for (int e = 0; e < NV; ++e) in[e] = e < nve ? __ldg(src + LPC * e) : 0.0;
                    const int k = kp + O * kq;
                    if (O == 1 || (O == 3 && CPW == 1)) {
                        // one cell per warp at o = 3: one weight at a time (NV >= 4 has no registers for more)
#pragma unroll
                        for (int m = 0; m < O2; ++m) {
                            const double w = __ldg(Wp + k * O2 + m);
#pragma unroll
                            for (int e = 0; e < NV; ++e) acc[m][e] = fma(w, in[e], acc[m][e]);
                        }
                    } else {
                        // the o^2 weights W[k][.] as 16-byte loads: blocks start 16-byte aligned (o = 3: 82 doubles per
                        // block, so the pair after the last weight exists); with CPW cells per warp a weight load touches
                        // CPW cache lines, and the L1 wavefronts of the weights bound the short-chunk kernel
                        constexpr int NPAIR = (O2 + 2) / 2;       // pairs that cover o^2 weights from either parity
                        const int b = (k * O2) & ~1, odd = (k * O2) & 1;
                        double2 t[NPAIR];
#pragma unroll
                        for (int q = 0; q < NPAIR; ++q)
                            if (2 * q < O2 + odd) t[q] = __ldg(reinterpret_cast<const double2 *>(Wp + b) + q);
#pragma unroll
                        for (int m = 0; m < O2; ++m) {
                            const double w = ((m + odd) & 1) ? t[(m + odd) >> 1].y : t[(m + odd) >> 1].x;
#pragma unroll
                            for (int e = 0; e < NV; ++e) acc[m][e] = fma(w, in[e], acc[m][e]);
                        }
                    }
                }
        }
#pragma unroll
        for (int mq = 0; mq < O; ++mq)
#pragma unroll
            for (int mp = 0; mp < O; ++mp) {
                double *dst = oz + (long long)(j * O + mq) * g.sY + (long long)(i * O + mp) * g.sX;
                const int m = mp + O * mq;
#pragma unroll
                for (int e = 0; e < NV; ++e)
                    if (e < nve) __stcs(dst + LPC * e, acc[m][e]);
            }
    }
}

static bool xy_apply_streams(int O) { return (O == 2 || O == 3) && !getenv("SLDG_APPLY_DIRECT"); }
static int stream_segment_rows(int ny) { return ny < STREAM_LMAX ? ny : STREAM_LMAX; }

size_t xy_apply_stage_flags(const sldg_params *p)
{
    const int L = stream_segment_rows(p->n[1]), tx = stream_tx(p->order[0]);
    const size_t strips = (p->n[0] + tx - 1) / tx, segs = (p->n[1] + L - 1) / L;
    return strips * segs * (size_t)p->n[2] * p->order[2];
}

// one launch of the direct kernel over the v values [vbeg, vend): all cells (flags == nullptr, grid of 8 x 4 tiles) or
// only the cells of the non-stageable streaming blocks (grid of the streaming kernel)
static void launch_direct(sldg_ctx *c, const double *fin, double *fout, const int32_t *flags, int L, int nblk_x, int vbeg,
                          int vend)
{
    const GridDev &g = c->g;
    const int O = g.o[0], stx = stream_tx(O), span = vend - vbeg;
    // values per lane: as many as cover the range in one chunk, at most 5 (45 accumulators at o = 3)
    int nv = (span + 31) / 32;
    if (nv > 5) nv = 4;
    const int vchunks = (span + 32 * nv - 1) / (32 * nv);
    dim3 dgrid((unsigned)nblk_x, (unsigned)vchunks, (unsigned)g.N[2]);
#define LAUNCH_A(OO, NN) \
    xy_apply_direct_kernel<OO, NN><<<dgrid, 256, 0, c->stream>>>(fin, fout, c->hdr, c->W, g, flags, L, stx, vbeg, vend)
#define LAUNCH_AN(OO)                                                                                         \
    do {                                                                                                      \
        if (nv == 1) LAUNCH_A(OO, 1); else if (nv == 2) LAUNCH_A(OO, 2); else if (nv == 3) LAUNCH_A(OO, 3);   \
        else if (nv == 4) LAUNCH_A(OO, 4); else LAUNCH_A(OO, 5);                                              \
    } while (0)
    if (span <= 16 && O == 3) {
        dgrid.y = 1;
        xy_apply_direct_kernel<3, 2, 4><<<dgrid, 256, 0, c->stream>>>(fin, fout, c->hdr, c->W, g, flags, L, stx, vbeg, vend);
    } else if (O == 1) LAUNCH_AN(1); else if (O == 2) LAUNCH_AN(2); else LAUNCH_AN(3);
#undef LAUNCH_AN
#undef LAUNCH_A
    c->launches++;
}

cudaError_t launch_xy_apply(sldg_ctx *c, const double *fin, double *fout)
{
    const GridDev &g = c->g;
    const int O = g.o[0];
    const int tiles = ((g.n[0] + 7) / 8) * ((g.n[1] + 3) / 4);
    if (xy_apply_streams(O)) {
        // Which blocks can stream is decided on the device (scan of the headers); the streaming kernel does
        // those, the direct kernel the others (none in an ITG step; most of them in a solid-body rotation, where the
        // anchors change by many cells along a strip).  No host synchronisation.
        static const int vsplit = getenv("SLDG_APPLY_VSPLIT") ? atoi(getenv("SLDG_APPLY_VSPLIT")) : 1;
        const int stx = stream_tx(O);
        const int L = stream_segment_rows(g.n[1]);
        const int strips = (g.n[0] + stx - 1) / stx, segs = (g.n[1] + L - 1) / L;
        // v chunks of the streaming kernel.  A last chunk with fewer than 64 values (Pv = 144 at o = 3: 128 + 16) would
        // keep a whole block busy for as long as a full chunk -- its lanes are mostly idle, its FMAs are not fewer --
        // and double the kernel's time: that remainder goes to the direct kernel instead.
        int vstream = g.Pv;
        if (g.Pv > STREAM_VMAX && g.Pv % STREAM_VMAX != 0 && g.Pv % STREAM_VMAX < 64) vstream = g.Pv - g.Pv % STREAM_VMAX;
        const int VL = vstream < STREAM_VMAX ? vstream : STREAM_VMAX;
        const size_t ring = O == 3 ? StreamCfg<3>::RING : StreamCfg<2>::RING;
        xy_stageable_kernel<<<dim3((unsigned)(strips * segs), (unsigned)g.N[2]), 128, 0, c->stream>>>(
            c->hdr, g, L, VL, stx, ring, c->stage_ok, c->err);
        dim3 grid((unsigned)(strips * segs), (unsigned)((vstream + STREAM_VMAX - 1) / STREAM_VMAX), (unsigned)g.N[2]);
#define LAUNCH_S(OO, VS)                                                                                      \
    do {                                                                                                      \
        auto kern = xy_apply_stream_kernel<OO, VS>;                                                           \
        cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)stream_smem_bytes<OO>()); \
        kern<<<grid, 32 * (StreamCfg<OO>::TX * VS + 1), stream_smem_bytes<OO>(), c->stream>>>(                \
            fin, fout, c->hdr, c->W, g, L, c->stage_ok, vstream);                                             \
    } while (0)
        if (O == 3) LAUNCH_S(3, 2);
        else if (vsplit == 1) LAUNCH_S(2, 1);
        else LAUNCH_S(2, 2);
#undef LAUNCH_S
        c->launches += 2;
        launch_direct(c, fin, fout, c->stage_ok, L, strips * segs, 0, vstream);  // the non-stageable blocks
        if (vstream < g.Pv) launch_direct(c, fin, fout, nullptr, 0, tiles, vstream, g.Pv);  // the short last chunk
        return cudaGetLastError();
    }
    launch_direct(c, fin, fout, nullptr, 0, tiles, 0, g.Pv);
    return cudaGetLastError();
}
