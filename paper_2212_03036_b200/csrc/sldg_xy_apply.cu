// sldg_xy_apply.cu -- eq. (17):  out[ij,m] = sum_{rs} sum_k (C^{ij,m}_{rs,k} / W_m) in[rs,k]
// for every (z, v), with the weights the geometry kernel left in the workspace (Algorithm 3, PAPER.md:287-293:
// coefficients once per z node, reused for every v).
//
// Thread mapping everywhere: lane <-> v (contiguous in memory), so the weights of a target cell are
// warp-uniform, the control flow over the (up to 3x3) non-empty source cells is warp-uniform, and empty
// source cells cost nothing.
//
//   xy_apply_stream_kernel (o = 2, the default): a streaming stencil in SOURCE-row order.  A block owns a
//     strip of TX = 8 target cells in x, a segment of up to 128 target rows in y, one z node and one chunk
//     of <= 128 v values.  The prologue reads the segment's headers and takes the bounds of the anchors;
//     they fix a static schedule: target row j uses source rows j+aymin .. j+aymin+2 and the x window
//     [axmin, TX-1+axmax].  A producer warp streams the source rows (each row = the window's lines, all v
//     of the chunk, 40 KB) and each target row's packed weight blocks into shared-memory rings with
//     cp.async.bulk copies completing on mbarriers.  Sixteen consumer warps (cell x half of the v chunk)
//     wait for ONE source row at a time, add its contributions to the (up to three) target rows that
//     use it -- their partial sums live in registers -- release the row at once, and store a target row
//     when its last source row has been applied.  Because a source row is never held while others arrive,
//     all but one ring slot are in flight.  Every input line is fetched once per strip (x halo:
//     window/TX = 10/8), weights once.  Segments whose anchors vary too much fall back to direct loads.
//   xy_apply_direct_kernel (any o): warp <-> target cell, inputs through L1.
#include <stdlib.h>

#include "sldg_internal.cuh"

__device__ __forceinline__ int wrap_idx(int i, int n)
{
    int r = i % n;
    return r < 0 ? r + n : r;
}

// ---- mbarrier / bulk-copy primitives (PTX) --------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t ok;
    do {
        asm volatile(
            "{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
            : "=r"(ok)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
    } while (!ok);
}

// One source cell's contribution for two v values per lane: 4 inputs (k), 16 weights W[k][m] (o = 2).
__device__ __forceinline__ void fma_block_o2(double (&acc)[4][2], const double2 (&in)[4], const double *Wp)
{
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const double2 w01 = *reinterpret_cast<const double2 *>(Wp + k * 4);
        const double2 w23 = *reinterpret_cast<const double2 *>(Wp + k * 4 + 2);
        acc[0][0] = fma(w01.x, in[k].x, acc[0][0]);
        acc[0][1] = fma(w01.x, in[k].y, acc[0][1]);
        acc[1][0] = fma(w01.y, in[k].x, acc[1][0]);
        acc[1][1] = fma(w01.y, in[k].y, acc[1][1]);
        acc[2][0] = fma(w23.x, in[k].x, acc[2][0]);
        acc[2][1] = fma(w23.x, in[k].y, acc[2][1]);
        acc[3][0] = fma(w23.y, in[k].x, acc[3][0]);
        acc[3][1] = fma(w23.y, in[k].y, acc[3][1]);
    }
}

constexpr int STREAM_TX = 8;        // target cells per strip
constexpr int STREAM_LMAX = 128;    // target rows per segment
constexpr int STREAM_VMAX = 128;    // v values per chunk
constexpr int STREAM_CWARPS = 16;   // consumer warps: cell x v half
constexpr int STREAM_THREADS = 32 * (STREAM_CWARPS + 1);
constexpr int STREAM_NRMAX = 8;     // ring slots (barrier arrays)
constexpr int STREAM_NW = 5;        // weight stages (target rows)
constexpr int STREAM_WROW = 48;     // weight blocks per target row stage (8 cells, <= 9 each, typically 35)
constexpr int STREAM_NACC = 3;      // source rows per target row handled by the register accumulators
constexpr size_t STREAM_RING_BYTES = 160 * 1024;
constexpr size_t STREAM_WRING_BYTES = (size_t)STREAM_NW * STREAM_WROW * 128;
constexpr size_t STREAM_HDR_BYTES = (size_t)STREAM_LMAX * STREAM_TX * 16;
constexpr size_t STREAM_SMEM = STREAM_RING_BYTES + STREAM_WRING_BYTES + STREAM_HDR_BYTES + 512;

__global__ void __launch_bounds__(STREAM_THREADS, 1) xy_apply_stream_kernel(
    const double *__restrict__ fin, double *__restrict__ fout, const int4 *__restrict__ hdrg,
    const double *__restrict__ W, GridDev g, int L)
{
    constexpr int TX = STREAM_TX, NW = STREAM_NW, NACC = STREAM_NACC;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double *ring = reinterpret_cast<double *>(smem_raw);                                  // [NR][2 kq][2*RW][VL]
    double *wring = reinterpret_cast<double *>(smem_raw + STREAM_RING_BYTES);             // [NW][WROW][16]
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
    const int VL = min(STREAM_VMAX, g.Pv - v0);  // multiple of 16
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
        if (i0 + ci < nx) h = __ldg(hdrg + zc + (long long)(j0 + jr) * nx + i0 + ci);
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
    const size_t stage_doubles = (size_t)2 * 2 * RW * VL;
    int NR = (int)(STREAM_RING_BYTES / (stage_doubles * 8));
    NR = NR > STREAM_NRMAX ? STREAM_NRMAX : NR;
    const bool staged = NR >= 2 && S <= NACC && bnd[4] <= STREAM_WROW;
    const double *fz = fin + z * g.sZ + v0;
    double *oz = fout + z * g.sZ + v0;

    if (!staged) {
        // direct path: warp <-> cell, 64 v values per pass
        for (int c = warp; c < rows * TX; c += STREAM_THREADS / 32) {
            const int jr = c / TX, ci = c % TX;
            const int4 h = hdr[c];
            if (i0 + ci >= nx || !h.z) continue;
            const int i = i0 + ci, j = j0 + jr;
            const long long cellid = zc + (long long)j * nx + i;
            const int gx = wrap_idx(i + h.x, nx), gy = wrap_idx(j + h.y, ny);
            for (int v = 2 * lane; v < VL; v += 64) {
                double acc[4][2] = {};
                int nb = 0;
#pragma unroll 1
                for (int slot = 0; slot < 9; ++slot) {
                    if (!((h.z >> slot) & 1)) continue;
                    int r = gx + slot % 3, s = gy + slot / 3;
                    if (r >= nx) r -= nx;
                    if (s >= ny) s -= ny;
                    double2 in[4];
#pragma unroll
                    for (int k = 0; k < 4; ++k)
                        in[k] = __ldg(reinterpret_cast<const double2 *>(
                            fz + (long long)(2 * s + (k >> 1)) * g.sY + (long long)(2 * r + (k & 1)) * g.sX + v));
                    fma_block_o2(acc, in, W + ((size_t)cellid * 9 + nb++) * 16);
                }
#pragma unroll
                for (int m = 0; m < 4; ++m)
                    *reinterpret_cast<double2 *>(oz + (long long)(2 * j + (m >> 1)) * g.sY +
                                                 (long long)(2 * i + (m & 1)) * g.sX + v) =
                        make_double2(acc[m][0], acc[m][1]);
            }
        }
        return;
    }

    const int nsrc = rows + S - 1;  // source rows y' = 0 .. nsrc-1, Y = j0 + aymin + y'

    if (warp == STREAM_CWARPS) {
        // ---------------- producer warp -------------------------------------------------------------------
        const int wx0 = wrap_idx(i0 + axmin, nx);       // first cell of the x window (wrapped)
        const int n1 = min(RW, nx - wx0);               // cells before the periodic seam
        const bool runs = (g.sX == (long long)VL) && RW <= nx;  // window lines contiguous in memory (z,y,x order)
        const uint32_t row_bytes = (uint32_t)(stage_doubles * 8);
        for (int k = 0; k < nsrc; ++k) {
            const int st = k % NR;
            if (k >= NR) mbar_wait(&empty[st], ((k / NR) & 1) ^ 1);
            if (lane == 0) mbar_arrive_expect_tx(&full[st], row_bytes);
            __syncwarp();
            const int sY = wrap_idx(j0 + aymin + k, ny);
            double *dst = ring + (size_t)st * stage_doubles;
            if (runs) {
                // per kq: one copy up to the seam, one after it
                if (lane < 4) {
                    const int kq = lane & 1, part = lane >> 1;
                    const int c0 = part ? 0 : wx0, nc = part ? RW - n1 : n1, off = part ? n1 : 0;
                    if (nc > 0)
                        bulk_g2s(dst + ((size_t)kq * 2 * RW + 2 * off) * VL,
                                 fz + (long long)(2 * sY + kq) * g.sY + (long long)(2 * c0) * g.sX,
                                 (uint32_t)(2 * nc * VL * 8), &full[st]);
                }
            } else {
                for (int l = lane; l < 4 * RW; l += 32) {
                    const int kq = l / (2 * RW), xd = l - kq * 2 * RW;
                    const int r = (wx0 + (xd >> 1)) % nx;  // the window may be wider than the periodic box
                    bulk_g2s(dst + ((size_t)kq * 2 * RW + xd) * VL,
                             fz + (long long)(2 * sY + kq) * g.sY + (long long)(2 * r + (xd & 1)) * g.sX,
                             (uint32_t)(VL * 8), &full[st]);
                }
            }
            // weights of target row k (first used with source row k)
            if (k < rows) {
                const int ws = k % NW;
                if (k >= NW) mbar_wait(&wempty[ws], ((k / NW) & 1) ^ 1);
                const int ci = lane;                      // one packed run of weight blocks per cell
                int cnt = 0, off = 0;
                if (ci < TX) {
                    const int4 h = hdr[k * TX + ci];
                    cnt = __popc(h.z);
                    off = h.w;
                }
                int tot = cnt;
#pragma unroll
                for (int o = 1; o < TX; o <<= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
                if (lane == 0) mbar_arrive_expect_tx(&wfull[ws], (uint32_t)(tot * 128));
                __syncwarp();
                if (cnt > 0) {
                    const long long cellid = zc + (long long)(j0 + k) * nx + i0 + ci;
                    bulk_g2s(wring + ((size_t)ws * STREAM_WROW + off) * 16, W + (size_t)cellid * 9 * 16,
                             (uint32_t)(cnt * 128), &wfull[ws]);
                }
            }
        }
        return;
    }

    // ---------------- consumer warps: cell = warp / 2, v half = warp % 2 -------------------------------------
    const int ci = warp >> 1, vh = warp & 1;
    const int v = vh * 64 + 2 * lane;
    const bool live = (i0 + ci < nx) && (v < VL);
    double acc[NACC][4][2];
#pragma unroll
    for (int a = 0; a < NACC; ++a)
#pragma unroll
        for (int m = 0; m < 4; ++m) acc[a][m][0] = acc[a][m][1] = 0.0;

    // one step: source row k; target rows k, k-1, k-2 (accumulator sets are indexed by row mod 3, static
    // because the step loop is unrolled by 3)
    for (int kb = 0; kb < rows + NACC - 1; kb += NACC) {
#pragma unroll
        for (int u = 0; u < NACC; ++u) {
            const int k = kb + u;
            if (k >= rows + NACC - 1) break;
            if (k < rows) mbar_wait(&wfull[k % NW], (k / NW) & 1);
            if (k < nsrc) {
                const int st = k % NR;
                mbar_wait(&full[st], (k / NR) & 1);
                const double *srow = ring + (size_t)st * stage_doubles + v;
#pragma unroll
                for (int d = 0; d < NACC; ++d) {
                    const int jr = k - d;
                    if (jr < 0 || jr >= rows) continue;
                    const int4 h = hdr[jr * TX + ci];
                    const int dy = d - (h.y - aymin);
                    if (!live || dy < 0 || dy > 2) continue;
                    const int mrow = (h.z >> (3 * dy)) & 7;
                    if (!mrow) continue;
                    const double *Wp = wring + ((size_t)(jr % NW) * STREAM_WROW + h.w +
                                                __popc(h.z & ((1 << (3 * dy)) - 1))) * 16;
                    const int bx = ci + h.x - axmin;
#pragma unroll
                    for (int dx = 0; dx < 3; ++dx) {
                        if (!((mrow >> dx) & 1)) continue;
                        const double *src = srow + (size_t)(2 * (bx + dx)) * VL;
                        double2 in[4];
                        in[0] = *reinterpret_cast<const double2 *>(src);
                        in[1] = *reinterpret_cast<const double2 *>(src + VL);
                        in[2] = *reinterpret_cast<const double2 *>(src + (size_t)2 * RW * VL);
                        in[3] = *reinterpret_cast<const double2 *>(src + (size_t)2 * RW * VL + VL);
                        fma_block_o2(acc[(u - d + NACC) % NACC], in, Wp);
                        Wp += 16;
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[st]);
            }
            // target row k - 2 has seen all its source rows
            const int jd = k - (NACC - 1);
            if (jd >= 0 && jd < rows) {
                constexpr int unused = 0;
                (void)unused;
                double(&a)[4][2] = acc[(u + 1) % NACC];  // (u - 2 + 3) % 3
                if (live && hdr[jd * TX + ci].z) {
                    const int i = i0 + ci, j = j0 + jd;
#pragma unroll
                    for (int m = 0; m < 4; ++m)
                        __stcs(reinterpret_cast<double2 *>(oz + (long long)(2 * j + (m >> 1)) * g.sY +
                                                           (long long)(2 * i + (m & 1)) * g.sX + v),
                               make_double2(a[m][0], a[m][1]));
                }
#pragma unroll
                for (int m = 0; m < 4; ++m) a[m][0] = a[m][1] = 0.0;
                __syncwarp();
                if (lane == 0) mbar_arrive(&wempty[jd % NW]);
            }
        }
    }
}

// --------------------------------------------------------------------------------------------------
// direct apply (any o): block = 8 warps, a tile of 8x4 target cells at one z node and one chunk of
// 32*NVT v values; warp <-> target cell (4 cells per warp), lane <-> v.  Inputs through L1.
// --------------------------------------------------------------------------------------------------
template <int O, int NVT>
__global__ void __launch_bounds__(256) xy_apply_direct_kernel(const double *__restrict__ fin,
                                                              double *__restrict__ fout,
                                                              const int4 *__restrict__ hdrg,
                                                              const double *__restrict__ W, GridDev g)
{
    constexpr int O2 = O * O, TX = 8, TY = 4;
    const int nx = g.n[0], ny = g.n[1];
    const int tiles_x = (nx + TX - 1) / TX;
    const int tile_i = (blockIdx.x % tiles_x) * TX, tile_j = (blockIdx.x / tiles_x) * TY;
    const int z = blockIdx.z;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int v = (blockIdx.y * 32 + lane) * NVT;
    if (v >= g.Pv) return;
    const long long ncell = (long long)nx * ny;
    const double *fz = fin + z * g.sZ + v;
    double *oz = fout + z * g.sZ + v;

    for (int c = warp; c < TX * TY; c += 8) {
        const int i = tile_i + (c % TX), j = tile_j + (c / TX);
        if (i >= nx || j >= ny) continue;
        const long long cellid = (long long)z * ncell + (long long)j * nx + i;
        const int4 h = __ldg(hdrg + cellid);
        const int ax = wrap_idx(i + h.x, nx);
        const int ay = wrap_idx(j + h.y, ny);
        const int msk = h.z;
        int nb = 0;
        double acc[O2][NVT];
#pragma unroll
        for (int m = 0; m < O2; ++m)
#pragma unroll
            for (int e = 0; e < NVT; ++e) acc[m][e] = 0.0;
#pragma unroll 1
        for (int slot = 0; slot < 9; ++slot) {
            if (!((msk >> slot) & 1)) continue;
            int r = ax + slot % 3, s = ay + slot / 3;
            if (r >= nx) r -= nx;
            if (s >= ny) s -= ny;
            const double *Wp = W + ((size_t)cellid * 9 + nb++) * (O2 * O2);
#pragma unroll
            for (int kq = 0; kq < O; ++kq)
#pragma unroll
                for (int kp = 0; kp < O; ++kp) {
                    const double *src = fz + (long long)(s * O + kq) * g.sY + (long long)(r * O + kp) * g.sX;
                    double in[NVT];
                    if (NVT == 2) {
                        double2 t = __ldg(reinterpret_cast<const double2 *>(src));
                        in[0] = t.x;
                        in[NVT - 1] = t.y;
                    } else {
                        in[0] = __ldg(src);
                    }
                    const int k = kp + O * kq;
#pragma unroll
                    for (int m = 0; m < O2; ++m) {
                        const double w = __ldg(Wp + k * O2 + m);
#pragma unroll
                        for (int e = 0; e < NVT; ++e) acc[m][e] = fma(w, in[e], acc[m][e]);
                    }
                }
        }
#pragma unroll
        for (int mq = 0; mq < O; ++mq)
#pragma unroll
            for (int mp = 0; mp < O; ++mp) {
                double *dst = oz + (long long)(j * O + mq) * g.sY + (long long)(i * O + mp) * g.sX;
                const int m = mp + O * mq;
                if (NVT == 2)
                    *reinterpret_cast<double2 *>(dst) = make_double2(acc[m][0], acc[m][NVT - 1]);
                else
                    dst[0] = acc[m][0];
            }
    }
}

cudaError_t launch_xy_apply(sldg_ctx *c, const double *fin, double *fout)
{
    const GridDev &g = c->g;
    const int O = g.o[0];
    if (O == 2 && !getenv("SLDG_APPLY_DIRECT")) {
        auto kern = xy_apply_stream_kernel;
        cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)STREAM_SMEM);
        const int L = g.n[1] < STREAM_LMAX ? g.n[1] : STREAM_LMAX;
        const int strips = (g.n[0] + STREAM_TX - 1) / STREAM_TX, segs = (g.n[1] + L - 1) / L;
        dim3 grid((unsigned)(strips * segs), (unsigned)((g.Pv + STREAM_VMAX - 1) / STREAM_VMAX), (unsigned)g.N[2]);
        kern<<<grid, STREAM_THREADS, STREAM_SMEM, c->stream>>>(fin, fout, c->hdr, c->W, g, L);
        c->launches++;
        return cudaGetLastError();
    }
    constexpr int NVT = 2;
    const int tiles = ((g.n[0] + 7) / 8) * ((g.n[1] + 3) / 4);
    const int vchunks = (g.Pv + 32 * NVT - 1) / (32 * NVT);
    dim3 grid((unsigned)tiles, (unsigned)vchunks, (unsigned)g.N[2]);
#define LAUNCH_A(OO) \
    xy_apply_direct_kernel<OO, NVT><<<grid, 256, 0, c->stream>>>(fin, fout, c->hdr, c->W, g)
    if (O == 1) LAUNCH_A(1); else if (O == 2) LAUNCH_A(2); else LAUNCH_A(3);
#undef LAUNCH_A
    c->launches++;
    return cudaGetLastError();
}
