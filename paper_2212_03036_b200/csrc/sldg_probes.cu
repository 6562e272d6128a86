// sldg_probes.cu -- measurement helpers of libsldg (not on the hot path): the fp64 FMA roof of the device, against
// which the ALU-bound kernels (2d geometry, 2d apply at o = 3; SURVEY.md 8(d) "Roofline per step")
// are scored, and the count of weight blocks the geometry produced (the flop count of the 2d apply).
#include "sldg_internal.cuh"

namespace {

// CH independent FMA chains per thread, each fed by its predecessor only: the fp64 pipe sees CH * warps independent
// instructions per scheduler.  8 warps per scheduler x 8 chains hide the pipe's latency many times over.
template <int CH>
__global__ void __launch_bounds__(256) fp64_fma_kernel(double *out, int iters, double a, double b)
{
    double x[CH];
#pragma unroll
    for (int k = 0; k < CH; ++k) x[k] = (double)(threadIdx.x + k) * 1e-3;
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u)
#pragma unroll
            for (int k = 0; k < CH; ++k) x[k] = fma(x[k], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < CH; ++k) s += x[k];
    if (s == 123.456) out[0] = s;  // never true; keeps the chains alive
}

__global__ void __launch_bounds__(256) count_blocks_kernel(const int4 *__restrict__ hdr, long long n,
                                                           unsigned long long *out)
{
    unsigned long long acc = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        acc += (unsigned)hdr[i].w;
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
    if ((threadIdx.x & 31) == 0 && acc) atomicAdd(out, acc);
}

}  // namespace

extern "C" int sldg_debug_fp64_peak(sldg_ctx *c, int repeats, double *tflops_host)
{
    if (!c || !tflops_host || repeats < 1) return SLDG_EINVAL;
    constexpr int CH = 8;
    const int iters = 4096, blocks = c->sm_count * 8, threads = 256;
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return SLDG_ECUDA;
    double best = 0.0;
    for (int r = 0; r <= repeats; ++r) {  // the first launch warms up
        cudaEventRecord(e0, c->stream);
        fp64_fma_kernel<CH><<<blocks, threads, 0, c->stream>>>(c->scalar_ws, iters, 0.999999, 1e-9);
        cudaEventRecord(e1, c->stream);
        c->launches++;
        if (cudaEventSynchronize(e1) != cudaSuccess) return SLDG_ECUDA;
        float ms = 0.0f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double flops = 2.0 * CH * 8.0 * iters * (double)blocks * threads;
        if (r > 0 && ms > 0.0f && flops / (ms * 1e-3) > best) best = flops / (ms * 1e-3);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *tflops_host = best * 1e-12;
    return cudaGetLastError() == cudaSuccess ? SLDG_OK : SLDG_ECUDA;
}

// number of non-empty (target cell, source cell) weight blocks of the last geometry, summed over all z nodes
cudaError_t count_weight_blocks(sldg_ctx *c, long long *total_host)
{
    const long long n = (long long)c->g.N[2] * c->g.n[0] * c->g.n[1];
    unsigned long long *cnt = reinterpret_cast<unsigned long long *>(c->scalar_ws) + 1;
    cudaError_t e = cudaMemsetAsync(cnt, 0, 8, c->stream);
    if (e != cudaSuccess) return e;
    count_blocks_kernel<<<c->sm_count * 4, 256, 0, c->stream>>>(c->hdr, n, cnt);
    c->launches++;
    unsigned long long v = 0;
    e = cudaMemcpyAsync(&v, cnt, 8, cudaMemcpyDeviceToHost, c->stream);
    if (e != cudaSuccess) return e;
    e = cudaStreamSynchronize(c->stream);
    *total_host = (long long)v;
    return e;
}
