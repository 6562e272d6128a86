// sldg_sweep_common.cuh -- device helpers shared by the 1d sweep kernels (sldg_sweeps.cu, sldg_fused_sweeps.cu).
#pragma once
#include "sldg_internal.cuh"

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

