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
    // Mass: w^T (A + B) = w^T holds for the exact matrices; the Horner values miss it by a few
    // 1e-17 with a sign that depends smoothly on alpha, which adds up to a drift of ~1.5e-16 per sweep (measured).
    // The defect of every column goes into its diagonal entry, which leaves an unbiased rounding error.  At
    // alpha = 0 (A = I, B = 0 exactly) the defect is exactly 0: integer shifts stay bit-exact copies.
#pragma unroll
    for (int m = 0; m < O; ++m) {
        double sum = 0.0;
#pragma unroll
        for (int j = 0; j < O; ++j) sum = fma(sp.w[j], A[j][m] + B[j][m], sum);
        A[m][m] = fma(sp.w[m] - sum, sp.iw[m], A[m][m]);
    }
}

__device__ __forceinline__ int wrapi(int i, int n)
{
    int r = i % n;
    return r < 0 ? r + n : r;
}

