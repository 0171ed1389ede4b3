// su3.cuh -- SU(3) link times half-spinor (2 spins x 3 colours), shared by the stencil kernels.
#pragma once

// v = U u (DAG = 0) or U^dag u (DAG = 1) for the two spins of a half-spinor
template <int DAG, typename F>
__device__ __forceinline__ void su3_mul_half(const F* U, const F* u, F* v) {
#pragma unroll
    for (int sp = 0; sp < 2; sp++)
#pragma unroll
        for (int a = 0; a < 3; a++) {
            F re = 0, im = 0;
#pragma unroll
            for (int b = 0; b < 3; b++) {
                const F ur = DAG ? U[(b * 3 + a) * 2] : U[(a * 3 + b) * 2];
                const F ui = DAG ? -U[(b * 3 + a) * 2 + 1] : U[(a * 3 + b) * 2 + 1];
                const F xr = u[sp * 6 + 2 * b], xi = u[sp * 6 + 2 * b + 1];
                // one FMA per statement (a single expression would cost FMUL + FFMA + FADD)
                re += ur * xr; re -= ui * xi;
                im += ur * xi; im += ui * xr;
            }
            v[sp * 6 + 2 * a] = re;
            v[sp * 6 + 2 * a + 1] = im;
        }
}

