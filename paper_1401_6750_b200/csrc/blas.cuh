// blas.cuh -- device scalars of a running CG and the deterministic grid reduction used by every
// kernel with a norm epilogue (row a3 of SURVEY.md sec 8: "reduced via warp shuffles").
#pragma once
#include "common.cuh"

// Device-resident CG state: alpha/beta/stopping are computed by the LAST block of the kernel that
// produced the norm, so the host never has to feed scalars back (SURVEY.md sec 7 hard part 4).
struct CgScalars {
    double gamma;      // ||z||^2 of the current search direction
    double ww;         // ||Mhat p||^2
    double rr;         // ||r||^2 (iterated)
    double alpha, beta;
    double target2;    // stop when rr <= target2
    double slot[8];    // generic results (norms for setup / true residual)
    int done;          // set once rr <= target2: later kernels of the solve become no-ops
    int iters;
    int pad[2];
};

// what the last block does with the reduced sum
enum {
    RED_NONE = 0,
    RED_WW,        // ww = sum; alpha = gamma / ww
    RED_RR,        // rr = sum; iters++; done = rr <= target2
    RED_ZZ,        // beta = sum / gamma; gamma = sum
    RED_ZZ_INIT,   // gamma = sum; beta = 0
    RED_SLOT0      // slot[k] = sum for RED_SLOT0 + k
};

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Block-wide sum (result valid in thread 0). blockDim.x multiple of 32, <= 1024.
__device__ __forceinline__ double block_sum(double v, double* sm /* >= 32 doubles */) {
    v = warp_sum(v);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) sm[w] = v;
    __syncthreads();
    if (w == 0) {
        v = (lane < (int)((blockDim.x + 31) >> 5)) ? sm[lane] : 0.0;
        v = warp_sum(v);
    }
    return v;
}

// Deterministic grid reduction: every block deposits its partial, the last one to arrive sums all
// partials in a fixed order and applies `op` to the CG scalars.  Must be reached by all threads.
__device__ __forceinline__ void grid_reduce(double v, double* partials, unsigned int* counter,
                                            CgScalars* sc, int op, double* sm) {
    __shared__ bool is_last;
    v = block_sum(v, sm);
    if (threadIdx.x == 0) {
        partials[blockIdx.x] = v;
        __threadfence();
        unsigned int t = atomicAdd(counter, 1u);
        is_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (is_last) {
        __threadfence();
        double s = 0.0;
        for (unsigned int i = threadIdx.x; i < gridDim.x; i += blockDim.x) s += __ldcg(partials + i);
        s = block_sum(s, sm);
        if (threadIdx.x == 0) {
            *counter = 0;
            switch (op) {
                case RED_WW: sc->ww = s; sc->alpha = sc->gamma / s; break;
                case RED_RR: sc->rr = s; sc->iters += 1; if (s <= sc->target2) sc->done = 1; break;
                case RED_ZZ: sc->beta = s / sc->gamma; sc->gamma = s; break;
                case RED_ZZ_INIT: sc->gamma = s; sc->beta = 0.0; break;
                default: if (op >= RED_SLOT0) sc->slot[op - RED_SLOT0] = s; break;
            }
        }
    }
}
