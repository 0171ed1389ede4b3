// blas.cuh -- device scalars / state machine of a running CG and the deterministic grid reduction
// used by every kernel with a norm epilogue (row a3 of SURVEY.md sec 8: "reduced via warp shuffles").
#pragma once
#include "common.cuh"

// Device-resident CG state.  alpha/beta, the stopping test AND the decision to pause for a reliable
// update are taken by the LAST block of the kernel that produced the norm, so the host never feeds
// scalars back (SURVEY.md sec 7 hard part 4).  Every solver kernel carries a guard: it runs only
// while `done` has the value it was enqueued for, so the host can enqueue iterations and
// reliable-update blocks speculatively, ahead of the device, without changing the result:
//   done = 0  iterating            (iteration kernels run, reliable-update kernels are no-ops)
//   done = 1  paused: the iterated ||r||^2 met the target, dropped by delta^2, or the cap was hit
//             (reliable-update kernels run, iteration kernels are no-ops)
//   done = 2  converged: outer-precision ||bhat - Mhat y||^2 <= target2      (everything is a no-op)
//   done = 3  failed: iteration cap reached or NaN                           (everything is a no-op)
struct CgScalars {
    double gamma;      // ||z||^2 of the current search direction
    double ww;         // ||Mhat p||^2
    double rr;         // ||r||^2 (iterated)
    double alpha, beta;
    double target2;    // rho^2 ||eta||^2
    double ru2;        // pause for a reliable update when rr <= ru2 (= delta^2 ||r||^2 at the last update)
    double rr_true;    // ||bhat - Mhat y||^2 at the last reliable update (outer precision)
    double rho2, delta2;
    double slot[8];    // generic results (slot 0: ||eta||^2)
    int done;
    int iters;
    int max_iter;
    int n_ru;          // reliable updates so far
    int x_zero;        // x == 0 by construction (start of a solve / after a reliable update): x is neither read nor zero-filled
    int y_zero;        // y == 0 by construction (no reliable update yet): y is not read
    int x_pend;        // x still lacks alpha * p of the last iteration: that axpy rides in the NEXT update_p (which reads p
                       // anyway) instead of update_xr, or in ru_begin when the solve pauses first; alpha and p are
                       // unchanged until then
    int iters_at_ru;   // iteration count at the last reliable update (a reliable update is forced every 100 iterations)
    int stall;         // consecutive reliable updates that did not halve the true residual while far from the target
    int pause_iter[CG_MAX_PAUSES];   // iteration count at each pause (replayed by the host as a launch plan)
};

#define TM_MAXNB 8                // sources solved together at most (every kernel launch covers all of them)
#define TM_PSTRIDE (1 << 18)     // doubles between the reduction partials of consecutive sources of a grouped solve

enum { GUARD_ALWAYS = 0, GUARD_ITER = 1, GUARD_RU = 2 };     // run iff guard == 0 || done == guard - 1
__device__ __forceinline__ bool guard_skip(const CgScalars* sc, int guard) {
    return guard != GUARD_ALWAYS && sc->done != guard - 1;
}

// what the last block does with the reduced sum
enum {
    RED_NONE = 0,
    RED_WW,        // ww = sum; alpha = gamma / ww
    RED_RR,        // rr = sum; iters++; pause (done = 1) on target / reliable-update trigger / cap / NaN
    RED_ZZ,        // beta = gamma > 0 ? sum / gamma : 0; gamma = sum
    RED_START,     // sum = ||bhat||^2: target2, ru2, rr; done = 0 (or 1 when already converged / no iterations allowed)
    RED_RU,        // sum = ||bhat - Mhat y||^2: converged (2) | failed (3) | resume (0) with a new ru2
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

// what the reduced sum `s` does to the CG state (one thread)
__device__ __forceinline__ void apply_red_op(CgScalars* sc, int op, double s) {
    switch (op) {
        case RED_WW:
            // the update_p that ran just before this Dslash has applied the pending alpha * p to x (with the OLD alpha)
            if (sc->x_pend) { sc->x_zero = 0; sc->x_pend = 0; }
            sc->ww = s; sc->alpha = sc->gamma / s;
            break;
        case RED_RR:
            sc->rr = s; sc->iters += 1; sc->x_pend = 1;
            if (!(s > sc->target2) || !(s > sc->ru2) || sc->iters >= sc->max_iter || sc->iters - sc->iters_at_ru >= 100)
                sc->done = 1;
            break;
        case RED_ZZ: sc->beta = sc->gamma > 0.0 ? s / sc->gamma : 0.0; sc->gamma = s; break;
        case RED_START:
            sc->target2 = sc->rho2 * sc->slot[0];
            sc->rr = s; sc->rr_true = s; sc->ru2 = sc->delta2 * s;
            sc->done = (s > sc->target2 && sc->max_iter > 0) ? 0 : 1;
            break;
        case RED_RU:
            if (sc->n_ru < CG_MAX_PAUSES) sc->pause_iter[sc->n_ru] = sc->iters;
            // stagnation: the iterated residual fell by delta (or met the target) but the TRUE residual did not even
            // halve, twice in a row, while still more than 2x above the target -> the sloppy precision's floor is
            // reached (e.g. pure fp32 asked for 1e-8); give up instead of iterating to max_iter
            if (sc->n_ru > 0 && s > 0.25 * sc->rr_true && s > 4.0 * sc->target2) sc->stall += 1; else sc->stall = 0;
            sc->n_ru += 1;
            sc->rr_true = s;
            sc->iters_at_ru = sc->iters;
            sc->x_zero = 1; sc->y_zero = 0; sc->x_pend = 0;      // ru_begin folded x (and the pending alpha p) into y
            if (!(s == s)) sc->done = 3;
            else if (s <= sc->target2) sc->done = 2;
            else if (sc->iters >= sc->max_iter || sc->stall >= 2) sc->done = 3;
            else { sc->rr = s; sc->ru2 = sc->delta2 * s; sc->done = 0; }
            break;
        default: if (op >= RED_SLOT0) sc->slot[op - RED_SLOT0] = s; break;
    }
}

// Per-block partial only (no fence, no atomic, no last-block tail): used by the Dslash kernels, whose 8192
// short-lived CTAs would each hold their SM slot ~1 us longer for the fence + atomic of grid_reduce (measured:
// +13.5 us on a 66 us launch).  reduce_finish_kernel (blas.cu), enqueued right behind, sums the partials in
// a fixed order and applies the op.  Must be reached by all threads of the block.
__device__ __forceinline__ void block_partial_at(double v, double* partials, int slot, double* sm) {
    v = block_sum(v, sm);
    if (threadIdx.x == 0) partials[slot] = v;
}
__device__ __forceinline__ void block_partial(double v, double* partials, double* sm) {
    block_partial_at(v, partials, blockIdx.x, sm);
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
        // fixed-order sum of the per-block partials, 16 independent loads in flight per thread (a dependent
        // one-load-per-round loop over 8192 partials costs ~10 us of L2 latency at the tail of every Dslash)
        double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
        const unsigned int n = gridDim.x, bd = blockDim.x;
        unsigned int i = threadIdx.x;
        for (; i + 15u * bd < n; i += 16u * bd) {
            double v[16];
#pragma unroll
            for (int k = 0; k < 16; k++) v[k] = __ldcg(partials + i + (unsigned)k * bd);
#pragma unroll
            for (int k = 0; k < 16; k += 4) { s0 += v[k]; s1 += v[k + 1]; s2 += v[k + 2]; s3 += v[k + 3]; }
        }
        for (; i < n; i += bd) s0 += __ldcg(partials + i);
        double s = (s0 + s1) + (s2 + s3);
        s = block_sum(s, sm);
        if (threadIdx.x == 0) {
            *counter = 0;
            apply_red_op(sc, op, s);
        }
    }
}
