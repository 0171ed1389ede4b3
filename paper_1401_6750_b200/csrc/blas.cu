// blas.cu -- BLAS-1 updates and norms of the CG, fused per update step.
// Work item = (site h, group g of 8 reals): identical (site, component) mapping in every storage
// precision, coalesced 16-byte accesses across h, so mixed-precision updates need no reshuffle.
#include <type_traits>
#include "kernels.h"

template <typename Fn> static tm_status dispatch_prec(tm_ctx* ctx, tm_prec p, Fn&& f) {
    switch (p) {
        case TM_F64:  return f((double*)nullptr);
        case TM_F32:  return f((float*)nullptr);
        case TM_F16:  return f((__half*)nullptr);
        case TM_BF16: return f((__nv_bfloat16*)nullptr);
    }
    return tm_fail(ctx, TM_EPREC, "unknown precision");
}
#define TAGTYPE(tag) typename std::remove_pointer<decltype(tag)>::type

// Grouped solves (ctx->nb = 2 | 4): blockIdx.y selects the source; consecutive sources' vectors sit one parity vector
// (24 Vh elements of their own type) apart, their CG states, reduction partials and counters one slot apart.
template <typename S> __device__ __forceinline__ S* src_vec(S* p, int src, int Vh) {
    return p ? p + (size_t)src * 24 * (size_t)Vh : p;
}
static inline dim3 pair_grid(const tm_ctx* ctx, unsigned gx) { return dim3(gx, (unsigned)(ctx->nb > 1 ? ctx->nb : 1)); }

static inline unsigned items_grid(const tm_ctx* ctx, int block, int nparity = 1) {
    return (unsigned)((3 * ctx->Vh * nparity + block - 1) / block);
}

// ------------------------------------------------------------------ copy / convert
template <typename Sd, typename Ss>
__global__ void copy_kernel(Sd* __restrict__ dst, const Ss* __restrict__ src, int Vh) {
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= 3L * Vh) return;
    const int g = (int)(i / Vh), h = (int)(i % Vh);
    typename Prec<Ss>::F a[8];
    typename Prec<Sd>::F b[8];
    load8<Ss>(src, Vh, h, g, a);
#pragma unroll
    for (int k = 0; k < 8; k++) b[k] = (typename Prec<Sd>::F)a[k];
    store8<Sd>(dst, Vh, h, g, b);
}

tm_status blas_zero(tm_ctx* ctx, void* v, tm_prec p, cudaStream_t st) {
    TM_CUDA(ctx, cudaMemsetAsync(v, 0, tm_parity_bytes(ctx, p), st));
    return TM_OK;
}

tm_status blas_copy(tm_ctx* ctx, void* dst, tm_prec pd, const void* src, tm_prec ps, cudaStream_t st) {
    if (pd == ps) {
        TM_CUDA(ctx, cudaMemcpyAsync(dst, src, tm_parity_bytes(ctx, pd), cudaMemcpyDeviceToDevice, st));
        return TM_OK;
    }
    return dispatch_prec(ctx, pd, [&](auto* td) {
        return dispatch_prec(ctx, ps, [&](auto* ts) {
            typedef TAGTYPE(td) Sd;
            typedef TAGTYPE(ts) Ss;
            copy_kernel<Sd, Ss><<<items_grid(ctx, 256), 256, 0, st>>>((Sd*)dst, (const Ss*)src, (int)ctx->Vh);
            TM_LAUNCH_CHECK(ctx, "copy_kernel");
            return TM_OK;
        });
    });
}

// ------------------------------------------------------------------ dst = A^-1 src
template <typename S>
__global__ void twist_inv_kernel(S* __restrict__ dst, const S* __restrict__ src, int Vh,
                                 typename Prec<S>::F a, int dst_mul, int src_mul) {
    typedef typename Prec<S>::F F;
    dst = src_vec(dst, blockIdx.y * dst_mul, Vh); src = src_vec(src, blockIdx.y * src_mul, Vh);
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= 3L * Vh) return;
    const int g = (int)(i / Vh), h = (int)(i % Vh);
    F v[8];
    load8<S>(src, Vh, h, g, v);
    // reals 8g..8g+7: spin = (8g + k)/6 ; upper spins (0,1) are reals 0..11, lower 12..23
    const F n = F(1) / (F(1) + a * a);
#pragma unroll
    for (int k = 0; k < 8; k += 2) {
        const bool upper = (8 * g + k) < 12;
        const F s = upper ? a : -a;                 // A^-1 = (1 - i s)/(1+a^2) on this chirality
        const F re = v[k], im = v[k + 1];
        v[k] = n * (re + s * im);
        v[k + 1] = n * (im - s * re);
    }
    store8<S>(dst, Vh, h, g, v);
}

// dst = A^-1 src + c * add   (odd-site reconstruction s_o = A^-1 eta_o + kappa [A^-1 D_oe y], solver.cu)
template <typename S>
__global__ void twist_inv_axpy_kernel(S* __restrict__ dst, const S* __restrict__ src, const S* __restrict__ add, int Vh,
                                      typename Prec<S>::F a, typename Prec<S>::F c, int dst_mul, int src_mul, int add_mul) {
    typedef typename Prec<S>::F F;
    dst = src_vec(dst, blockIdx.y * dst_mul, Vh); src = src_vec(src, blockIdx.y * src_mul, Vh);
    add = src_vec(add, blockIdx.y * add_mul, Vh);
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= 3L * Vh) return;
    const int g = (int)(i / Vh), h = (int)(i % Vh);
    F v[8], w[8];
    load8<S>(src, Vh, h, g, v);
    load8<S>(add, Vh, h, g, w);
    const F n = F(1) / (F(1) + a * a);
#pragma unroll
    for (int k = 0; k < 8; k += 2) {
        const bool upper = (8 * g + k) < 12;
        const F s = upper ? a : -a;
        const F re = v[k], im = v[k + 1];
        v[k] = n * (re + s * im) + c * w[k];
        v[k + 1] = n * (im - s * re) + c * w[k + 1];
    }
    store8<S>(dst, Vh, h, g, v);
}
tm_status blas_twist_inv_axpy(tm_ctx* ctx, void* dst, const void* src, const void* add, tm_prec p, double kappa,
                              double mu, double c, cudaStream_t st, int dst_mul, int src_mul, int add_mul) {
    const double a = 2.0 * kappa * mu;
    return dispatch_prec(ctx, p, [&](auto* t) {
        typedef TAGTYPE(t) S;
        typedef typename Prec<S>::F F;
        twist_inv_axpy_kernel<S><<<pair_grid(ctx, items_grid(ctx, 256)), 256, 0, st>>>((S*)dst, (const S*)src, (const S*)add, (int)ctx->Vh, (F)a, (F)c,
                                                                                             dst_mul, src_mul, add_mul);
        TM_LAUNCH_CHECK(ctx, "twist_inv_axpy_kernel");
        return TM_OK;
    });
}

tm_status blas_twist_inv(tm_ctx* ctx, void* dst, const void* src, tm_prec p, double kappa, double mu,
                         int dagger, cudaStream_t st, int dst_mul, int src_mul) {
    const double a = 2.0 * kappa * mu * (dagger ? -1.0 : 1.0);
    return dispatch_prec(ctx, p, [&](auto* t) {
        typedef TAGTYPE(t) S;
        twist_inv_kernel<S><<<pair_grid(ctx, items_grid(ctx, 256)), 256, 0, st>>>((S*)dst, (const S*)src, (int)ctx->Vh,
                                                               (typename Prec<S>::F)a, dst_mul, src_mul);
        TM_LAUNCH_CHECK(ctx, "twist_inv_kernel");
        return TM_OK;
    });
}

// ------------------------------------------------------------------ reliable update, part 1: y += x (+ alpha p) ; x = 0
template <typename Sy, typename Sx, typename Sp>
__global__ void ru_begin_kernel(Sy* __restrict__ y, Sx* __restrict__ x, const Sp* __restrict__ p, int Vh, const CgScalars* sc,
                                int y_mul) {
    sc += blockIdx.y; y = src_vec(y, blockIdx.y * y_mul, Vh); x = src_vec(x, blockIdx.y, Vh); p = src_vec(p, blockIdx.y, Vh);
    if (guard_skip(sc, GUARD_RU)) return;
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= 3L * Vh) return;
    const int g = (int)(i / Vh), h = (int)(i % Vh);
    // y += x ; x = 0, with both vectors possibly "zero by construction" (CgScalars::x_zero / y_zero: then they are
    // not read, and x is not zero-filled -- RED_RU raises x_zero instead); x_pend: the axpy of the last iteration has
    // not reached x yet (it rides in the next update_p) and is applied here, in x's precision, before x goes into y
    const bool xz = sc->x_zero != 0, yz = sc->y_zero != 0, pend = sc->x_pend != 0;
    if (xz && !pend && !yz) return;
    typedef typename Prec<Sx>::F FA;
    FA a[8];
    typename Prec<Sy>::F b[8];
#pragma unroll
    for (int k = 0; k < 8; k++) { a[k] = 0; b[k] = 0; }
    if (!xz) load8<Sx>(x, Vh, h, g, a);
    if (pend) {
        const FA alpha = (FA)sc->alpha;
        typename Prec<Sp>::F vp[8];
        load8<Sp>(p, Vh, h, g, vp);
#pragma unroll
        for (int k = 0; k < 8; k++) a[k] += alpha * (FA)vp[k];
    }
    if (!yz) load8<Sy>(y, Vh, h, g, b);
#pragma unroll
    for (int k = 0; k < 8; k++) b[k] += (typename Prec<Sy>::F)a[k];
    store8<Sy>(y, Vh, h, g, b);
}

tm_status blas_ru_begin(tm_ctx* ctx, void* y, tm_prec po, void* x, tm_prec pacc, const void* p, tm_prec psl, cudaStream_t st,
                        int y_mul) {
    const dim3 grid = pair_grid(ctx, items_grid(ctx, 256));
    const int Vh = (int)ctx->Vh;
    const CgScalars* sc = ctx->d_scal;
#define RUB(SY, SX, SP) ru_begin_kernel<SY, SX, SP><<<grid, 256, 0, st>>>((SY*)y, (SX*)x, (const SP*)p, Vh, sc, y_mul)
    if (po == TM_F64 && pacc == TM_F64 && psl == TM_F64) RUB(double, double, double);
    else if (po == TM_F64 && pacc == TM_F32 && psl == TM_F32) RUB(double, float, float);
    else if (po == TM_F64 && pacc == TM_F32 && psl == TM_F16) RUB(double, float, __half);
    else if (po == TM_F64 && pacc == TM_F32 && psl == TM_BF16) RUB(double, float, __nv_bfloat16);
    else if (po == TM_F32 && pacc == TM_F32 && psl == TM_F32) RUB(float, float, float);
    else if (po == TM_F32 && pacc == TM_F32 && psl == TM_F16) RUB(float, float, __half);
    else if (po == TM_F32 && pacc == TM_F32 && psl == TM_BF16) RUB(float, float, __nv_bfloat16);
    else return tm_fail(ctx, TM_EPREC, "ru_begin: unsupported precision triple");
#undef RUB
    TM_LAUNCH_CHECK(ctx, "ru_begin_kernel");
    return TM_OK;
}

// ------------------------------------------------------------------ r = b - m (acc), rs = b - m (sloppy), ||b - m||^2
// m == NULL: r = rs = b (start of a solve).  SA == SL: rs is not written (r is the sloppy vector).
template <typename SO, typename SA, typename SL>
__global__ void __launch_bounds__(256) residual_kernel(SA* __restrict__ r, SL* __restrict__ rs, const SO* __restrict__ b,
                                                       const SO* __restrict__ m, int Vh, int red_op, int guard,
                                                       double* partials, unsigned int* counter, CgScalars* sc) {
    typedef typename Prec<SO>::F FO;
    typedef typename Prec<SA>::F FA;
    typedef typename Prec<SL>::F FL;
    __shared__ double sm[32];
    {
        const int src = blockIdx.y;
        sc += src; partials += src * TM_PSTRIDE; counter += src;
        r = src_vec(r, src, Vh); rs = src_vec(rs, src, Vh); b = src_vec(b, src, Vh); m = src_vec(m, src, Vh);
    }
    if (guard_skip(sc, guard)) return;
    double nrm = 0.0;
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < 3L * Vh; i += (long)gridDim.x * blockDim.x) {
        const int g = (int)(i / Vh), h = (int)(i % Vh);
        FO vb[8];
        load8<SO>(b, Vh, h, g, vb);
        if (m) {
            FO vm[8];
            load8<SO>(m, Vh, h, g, vm);
#pragma unroll
            for (int k = 0; k < 8; k++) vb[k] -= vm[k];
        }
        FA va[8];
#pragma unroll
        for (int k = 0; k < 8; k++) { nrm += (double)vb[k] * (double)vb[k]; va[k] = (FA)vb[k]; }
        if (r) store8<SA>(r, Vh, h, g, va);          // r == NULL: the residual lives in sloppy storage only
        if (!std::is_same<SA, SL>::value) {
            FL vs[8];
#pragma unroll
            for (int k = 0; k < 8; k++) vs[k] = (FL)vb[k];
            store8<SL>(rs, Vh, h, g, vs);
        }
    }
    grid_reduce(nrm, partials, counter, sc, red_op, sm);
}

static inline unsigned red_grid(const tm_ctx* ctx, long items, int block) {
    long g = (items + block - 1) / block;
    long cap = (long)ctx->sm_count * 16;
    return (unsigned)(g < cap ? g : cap);
}

template <typename SO, typename SA, typename SL>
static tm_status residual_launch(tm_ctx* ctx, void* r, void* rs, const void* b, const void* m, int red_op, int guard,
                                 cudaStream_t st) {
    const dim3 grid = pair_grid(ctx, red_grid(ctx, 3L * ctx->Vh, 256));
    residual_kernel<SO, SA, SL><<<grid, 256, 0, st>>>((SA*)r, (SL*)rs, (const SO*)b, (const SO*)m, (int)ctx->Vh, red_op,
                                                     guard, ctx->d_partials, ctx->d_counter, ctx->d_scal);
    TM_LAUNCH_CHECK(ctx, "residual_kernel");
    return TM_OK;
}

tm_status blas_residual(tm_ctx* ctx, void* r, tm_prec pacc, void* rs, tm_prec psl, const void* b, const void* m,
                        tm_prec po, int red_op, int guard, cudaStream_t st) {
    if (po == TM_F64) {
        if (pacc == TM_F64 && psl == TM_F64) return residual_launch<double, double, double>(ctx, r, rs, b, m, red_op, guard, st);
        if (pacc == TM_F32 && psl == TM_F32) return residual_launch<double, float, float>(ctx, r, rs, b, m, red_op, guard, st);
        if (pacc == TM_F32 && psl == TM_F16) return residual_launch<double, float, __half>(ctx, r, rs, b, m, red_op, guard, st);
        if (pacc == TM_F32 && psl == TM_BF16) return residual_launch<double, float, __nv_bfloat16>(ctx, r, rs, b, m, red_op, guard, st);
    } else if (po == TM_F32 && pacc == TM_F32) {
        if (psl == TM_F32) return residual_launch<float, float, float>(ctx, r, rs, b, m, red_op, guard, st);
        if (psl == TM_F16) return residual_launch<float, float, __half>(ctx, r, rs, b, m, red_op, guard, st);
        if (psl == TM_BF16) return residual_launch<float, float, __nv_bfloat16>(ctx, r, rs, b, m, red_op, guard, st);
    }
    return tm_fail(ctx, TM_EPREC, "residual: unsupported precision combination");
}

// ------------------------------------------------------------------ ||v||^2
template <typename S>
__global__ void __launch_bounds__(256) norm_kernel(const S* __restrict__ v, long Vh_items, int Vh, int red_op,
                                                   double* partials, unsigned int* counter, CgScalars* sc) {
    typedef typename Prec<S>::F F;
    __shared__ double sm[32];
    double nrm = 0.0;
    // Vh_items = 3 * (number of sites in the field): a full-lattice field is two consecutive parity blocks
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < Vh_items; i += (long)gridDim.x * blockDim.x) {
        const long blk = i / (3L * Vh);
        const long j = i - blk * 3L * Vh;
        const int g = (int)(j / Vh), h = (int)(j % Vh);
        F a[8];
        load8<S>(v + blk * 24L * Vh, Vh, h, g, a);
#pragma unroll
        for (int k = 0; k < 8; k++) nrm += (double)a[k] * (double)a[k];
    }
    grid_reduce(nrm, partials, counter, sc, red_op, sm);
}

static tm_status norm_impl(tm_ctx* ctx, const void* v, tm_prec p, int red_op, int nparity, cudaStream_t st) {
    const long items = 3L * ctx->Vh * nparity;
    const unsigned grid = red_grid(ctx, items, 256);
    return dispatch_prec(ctx, p, [&](auto* t) {
        typedef TAGTYPE(t) S;
        norm_kernel<S><<<grid, 256, 0, st>>>((const S*)v, items, (int)ctx->Vh, red_op, ctx->d_partials,
                                             ctx->d_counter, ctx->d_scal);
        TM_LAUNCH_CHECK(ctx, "norm_kernel");
        return TM_OK;
    });
}
tm_status blas_norm(tm_ctx* ctx, const void* v, tm_prec p, int red_op, cudaStream_t st) { return norm_impl(ctx, v, p, red_op, 1, st); }
tm_status blas_norm_full(tm_ctx* ctx, const void* v, tm_prec p, int red_op, cudaStream_t st) { return norm_impl(ctx, v, p, red_op, 2, st); }

// ------------------------------------------------------------------ r -= alpha w ; ||r||^2
// (x += alpha p, the other half of the textbook update, is deferred to the next update_p -- which reads p anyway -- or
//  to ru_begin when the solve pauses first: CgScalars::x_pend.  Same operations on x in the same order, one read of
//  p per iteration less.)
template <typename SA, typename SL>
__global__ void __launch_bounds__(256) update_xr_kernel(SA* __restrict__ r, const SL* __restrict__ w,
                                                        SL* __restrict__ rs, int Vh, double* partials,
                                                        unsigned int* counter, CgScalars* sc) {
    typedef typename Prec<SA>::F FA;
    typedef typename Prec<SL>::F FL;
    __shared__ double sm[32];
    {
        const int src = blockIdx.y;
        sc += src; partials += src * TM_PSTRIDE; counter += src;
        r = src_vec(r, src, Vh); w = src_vec(w, src, Vh); rs = src_vec(rs, src, Vh);
    }
    if (guard_skip(sc, GUARD_ITER)) return;
    const FA alpha = (FA)sc->alpha;
    double nrm = 0.0;
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < 3L * Vh; i += (long)gridDim.x * blockDim.x) {
        const int g = (int)(i / Vh), h = (int)(i % Vh);
        FA vr[8];
        FL vw[8];
        if (r) load8<SA>(r, Vh, h, g, vr);
        else {                                       // r == NULL: the residual lives in sloppy storage only
            FL vs[8];
            load8<SL>(rs, Vh, h, g, vs);
#pragma unroll
            for (int k = 0; k < 8; k++) vr[k] = (FA)vs[k];
        }
        load8<SL>(w, Vh, h, g, vw);
#pragma unroll
        for (int k = 0; k < 8; k++) {
            vr[k] -= alpha * (FA)vw[k];
            nrm += (double)vr[k] * (double)vr[k];
        }
        if (r) store8<SA>(r, Vh, h, g, vr);
        if (!std::is_same<SA, SL>::value) {
            FL vs[8];
#pragma unroll
            for (int k = 0; k < 8; k++) vs[k] = (FL)vr[k];
            store8<SL>(rs, Vh, h, g, vs);
        }
    }
    grid_reduce(nrm, partials, counter, sc, RED_RR, sm);
}

tm_status blas_update_xr(tm_ctx* ctx, void* r, tm_prec pacc, const void* w, void* rs, tm_prec psl, cudaStream_t st) {
    const dim3 grid = pair_grid(ctx, red_grid(ctx, 3L * ctx->Vh, 256));
    const int Vh = (int)ctx->Vh;
    double* pa = ctx->d_partials; unsigned int* cn = ctx->d_counter; CgScalars* sc = ctx->d_scal;
    if (pacc == TM_F64 && psl == TM_F64)
        update_xr_kernel<double, double><<<grid, 256, 0, st>>>((double*)r, (const double*)w, (double*)rs, Vh, pa, cn, sc);
    else if (pacc == TM_F32 && psl == TM_F32)
        update_xr_kernel<float, float><<<grid, 256, 0, st>>>((float*)r, (const float*)w, (float*)rs, Vh, pa, cn, sc);
    else if (pacc == TM_F32 && psl == TM_F16)
        update_xr_kernel<float, __half><<<grid, 256, 0, st>>>((float*)r, (const __half*)w, (__half*)rs, Vh, pa, cn, sc);
    else if (pacc == TM_F32 && psl == TM_BF16)
        update_xr_kernel<float, __nv_bfloat16><<<grid, 256, 0, st>>>((float*)r, (const __nv_bfloat16*)w, (__nv_bfloat16*)rs, Vh, pa, cn, sc);
    else return tm_fail(ctx, TM_EPREC, "update_xr: unsupported precision pair");
    TM_LAUNCH_CHECK(ctx, "update_xr_kernel");
    return TM_OK;
}

// ------------------------------------------------------------------ x += alpha_old p (if pending) ; p = z + beta p
template <typename SA, typename S>
__global__ void update_p_kernel(S* __restrict__ p, const S* __restrict__ z, SA* __restrict__ x, int Vh, const CgScalars* sc) {
    typedef typename Prec<S>::F F;
    typedef typename Prec<SA>::F FA;
    sc += blockIdx.y; p = src_vec(p, blockIdx.y, Vh); z = src_vec(z, blockIdx.y, Vh); x = src_vec(x, blockIdx.y, Vh);
    if (guard_skip(sc, GUARD_ITER)) return;
    const F beta = (F)sc->beta;
    // the axpy of the previous iteration (CgScalars::x_pend): alpha is still that iteration's (the next RED_WW replaces
    // it, and marks x as up to date), p is still its search direction
    const bool pend = sc->x_pend != 0, xz = sc->x_zero != 0;
    const FA alpha = (FA)sc->alpha;
    const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= 3L * Vh) return;
    const int g = (int)(i / Vh), h = (int)(i % Vh);
    F vp[8], vz[8];
    load8<S>(z, Vh, h, g, vz);
    if (beta != F(0) || pend) load8<S>(p, Vh, h, g, vp);
    if (pend) {
        FA vx[8];
        if (xz) {                   // first update after a (re)start: x is zero by construction
#pragma unroll
            for (int k = 0; k < 8; k++) vx[k] = 0;
        } else load8<SA>(x, Vh, h, g, vx);
#pragma unroll
        for (int k = 0; k < 8; k++) vx[k] += alpha * (FA)vp[k];
        store8<SA>(x, Vh, h, g, vx);
    }
    if (beta != F(0)) {             // beta == 0: first iteration of a solve, p is uninitialised, p = z
#pragma unroll
        for (int k = 0; k < 8; k++) vp[k] = vz[k] + beta * vp[k];
    } else {
#pragma unroll
        for (int k = 0; k < 8; k++) vp[k] = vz[k];
    }
    store8<S>(p, Vh, h, g, vp);
}

tm_status blas_update_p(tm_ctx* ctx, void* p, const void* z, tm_prec psl, void* x, tm_prec pacc, cudaStream_t st) {
    const dim3 grid = pair_grid(ctx, items_grid(ctx, 256));
    const int Vh = (int)ctx->Vh;
    const CgScalars* sc = ctx->d_scal;
    if (pacc == TM_F64 && psl == TM_F64) update_p_kernel<double, double><<<grid, 256, 0, st>>>((double*)p, (const double*)z, (double*)x, Vh, sc);
    else if (pacc == TM_F32 && psl == TM_F32) update_p_kernel<float, float><<<grid, 256, 0, st>>>((float*)p, (const float*)z, (float*)x, Vh, sc);
    else if (pacc == TM_F32 && psl == TM_F16) update_p_kernel<float, __half><<<grid, 256, 0, st>>>((__half*)p, (const __half*)z, (float*)x, Vh, sc);
    else if (pacc == TM_F32 && psl == TM_BF16) update_p_kernel<float, __nv_bfloat16><<<grid, 256, 0, st>>>((__nv_bfloat16*)p, (const __nv_bfloat16*)z, (float*)x, Vh, sc);
    else return tm_fail(ctx, TM_EPREC, "update_p: unsupported precision pair");
    TM_LAUNCH_CHECK(ctx, "update_p_kernel");
    return TM_OK;
}

// ------------------------------------------------------------------ scalars
__global__ void scal_init_kernel(CgScalars* sc, double rho2, double delta2, int max_iter, double eta2) {
    CgScalars z;
    memset(&z, 0, sizeof(z));
    z.rho2 = rho2; z.delta2 = delta2; z.max_iter = max_iter;
    z.x_zero = 1; z.y_zero = 1;
    z.slot[0] = eta2;               // ||eta||^2 when the caller knows it (else 0, filled by the norm kernel)
    sc[blockIdx.x] = z;
}
tm_status scal_init(tm_ctx* ctx, double rho2, double delta2, int max_iter, double eta2, cudaStream_t st) {
    scal_init_kernel<<<ctx->nb > 1 ? ctx->nb : 1, 1, 0, st>>>(ctx->d_scal, rho2, delta2, max_iter, eta2);
    TM_LAUNCH_CHECK(ctx, "scal_init_kernel");
    return TM_OK;
}
tm_status scal_get(tm_ctx* ctx, CgScalars* v, cudaStream_t st) {
    TM_CUDA(ctx, cudaMemcpyAsync(ctx->h_scal, ctx->d_scal, TM_MAXNB * sizeof(CgScalars), cudaMemcpyDeviceToHost, st));
    TM_CUDA(ctx, cudaStreamSynchronize(st));
    for (int b = 0; b < TM_MAXNB; b++) v[b] = ctx->h_scal[b];
    return TM_OK;
}

// ------------------------------------------------------------------ second stage of the Dslash norm epilogue
// one block: fixed-order sum of the n per-block partials a Dslash kernel left behind, then the op on the CG state
__global__ void __launch_bounds__(1024) reduce_finish_kernel(const double* __restrict__ partials, unsigned int n,
                                                             CgScalars* sc, int op, int guard) {
    __shared__ double sm[32];
    sc += blockIdx.x; partials += blockIdx.x * TM_PSTRIDE;      // one block per source of a paired solve
    if (guard_skip(sc, guard)) return;
    double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
    unsigned int i = threadIdx.x;
    for (; i + 3u * 1024u < n; i += 4u * 1024u) {
        s0 += partials[i]; s1 += partials[i + 1024u]; s2 += partials[i + 2048u]; s3 += partials[i + 3072u];
    }
    for (; i < n; i += 1024u) s0 += partials[i];
    double s = (s0 + s1) + (s2 + s3);
    s = block_sum(s, sm);
    if (threadIdx.x == 0) apply_red_op(sc, op, s);
}
tm_status tm_reduce_finish(tm_ctx* ctx, unsigned int nblocks, int op, int guard, cudaStream_t st) {
    reduce_finish_kernel<<<ctx->nb > 1 ? ctx->nb : 1, 1024, 0, st>>>(ctx->d_partials, nblocks, ctx->d_scal, op, guard);
    TM_LAUNCH_CHECK(ctx, "reduce_finish_kernel");
    return TM_OK;
}

// ------------------------------------------------------------------ complex128 accumulate
__global__ void accumulate_kernel(double* __restrict__ acc, const double* __restrict__ x, size_t n) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) acc[i] += x[i];
}
tm_status tm_accumulate(tm_ctx* ctx, void* d_acc, const void* d_x, size_t n, cudaStream_t st) {
    const size_t nr = 2 * n;
    accumulate_kernel<<<(unsigned)((nr + 255) / 256), 256, 0, st>>>((double*)d_acc, (const double*)d_x, nr);
    TM_LAUNCH_CHECK(ctx, "accumulate_kernel");
    return TM_OK;
}
