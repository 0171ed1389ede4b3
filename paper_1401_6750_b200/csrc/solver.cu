// solver.cu -- eq. 2.1: M s = eta by even-odd preconditioned CG on Mhat^dag Mhat
// (SURVEY.md sec 8 rows a2-a5).  CGLS recurrences in `sloppy` storage, x and r accumulated in
// >= fp32, reliable updates and the final true-residual test in `outer` precision.
//
//   Mhat   = A - kappa^2 D_eo A^-1 D_oe            (A = 1 + 2 i kappa mu g5)
//   bhat_e = eta_e + kappa D_eo A^-1 eta_o
//   s_o    = A^-1 (eta_o + kappa D_oe s_e)
// With s_o reconstructed this way eta - M s vanishes on odd sites and equals bhat - Mhat s_e on even
// sites, so ||bhat - Mhat y|| / ||eta|| evaluated in `outer` precision IS the true residual.
//
// Control flow lives on the device (blas.cuh, CgScalars): the last block of every reducing kernel
// computes alpha / beta, decides when to pause for a reliable update and when the solve is over;
// every kernel is guarded by that state.  The host only enqueues:
//   iteration block  (GUARD_ITER)  z = Mhat^dag r ; p = z + beta p ; w = Mhat p ; x += alpha p, r -= alpha w
//   update block     (GUARD_RU)    y += x, x = 0 ; r = bhat - Mhat y in outer precision ; resume | finish
//   tail             (always)      s_o = A^-1 (eta_o + kappa D_oe y)
// along the plan recorded by the previous solve with the same parameters, and reads the state back
// once at the end (one host synchronisation per solve when the plan fits; otherwise it keeps
// enqueueing [iteration, update] pairs and polls).
#include <math.h>
#include "kernels.h"

// out = Mhat in (dagger: Mhat^dag in) on even sites; tmp: odd-parity scratch of the same precision
static tm_status apply_mhat(tm_ctx* ctx, void* out, const void* in, void* tmp, int dagger, double kappa,
                            double mu, tm_prec prec, tm_recon recon, int red_op, int guard, cudaStream_t st) {
    DslashCall k;
    memset(&k, 0, sizeof(k));
    k.kappa = kappa; k.mu = mu; k.dagger = dagger; k.guard = guard;
    k.out = tmp; k.in = in; k.out_parity = 1; k.post = 1; k.coef = 1.0; k.red_op = RED_NONE;
    TM_TRY(tm_dslash_launch(ctx, k, prec, recon, st));
    k.out = out; k.in = tmp; k.x = in; k.out_parity = 0; k.post = 0; k.xmode = 2; k.coef = -kappa * kappa;
    k.red_op = red_op;
    return tm_dslash_launch(ctx, k, prec, recon, st);
}

tm_status tm_solve_internal(tm_ctx* ctx, void* d_s, const void* d_eta, double kappa, double mu,
                            const tm_solve_params* P, tm_solve_info* info, cudaStream_t st) {
    if (!P) return tm_fail(ctx, TM_EARG, "solve: null params");
    const tm_prec po = P->outer, ps = P->sloppy;
    if (po != TM_F64 && po != TM_F32) return tm_fail(ctx, TM_EPREC, "solve: outer precision must be f32 or f64");
    if ((int)ps < 0 || (int)ps > 3) return tm_fail(ctx, TM_EPREC, "solve: unknown sloppy precision");
    if (tm_prec_size(ps) > tm_prec_size(po)) return tm_fail(ctx, TM_EPREC, "solve: sloppy precision wider than outer");
    if (P->recon != TM_R12 && P->recon != TM_R18) return tm_fail(ctx, TM_EARG, "solve: recon must be 12 or 18");
    if (!(P->rho > 0) || P->max_iter < 0) return tm_fail(ctx, TM_EARG, "solve: rho must be > 0, max_iter >= 0");
    const tm_prec pa = (ps == TM_F64) ? TM_F64 : TM_F32;        // accumulate precision of x, r
    const tm_recon rc = P->recon;
    const double delta = (P->delta > 0 && P->delta < 1) ? P->delta : 0.1;
    const size_t bo = tm_parity_bytes(ctx, po), bs = tm_parity_bytes(ctx, ps), ba = tm_parity_bytes(ctx, pa);

    cudaEvent_t e0 = ctx->ev[0], e1 = ctx->ev[1];
    TM_CUDA(ctx, cudaEventRecord(e0, st));

    void *p, *w, *z, *tmp, *rs, *x, *r, *b, *tmpo, *mo;
    TM_TRY(tm_ws(ctx, WS_SL_P, bs, &p));
    TM_TRY(tm_ws(ctx, WS_SL_W, bs, &w));
    TM_TRY(tm_ws(ctx, WS_SL_Z, bs, &z));
    TM_TRY(tm_ws(ctx, WS_SL_TMP, bs, &tmp));
    TM_TRY(tm_ws(ctx, WS_AC_X, ba, &x));
    TM_TRY(tm_ws(ctx, WS_AC_R, ba, &r));
    if (pa != ps) TM_TRY(tm_ws(ctx, WS_SL_R, bs, &rs)); else rs = r;
    TM_TRY(tm_ws(ctx, WS_OU_B, bo, &b));
    TM_TRY(tm_ws(ctx, WS_OU_TMP, bo, &tmpo));
    TM_TRY(tm_ws(ctx, WS_OU_TMP2, bo, &mo));

    const char* eta_e = (const char*)d_eta;
    const char* eta_o = eta_e + bo;
    char* y = (char*)d_s;                  // the even half of the solution is accumulated in place
    char* s_o = y + bo;

    // ---- setup (no host synchronisation): state, ||eta||^2, bhat, y = x = 0, r = rs = bhat
    TM_TRY(scal_init(ctx, P->rho * P->rho, delta * delta, P->max_iter, st));
    TM_TRY(blas_norm_full(ctx, d_eta, po, RED_SLOT0 + 0, st));
    TM_TRY(blas_twist_inv(ctx, tmpo, eta_o, po, kappa, mu, 0, st));
    {
        DslashCall k;
        memset(&k, 0, sizeof(k));
        k.out = b; k.in = tmpo; k.x = eta_e; k.out_parity = 0; k.kappa = kappa; k.mu = mu;
        k.xmode = 1; k.coef = kappa; k.red_op = RED_NONE;
        TM_TRY(tm_dslash_launch(ctx, k, po, rc, st));
    }
    TM_TRY(blas_zero(ctx, y, po, st));
    TM_TRY(blas_zero(ctx, x, pa, st));
    TM_TRY(blas_residual(ctx, r, pa, rs, ps, b, nullptr, po, RED_START, GUARD_ALWAYS, st));

    auto iteration = [&]() -> tm_status {
        TM_TRY(apply_mhat(ctx, z, rs, tmp, 1, kappa, mu, ps, rc, RED_ZZ, GUARD_ITER, st));
        TM_TRY(blas_update_p(ctx, p, z, ps, st));
        TM_TRY(apply_mhat(ctx, w, p, tmp, 0, kappa, mu, ps, rc, RED_WW, GUARD_ITER, st));
        return blas_update_xr(ctx, x, r, pa, p, w, rs, ps, st);
    };
    auto update = [&]() -> tm_status {
        TM_TRY(blas_ru_begin(ctx, y, po, x, pa, st));
        TM_TRY(apply_mhat(ctx, mo, y, tmpo, 0, kappa, mu, po, rc, RED_NONE, GUARD_RU, st));
        return blas_residual(ctx, r, pa, rs, ps, b, mo, po, RED_RU, GUARD_RU, st);
    };
    auto tail = [&]() -> tm_status {
        DslashCall k;
        memset(&k, 0, sizeof(k));
        k.out = s_o; k.in = y; k.x = eta_o; k.out_parity = 1; k.kappa = kappa; k.mu = mu;
        k.xmode = 1; k.post = 1; k.coef = kappa; k.red_op = RED_NONE;
        TM_TRY(tm_dslash_launch(ctx, k, po, rc, st));
        TM_CUDA(ctx, cudaEventRecord(e1, st));
        return TM_OK;
    };

    CgPlan& plan = ctx->plan[(int)ps];
    const bool have_plan = plan.valid && plan.sloppy == (int)ps && plan.outer == (int)po && plan.recon == (int)rc
                        && plan.max_iter == P->max_iter && plan.rho == P->rho && plan.delta == delta;
    CgScalars sc;
    bool tail_valid = false;
    long enq = 0;                                   // iteration blocks enqueued so far
    if (have_plan) {
        for (int k = 0; k < plan.n_pause; k++) {
            for (; enq < plan.pause_iter[k]; enq++) TM_TRY(iteration());
            TM_TRY(update());
        }
        TM_TRY(tail());
        tail_valid = true;
    } else {
        TM_TRY(update());                           // covers "already converged at x = 0" (state 1 after RED_START)
    }
    TM_TRY(scal_get(ctx, &sc, st));
    while (sc.done < 2) {
        // off plan (first solve with these parameters, or this source behaves differently):
        // [iteration, update] pairs, polled every few pairs
        const int burst = 4;
        for (int k = 0; k < burst; k++) { TM_TRY(iteration()); TM_TRY(update()); enq++; }
        tail_valid = false;
        TM_TRY(scal_get(ctx, &sc, st));
        if (enq > (long)P->max_iter + 8 * (long)CG_MAX_PAUSES + 64 && sc.done < 2)
            return tm_fail(ctx, TM_ECUDA, "solve: device state machine did not terminate");
    }
    if (!tail_valid) {
        TM_TRY(tail());
        TM_CUDA(ctx, cudaEventSynchronize(e1));
    }
    // remember where this solve paused: the launch plan of the next one
    plan.valid = sc.n_ru <= CG_MAX_PAUSES;
    plan.sloppy = (int)ps; plan.outer = (int)po; plan.recon = (int)rc; plan.max_iter = P->max_iter;
    plan.rho = P->rho; plan.delta = delta;
    plan.n_pause = sc.n_ru < CG_MAX_PAUSES ? sc.n_ru : CG_MAX_PAUSES;
    for (int k = 0; k < plan.n_pause; k++) plan.pause_iter[k] = sc.pause_iter[k];

    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    const double eta2 = sc.slot[0];
    const double resid = eta2 > 0 ? sqrt(sc.rr_true / eta2) : 0.0;
    if (info) {
        info->iters = sc.iters;
        info->reliable_updates = sc.n_ru;
        info->true_resid = resid;
        info->ms = ms;
    }
    if (sc.done != 2) {
        snprintf(ctx->err, sizeof(ctx->err), "solve: rho = %g not reached in %d iterations (true residual %g)",
                 P->rho, sc.iters, resid);
        return TM_ENOCONV;
    }
    return TM_OK;
}

extern "C" tm_status tm_cg_solve(tm_ctx* ctx, void* d_s, const void* d_eta, double kappa, double mu,
                                 const tm_solve_params* params, tm_solve_info* info, void* stream) {
    if (!ctx || !d_s || !d_eta || !params) return tm_fail(ctx, TM_EARG, "tm_cg_solve: null argument");
    cudaStream_t st = (cudaStream_t)stream;
    TM_CUDA(ctx, cudaSetDevice(ctx->device));
    const tm_prec po = params->outer;
    if (po != TM_F64 && po != TM_F32) return tm_fail(ctx, TM_EPREC, "tm_cg_solve: outer precision must be f32 or f64");
    void *eta_i, *s_i;
    TM_TRY(tm_ws(ctx, WS_OU_ETA, 2 * tm_parity_bytes(ctx, po), &eta_i));
    TM_TRY(tm_ws(ctx, WS_OU_S, 2 * tm_parity_bytes(ctx, po), &s_i));
    TM_TRY(tm_import_launch(ctx, eta_i, d_eta, po, st));
    tm_status s = tm_solve_internal(ctx, s_i, eta_i, kappa, mu, params, info, st);
    if (s != TM_OK && s != TM_ENOCONV) return s;
    TM_TRY(tm_export_launch(ctx, d_s, s_i, po, st));
    TM_CUDA(ctx, cudaStreamSynchronize(st));
    return s;
}
