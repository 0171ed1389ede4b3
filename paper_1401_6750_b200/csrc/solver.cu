// solver.cu -- eq. 2.1: M s = eta by even-odd preconditioned CG on Mhat^dag Mhat
// (SURVEY.md sec 8 rows a2-a5).  CGLS recurrences in `sloppy` storage, x and r accumulated in
// >= fp32, reliable updates and the final true-residual test in `outer` precision.
//
//   Mhat   = A - kappa^2 D_eo A^-1 D_oe            (A = 1 + 2 i kappa mu g5)
//   bhat_e = eta_e + kappa D_eo A^-1 eta_o
//   s_o    = A^-1 (eta_o + kappa D_oe s_e)
// With s_o reconstructed this way eta - M s vanishes on odd sites and equals bhat - Mhat s_e on even
// sites, so ||bhat - Mhat y|| / ||eta|| evaluated in `outer` precision IS the true residual.
#include <math.h>
#include "kernels.h"

struct MhatWork { void* tmp; };

// out = Mhat in (dagger: Mhat^dag in) on even sites; tmp: odd-parity scratch of the same precision
static tm_status apply_mhat(tm_ctx* ctx, void* out, const void* in, void* tmp, int dagger, double kappa,
                            double mu, tm_prec prec, tm_recon recon, int red_op, int check_done, cudaStream_t st) {
    DslashCall k;
    memset(&k, 0, sizeof(k));
    k.kappa = kappa; k.mu = mu; k.dagger = dagger; k.check_done = check_done;
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

    void *p, *w, *z, *tmp, *rs, *x, *r, *y, *b, *ro, *tmpo, *mo;
    TM_TRY(tm_ws(ctx, WS_SL_P, bs, &p));
    TM_TRY(tm_ws(ctx, WS_SL_W, bs, &w));
    TM_TRY(tm_ws(ctx, WS_SL_Z, bs, &z));
    TM_TRY(tm_ws(ctx, WS_SL_TMP, bs, &tmp));
    TM_TRY(tm_ws(ctx, WS_AC_X, ba, &x));
    TM_TRY(tm_ws(ctx, WS_AC_R, ba, &r));
    if (pa != ps) TM_TRY(tm_ws(ctx, WS_SL_R, bs, &rs)); else rs = r;
    TM_TRY(tm_ws(ctx, WS_OU_Y, bo, &y));
    TM_TRY(tm_ws(ctx, WS_OU_B, bo, &b));
    TM_TRY(tm_ws(ctx, WS_OU_R, bo, &ro));
    TM_TRY(tm_ws(ctx, WS_OU_TMP, bo, &tmpo));
    TM_TRY(tm_ws(ctx, WS_OU_TMP2, bo, &mo));

    const char* eta_e = (const char*)d_eta;
    const char* eta_o = eta_e + bo;
    char* s_e = (char*)d_s;
    char* s_o = s_e + bo;

    CgScalars sc;
    memset(&sc, 0, sizeof(sc));
    TM_TRY(scal_set(ctx, sc, st));

    // ||eta||^2 ; bhat = eta_e + kappa D_eo A^-1 eta_o
    TM_TRY(blas_norm_full(ctx, d_eta, po, RED_SLOT0 + 0, st));
    TM_TRY(blas_twist_inv(ctx, tmpo, eta_o, po, kappa, mu, 0, st));
    {
        DslashCall k;
        memset(&k, 0, sizeof(k));
        k.out = b; k.in = tmpo; k.x = eta_e; k.out_parity = 0; k.kappa = kappa; k.mu = mu;
        k.xmode = 1; k.coef = kappa; k.red_op = RED_SLOT0 + 1;
        TM_TRY(tm_dslash_launch(ctx, k, po, rc, st));
    }
    TM_TRY(scal_get(ctx, &sc, st));
    const double eta2 = sc.slot[0];
    int iters = 0, n_ru = 0, converged = 0;
    double rr_true = sc.slot[1];
    TM_TRY(blas_zero(ctx, y, po, st));
    if (eta2 == 0.0) {
        converged = 1; rr_true = 0.0;
    } else {
        const double target2 = P->rho * P->rho * eta2;
        if (rr_true <= target2) converged = 1;
        if (!converged) {
            TM_TRY(scal_set_done_target(ctx, 0, target2, st));
            TM_TRY(blas_copy(ctx, ro, po, b, po, st));
            TM_TRY(blas_zero(ctx, x, pa, st));
            TM_TRY(blas_copy(ctx, r, pa, ro, po, st));
            if (pa != ps) TM_TRY(blas_copy(ctx, rs, ps, ro, po, st));
            // z = Mhat^dag r ; p = z ; gamma = ||z||^2
            TM_TRY(apply_mhat(ctx, z, rs, tmp, 1, kappa, mu, ps, rc, RED_ZZ_INIT, 0, st));
            TM_TRY(blas_copy(ctx, p, ps, z, ps, st));
            double rr_ru = rr_true;
            while (true) {
                // w = Mhat p ; alpha = gamma / ||w||^2
                TM_TRY(apply_mhat(ctx, w, p, tmp, 0, kappa, mu, ps, rc, RED_WW, 1, st));
                // x += alpha p ; r -= alpha w ; rr
                TM_TRY(blas_update_xr(ctx, x, r, pa, p, w, rs, ps, st));
                TM_TRY(scal_get(ctx, &sc, st));
                iters = sc.iters;
                const bool out_of_iters = iters >= P->max_iter;
                if (sc.done || out_of_iters || sc.rr <= delta * delta * rr_ru || !(sc.rr == sc.rr)) {
                    // reliable update: y += x ; x = 0 ; r = bhat - Mhat y in outer precision
                    TM_TRY(blas_axpy1(ctx, y, po, x, pa, st));
                    TM_TRY(blas_zero(ctx, x, pa, st));
                    TM_TRY(apply_mhat(ctx, mo, y, tmpo, 0, kappa, mu, po, rc, RED_NONE, 0, st));
                    TM_TRY(blas_xmy_norm(ctx, ro, b, mo, po, RED_SLOT0 + 2, st));
                    TM_TRY(scal_get(ctx, &sc, st));
                    rr_true = sc.slot[2];
                    n_ru++;
                    if (rr_true <= target2) { converged = 1; break; }
                    if (out_of_iters || !(rr_true == rr_true)) break;
                    rr_ru = rr_true;
                    TM_TRY(scal_set_done_target(ctx, 0, target2, st));
                    TM_TRY(blas_copy(ctx, r, pa, ro, po, st));
                    if (pa != ps) TM_TRY(blas_copy(ctx, rs, ps, ro, po, st));
                }
                // z = Mhat^dag r ; beta = ||z||^2 / gamma ; p = z + beta p
                TM_TRY(apply_mhat(ctx, z, rs, tmp, 1, kappa, mu, ps, rc, RED_ZZ, 1, st));
                TM_TRY(blas_update_p(ctx, p, z, ps, st));
            }
        }
    }
    // s_e = y ; s_o = A^-1 (eta_o + kappa D_oe s_e)
    TM_TRY(blas_copy(ctx, s_e, po, y, po, st));
    {
        DslashCall k;
        memset(&k, 0, sizeof(k));
        k.out = s_o; k.in = y; k.x = eta_o; k.out_parity = 1; k.kappa = kappa; k.mu = mu;
        k.xmode = 1; k.post = 1; k.coef = kappa; k.red_op = RED_NONE;
        TM_TRY(tm_dslash_launch(ctx, k, po, rc, st));
    }
    TM_CUDA(ctx, cudaEventRecord(e1, st));
    TM_CUDA(ctx, cudaEventSynchronize(e1));
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    if (info) {
        info->iters = iters;
        info->reliable_updates = n_ru;
        info->true_resid = eta2 > 0 ? sqrt(rr_true / eta2) : 0.0;
        info->ms = ms;
    }
    if (!converged) {
        snprintf(ctx->err, sizeof(ctx->err), "solve: rho = %g not reached in %d iterations (true residual %g)",
                 P->rho, iters, eta2 > 0 ? sqrt(rr_true / eta2) : 0.0);
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
