// hpe.cu -- Hopping Parameter Expansion of the plain loop estimator ("... time-dilution and the Hopping
// Parameter Expansion (HPE) [7], and all the possible combinations of these"; reading 23).
//
// With the site-local A = 1 + 2 i kappa mu g5 and the hopping part H = A - M = kappa D,
//     M^-1 = sum_{k<n} (A^-1 H)^k A^-1 + (A^-1 H)^n M^-1        exactly, for every n,
// so the loop tr[X_i M^-1] is an exact part plus a remainder that the SAME solution s = M^-1 eta estimates:
//     l_i = eta^dag X_i (A^-1 H)^{n_i} s  +  E_i,      n_i = order (<= 4) for X_i = G_n,  min(order, 2) for X_i = G_n D_m.
// Per source this costs n applications of the hopping term (two parity Dslash launches each, twist inverse in the
// epilogue) and one or two plain contractions (the primitive of contract.cu with the pair swapped and mu = 0, as in
// dilution.cu).  Up to these orders E_i is site- and gauge-independent (every extent >= 4): closed forms below, built
// by multiplying out the 4 x 4 matrices on the host -- the oracle gets the same numbers by brute force over the 12 V
// unit vectors.
#include <math.h>
#include <complex>
#include <vector>
#include "kernels.h"

typedef std::complex<double> cd;
struct M4 { cd m[4][4]; };
static M4 m4_mul(const M4& a, const M4& b) {
    M4 c;
    for (int i = 0; i < 4; i++)
        for (int j = 0; j < 4; j++) {
            cd s = 0;
            for (int k = 0; k < 4; k++) s += a.m[i][k] * b.m[k][j];
            c.m[i][j] = s;
        }
    return c;
}
static M4 m4_lin(cd x, const M4& a, cd y, const M4& b) {
    M4 c;
    for (int i = 0; i < 4; i++)
        for (int j = 0; j < 4; j++) c.m[i][j] = x * a.m[i][j] + y * b.m[i][j];
    return c;
}
static cd m4_tr(const M4& a) { return a.m[0][0] + a.m[1][1] + a.m[2][2] + a.m[3][3]; }

// E[i] per site of a timeslice (p = 0), i = 0..79; chiral basis of dslash.cu: g_mu = [[0, B],[B^dag, 0]], B_k = -i s_k, B_t = 1
static void hpe_constants(double kappa, double mu, int n_loc, int n_der, cd* E) {
    const cd I(0, 1);
    cd sig[4][2][2] = {{{0, 1}, {1, 0}}, {{0, -I}, {I, 0}}, {{1, 0}, {0, -1}}, {{1, 0}, {0, 1}}};
    M4 one, gam[4], g5;
    memset(&one, 0, sizeof(one));
    for (int i = 0; i < 4; i++) one.m[i][i] = 1;
    for (int m = 0; m < 4; m++) {
        memset(&gam[m], 0, sizeof(M4));
        for (int i = 0; i < 2; i++)
            for (int j = 0; j < 2; j++) {
                const cd Bm = (m < 3) ? -I * sig[m][i][j] : sig[3][i][j];
                gam[m].m[i][2 + j] = Bm;
                gam[m].m[2 + j][i] = std::conj(Bm);
            }
    }
    g5 = one;
    for (int m = 0; m < 4; m++) g5 = m4_mul(g5, gam[m]);
    const double a = 2.0 * kappa * mu;
    const M4 B = m4_lin(1.0 / (1.0 + a * a), one, -I * a / (1.0 + a * a), g5);          // A^-1
    // sum over mu of the two out-and-back paths: (1 - g) B (1 + g) + (1 + g) B (1 - g)
    M4 back;
    memset(&back, 0, sizeof(back));
    for (int m = 0; m < 4; m++) {
        const M4 pm = m4_lin(1, one, -1, gam[m]), pp = m4_lin(1, one, 1, gam[m]);
        back = m4_lin(1, back, 1, m4_lin(1, m4_mul(m4_mul(pm, B), pp), 1, m4_mul(m4_mul(pp, B), pm)));
    }
    for (int n = 0; n < 16; n++) {
        M4 G = one;
        for (int m = 0; m < 4; m++)
            if ((n >> m) & 1) G = m4_mul(G, gam[m]);
        const M4 GB = m4_mul(G, B);
        cd e = 0;
        if (n_loc >= 1) e += 3.0 * m4_tr(GB);
        if (n_loc >= 3) e += 3.0 * kappa * kappa * m4_tr(m4_mul(m4_mul(GB, back), B));
        E[n] = e;
        for (int m = 0; m < 4; m++)
            E[16 + 16 * m + n] = n_der >= 2 ? 3.0 * kappa * m4_tr(m4_mul(m4_mul(GB, gam[m]), B)) : cd(0);
    }
}

// v = eps_n * prim[f = 1][idx] from prim_loc (i < 16) or prim_der, plus E_i * sites at the p = 0 entries;
// dst = v | acc0 += v | acc1 += v | copy = v   (as plain_assemble_kernel of dilution.cu)
__global__ void hpe_assemble_kernel(double2* __restrict__ dst, double2* __restrict__ acc0, double2* __restrict__ acc1,
                                    double2* __restrict__ copy, const double2* __restrict__ prim_loc,
                                    const double2* __restrict__ prim_der, const double2* __restrict__ E,
                                    const unsigned char* __restrict__ pzero, size_t per_f, int nmom, int T) {
    const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= per_f) return;
    const int i = (int)(idx / ((size_t)nmom * T));
    const int k = (int)((idx / T) % nmom);
    const int n = i < 16 ? i : (i - 16) & 15;
    const double eps = (__popc(n) & 1) ? -1.0 : 1.0;
    double2 v = (i < 16 ? prim_loc : prim_der)[per_f + idx];
    v.x *= eps; v.y *= eps;
    if (pzero[k]) { const double2 e = E[i]; v.x += e.x; v.y += e.y; }
    if (dst) dst[idx] = v;
    if (acc0) { double2 a = acc0[idx]; a.x += v.x; a.y += v.y; acc0[idx] = a; }
    if (acc1) { double2 a = acc1[idx]; a.x += v.x; a.y += v.y; acc1[idx] = a; }
    if (copy) copy[idx] = v;
}
__global__ void hpe_combine_kernel(double* __restrict__ out, const double* __restrict__ sums, double inv_lp, double inv_hp,
                                   size_t n) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    out[i] = sums[i] * inv_lp + (sums[2 * n + i] - sums[n + i]) * inv_hp;
}

// out = A^-1 H in on full-lattice internal fields: out_p = A^-1 (kappa D_pq in_q), p = 0, 1
static tm_status hpe_hop(tm_ctx* ctx, void* out, const void* in, double kappa, double mu, tm_prec prec, cudaStream_t st) {
    const size_t pb = tm_parity_bytes(ctx, prec);
    const tm_recon rc = prec == TM_F64 ? TM_R18 : TM_R12;
    for (int p = 0; p < 2; p++) {
        DslashCall k;
        memset(&k, 0, sizeof(k));
        k.out = (char*)out + p * pb; k.in = (const char*)in + (1 - p) * pb;
        k.out_parity = p; k.xmode = 0; k.post = 1; k.coef = kappa; k.kappa = kappa; k.mu = mu; k.red_op = RED_NONE;
        TM_TRY(tm_dslash_launch(ctx, k, prec, rc, st));
    }
    return TM_OK;
}

struct HpeTables {              // device block: E[80] complex, then one flag per momentum (p == 0)
    double2* E;
    unsigned char* pzero;
};
static tm_status hpe_orders(tm_ctx* ctx, int order, int* n_loc, int* n_der) {
    if (order < 0 || order > 4) return tm_fail(ctx, TM_EARG, "hpe: order must be 0..4");
    for (int d = 0; d < 4; d++)
        if (order > 0 && ctx->X[d] < 4)
            return tm_fail(ctx, TM_EDIM, "hpe: every extent must be >= 4 (shorter paths close around the torus)");
    *n_loc = order; *n_der = order < 2 ? order : 2;
    return TM_OK;
}
static tm_status hpe_tables(tm_ctx* ctx, HpeTables* Tb, double kappa, double mu, int n_loc, int n_der, const int* h_momenta,
                            int nmom, cudaStream_t st) {
    std::vector<unsigned char> host(80 * 16 + (size_t)nmom);
    cd E[80];
    hpe_constants(kappa, mu, n_loc, n_der, E);
    const double n3 = (double)ctx->X[0] * ctx->X[1] * ctx->X[2];
    for (int i = 0; i < 80; i++) { ((double*)host.data())[2 * i] = n3 * E[i].real(); ((double*)host.data())[2 * i + 1] = n3 * E[i].imag(); }
    for (int k = 0; k < nmom; k++)
        host[80 * 16 + k] = (h_momenta[3 * k] == 0 && h_momenta[3 * k + 1] == 0 && h_momenta[3 * k + 2] == 0) ? 1 : 0;
    void* d;
    TM_TRY(tm_ws(ctx, WS_HPE_TAB, host.size(), &d));
    TM_CUDA(ctx, cudaMemcpyAsync(d, host.data(), host.size(), cudaMemcpyHostToDevice, st));
    TM_CUDA(ctx, cudaStreamSynchronize(st));              // host is a local vector
    Tb->E = (double2*)d;
    Tb->pzero = (unsigned char*)d + 80 * 16;
    return TM_OK;
}

// the two remainders of one (eta, s) pair in internal layout, precision acc: prim_loc / prim_der = primitive arrays
// [2][80][nmom][T] of (eta, (A^-1 H)^{n_loc} s) and (eta, (A^-1 H)^{n_der} s); prim_der == prim_loc when the orders agree
static tm_status hpe_remainders(tm_ctx* ctx, void** prim_loc, void** prim_der, const void* eta_i, const void* s_i,
                                double kappa, double mu, int n_loc, int n_der, const int* h_momenta, int nmom, tm_prec acc,
                                cudaStream_t st) {
    const size_t fb = 2 * tm_parity_bytes(ctx, acc);
    const size_t nprim = (size_t)2 * 80 * nmom * ctx->X[3] * 16;
    void *va, *vb, *pl, *pd;
    TM_TRY(tm_ws(ctx, WS_HPE_A, fb, &va));
    TM_TRY(tm_ws(ctx, WS_HPE_B, fb, &vb));
    TM_TRY(tm_ws(ctx, WS_TD_PRIM, 2 * nprim, &pl));
    pd = (char*)pl + nprim;
    const void* v = s_i;
    const void* v_der = s_i;
    for (int k = 1; k <= n_loc; k++) {
        void* o = (k & 1) ? va : vb;
        TM_TRY(hpe_hop(ctx, o, v, kappa, mu, acc, st));
        v = o;
        if (k == n_der) {
            if (n_loc > n_der + 1) {            // va is overwritten two steps later: keep the order-n_der vector
                void* keep;
                TM_TRY(tm_ws(ctx, WS_HPE_C, fb, &keep));
                TM_CUDA(ctx, cudaMemcpyAsync(keep, o, fb, cudaMemcpyDeviceToDevice, st));
                v_der = keep;
            } else v_der = o;
        }
    }
    if (n_der == 0) v_der = s_i;
    // plain bilinears eta^dag X_i v from the primitive with the pair swapped and mu = 0 (dilution.cu)
    TM_TRY(tm_contract_internal(ctx, pl, eta_i, v, 0.0, 0.0, h_momenta, nmom, acc, st));
    *prim_loc = pl;
    if (n_der == n_loc) *prim_der = pl;
    else {
        TM_TRY(tm_contract_internal(ctx, pd, eta_i, v_der, 0.0, 0.0, h_momenta, nmom, acc, st));
        *prim_der = pd;
    }
    return TM_OK;
}

extern "C" tm_status loop_hpe_project(tm_ctx* ctx, void* d_out, const void* d_eta, const void* d_s, double kappa, double mu,
                                      const int* h_momenta, int nmom, int order, tm_prec acc, void* stream) {
    if (!ctx || !d_out || !d_eta || !d_s) return tm_fail(ctx, TM_EARG, "loop_hpe_project: null argument");
    if (acc != TM_F64 && acc != TM_F32) return tm_fail(ctx, TM_EPREC, "loop_hpe_project: acc must be f32 or f64");
    if (nmom < 1 || !h_momenta) return tm_fail(ctx, TM_EARG, "loop_hpe_project: need at least one momentum");
    int n_loc, n_der;
    TM_TRY(hpe_orders(ctx, order, &n_loc, &n_der));
    cudaStream_t st = (cudaStream_t)stream;
    TM_CUDA(ctx, cudaSetDevice(ctx->device));
    const size_t per_f = (size_t)80 * nmom * ctx->X[3];
    void *ei, *si, *pl, *pd;
    TM_TRY(tm_ws(ctx, WS_CT_ETA, 2 * tm_parity_bytes(ctx, acc), &ei));
    TM_TRY(tm_ws(ctx, WS_CT_S, 2 * tm_parity_bytes(ctx, acc), &si));
    TM_TRY(tm_import_launch(ctx, ei, d_eta, acc, st));
    TM_TRY(tm_import_launch(ctx, si, d_s, acc, st));
    HpeTables Tb;
    TM_TRY(hpe_tables(ctx, &Tb, kappa, mu, n_loc, n_der, h_momenta, nmom, st));
    TM_TRY(hpe_remainders(ctx, &pl, &pd, ei, si, kappa, mu, n_loc, n_der, h_momenta, nmom, acc, st));
    hpe_assemble_kernel<<<(unsigned)((per_f + 255) / 256), 256, 0, st>>>((double2*)d_out, nullptr, nullptr, nullptr,
                                                                        (const double2*)pl, (const double2*)pd, Tb.E, Tb.pzero,
                                                                        per_f, nmom, ctx->X[3]);
    TM_LAUNCH_CHECK(ctx, "hpe_assemble_kernel");
    return TM_OK;
}

// full-lattice field precision conversion (two parity blocks)
static tm_status hpe_convert_full(tm_ctx* ctx, void* dst, tm_prec pd, const void* src, tm_prec ps, cudaStream_t st) {
    for (int p = 0; p < 2; p++)
        TM_TRY(blas_copy(ctx, (char*)dst + p * tm_parity_bytes(ctx, pd), pd,
                         (const char*)src + p * tm_parity_bytes(ctx, ps), ps, st));
    return TM_OK;
}

extern "C" tm_status tsm_estimate_hpe(tm_ctx* ctx, void* d_out, void* d_per_source, const tsm_params* P, int order,
                                      tsm_info* info, void* stream) {
    if (!ctx) return TM_EARG;
    if (!P || !d_out) return tm_fail(ctx, TM_EARG, "tsm_estimate_hpe: null argument");
    if (P->n_lp < 1 || P->n_hp < 0 || P->n_hp > P->n_lp)
        return tm_fail(ctx, TM_EARG, "tsm_estimate_hpe: need 1 <= n_lp and 0 <= n_hp <= n_lp");
    if (P->nmom < 1 || !P->h_momenta) return tm_fail(ctx, TM_EARG, "tsm_estimate_hpe: need at least one momentum");
    if (P->src_first < 0 || P->src_stride < 0) return tm_fail(ctx, TM_EARG, "tsm_estimate_hpe: src_first and src_stride must be >= 0");
    for (int pass = 0; pass < (P->n_hp ? 2 : 1); pass++) {
        const tm_prec po = pass ? P->hp.outer : P->lp.outer, ac = pass ? P->contract_acc_hp : P->contract_acc_lp;
        if (po != TM_F32 && po != TM_F64) return tm_fail(ctx, TM_EPREC, "tsm_estimate_hpe: outer precisions must be f32 or f64");
        if (ac != TM_F32 && ac != TM_F64) return tm_fail(ctx, TM_EPREC, "tsm_estimate_hpe: contraction precisions must be f32 or f64");
    }
    int n_loc, n_der;
    TM_TRY(hpe_orders(ctx, order, &n_loc, &n_der));
    cudaStream_t st = (cudaStream_t)stream;
    TM_CUDA(ctx, cudaSetDevice(ctx->device));
    TM_TRY(tm_lane_use(ctx, 0));
    const long launches0 = ctx->launches;
    const int T = ctx->X[3];
    const size_t per_f = (size_t)80 * P->nmom * T;            // complex entries of one per-source array
    const size_t nrd = 2 * per_f;                             // doubles
    const unsigned agrid = (unsigned)((per_f + 255) / 256);
    const long stride = P->src_stride > 0 ? P->src_stride : 1;
    int group = ctx->opt_group ? ctx->opt_group : TM_MAXNB;
    {
        size_t free_b = 0, total_b = 0;
        TM_CUDA(ctx, cudaMemGetInfo(&free_b, &total_b));
        const tm_solve_params& big = P->n_hp ? P->hp : P->lp;
        const double need = 7.0 * (double)tm_parity_bytes(ctx, big.outer) + 7.0 * (double)tm_parity_bytes(ctx, TM_F32);
        while (!ctx->opt_group && group > 1 && (double)group * need > 0.45 * (double)total_b) group /= 2;
    }
    HpeTables Tb;
    TM_TRY(hpe_tables(ctx, &Tb, P->kappa, P->mu, n_loc, n_der, P->h_momenta, P->nmom, st));
    double* sums;
    TM_TRY(tm_ws(ctx, WS_TD_ACC, 3 * nrd * sizeof(double), (void**)&sums));
    TM_CUDA(ctx, cudaMemsetAsync(sums, 0, 3 * nrd * sizeof(double), st));
    double2* S_lp = (double2*)sums, *S_lpc = S_lp + per_f, *S_hp = S_lp + 2 * per_f;
    cudaEvent_t e0 = ctx->ev[2], e1 = ctx->ev[3];
    TM_CUDA(ctx, cudaEventRecord(e0, st));
    double ms_lp = 0, ms_hp = 0, worst_lp = 0, worst_hp = 0;
    long it_lp = 0, it_hp = 0;
    int noconv = 0;
    const size_t z4_bytes = 3 * ctx->V;
    for (int pass = 0; pass < (P->n_hp ? 2 : 1); pass++) {
        const int nsrc = pass ? P->n_hp : P->n_lp;
        const tm_solve_params* sp = pass ? &P->hp : &P->lp;
        const tm_prec po = sp->outer, ac = pass ? P->contract_acc_hp : P->contract_acc_lp;
        const size_t fbo = 2 * tm_parity_bytes(ctx, po), fba = 2 * tm_parity_bytes(ctx, ac);
        void *eta_o, *s_o;
        TM_TRY(tm_ws(ctx, po == TM_F32 ? WS_TSM_ETA32 : WS_TSM_ETA64, TM_MAXNB * fbo, &eta_o));
        TM_TRY(tm_ws(ctx, po == TM_F32 ? WS_TSM_S32 : WS_TSM_S64, TM_MAXNB * fbo, &s_o));
        for (int r0 = 0; r0 < nsrc;) {
            int nb = 1;
            while (2 * nb <= nsrc - r0 && 2 * nb <= group && 2 * nb <= TM_MAXNB) nb *= 2;
            for (int b = 0; b < nb; b++) {
                const int r = r0 + b;
                TM_TRY(tm_z4_expand(ctx, (char*)eta_o + (size_t)b * fbo, po, P->d_z4 ? P->d_z4 + (size_t)r * z4_bytes : nullptr,
                                    P->seed, (unsigned long long)(P->src_first + (long)r * stride), st));
            }
            SolveJob sj;
            TM_TRY(tm_solve_begin(ctx, &sj, s_o, eta_o, P->kappa, P->mu, sp, st, 12.0 * (double)ctx->V, nb));
            tm_solve_info si[TM_MAXNB];
            tm_status s = tm_solve_end(ctx, &sj, si);
            if (s != TM_OK && s != TM_ENOCONV) return s;
            for (int b = 0; b < nb; b++) {
                const int r = r0 + b;
                if (pass) { ms_hp += si[b].ms; it_hp += si[b].iters; worst_hp = fmax(worst_hp, si[b].true_resid); }
                else      { ms_lp += si[b].ms; it_lp += si[b].iters; worst_lp = fmax(worst_lp, si[b].true_resid); }
                if (!(si[b].true_resid <= sp->rho * (1.0 + 1e-12))) noconv++;
                void *s_c = (char*)s_o + (size_t)b * fbo, *eta_c = (char*)eta_o + (size_t)b * fbo;
                if (ac != po) {
                    void *sbuf, *ebuf;
                    TM_TRY(tm_ws(ctx, WS_CT_S, fba, &sbuf));
                    TM_TRY(tm_ws(ctx, WS_CT_ETA, fba, &ebuf));
                    TM_TRY(hpe_convert_full(ctx, sbuf, ac, s_c, po, st));
                    TM_TRY(hpe_convert_full(ctx, ebuf, ac, eta_c, po, st));
                    s_c = sbuf; eta_c = ebuf;
                }
                void *pl, *pd;
                TM_TRY(hpe_remainders(ctx, &pl, &pd, eta_c, s_c, P->kappa, P->mu, n_loc, n_der, P->h_momenta, P->nmom, ac, st));
                double2* copy = d_per_source ? (double2*)d_per_source + (size_t)(pass ? P->n_lp + r : r) * per_f : nullptr;
                hpe_assemble_kernel<<<agrid, 256, 0, st>>>(nullptr, pass ? S_hp : S_lp, (!pass && r < P->n_hp) ? S_lpc : nullptr, copy,
                                                           (const double2*)pl, (const double2*)pd, Tb.E, Tb.pzero, per_f, P->nmom, T);
                TM_LAUNCH_CHECK(ctx, "hpe_assemble_kernel");
            }
            r0 += nb;
        }
    }
    hpe_combine_kernel<<<(unsigned)((nrd + 255) / 256), 256, 0, st>>>((double*)d_out, sums, 1.0 / P->n_lp,
                                                                     P->n_hp ? 1.0 / P->n_hp : 0.0, nrd);
    TM_LAUNCH_CHECK(ctx, "hpe_combine_kernel");
    TM_CUDA(ctx, cudaEventRecord(e1, st));
    TM_CUDA(ctx, cudaEventSynchronize(e1));
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    if (info) {
        info->ms_total = ms; info->ms_lp_solve = ms_lp; info->ms_hp_solve = ms_hp;
        info->ms_contract = ms - ms_lp - ms_hp;
        info->iters_lp = it_lp; info->iters_hp = it_hp;
        info->worst_resid_lp = worst_lp; info->worst_resid_hp = worst_hp;
        info->launches = (int)(ctx->launches - launches0);
        info->lanes = 1;
    }
    if (noconv) {
        snprintf(ctx->err, sizeof(ctx->err), "tsm_estimate_hpe: %d solve(s) missed their rho (worst LP %g, HP %g)",
                 noconv, worst_lp, worst_hp);
        return TM_ENOCONV;
    }
    return TM_OK;
}
