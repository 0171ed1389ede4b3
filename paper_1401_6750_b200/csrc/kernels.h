// kernels.h -- internal (non-exported) entry points shared by the translation units of libtmloops.
#pragma once
#include "common.cuh"
#include "blas.cuh"

// ---- dslash.cu ----------------------------------------------------------------------------
// out_p = post( xterm(x) + coef * D_pq in ),  xmode: 0 none | 1 x | 2 A x ; post: 0 none | 1 A^-1
struct DslashCall {
    void* out; const void* in; const void* x;
    int out_parity, dagger;
    double kappa, mu, coef;
    int xmode, post;
    int red_op;        // RED_* applied to ||out||^2 (RED_NONE: no norm)
    int guard;         // GUARD_ALWAYS | GUARD_ITER | GUARD_RU (blas.cuh)
    int mul_in, mul_x, mul_out;   // paired solves: source stride of each operand in parity vectors (0 = 1)
};
tm_status tm_dslash_launch(tm_ctx* ctx, const DslashCall& c, tm_prec prec, tm_recon recon, cudaStream_t st);

// ---- layout.cu ----------------------------------------------------------------------------
tm_status tm_import_launch(tm_ctx* ctx, void* d_internal, const void* d_canon, tm_prec prec, cudaStream_t st);
tm_status tm_export_launch(tm_ctx* ctx, void* d_canon, const void* d_internal, tm_prec prec, cudaStream_t st);
// Z4 noise into a full-lattice internal field: packed exponents (d_z4 != NULL) or counter hash;
// t_only >= 0: restricted to that timeslice (time dilution), zero elsewhere
tm_status tm_z4_expand(tm_ctx* ctx, void* d_internal, tm_prec prec, const unsigned char* d_z4,
                       unsigned long long seed, unsigned long long r, cudaStream_t st, int t_only = -1);

// ---- blas.cu ------------------------------------------------------------------------------
// parity-vector operations (n = 24*Vh reals each); all asynchronous on st
tm_status blas_zero(tm_ctx* ctx, void* v, tm_prec p, cudaStream_t st);
tm_status blas_copy(tm_ctx* ctx, void* dst, tm_prec pd, const void* src, tm_prec ps, cudaStream_t st);
// dst = A^-1 src  (site-local twist inverse)
// (paired solves: *_mul = distance of source 1's vector behind source 0's, in parity vectors: 1 for solver
//  workspaces, 2 for the halves of full-lattice fields, which keep each source's [even][odd] contiguous)
tm_status blas_twist_inv(tm_ctx* ctx, void* dst, const void* src, tm_prec p, double kappa, double mu,
                         int dagger, cudaStream_t st, int dst_mul = 1, int src_mul = 1);
// dst = A^-1 src + c * add
tm_status blas_twist_inv_axpy(tm_ctx* ctx, void* dst, const void* src, const void* add, tm_prec p, double kappa,
                              double mu, double c, cudaStream_t st, int dst_mul = 1, int src_mul = 1, int add_mul = 1);
// ||v||^2 -> red_op
tm_status blas_norm(tm_ctx* ctx, const void* v, tm_prec p, int red_op, cudaStream_t st);
// full-lattice norm (2 parities)
tm_status blas_norm_full(tm_ctx* ctx, const void* v, tm_prec p, int red_op, cudaStream_t st);
// CG kernels driven by the device-resident state (CgScalars); each runs only in its guard state:
//   r -= alpha w ; ||r||^2 -> RED_RR ; sloppy copy rs of r                            (GUARD_ITER)
//   (the x += alpha p of the same iteration is deferred: CgScalars::x_pend)
tm_status blas_update_xr(tm_ctx* ctx, void* r, tm_prec pacc, const void* w, void* rs, tm_prec psl, cudaStream_t st);
//   x += alpha p of the PREVIOUS iteration if pending ; p = z + beta p (p = z when beta == 0: first iteration)  (GUARD_ITER)
tm_status blas_update_p(tm_ctx* ctx, void* p, const void* z, tm_prec psl, void* x, tm_prec pacc, cudaStream_t st);
//   y += x (+ the pending alpha p) ; x = 0                                                    (GUARD_RU)
tm_status blas_ru_begin(tm_ctx* ctx, void* y, tm_prec po, void* x, tm_prec pacc, const void* p, tm_prec psl, cudaStream_t st,
                        int y_mul = 1);
//   r = b - m (acc precision) ; rs = b - m (sloppy) ; ||b - m||^2 -> red_op (RED_START: m == NULL,
//   GUARD_ALWAYS; RED_RU: GUARD_RU)
tm_status blas_residual(tm_ctx* ctx, void* r, tm_prec pacc, void* rs, tm_prec psl, const void* b, const void* m,
                        tm_prec po, int red_op, int guard, cudaStream_t st);
// second stage of a Dslash norm epilogue: sum the nblocks per-block partials, apply red_op (same guard as the Dslash)
tm_status tm_reduce_finish(tm_ctx* ctx, unsigned int nblocks, int op, int guard, cudaStream_t st);
// reset the device state for a new solve (no host synchronisation)
// eta2 > 0: ||eta||^2 known to the caller (Z4 noise: 12 V exactly), no norm kernel needed
tm_status scal_init(tm_ctx* ctx, double rho2, double delta2, int max_iter, double eta2, cudaStream_t st);
tm_status scal_get(tm_ctx* ctx, CgScalars* v /*[TM_MAXNB]*/, cudaStream_t st);   // download + sync

// ---- solver.cu ----------------------------------------------------------------------------
// eta, s: full-lattice internal fields of precision params->outer
struct SolveJob {                       // one solve in flight (solver.cu: tm_solve_begin / tm_solve_end)
    tm_solve_params P;
    int nb;                             // sources solved together (1 | 2 | 4)
    tm_prec po, ps, pa; tm_recon rc;
    double kappa, mu, delta;
    cudaStream_t st;
    void *p, *w, *z, *tmp, *rs, *x, *r, *b, *tmpo, *mo;
    char *y, *s_o; const char* eta_o;
    cudaEvent_t e0, e1, e_scal;
    CgScalars* h_scal;
    bool tail_valid; long enq;
};
// eta_norm2 > 0: ||eta||^2 known exactly to the caller (skips the norm kernel); 0: computed.
// nb = 2 | 4: that many sources solved in lockstep (every kernel launch covers all of them; needs eta_norm2): d_eta
// and d_s hold nb full-lattice fields back to back, tm_solve_end fills info[0..nb-1]
tm_status tm_solve_begin(tm_ctx* ctx, SolveJob* job, void* d_s, const void* d_eta, double kappa, double mu,
                         const tm_solve_params* params, cudaStream_t st, double eta_norm2 = 0.0, int nb = 1);
tm_status tm_solve_end(tm_ctx* ctx, SolveJob* job, tm_solve_info* info);
tm_status tm_solve_internal(tm_ctx* ctx, void* d_s, const void* d_eta, double kappa, double mu,
                            const tm_solve_params* params, tm_solve_info* info, cudaStream_t st);

// ---- contract.cu --------------------------------------------------------------------------
// s, eta: full-lattice internal fields of precision acc (TM_F32 | TM_F64); out: complex128 [2][80][nmom][T]
tm_status tm_contract_internal(tm_ctx* ctx, void* d_out, const void* d_s, const void* d_eta,
                               double kappa, double mu, const int* h_momenta, int nmom, tm_prec acc,
                               cudaStream_t st, int t_first = 0, int nt = 0 /* 0: all timeslices */,
                               int merge = 0);
// merge (whole-vector fp32 calls on the TMA path only: tm_contract_merge_ok): the z-sum and the assembly are linear in
// the x/y partial sums Q, so sources whose loops are only ever ADDED (LP sources without an HP partner, no per-source
// output) can share them: bit 0 = add this source's Q to what the workspace holds, bit 1 = stop after the x/y stage
// (d_out untouched).  A group of n sources calls with merge = 2, 3, ..., 3, 1 and gets the SUM of the n loops in d_out.
bool tm_contract_merge_ok(const tm_ctx* ctx, tm_prec acc);
// contract_tma.cu: TMA-staged fast path of the site + x/y-DFT stage (fp32, Lx <= 32)
bool tm_contract_tma_usable(const tm_ctx* ctx);
// half0: the s-family derivative slots receive only the forward half F_mu (AssembleArgs::half0 restores the rest)
tm_status tm_contract_xy_tma(tm_ctx* ctx, void* qbuf, const void* d_s, const void* d_eta, const void* gauge,
                             const void* wx, const void* wy, int prune, int half0, int t_first, int nt, cudaStream_t st,
                             int q_add = 0);
// contract_mma.cu: the same with the x-stage DFT on the tensor cores (mma.sync tf32, split-fp32 operands)
bool tm_contract_mma_usable(const tm_ctx* ctx);
tm_status tm_contract_xy_mma(tm_ctx* ctx, void* qbuf, const void* d_s, const void* d_eta, const void* gauge,
                             const void* wx, const void* wy, int prune, int t_first, int nt, cudaStream_t st);
void tm_contract_qidx(short* qidx, int prune, int* nq);   // contract.cu: layout of the x/y partial sums Q
// acc += x on complex128 arrays of n complex numbers
tm_status tm_accumulate(tm_ctx* ctx, void* d_acc, const void* d_x, size_t n, cudaStream_t st);
