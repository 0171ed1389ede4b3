/* tmloops.h -- C ABI of the B200-native Truncated-Solver-Method loop estimator.
 *
 * One shared library (libtmloops.so, sm_100a) implementing the data-parallel hot path of
 * arXiv:1401.6750 ("A QUDA-branch to compute disconnected diagrams in GPUs"):
 *   eq. 2.1     M |s_r> = |eta_r>                          -> tm_cg_solve
 *   sec 2.1  Truncated Solver Method, N_LP + N_HP        -> tsm_estimate
 *   sec 2.1.1     one-end trick, 160 insertions, p^2 <= 9     -> loop_contract_project
 *   sec 2.2  colour-traced contraction, covariant derivative, time-slice array
 *   [B:ns] = BASELINE.json north_star: the operator
 *     M = (1 + 2 i kappa mu gamma5 tau3) - kappa sum_mu [(1-gamma_mu) U_mu(x) d_{x+mu,y}
 *                                                      + (1+gamma_mu) U_mu^dag(x-mu) d_{x-mu,y}]  -> tm_dslash
 *
 * No CUDA or torch types: device pointers are plain void* ("d_" prefix = device memory,
 * "h_" = host memory), streams are void* holding a cudaStream_t (NULL = default stream).
 *
 * Conventions: dims = {Lx,Ly,Lz,T}, all even; canonical site index
 * ((t*Lz+z)*Ly+y)*Lx+x; directions mu = 0..3 = x,y,z,t; parity = (x+y+z+t)&1;
 * canonical spinor  complex128 [V][4 spin][3 colour]; canonical gauge complex128 [V][4 mu][3][3];
 * Hermitian chiral gamma basis, gamma5 = diag(1,1,-1,-1); periodic in space,
 * psi(t+T) = t_boundary * psi(t).  tau3 -> +1; pass mu < 0 for the other flavour.
 *
 * Internal fields (what tm_dslash works on, so a timed loop holds nothing but the kernel):
 * per parity, [24/CV chunks][V/2 sites] vectors of 16 bytes (CV = 2/4/8 reals for
 * f64/f32/16-bit); a full-lattice internal field is the even block followed by the odd block.
 * Use tm_field_bytes / tm_field_import / tm_field_export; never index them by hand.
 *
 * Ownership: the caller owns every field / output buffer and the stream.  The context owns
 * its private gauge copies (one per precision x reconstruct actually used, built lazily from
 * the fp64 master) and solver workspaces.  Errors: every call returns tm_status; nothing
 * throws or aborts across the ABI; text of the last error via tm_last_error.  There is NO CPU
 * fallback: without a CUDA device tm_create fails with TM_ECUDA.
 * Calls are stream-ordered; those that fill an *_info struct synchronise the stream at the end.
 * One stream at a time per context: state the context builds lazily (reduced-precision gauge copies, contraction
 * tables, workspaces) is ordered on the stream of the call that built it, so a caller that moves a context to another
 * stream must order the two streams itself (event or synchronisation).  A context is not thread-safe.
 */
#ifndef TMLOOPS_H
#define TMLOOPS_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct tm_ctx tm_ctx;
typedef enum { TM_OK = 0, TM_EARG = 1, TM_EDIM = 2, TM_EPREC = 3, TM_ECUDA = 4, TM_ENOCONV = 5,
               TM_EALLOC = 6 } tm_status;
typedef enum { TM_F64 = 0, TM_F32 = 1, TM_F16 = 2, TM_BF16 = 3 } tm_prec;
typedef enum { TM_R18 = 18, TM_R12 = 12 } tm_recon;
/* tm_dslash operations ([B:ns] operator; A = 1 + 2 i kappa mu gamma5 is the site-diagonal part,
 * D the hopping sum, "p" the output parity, "q" the other one):
 *   TM_OP_HOP        out_p = D_pq in_q
 *   TM_OP_HOP_TWINV  out_p = A^-1 D_pq in_q
 *   TM_OP_XPAY       out_p = A x_p - kappa^2 D_pq in_q
 *   TM_OP_M_FULL     out = M in on the full lattice (in, out: full-lattice internal fields)
 *   TM_OP_MHAT       out_e = (A - kappa^2 D_eo A^-1 D_oe) in_e   (even-odd Schur complement)
 * dagger != 0 applies the adjoint (gamma_mu -> -gamma_mu in the projectors, mu -> -mu). */
typedef enum { TM_OP_HOP = 0, TM_OP_HOP_TWINV = 1, TM_OP_XPAY = 2, TM_OP_M_FULL = 3,
               TM_OP_MHAT = 4 } tm_op;

/* dims: {Lx,Ly,Lz,T}, each even and >= 2 (TM_EDIM otherwise); t_boundary: +1 | -1;
 * device: CUDA ordinal.  TM_ECUDA if no usable device. */
tm_status tm_create(tm_ctx** ctx, const int dims[4], int t_boundary, int device);
tm_status tm_destroy(tm_ctx* ctx);
const char* tm_last_error(const tm_ctx* ctx);

/* Context options (no environment variables, no global state: everything lives in the opaque context).
 *   TM_OPT_GROUP          sources solved per launch by tsm_estimate*: 0 = automatic (8, halved until the workspaces
 *                         fit the device memory), or 1 | 2 | 4 | 8
 *   TM_OPT_CONTRACT_PATH  site + x/y-DFT stage of the contraction: 0 = automatic (fastest usable), 1 = generic kernel
 *                         (read-only-cache loads; any Lx, fp64), 2 = TMA-staged fp32 kernel with the DFT on the fp32 pipe
 *                         (x-stage folded over the sites {x, L-x, L/2-x, L/2+x} where Lx is 16, 24 or 32; whole-vector
 *                         calls keep only the forward half of the s-family derivative and restore the rest in the
 *                         assembly), 3 = TMA-staged fp32 kernel with the x-stage of the DFT on the tensor cores (tf32
 *                         MMAs on split-fp32 operands, hi*hi + lo*hi + hi*lo: same 1e-5 bound; whole-vector calls; never
 *                         the automatic choice: measured slower than 2), 4 = kernel 2 without the fold and with both
 *                         halves of every derivative (the plain form; what single-timeslice calls of 2 also use for the
 *                         derivative); 2, 3 and 4 need Lx <= 32 and fall back to 1 otherwise
 *   TM_OPT_POISON         debugging aid (compute-sanitizer's initcheck is not available everywhere): 1 = every workspace
 *                         the context allocates from now on starts as 0xFF bytes, i.e. NaN in all four storage
 *                         precisions, so that a read of never-written workspace memory reaches the results
 *   TM_OPT_LANES          jobs in flight in tsm_estimate*, each on a lane of its own (stream + workspaces): 0 = automatic
 *                         (one when the sources are solved 8 per launch -- such kernels fill the GPU --, else two), 1, 2.
 *                         On one lane the solve / contraction phases follow one another on one stream and the phase
 *                         times of tsm_info add up to the total; estimates of one and two lanes differ only by the order
 *                         of the fp64 accumulation
 * TM_EARG for an unknown option or value. */
typedef enum { TM_OPT_GROUP = 0, TM_OPT_CONTRACT_PATH = 1, TM_OPT_POISON = 2, TM_OPT_LANES = 3 } tm_option;
tm_status tm_set_option(tm_ctx* ctx, tm_option opt, int value);

/* d_U: device, canonical complex128 [V][4][3][3].  Copied into the context (fp64 master) asynchronously on stream;
 * previously built reduced-precision copies are marked stale and repacked on their next use.
 * tm_load_gauge_host: the same from HOST memory (pinned for a truly asynchronous copy); the buffer must stay valid
 * until the stream has passed the call.
 * Streams: every call is stream-ordered on the stream it is given.  The context's lazily built state is ordered across
 * streams by events: a call on another stream than the one that uploaded the master or packed a reduced-precision copy
 * waits (on the device) for that upload / pack before using it, and a new upload waits for the packs of the previous
 * master.  What the library cannot know is which kernels of OTHER streams still read the previous gauge field or a
 * workspace: load a new gauge field, and share one context between streams, only at points where the caller has
 * ordered those streams itself (one context per stream is the simple rule; tsm_estimate's own lanes are ordered inside). */
tm_status tm_load_gauge(tm_ctx* ctx, const void* d_U, void* stream);
tm_status tm_load_gauge_host(tm_ctx* ctx, const void* h_U, void* stream);

/* bytes of an internal field of the given storage precision (full_lattice: 0 = one parity). */
size_t tm_field_bytes(const tm_ctx* ctx, tm_prec prec, int full_lattice);
/* canonical complex128 full-lattice spinor <-> internal full-lattice field (device, device). */
tm_status tm_field_import(tm_ctx* ctx, void* d_internal, const void* d_canon, tm_prec prec, void* stream);
tm_status tm_field_export(tm_ctx* ctx, void* d_canon, const void* d_internal, tm_prec prec, void* stream);

/* One application of the operator pieces above on INTERNAL fields (device).
 * d_out, d_in: parity fields (full-lattice fields for TM_OP_M_FULL); d_x: parity field, used by
 * TM_OP_XPAY only (else NULL); out_parity 0 = even, 1 = odd (ignored by M_FULL / MHAT).
 * d_out must not alias d_in.  Asynchronous on stream. */
tm_status tm_dslash(tm_ctx* ctx, void* d_out, const void* d_in, const void* d_x, tm_op op,
                    int out_parity, int dagger, double kappa, double mu, tm_prec prec,
                    tm_recon recon, void* stream);

/* Row f3 of SURVEY.md sec 8 (multi-source Dslash; the N_LP ~ 1e2-1e3 sources are independent): the
 * operator pieces HOP, HOP_TWINV, XPAY of tm_dslash (reconstruct-12) applied to nb = 1, 2, 4 or 8 parity fields in
 * one launch.  d_out, d_in, d_x: nb internal parity fields back to back (source b at byte offset
 * b * tm_field_bytes(prec, 0)).  CTAs nb*k .. nb*k + nb-1 work on the same sites of the nb sources, so every link
 * crosses HBM once per group (the later readers find it in L2).  Results are bit-identical to nb tm_dslash calls.
 * tsm_estimate solves its sources in such groups (8 by default).  Asynchronous on stream. */
tm_status tm_dslash_multi(tm_ctx* ctx, void* d_out, const void* d_in, const void* d_x, int nb, tm_op op,
                          int out_parity, int dagger, double kappa, double mu, tm_prec prec, void* stream);

/* eq. 2.1: even-odd preconditioned CG on Mhat^dag Mhat (CGLS recurrences, x0 = 0) in `sloppy`
 * storage with reliable updates in `outer` precision (TM_F32 or TM_F64, >= sloppy).
 * Stops when the true residual ||eta - M s|| / ||eta|| evaluated in `outer` precision is <= rho.
 * delta: reliable-update trigger (iterated residual dropped by this factor; <= 0 -> 0.1). */
typedef struct { tm_prec sloppy, outer; tm_recon recon; double rho; int max_iter; double delta; } tm_solve_params;
typedef struct { int iters; int reliable_updates; double true_resid; double ms; } tm_solve_info;
/* d_s (out), d_eta (in): device canonical complex128 full-lattice spinors.
 * TM_ENOCONV if rho is not reached within max_iter (d_s and info are still filled). */
tm_status tm_cg_solve(tm_ctx* ctx, void* d_s, const void* d_eta, double kappa, double mu,
                      const tm_solve_params* params, tm_solve_info* info, void* stream);

/* sec 2.1.1 / 2.2: the 160 insertions of (s, eta), momentum-projected per timeslice:
 *   d_out[((f*80 + i)*nmom + k)*T + t] = sum_{x,y,z} exp(+2 pi i p_k.x / L) l_{f,i}(x,y,z,t)
 *   l_{0,n} = s^dag g5 G_n s,  l_{0,16+16m+n} = s^dag g5 G_n D_m s,
 *   l_{1,n} = s^dag g5 G_n g,  l_{1,16+16m+n} = s^dag g5 G_n D_m g,  g = g5 eta - 2 i kappa mu s,
 *   G_n = g_x^b0 g_y^b1 g_z^b2 g_t^b3 (n = b0+2b1+4b2+8b3), D_m the symmetric covariant difference.
 * d_s, d_eta: device canonical complex128; d_out: device complex128 [2][80][nmom][T];
 * h_momenta: host int [nmom][3] = (px,py,pz); at most 4 distinct |px| values (TM_EARG otherwise);
 * acc: TM_F64 or TM_F32 (arithmetic and accumulation precision of the site and DFT stages). */
tm_status loop_contract_project(tm_ctx* ctx, void* d_out, const void* d_s, const void* d_eta,
                                double kappa, double mu, const int* h_momenta, int nmom,
                                tm_prec acc, void* stream);

/* The same call on fields that are already in the internal layout of precision acc (full-lattice fields made by
 * tm_field_import: what the TSM loop hands to the contraction after a solve) -- no canonical -> internal conversion
 * inside, so it times and profiles as the loop runs it.  d_s_int, d_eta_int: tm_field_bytes(acc, 1) bytes each. */
tm_status loop_contract_project_fields(tm_ctx* ctx, void* d_out, const void* d_s_int, const void* d_eta_int,
                                       double kappa, double mu, const int* h_momenta, int nmom,
                                       tm_prec acc, void* stream);

/* loop_contract_project_fields for callers that cannot allocate (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): same arguments, same result (the generic contraction kernels; fp32 results agree
 * with the automatic path within the fp32 bound, fp64 within rounding of the DFT weights), but the call performs NO
 * cudaMalloc / cudaFree / cudaMemcpy or other allocating routine.  Its scratch -- x/y partial sums, z-stage sums, DFT
 * weight tables, momentum list -- lives in one file-scope device array of loop_contract_static_scratch_bytes() = 16 MiB
 * that every GPU which loads the library holds until the process exits; the tables are written by a kernel from
 * kernel arguments.  Limits and rules:
 *   - the lattice / momentum set must fit: tables + Lz*T*NQ*320*sizeof(acc) + T*NQ*7*320*8 bytes <= 16 MiB, NQ = 29
 *     (all px^2 + py^2 <= 9) or 49; e.g. 4^3x8 in fp64, 8^3x16 in fp32.  TM_EDIM with the sizes in the message otherwise;
 *   - nmom <= 128 (TM_EARG otherwise);
 *   - the packed gauge copy of precision acc is context state, not scratch, and must exist: one call of
 *     loop_contract_project_fields with the same acc after tm_load_gauge creates it (TM_EARG otherwise);
 *   - ALL calls on one device share the array (whatever the context): calls that overlap on the GPU, i.e. on different
 *     streams without ordering, race.  Calls on one stream are safe.  The array keeps the last call's contents; nothing in
 *     it needs clearing (a call writes every element before reading it);
 *   - the first call on a device does the one-time set-up (cudaGetSymbolAddress of the array, upload of the 192-byte
 *     Gamma table into constant memory): do one call before starting a graph capture. */
tm_status loop_contract_project_fields_static(tm_ctx* ctx, void* d_out, const void* d_s_int, const void* d_eta_int,
                                              double kappa, double mu, const int* h_momenta, int nmom,
                                              tm_prec acc, void* stream);
size_t loop_contract_static_scratch_bytes(void);

/* PAPER.md:88 ("GPU kernels to contract a single time slice or a whole vector", for time-dilution): the same call
 * restricted to ONE timeslice t0 -- 1/T of the work.  d_out keeps the shape [2][80][nmom][T]: column t0 is
 * computed, every other column is set to zero. */
tm_status loop_contract_project_timeslice(tm_ctx* ctx, void* d_out, const void* d_s, const void* d_eta,
                                          double kappa, double mu, const int* h_momenta, int nmom, int t0,
                                          tm_prec acc, void* stream);

/* Row f3 variant (reading 5): the same 160 projected insertions with the generalised one-end trick's
 * D_W applied EXPLICITLY: g = g5 D_W s = g5 (M s) - 2 i kappa mu s instead of g5 eta - 2 i kappa mu s, i.e. the loops
 * of (s, eta := M s); it differs from loop_contract_project by the bilinears of g5 (eta - M s) and costs one extra
 * full operator application (in precision acc, reconstruct-12 for TM_F32, -18 for TM_F64). */
tm_status loop_contract_project_explicit(tm_ctx* ctx, void* d_out, const void* d_s, double kappa, double mu,
                                         const int* h_momenta, int nmom, tm_prec acc, void* stream);

/* Row f3 variant (reading 4): the same output with the left-right SYMMETRISED derivative in the 128
 * one-derivative insertions, l[f][16+16m+n] = 1/2 [ s^dag g5 G_n (D_m psi) - (D_m s)^dag g5 G_n psi ] (psi = s | g);
 * ultra-local entries as in loop_contract_project.  Obtained from the same primitive with the arguments swapped
 * (two contraction passes + a small assembly kernel); h_momenta must contain -p for every p (TM_EARG otherwise). */
tm_status loop_contract_project_sym(tm_ctx* ctx, void* d_out, const void* d_s, const void* d_eta,
                                    double kappa, double mu, const int* h_momenta, int nmom,
                                    tm_prec acc, void* stream);

/* sec 2.1: L_TSM = (1/N_LP) sum_{r<N_LP} l_r^LP + (1/N_HP) sum_{r<N_HP} (l_r^HP - l_r^LP);
 * the HP sources are the first n_hp of the LP sources.  Z4 noise eta_r[c] = i^k, c = (site*4+spin)*3+col:
 * d_z4 != NULL: packed exponents, byte j of source r holds k[4j+m] in bits 2m..2m+1,
 *               layout [n_lp][3V] bytes (device);
 * d_z4 == NULL: generated on the device from `seed` with the counter hash of DESIGN.md
 *               (k = h(seed, r, c) & 3). */
/* Sharding by source (the sources are independent): local source j = 0..n_lp-1 of a call
 * is the GLOBAL source r = src_first + j * src_stride (src_stride 0 is read as 1), which names its noise stream
 * h(seed, r, .); d_z4 is indexed by the local j.  Rank k of W ranks takes src_first = k, src_stride = W, so the first
 * N_HP global sources -- the ones that also get an HP solve -- are spread evenly: n_hp = ceil((N_HP - k) / W).
 * d_solutions: optional (NULL ok) device complex128 [n_lp + n_hp][V][4][3], receives every solution s_r in canonical
 * layout (LP first, then HP) so that a checker can evaluate residuals and loops of the run's own solutions. */
typedef struct { int n_lp, n_hp; tm_solve_params lp, hp; double kappa, mu;
                 const int* h_momenta; int nmom; tm_prec contract_acc_lp, contract_acc_hp;
                 const unsigned char* d_z4; unsigned long long seed;
                 int src_first, src_stride; void* d_solutions; } tsm_params;
typedef struct { double ms_total, ms_lp_solve, ms_hp_solve, ms_contract; long iters_lp, iters_hp;
                 double worst_resid_lp, worst_resid_hp; int launches; int lanes; } tsm_info;
/* tsm_info: ms_* are device times (CUDA events); with lanes = 1 the three phase times add up to ms_total, with two lanes
 * the solve times of the lanes overlap and their sums are halved; lanes = jobs that were in flight (TM_OPT_LANES). */
/* d_out: device complex128 [2][80][nmom][T]; d_per_source: optional (NULL ok) device complex128
 * [n_lp + n_hp][2][80][nmom][T] receiving every per-source array (LP first, then HP).
 * TM_ENOCONV if any solve missed its rho (outputs still filled). */
tm_status tsm_estimate(tm_ctx* ctx, void* d_out, void* d_per_source, const tsm_params* params,
                       tsm_info* info, void* stream);
/* The same loop, stopped before the division: d_sums = complex128 [3][2][80][nmom][T] receives the raw accumulators
 * S_LP = sum_r l_r^LP (all n_lp local sources), S_LPc = sum_{r<n_hp} l_r^LP, S_HP = sum_{r<n_hp} l_r^HP.  With sources
 * sharded over ranks (src_first / src_stride above) the only exchange of a multi-GPU run is one all-reduce (sum) of
 * these three arrays, followed by tsm_combine_sums on every rank:
 *   d_out = S_LP / n_lp_total + (S_HP - S_LPc) / n_hp_total      (n_hp_total = 0: the second term is dropped). */
tm_status tsm_partial_sums(tm_ctx* ctx, void* d_sums, void* d_per_source, const tsm_params* params,
                           tsm_info* info, void* stream);
tm_status tsm_combine_sums(tm_ctx* ctx, void* d_out, const void* d_sums, int n_lp_total, int n_hp_total,
                           int nmom, void* stream);
/* Same with HOST buffers (PAPER.md:104-106 names source generation and transfers as the bottlenecks of the paper's own
 * code; Fig. 4 / PAPER.md:115 is the all-on-GPU scheme): h_z4 (pinned or pageable host memory, [n_lp][3V] bytes, may be
 * NULL -> seed) is uploaded by a copy stream in group-sized chunks that run ahead of the solves (the whole packed noise
 * stays resident on the device when it fits a quarter of the free memory, else it is staged source by source), and
 * h_out (complex128 [2][80][nmom][T]) is copied back, all inside the call, which returns after the copy back.
 * tsm_partial_sums_host: the same for the raw accumulators, h_sums = complex128 [3][2][80][nmom][T]. */
tm_status tsm_estimate_host(tm_ctx* ctx, void* h_out, const unsigned char* h_z4,
                            const tsm_params* params, tsm_info* info, void* stream);
tm_status tsm_partial_sums_host(tm_ctx* ctx, void* h_sums, const unsigned char* h_z4,
                                const tsm_params* params, tsm_info* info, void* stream);

/* Row f4 of SURVEY.md sec 8 -- time dilution ("we also worked with time-dilution [6], so there are GPU
 * kernels to contract a single time slice or a whole vector"; it combines with the TSM; reading 22).
 *
 * loop_plain_project_timeslice: the plain bilinears of a pair (a, b) on timeslice t0 (t0 = -1: on every timeslice),
 *   d_out[(i*nmom + k)*T + t] = sum_{x,y,z} exp(+2 pi i p_k.x / L) a(x,t)^dag X_i b(x,t),
 *   X_n = G_n (n < 16), X_{16+16m+n} = G_n D_m (D_m acting on b);  columns t != t0 are set to zero.
 * d_a, d_b: device canonical complex128 spinors; d_out: device complex128 [80][nmom][T].
 *
 * tsm_estimate_time_diluted: the TSM estimator of the time-diluted plain loops.  For every noise vector r and every
 * timeslice t0: eta_r^(t0) = eta_r restricted to t0, M s = eta_r^(t0) (LP for all r, HP as well for r < n_hp; the T
 * diluted sources of a noise vector are solved 8 per launch), l_r[i][k][t0] = the bilinear above of (eta_r^(t0), s) on
 * timeslice t0 -- T solves and T single-timeslice contractions per noise vector and pass -- then
 *   d_out = (1/n_lp) sum_r l_r^LP + (1/n_hp) sum_{r<n_hp} (l_r^HP - l_r^LP)          complex128 [80][nmom][T].
 * d_per_source: optional (NULL ok) [n_lp + n_hp][80][nmom][T].  params as for tsm_estimate (d_solutions is not used);
 * TM_ENOCONV if any solve missed its rho (outputs still filled).  Synchronises the stream at the end. */
tm_status loop_plain_project_timeslice(tm_ctx* ctx, void* d_out, const void* d_a, const void* d_b,
                                       const int* h_momenta, int nmom, int t0, tm_prec acc, void* stream);
tm_status tsm_estimate_time_diluted(tm_ctx* ctx, void* d_out, void* d_per_source, const tsm_params* params,
                                    tsm_info* info, void* stream);

/* Row f4 of SURVEY.md sec 8, second half -- Hopping Parameter Expansion ("... time-dilution and the Hopping
 * Parameter Expansion (HPE) [7], and all the possible combinations of these"; reading 23).
 * With A = 1 + 2 i kappa mu g5 and H = A - M (kappa times the hopping term):
 *   M^-1 = sum_{k<n} (A^-1 H)^k A^-1 + (A^-1 H)^n M^-1   for every n,
 * so the plain loop estimator splits into an exact part and a remainder estimated with the same solution:
 *   d_out[(i*nmom + k)*T + t] = sum_{x,y,z} exp(+2 pi i p_k.x / L) eta(x,t)^dag X_i ((A^-1 H)^{n_i} s)(x,t) + E_i(p_k),
 *   X_n = G_n (n < 16): n_i = order;  X_{16+16m+n} = G_n D_m: n_i = min(order, 2);  order = 0..4 (0: the plain estimator);
 *   E_i = the site- and gauge-independent trace of X_i sum_{k<n_i} (A^-1 H)^k A^-1 (closed forms, nonzero at p = 0 only).
 * loop_hpe_project: one (eta, s) pair, device canonical complex128 spinors; d_out: device complex128 [80][nmom][T].
 * tsm_estimate_hpe: the TSM estimator of these loops (whole-volume Z4 sources, solved 8 per launch; LP for all n_lp
 *   sources, HP as well for the first n_hp): d_out = (1/n_lp) sum_r l_r^LP + (1/n_hp) sum_{r<n_hp} (l_r^HP - l_r^LP),
 *   complex128 [80][nmom][T]; d_per_source: optional (NULL ok) [n_lp + n_hp][80][nmom][T]; params as for tsm_estimate
 *   (d_solutions is not used).  TM_ENOCONV if any solve missed its rho (outputs still filled); synchronises the stream.
 * TM_EDIM if order > 0 and an extent is < 4 (paths of fewer than 4 hops would close around the torus), TM_EARG for an
 * order outside 0..4. */
tm_status loop_hpe_project(tm_ctx* ctx, void* d_out, const void* d_eta, const void* d_s, double kappa, double mu,
                           const int* h_momenta, int nmom, int order, tm_prec acc, void* stream);
tm_status tsm_estimate_hpe(tm_ctx* ctx, void* d_out, void* d_per_source, const tsm_params* params, int order,
                           tsm_info* info, void* stream);

/* sec 2.1.1 (Fig. 2): binary storage of partial sums, on the device, in momentum space.
 * File k = 0, 1, 2, ... (the paper's File.2^k) holds the SUM of the per-source arrays of the 2^k sources
 * r = 2^k - 1 ... 2^(k+1) - 2, so n sources need loop_binary_nfiles(n) = ceil(log2(n + 1)) arrays instead of n.
 *   loop_binary_accumulate: d_files[k(r)] += d_loop   (k(r) = floor(log2(r + 1)))
 *   loop_binary_recover:    d_out = (sum of the files named by the binary digits of N) / N
 *                           ("Reconstruction is straightforward, taking into account the base-2 structure";
 *                           Fig. 2: N = 13 = 1101b -> the files holding 8, 4 and 1 sources).
 * d_files: device complex128 [nfiles][len], zeroed by the caller before the first source; d_loop, d_out:
 * device complex128 [len]; len = number of complex entries of one per-source array (160 * nmom * T).
 * n_stored = number of sources accumulated so far.  Recoverable N: any N whose binary digits name COMPLETE files, and
 * N = n_stored itself (the sum of every file, the partially filled last one included, divided by n_stored) -- so a run
 * of 500 + 20 sources can always recover its own full estimate; recover returns TM_EARG for any other N.
 * Asynchronous on stream. */
int loop_binary_nfiles(int n_sources);
tm_status loop_binary_accumulate(tm_ctx* ctx, void* d_files, const void* d_loop, int r, size_t len, void* stream);
tm_status loop_binary_recover(tm_ctx* ctx, void* d_out, const void* d_files, int n_stored, int N, size_t len,
                              void* stream);
/* tsm_estimate that also fills the binary-storage files (either may be NULL):
 *   d_files_lp   [loop_binary_nfiles(n_lp)][2][80][nmom][T]: file k += l_r^LP              for every r < n_lp
 *   d_files_corr [loop_binary_nfiles(n_hp)][2][80][nmom][T]: file k += l_r^HP - l_r^LP     for every r < n_hp
 * so that the TSM estimate of any (N_LP', N_HP') with complete files is
 *   recover(files_lp, N_LP') + recover(files_corr, N_HP').  Both are zeroed inside the call. */
tm_status tsm_estimate_binary(tm_ctx* ctx, void* d_out, void* d_files_lp, void* d_files_corr,
                              const tsm_params* params, tsm_info* info, void* stream);

/* Measured fp32 FMA peak of the device in TFLOP/s (2 flop per FMA lane): the ALU roofline denominator of the contraction
 * kernel (measure it, do not quote it).  mode 0: scalar FFMA, mode 1: packed FFMA2 (the instruction
 * the contraction and the fp32 Dslash issue); iters rounds of 16 independent FMAs per thread, best of 3 launches.
 * Synchronises the stream. */
tm_status tm_fma_peak(tm_ctx* ctx, int mode, int iters, double* tflops, void* stream);

/* number of kernels launched by this context so far (bench.py's gpu_launches) */
long tm_launch_count(const tm_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif
