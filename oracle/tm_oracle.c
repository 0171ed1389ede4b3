/* tm_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, double-precision, full-lattice statement of what the TSM
 * disconnected-loop hot path of arXiv:1401.6750 computes.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may call it.  It shares no code, header, table or helper with the CUDA path
 * (paper_1401_6750_b200/csrc) and uses none of that path's devices: no
 * even-odd preconditioning, no spin-projection trick, no link reconstruction,
 * no separable DFT, no fusion.  OpenMP over sites only changes summation
 * order in the global dot products.
 *
 * Passages followed (PAPER.md = /root/reference/PAPER.md; [B:ns] =
 * BASELINE.json north_star; readings = DESIGN.md "Readings of the paper"):
 *   eq. 2.1  PAPER.md:50        M |s_r> = |eta_r>                  -> orc_solve
 *   [B:ns]                      M = (1 + 2 i kappa mu g5 tau3) - kappa * sum_mu
 *                               [(1-g_mu) U_mu(x) d_{x+mu,y} + (1+g_mu) U_mu^dag(x-mu) d_{x-mu,y}]
 *                                                                   -> orc_apply_M
 *   sec 2.1  PAPER.md:56-58     TSM: N_LP low precision + N_HP correction -> orc_tsm_combine
 *   sec 2.1.1, Fig. 2  binary storage of partial sums       -> orc_binary_store / _recover
 *   sec 2.1.1 PAPER.md:72       one-end trick, 16 ultra-local + 64 one-derivative
 *                               insertions, with/without tau3 = 160  -> orc_loops_sites
 *   sec 2.2  PAPER.md:86        colour trace, Dirac indices open; covariant derivative
 *                                                                   -> orc_cov_deriv
 *   sec 2.2/2.3 PAPER.md:88,94-100  "array with a time-slice index", Fourier
 *                               transform, cut in p^2               -> orc_loops_project
 *   sec 2.2  PAPER.md:88, 92    time-dilution: sources on one timeslice, "contract a single
 *                               time slice"                         -> orc_time_dilute, orc_plain_loops_project
 *   sec 2.3  PAPER.md:92        Hopping Parameter Expansion [7]: M^-1 = sum_{k<n} (A^-1 H)^k A^-1 + (A^-1 H)^n M^-1
 *                                                                   -> orc_apply_AinvH, orc_hpe_exact
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"): gamma algebra; gamma5-
 * hermiticity; free-field plane waves vs the momentum-space closed form;
 * gauge covariance / invariance; dense assembly + LU on 2^4; full-dilution
 * loops vs traces of dense inverses; summation by parts; numpy.fft cross-check
 * of the projection; TSM identity; Fig. 2's 13-source example of the binary
 * storage; time dilution: exact spin-colour-site dilution of one timeslice vs the
 * trace of the dense inverse, dense-D_m einsum, linearity in t0; HPE: A^-1 H against the
 * dense matrices, the expansion identity and the exact part against traces of dense
 * matrices on 2^4, the closed forms of the exact part on 4^4.  No function here
 * is "parity unpinned".
 *
 * Conventions (readings 1-7,15,16): dims = {Lx,Ly,Lz,T}; site index
 * ((t*Lz+z)*Ly+y)*Lx+x; directions mu = 0,1,2,3 = x,y,z,t; spinor
 * psi[site*12 + spin*3 + colour]; link U[((site*4+mu)*3+row)*3+col];
 * periodic in space, psi(t+T) = tb * psi(t) in time (tb = +1 | -1);
 * Hermitian chiral gamma basis, gamma5 = g_x g_y g_z g_t = diag(1,1,-1,-1);
 * Gamma_n = g_x^b0 g_y^b1 g_z^b2 g_t^b3, n = b0 + 2 b1 + 4 b2 + 8 b3.
 */
#define _GNU_SOURCE
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cplx;

/* ------------------------------------------------------------------ gamma */
/* reading 2: g_k = [[0, -i sigma_k],[i sigma_k, 0]], g_t = [[0,1],[1,0]]   */
static void gamma_mat(int mu, cplx g[4][4])
{
    memset(g, 0, 16 * sizeof(cplx));
    switch (mu) {
    case 0: /* sigma_x = [[0,1],[1,0]] */
        g[0][3] = -I; g[1][2] = -I; g[2][1] = I;  g[3][0] = I;  break;
    case 1: /* sigma_y = [[0,-i],[i,0]] : -i*sigma_y = [[0,-1],[1,0]] */
        g[0][3] = -1; g[1][2] = 1;  g[2][1] = 1;  g[3][0] = -1; break;
    case 2: /* sigma_z = diag(1,-1) */
        g[0][2] = -I; g[1][3] = I;  g[2][0] = I;  g[3][1] = -I; break;
    case 3:
        g[0][2] = 1;  g[1][3] = 1;  g[2][0] = 1;  g[3][1] = 1;  break;
    default: /* gamma5 */
        g[0][0] = 1;  g[1][1] = 1;  g[2][2] = -1; g[3][3] = -1; break;
    }
}

static void mat4_mul(cplx c[4][4], cplx a[4][4], cplx b[4][4])
{
    cplx t[4][4];
    for (int i = 0; i < 4; i++)
        for (int j = 0; j < 4; j++) {
            cplx s = 0;
            for (int k = 0; k < 4; k++) s += a[i][k] * b[k][j];
            t[i][j] = s;
        }
    memcpy(c, t, sizeof(t));
}

/* reading 3: Gamma_n = g_x^b0 g_y^b1 g_z^b2 g_t^b3 */
static void Gamma_mat(int n, cplx G[4][4])
{
    memset(G, 0, 16 * sizeof(cplx));
    for (int i = 0; i < 4; i++) G[i][i] = 1;
    for (int mu = 0; mu < 4; mu++)
        if ((n >> mu) & 1) {
            cplx g[4][4];
            gamma_mat(mu, g);
            mat4_mul(G, G, g);
        }
}

void orc_gamma(int mu, cplx *out)   { cplx g[4][4]; gamma_mat(mu, g); memcpy(out, g, sizeof(g)); }
void orc_Gamma(int n, cplx *out)    { cplx g[4][4]; Gamma_mat(n, g);  memcpy(out, g, sizeof(g)); }

/* ------------------------------------------------------------- geometry */
static inline long site_of(const int d[4], int x, int y, int z, int t)
{
    return (((long)t * d[2] + z) * d[1] + y) * d[0] + x;
}

/* neighbour of (c[0..3]) displaced by dir (+1|-1) along mu; *sign gets the
 * time-boundary factor tb when the hop wraps around in t (reading 7). */
static inline long neighbour(const int d[4], const int c[4], int mu, int dir, int tb, double *sign)
{
    int n[4] = { c[0], c[1], c[2], c[3] };
    *sign = 1.0;
    n[mu] += dir;
    if (n[mu] >= d[mu]) { n[mu] -= d[mu]; if (mu == 3) *sign = tb; }
    if (n[mu] < 0)      { n[mu] += d[mu]; if (mu == 3) *sign = tb; }
    return site_of(d, n[0], n[1], n[2], n[3]);
}

static inline void coords_of(const int d[4], long s, int c[4])
{
    c[0] = (int)(s % d[0]); s /= d[0];
    c[1] = (int)(s % d[1]); s /= d[1];
    c[2] = (int)(s % d[2]); s /= d[2];
    c[3] = (int)s;
}

/* v[spin][a] = sum_b U[a][b] psi[spin][b]   (dag=0)
 * v[spin][a] = sum_b conj(U[b][a]) psi[spin][b] (dag=1) */
static inline void su3_mul(cplx v[4][3], const cplx *U, const cplx *psi, int dag)
{
    for (int s = 0; s < 4; s++)
        for (int a = 0; a < 3; a++) {
            cplx acc = 0;
            for (int b = 0; b < 3; b++)
                acc += (dag ? conj(U[b * 3 + a]) : U[a * 3 + b]) * psi[s * 3 + b];
            v[s][a] = acc;
        }
}

/* ------------------------------------------------------------ operator M */
/* [B:ns]:  (M psi)(x) = psi(x) + 2 i kappa mu gamma5 psi(x)
 *            - kappa sum_mu [ (1-g_mu) U_mu(x) psi(x+mu) + (1+g_mu) U_mu^dag(x-mu) psi(x-mu) ]
 * dagger=1: the conjugate transpose written out from the definition:
 *          (M^dag psi)(x) = psi(x) - 2 i kappa mu gamma5 psi(x)
 *            - kappa sum_mu [ (1+g_mu) U_mu(x) psi(x+mu) + (1-g_mu) U_mu^dag(x-mu) psi(x-mu) ]
 * (tau3 -> +1, the up flavour; mu < 0 gives the down flavour -- reading 1). */
void orc_apply_M(cplx *out, const cplx *in, const cplx *U, const int *dims, int tb,
                 double kappa, double mu, int dagger)
{
    const long V = (long)dims[0] * dims[1] * dims[2] * dims[3];
    cplx g[5][4][4];
    for (int m = 0; m < 5; m++) gamma_mat(m, g[m]);
    const double gs = dagger ? -1.0 : 1.0; /* sign in front of gamma_mu in the forward hop is -gs */
#pragma omp parallel for schedule(static)
    for (long x = 0; x < V; x++) {
        int c[4];
        coords_of(dims, x, c);
        cplx hop[4][3];
        memset(hop, 0, sizeof(hop));
        for (int m = 0; m < 4; m++) {
            double sg;
            cplx v[4][3];
            /* forward: (1 - gs*g_mu) U_mu(x) psi(x+mu) */
            long xp = neighbour(dims, c, m, +1, tb, &sg);
            su3_mul(v, U + (x * 4 + m) * 9, in + xp * 12, 0);
            for (int s = 0; s < 4; s++)
                for (int a = 0; a < 3; a++) {
                    cplx acc = v[s][a];
                    for (int s2 = 0; s2 < 4; s2++) acc -= gs * g[m][s][s2] * v[s2][a];
                    hop[s][a] += sg * acc;
                }
            /* backward: (1 + gs*g_mu) U_mu^dag(x-mu) psi(x-mu) */
            long xm = neighbour(dims, c, m, -1, tb, &sg);
            su3_mul(v, U + (xm * 4 + m) * 9, in + xm * 12, 1);
            for (int s = 0; s < 4; s++)
                for (int a = 0; a < 3; a++) {
                    cplx acc = v[s][a];
                    for (int s2 = 0; s2 < 4; s2++) acc += gs * g[m][s][s2] * v[s2][a];
                    hop[s][a] += sg * acc;
                }
        }
        for (int s = 0; s < 4; s++)
            for (int a = 0; a < 3; a++) {
                cplx g5psi = 0;
                for (int s2 = 0; s2 < 4; s2++) g5psi += g[4][s][s2] * in[x * 12 + s2 * 3 + a];
                out[x * 12 + s * 3 + a] = in[x * 12 + s * 3 + a]
                                          + gs * 2.0 * I * kappa * mu * g5psi
                                          - kappa * hop[s][a];
            }
    }
}

/* ----------------------------------------------------------------- solve */
static double norm2(const cplx *a, long n)
{
    double s = 0;
#pragma omp parallel for reduction(+ : s) schedule(static)
    for (long i = 0; i < n; i++) s += creal(a[i]) * creal(a[i]) + cimag(a[i]) * cimag(a[i]);
    return s;
}

/* eq. 2.1: find s with ||eta - M s|| / ||eta|| <= rho  (reading 8).
 * Route: unpreconditioned CG on the normal equations M^dag M s = M^dag eta on
 * the full lattice (CGLS form, residual of M s = eta tracked), s0 = 0
 * (reading 9).  Stops at the first iterate whose recurrence residual meets rho;
 * *true_resid is recomputed from scratch with orc_apply_M.
 * Returns 0 on convergence, 1 if max_iter was hit. */
int orc_solve(cplx *s, const cplx *eta, const cplx *U, const int *dims, int tb,
              double kappa, double mu, double rho, int max_iter,
              int *iters, double *true_resid)
{
    const long n = 12L * dims[0] * dims[1] * dims[2] * dims[3];
    cplx *r = malloc(n * sizeof(cplx)), *z = malloc(n * sizeof(cplx));
    cplx *p = malloc(n * sizeof(cplx)), *w = malloc(n * sizeof(cplx));
    const double eta2 = norm2(eta, n);
    int k = 0, status = 1;
    memset(s, 0, n * sizeof(cplx));
    memcpy(r, eta, n * sizeof(cplx));
    if (eta2 == 0.0) { status = 0; goto done; }
    orc_apply_M(z, r, U, dims, tb, kappa, mu, 1);
    memcpy(p, z, n * sizeof(cplx));
    double gam = norm2(z, n);
    if (sqrt(norm2(r, n)) <= rho * sqrt(eta2)) status = 0;
    while (status && k < max_iter) {
        orc_apply_M(w, p, U, dims, tb, kappa, mu, 0);
        const double alpha = gam / norm2(w, n);
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; i++) { s[i] += alpha * p[i]; r[i] -= alpha * w[i]; }
        k++;
        if (sqrt(norm2(r, n)) <= rho * sqrt(eta2)) { status = 0; break; }
        orc_apply_M(z, r, U, dims, tb, kappa, mu, 1);
        const double gam2 = norm2(z, n);
        const double beta = gam2 / gam;
        gam = gam2;
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; i++) p[i] = z[i] + beta * p[i];
    }
done:
    if (iters) *iters = k;
    if (true_resid) {
        if (eta2 == 0.0) *true_resid = 0.0;
        else {
            orc_apply_M(w, s, U, dims, tb, kappa, mu, 0);
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; i++) w[i] = eta[i] - w[i];
            *true_resid = sqrt(norm2(w, n) / eta2);
        }
    }
    free(r); free(z); free(p); free(w);
    return status;
}

/* ||eta - M s|| / ||eta|| with the fp64 operator (reading 8) */
double orc_true_residual(const cplx *s, const cplx *eta, const cplx *U, const int *dims, int tb,
                         double kappa, double mu)
{
    const long n = 12L * dims[0] * dims[1] * dims[2] * dims[3];
    cplx *w = malloc(n * sizeof(cplx));
    orc_apply_M(w, s, U, dims, tb, kappa, mu, 0);
#pragma omp parallel for schedule(static)
    for (long i = 0; i < n; i++) w[i] = eta[i] - w[i];
    double r = sqrt(norm2(w, n) / norm2(eta, n));
    free(w);
    return r;
}

/* --------------------------------------------------- covariant derivative */
/* reading 4 / PAPER.md:86: (D_mu psi)(x) = 1/2 [ U_mu(x) psi(x+mu) - U_mu^dag(x-mu) psi(x-mu) ],
 * same boundary condition as M. */
static void cov_deriv_site(cplx out[12], const cplx *psi, const cplx *U, const int *dims, int tb,
                           long x, int m)
{
    int c[4];
    double sf, sb;
    cplx vf[4][3], vb[4][3];
    coords_of(dims, x, c);
    long xp = neighbour(dims, c, m, +1, tb, &sf);
    long xm = neighbour(dims, c, m, -1, tb, &sb);
    su3_mul(vf, U + (x * 4 + m) * 9, psi + xp * 12, 0);
    su3_mul(vb, U + (xm * 4 + m) * 9, psi + xm * 12, 1);
    for (int s = 0; s < 4; s++)
        for (int a = 0; a < 3; a++) out[s * 3 + a] = 0.5 * (sf * vf[s][a] - sb * vb[s][a]);
}

void orc_cov_deriv(cplx *out, const cplx *psi, const cplx *U, const int *dims, int tb, int m)
{
    const long V = (long)dims[0] * dims[1] * dims[2] * dims[3];
#pragma omp parallel for schedule(static)
    for (long x = 0; x < V; x++) cov_deriv_site(out + x * 12, psi, U, dims, tb, x, m);
}

/* ------------------------------------------------------------------ loops */
/* phi^dag X psi at one site: sum_{a,b,c} conj(phi[a][c]) X[a][b] psi[b][c]
 * ("traces were taken in color space, leaving the Dirac ... indices open") */
static inline cplx bilinear(const cplx *phi, cplx X[4][4], const cplx *psi)
{
    cplx acc = 0;
    for (int a = 0; a < 4; a++)
        for (int b = 0; b < 4; b++) {
            if (X[a][b] == 0) continue;
            cplx tr = 0;
            for (int c = 0; c < 3; c++) tr += conj(phi[a * 3 + c]) * psi[b * 3 + c];
            acc += X[a][b] * tr;
        }
    return acc;
}

/* g(x) = gamma5 eta(x) - 2 i kappa mu s(x)   (reading 5; = gamma5 D_W s when M s = eta) */
static void make_g(cplx *g, const cplx *s, const cplx *eta, long V, double kappa, double mu)
{
    cplx g5[4][4];
    gamma_mat(4, g5);
#pragma omp parallel for schedule(static)
    for (long x = 0; x < V; x++)
        for (int a = 0; a < 4; a++)
            for (int c = 0; c < 3; c++) {
                cplx t = 0;
                for (int b = 0; b < 4; b++) t += g5[a][b] * eta[x * 12 + b * 3 + c];
                g[x * 12 + a * 3 + c] = t - 2.0 * I * kappa * mu * s[x * 12 + a * 3 + c];
            }
}

/* The 160 insertions at site x (readings 3-6), out[f*80 + i]:
 *   out[0*80 + n]         = s^dag g5 Gamma_n s          (ultra-local, "with tau3")
 *   out[0*80 + 16+16m+n]  = s^dag g5 Gamma_n D_m s      (one-derivative)
 *   out[1*80 + n]         = s^dag g5 Gamma_n g          ("without tau3")
 *   out[1*80 + 16+16m+n]  = s^dag g5 Gamma_n D_m g                                  */
static void loops_at_site(cplx out[160], const cplx *s, const cplx *g, const cplx *U,
                          const int *dims, int tb, long x, cplx g5G[16][4][4])
{
    const cplx *fam[2] = { s, g };
    for (int f = 0; f < 2; f++) {
        for (int n = 0; n < 16; n++)
            out[f * 80 + n] = bilinear(s + x * 12, g5G[n], fam[f] + x * 12);
        for (int m = 0; m < 4; m++) {
            cplx d[12];
            cov_deriv_site(d, fam[f], U, dims, tb, x, m);
            for (int n = 0; n < 16; n++)
                out[f * 80 + 16 + 16 * m + n] = bilinear(s + x * 12, g5G[n], d);
        }
    }
}

/* Variant of reading 4: the left-right symmetrised derivative,
 *   out[f*80 + 16+16m+n] = 1/2 [ s^dag g5 Gamma_n (D_m psi) - (D_m s)^dag g5 Gamma_n psi ],  psi = s (f = 0) | g (f = 1);
 * the ultra-local entries are those of loops_at_site.  Written from the definition: D_m applied to s as well. */
static void loops_at_site_sym(cplx out[160], const cplx *s, const cplx *g, const cplx *U,
                              const int *dims, int tb, long x, cplx g5G[16][4][4])
{
    const cplx *fam[2] = { s, g };
    for (int f = 0; f < 2; f++) {
        for (int n = 0; n < 16; n++)
            out[f * 80 + n] = bilinear(s + x * 12, g5G[n], fam[f] + x * 12);
        for (int m = 0; m < 4; m++) {
            cplx dpsi[12], ds[12];
            cov_deriv_site(dpsi, fam[f], U, dims, tb, x, m);
            cov_deriv_site(ds, s, U, dims, tb, x, m);
            for (int n = 0; n < 16; n++)
                out[f * 80 + 16 + 16 * m + n] = 0.5 * (bilinear(s + x * 12, g5G[n], dpsi)
                                                       - bilinear(ds, g5G[n], fam[f] + x * 12));
        }
    }
}

static void make_g5G(cplx g5G[16][4][4])
{
    cplx g5[4][4];
    gamma_mat(4, g5);
    for (int n = 0; n < 16; n++) {
        cplx G[4][4];
        Gamma_mat(n, G);
        mat4_mul(g5G[n], g5, G);
    }
}

/* per-site loops for nsites listed sites: out[k*160 + f*80 + i] */
void orc_loops_sites(cplx *out, const cplx *s, const cplx *eta, const cplx *U, const int *dims,
                     int tb, double kappa, double mu, const long *sites, long nsites)
{
    const long V = (long)dims[0] * dims[1] * dims[2] * dims[3];
    cplx *g = malloc(V * 12 * sizeof(cplx));
    cplx g5G[16][4][4];
    make_g5G(g5G);
    make_g(g, s, eta, V, kappa, mu);
#pragma omp parallel for schedule(static)
    for (long k = 0; k < nsites; k++) loops_at_site(out + k * 160, s, g, U, dims, tb, sites[k], g5G);
    free(g);
}

/* PAPER.md:88,94-100 + readings 15,16: for timeslices t0 <= t < t1
 *   out[((f*80+i)*nmom + k)*T + t] = sum_{x,y,z} exp(+2 pi i (px x/Lx + py y/Ly + pz z/Lz)) l_{f,i}(x,y,z,t)
 * by the direct sum.  momenta: int [nmom][3] = (px,py,pz).  Entries of out for
 * other t are left untouched. */
static void loops_project_impl(cplx *out, const cplx *s, const cplx *eta, const cplx *U, const int *dims,
                               int tb, double kappa, double mu, const int *momenta, int nmom,
                               int t0, int t1, int sym)
{
    const int Lx = dims[0], Ly = dims[1], Lz = dims[2], T = dims[3];
    const long V = (long)Lx * Ly * Lz * T, V3 = (long)Lx * Ly * Lz;
    cplx *g = malloc(V * 12 * sizeof(cplx));
    cplx *l = malloc(V3 * 160 * sizeof(cplx));
    cplx g5G[16][4][4];
    make_g5G(g5G);
    make_g(g, s, eta, V, kappa, mu);
    for (int t = t0; t < t1; t++) {
#pragma omp parallel for schedule(static)
        for (long k = 0; k < V3; k++) {
            if (sym) loops_at_site_sym(l + k * 160, s, g, U, dims, tb, (long)t * V3 + k, g5G);
            else     loops_at_site(l + k * 160, s, g, U, dims, tb, (long)t * V3 + k, g5G);
        }
#pragma omp parallel for schedule(dynamic, 1)
        for (int q = 0; q < nmom; q++) {
            cplx acc[160];
            memset(acc, 0, sizeof(acc));
            for (int z = 0; z < Lz; z++)
                for (int y = 0; y < Ly; y++)
                    for (int x = 0; x < Lx; x++) {
                        const double ph = 2.0 * M_PI * ((double)momenta[q * 3 + 0] * x / Lx
                                                        + (double)momenta[q * 3 + 1] * y / Ly
                                                        + (double)momenta[q * 3 + 2] * z / Lz);
                        const cplx e = cos(ph) + I * sin(ph);
                        const cplx *lx = l + (((long)z * Ly + y) * Lx + x) * 160;
                        for (int j = 0; j < 160; j++) acc[j] += e * lx[j];
                    }
            for (int j = 0; j < 160; j++) out[((long)j * nmom + q) * T + t] = acc[j];
        }
    }
    free(g); free(l);
}

void orc_loops_project(cplx *out, const cplx *s, const cplx *eta, const cplx *U, const int *dims,
                       int tb, double kappa, double mu, const int *momenta, int nmom,
                       int t0, int t1)
{
    loops_project_impl(out, s, eta, U, dims, tb, kappa, mu, momenta, nmom, t0, t1, 0);
}

/* same with the symmetrised derivative (loops_at_site_sym) */
void orc_loops_project_sym(cplx *out, const cplx *s, const cplx *eta, const cplx *U, const int *dims,
                           int tb, double kappa, double mu, const int *momenta, int nmom,
                           int t0, int t1)
{
    loops_project_impl(out, s, eta, U, dims, tb, kappa, mu, momenta, nmom, t0, t1, 1);
}

/* ------------------------------------------------------- time dilution (row f4) */
/* PAPER.md:88 "we also worked with time-dilution [6], so there are GPU kernels to contract a single time slice or a
 * whole vector" + DESIGN.md reading 22.  A time-diluted source eta^(t0) is the noise vector restricted to timeslice t0
 * (zero elsewhere); with M s^(t0) = eta^(t0) the plain stochastic estimator of the loop on that timeslice is
 *     l[i][k][t0] = sum_{x in t0} exp(+2 pi i p_k.x/L)  eta^(t0)(x)^dag  X_i  s^(t0)(x),
 *     X_n = Gamma_n (n < 16),   X_{16+16m+n} = Gamma_n D_m   (D_m acting on s: reading 4)
 * (E[eta eta^dag] = 1 on the timeslice, so E[l] = sum_x e^{ipx} tr[X_i M^-1(x,x)]; the noise of the other T-1
 * timeslices never enters: that is the variance reduction).  The function below is the bilinear itself for any pair
 * (a, b) and timeslices t0 <= t < t1, by the direct sum:
 *     out[(i*nmom + k)*T + t] = sum_{x,y,z} exp(+2 pi i p_k.x/L) a(x,t)^dag X_i b(x,t);
 * entries of out for other t are left untouched. */
void orc_plain_loops_project(cplx *out, const cplx *a, const cplx *b, const cplx *U, const int *dims,
                             int tb, const int *momenta, int nmom, int t0, int t1)
{
    const int Lx = dims[0], Ly = dims[1], Lz = dims[2], T = dims[3];
    const long V3 = (long)Lx * Ly * Lz;
    cplx *l = malloc(V3 * 80 * sizeof(cplx));
    cplx G[16][4][4];
    for (int n = 0; n < 16; n++) Gamma_mat(n, G[n]);
    for (int t = t0; t < t1; t++) {
#pragma omp parallel for schedule(static)
        for (long k = 0; k < V3; k++) {
            const long x = (long)t * V3 + k;
            cplx *o = l + k * 80;
            for (int n = 0; n < 16; n++) o[n] = bilinear(a + x * 12, G[n], b + x * 12);
            for (int m = 0; m < 4; m++) {
                cplx d[12];
                cov_deriv_site(d, b, U, dims, tb, x, m);
                for (int n = 0; n < 16; n++) o[16 + 16 * m + n] = bilinear(a + x * 12, G[n], d);
            }
        }
#pragma omp parallel for schedule(dynamic, 1)
        for (int q = 0; q < nmom; q++) {
            cplx acc[80];
            memset(acc, 0, sizeof(acc));
            for (int z = 0; z < Lz; z++)
                for (int y = 0; y < Ly; y++)
                    for (int x = 0; x < Lx; x++) {
                        const double ph = 2.0 * M_PI * ((double)momenta[q * 3 + 0] * x / Lx
                                                        + (double)momenta[q * 3 + 1] * y / Ly
                                                        + (double)momenta[q * 3 + 2] * z / Lz);
                        const cplx e = cos(ph) + I * sin(ph);
                        const cplx *lx = l + (((long)z * Ly + y) * Lx + x) * 80;
                        for (int j = 0; j < 80; j++) acc[j] += e * lx[j];
                    }
            for (int j = 0; j < 80; j++) out[((long)j * nmom + q) * T + t] = acc[j];
        }
    }
    free(l);
}

/* eta^(t0): the noise vector restricted to timeslice t0 (PAPER.md:88 time-dilution; reading 22) */
void orc_time_dilute(cplx *out, const cplx *eta, const int *dims, int t0)
{
    const long V3 = (long)dims[0] * dims[1] * dims[2], V = V3 * dims[3];
    for (long j = 0; j < V * 12; j++) out[j] = 0;
    for (long j = 0; j < V3 * 12; j++) out[(long)t0 * V3 * 12 + j] = eta[(long)t0 * V3 * 12 + j];
}

/* ------------------------------------------------------- hopping parameter expansion (row f4) */
/* PAPER.md:92 "... variance reduction methods, namely the TSM, the one-end trick ..., time-dilution and the Hopping
 * Parameter Expansion (HPE) [7]" + DESIGN.md reading 23.  Split M = A - H with the site-local A = 1 + 2 i kappa mu g5
 * and the hopping part H = A - M (= kappa * sum of the eight hops).  For every n >= 0, exactly,
 *     M^-1 = sum_{k<n} (A^-1 H)^k A^-1  +  (A^-1 H)^n M^-1 .
 * The loop tr[X M^-1] is the sum of an exact part (first sum: no noise) and a remainder estimated stochastically with
 * the same solution s = M^-1 eta:  eta^dag X (A^-1 H)^n s.
 *
 * orc_apply_AinvH: out = A^-1 (A in - M in), one factor of the expansion, from the definition H = A - M;
 * A^-1 = (1 - 2 i kappa mu g5) / (1 + 4 kappa^2 mu^2) because g5^2 = 1. */
void orc_apply_AinvH(cplx *out, const cplx *in, const cplx *U, const int *dims, int tb, double kappa, double mu)
{
    const long V = (long)dims[0] * dims[1] * dims[2] * dims[3];
    cplx g5[4][4];
    gamma_mat(4, g5);
    const double a = 2.0 * kappa * mu;
    cplx *Min = malloc(V * 12 * sizeof(cplx));
    orc_apply_M(Min, in, U, dims, tb, kappa, mu, 0);
    for (long x = 0; x < V; x++)
        for (int c = 0; c < 3; c++) {
            cplx w[4];                          /* w = A in - M in at this site and colour */
            for (int s = 0; s < 4; s++) {
                cplx g5in = 0;
                for (int s2 = 0; s2 < 4; s2++) g5in += g5[s][s2] * in[x * 12 + s2 * 3 + c];
                w[s] = in[x * 12 + s * 3 + c] + I * a * g5in - Min[x * 12 + s * 3 + c];
            }
            for (int s = 0; s < 4; s++) {
                cplx g5w = 0;
                for (int s2 = 0; s2 < 4; s2++) g5w += g5[s][s2] * w[s2];
                out[x * 12 + s * 3 + c] = (w[s] - I * a * g5w) / (1.0 + a * a);
            }
        }
    free(Min);
}

/* Exact part of the expansion, by brute force (column j of the operator from the unit vector e_j, for all 12 V of them):
 *     out[(i*nmom + q)*T + t] = sum_{x in t} exp(+2 pi i p_q.x/L) tr_{spin,colour}[ ( X_i S_i )(x,x) ],
 *     S_i = sum_{k < n_i} (A^-1 H)^k A^-1,   n_i = order_local for the ultra-local X_i = Gamma_n (i < 16),
 *                                            n_i = order_deriv for X_{16+16m+n} = Gamma_n D_m.
 * O(V^2): for the small lattices of the tests only. */
void orc_hpe_exact(cplx *out, const cplx *U, const int *dims, int tb, double kappa, double mu,
                   int order_local, int order_deriv, const int *momenta, int nmom)
{
    const int Lx = dims[0], Ly = dims[1], Lz = dims[2], T = dims[3];
    const long V = (long)Lx * Ly * Lz * T;
    const double a = 2.0 * kappa * mu;
    const int nmax = order_local > order_deriv ? order_local : order_deriv;
    cplx G[16][4][4], g5[4][4];
    for (int n = 0; n < 16; n++) Gamma_mat(n, G[n]);
    gamma_mat(4, g5);
    cplx *site = calloc(V * 80, sizeof(cplx));          /* tr[(X_i S_i)(x,x)] for every site x */
    cplx *w = malloc(V * 12 * sizeof(cplx)), *w2 = malloc(V * 12 * sizeof(cplx));
    cplx *Sl = malloc(V * 12 * sizeof(cplx)), *Sd = malloc(V * 12 * sizeof(cplx));
    for (long x0 = 0; x0 < V; x0++)
        for (int j = 0; j < 12; j++) {
            /* w = A^-1 e_j (k = 0), then w <- A^-1 H w; Sl, Sd = the partial sums applied to e_j */
            for (long i = 0; i < V * 12; i++) { w[i] = 0; Sl[i] = 0; Sd[i] = 0; }
            const int sp = j / 3, c = j % 3;
            for (int s = 0; s < 4; s++) w[x0 * 12 + s * 3 + c] = ((s == sp ? 1.0 : 0.0) - I * a * g5[s][sp]) / (1.0 + a * a);
            for (int k = 0; k < nmax; k++) {
                if (k < order_local) for (long i = 0; i < V * 12; i++) Sl[i] += w[i];
                if (k < order_deriv) for (long i = 0; i < V * 12; i++) Sd[i] += w[i];
                if (k + 1 < nmax) {
                    orc_apply_AinvH(w2, w, U, dims, tb, kappa, mu);
                    memcpy(w, w2, V * 12 * sizeof(cplx));
                }
            }
            /* diagonal entry (x0, j) of X_i S_i: component j at site x0 of X_i applied to the column */
            for (int n = 0; n < 16; n++) {
                cplx acc = 0;
                for (int s2 = 0; s2 < 4; s2++) acc += G[n][sp][s2] * Sl[x0 * 12 + s2 * 3 + c];
                site[x0 * 80 + n] += acc;
            }
            for (int m = 0; m < 4; m++) {
                cplx d[12];
                cov_deriv_site(d, Sd, U, dims, tb, x0, m);
                for (int n = 0; n < 16; n++) {
                    cplx acc = 0;
                    for (int s2 = 0; s2 < 4; s2++) acc += G[n][sp][s2] * d[s2 * 3 + c];
                    site[x0 * 80 + 16 + 16 * m + n] += acc;
                }
            }
        }
    for (int q = 0; q < nmom; q++)
        for (int t = 0; t < T; t++) {
            cplx acc[80];
            memset(acc, 0, sizeof(acc));
            for (int z = 0; z < Lz; z++)
                for (int y = 0; y < Ly; y++)
                    for (int x = 0; x < Lx; x++) {
                        const double ph = 2.0 * M_PI * ((double)momenta[q * 3 + 0] * x / Lx
                                                        + (double)momenta[q * 3 + 1] * y / Ly
                                                        + (double)momenta[q * 3 + 2] * z / Lz);
                        const cplx e = cos(ph) + I * sin(ph);
                        const cplx *lx = site + ((((long)t * Lz + z) * Ly + y) * Lx + x) * 80;
                        for (int i = 0; i < 80; i++) acc[i] += e * lx[i];
                    }
            for (int i = 0; i < 80; i++) out[((long)i * nmom + q) * T + t] = acc[i];
        }
    free(site); free(w); free(w2); free(Sl); free(Sd);
}

/* sec 2.1 + reading 14:
 *   L_TSM = (1/N_LP) sum_{r<N_LP} l_r^LP + (1/N_HP) sum_{r<N_HP} (l_r^HP - l_r^LP)
 * lp: [n_lp][len], hp: [n_hp][len] (HP sources = first n_hp LP sources). */
void orc_tsm_combine(cplx *out, const cplx *lp, int n_lp, const cplx *hp, int n_hp, long len)
{
    for (long j = 0; j < len; j++) {
        cplx a = 0, b = 0;
        for (int r = 0; r < n_lp; r++) a += lp[(long)r * len + j];
        for (int r = 0; r < n_hp; r++) b += hp[(long)r * len + j] - lp[(long)r * len + j];
        out[j] = a / n_lp + (n_hp > 0 ? b / n_hp : 0);
    }
}

/* sec 2.1.1 (Fig. 2) + DESIGN.md reading 21: binary storage of partial sums.
 * "in File.1 we store the contractions generated with one stochastic source, in File.2 we store the
 * sum of the contractions coming from the second and the third stochastic source, and so on":
 * file k = 0,1,2,... (the paper's File.2^k) holds the sum over the 2^k sources r = 2^k - 1 ... 2^(k+1) - 2.
 * per_source: [n][len]; files: [nfiles][len] with nfiles = floor(log2(n)) + 1 (the last file may be
 * incomplete when n + 1 is not a power of two); counts[k] = number of sources summed into file k. */
void orc_binary_store(cplx *files, int *counts, const cplx *per_source, int n, long len)
{
    int nfiles = 0;
    while (((1L << nfiles) - 1) < n) nfiles++;          /* smallest K with 2^K - 1 >= n */
    for (int k = 0; k < nfiles; k++) {
        counts[k] = 0;
        for (long j = 0; j < len; j++) files[(long)k * len + j] = 0;
    }
    for (int r = 0; r < n; r++) {
        int k = 0;
        while (((1L << (k + 1)) - 1) <= r) k++;          /* 2^k - 1 <= r < 2^(k+1) - 1 */
        counts[k] += 1;
        for (long j = 0; j < len; j++) files[(long)k * len + j] += per_source[(long)r * len + j];
    }
}

/* "Reconstruction is straightforward, taking into account the base-2 structure": the estimator from N
 * sources is the sum of the files whose weight 2^k is a binary digit of N, divided by N (Fig. 2:
 * N = 13 = 1101b -> the files with 1, 4 and 8 sources).  "With this storage method one can recover the
 * data for any number of sources": the one N the digits rule cannot serve while the last
 * file is still filling is the number of sources stored so far, n = sum_k counts[k]; for N = n the
 * estimator is the sum of EVERY file, the partial one included, divided by n (reading 21).
 * Returns 0, or -1 when N is neither n nor made of complete files (counts[k] == 2^k). */
int orc_binary_recover(cplx *out, const cplx *files, const int *counts, int nfiles, int N, long len)
{
    if (N < 1) return -1;
    long n = 0;
    for (int k = 0; k < nfiles; k++) n += counts[k];
    if (N == n) {                                        /* everything stored so far */
        for (long j = 0; j < len; j++) {
            out[j] = 0;
            for (int k = 0; k < nfiles; k++) out[j] += files[(long)k * len + j];
            out[j] /= N;
        }
        return 0;
    }
    for (int k = 0; (1L << k) <= N; k++)
        if ((N >> k) & 1)
            if (k >= nfiles || counts[k] != (1 << k)) return -1;
    for (long j = 0; j < len; j++) out[j] = 0;
    for (int k = 0; (1L << k) <= N; k++)
        if ((N >> k) & 1)
            for (long j = 0; j < len; j++) out[j] += files[(long)k * len + j];
    for (long j = 0; j < len; j++) out[j] /= N;
    return 0;
}
