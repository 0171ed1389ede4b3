// contract.cu -- fused one-end-trick contraction + momentum projection.
//
// PAPER.md:86 "traces were taken in color space, leaving the Dirac ... indices open";
// PAPER.md:72 "all ultra-local and one-derivative insertions, with and without tau3 ... 160 insertions";
// PAPER.md:88 "returning an array with a time-slice index"; PAPER.md:94-100 Fourier transform + p^2 cut.
//
// Per site x the kernel forms the 10 spinors  psi_{fam,d}:  fam in {s, eta},  d = 0: psi(x),
// d = 1+mu: 2 D_mu psi(x) = U_mu(x) psi(x+mu) - U_mu^dag(x-mu) psi(x-mu)   (PAPER.md:86 covariant derivative)
// and their colour-traced outer products with s,
//     C_{fam,d}[a][b](x) = sum_c conj(s_{a c}(x)) psi_{fam,d; b c}(x)       (16 complex each, 160 in total)
// which never leave the SM: they are reduced against cos/sin(2 pi m x / Lx) along x (m = 0..3) and
// cos/sin(2 pi n y / Ly) along y inside the CTA that owns one (z,t) plane (separable partial DFT, real
// weights).  A second small kernel does the z sum, assembles the complex exponential for every
// requested momentum and applies the site-independent change of basis
//     l_{0,n} = sum_a ph_n(a) C_{s,d}[a][perm_n(a)]   with (g5 Gamma_n)[a][b] = ph_n(a) delta_{b,perm_n(a)}
//     l_{1,n} = sum_a ph_n(a) g5(perm_n(a)) C_{eta,d}[a][perm_n(a)] - 2 i kappa mu l_{0,n}
// (g = g5 eta - 2 i kappa mu s, reading 5), times 1/2 for the derivative insertions.
//
// Kernel 1 is warp-specialised (see contract_xy_kernel): producer warps (lane = x) compute the 16
// complex numbers of C_{fam,d}(x) into a shared-memory ring of row buffers, consumer warps (thread =
// one complex component) do the x-sum with 7 real weights and the y-stage update of their NQ register
// accumulators Q[(m,n),(cos|sin)x,(cos|sin)y].
#include <math.h>
#include <complex>
#include <vector>
#include "contract.cuh"

// Warp-specialised CTA, one (z,t) plane per CTA:
//   NP producer warps (lane = x): jobs (fam, d) of one row chunk -> psi_{fam,d}(x), colour-traced outer
//     product with s(x) -> row buffer (NS-stage ring in shared memory)
//   CT_NC consumer warps (thread = complex component): x-sum of the row buffer with the 7 real weights,
//     y-stage update of the NQ register accumulators; written to qbuf at the end of the plane.
// Producers never hold the Q accumulators and consumers never hold spinors, so neither role pays the
// other's registers; the ring lets the global loads of row y+1 overlap the DFT of row y.
template <typename S, int R, int PRUNE, int NP, int NS>
__global__ void __launch_bounds__((NP + CT_NC) * 32, 1) contract_xy_kernel(ContractArgs A) {
    typedef S F;
    typedef typename P2<F>::T T;
    constexpr int NQ = QLayout<PRUNE>::NQ;
    constexpr int NTHREADS = (NP + CT_NC) * 32;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* buf = reinterpret_cast<T*>(smem_raw);                     // [NS][160][CT_BSC]
    F* swx = reinterpret_cast<F*>(buf + (size_t)NS * CT_NCC * CT_BSC);   // [Lx][8]
    F* swy = swx + (size_t)A.g.X0 * 8;                           // [Ly][8]
    const Geom& g = A.g;
    const int zt = blockIdx.x + A.t_first * g.X2;
    const int z = zt % g.X2, t = zt / g.X2;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int i = threadIdx.x; i < g.X0 * 8; i += NTHREADS) swx[i] = ((const F*)A.wx)[i];
    for (int i = threadIdx.x; i < g.X1 * 8; i += NTHREADS) swy[i] = ((const F*)A.wy)[i];
    __syncthreads();

    const int nxc = (g.X0 + 31) / 32;
    const int niter = g.X1 * nxc;
    // barrier ids: full[st] = 1 + st, empty[st] = 1 + NS + st
    if (warp < NP) {
        // ================================================================ producers
        const S* sfield = (const S*)A.s;
        const S* efield = (const S*)A.eta;
        const S* gauge = (const S*)A.gauge;
        const size_t Vh = g.Vh;
        const size_t pblk = Vh * 24;
        for (int it = 0; it < niter; it++) {
            const int st = it % NS;
            const int y = it / nxc, xc = it - y * nxc;
            const int x = xc * 32 + lane;
            T* rowbuf = buf + (size_t)st * CT_NCC * CT_BSC;
            if (it >= NS) named_bar_sync(1 + NS + st, NTHREADS);
            if (x < g.X0) {
                const int par = (x + y + z + t) & 1;
                const int row = ((t * g.X2 + z) * g.X1 + y) * g.X0;      // lex index of x = 0
                const size_t h = (size_t)(row + x) >> 1;
                T sv[12];
                load_spinor_pairs<S>(sfield + par * pblk, Vh, h, sv);
                // ---- heavy jobs: derivative directions
#pragma unroll 1
                for (int job = warp; job < 8; job += NP) {
                    const int fam = job >> 2, mu = job & 3;
                    const S* pfield = fam ? efield : sfield;
                    int lf, lb;
                    bool wf = false, wb = false;
                    if (mu == 0) {
                        lf = row + (x + 1 == g.X0 ? 0 : x + 1);
                        lb = row + (x == 0 ? g.X0 - 1 : x - 1);
                    } else if (mu == 1) {
                        const int sd = g.X0;
                        lf = (y + 1 == g.X1) ? row + x - (g.X1 - 1) * sd : row + x + sd;
                        lb = (y == 0) ? row + x + (g.X1 - 1) * sd : row + x - sd;
                    } else if (mu == 2) {
                        const int sd = g.X0 * g.X1;
                        lf = (z + 1 == g.X2) ? row + x - (g.X2 - 1) * sd : row + x + sd;
                        lb = (z == 0) ? row + x + (g.X2 - 1) * sd : row + x - sd;
                    } else {
                        const int sd = g.X0 * g.X1 * g.X2;
                        if (t + 1 == g.X3) { lf = row + x - (g.X3 - 1) * sd; wf = true; } else lf = row + x + sd;
                        if (t == 0) { lb = row + x + (g.X3 - 1) * sd; wb = true; } else lb = row + x - sd;
                    }
                    const size_t hf = (size_t)lf >> 1, hb = (size_t)lb >> 1;
                    T nb[12], psi[12];
                    F U[18];
#pragma unroll
                    for (int i = 0; i < 12; i++) psi[i] = P2<F>::make(0, 0);
                    load_spinor_pairs<S>(pfield + (1 - par) * pblk, Vh, hf, nb);
                    load_link<S, R, LD_DEFAULT>(gauge, Vh, par, mu, h, U);
                    if (wf) {
#pragma unroll
                        for (int i = 0; i < 12; i++) nb[i] = P2<F>::mul_s((F)A.tb, nb[i]);
                    }
                    su3_macc<0, 0, F>(U, nb, psi);
                    load_spinor_pairs<S>(pfield + (1 - par) * pblk, Vh, hb, nb);
                    load_link<S, R, LD_DEFAULT>(gauge, Vh, 1 - par, mu, hb, U);
                    if (wb) {
#pragma unroll
                        for (int i = 0; i < 12; i++) nb[i] = P2<F>::mul_s((F)A.tb, nb[i]);
                    }
                    su3_macc<1, 1, F>(U, nb, psi);
                    outer_store<F>(sv, psi, rowbuf, fam * 5 + 1 + mu, lane);
                }
                // ---- light jobs (d = 0), rotated over the producer warps
                const int lw = (2 * it) % NP;
                if (warp == lw) outer_store<F>(sv, sv, rowbuf, 0, lane);
                if (warp == (lw + 1) % NP) {
                    T ev[12];
                    load_spinor_pairs<S>(efield + par * pblk, Vh, h, ev);
                    outer_store<F>(sv, ev, rowbuf, 5, lane);
                }
            }
            __syncwarp();
            named_bar_arrive(1 + st, NTHREADS);
        }
    } else {
        // ================================================================ consumers
        const int cc = threadIdx.x - NP * 32;        // 0..159
        T Q[NQ];
#pragma unroll
        for (int q = 0; q < NQ; q++) Q[q] = P2<F>::make(0, 0);
        T a0 = P2<F>::make(0, 0), ac[3], as[3];
#pragma unroll
        for (int m = 0; m < 3; m++) { ac[m] = P2<F>::make(0, 0); as[m] = P2<F>::make(0, 0); }
        for (int it = 0; it < niter; it++) {
            const int st = it % NS;
            const int y = it / nxc, xc = it - y * nxc;
            const T* v = buf + ((size_t)st * CT_NCC + cc) * CT_BSC;
            const F* w = swx + (size_t)xc * 32 * 8;
            const int nvalid = min(32, g.X0 - xc * 32);
            named_bar_sync(1 + st, NTHREADS);
#pragma unroll 4
            for (int l = 0; l < nvalid; l++) {
                const T val = v[l];
                const F* wl = w + l * 8;
                a0 = P2<F>::add(a0, val);
#pragma unroll
                for (int m = 0; m < 3; m++) {
                    ac[m] = P2<F>::fma_s(wl[2 * m + 1], val, ac[m]);
                    as[m] = P2<F>::fma_s(wl[2 * m + 2], val, as[m]);
                }
            }
            if (it + NS < niter) named_bar_arrive(1 + NS + st, NTHREADS);
            if (xc == nxc - 1) {
                // ---------------------------------------------------------------- y-stage
                const F* wl = swy + y * 8;
                F cy[4], sy[4];
                cy[0] = 1; sy[0] = 0;
                cy[1] = wl[1]; sy[1] = wl[2]; cy[2] = wl[3]; sy[2] = wl[4]; cy[3] = wl[5]; sy[3] = wl[6];
                int q = 0;
#pragma unroll
                for (int m = 0; m < 4; m++)
#pragma unroll
                    for (int n = 0; n < 4; n++) {
                        if (!PRUNE || m * m + n * n <= 9) {
                            const T xcm = m ? ac[m - 1] : a0;
                            if (n == 0) Q[q] = P2<F>::add(Q[q], xcm); else Q[q] = P2<F>::fma_s(cy[n], xcm, Q[q]);
                            q++;
                            if (n > 0) { Q[q] = P2<F>::fma_s(sy[n], xcm, Q[q]); q++; }
                            if (m > 0) {
                                if (n == 0) Q[q] = P2<F>::add(Q[q], as[m - 1]); else Q[q] = P2<F>::fma_s(cy[n], as[m - 1], Q[q]);
                                q++;
                            }
                            if (m > 0 && n > 0) { Q[q] = P2<F>::fma_s(sy[n], as[m - 1], Q[q]); q++; }
                        }
                    }
                a0 = P2<F>::make(0, 0);
#pragma unroll
                for (int m = 0; m < 3; m++) { ac[m] = P2<F>::make(0, 0); as[m] = P2<F>::make(0, 0); }
            }
        }
        T* qb = reinterpret_cast<T*>((F*)A.qbuf + (size_t)zt * NQ * CT_THREADS) + cc;
#pragma unroll
        for (int q = 0; q < NQ; q++) qb[(size_t)q * CT_NCC] = Q[q];
    }
}

// ------------------------------------------------------------------ kernel 2: z-sum + assembly
struct GammaTable {
    signed char perm[16][4];     // column of the nonzero of row a of g5 Gamma_n
    signed char phre[16][4];     // its value (one of +-1, +-i)
    signed char phim[16][4];
};
__constant__ GammaTable c_gamma;

struct AssembleArgs {
    const void* qbuf;          // [T*Lz][NQ][320] (F precision): x/y partial sums per (z,t) plane
    double* zbuf;              // [T][NQ][7][320]: z-stage sums with weights 1, c1, s1, c2, s2, c3, s3
    void* out;                 // complex128 [2][80][nmom][T]
    const int* mom;            // [nmom][3]
    const short* qidx;         // [4][4][4]: index of Qcc, Qcs, Qsc, Qss for (m,n), -1 if absent
    const double* wz;          // [Lz][8]
    int nmom, T, Lz, NQ;
    int t_first;               // first timeslice handled (blockIdx.y = 0)
    double twokmu;             // 2 kappa mu
    int half0;                 // s-family derivative slots hold only the forward half F_mu (contract_mma.cu); every
                               // timeslice must have been summed
    int L[3];                  // Lx, Ly, Lz
    // by-value copies (constant bank: no dependent global loads at the start of each of the nmom x T small CTAs of the
    // assembly); mom_v is used when nmom <= AS_MOMV, else the kernel reads A.mom
    short qidx_v[64];
    int mom_v[3 * 128];
};
#define AS_MOMV 128

// z-stage: every x/y partial sum is read exactly once and reduced against the 7 real z-weights
template <typename F>
__global__ void __launch_bounds__(CT_THREADS) contract_zsum_kernel(AssembleArgs A) {
    const int q = blockIdx.x, t = blockIdx.y + A.t_first, jr = threadIdx.x;
    const F* qb = (const F*)A.qbuf + ((size_t)t * A.Lz * A.NQ + q) * CT_THREADS + jr;
    double acc[7];
#pragma unroll
    for (int k = 0; k < 7; k++) acc[k] = 0.0;
    // the 6 weights of a z value from shared memory: as global loads they were 6 of the 7 loads of an iteration and kept
    // the data loads from overlapping
    extern __shared__ double swz[];                         // [Lz][8]
    for (int i = threadIdx.x; i < A.Lz * 8; i += CT_THREADS) swz[i] = A.wz[i];
    __syncthreads();
#pragma unroll 4
    for (int z = 0; z < A.Lz; z++) {
        const double v = (double)qb[(size_t)z * A.NQ * CT_THREADS];
        const double* w = swz + z * 8;
        acc[0] += v;
#pragma unroll
        for (int k = 1; k < 7; k++) acc[k] += w[k] * v;
    }
    double* zb = A.zbuf + (((size_t)t * A.NQ + q) * 7) * CT_THREADS + jr;
#pragma unroll
    for (int k = 0; k < 7; k++) zb[(size_t)k * CT_THREADS] = acc[k];
}

// assembly of exp(+2 pi i p.x / L) for every requested momentum from the (cos|sin)^3 sums, then the
// site-independent Gamma change of basis
__global__ void __launch_bounds__(CT_THREADS) contract_assemble_kernel(AssembleArgs A) {
    __shared__ double zre[CT_THREADS], zim[CT_THREADS];
    __shared__ double zre_tm[32], zim_tm[32];               // half0: the t-derivative slot of the s family at t - 1
    // every thread reads its own row of the Gamma table: from __constant__ memory that serialises in the constant
    // cache (16 distinct addresses per warp and access), so the table is staged in shared memory once per CTA
    __shared__ GammaTable sg;
    const int k = blockIdx.x, t = blockIdx.y + A.t_first;
    const int jr = threadIdx.x;
    if (jr < (int)(sizeof(GammaTable) / 4)) reinterpret_cast<int*>(&sg)[jr] = reinterpret_cast<const int*>(&c_gamma)[jr];
    const int* momk = A.nmom <= AS_MOMV ? A.mom_v + 3 * k : A.mom + 3 * k;
    const int px = momk[0], py = momk[1], pz = momk[2];
    const int m = abs(px), n = abs(py), l = abs(pz);
    const double sx = px < 0 ? -1.0 : 1.0, sy = py < 0 ? -1.0 : 1.0, sz = pz < 0 ? -1.0 : 1.0;
    const short* qi = A.qidx_v + (m * 4 + n) * 4;
    // Z(tq) = sum over the timeslice of exp(+i p.x) times real component jr
    auto Zof = [&](int tq, double& re, double& im) {
        const double* zb = A.zbuf + (size_t)tq * A.NQ * 7 * CT_THREADS + jr;
        // X[c] = sum_z cos(2 pi l z / L) Q_X(z), X[s] = sum_z sin(...) Q_X(z) for X in cc, cs, sc, ss
        double C[4], S[4];
#pragma unroll
        for (int x = 0; x < 4; x++) {
            const int iq = qi[x];
            C[x] = 0.0; S[x] = 0.0;
            if (iq >= 0) {
                const double* e = zb + (size_t)iq * 7 * CT_THREADS;
                C[x] = l ? e[(size_t)(2 * l - 1) * CT_THREADS] : e[0];
                S[x] = l ? e[(size_t)(2 * l) * CT_THREADS] : 0.0;
            }
        }
        // (cos mx + i sx sin mx)(cos ny + i sy sin ny)(cos lz + i sz sin lz)
        const double wrC = C[0] - sx * sy * C[3], wiC = sx * C[2] + sy * C[1];
        const double wrS = S[0] - sx * sy * S[3], wiS = sx * S[2] + sy * S[1];
        re = wrC - sz * wiS;
        im = wiC + sz * wrS;
    };
    Zof(t, zre[jr], zim[jr]);
    if (A.half0 && jr >= 4 * 32 && jr < 5 * 32) Zof(t == 0 ? A.T - 1 : t - 1, zre_tm[jr - 4 * 32], zim_tm[jr - 4 * 32]);
    __syncthreads();
    if (jr < 160) {
        const int f = jr / 80, i = jr % 80;
        const int nG = i < 16 ? i : (i - 16) & 15;
        const int d = i < 16 ? 0 : 1 + ((i - 16) >> 4);
        const double scale = d ? 0.5 : 1.0;
        // half0: C~[a][b](p,t) = F~[a][b](p,t) - e^{i p_mu} conj(F~[b][a](-p,t')), and for real fields Z(-p) = conj(Z(p))
        double phr = 1.0, phi = 0.0;
        if (A.half0 && d >= 1 && d <= 3) sincospi(2.0 * (double)momk[d - 1] / (double)A.L[d - 1], &phi, &phr);
        const double* br_ = (d == 4) ? zre_tm - 4 * 32 : zre;
        const double* bi_ = (d == 4) ? zim_tm - 4 * 32 : zim;
        double l0r = 0, l0i = 0, l1r = 0, l1i = 0;
#pragma unroll
        for (int a = 0; a < 4; a++) {
            const int bcol = sg.perm[nG][a];
            const double pr = sg.phre[nG][a], pi = sg.phim[nG][a];
            {   // s family: raw complex value = (Z[re comp]) + i (Z[im comp]) with each Z complex
                const int j = (d * 32) + (a * 4 + bcol) * 2;
                double rr = zre[j] - zim[j + 1], ri = zim[j] + zre[j + 1];
                if (A.half0 && d) {
                    const int jt = (d * 32) + (bcol * 4 + a) * 2;            // transposed component
                    const double cr = br_[jt] + bi_[jt + 1], ci = bi_[jt] - br_[jt + 1];   // conj(F~[b][a](-p))
                    rr -= phr * cr - phi * ci;
                    ri -= phr * ci + phi * cr;
                }
                l0r += pr * rr - pi * ri;
                l0i += pr * ri + pi * rr;
            }
            if (f) {
                const int j = ((5 + d) * 32) + (a * 4 + bcol) * 2;
                const double g5 = bcol < 2 ? 1.0 : -1.0;
                const double rr = g5 * (zre[j] - zim[j + 1]), ri = g5 * (zim[j] + zre[j + 1]);
                l1r += pr * rr - pi * ri;
                l1i += pr * ri + pi * rr;
            }
        }
        double outr, outi;
        if (f == 0) { outr = scale * l0r; outi = scale * l0i; }
        else {      // l1 - 2 i kappa mu l0
            outr = scale * (l1r + A.twokmu * l0i);
            outi = scale * (l1i - A.twokmu * l0r);
        }
        double* o = (double*)A.out + 2 * ((((size_t)f * 80 + i) * A.nmom + k) * A.T + t);
        o[0] = outr; o[1] = outi;
    }
}

// ------------------------------------------------------------------ host side
typedef std::complex<double> cd;
static void mat4mul(cd c[4][4], const cd a[4][4], const cd b[4][4]) {
    cd t[4][4];
    for (int i = 0; i < 4; i++)
        for (int j = 0; j < 4; j++) {
            cd s = 0;
            for (int k = 0; k < 4; k++) s += a[i][k] * b[k][j];
            t[i][j] = s;
        }
    memcpy(c, t, sizeof(t));
}

// chiral basis of dslash.cu: g_mu = [[0, B],[B^dag, 0]], B_k = -i sigma_k, B_t = 1
static void build_gamma_table(GammaTable* G) {
    const cd I(0, 1);
    cd sig[4][2][2] = {{{0, 1}, {1, 0}}, {{0, -I}, {I, 0}}, {{1, 0}, {0, -1}}, {{1, 0}, {0, 1}}};
    cd gam[4][4][4];
    memset(gam, 0, sizeof(gam));
    for (int mu = 0; mu < 4; mu++)
        for (int i = 0; i < 2; i++)
            for (int j = 0; j < 2; j++) {
                const cd B = (mu < 3) ? -I * sig[mu][i][j] : sig[3][i][j];
                gam[mu][i][2 + j] = B;
                gam[mu][2 + j][i] = std::conj(B);      // B^dag[j][i]
            }
    cd g5[4][4];
    memset(g5, 0, sizeof(g5));
    for (int i = 0; i < 4; i++) g5[i][i] = 1;
    for (int mu = 0; mu < 4; mu++) mat4mul(g5, g5, gam[mu]);   // g5 = gx gy gz gt
    for (int n = 0; n < 16; n++) {
        cd M[4][4];
        memcpy(M, g5, sizeof(M));
        for (int mu = 0; mu < 4; mu++)
            if ((n >> mu) & 1) mat4mul(M, M, gam[mu]);
        for (int a = 0; a < 4; a++) {
            int col = -1;
            for (int b = 0; b < 4; b++)
                if (std::abs(M[a][b]) > 0.5) col = b;
            G->perm[n][a] = (signed char)col;
            G->phre[n][a] = (signed char)lround(M[a][col].real());
            G->phim[n][a] = (signed char)lround(M[a][col].imag());
        }
    }
}

// weights[x][8] = 1, cos(2 pi x/L), sin(2 pi x/L), cos(2 pi 2x/L), sin(..), cos(2 pi 3x/L), sin(..), 0
static void fill_weights(double* w, int L) {
    for (int x = 0; x < L; x++) {
        w[x * 8 + 0] = 1.0; w[x * 8 + 7] = 0.0;
        for (int m = 1; m < 4; m++) {
            const int r = (m * x) % L;                  // exact argument reduction
            const double th = 2.0 * M_PI * (double)r / (double)L;
            w[x * 8 + 2 * m - 1] = cos(th);
            w[x * 8 + 2 * m] = sin(th);
        }
    }
}

struct ContractTables {      // device block layout (offsets in bytes)
    size_t off_wx32, off_wy32, off_wx64, off_wy64, off_wz, off_mom, off_qidx, total;
};
static ContractTables table_layout(const tm_ctx* c, int nmom) {
    ContractTables L;
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t r = o; o += (bytes + 255) & ~(size_t)255; return r; };
    L.off_wx32 = take((size_t)c->X[0] * 8 * 4);
    L.off_wy32 = take((size_t)c->X[1] * 8 * 4);
    L.off_wx64 = take((size_t)c->X[0] * 8 * 8);
    L.off_wy64 = take((size_t)c->X[1] * 8 * 8);
    L.off_wz = take((size_t)c->X[2] * 8 * 8);
    L.off_mom = take((size_t)nmom * 3 * 4);
    L.off_qidx = take(64 * 2);
    L.total = o;
    return L;
}

void tm_contract_qidx(short* qidx, int prune, int* nq) {
    int q = 0;
    for (int m = 0; m < 4; m++)
        for (int n = 0; n < 4; n++) {
            short* e = qidx + (m * 4 + n) * 4;
            e[0] = e[1] = e[2] = e[3] = -1;
            if (!prune || m * m + n * n <= 9) {
                e[0] = (short)q++;
                if (n > 0) e[1] = (short)q++;
                if (m > 0) e[2] = (short)q++;
                if (m > 0 && n > 0) e[3] = (short)q++;
            }
        }
    *nq = q;
}

template <typename S> struct XyConfig;
template <> struct XyConfig<float>  { static constexpr int NP = 8, NS = 3; };
template <> struct XyConfig<double> { static constexpr int NP = 4, NS = 2; };

template <typename S, int R>
static tm_status launch_xy(tm_ctx* ctx, const ContractArgs& A, int prune, int nt, cudaStream_t st) {
    constexpr int NP = XyConfig<S>::NP, NS = XyConfig<S>::NS;
    constexpr int NT = (NP + CT_NC) * 32;
    const size_t smem = (size_t)NS * CT_NCC * CT_BSC * 2 * sizeof(S) + (size_t)(ctx->X[0] + ctx->X[1]) * 8 * sizeof(S);
    if (smem > 227 * 1024) return tm_fail(ctx, TM_EDIM, "contract: Lx + Ly too large for the shared-memory weight tables");
    const unsigned grid = (unsigned)(ctx->X[2] * nt);
    if (prune) {
        TM_CUDA(ctx, cudaFuncSetAttribute(contract_xy_kernel<S, R, 1, NP, NS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        contract_xy_kernel<S, R, 1, NP, NS><<<grid, NT, smem, st>>>(A);
    } else {
        TM_CUDA(ctx, cudaFuncSetAttribute(contract_xy_kernel<S, R, 0, NP, NS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        contract_xy_kernel<S, R, 0, NP, NS><<<grid, NT, smem, st>>>(A);
    }
    TM_LAUNCH_CHECK(ctx, "contract_xy_kernel");
    return TM_OK;
}

tm_status tm_contract_internal(tm_ctx* ctx, void* d_out, const void* d_s, const void* d_eta, double kappa,
                               double mu, const int* h_momenta, int nmom, tm_prec acc, cudaStream_t st,
                               int t_first, int nt, int merge) {
    if (nt <= 0) { t_first = 0; nt = ctx->X[3]; }                 // default: every timeslice
    if (merge && (nt != ctx->X[3] || !tm_contract_merge_ok(ctx, acc)))
        return tm_fail(ctx, TM_EARG, "contract: merged sources need a whole-vector fp32 call on the TMA path");
    if (t_first < 0 || t_first + nt > ctx->X[3]) return tm_fail(ctx, TM_EARG, "contract: timeslice range outside the lattice");
    if (acc != TM_F64 && acc != TM_F32) return tm_fail(ctx, TM_EPREC, "contract: acc must be f32 or f64");
    if (!h_momenta || nmom < 1) return tm_fail(ctx, TM_EARG, "contract: need at least one momentum");
    int prune = 1;
    for (int k = 0; k < nmom; k++) {
        const int px = h_momenta[3 * k], py = h_momenta[3 * k + 1], pz = h_momenta[3 * k + 2];
        if (abs(px) > 3 || abs(py) > 3 || abs(pz) > 3)
            return tm_fail(ctx, TM_EARG, "contract: momentum components must lie in [-3, 3]");
        if (px * px + py * py > 9) prune = 0;
    }
    // tables (rebuilt only when the momentum list changes)
    const ContractTables L = table_layout(ctx, nmom);
    std::vector<unsigned char> host(L.total, 0);
    {
        std::vector<double> w((size_t)8 * (ctx->X[0] > ctx->X[1] ? ctx->X[0] : ctx->X[1]));
        fill_weights(w.data(), ctx->X[0]);
        for (int i = 0; i < ctx->X[0] * 8; i++) { ((float*)(host.data() + L.off_wx32))[i] = (float)w[i]; ((double*)(host.data() + L.off_wx64))[i] = w[i]; }
        fill_weights(w.data(), ctx->X[1]);
        for (int i = 0; i < ctx->X[1] * 8; i++) { ((float*)(host.data() + L.off_wy32))[i] = (float)w[i]; ((double*)(host.data() + L.off_wy64))[i] = w[i]; }
        fill_weights((double*)(host.data() + L.off_wz), ctx->X[2]);
        memcpy(host.data() + L.off_mom, h_momenta, (size_t)nmom * 12);
        int nq;
        tm_contract_qidx((short*)(host.data() + L.off_qidx), prune, &nq);
    }
    static_assert(sizeof(int) == 4, "int momenta");
    if (!ctx->h_contract_tables || ctx->contract_tables_bytes != L.total
        || memcmp(ctx->h_contract_tables, host.data(), L.total) != 0) {
        TM_CUDA(ctx, cudaStreamSynchronize(st));
        if (ctx->d_contract_tables) cudaFree(ctx->d_contract_tables);
        free(ctx->h_contract_tables);
        ctx->d_contract_tables = nullptr;
        ctx->h_contract_tables = malloc(L.total);
        if (!ctx->h_contract_tables) return tm_fail(ctx, TM_EALLOC, "contract: host allocation failed");
        memcpy(ctx->h_contract_tables, host.data(), L.total);
        ctx->contract_tables_bytes = L.total;
        if (cudaMalloc(&ctx->d_contract_tables, L.total) != cudaSuccess) {
            cudaGetLastError(); ctx->d_contract_tables = nullptr; free(ctx->h_contract_tables); ctx->h_contract_tables = nullptr;
            return tm_fail(ctx, TM_EALLOC, "contract: out of device memory");
        }
        TM_CUDA(ctx, cudaMemcpy(ctx->d_contract_tables, ctx->h_contract_tables, L.total, cudaMemcpyHostToDevice));
        GammaTable G;
        build_gamma_table(&G);
        TM_CUDA(ctx, cudaMemcpyToSymbol(c_gamma, &G, sizeof(G)));
    }
    const unsigned char* tb = (const unsigned char*)ctx->d_contract_tables;
    const int nq = prune ? 29 : 49;
    const size_t fsz = acc == TM_F64 ? 8 : 4;
    void* qbuf;
    TM_TRY(tm_ws(ctx, WS_CT_PLANES, (size_t)ctx->X[2] * ctx->X[3] * nq * CT_THREADS * fsz, &qbuf));
    const tm_recon rc = acc == TM_F64 ? TM_R18 : TM_R12;
    const void* gauge = nullptr;
    TM_TRY(tm_get_gauge(ctx, acc, rc, st, &gauge));

    ContractArgs A;
    A.s = d_s; A.eta = d_eta; A.gauge = gauge; A.qbuf = qbuf;
    A.wx = tb + (acc == TM_F64 ? L.off_wx64 : L.off_wx32);
    A.wy = tb + (acc == TM_F64 ? L.off_wy64 : L.off_wy32);
    A.g = tm_geom(ctx);
    A.tb = (double)ctx->tb;
    A.t_first = t_first;
    // The forward-only s family (half0: the backward half of the s-family derivative is the shifted conjugate transpose
    // of the forward half and is restored by contract_assemble_kernel from the same sums) needs timeslice t - 1 in the
    // assembly: whole-vector launches only.  contract_tma.cu uses it except under TM_OPT_CONTRACT_PATH 4; contract_mma.cu
    // always (measured at c4, profiles/r02_contract_paths.md: slower than contract_tma.cu although it issues fewer
    // FFMA2, so it is not the automatic choice).
    const bool whole = nt == ctx->X[3];
    const bool mma = acc == TM_F32 && whole && ctx->opt_contract == 3 && tm_contract_mma_usable(ctx);
    const bool tma = acc == TM_F32 && !mma && ctx->opt_contract != 1 && tm_contract_tma_usable(ctx);
    const bool half0 = mma || (tma && whole && ctx->opt_contract != 4);
    if (acc == TM_F64) TM_TRY((launch_xy<double, 18>(ctx, A, prune, nt, st)));
    else if (mma) TM_TRY(tm_contract_xy_mma(ctx, qbuf, d_s, d_eta, gauge, A.wx, A.wy, prune, t_first, nt, st));
    else if (tma) TM_TRY(tm_contract_xy_tma(ctx, qbuf, d_s, d_eta, gauge, A.wx, A.wy, prune, half0 ? 1 : 0, t_first, nt, st, merge & 1));
    else TM_TRY((launch_xy<float, 12>(ctx, A, prune, nt, st)));
    if (merge & 2) return TM_OK;                // the group's last source runs the z-sum and the assembly

    AssembleArgs B;
    B.qbuf = qbuf; B.out = d_out;
    TM_TRY(tm_ws(ctx, WS_CT_OUT, (size_t)ctx->X[3] * nq * 7 * CT_THREADS * sizeof(double), (void**)&B.zbuf));
    B.mom = (const int*)(tb + L.off_mom);
    B.qidx = (const short*)(tb + L.off_qidx);
    memcpy(B.qidx_v, host.data() + L.off_qidx, sizeof(B.qidx_v));
    memset(B.mom_v, 0, sizeof(B.mom_v));
    if (nmom <= AS_MOMV) memcpy(B.mom_v, h_momenta, (size_t)nmom * 12);
    B.wz = (const double*)(tb + L.off_wz);
    B.nmom = nmom; B.T = ctx->X[3]; B.Lz = ctx->X[2]; B.NQ = nq; B.t_first = t_first;
    B.twokmu = 2.0 * kappa * mu;
    B.half0 = half0 ? 1 : 0;
    B.L[0] = ctx->X[0]; B.L[1] = ctx->X[1]; B.L[2] = ctx->X[2];
    dim3 zgrid((unsigned)nq, (unsigned)nt);
    if (acc == TM_F64) contract_zsum_kernel<double><<<zgrid, CT_THREADS, (size_t)B.Lz * 64, st>>>(B);
    else contract_zsum_kernel<float><<<zgrid, CT_THREADS, (size_t)B.Lz * 64, st>>>(B);
    TM_LAUNCH_CHECK(ctx, "contract_zsum_kernel");
    dim3 grid((unsigned)nmom, (unsigned)nt);
    contract_assemble_kernel<<<grid, CT_THREADS, 0, st>>>(B);
    TM_LAUNCH_CHECK(ctx, "contract_assemble_kernel");
    return TM_OK;
}

// the path tm_contract_internal takes for a whole-vector call of precision acc is the TMA kernel (what merging needs)
bool tm_contract_merge_ok(const tm_ctx* ctx, tm_prec acc) {
    return acc == TM_F32 && ctx->opt_contract != 1 && ctx->opt_contract != 3 && tm_contract_tma_usable(ctx);
}

extern "C" tm_status loop_contract_project(tm_ctx* ctx, void* d_out, const void* d_s, const void* d_eta,
                                           double kappa, double mu, const int* h_momenta, int nmom,
                                           tm_prec acc, void* stream) {
    if (!ctx || !d_out || !d_s || !d_eta) return tm_fail(ctx, TM_EARG, "loop_contract_project: null argument");
    if (acc != TM_F64 && acc != TM_F32) return tm_fail(ctx, TM_EPREC, "loop_contract_project: acc must be f32 or f64");
    cudaStream_t st = (cudaStream_t)stream;
    TM_CUDA(ctx, cudaSetDevice(ctx->device));
    void *si, *ei;
    TM_TRY(tm_ws(ctx, WS_CT_S, 2 * tm_parity_bytes(ctx, acc), &si));
    TM_TRY(tm_ws(ctx, WS_CT_ETA, 2 * tm_parity_bytes(ctx, acc), &ei));
    TM_TRY(tm_import_launch(ctx, si, d_s, acc, st));
    TM_TRY(tm_import_launch(ctx, ei, d_eta, acc, st));
    return tm_contract_internal(ctx, d_out, si, ei, kappa, mu, h_momenta, nmom, acc, st);
}

extern "C" tm_status loop_contract_project_fields(tm_ctx* ctx, void* d_out, const void* d_s_int, const void* d_eta_int,
                                                  double kappa, double mu, const int* h_momenta, int nmom,
                                                  tm_prec acc, void* stream) {
    if (!ctx || !d_out || !d_s_int || !d_eta_int) return tm_fail(ctx, TM_EARG, "loop_contract_project_fields: null argument");
    if (acc != TM_F64 && acc != TM_F32) return tm_fail(ctx, TM_EPREC, "loop_contract_project_fields: acc must be f32 or f64");
    TM_CUDA(ctx, cudaSetDevice(ctx->device));
    return tm_contract_internal(ctx, d_out, d_s_int, d_eta_int, kappa, mu, h_momenta, nmom, acc, (cudaStream_t)stream);
}

extern "C" tm_status loop_contract_project_explicit(tm_ctx* ctx, void* d_out, const void* d_s, double kappa, double mu,
                                                    const int* h_momenta, int nmom, tm_prec acc, void* stream) {
    if (!ctx || !d_out || !d_s) return tm_fail(ctx, TM_EARG, "loop_contract_project_explicit: null argument");
    if (acc != TM_F64 && acc != TM_F32) return tm_fail(ctx, TM_EPREC, "loop_contract_project_explicit: acc must be f32 or f64");
    cudaStream_t st = (cudaStream_t)stream;
    TM_CUDA(ctx, cudaSetDevice(ctx->device));
    const size_t pb = tm_parity_bytes(ctx, acc);
    void *si, *ms;
    TM_TRY(tm_ws(ctx, WS_CT_S, 2 * pb, &si));
    TM_TRY(tm_ws(ctx, WS_CT_ETA, 2 * pb, &ms));
    TM_TRY(tm_import_launch(ctx, si, d_s, acc, st));
    // ms = M s: out_p = A s_p - kappa D_pq s_q for both parities
    const tm_recon rc = acc == TM_F64 ? TM_R18 : TM_R12;
    for (int p = 0; p < 2; p++) {
        DslashCall k;
        memset(&k, 0, sizeof(k));
        k.out = (char*)ms + p * pb; k.in = (const char*)si + (1 - p) * pb; k.x = (const char*)si + p * pb;
        k.out_parity = p; k.xmode = 2; k.coef = -kappa; k.kappa = kappa; k.mu = mu; k.red_op = RED_NONE;
        TM_TRY(tm_dslash_launch(ctx, k, acc, rc, st));
    }
    return tm_contract_internal(ctx, d_out, si, ms, kappa, mu, h_momenta, nmom, acc, st);
}

// ------------------------------------------------------------------ row f3 variant: symmetrised derivative
// l_sym[f][16+16m+n] = 1/2 [ s^dag g5 G_n (D_m psi) - (D_m s)^dag g5 G_n psi ],  psi = s | g.
// The second term is a relabeling of the same primitive: with (g5 G_n)^dag = eta_n g5 G_n and g5 G_n g5 = eps_n G_n,
//   (D s)^dag g5 G_n s = eta_n conj( s^dag g5 G_n D s )                                  -> A[0] of prim(s, eta)
//   (D s)^dag g5 G_n g = eta_n conj( eps_n (B[1] + 2 i kappa mu B[0]) + 2 i kappa mu A[0] ),  B = prim(eta, s)
// site by site, i.e. after projection the same expressions with p -> -p inside the conj (the momentum list must be
// closed under p -> -p).  Two contraction passes + this assembly; the ultra-local entries are A's.
__global__ void sym_assemble_kernel(double2* __restrict__ out, const double2* __restrict__ A, const double2* __restrict__ B,
                                    const int* __restrict__ negidx, unsigned eta_neg, unsigned eps_neg, double twokmu,
                                    int nmom, int T) {
    const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const size_t per_f = (size_t)80 * nmom * T;
    if (idx >= 2 * per_f) return;
    const int f = (int)(idx / per_f);
    size_t r = idx % per_f;
    const int i = (int)(r / ((size_t)nmom * T));
    r %= (size_t)nmom * T;
    const int k = (int)(r / T), t = (int)(r % T);
    if (i < 16) { out[idx] = A[idx]; return; }
    const int n = (i - 16) & 15;
    const double es = (eta_neg >> n) & 1u ? -1.0 : 1.0, ps = (eps_neg >> n) & 1u ? -1.0 : 1.0;
    const size_t at_neg = ((size_t)i * nmom + negidx[k]) * T + t;         // entry (f = 0, i, -p_k, t)
    const double2 a0n = A[at_neg];
    double2 y;                                                              // the bracket of the second term at -p
    if (f == 0) y = a0n;
    else {
        const double2 b0 = B[at_neg], b1 = B[per_f + at_neg];
        y.x = ps * (b1.x - twokmu * b0.y) - twokmu * a0n.y;
        y.y = ps * (b1.y + twokmu * b0.x) + twokmu * a0n.x;
    }
    const double2 a = A[idx];
    out[idx] = make_double2(0.5 * (a.x - es * y.x), 0.5 * (a.y + es * y.y));
}

extern "C" tm_status loop_contract_project_sym(tm_ctx* ctx, void* d_out, const void* d_s, const void* d_eta,
                                               double kappa, double mu, const int* h_momenta, int nmom,
                                               tm_prec acc, void* stream) {
    if (!ctx || !d_out || !d_s || !d_eta) return tm_fail(ctx, TM_EARG, "loop_contract_project_sym: null argument");
    if (acc != TM_F64 && acc != TM_F32) return tm_fail(ctx, TM_EPREC, "loop_contract_project_sym: acc must be f32 or f64");
    if (!h_momenta || nmom < 1) return tm_fail(ctx, TM_EARG, "loop_contract_project_sym: need at least one momentum");
    std::vector<int> neg(nmom, -1);
    for (int k = 0; k < nmom; k++)
        for (int j = 0; j < nmom; j++)
            if (h_momenta[3 * j] == -h_momenta[3 * k] && h_momenta[3 * j + 1] == -h_momenta[3 * k + 1]
                && h_momenta[3 * j + 2] == -h_momenta[3 * k + 2]) { neg[k] = j; break; }
    for (int k = 0; k < nmom; k++)
        if (neg[k] < 0) return tm_fail(ctx, TM_EARG, "loop_contract_project_sym: the momentum list must contain -p for every p");
    // signs of the Gamma algebra, multiplied out here (independent of the oracle)
    unsigned eta_neg = 0, eps_neg = 0;
    {
        const cd I(0, 1);
        cd sig[4][2][2] = {{{0, 1}, {1, 0}}, {{0, -I}, {I, 0}}, {{1, 0}, {0, -1}}, {{1, 0}, {0, 1}}};
        cd gam[4][4][4], g5[4][4];
        memset(gam, 0, sizeof(gam));
        for (int m = 0; m < 4; m++)
            for (int i = 0; i < 2; i++)
                for (int j = 0; j < 2; j++) {
                    const cd Bm = (m < 3) ? -I * sig[m][i][j] : sig[3][i][j];
                    gam[m][i][2 + j] = Bm;
                    gam[m][2 + j][i] = std::conj(Bm);
                }
        memset(g5, 0, sizeof(g5));
        for (int i = 0; i < 4; i++) g5[i][i] = 1;
        for (int m = 0; m < 4; m++) mat4mul(g5, g5, gam[m]);
        for (int n = 0; n < 16; n++) {
            cd G[4][4], M[4][4], W[4][4];
            memset(G, 0, sizeof(G));
            for (int i = 0; i < 4; i++) G[i][i] = 1;
            for (int m = 0; m < 4; m++)
                if ((n >> m) & 1) mat4mul(G, G, gam[m]);
            mat4mul(M, g5, G);                       // g5 Gamma_n
            mat4mul(W, M, g5);                       // g5 Gamma_n g5
            // M^dag = eta M and W = eps G: read the sign off a nonzero entry
            for (int a = 0; a < 4; a++)
                for (int b = 0; b < 4; b++) {
                    if (std::abs(M[a][b]) > 0.5 && std::abs(std::conj(M[b][a]) + M[a][b]) < 1e-12) eta_neg |= 1u << n;
                    if (std::abs(G[a][b]) > 0.5 && std::abs(W[a][b] + G[a][b]) < 1e-12) eps_neg |= 1u << n;
                }
        }
    }
    cudaStream_t st = (cudaStream_t)stream;
    TM_CUDA(ctx, cudaSetDevice(ctx->device));
    const size_t pb = tm_parity_bytes(ctx, acc);
    const size_t nout = (size_t)160 * nmom * ctx->X[3];
    void *si, *ei, *A, *B, *dneg;
    TM_TRY(tm_ws(ctx, WS_CT_S, 2 * pb, &si));
    TM_TRY(tm_ws(ctx, WS_CT_ETA, 2 * pb, &ei));
    TM_TRY(tm_ws(ctx, WS_API_A, nout * 16, &A));
    TM_TRY(tm_ws(ctx, WS_API_B, nout * 16, &B));
    TM_TRY(tm_ws(ctx, WS_API_C, (size_t)nmom * sizeof(int), &dneg));
    TM_CUDA(ctx, cudaMemcpyAsync(dneg, neg.data(), (size_t)nmom * sizeof(int), cudaMemcpyHostToDevice, st));
    TM_CUDA(ctx, cudaStreamSynchronize(st));         // neg is a local host vector
    TM_TRY(tm_import_launch(ctx, si, d_s, acc, st));
    TM_TRY(tm_import_launch(ctx, ei, d_eta, acc, st));
    TM_TRY(tm_contract_internal(ctx, A, si, ei, kappa, mu, h_momenta, nmom, acc, st));
    TM_TRY(tm_contract_internal(ctx, B, ei, si, kappa, mu, h_momenta, nmom, acc, st));
    sym_assemble_kernel<<<(unsigned)((nout + 255) / 256), 256, 0, st>>>((double2*)d_out, (const double2*)A, (const double2*)B,
                                                                       (const int*)dneg, eta_neg, eps_neg, 2.0 * kappa * mu,
                                                                       nmom, ctx->X[3]);
    TM_LAUNCH_CHECK(ctx, "sym_assemble_kernel");
    return TM_OK;
}

// A12 of SURVEY.md sec 2 ("GPU kernels to contract a single time slice or a whole vector"): the same 160
// projected insertions for ONE timeslice t0 (what a time-diluted source needs); 1/T of the work of the whole-vector
// call.  d_out keeps the [2][80][nmom][T] shape: column t0 is computed, every other column is zero.
extern "C" tm_status loop_contract_project_timeslice(tm_ctx* ctx, void* d_out, const void* d_s, const void* d_eta,
                                                     double kappa, double mu, const int* h_momenta, int nmom, int t0,
                                                     tm_prec acc, void* stream) {
    if (!ctx || !d_out || !d_s || !d_eta) return tm_fail(ctx, TM_EARG, "loop_contract_project_timeslice: null argument");
    if (acc != TM_F64 && acc != TM_F32) return tm_fail(ctx, TM_EPREC, "loop_contract_project_timeslice: acc must be f32 or f64");
    if (t0 < 0 || t0 >= ctx->X[3]) return tm_fail(ctx, TM_EARG, "loop_contract_project_timeslice: t0 outside the lattice");
    if (nmom < 1) return tm_fail(ctx, TM_EARG, "loop_contract_project_timeslice: need at least one momentum");
    cudaStream_t st = (cudaStream_t)stream;
    TM_CUDA(ctx, cudaSetDevice(ctx->device));
    void *si, *ei;
    TM_TRY(tm_ws(ctx, WS_CT_S, 2 * tm_parity_bytes(ctx, acc), &si));
    TM_TRY(tm_ws(ctx, WS_CT_ETA, 2 * tm_parity_bytes(ctx, acc), &ei));
    TM_TRY(tm_import_launch(ctx, si, d_s, acc, st));
    TM_TRY(tm_import_launch(ctx, ei, d_eta, acc, st));
    TM_CUDA(ctx, cudaMemsetAsync(d_out, 0, (size_t)160 * nmom * ctx->X[3] * 16, st));
    return tm_contract_internal(ctx, d_out, si, ei, kappa, mu, h_momenta, nmom, acc, st, t0, 1);
}

// =====================================================================================================
// loop_contract_project_fields_static: the contraction + projection for callers that cannot allocate
// (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).
//
// Same kernels as loop_contract_project_fields on its generic path (contract_xy_kernel, contract_zsum_kernel,
// contract_assemble_kernel); what differs is where their scratch lives: the x/y partial sums Q, the z-stage sums and the
// small tables (DFT weights, momentum list, accumulator index) sit in ONE file-scope device array of
// TM_STATIC_SCRATCH_BYTES instead of context workspaces, and the tables are written by a kernel from values passed as
// kernel arguments (no cudaMalloc, cudaFree, cudaMemcpy or other allocating call on this path).  Every GPU that loads
// the library holds the array until the process exits.  All calls, of all contexts, on one device share it: calls
// that overlap on the GPU (different streams) race.  It keeps the last call's contents; nothing in it has to start at
// zero (every element a call reads is written by that call first).
#define TM_STATIC_SCRATCH_BYTES ((size_t)16 << 20)
#define TM_STATIC_MAX_MOM 128
static __device__ __align__(256) unsigned char g_static_scratch[TM_STATIC_SCRATCH_BYTES];

struct StaticTablesArgs {
    int mom[3 * TM_STATIC_MAX_MOM];
    short qidx[64];
    int nmom, L[3];
    unsigned off_wx32, off_wy32, off_wx64, off_wy64, off_wz, off_mom, off_qidx;
};

// the tables of tm_contract_internal, built on the device: w[x][8] = 1, c1, s1, c2, s2, c3, s3, 0 with
// c_m + i s_m = exp(2 pi i m x / L) (exact argument reduction, as fill_weights does on the host)
__global__ void static_tables_kernel(unsigned char* tb, StaticTablesArgs A) {
    for (int i = threadIdx.x; i < (A.L[0] + A.L[1] + A.L[2]) * 8; i += blockDim.x) {
        int d = 0, j = i;
        if (j >= A.L[0] * 8) { j -= A.L[0] * 8; d = 1; }
        if (d == 1 && j >= A.L[1] * 8) { j -= A.L[1] * 8; d = 2; }
        const int x = j >> 3, k = j & 7, L = A.L[d];
        double w = k == 0 ? 1.0 : 0.0;
        if (k >= 1 && k <= 6) {
            const int m = (k + 1) >> 1;
            const double th = 2.0 * (double)((m * x) % L) / (double)L;
            w = (k & 1) ? cospi(th) : sinpi(th);
        }
        if (d == 0) { ((float*)(tb + A.off_wx32))[j] = (float)w; ((double*)(tb + A.off_wx64))[j] = w; }
        else if (d == 1) { ((float*)(tb + A.off_wy32))[j] = (float)w; ((double*)(tb + A.off_wy64))[j] = w; }
        else ((double*)(tb + A.off_wz))[j] = w;
    }
    for (int i = threadIdx.x; i < 3 * A.nmom; i += blockDim.x) ((int*)(tb + A.off_mom))[i] = A.mom[i];
    for (int i = threadIdx.x; i < 64; i += blockDim.x) ((short*)(tb + A.off_qidx))[i] = A.qidx[i];
}

// Device address of g_static_scratch, looked up once per device (in host code the array's name is only a host-side
// stand-in for the symbol, not a device address) together with the one-time upload of the Gamma table.
static unsigned char* g_static_ptr[64];
static tm_status static_setup(tm_ctx* ctx, unsigned char** out) {
    const int dev = ctx->device;
    if (dev < 0 || dev >= 64) return tm_fail(ctx, TM_EARG, "loop_contract_project_fields_static: device ordinal above 63");
    if (!g_static_ptr[dev]) {                                  // ctx->device is current (the caller set it)
        void* p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess || !p) return tm_cuda_fail(ctx, e, "cudaGetSymbolAddress(g_static_scratch)");
        GammaTable G;
        build_gamma_table(&G);
        TM_CUDA(ctx, cudaMemcpyToSymbol(c_gamma, &G, sizeof(G)));   // the same values the allocating path uploads
        g_static_ptr[dev] = (unsigned char*)p;
    }
    *out = g_static_ptr[dev];
    return TM_OK;
}

extern "C" size_t loop_contract_static_scratch_bytes(void) { return TM_STATIC_SCRATCH_BYTES; }

extern "C" tm_status loop_contract_project_fields_static(tm_ctx* ctx, void* d_out, const void* d_s_int,
                                                         const void* d_eta_int, double kappa, double mu,
                                                         const int* h_momenta, int nmom, tm_prec acc, void* stream) {
    if (!ctx || !d_out || !d_s_int || !d_eta_int || !h_momenta)
        return tm_fail(ctx, TM_EARG, "loop_contract_project_fields_static: null argument");
    if (acc != TM_F64 && acc != TM_F32) return tm_fail(ctx, TM_EPREC, "loop_contract_project_fields_static: acc must be f32 or f64");
    if (nmom < 1 || nmom > TM_STATIC_MAX_MOM)
        return tm_fail(ctx, TM_EARG, "loop_contract_project_fields_static: 1 <= nmom <= 128 (the momentum list travels as a kernel argument)");
    cudaStream_t st = (cudaStream_t)stream;
    TM_CUDA(ctx, cudaSetDevice(ctx->device));
    int prune = 1;
    for (int k = 0; k < nmom; k++) {
        const int px = h_momenta[3 * k], py = h_momenta[3 * k + 1], pz = h_momenta[3 * k + 2];
        if (abs(px) > 3 || abs(py) > 3 || abs(pz) > 3)
            return tm_fail(ctx, TM_EARG, "contract: momentum components must lie in [-3, 3]");
        if (px * px + py * py > 9) prune = 0;
    }
    // layout of the static array: tables | Q[T*Lz][NQ][320] (acc precision) | Z[T][NQ][7][320] (double)
    const ContractTables L = table_layout(ctx, nmom);
    const int nq = prune ? 29 : 49;
    const size_t fsz = acc == TM_F64 ? 8 : 4;
    const size_t qbytes = ((size_t)ctx->X[2] * ctx->X[3] * nq * CT_THREADS * fsz + 255) & ~(size_t)255;
    const size_t zbytes = (size_t)ctx->X[3] * nq * 7 * CT_THREADS * sizeof(double);
    const size_t need = L.total + qbytes + zbytes;
    if (need > TM_STATIC_SCRATCH_BYTES) {
        char msg[200];
        snprintf(msg, sizeof(msg), "loop_contract_project_fields_static: this lattice / momentum set needs %zu bytes of scratch, "
                 "the static array holds %zu (use loop_contract_project_fields)", need, (size_t)TM_STATIC_SCRATCH_BYTES);
        return tm_fail(ctx, TM_EDIM, msg);
    }
    // the packed gauge copy is context state, not scratch: it must exist already (packing allocates)
    const tm_recon rc = acc == TM_F64 ? TM_R18 : TM_R12;
    const int r = rc == TM_R12 ? 1 : 0;
    if (!ctx->gauge[acc][r] || !ctx->gauge_valid[acc][r])
        return tm_fail(ctx, TM_EARG, "loop_contract_project_fields_static: no packed gauge copy of this precision yet; one call of "
                                     "loop_contract_project_fields with the same acc after tm_load_gauge packs it");
    if (ctx->gauge_ev[acc][r] && ctx->gauge_st[acc][r] != st) TM_CUDA(ctx, cudaStreamWaitEvent(st, ctx->gauge_ev[acc][r], 0));
    unsigned char* tb = nullptr;
    TM_TRY(static_setup(ctx, &tb));

    StaticTablesArgs T;
    memset(&T, 0, sizeof(T));
    memcpy(T.mom, h_momenta, (size_t)nmom * 12);
    int nq_chk;
    tm_contract_qidx(T.qidx, prune, &nq_chk);
    T.nmom = nmom; T.L[0] = ctx->X[0]; T.L[1] = ctx->X[1]; T.L[2] = ctx->X[2];
    T.off_wx32 = (unsigned)L.off_wx32; T.off_wy32 = (unsigned)L.off_wy32; T.off_wx64 = (unsigned)L.off_wx64;
    T.off_wy64 = (unsigned)L.off_wy64; T.off_wz = (unsigned)L.off_wz; T.off_mom = (unsigned)L.off_mom; T.off_qidx = (unsigned)L.off_qidx;
    static_tables_kernel<<<1, 256, 0, st>>>(tb, T);
    TM_LAUNCH_CHECK(ctx, "static_tables_kernel");

    void* qbuf = tb + L.total;
    ContractArgs A;
    A.s = d_s_int; A.eta = d_eta_int; A.gauge = ctx->gauge[acc][r]; A.qbuf = qbuf;
    A.wx = tb + (acc == TM_F64 ? L.off_wx64 : L.off_wx32);
    A.wy = tb + (acc == TM_F64 ? L.off_wy64 : L.off_wy32);
    A.g = tm_geom(ctx);
    A.tb = (double)ctx->tb;
    A.t_first = 0;
    const int nt = ctx->X[3];
    if (acc == TM_F64) TM_TRY((launch_xy<double, 18>(ctx, A, prune, nt, st)));
    else TM_TRY((launch_xy<float, 12>(ctx, A, prune, nt, st)));

    AssembleArgs B;
    B.qbuf = qbuf; B.out = d_out;
    B.zbuf = (double*)(tb + L.total + qbytes);
    B.mom = (const int*)(tb + L.off_mom);
    B.qidx = (const short*)(tb + L.off_qidx);
    memcpy(B.qidx_v, T.qidx, sizeof(B.qidx_v));
    memset(B.mom_v, 0, sizeof(B.mom_v));
    memcpy(B.mom_v, h_momenta, (size_t)nmom * 12);
    B.wz = (const double*)(tb + L.off_wz);
    B.nmom = nmom; B.T = nt; B.Lz = ctx->X[2]; B.NQ = nq; B.t_first = 0;
    B.twokmu = 2.0 * kappa * mu;
    B.half0 = 0;
    B.L[0] = ctx->X[0]; B.L[1] = ctx->X[1]; B.L[2] = ctx->X[2];
    dim3 zgrid((unsigned)nq, (unsigned)nt);
    if (acc == TM_F64) contract_zsum_kernel<double><<<zgrid, CT_THREADS, (size_t)B.Lz * 64, st>>>(B);
    else contract_zsum_kernel<float><<<zgrid, CT_THREADS, (size_t)B.Lz * 64, st>>>(B);
    TM_LAUNCH_CHECK(ctx, "contract_zsum_kernel");
    dim3 grid((unsigned)nmom, (unsigned)nt);
    contract_assemble_kernel<<<grid, CT_THREADS, 0, st>>>(B);
    TM_LAUNCH_CHECK(ctx, "contract_assemble_kernel");
    return TM_OK;
}
