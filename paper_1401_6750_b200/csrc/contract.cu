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
// Kernel 1 thread roles (320 threads = 10 warps per CTA):
//   phase A: warp g = fam*5 + d, lane = x: computes the 32 reals of C_{fam,d}(x) -> shared memory
//   phase B: thread jr = one of the 320 real components: x-sum with 7 real weights, then the y-stage
//            update of its NQ register accumulators Q[(m,n),(cos|sin)x,(cos|sin)y].
#include <math.h>
#include <complex>
#include <vector>
#include "kernels.h"
#include "su3.cuh"

#define CT_THREADS 320

template <int PRUNE> struct QLayout { static constexpr int NQ = PRUNE ? 29 : 49; };

struct ContractArgs {
    const void* s;         // full-lattice internal field (even block, odd block)
    const void* eta;
    const void* gauge;
    void* qbuf;            // [T*Lz][NQ][320]
    const void* wx;        // [Lx][8]: 1, c1, s1, c2, s2, c3, s3, 0   (F precision)
    const void* wy;        // [Ly][8]
    Geom g;
    double tb;
};

template <typename F> struct BufStride;
template <> struct BufStride<float>  { static constexpr int V = 36; };
template <> struct BufStride<double> { static constexpr int V = 34; };

// full 4-spin SU(3) multiply
template <int DAG, typename F>
__device__ __forceinline__ void su3_mul_full(const F* U, const F* in, F* out) {
    su3_mul_half<DAG>(U, in, out);
    su3_mul_half<DAG>(U, in + 12, out + 12);
}

template <typename S, int R, int PRUNE, int NBUF>
__global__ void __launch_bounds__(CT_THREADS) contract_xy_kernel(ContractArgs A) {
    typedef S F;
    constexpr int BS = BufStride<F>::V;
    constexpr int NQ = QLayout<PRUNE>::NQ;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    F* buf = reinterpret_cast<F*>(smem_raw);                 // [NBUF][320][BS]
    F* swx = buf + (size_t)NBUF * CT_THREADS * BS;           // [Lx][8]
    F* swy = swx + (size_t)A.g.X0 * 8;                       // [Ly][8]
    const Geom& g = A.g;
    const int zt = blockIdx.x;
    const int z = zt % g.X2, t = zt / g.X2;
    const int lane = threadIdx.x & 31, grp = threadIdx.x >> 5;
    const int fam = grp / 5, d = grp % 5;
    const int jr = threadIdx.x;
    for (int i = threadIdx.x; i < g.X0 * 8; i += CT_THREADS) swx[i] = ((const F*)A.wx)[i];
    for (int i = threadIdx.x; i < g.X1 * 8; i += CT_THREADS) swy[i] = ((const F*)A.wy)[i];
    __syncthreads();

    const S* sfield = (const S*)A.s;
    const S* pfield = fam ? (const S*)A.eta : (const S*)A.s;
    const S* gauge = (const S*)A.gauge;
    const size_t Vh = g.Vh;
    const size_t pblk = Vh * 24;

    F Q[NQ];
#pragma unroll
    for (int q = 0; q < NQ; q++) Q[q] = 0;
    int b = 0;
    const int nxc = (g.X0 + 31) / 32;
    for (int y = 0; y < g.X1; y++) {
        F xc_[4], xs_[4];
#pragma unroll
        for (int m = 0; m < 4; m++) { xc_[m] = 0; xs_[m] = 0; }
        for (int xc = 0; xc < nxc; xc++) {
            const int x = xc * 32 + lane;
            F* mybuf = buf + (size_t)b * CT_THREADS * BS;
            // ---------------------------------------------------------------- phase A
            if (x < g.X0) {
                const int par = (x + y + z + t) & 1;
                const int row = ((t * g.X2 + z) * g.X1 + y) * g.X0;      // lex index of x = 0
                const size_t h = (size_t)(row + x) >> 1;
                F sv[24], psi[24];
                load_spinor<S>(sfield + par * pblk, Vh, h, sv);
                if (d == 0) {
                    if (fam) load_spinor<S>(pfield + par * pblk, Vh, h, psi);
                    else {
#pragma unroll
                        for (int i = 0; i < 24; i++) psi[i] = sv[i];
                    }
                } else {
                    const int mu = d - 1;
                    // neighbour lex indices and boundary signs
                    int lf, lb;
                    F sf = 1, sb = 1;
                    if (mu == 0) {
                        lf = row + (x + 1 == g.X0 ? 0 : x + 1);
                        lb = row + (x == 0 ? g.X0 - 1 : x - 1);
                    } else if (mu == 1) {
                        const int st = g.X0;
                        lf = (y + 1 == g.X1) ? row + x - (g.X1 - 1) * st : row + x + st;
                        lb = (y == 0) ? row + x + (g.X1 - 1) * st : row + x - st;
                    } else if (mu == 2) {
                        const int st = g.X0 * g.X1;
                        lf = (z + 1 == g.X2) ? row + x - (g.X2 - 1) * st : row + x + st;
                        lb = (z == 0) ? row + x + (g.X2 - 1) * st : row + x - st;
                    } else {
                        const int st = g.X0 * g.X1 * g.X2;
                        if (t + 1 == g.X3) { lf = row + x - (g.X3 - 1) * st; sf = (F)A.tb; } else lf = row + x + st;
                        if (t == 0) { lb = row + x + (g.X3 - 1) * st; sb = (F)A.tb; } else lb = row + x - st;
                    }
                    const size_t hf = (size_t)lf >> 1, hb = (size_t)lb >> 1;
                    F nb[24], U[18], tmp[24];
                    load_spinor<S>(pfield + (1 - par) * pblk, Vh, hf, nb);
                    load_link<S, R, LD_DEFAULT>(gauge, Vh, par, mu, h, U);
                    su3_mul_full<0>(U, nb, psi);
                    load_spinor<S>(pfield + (1 - par) * pblk, Vh, hb, nb);
                    load_link<S, R, LD_DEFAULT>(gauge, Vh, 1 - par, mu, hb, U);
                    su3_mul_full<1>(U, nb, tmp);
#pragma unroll
                    for (int i = 0; i < 24; i++) psi[i] = sf * psi[i] - sb * tmp[i];
                }
                // C[a][b] = sum_c conj(s_ac) psi_bc
                F* out = mybuf + (size_t)(grp * 32) * BS + lane;
#pragma unroll
                for (int a = 0; a < 4; a++)
#pragma unroll
                    for (int bb = 0; bb < 4; bb++) {
                        F re = 0, im = 0;
#pragma unroll
                        for (int c = 0; c < 3; c++) {
                            const F sr = sv[(a * 3 + c) * 2], si = sv[(a * 3 + c) * 2 + 1];
                            const F pr = psi[(bb * 3 + c) * 2], pi = psi[(bb * 3 + c) * 2 + 1];
                            re += sr * pr + si * pi;
                            im += sr * pi - si * pr;
                        }
                        out[(size_t)((a * 4 + bb) * 2) * BS] = re;
                        out[(size_t)((a * 4 + bb) * 2 + 1) * BS] = im;
                    }
            }
            __syncthreads();
            // ---------------------------------------------------------------- phase B: x-sum
            {
                const int nvalid = min(32, g.X0 - xc * 32);
                const F* v = mybuf + (size_t)jr * BS;
                const F* w = swx + (size_t)xc * 32 * 8;
                for (int l = 0; l < nvalid; l++) {
                    const F val = v[l];
                    const F* wl = w + l * 8;
                    xc_[0] += val;
                    xc_[1] += wl[1] * val; xs_[1] += wl[2] * val;
                    xc_[2] += wl[3] * val; xs_[2] += wl[4] * val;
                    xc_[3] += wl[5] * val; xs_[3] += wl[6] * val;
                }
            }
            if (NBUF == 2) b ^= 1; else __syncthreads();
        }
        // -------------------------------------------------------------------- y-stage
        {
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
                        Q[q++] += cy[n] * xc_[m];
                        if (n > 0) Q[q++] += sy[n] * xc_[m];
                        if (m > 0) Q[q++] += cy[n] * xs_[m];
                        if (m > 0 && n > 0) Q[q++] += sy[n] * xs_[m];
                    }
                }
        }
    }
    F* qb = (F*)A.qbuf + (size_t)zt * NQ * CT_THREADS + jr;
#pragma unroll
    for (int q = 0; q < NQ; q++) qb[(size_t)q * CT_THREADS] = Q[q];
}

// ------------------------------------------------------------------ kernel 2: z-sum + assembly
struct GammaTable {
    signed char perm[16][4];     // column of the nonzero of row a of g5 Gamma_n
    signed char phre[16][4];     // its value (one of +-1, +-i)
    signed char phim[16][4];
};
__constant__ GammaTable c_gamma;

struct AssembleArgs {
    const void* qbuf;
    void* out;                 // complex128 [2][80][nmom][T]
    const int* mom;            // [nmom][3]
    const short* qidx;         // [4][4][4]: index of Qcc, Qcs, Qsc, Qss for (m,n), -1 if absent
    const double* wz;          // [Lz][8]
    int nmom, T, Lz, NQ;
    double twokmu;             // 2 kappa mu
};

template <typename F>
__global__ void __launch_bounds__(CT_THREADS) contract_assemble_kernel(AssembleArgs A) {
    __shared__ double zre[CT_THREADS], zim[CT_THREADS];
    const int k = blockIdx.x, t = blockIdx.y;
    const int jr = threadIdx.x;
    const int px = A.mom[3 * k], py = A.mom[3 * k + 1], pz = A.mom[3 * k + 2];
    const int m = abs(px), n = abs(py), l = abs(pz);
    const double sx = px < 0 ? -1.0 : 1.0, sy = py < 0 ? -1.0 : 1.0, sz = pz < 0 ? -1.0 : 1.0;
    const short* qi = A.qidx + (m * 4 + n) * 4;
    const int icc = qi[0], ics = qi[1], isc = qi[2], iss = qi[3];
    const F* qb = (const F*)A.qbuf + (size_t)t * A.Lz * A.NQ * CT_THREADS + jr;
    double ar = 0, ai = 0;
    for (int z = 0; z < A.Lz; z++) {
        const F* q = qb + (size_t)z * A.NQ * CT_THREADS;
        const double cc = (double)q[(size_t)icc * CT_THREADS];
        const double cs = ics >= 0 ? (double)q[(size_t)ics * CT_THREADS] : 0.0;
        const double sc = isc >= 0 ? (double)q[(size_t)isc * CT_THREADS] : 0.0;
        const double ss = iss >= 0 ? (double)q[(size_t)iss * CT_THREADS] : 0.0;
        // (cos mx + i sx sin mx)(cos ny + i sy sin ny)
        const double wr = cc - sx * sy * ss, wi = sx * sc + sy * cs;
        const double cz = l ? A.wz[z * 8 + 2 * l - 1] : 1.0, szv = l ? sz * A.wz[z * 8 + 2 * l] : 0.0;
        ar += cz * wr - szv * wi;
        ai += cz * wi + szv * wr;
    }
    zre[jr] = ar; zim[jr] = ai;
    __syncthreads();
    if (jr < 160) {
        const int f = jr / 80, i = jr % 80;
        const int nG = i < 16 ? i : (i - 16) & 15;
        const int d = i < 16 ? 0 : 1 + ((i - 16) >> 4);
        const double scale = d ? 0.5 : 1.0;
        double l0r = 0, l0i = 0, l1r = 0, l1i = 0;
#pragma unroll
        for (int a = 0; a < 4; a++) {
            const int bcol = c_gamma.perm[nG][a];
            const double pr = c_gamma.phre[nG][a], pi = c_gamma.phim[nG][a];
            {   // s family: raw complex value = (Z[re comp]) + i (Z[im comp]) with each Z complex
                const int j = (d * 32) + (a * 4 + bcol) * 2;
                const double rr = zre[j] - zim[j + 1], ri = zim[j] + zre[j + 1];
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

static void build_qidx(short* qidx, int prune, int* nq) {
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

template <typename S, int R>
static tm_status launch_xy(tm_ctx* ctx, const ContractArgs& A, int prune, cudaStream_t st) {
    constexpr int BS = BufStride<S>::V;
    constexpr int NBUF = sizeof(S) == 4 ? 2 : 1;
    const size_t smem = (size_t)NBUF * CT_THREADS * BS * sizeof(S) + (size_t)(ctx->X[0] + ctx->X[1]) * 8 * sizeof(S);
    if (smem > 227 * 1024) return tm_fail(ctx, TM_EDIM, "contract: Lx + Ly too large for the shared-memory weight tables");
    const unsigned grid = (unsigned)(ctx->X[2] * ctx->X[3]);
    if (prune) {
        TM_CUDA(ctx, cudaFuncSetAttribute(contract_xy_kernel<S, R, 1, NBUF>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        contract_xy_kernel<S, R, 1, NBUF><<<grid, CT_THREADS, smem, st>>>(A);
    } else {
        TM_CUDA(ctx, cudaFuncSetAttribute(contract_xy_kernel<S, R, 0, NBUF>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        contract_xy_kernel<S, R, 0, NBUF><<<grid, CT_THREADS, smem, st>>>(A);
    }
    TM_LAUNCH_CHECK(ctx, "contract_xy_kernel");
    return TM_OK;
}

tm_status tm_contract_internal(tm_ctx* ctx, void* d_out, const void* d_s, const void* d_eta, double kappa,
                               double mu, const int* h_momenta, int nmom, tm_prec acc, cudaStream_t st) {
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
        build_qidx((short*)(host.data() + L.off_qidx), prune, &nq);
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
    if (acc == TM_F64) TM_TRY((launch_xy<double, 18>(ctx, A, prune, st)));
    else TM_TRY((launch_xy<float, 12>(ctx, A, prune, st)));

    AssembleArgs B;
    B.qbuf = qbuf; B.out = d_out;
    B.mom = (const int*)(tb + L.off_mom);
    B.qidx = (const short*)(tb + L.off_qidx);
    B.wz = (const double*)(tb + L.off_wz);
    B.nmom = nmom; B.T = ctx->X[3]; B.Lz = ctx->X[2]; B.NQ = nq;
    B.twokmu = 2.0 * kappa * mu;
    dim3 grid((unsigned)nmom, (unsigned)ctx->X[3]);
    if (acc == TM_F64) contract_assemble_kernel<double><<<grid, CT_THREADS, 0, st>>>(B);
    else contract_assemble_kernel<float><<<grid, CT_THREADS, 0, st>>>(B);
    TM_LAUNCH_CHECK(ctx, "contract_assemble_kernel");
    return TM_OK;
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
