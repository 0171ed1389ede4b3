// contract_tma.cu -- TMA-staged fast path of the fused contraction + projection kernel (fp32, Lx <= 32).
//
// Same mathematics and the same output (qbuf) as contract_xy_kernel in contract.cu (SURVEY.md sec 8
// rows a6-a8); what changes is how operands reach the SM and how much arithmetic is
// left per site.  One CTA per (z,t) plane, 14 warps:
//   warp 13      loader: one thread issues, per y-row, the TMA tensor copies (cp.async.bulk.tensor) that
//                land the rows of s and eta the row needs (centre, y+-1, z+-1, t+-1), the row's 4
//                forward links and the 3 backward links of the y-1, z-1, t-1 rows in shared memory,
//                completion signalled on an mbarrier (ring of 2 stages, or 3 with HALF0)
//   warps 0..7   producers, one fixed (fam, mu) derivative job each (+ a share of the d = 0 jobs): operands
//                come from shared memory at compile-time offsets (no global address arithmetic, no
//                long-scoreboard stalls), 16 complex outer-product values per site -> row buffer
//   warps 8..12  consumers: thread = complex component; x-sum with 7 real weights, y-stage accumulators
// Lane l of a producer handles the site of parity p = l / Xh with in-row half index idx = l % Xh
// (x = 2 idx + (p ^ row parity)), so that every shared-memory operand read is a contiguous run of
// 16-byte vectors.
//
// The kernel is bound by instruction issue (ncu: no pipe above 55 %, issue slots the scarce resource; an FFMA2
// costs one slot but two fp32-pipe cycles), so round 2 removed instructions (profiles/r02_contract_f32.md):
//   * LX > 0 (Lx = 16, 24, 32): folded x-stage -- the consumers combine the four sites {x, L-x, L/2-x, L/2+x}, on which
//     every cos / sin weight has the same absolute value, before weighting (15 packed operations per 4 sites instead
//     of 28); the weights are kernel parameters (constant bank -> uniform-register operands of FFMA2, no
//     shared-memory weight table); the producers store site x at the folded column fold_col(x);
//   * HALF0 (whole-vector launches): the s-family derivative slots receive only the forward half
//     F_mu = s^dag (x) U_mu(x) s(x + mu); the backward half is its shifted conjugate transpose and is restored by
//     contract_assemble_kernel from the same sums.  The s-family warps then do the d = 0 columns of both families, the
//     three backward rows of s are not staged (3 input stages fit), -14 % fp32 work;
//   * complex multiplies as one FFMA2 (real coefficient, broadcast scalar) + two scalar FFMA (imaginary coefficient):
//     no (-im, re) operand pair has to be built (P2::fma_si);
//   * d = 0 columns read straight from the stage instead of selected among registers at run time.
// TM_OPT_CONTRACT_PATH 4 launches the kernel without the first two (LX = 0, HALF0 = 0): the reference the tests
// compare with, and the only form a single-timeslice launch can take for HALF0 (it needs timeslice t - 1).
#include "contract.cuh"
#include "tma.cuh"

// NP producer warps (one (fam, mu) derivative job each), then CT_NC consumer warps and the loader warp
#define TX_NTHREADS(NP) (((NP) + CT_NC + 1) * 32)
#define TX_NCOMP(NP) (((NP) + CT_NC) * 32)    // threads taking part in the row-buffer barriers
#define TX_NSC 2                               // row-buffer stages
#ifndef TX_PF
#define TX_PF 1000                                // L2 prefetch distance in rows
#endif

struct TmaContractArgs {
    void* qbuf;            // [T*Lz][NQ][320] float
    const float* wx;       // [Lx][8]
    const float* wy;       // [Ly][8]
    Geom g;
    float tb;
    int t_first;           // first timeslice of the launch
    int q_add;             // add this source's partial sums to what qbuf holds (merged LP groups, tsm.cu) instead of overwriting
    float wf[7][6];        // folded x-stage (LX > 0): c1, s1, c2, s2, c3, s3 at x = j + 1, j < LX / 4 - 1 (kernel
                           // parameters live in the constant bank: FFMA2 takes them as uniform-register operands)
};

// shared-memory plan (bytes), every TMA destination 128-byte aligned
struct TxPlan {
    int nsi;               // input stages: 2, or 3 when the s family needs no backward rows (HALF0)
    int nrow_s;            // staged spinor rows of the s family: 7, or 4 with HALF0 (centre, y+1, z+1, t+1)
    int seg;               // bytes of one segment: Xh float4
    int row;               // one spinor row block: 12 segments, padded to 128
    int gf, gb;            // forward-link block (24 segments), one backward-link block (6 segments)
    int stage;             // one input stage: (nrow_s + 7) rows + gf + 3 gb
    int off_c, off_wx, off_wy, off_bar, total;
};
__host__ __device__ inline int tx_pad128(int b) { return (b + 127) & ~127; }
__host__ __device__ inline TxPlan tx_plan(int Lx, int Ly, int half0) {
    TxPlan P;
    P.nsi = half0 ? 3 : 2;
    P.nrow_s = half0 ? 4 : 7;
    P.seg = (Lx / 2) * 16;
    P.row = tx_pad128(12 * P.seg);
    P.gf = tx_pad128(24 * P.seg);
    P.gb = tx_pad128(6 * P.seg);
    P.stage = (P.nrow_s + 7) * P.row + P.gf + 3 * P.gb;
    P.off_c = P.nsi * P.stage;
    P.off_wx = P.off_c + TX_NSC * CT_NCC * CT_BSC * 8;
    P.off_wy = P.off_wx + 2 * 32 * 8 * 4;
    P.off_bar = tx_pad128(P.off_wy + Ly * 8 * 4);
    P.total = P.off_bar + 64;
    return P;
}

// ------------------------------------------------------------------ shared-memory operand reads
typedef P2<float>::T T2;

// 12 complex numbers of the site (parity q, in-row index idx) of a staged spinor row
__device__ __forceinline__ void lds_spinor(const float4* rowblk, int Xh, int q, int idx, T2* v) {
#pragma unroll
    for (int k = 0; k < 6; k++) {
        const float4 f = rowblk[(q * 6 + k) * Xh + idx];
        v[2 * k] = P2<float>::make(f.x, f.y);
        v[2 * k + 1] = P2<float>::make(f.z, f.w);
    }
}
// link stored as 3 segments starting at segment `seg0` of a link block; row 2 = conj(row0 x row1)
__device__ __forceinline__ void lds_link(const float4* blk, int Xh, int seg0, int idx, float* u) {
#pragma unroll
    for (int k = 0; k < 3; k++) {
        const float4 f = blk[(seg0 + k) * Xh + idx];
        u[4 * k] = f.x; u[4 * k + 1] = f.y; u[4 * k + 2] = f.z; u[4 * k + 3] = f.w;
    }
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const int i = (c + 1) % 3, j = (c + 2) % 3;
        const float ar = u[2 * i], ai = u[2 * i + 1], br = u[6 + 2 * j], bi = u[6 + 2 * j + 1];
        const float cr = u[2 * j], ci = u[2 * j + 1], dr = u[6 + 2 * i], di = u[6 + 2 * i + 1];
        float re = ar * br; re -= ai * bi; re -= cr * dr; re += ci * di;
        float im = ar * bi; im += ai * br; im -= cr * di; im -= ci * dr;
        u[12 + 2 * c] = re;
        u[12 + 2 * c + 1] = -im;
    }
}

// row blocks of one input stage, in the order the loader fills them
enum { ROW_C = 0, ROW_YP, ROW_YM, ROW_ZP, ROW_ZM, ROW_TP, ROW_TM };

// Folded x-stage (compile-time LX = Lx, a multiple of 4).  cos / sin(2 pi m x / L), m <= 3, take the same absolute
// values on the four sites {j, L - j, L/2 - j, L/2 + j}, so the consumers first form the four sign combinations of a
// group (8 adds) and then need 7 weighted accumulations per group instead of 28: 15 packed operations per 4 sites.  The
// producers store site x at row-buffer column fold_col(x): group j occupies columns 4j .. 4j + 3 (two 16-byte reads);
// group 0 holds the self-mirrored sites 0, L/2 and L/4, 3L/4, whose weights are 0 and +-1.
template <int LX> __device__ __forceinline__ int fold_col(int x) {
    if (x == 0) return 0;
    if (x == LX / 2) return 1;
    if (x == LX / 4) return 2;
    if (x == 3 * LX / 4) return 3;
    if (x < LX / 4) return 4 * x;
    if (x < LX / 2) return 4 * (LX / 2 - x) + 2;
    if (x < 3 * LX / 4) return 4 * (x - LX / 2) + 3;
    return 4 * (LX - x) + 1;
}
__device__ __forceinline__ T2 sub2(T2 a, T2 b) { T2 d; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }

struct TxShared {             // resolved shared-memory pointers of the CTA
    unsigned char* in;        // [P.nsi] input stages
    T2* cbuf;                 // [TX_NSC][160][CT_BSC]
    float* swx;               // [2 row parities][32 columns][8]
    float* swy;               // [Ly][8]
    unsigned bar_full, bar_empty;   // shared-space addresses of in_full[0], in_empty[0] (8 bytes apart per stage)
};

// producer warp: fixed derivative job (fam, mu) for every row of the plane, plus the rotating d = 0 jobs.
// One copy of the code for all directions (the direction only selects loop-invariant shared-memory
// offsets), so the 8 producer warps share the instruction cache.
template <int LX, int HALF0>
__device__ __forceinline__ void producer_rows(const TxShared& sh, const TxPlan& Prt, const Geom& g, int z, int t,
                                              int warp, int lane, float tb) {
    // with a compile-time row length every stage offset below is an immediate of its LDS (no address arithmetic)
    const int Xh = LX > 0 ? LX / 2 : g.Xh;
    const TxPlan P = LX > 0 ? tx_plan(LX, 2, HALF0) : Prt;        // the fields used here depend on Lx and HALF0 only
    const int fam = warp >> 2, mu = warp & 3;
    const int p = lane / Xh, idx = lane - p * Xh;
    const bool active = lane < g.X0;
    const float sgn_f = (mu == 3 && t + 1 == g.X3) ? tb : 1.f;
    const float sgn_b = (mu == 3 && t == 0) ? tb : 1.f;
    // byte offsets inside an input stage (float4 index = segment * Xh + idx)
    constexpr int NSI = HALF0 ? 3 : 2;
    // rows of a stage: the s family (7 rows in the order of the enum, or with HALF0 centre, y+1, z+1, t+1), then eta (7)
    const int fam_off = fam ? P.nrow_s * P.row : 0;
    const int rf = mu == 0 ? ROW_C : (HALF0 && fam == 0) ? mu : mu == 1 ? ROW_YP : mu == 2 ? ROW_ZP : ROW_TP;
    const int rb = mu == 0 ? ROW_C : mu == 1 ? ROW_YM : mu == 2 ? ROW_ZM : ROW_TM;
    const int idx_up = idx + 1 == Xh ? 0 : idx + 1, idx_dn = idx == 0 ? Xh - 1 : idx - 1;
    const int gbase = (P.nrow_s + 7) * P.row;
    const int off_sv = ((p * 6) * Xh + idx) * 16;                                   // centre s
    const int off_ev = P.nrow_s * P.row + off_sv;                                   // centre eta
    const int off_uf = gbase + (((p * 4 + mu) * 3) * Xh + idx) * 16;                // U_mu(x)
    // backward link U_mu(x - mu): mu = 0 from the row's own forward block, else from the staged neighbour row
    const int ub_blk = mu == 0 ? gbase + (((1 - p) * 4) * 3) * Xh * 16
                               : gbase + P.gf + (mu - 1) * P.gb + ((1 - p) * 3) * Xh * 16;
    const int nbf_blk = fam_off + rf * P.row + ((1 - p) * 6) * Xh * 16;
    const int nbb_blk = fam_off + rb * P.row + ((1 - p) * 6) * Xh * 16;
    const int seg = Xh * 16;
    // row-buffer column of this lane's site for x = 2 idx (+ 1): the site column itself, or its folded position
    const int col_e = LX > 0 ? fold_col<(LX > 0 ? LX : 4)>(2 * idx) : lane;
    const int col_o = LX > 0 ? fold_col<(LX > 0 ? LX : 4)>(2 * idx + 1) : lane;
    for (int y = 0; y < g.X1; y++) {
        const int si = y % NSI, sc = y % TX_NSC;
        const unsigned char* stage = sh.in + (size_t)si * P.stage;
        T2* rowbuf = sh.cbuf + (size_t)sc * CT_NCC * CT_BSC;
        mbar_wait(sh.bar_full + 8 * si, (y / NSI) & 1);
        if (y >= TX_NSC) named_bar_sync(1 + TX_NSC + sc, TX_NCOMP(8));
        if (active) {
            const int xo = (p ^ (y + z + t)) & 1;                 // x = 2 idx + xo
            const int col = xo ? col_o : col_e;
            const int idx_f = mu == 0 ? (xo ? idx_up : idx) : idx;
            const int idx_b = mu == 0 ? (xo ? idx : idx_dn) : idx;
            T2 sv[12];
#pragma unroll
            for (int k = 0; k < 6; k++) {
                const float4 f = *reinterpret_cast<const float4*>(stage + off_sv + k * seg);
                sv[2 * k] = P2<float>::make(f.x, f.y);
                sv[2 * k + 1] = P2<float>::make(f.z, f.w);
            }
            {
                // psi = U_mu(x) f(x+mu) - U_mu^dag(x-mu) f(x-mu)
                T2 psi[12], nb[12];
                float U[18];
#pragma unroll
                for (int i = 0; i < 12; i++) psi[i] = P2<float>::make(0.f, 0.f);
                const unsigned char* nf = stage + nbf_blk + idx_f * 16;
#pragma unroll
                for (int k = 0; k < 6; k++) {
                    const float4 f = *reinterpret_cast<const float4*>(nf + k * seg);
                    nb[2 * k] = P2<float>::make(f.x, f.y);
                    nb[2 * k + 1] = P2<float>::make(f.z, f.w);
                }
                if (sgn_f != 1.f) {
#pragma unroll
                    for (int i = 0; i < 12; i++) nb[i] = P2<float>::mul_s(sgn_f, nb[i]);
                }
                lds_link(reinterpret_cast<const float4*>(stage + off_uf), Xh, 0, 0, U);
                su3_macc<0, 0, float>(U, nb, psi);
                // HALF0: the s family keeps only the forward half F_mu; contract_assemble_kernel restores the backward
                // half from the same sums (it is the shifted conjugate transpose of the forward half)
                if (!(HALF0 && fam == 0)) {
                    const unsigned char* nbk = stage + nbb_blk + idx_b * 16;
#pragma unroll
                    for (int k = 0; k < 6; k++) {
                        const float4 f = *reinterpret_cast<const float4*>(nbk + k * seg);
                        nb[2 * k] = P2<float>::make(f.x, f.y);
                        nb[2 * k + 1] = P2<float>::make(f.z, f.w);
                    }
                    if (sgn_b != 1.f) {
#pragma unroll
                        for (int i = 0; i < 12; i++) nb[i] = P2<float>::mul_s(sgn_b, nb[i]);
                    }
                    lds_link(reinterpret_cast<const float4*>(stage + ub_blk + idx_b * 16), Xh, 0, 0, U);
                    su3_macc<1, 1, float>(U, nb, psi);
                }
                outer_store<float>(sv, psi, rowbuf, fam * 5 + 1 + mu, col);
            }
            // this warp's share of the two d = 0 jobs: column bb = mu of C_{fd,0}[a][bb] = sum_c conj(s_ac) f_{bb,c}
            // (splitting the two light jobs keeps the producer warps in step: every warp one column of its own family,
            // or with HALF0 the four s-family warps, which skip the backward half, one column of each family)
            if (!HALF0 || fam == 0) {
#pragma unroll
                for (int ff = 0; ff < (HALF0 ? 2 : 1); ff++) {
                    const int fd = HALF0 ? ff : fam;
                    const int bb = mu;
                    // spin component bb of the centre row of family fd, straight from the stage (complex number j sits
                    // in half j & 1 of segment j >> 1): no run-time selection among the registers of sv
                    const unsigned char* cb = stage + (fd ? off_ev : off_sv);
                    T2 f3[3];
#pragma unroll
                    for (int c = 0; c < 3; c++) {
                        const int j = 3 * bb + c;
                        f3[c] = *reinterpret_cast<const T2*>(cb + (j >> 1) * seg + (j & 1) * 8);
                    }
                    T2 acc[4];
#pragma unroll
                    for (int a = 0; a < 4; a++) acc[a] = P2<float>::make(0.f, 0.f);
#pragma unroll
                    for (int c = 0; c < 3; c++) {
                        float sre[4], sim[4];
#pragma unroll
                        for (int a = 0; a < 4; a++) { P2<float>::get(sv[a * 3 + c], sre[a], sim[a]); }
#pragma unroll
                        for (int a = 0; a < 4; a++) acc[a] = P2<float>::fma_s(sre[a], f3[c], acc[a]);
#pragma unroll
                        for (int a = 0; a < 4; a++) acc[a] = P2<float>::fma_si(-sim[a], f3[c], acc[a]);
                    }
                    T2* out = rowbuf + (size_t)(fd * 5 * 16 + bb) * CT_BSC + col;
#pragma unroll
                    for (int a = 0; a < 4; a++) out[(size_t)(a * 4) * CT_BSC] = acc[a];
                }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(sh.bar_empty + 8 * si);        // this warp is done reading the input stage
        named_bar_arrive(1 + sc, TX_NCOMP(8));
    }
}

template <int PRUNE, int LX, int HALF0, int NP>
__global__ void __launch_bounds__(TX_NTHREADS(NP), 1)
contract_xy_tma_kernel(const __grid_constant__ CUtensorMap tm_s, const __grid_constant__ CUtensorMap tm_e,
                       const __grid_constant__ CUtensorMap tm_gf, const __grid_constant__ CUtensorMap tm_gb,
                       TmaContractArgs A) {
    constexpr int NQ = QLayout<PRUNE>::NQ;
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    const Geom& g = A.g;
    constexpr int NSI = HALF0 ? 3 : 2;
    const TxPlan P = tx_plan(g.X0, g.X1, HALF0);
    TxShared sh;
    sh.in = smem_raw;
    sh.cbuf = reinterpret_cast<T2*>(smem_raw + P.off_c);
    sh.swx = reinterpret_cast<float*>(smem_raw + P.off_wx);
    sh.swy = reinterpret_cast<float*>(smem_raw + P.off_wy);
    sh.bar_full = smem_u32(smem_raw + P.off_bar);
    sh.bar_empty = sh.bar_full + 8 * NSI;
    const int zt = blockIdx.x + A.t_first * g.X2;
    const int z = zt % g.X2, t = zt / g.X2;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int Xh = g.Xh;

    // x-weight tables in column order: column l <-> x = 2 (l % Xh) + ((l / Xh) ^ row parity)
    for (int i = threadIdx.x; i < 2 * 32 * 8; i += TX_NTHREADS(NP)) {
        const int rp = i >> 8, l = (i >> 3) & 31, k = i & 7;
        float w = 0.f;
        if (l < g.X0) {
            const int x = 2 * (l % Xh) + ((l / Xh) ^ rp);
            w = A.wx[x * 8 + k];
        }
        sh.swx[i] = w;
    }
    for (int i = threadIdx.x; i < g.X1 * 8; i += TX_NTHREADS(NP)) sh.swy[i] = A.wy[i];
    if (threadIdx.x == 0) {
        for (int s = 0; s < NSI; s++) {
            mbar_init(sh.bar_full + 8 * s, 1);
            mbar_init(sh.bar_empty + 8 * s, NP);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == NP + CT_NC) {
        // ================================================================ loader
        if (lane == 0) {
            asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_s) : "memory");
            asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_e) : "memory");
            asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_gf) : "memory");
            asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_gb) : "memory");
            const unsigned in0 = smem_u32(sh.in);
            const int zp = z + 1 == g.X2 ? 0 : z + 1, zm = z == 0 ? g.X2 - 1 : z - 1;
            const int tp = t + 1 == g.X3 ? 0 : t + 1, tm = t == 0 ? g.X3 - 1 : t - 1;
            const unsigned bytes = (unsigned)((P.nrow_s + 7) * 12 + 24 + 18) * (unsigned)P.seg;
            for (int y = 0; y < g.X1; y++) {
                const int si = y % NSI;
                const unsigned full = sh.bar_full + 8 * si;
                if (y >= NSI) mbar_wait_relaxed(sh.bar_empty + 8 * si, ((y / NSI) - 1) & 1);
                mbar_expect_tx(full, bytes);
                const int yp = y + 1 == g.X1 ? 0 : y + 1, ym = y == 0 ? g.X1 - 1 : y - 1;
                // float coordinate of the first site of row (yy, zz, tt) inside a parity block: 4 * (lex / 2)
                auto c0 = [&](int yy, int zz, int tt) { return 2 * (((tt * g.X2 + zz) * g.X1 + yy) * g.X0); };
                const int rc[7] = {c0(y, z, t), c0(yp, z, t), c0(ym, z, t), c0(y, zp, t), c0(y, zm, t), c0(y, z, tp), c0(y, z, tm)};
                const unsigned st0 = in0 + (unsigned)si * (unsigned)P.stage;
                if (HALF0) {        // s family: centre and forward rows only
#pragma unroll
                    for (int r = 0; r < 4; r++) tma_load_2d(st0 + (unsigned)(r * P.row), &tm_s, full, rc[r == 0 ? 0 : 2 * r - 1], 0);
                } else {
#pragma unroll
                    for (int r = 0; r < 7; r++) tma_load_2d(st0 + (unsigned)(r * P.row), &tm_s, full, rc[r], 0);
                }
#pragma unroll
                for (int r = 0; r < 7; r++) tma_load_2d(st0 + (unsigned)((P.nrow_s + r) * P.row), &tm_e, full, rc[r], 0);
                const unsigned gbase = st0 + (unsigned)((P.nrow_s + 7) * P.row);
                tma_load_4d(gbase, &tm_gf, full, rc[0], 0, 0, 0);
                tma_load_4d(gbase + (unsigned)P.gf, &tm_gb, full, rc[2], 0, 1, 0);
                tma_load_4d(gbase + (unsigned)(P.gf + P.gb), &tm_gb, full, rc[4], 0, 2, 0);
                tma_load_4d(gbase + (unsigned)(P.gf + 2 * P.gb), &tm_gb, full, rc[6], 0, 3, 0);
                // pull the rows a few iterations ahead into L2 (costs no shared memory): the y+1 row of
                // iteration y + TX_PF is the only one of its y-window not requested before
                const int ya = y + TX_PF;
                if (ya < g.X1) {
                    const int yb = ya + 1 == g.X1 ? 0 : ya + 1;
                    const int pc[5] = {c0(yb, z, t), c0(ya, zp, t), c0(ya, zm, t), c0(ya, z, tp), c0(ya, z, tm)};
#pragma unroll
                    for (int r = 0; r < 5; r++) { tma_prefetch_2d(&tm_s, pc[r], 0); tma_prefetch_2d(&tm_e, pc[r], 0); }
                    tma_prefetch_4d(&tm_gf, pc[0], 0, 0, 0);
                    tma_prefetch_4d(&tm_gb, pc[2], 0, 2, 0);
                    tma_prefetch_4d(&tm_gb, pc[4], 0, 3, 0);
                }
            }
        }
    } else if (warp < NP) {
        // ================================================================ producers
        producer_rows<LX, HALF0>(sh, P, g, z, t, warp, lane, A.tb);
    } else {
        // ================================================================ consumers
        typedef P2<float> PP;
        const int cc = threadIdx.x - NP * 32;           // 0..159
        T2 Q[NQ];
#pragma unroll
        for (int q = 0; q < NQ; q++) Q[q] = PP::make(0.f, 0.f);
        for (int y = 0; y < g.X1; y++) {
            const int sc = y % TX_NSC;
            const T2* v = sh.cbuf + ((size_t)sc * CT_NCC + cc) * CT_BSC;
            const float* w = sh.swx + ((y + z + t) & 1) * 256;
            T2 a0 = PP::make(0.f, 0.f), ac[3], as[3];
#pragma unroll
            for (int m = 0; m < 3; m++) { ac[m] = PP::make(0.f, 0.f); as[m] = PP::make(0.f, 0.f); }
            named_bar_sync(1 + sc, TX_NCOMP(NP));
            if (LX > 0) {
                // folded x-stage: see fold_col
                const ulonglong2* v4 = reinterpret_cast<const ulonglong2*>(v);
                {
                    const ulonglong2 q0 = v4[0], q1 = v4[1];       // C(0), C(L/2); C(L/4), C(3L/4)
                    const T2 Pp = PP::add(q0.x, q0.y), Mm = sub2(q0.x, q0.y);
                    const T2 Ee = PP::add(q1.x, q1.y), Oo = sub2(q1.x, q1.y);
                    a0 = PP::add(Pp, Ee);
                    ac[1] = sub2(Pp, Ee);
                    ac[0] = Mm; ac[2] = Mm;
                    as[0] = Oo; as[2] = sub2(as[2], Oo);
                }
#pragma unroll
                for (int j = 1; j < (LX > 0 ? LX / 4 : 1); j++) {
                    const ulonglong2 q0 = v4[2 * j], q1 = v4[2 * j + 1];   // C(j), C(L-j); C(L/2-j), C(L/2+j)
                    const T2 E1 = PP::add(q0.x, q0.y), O1 = sub2(q0.x, q0.y);
                    const T2 E2 = PP::add(q1.x, q1.y), O2 = sub2(q1.y, q1.x);
                    const T2 Pp = PP::add(E1, E2), Mm = sub2(E1, E2), Rr = PP::add(O1, O2), Ss = sub2(O1, O2);
                    const float* wj = A.wf[j - 1];
                    a0 = PP::add(a0, Pp);
                    ac[0] = PP::fma_s(wj[0], Mm, ac[0]);
                    as[0] = PP::fma_s(wj[1], Ss, as[0]);
                    ac[1] = PP::fma_s(wj[2], Pp, ac[1]);
                    as[1] = PP::fma_s(wj[3], Rr, as[1]);
                    ac[2] = PP::fma_s(wj[4], Mm, ac[2]);
                    as[2] = PP::fma_s(wj[5], Ss, as[2]);
                }
            } else {
#pragma unroll 4
                for (int l = 0; l < g.X0; l++) {
                    const T2 val = v[l];
                    const float* wl = w + l * 8;
                    a0 = PP::add(a0, val);
#pragma unroll
                    for (int m = 0; m < 3; m++) {
                        ac[m] = PP::fma_s(wl[2 * m + 1], val, ac[m]);
                        as[m] = PP::fma_s(wl[2 * m + 2], val, as[m]);
                    }
                }
            }
            if (y + TX_NSC < g.X1) named_bar_arrive(1 + TX_NSC + sc, TX_NCOMP(NP));
            const float* wl = sh.swy + y * 8;
            float cy[4], sy[4];
            cy[0] = 1.f; sy[0] = 0.f;
            cy[1] = wl[1]; sy[1] = wl[2]; cy[2] = wl[3]; sy[2] = wl[4]; cy[3] = wl[5]; sy[3] = wl[6];
            int q = 0;
#pragma unroll
            for (int m = 0; m < 4; m++)
#pragma unroll
                for (int n = 0; n < 4; n++) {
                    if (!PRUNE || m * m + n * n <= 9) {
                        const T2 xcm = m ? ac[m - 1] : a0;
                        if (n == 0) Q[q] = PP::add(Q[q], xcm); else Q[q] = PP::fma_s(cy[n], xcm, Q[q]);
                        q++;
                        if (n > 0) { Q[q] = PP::fma_s(sy[n], xcm, Q[q]); q++; }
                        if (m > 0) {
                            if (n == 0) Q[q] = PP::add(Q[q], as[m - 1]); else Q[q] = PP::fma_s(cy[n], as[m - 1], Q[q]);
                            q++;
                        }
                        if (m > 0 && n > 0) { Q[q] = PP::fma_s(sy[n], as[m - 1], Q[q]); q++; }
                    }
                }
        }
        T2* qb = reinterpret_cast<T2*>((float*)A.qbuf + (size_t)zt * NQ * CT_THREADS) + cc;
        if (A.q_add) {
#pragma unroll
            for (int q = 0; q < NQ; q++) Q[q] = PP::add(Q[q], qb[(size_t)q * CT_NCC]);
        }
#pragma unroll
        for (int q = 0; q < NQ; q++) qb[(size_t)q * CT_NCC] = Q[q];
    }
}

// ------------------------------------------------------------------ host side
bool tm_contract_tma_usable(const tm_ctx* ctx) {
    if (ctx->X[0] > 32) return false;
    if (4 * ctx->Vh >= (size_t)1 << 31) return false;             // TMA coordinates are int32
    const TxPlan P = tx_plan(ctx->X[0], ctx->X[1], 0);       // the larger of the two plans
    if (P.total > 227 * 1024 || tx_plan(ctx->X[0], ctx->X[1], 1).total > 227 * 1024) return false;
    return get_encode_fn() != nullptr;
}

// s, eta: fp32 full-lattice internal fields; gauge: fp32 reconstruct-12 internal copy; wx, wy: float tables
tm_status tm_contract_xy_tma(tm_ctx* ctx, void* qbuf, const void* d_s, const void* d_eta, const void* gauge,
                             const void* wx, const void* wy, int prune, int half0, int t_first, int nt, cudaStream_t st,
                             int q_add) {
    const int Xh = ctx->Xh;
    const cuuint64_t Vh = ctx->Vh;
    CUtensorMap ms, me, mgf, mgb;
    {
        const cuuint64_t dims[2] = {4 * Vh, 12};
        const cuuint64_t strides[1] = {Vh * 16};
        const cuuint32_t box[2] = {(cuuint32_t)(4 * Xh), 12};
        if (!encode_map(&ms, d_s, 2, dims, strides, box) || !encode_map(&me, d_eta, 2, dims, strides, box))
            return tm_fail(ctx, TM_ECUDA, "contract: cuTensorMapEncodeTiled failed (spinor)");
    }
    {
        const cuuint64_t dims[4] = {4 * Vh, 3, 4, 2};
        const cuuint64_t strides[3] = {Vh * 16, 3 * Vh * 16, 12 * Vh * 16};
        const cuuint32_t boxf[4] = {(cuuint32_t)(4 * Xh), 3, 4, 2};
        const cuuint32_t boxb[4] = {(cuuint32_t)(4 * Xh), 3, 1, 2};
        if (!encode_map(&mgf, gauge, 4, dims, strides, boxf) || !encode_map(&mgb, gauge, 4, dims, strides, boxb))
            return tm_fail(ctx, TM_ECUDA, "contract: cuTensorMapEncodeTiled failed (gauge)");
    }
    TmaContractArgs A;
    A.qbuf = qbuf; A.wx = (const float*)wx; A.wy = (const float*)wy;
    A.g = tm_geom(ctx);
    A.tb = (float)ctx->tb;
    A.t_first = t_first;
    A.q_add = q_add;
    const TxPlan P = tx_plan(ctx->X[0], ctx->X[1], half0);
    const unsigned grid = (unsigned)(ctx->X[2] * nt);
    // folded x-stage for the extents the configurations use (any multiple of 4 would do); other extents take the
    // plain weighted sum over the row
    const int L = ctx->X[0];
    const int lx = (ctx->opt_contract != 4 && (L == 32 || L == 24 || L == 16)) ? L : 0;
    memset(A.wf, 0, sizeof(A.wf));
    for (int j = 1; lx && j < lx / 4; j++)
        for (int m = 1; m < 4; m++) {
            const double th = 2.0 * M_PI * (double)((m * j) % lx) / (double)lx;      // exact argument reduction
            A.wf[j - 1][2 * m - 2] = (float)cos(th);
            A.wf[j - 1][2 * m - 1] = (float)sin(th);
        }
#define TX_LAUNCH1(PR, LXV, H0, NPV)                                                                                    \
    do {                                                                                                                \
        TM_CUDA(ctx, cudaFuncSetAttribute(contract_xy_tma_kernel<PR, LXV, H0, NPV>,                                     \
                                          cudaFuncAttributeMaxDynamicSharedMemorySize, P.total));                       \
        contract_xy_tma_kernel<PR, LXV, H0, NPV><<<grid, TX_NTHREADS(NPV), P.total, st>>>(ms, me, mgf, mgb, A);         \
    } while (0)
#define TX_LAUNCH(PR, LXV)                                                                                              \
    do {                                                                                                                \
        if (half0) TX_LAUNCH1(PR, LXV, 1, 8);                                                                           \
        else TX_LAUNCH1(PR, LXV, 0, 8);                                                                                 \
    } while (0)
    if (prune) {
        if (lx == 32) TX_LAUNCH(1, 32); else if (lx == 24) TX_LAUNCH(1, 24); else if (lx == 16) TX_LAUNCH(1, 16); else TX_LAUNCH(1, 0);
    } else {
        if (lx == 32) TX_LAUNCH(0, 32); else if (lx == 24) TX_LAUNCH(0, 24); else if (lx == 16) TX_LAUNCH(0, 16); else TX_LAUNCH(0, 0);
    }
#undef TX_LAUNCH
#undef TX_LAUNCH1
    TM_LAUNCH_CHECK(ctx, "contract_xy_tma_kernel");
    return TM_OK;
}
