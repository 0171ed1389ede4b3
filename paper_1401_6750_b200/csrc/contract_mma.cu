// contract_mma.cu -- fused contraction + projection, site stage and x/y-DFT, third implementation (fp32, Lx <= 32,
// whole-vector launches; TM_OPT_CONTRACT_PATH 3; measured slower than contract_tma.cu, so never the automatic choice).
//
// Same mathematics as contract_xy_kernel in contract.cu and the same
// TMA operand staging as contract_tma.cu.  contract_tma.cu is bound by how well two lock-stepped producer warps per
// SM sub-partition keep the fp32 pipe busy (ncu: pipe 50 % active, issue slots 50 %, 3800 cycles per lattice row for
// 1700 cycles of pipe work), whatever the consumers do.  Three changes:
//
// (1) No producer / consumer split and no CTA-wide barrier.  16 symmetric warps (4 per sub-partition); warp
//     (fam, mu, h) owns the 8 complex components C_{fam,1+mu}[a][b], b in {2h, 2h+1}, of every row of the plane:
//     it forms them (lane = site), transposes them through a private 2 KB shared-memory tile (__syncwarp only), and
//     reduces them over x itself.  Warps meet only at the mbarriers of the input stages (3-stage ring).
// (2) The x-sum  X[comp][k] = sum_l C[comp][l] W[l][k]  (16 real rows x 32 sites x 8 weights per tile) runs on the
//     tensor pipe, which is otherwise idle: mma.sync.m16n8k8 tf32 with split-fp32 operands, C = C_hi + C_lo,
//     W = W_hi + W_lo, three MMAs (hi*hi + lo*hi + hi*lo); dropped terms are O(2^-21) relative, the 1e-5 bound of the
//     fp32 contraction holds (measured 2-4e-7).  The split needs the operand in registers anyway, which is why this is
//     the register-operand mma.sync and not tcgen05.mma (a shared-memory A operand would need a second, lo, tile
//     written by the producers).  D fragments feed the y-stage accumulators directly: thread (g, t) of a tile owns
//     component g and the x-weights of D columns 2t, 2t+1; columns are ordered so that no thread needs more than
//     10 (unpruned: 14) complex accumulators per tile.
// (3) Half the SU(3) work of the s family.  With a_mu(y) = U_mu(y) s(y+mu) the backward half of the derivative is the
//     shifted conjugate transpose of the forward half,
//         s^dag(x) (x) U_mu^dag(x-mu) s(x-mu) [a][b]  =  conj( F_mu[b][a](x-mu) ),   F_mu(y) = s^dag(y) (x) a_mu(y),
//     so the s-family warps form only F_mu (one SU(3) product on two spins, forward rows and links only) and the
//     assembly kernel restores  F~[a][b](p,t) - e^{i p_mu} conj(F~[b][a](-p, t'))  (t' = t-1 for mu = t) from the same
//     (cos|sin)^3 sums (AssembleArgs::half0).  The 8 s-family warps use the time saved for the two ultra-local
//     families (a quarter-tile each).
#include <vector>
#include <utility>
#include "contract.cuh"
#include "tma.cuh"

#define MX_NW 16
#define MX_NTHREADS (MX_NW * 32)
#define MX_NSI 3                               // input stages
#define MX_BS 32                               // tile stride in complex numbers (32 sites)
#define MX_TILE_BYTES (8 * MX_BS * 8)          // 8 complex components x 32 sites
#define MX_NTILES_SMEM (MX_NW + MX_NW / 2)     // one per warp + the ultra-local quarter-tiles of the s-family warps

struct MmaSlots {              // y-stage accumulators of thread t (= lane & 3) of a tile: slot j < NA takes D column 2t,
    signed char q[4][16];      //   slot NA + j column 2t + 1; q = index into the Q layout of contract.cu (-1: unused),
    signed char sel[4][16];    //   sel = entry of the y-weight row (1, c1, s1, c2, s2, c3, s3, 0) it is multiplied with
};

struct MmaContractArgs {
    void* qbuf;            // [T*Lz][NQ][320] float
    const float* wx;       // [Lx][8]
    const float* wy;       // [Ly][8]
    Geom g;
    float tb;
    int t_first;           // first timeslice of the launch
    MmaSlots slots;
};

// x-weight (entry of the weight row) of D column n; column 1 repeats the constant weight so that the 7 accumulators
// of the m = 0 sums split 4 + 3 over the two columns of thread 0
__device__ __constant__ signed char c_mx_wsel[8] = {0, 0, 1, 5, 2, 6, 3, 4};

// row blocks of one input stage, in the order the loader fills them: s needs only the forward neighbours
enum { SR_C = 0, SR_YP, SR_ZP, SR_TP, ER_C, ER_YP, ER_YM, ER_ZP, ER_ZM, ER_TP, ER_TM, MX_NROWS };

// shared-memory plan (bytes), every TMA destination 128-byte aligned
struct MxPlan {
    int seg;               // bytes of one segment: Xh float4
    int row;               // one spinor row block: 12 segments, padded to 128
    int gf, gb;            // forward-link block (24 segments), one backward-link block (6 segments)
    int stage;             // one input stage: 11 rows + gf + 3 gb
    int off_tile, off_bt, off_cf, off_bar, total;
};
__host__ __device__ inline int mx_pad128(int b) { return (b + 127) & ~127; }
__host__ __device__ inline MxPlan mx_plan(int Lx, int Ly) {
    MxPlan P;
    P.seg = (Lx / 2) * 16;
    P.row = mx_pad128(12 * P.seg);
    P.gf = mx_pad128(24 * P.seg);
    P.gb = mx_pad128(6 * P.seg);
    P.stage = MX_NROWS * P.row + P.gf + 3 * P.gb;
    P.off_tile = MX_NSI * P.stage;
    P.off_bt = P.off_tile + MX_NTILES_SMEM * MX_TILE_BYTES;
    P.off_cf = P.off_bt + 2 * 4 * 32 * 16;
    P.off_bar = mx_pad128(P.off_cf + Ly * 4 * 16 * 4);
    P.total = P.off_bar + 64;
    return P;
}

typedef P2<float>::T T2;

// link stored as 3 float4 segments; row 2 = conj(row0 x row1)
// (sgn = +-1 multiplies the link: rows 0 and 1 are scaled before the cross product, which then needs no sign of its
// own for the first factor and one for the second: row 2 = conj((sgn row0) x row1))
__device__ __forceinline__ void mx_lds_link(const unsigned char* p, int seg, float* u, float sgn) {
    float r1[6];
#pragma unroll
    for (int k = 0; k < 3; k++) {
        const float4 f = *reinterpret_cast<const float4*>(p + k * seg);
        u[4 * k] = f.x; u[4 * k + 1] = f.y; u[4 * k + 2] = f.z; u[4 * k + 3] = f.w;
    }
#pragma unroll
    for (int i = 0; i < 6; i++) { r1[i] = u[6 + i]; u[i] *= sgn; u[6 + i] *= sgn; }
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const int i = (c + 1) % 3, j = (c + 2) % 3;
        const float ar = u[2 * i], ai = u[2 * i + 1], br = r1[2 * j], bi = r1[2 * j + 1];
        const float cr = u[2 * j], ci = u[2 * j + 1], dr = r1[2 * i], di = r1[2 * i + 1];
        float re = ar * br; re -= ai * bi; re -= cr * dr; re += ci * di;
        float im = ar * bi; im += ai * br; im -= cr * di; im -= ci * dr;
        u[12 + 2 * c] = re;
        u[12 + 2 * c + 1] = -im;
    }
}
// NCH consecutive 16-byte chunks (2 complex numbers each) of one site of a staged spinor row
template <int NCH>
__device__ __forceinline__ void mx_lds_pairs(const unsigned char* p, int seg, T2* v) {
#pragma unroll
    for (int k = 0; k < NCH; k++) {
        const float4 f = *reinterpret_cast<const float4*>(p + k * seg);
        v[2 * k] = P2<float>::make(f.x, f.y);
        v[2 * k + 1] = P2<float>::make(f.z, f.w);
    }
}

// out[sp][a] (+|-)= sum_b U[a][b] in[sp][b] (DAG: U^dag) for the two spins of a half spinor (6 pairs); NEG subtracts
template <int DAG, int NEG>
__device__ __forceinline__ void mx_su3_half(const float* U, const T2* in, T2* out) {
    typedef P2<float> PP;
#pragma unroll
    for (int b = 0; b < 3; b++) {
        T2 ib[2];
#pragma unroll
        for (int sp = 0; sp < 2; sp++) ib[sp] = times_i<float>(in[sp * 3 + b]);
        float ur[3], ui[3];
#pragma unroll
        for (int a = 0; a < 3; a++) {
            ur[a] = DAG ? U[(b * 3 + a) * 2] : U[(a * 3 + b) * 2];
            ui[a] = DAG ? -U[(b * 3 + a) * 2 + 1] : U[(a * 3 + b) * 2 + 1];
            if (NEG) { ur[a] = -ur[a]; ui[a] = -ui[a]; }
        }
#pragma unroll
        for (int a = 0; a < 3; a++)
#pragma unroll
            for (int sp = 0; sp < 2; sp++) out[sp * 3 + a] = PP::fma_s(ur[a], in[sp * 3 + b], out[sp * 3 + a]);
#pragma unroll
        for (int a = 0; a < 3; a++)
#pragma unroll
            for (int sp = 0; sp < 2; sp++) out[sp * 3 + a] = PP::fma_s(ui[a], ib[sp], out[sp * 3 + a]);
    }
}

__device__ __forceinline__ void mma_tf32(float& d0, float& d1, float& d2, float& d3, unsigned a0, unsigned a1, unsigned a2,
                                         unsigned a3, unsigned b0, unsigned b1) {
    asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, {%0, %1, %2, %3};"
                 : "+f"(d0), "+f"(d1), "+f"(d2), "+f"(d3)
                 : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
#define MX_TF32_MASK 0xffffe000u

// x-sum of one tile on the tensor pipe + y-stage update.  tile: [8 components][32 columns] complex, column XOR 8 for
// odd components; thread (gg, tt) reads row gg; bt: this lane's B fragments of the row parity, [4 k-steps] 32 apart.
template <int NA>
__device__ __forceinline__ void mx_dft_tile(const T2* tile, const float4* bt, int gg, int tt, const float* cy, T2* Q) {
    typedef P2<float> PP;
    float d0 = 0.f, d1 = 0.f, d2 = 0.f, d3 = 0.f;        // three independent accumulation chains (MMA latency)
    float e0 = 0.f, e1 = 0.f, e2 = 0.f, e3 = 0.f, f0 = 0.f, f1 = 0.f, f2 = 0.f, f3 = 0.f;
    const float4* arow = reinterpret_cast<const float4*>(tile + gg * MX_BS);
    const int swz = (gg & 1) << 2;
#pragma unroll
    for (int ks = 0; ks < 4; ks++) {
        const float4 a = arow[(4 * ks + tt) ^ swz];          // (re, im) of logical columns 8 ks + 2t, + 1
        const float4 b = bt[ks * 32];
        const unsigned h0 = __float_as_uint(a.x) & MX_TF32_MASK, h1 = __float_as_uint(a.y) & MX_TF32_MASK;
        const unsigned h2 = __float_as_uint(a.z) & MX_TF32_MASK, h3 = __float_as_uint(a.w) & MX_TF32_MASK;
        const float l0 = a.x - __uint_as_float(h0), l1 = a.y - __uint_as_float(h1);
        const float l2 = a.z - __uint_as_float(h2), l3 = a.w - __uint_as_float(h3);
        const unsigned bh0 = __float_as_uint(b.x), bh1 = __float_as_uint(b.y);
        const unsigned bl0 = __float_as_uint(b.z), bl1 = __float_as_uint(b.w);
        mma_tf32(e0, e1, e2, e3, __float_as_uint(l0), __float_as_uint(l1), __float_as_uint(l2), __float_as_uint(l3), bh0, bh1);
        mma_tf32(f0, f1, f2, f3, h0, h1, h2, h3, bl0, bl1);
        mma_tf32(d0, d1, d2, d3, h0, h1, h2, h3, bh0, bh1);
    }
    d0 += e0 + f0; d1 += e1 + f1; d2 += e2 + f2; d3 += e3 + f3;
    // D rows gg, gg + 8 = re, im of component gg; columns 2t, 2t + 1
    const T2 va = PP::make(d0, d2), vb = PP::make(d1, d3);
#pragma unroll
    for (int j = 0; j < NA; j++) {
        Q[j] = PP::fma_s(cy[j], va, Q[j]);
        Q[NA + j] = PP::fma_s(cy[NA + j], vb, Q[NA + j]);
    }
}

template <int PRUNE, int XH>        // XH: Lx / 2 at compile time (shared-memory offsets become immediates), 0 = run time
__global__ void __launch_bounds__(MX_NTHREADS, 1)
contract_xy_mma_kernel(const __grid_constant__ CUtensorMap tm_s, const __grid_constant__ CUtensorMap tm_e,
                       const __grid_constant__ CUtensorMap tm_gf, const __grid_constant__ CUtensorMap tm_gb,
                       const __grid_constant__ MmaContractArgs A) {
    typedef P2<float> PP;
    constexpr int NQ = QLayout<PRUNE>::NQ;
    constexpr int NA = PRUNE ? 5 : 7;                   // accumulators per D column
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    const Geom& g = A.g;
    const int Xh = XH ? XH : g.Xh;
    const int X0 = 2 * Xh;
    const MxPlan P = mx_plan(X0, g.X1);
    float4* bt = reinterpret_cast<float4*>(smem_raw + P.off_bt);       // [2 row parities][4 k-steps][32 lanes]
    float* cf = reinterpret_cast<float*>(smem_raw + P.off_cf);         // [Ly][4][16]
    const unsigned bar_full = smem_u32(smem_raw + P.off_bar), bar_empty = bar_full + 8 * MX_NSI;
    const int zt = blockIdx.x + A.t_first * g.X2;
    const int z = zt % g.X2, t = zt / g.X2;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

    // tiles start at zero: the columns of inactive lanes (Lx < 32) and rows 4..7 of the quarter-tiles are never
    // written and must contribute nothing
    for (int i = threadIdx.x; i < MX_NTILES_SMEM * MX_TILE_BYTES / 16; i += MX_NTHREADS)
        reinterpret_cast<float4*>(smem_raw + P.off_tile)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    // B fragments (x-weights, split into tf32 hi + lo) of lane (g, t) for k-step ks: logical columns 8 ks + 2t, + 1;
    // column l <-> x = 2 (l % Xh) + ((l / Xh) ^ row parity)
    for (int i = threadIdx.x; i < 2 * 4 * 32; i += MX_NTHREADS) {
        const int rp = i >> 7, ks = (i >> 5) & 3, ln = i & 31;
        const int gq = ln >> 2, tq = ln & 3;
        float hi[2], lo[2];
#pragma unroll
        for (int j = 0; j < 2; j++) {
            const int l = 8 * ks + 2 * tq + j;
            float w = 0.f;
            if (l < X0) {
                const int x = 2 * (l % Xh) + ((l / Xh) ^ rp);
                w = A.wx[x * 8 + c_mx_wsel[gq]];
            }
            hi[j] = __uint_as_float(__float_as_uint(w) & MX_TF32_MASK);
            lo[j] = w - hi[j];
        }
        bt[i] = make_float4(hi[0], hi[1], lo[0], lo[1]);
    }
    for (int i = threadIdx.x; i < g.X1 * 4 * 16; i += MX_NTHREADS) {
        const int y = i >> 6, tq = (i >> 4) & 3, j = i & 15;
        cf[i] = A.wy[y * 8 + A.slots.sel[tq][j]];
    }
    if (threadIdx.x == 0) {
        for (int s = 0; s < MX_NSI; s++) {
            mbar_init(bar_full + 8 * s, 1);
            mbar_init(bar_empty + 8 * s, MX_NW);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // ---- this warp's job
    const int fam = warp >> 3, mu = (warp >> 1) & 3, h = warp & 1;
    const int p = lane / Xh, idx = lane - p * Xh;       // site of this lane: parity block p, in-row half index idx
    const bool active = lane < X0;
    const float sgn_f = (mu == 3 && t + 1 == g.X3) ? A.tb : 1.f;
    const float sgn_b = (mu == 3 && t == 0) ? A.tb : 1.f;
    const int seg = Xh * 16;
    const int idx_up = idx + 1 == Xh ? 0 : idx + 1, idx_dn = idx == 0 ? Xh - 1 : idx - 1;
    const int off_sv = SR_C * P.row + ((p * 6) * Xh + idx) * 16;                         // centre s, chunk 0
    const int off_uf = MX_NROWS * P.row + (((p * 4 + mu) * 3) * Xh + idx) * 16;        // U_mu(x)
    // backward link U_mu(x - mu): mu = 0 from the row's own forward block, else from the staged neighbour row
    const int ub_blk = mu == 0 ? MX_NROWS * P.row + (((1 - p) * 4) * 3) * Xh * 16
                               : MX_NROWS * P.row + P.gf + (mu - 1) * P.gb + ((1 - p) * 3) * Xh * 16;
    const int rf = fam == 0 ? (mu == 0 ? SR_C : mu == 1 ? SR_YP : mu == 2 ? SR_ZP : SR_TP)
                            : (mu == 0 ? ER_C : mu == 1 ? ER_YP : mu == 2 ? ER_ZP : ER_TP);
    const int rb = mu == 0 ? ER_C : mu == 1 ? ER_YM : mu == 2 ? ER_ZM : ER_TM;       // s family: no backward half
    const int nbf_blk = rf * P.row + ((1 - p) * 6 + 3 * h) * Xh * 16;                  // spins 2h, 2h+1 of the neighbour
    const int nbb_blk = rb * P.row + ((1 - p) * 6 + 3 * h) * Xh * 16;
    // ultra-local quarter job of the s-family warps: column b0 of C_{f0,0}[a][b0] = sum_c conj(s_ac) f_{b0,c}
    const int f0 = (warp >> 2) & 1, b0 = warp & 3;
    const int off_q = (f0 ? ER_C : SR_C) * P.row + ((p * 6 + ((6 * b0) >> 2)) * Xh + idx) * 16;
    T2* tile = reinterpret_cast<T2*>(smem_raw + P.off_tile + warp * MX_TILE_BYTES);
    T2* qtile = reinterpret_cast<T2*>(smem_raw + P.off_tile + (MX_NW + (warp & 7)) * MX_TILE_BYTES);
    const int gg = lane >> 2, tt = lane & 3;

    // ---- loader (lane 0 of warp 0): 15 TMA tensor copies per row
    const bool loader = warp == 0 && lane == 0;
    const unsigned in0 = smem_u32(smem_raw);
    const int zp = z + 1 == g.X2 ? 0 : z + 1, zm = z == 0 ? g.X2 - 1 : z - 1;
    const int tp = t + 1 == g.X3 ? 0 : t + 1, tm = t == 0 ? g.X3 - 1 : t - 1;
    const unsigned bytes = (unsigned)(MX_NROWS * 12 + 24 + 18) * (unsigned)P.seg;
    auto issue_row = [&](int y) {
        const int si = y % MX_NSI;
        const unsigned full = bar_full + 8 * si;
        mbar_expect_tx(full, bytes);
        const int yp = y + 1 == g.X1 ? 0 : y + 1, ym = y == 0 ? g.X1 - 1 : y - 1;
        // float coordinate of the first site of row (yy, zz, t4) inside a parity block: 4 * (lex / 2)
        auto c0 = [&](int yy, int zz, int t4) { return 2 * (((t4 * g.X2 + zz) * g.X1 + yy) * X0); };
        const int cC = c0(y, z, t), cYP = c0(yp, z, t), cYM = c0(ym, z, t), cZP = c0(y, zp, t), cZM = c0(y, zm, t),
                  cTP = c0(y, z, tp), cTM = c0(y, z, tm);
        const unsigned st0 = in0 + (unsigned)si * (unsigned)P.stage;
        tma_load_2d(st0 + (unsigned)(SR_C * P.row), &tm_s, full, cC, 0);
        tma_load_2d(st0 + (unsigned)(SR_YP * P.row), &tm_s, full, cYP, 0);
        tma_load_2d(st0 + (unsigned)(SR_ZP * P.row), &tm_s, full, cZP, 0);
        tma_load_2d(st0 + (unsigned)(SR_TP * P.row), &tm_s, full, cTP, 0);
        tma_load_2d(st0 + (unsigned)(ER_C * P.row), &tm_e, full, cC, 0);
        tma_load_2d(st0 + (unsigned)(ER_YP * P.row), &tm_e, full, cYP, 0);
        tma_load_2d(st0 + (unsigned)(ER_YM * P.row), &tm_e, full, cYM, 0);
        tma_load_2d(st0 + (unsigned)(ER_ZP * P.row), &tm_e, full, cZP, 0);
        tma_load_2d(st0 + (unsigned)(ER_ZM * P.row), &tm_e, full, cZM, 0);
        tma_load_2d(st0 + (unsigned)(ER_TP * P.row), &tm_e, full, cTP, 0);
        tma_load_2d(st0 + (unsigned)(ER_TM * P.row), &tm_e, full, cTM, 0);
        const unsigned gbase = st0 + (unsigned)(MX_NROWS * P.row);
        tma_load_4d(gbase, &tm_gf, full, cC, 0, 0, 0);
        tma_load_4d(gbase + (unsigned)P.gf, &tm_gb, full, cYM, 0, 1, 0);
        tma_load_4d(gbase + (unsigned)(P.gf + P.gb), &tm_gb, full, cZM, 0, 2, 0);
        tma_load_4d(gbase + (unsigned)(P.gf + 2 * P.gb), &tm_gb, full, cTM, 0, 3, 0);
    };
    if (loader) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_s) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_e) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_gf) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tm_gb) : "memory");
        for (int y = 0; y < MX_NSI - 1 && y < g.X1; y++) issue_row(y);
    }
    __syncwarp();

#ifndef MX_STAGGER_NS
#define MX_STAGGER_NS 550
#endif
    // The 4 warps of a sub-partition run the same phases (operand loads from shared memory, fp32 pipe, tile
    // transpose, tensor pipe) and nothing but the arrival of a row couples them, so started together they stay in
    // step and the shared-memory and fp32 phases add up instead of overlapping.  Start them a quarter of a row apart.
    if (MX_STAGGER_NS) __nanosleep(MX_STAGGER_NS * (warp >> 2));
    T2 Q[2 * NA], Qq[2 * NA];                           // y-stage accumulators: own tile, ultra-local quarter-tile
#pragma unroll
    for (int j = 0; j < 2 * NA; j++) { Q[j] = PP::make(0.f, 0.f); Qq[j] = PP::make(0.f, 0.f); }

    for (int y = 0; y < g.X1; y++) {
        const int si = y % MX_NSI;
        if (loader && y + MX_NSI - 1 < g.X1) {
            // row y + 2 goes where row y - 1 was: wait until all 16 warps have released that stage
            const int yl = y + MX_NSI - 1;
            if (yl >= MX_NSI) mbar_wait(bar_empty + 8 * (yl % MX_NSI), ((yl / MX_NSI) - 1) & 1);
            issue_row(yl);
        }
        __syncwarp();
        const unsigned char* stage = smem_raw + (size_t)si * P.stage;
        mbar_wait(bar_full + 8 * si, (y / MX_NSI) & 1);
        if (active) {
            const int xo = (p ^ (y + z + t)) & 1;                 // x = 2 idx + xo
            const int idx_f = mu == 0 ? (xo ? idx_up : idx) : idx;
            const int idx_b = mu == 0 ? (xo ? idx : idx_dn) : idx;
            T2 sv[12];
            mx_lds_pairs<6>(stage + off_sv, seg, sv);
            T2 psi[6], nb[6];
            float U[18];
#pragma unroll
            for (int i = 0; i < 6; i++) psi[i] = PP::make(0.f, 0.f);
            // forward half: U_mu(x) f(x+mu), spins 2h, 2h+1
            // (the time-boundary sign of a wrapping hop goes onto the 18 link reals: no branch, no copy of nb)
            mx_lds_pairs<3>(stage + nbf_blk + idx_f * 16, seg, nb);
            mx_lds_link(stage + off_uf, seg, U, sgn_f);
            mx_su3_half<0, 0>(U, nb, psi);
            if (fam) {
                // eta family: minus the backward half U_mu^dag(x-mu) eta(x-mu)
                mx_lds_pairs<3>(stage + nbb_blk + idx_b * 16, seg, nb);
                mx_lds_link(stage + ub_blk + idx_b * 16, seg, U, sgn_b);
                mx_su3_half<1, 1>(U, nb, psi);
            }
            // C[a][2h + bl] = sum_c conj(s_ac) psi_{bl,c}  ->  tile row a * 2 + bl
            T2 acc[8];
#pragma unroll
            for (int i = 0; i < 8; i++) acc[i] = PP::make(0.f, 0.f);
#pragma unroll
            for (int c = 0; c < 3; c++) {
                float sre[4], sim[4];
                T2 ip[2];
#pragma unroll
                for (int a = 0; a < 4; a++) { PP::get(sv[a * 3 + c], sre[a], sim[a]); sim[a] = -sim[a]; }
#pragma unroll
                for (int bl = 0; bl < 2; bl++) ip[bl] = times_i<float>(psi[bl * 3 + c]);
#pragma unroll
                for (int a = 0; a < 4; a++)
#pragma unroll
                    for (int bl = 0; bl < 2; bl++) acc[a * 2 + bl] = PP::fma_s(sre[a], psi[bl * 3 + c], acc[a * 2 + bl]);
#pragma unroll
                for (int a = 0; a < 4; a++)
#pragma unroll
                    for (int bl = 0; bl < 2; bl++) acc[a * 2 + bl] = PP::fma_s(sim[a], ip[bl], acc[a * 2 + bl]);
            }
            {
                const int col0 = lane, col1 = lane ^ 8;        // odd tile rows: column XOR 8
#pragma unroll
                for (int i = 0; i < 8; i++) tile[i * MX_BS + ((i & 1) ? col1 : col0)] = acc[i];
            }
            if (fam == 0) {
                // ultra-local quarter job: C_{f0,0}[a][b0] = sum_c conj(s_ac) f_{b0,c}, f = s | eta at this site
                const float4 q0 = *reinterpret_cast<const float4*>(stage + off_q);
                const float4 q1 = *reinterpret_cast<const float4*>(stage + off_q + seg);
                T2 f3[3];
                if (b0 & 1) { f3[0] = PP::make(q0.z, q0.w); f3[1] = PP::make(q1.x, q1.y); f3[2] = PP::make(q1.z, q1.w); }
                else        { f3[0] = PP::make(q0.x, q0.y); f3[1] = PP::make(q0.z, q0.w); f3[2] = PP::make(q1.x, q1.y); }
                T2 a4[4];
#pragma unroll
                for (int a = 0; a < 4; a++) a4[a] = PP::make(0.f, 0.f);
#pragma unroll
                for (int c = 0; c < 3; c++) {
                    const T2 ip = times_i<float>(f3[c]);
                    float sre[4], sim[4];
#pragma unroll
                    for (int a = 0; a < 4; a++) { PP::get(sv[a * 3 + c], sre[a], sim[a]); }
#pragma unroll
                    for (int a = 0; a < 4; a++) a4[a] = PP::fma_s(sre[a], f3[c], a4[a]);
#pragma unroll
                    for (int a = 0; a < 4; a++) a4[a] = PP::fma_s(-sim[a], ip, a4[a]);
                }
                const int col0 = lane, col1 = lane ^ 8;
#pragma unroll
                for (int a = 0; a < 4; a++) qtile[a * MX_BS + ((a & 1) ? col1 : col0)] = a4[a];
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_empty + 8 * si);           // this warp is done reading the input stage
        // ---- x-sum on the tensor pipe, y-stage in registers
        const int rp = (y + z + t) & 1;
        float cy[16];
        {
            const float4* c4 = reinterpret_cast<const float4*>(cf + (y * 4 + tt) * 16);
#pragma unroll
            for (int k = 0; k < (2 * NA + 3) / 4; k++) {
                const float4 f = c4[k];
                cy[4 * k] = f.x; cy[4 * k + 1] = f.y; cy[4 * k + 2] = f.z; cy[4 * k + 3] = f.w;
            }
        }
        mx_dft_tile<NA>(tile, bt + rp * 4 * 32 + lane, gg, tt, cy, Q);
        if (fam == 0) mx_dft_tile<NA>(qtile, bt + rp * 4 * 32 + lane, gg, tt, cy, Qq);
        __syncwarp();                                             // tile reads done before the next row's stores
    }
    // ---- partial sums of the plane: component of tile row gg
    T2* qb = reinterpret_cast<T2*>((float*)A.qbuf + (size_t)zt * NQ * CT_THREADS);
    {
        const int cc = (fam * 5 + 1 + mu) * 16 + (gg >> 1) * 4 + 2 * h + (gg & 1);
#pragma unroll
        for (int j = 0; j < 2 * NA; j++) {
            const int q = A.slots.q[tt][j];
            if (q >= 0) qb[(size_t)q * CT_NCC + cc] = Q[j];
        }
    }
    if (fam == 0 && gg < 4) {
        const int cc = f0 * 80 + gg * 4 + b0;
#pragma unroll
        for (int j = 0; j < 2 * NA; j++) {
            const int q = A.slots.q[tt][j];
            if (q >= 0) qb[(size_t)q * CT_NCC + cc] = Qq[j];
        }
    }
}

// ------------------------------------------------------------------ host side

static bool mx_build_slots(MmaSlots* S, int prune) {
    short qidx[64];
    int nq;
    tm_contract_qidx(qidx, prune, &nq);
    const int NA = prune ? 5 : 7;
    typedef std::vector<std::pair<int, int>> List;
    // accumulators fed by the x-sum (m, cos | sin): for every allowed n the cos-y one and, for n > 0, the sin-y one
    auto entries = [&](int m, int part) {
        List out;
        for (int n = 0; n < 4; n++) {
            const short* e = qidx + (m * 4 + n) * 4;
            if (e[0] < 0) continue;
            const int base = part ? 2 : 0;
            out.push_back({e[base], n == 0 ? 0 : 2 * n - 1});
            if (n > 0) out.push_back({e[base + 1], 2 * n});
        }
        return out;
    };
    memset(S, 0, sizeof(*S));
    for (int t = 0; t < 4; t++)
        for (int j = 0; j < 16; j++) { S->q[t][j] = -1; S->sel[t][j] = 7; }
    List colA[4], colB[4];
    {
        const List m0 = entries(0, 0);
        for (size_t k = 0; k < m0.size(); k++) (k < 4 ? colA[0] : colB[0]).push_back(m0[k]);
    }
    colA[1] = entries(1, 0); colB[1] = entries(3, 0);
    colA[2] = entries(1, 1); colB[2] = entries(3, 1);
    colA[3] = entries(2, 0); colB[3] = entries(2, 1);
    int total = 0;
    for (int t = 0; t < 4; t++) {
        if ((int)colA[t].size() > NA || (int)colB[t].size() > NA) return false;
        for (size_t k = 0; k < colA[t].size(); k++) { S->q[t][k] = (signed char)colA[t][k].first; S->sel[t][k] = (signed char)colA[t][k].second; }
        for (size_t k = 0; k < colB[t].size(); k++) { S->q[t][NA + k] = (signed char)colB[t][k].first; S->sel[t][NA + k] = (signed char)colB[t][k].second; }
        total += (int)(colA[t].size() + colB[t].size());
    }
    return total == nq;
}

bool tm_contract_mma_usable(const tm_ctx* ctx) {
    if (ctx->X[0] > 32) return false;
    if (4 * ctx->Vh >= (size_t)1 << 31) return false;             // TMA coordinates are int32
    const MxPlan P = mx_plan(ctx->X[0], ctx->X[1]);
    if (P.total > 227 * 1024) return false;
    return get_encode_fn() != nullptr;
}

// s, eta: fp32 full-lattice internal fields; gauge: fp32 reconstruct-12 internal copy; wx, wy: float tables
tm_status tm_contract_xy_mma(tm_ctx* ctx, void* qbuf, const void* d_s, const void* d_eta, const void* gauge,
                             const void* wx, const void* wy, int prune, int t_first, int nt, cudaStream_t st) {
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
    MmaContractArgs A;
    A.qbuf = qbuf; A.wx = (const float*)wx; A.wy = (const float*)wy;
    A.g = tm_geom(ctx);
    A.tb = (float)ctx->tb;
    A.t_first = t_first;
    if (!mx_build_slots(&A.slots, prune)) return tm_fail(ctx, TM_ECUDA, "contract: accumulator slots do not cover the Q layout");
    const MxPlan P = mx_plan(ctx->X[0], ctx->X[1]);
    const unsigned grid = (unsigned)(ctx->X[2] * nt);
#define MX_LAUNCH(PR, XH)                                                                                              \
    do {                                                                                                               \
        TM_CUDA(ctx, cudaFuncSetAttribute(contract_xy_mma_kernel<PR, XH>, cudaFuncAttributeMaxDynamicSharedMemorySize, \
                                          P.total));                                                                   \
        contract_xy_mma_kernel<PR, XH><<<grid, MX_NTHREADS, P.total, st>>>(ms, me, mgf, mgb, A);                       \
    } while (0)
    if (prune) {
        if (Xh == 16) MX_LAUNCH(1, 16); else if (Xh == 12) MX_LAUNCH(1, 12); else if (Xh == 8) MX_LAUNCH(1, 8); else MX_LAUNCH(1, 0);
    } else {
        if (Xh == 16) MX_LAUNCH(0, 16); else MX_LAUNCH(0, 0);
    }
#undef MX_LAUNCH
    TM_LAUNCH_CHECK(ctx, "contract_xy_mma_kernel");
    return TM_OK;
}
