// factor.cu -- a1 (assemble A_j) + a2 (eliminate with partial pivoting) of SURVEY.md section 8(a).
//
// A_j = [delta_gg' L_{c,j,g} - S_{g'->g,j}]  (Eq. 40b), L_c block-diagonal in the ordinate
// (Eq. 8a-b), S_{(g,m,p),(g',m',p')} = delta_pp' (dx_j K_j[g][g'] / 4) w_m'  (Eq. 10 / 39,
// PAPER.md:154, 320, read as DESIGN.md A2). The matrix is assembled straight into on-chip memory and never
// written to HBM un-eliminated. Elimination is Gaussian elimination with partial (row) pivoting -- the same
// pivots `_gesv` takes in Alg. 2 -- carried through to the inverse (Gauss-Jordan, in
// place, implicit row exchange), because the iterate kernel streams A_j^{-1}.
#include "common.cuh"
#include <cooperative_groups.h>
#include <limits.h>
#include <string.h>

namespace {

constexpr int FACTOR_THREADS = 256;

// Entry (i, c) of A_j, every rounding explicit (bit-identical to an uncontracted evaluation).
__device__ __forceinline__ double a_entry(const ProblemView &P, int cell, int i, int c)
{
    const int N = P.N, G = P.G;
    const int p = i & 3, bm = i >> 2, m = bm % N, g = bm / N;
    const int pp = c & 3, bmc = c >> 2, mc = bmc % N, gc = bmc / N;
    const double dx = P.dx[cell];
    double val = 0.0;
    if (bm == bmc) val = lc_entry(p, pp, dx, P.sigma_t[(size_t)cell * G + g], P.v[g], P.dt, P.mu[m]);
    if (p == pp) {
        const double K = P.transfer[((size_t)cell * G + g) * G + gc];
        const double s = __dmul_rn(__dmul_rn(__dmul_rn(dx, K), 0.25), P.w[mc]); // dx K / 4 * w_m'
        val = __dsub_rn(val, s);
    }
    return val;
}

// One CTA per cell (grid-stride). W is the n x n working array, row-major with leading dimension ldw:
// in shared memory when it fits (ldw = n + 1, conflict-free column access), else in a per-CTA global scratch
// that stays L2-resident.
template <bool GLOBAL_W>
__global__ void __launch_bounds__(FACTOR_THREADS)
factor_gj_kernel(ProblemView P, double *__restrict__ Minv, double *__restrict__ scratch, int ldw, int *info)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int n = P.n;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NW = FACTOR_THREADS / 32;

    double *sm = reinterpret_cast<double *>(smem_raw);
    double *colk = sm;               // [n]
    double *prow = colk + n;         // [n]
    double *wmax = prow + n;         // [NW]
    int *widx = reinterpret_cast<int *>(wmax + NW); // [NW]
    int *rho = widx + NW;            // [n] pivot row of step k
    int *rhoinv = rho + n;           // [n]
    int *used = rhoinv + n;          // [n]
    double *Wsm = reinterpret_cast<double *>(used + n + ((n + NW) & 1)); // keep 8-byte alignment
    double *W = GLOBAL_W ? scratch + (size_t)blockIdx.x * n * ldw : Wsm;

    for (int cell = blockIdx.x; cell < P.J; cell += gridDim.x) {
        // ---- a1: assemble
        for (int i = warp; i < n; i += NW)
            for (int c = lane; c < n; c += 32) W[(size_t)i * ldw + c] = a_entry(P, cell, i, c);
        for (int i = tid; i < n; i += FACTOR_THREADS) used[i] = 0;
        __syncthreads();

        bool singular = false;
        // ---- a2: elimination, step k eliminates column k with the pivot row rho_k
        for (int k = 0; k < n; ++k) {
            double cand = -1.0;
            int ci = INT_MAX;
            for (int i = tid; i < n; i += FACTOR_THREADS) {
                const double vv = W[(size_t)i * ldw + k];
                colk[i] = vv;
                const double a = used[i] ? -1.0 : fabs(vv);
                if (a > cand) { cand = a; ci = i; }
            }
            // arg-max by warp shuffles: larger |entry| wins, ties go to the lower row
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                const double oc = __shfl_xor_sync(0xffffffffu, cand, o);
                const int oi = __shfl_xor_sync(0xffffffffu, ci, o);
                if (oc > cand || (oc == cand && oi < ci)) { cand = oc; ci = oi; }
            }
            if (lane == 0) { wmax[warp] = cand; widx[warp] = ci; }
            __syncthreads();
            double best = wmax[0];
            int r = widx[0];
#pragma unroll
            for (int q = 1; q < NW; ++q) {
                const double oc = wmax[q];
                const int oi = widx[q];
                if (oc > best || (oc == best && oi < r)) { best = oc; r = oi; }
            }
            if (!(best > 0.0)) { singular = true; break; } // uniform across the CTA
            const double inv = 1.0 / colk[r];
            for (int c = tid; c < n; c += FACTOR_THREADS)
                prow[c] = (c == k ? 1.0 : W[(size_t)r * ldw + c]) * inv;
            if (tid == 0) { used[r] = 1; rho[k] = r; rhoinv[r] = k; }
            __syncthreads();
            for (int i = warp; i < n; i += NW) {
                double *Wi = W + (size_t)i * ldw;
                if (i == r) {
                    for (int c = lane; c < n; c += 32) Wi[c] = prow[c];
                } else {
                    const double f = colk[i];
                    if (f != 0.0)
                        for (int c = lane; c < n; c += 32) {
                            const double base = (c == k) ? 0.0 : Wi[c];
                            Wi[c] = fma(-f, prow[c], base);
                        }
                }
            }
            __syncthreads();
        }
        if (singular) {
            if (tid == 0) atomicMin(info, cell + 1);
            // leave a NaN-free but meaningless block behind: zero it
            for (int e = tid; e < n * n; e += FACTOR_THREADS) Minv[(size_t)cell * n * n + e] = 0.0;
            __syncthreads();
            continue;
        }
        // ---- store A^{-1} column-major: Ainv[kappa][rho_j] = W[rho_kappa][j]  (un-scrambles the implicit exchange)
        double *out = Minv + (size_t)cell * n * n;
        for (int j = warp; j < n; j += NW) {
            const int col = rho[j];
            for (int i = lane; i < n; i += 32) out[(size_t)col * n + rhoinv[i]] = W[(size_t)i * ldw + j];
        }
        __syncthreads();
    }
}

namespace cg = cooperative_groups;

constexpr int FR_NB = 8; // panel width of every blocked factor kernel below

// Branch-free reciprocal: hardware seed (MUFU.RCP64H, relative error 2^-19.9) + one cubic Newton step. Measured on a
// B200 over 1.3e9 random arguments: at most 1 ulp from the correctly rounded 1 / x (one more quadratic step, two FMAs,
// makes it correctly rounded; they sat on every pivot step's critical path and bought nothing the 1e-11 parity bar
// can see). No special cases: zero / non-finite pivots are flagged separately as singular.
__device__ __forceinline__ double rcp_nr(double x)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    double e = fma(-x, r, 1.0);
    e = fma(e, e, e);
    return fma(r, e, r);
}

// ============================================================================================================
// n = 64: ONE WARP PER CELL, the working matrix in shared memory, rank-8 updates on the FP64 tensor path (DMMA):
// the production a1 + a2 kernel of the headline configuration.
// ============================================================================================================
// Partial pivoting makes the 64 pivot decisions of a cell strictly sequential, and each is a chain of dependent
// latencies (arg-max reduction, ballot, broadcast of the pivot row, one fused multiply-add). The throughput of the
// kernel is therefore (cells in flight per SM) / (length of that chain), and the chain is shortest when NOTHING in it
// crosses a warp: no CTA barrier, no exchange through another warp. So a cell belongs to one warp from assembly to
// store, six cells (warps) are resident per SM and drift apart in phase, which overlaps one cell's pivot chain with
// another cell's rank-8 update.
//   W      column-major in shared memory, leading dimension 66: lane l reads rows {2 l, 2 l + 1} of a column as one
//          conflict-free 16-byte access (assembly, panel phase, store), and the 8 x 8 accumulator fragments of
//          mma.sync.m8n8k4.f64 (lane holds row l / 4, columns 2 (l % 4), + 1) are conflict-free 8-byte accesses
//          (66 = 2 mod 8 spreads the four columns of a half-warp over all 32 banks).
//   phase P (panel of 8 columns, in registers, two rows per lane): per pivot step the local winner of the lane's two
//          rows (exact 64-bit compare, lower row on a tie), redux.sync.max on the high key word + ballot (exact tie
//          path behind a warp-uniform branch: first maximal |entry|), every lane scales its candidate row by a
//          branch-free reciprocal in the shadow of the reduction, the winner broadcasts its scaled row through 64
//          bytes of shared memory, 16 fused multiply-adds per lane.
//   phase U  W[:, c] += Z W_old[R, c] for the 56 other columns, Z = T[:, R] - I[:, R]: per 8 x 8 tile two
//          mma.sync.m8n8k4.f64 with the A fragments (Z, read from the eliminated panel in place) and the B fragments
//          (the 8 pivot rows of the column block, read before the block is touched) held in registers. A DMMA carries
//          8 fused multiply-adds per lane in ONE issue slot at the full rate of the FP64 pipe (measured on this B200:
//          16.5 cycles per DMMA and sub-partition = 64 FMA/clk/SM from one warp per sub-partition; the DFMA form of
//          the same update needs 8 issue slots and 4.5 shared-memory loads per 8 FMAs) -- DMMA_UPD = false keeps that
//          form for the A/B measurement DESIGN.md quotes.
//   store  rows and columns un-scrambled on the way out: lane l gathers rows {rho[2 l], rho[2 l + 1]} of column
//          rhoinv[c] and writes 16 contiguous bytes of column c of A^{-1}.
// Cells are handed out by an atomic counter (a static split would leave the sub-partitions that hold two of the six
// warps behind).
constexpr int WC_LD = 66;

struct WcShared {
    double W[64 * WC_LD];          // [column][row], column-major working matrix
    double prow[2][FR_NB];         // [step parity][c]: the scaled pivot row of the current step
    int rho[64], rhoinv[64];
};

__device__ __forceinline__ void dmma884(double &c0, double &c1, double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c0), "+d"(c1)
        : "d"(a), "d"(b));
}

// NT row tiles (8 rows each) of one column block: v[tile] += a0 z0[tile] + a1 z1[tile], the transposed rank-8 update of
// wc2_update_blocks with the B fragments (z0, z1: the eliminated panel) read from shared memory. Software-pipelined by
// hand: the compiler must assume that the store of a tile aliases the loads of the next one and, left alone, emits
// load -> DMMA -> dependent DMMA -> store tile after tile (~100 cycles of exposed latency per tile). Here the loads of
// the next four tiles are issued before the DMMAs of the current four, and the two dependent DMMAs of a tile are four
// issue slots (~66 cycles) apart, so the warp is bound by the 16.5 cycles a DMMA occupies its sub-partition's pipe.
// cp: the lane's double2 of tile 0 (tile stride: 4 double2 = 8 rows); zp0 / zp1: the lane's B-fragment entries of tile 0
// (tile stride 8 doubles).
template <int NT>
__device__ __forceinline__ void dmma_strip(double2 *cp, const double *zp0, const double *zp1, double a0, double a1)
{
    static_assert(NT % 4 == 0, "tiles are processed four at a time");
    double2 v[2][4];
    double z0[2][4], z1[2][4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        v[0][i] = cp[4 * i];
        z0[0][i] = zp0[8 * i];
        z1[0][i] = zp1[8 * i];
    }
#pragma unroll
    for (int bt = 0; bt < NT / 4; ++bt) {
        const int cur = bt & 1;
        if (bt + 1 < NT / 4) {
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int I = 4 * (bt + 1) + i;
                v[cur ^ 1][i] = cp[4 * I];
                z0[cur ^ 1][i] = zp0[8 * I];
                z1[cur ^ 1][i] = zp1[8 * I];
            }
        }
#pragma unroll
        for (int i = 0; i < 4; ++i) dmma884(v[cur][i].x, v[cur][i].y, a0, z0[cur][i]);
#pragma unroll
        for (int i = 0; i < 4; ++i) dmma884(v[cur][i].x, v[cur][i].y, a1, z1[cur][i]);
#pragma unroll
        for (int i = 0; i < 4; ++i) cp[4 * (4 * bt + i)] = v[cur][i];
    }
}

// a1 for one warp: rows {2 lane, 2 lane + 1} of every column of A_j into the column-major shared-memory array W
// (leading dimension ld). Same operations in the same order as a_entry(): bit-identical (asserted by
// tests/test_gpu_parity.py::test_production_assembly_bit_exact through oci_debug_get_factor_input).
__device__ __forceinline__ void assemble_rows2(const ProblemView &P, int cell, int lane, double *W, int ld,
                                               int bmc0 = 0, int bmc_step = 1, int rb0 = 0, int rb_step = 64)
{
    const int N = P.N, G = P.G, NB = N * G;
    const double dx = P.dx[cell];
    for (int rb = rb0; rb < P.n; rb += rb_step) { // row block: rows rb + 2 lane, + 1
        const int p0 = (lane & 1) * 2;
        const int bm = (rb >> 2) + (lane >> 1), m = bm % N, g = bm / N;
        const double sig = P.sigma_t[(size_t)cell * G + g], mu = P.mu[m];
        const double av = __dmul_rn(__dadd_rn(fabs(mu), __dmul_rn(dx, sig)), 0.5);
        const double gam = __ddiv_rn(dx, __dmul_rn(P.v[g], P.dt));
        const double h = __dmul_rn(mu, 0.5), hg = __dmul_rn(gam, 0.5), ga = __dadd_rn(gam, av);
        const double *Krow = P.transfer + ((size_t)cell * G + g) * G;
        for (int bmc = bmc0; bmc < NB; bmc += bmc_step) { // column block (g', m')
            const double Kw = __dmul_rn(__dmul_rn(__dmul_rn(dx, Krow[bmc / N]), 0.25), P.w[bmc % N]);
            const bool diag = bm == bmc;
#pragma unroll
            for (int pp = 0; pp < 4; ++pp) {
                double val[2];
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int p = p0 + e, d = pp - p;
                    double x = 0.0;
                    if (diag) { // Eq. 8b
                        if (d == 0) x = p < 2 ? av : ga;
                        else if (p == 0 && pp == 1) x = h;
                        else if (p == 1 && pp == 0) x = -h;
                        else if (p == 2 && pp == 3) x = h;
                        else if (p == 3 && pp == 2) x = -h;
                        else if (d == 2) x = hg;
                        else if (d == -2) x = -gam;
                    }
                    if (p == pp) x = __dsub_rn(x, Kw);
                    val[e] = x;
                }
                *reinterpret_cast<double2 *>(&W[(size_t)(4 * bmc + pp) * ld + rb + 2 * lane]) = make_double2(val[0], val[1]);
            }
        }
    }
}

template <bool DMMA_UPD, bool DUMP>
__global__ void __launch_bounds__(32)
factor_wc_kernel(ProblemView P, double *__restrict__ Minv, int *info, int *next_cell, double *__restrict__ dumpA, int dump_cell,
                 int /* role_mode: factor_wc2_kernel only */)
{
    constexpr int n = 64, LD = WC_LD, NPANEL = n / FR_NB;
    constexpr unsigned FULL = 0xffffffffu;
    extern __shared__ __align__(16) unsigned char wc_smem[];
    WcShared &sh = *reinterpret_cast<WcShared *>(wc_smem);
    double *W = sh.W;
    const int lane = threadIdx.x, lq = lane & 3, lg = lane >> 2;

    for (;;) {
        int cell = dump_cell;
        if (!DUMP) {
            if (lane == 0) cell = atomicAdd(next_cell, 1);
            cell = __shfl_sync(FULL, cell, 0);
        }
        if (cell >= P.J) break;
        assemble_rows2(P, cell, lane, W, LD);
        __syncwarp();
        if (DUMP) { // the assembled tile of the production kernel, row-major, for the bit-exactness test
            for (int e = lane; e < n * n; e += 32) dumpA[e] = W[(e & 63) * LD + (e >> 6)];
            break;
        }

        bool used0 = false, used1 = false; // rows 2 lane, 2 lane + 1 have been pivot rows
        bool singular = false;
        for (int pnl = 0; pnl < NPANEL; ++pnl) {
            // ================= phase P: the 64 x 8 panel in registers, two rows per lane =================
            double t[FR_NB][2];
#pragma unroll
            for (int c = 0; c < FR_NB; ++c) {
                const double2 v = *reinterpret_cast<const double2 *>(&W[(FR_NB * pnl + c) * LD + 2 * lane]);
                t[c][0] = v.x;
                t[c][1] = v.y;
            }
            int Rl[FR_NB];
            bool bad = false;
#pragma unroll
            for (int b = 0; b < FR_NB; ++b) {
                const unsigned long long key0 = used0 ? 0ull : (unsigned long long)__double_as_longlong(fabs(t[b][0]));
                const unsigned long long key1 = used1 ? 0ull : (unsigned long long)__double_as_longlong(fabs(t[b][1]));
                const bool e1 = key1 > key0; // the lane's own winner: the lower row on a tie
                const unsigned long long key = e1 ? key1 : key0;
                const unsigned khi = (unsigned)(key >> 32);
                const unsigned mhi = __reduce_max_sync(FULL, khi);
                const unsigned eball = __ballot_sync(FULL, e1);
                // in the shadow of the reduction: the lane's candidate row scaled by 1 / its candidate
                double tl[FR_NB];
#pragma unroll
                for (int c = 0; c < FR_NB; ++c) tl[c] = e1 ? t[c][1] : t[c][0];
                const double linv = rcp_nr(tl[b]);
                double scl[FR_NB];
#pragma unroll
                for (int c = 0; c < FR_NB; ++c) scl[c] = (c == b) ? linv : tl[c] * linv;
                bool cand = khi == mhi;
                const unsigned ball = __ballot_sync(FULL, cand);
                int src;
                if (__popc(ball) == 1) {
                    src = __ffs(ball) - 1;
                } else { // ties in the high word: low words, then the lowest lane (= the lowest row)
                    const unsigned klo = (unsigned)key;
                    const unsigned mlo = __reduce_max_sync(FULL, cand ? klo : 0u);
                    cand = cand && klo == mlo;
                    const unsigned b2 = __ballot_sync(FULL, cand);
                    src = b2 ? __ffs(b2) - 1 : 0;
                }
                if (mhi == 0u || mhi >= 0x7ff00000u) bad = true; // pivot with a zero high word (0, or a denormal below 2^-1042), inf, NaN, or no unused row
                const int esrc = (eball >> src) & 1;
                if (lane == src) {
                    double2 *dst = reinterpret_cast<double2 *>(sh.prow[b & 1]);
#pragma unroll
                    for (int c = 0; c < FR_NB / 2; ++c) dst[c] = make_double2(scl[2 * c], scl[2 * c + 1]);
                }
                __syncwarp(); // (two buffers alternate: no second barrier needed)
                double sp[FR_NB];
#pragma unroll
                for (int c = 0; c < FR_NB / 2; ++c) {
                    const double2 v = reinterpret_cast<const double2 *>(sh.prow[b & 1])[c];
                    sp[2 * c] = v.x;
                    sp[2 * c + 1] = v.y;
                }
                Rl[b] = 2 * src + esrc;
                const bool p0 = lane == src && esrc == 0, p1 = lane == src && esrc == 1;
                const double f0 = t[b][0], f1 = t[b][1];
#pragma unroll
                for (int c = 0; c < FR_NB; ++c) { // the pivot row becomes itself / pivot (= scl)
                    const double u0 = (c == b) ? -f0 * sp[b] : fma(-f0, sp[c], t[c][0]);
                    const double u1 = (c == b) ? -f1 * sp[b] : fma(-f1, sp[c], t[c][1]);
                    t[c][0] = p0 ? scl[c] : u0;
                    t[c][1] = p1 ? scl[c] : u1;
                }
                used0 = used0 || p0;
                used1 = used1 || p1;
                if (lane == b) { sh.rho[FR_NB * pnl + b] = Rl[b]; sh.rhoinv[Rl[b]] = FR_NB * pnl + b; }
            }
            if (bad) { singular = true; break; } // warp-uniform
            // the eliminated panel (its columns now hold T e_r) back in place
#pragma unroll
            for (int c = 0; c < FR_NB; ++c)
                *reinterpret_cast<double2 *>(&W[(FR_NB * pnl + c) * LD + 2 * lane]) = make_double2(t[c][0], t[c][1]);
            __syncwarp();

            // ================= phase U: rank-8 update of the other 56 columns =================
            if (DMMA_UPD) {
                const int rk0 = sh.rho[FR_NB * pnl + lq], rk1 = sh.rho[FR_NB * pnl + 4 + lq];
                double af[8][2]; // A fragments: Z[8 I + lg][4 h + lq]
#pragma unroll
                for (int I = 0; I < 8; ++I) {
                    const int row = 8 * I + lg;
                    af[I][0] = W[(FR_NB * pnl + lq) * LD + row] - (rk0 == row ? 1.0 : 0.0);
                    af[I][1] = W[(FR_NB * pnl + 4 + lq) * LD + row] - (rk1 == row ? 1.0 : 0.0);
                }
                for (int Jb = 0; Jb < 8; ++Jb) {
                    if (Jb == pnl) continue;
                    // B fragments: W_old[R[4 h + lq]][8 Jb + lg], read before any lane touches this column block
                    const double bf0 = W[(8 * Jb + lg) * LD + rk0], bf1 = W[(8 * Jb + lg) * LD + rk1];
                    __syncwarp();
                    double *cp = &W[(8 * Jb + 2 * lq) * LD + lg];
#pragma unroll
                    for (int I = 0; I < 8; ++I) {
                        double c0 = cp[8 * I], c1 = cp[LD + 8 * I];
                        dmma884(c0, c1, af[I][0], bf0);
                        dmma884(c0, c1, af[I][1], bf1);
                        cp[8 * I] = c0;
                        cp[LD + 8 * I] = c1;
                    }
                }
            } else {
                double z[FR_NB][2];
#pragma unroll
                for (int b = 0; b < FR_NB; ++b) {
                    z[b][0] = t[b][0] - (Rl[b] == 2 * lane ? 1.0 : 0.0);
                    z[b][1] = t[b][1] - (Rl[b] == 2 * lane + 1 ? 1.0 : 0.0);
                }
                for (int c = 0; c < n; ++c) {
                    if ((c >> 3) == pnl) continue;
                    double rv[FR_NB];
#pragma unroll
                    for (int b = 0; b < FR_NB; ++b) rv[b] = W[c * LD + Rl[b]]; // uniform address
                    double2 v = *reinterpret_cast<const double2 *>(&W[c * LD + 2 * lane]);
                    __syncwarp(); // every lane has read the pivot rows of this column
#pragma unroll
                    for (int b = 0; b < FR_NB; ++b) { v.x = fma(z[b][0], rv[b], v.x); v.y = fma(z[b][1], rv[b], v.y); }
                    *reinterpret_cast<double2 *>(&W[c * LD + 2 * lane]) = v;
                }
            }
            __syncwarp();
        }

        double *out = Minv + (size_t)cell * n * n;
        if (singular) {
            if (lane == 0) atomicMin(info, cell + 1);
            for (int e = lane; e < n * n / 2; e += 32) reinterpret_cast<double2 *>(out)[e] = make_double2(0.0, 0.0);
            __syncwarp();
            continue;
        }
        // ---- store A^{-1} column-major: Ainv[rhoinv[i]][rho[j]] = W[i][j], i.e. out[c][r] = W[rho[r]][rhoinv[c]]
        const int i0 = sh.rho[2 * lane], i1 = sh.rho[2 * lane + 1];
#pragma unroll 4
        for (int c = 0; c < n; ++c) {
            const double *col = &W[sh.rhoinv[c] * LD];
            reinterpret_cast<double2 *>(out + (size_t)c * n)[lane] = make_double2(col[i0], col[i1]);
        }
        __syncwarp(); // every lane is done with W before the next cell's assembly overwrites it
    }
}

// ============================================================================================================
// n = 64, TWO WARPS PER CELL with look-ahead: the production a1 + a2 kernel of the headline configuration.
// ============================================================================================================
// Same data layout and arithmetic as factor_wc_kernel. ncu on that kernel (profiles/r02_factor.md): a warp that
// issues a DMMA cannot issue anything else for ~15 cycles, so the rank-8 update of one warp takes 16 cycles per DMMA
// whatever else there is to overlap, and phase U was 40 % of a cell's latency. Here warp A runs the pivot chain and
// warp B the updates: after panel p is eliminated, A updates ONLY column block p + 1 and goes straight on to
// eliminate it, while B applies update p to the other six blocks -- the classic look-ahead of blocked LU. One CTA
// barrier per panel (A: Z(p) is in shared memory; B: update p - 1 is complete). The critical path of a cell is its
// 64 pivot steps plus eight one-block updates; six cells (twelve warps) per SM.
// PAIRED (production): B does not apply every panel's update to every block. Panels are taken in pairs and a block that
// is not needed soon receives both updates of a pair in ONE pass over its accumulator tiles (wc2_update_blocks16, four
// DMMAs per tile): 9 block passes per pair instead of 14 -- the accumulator tiles of phase U are 55 % of the kernel's
// shared-memory wavefronts, the resource it saturates. The schedule is written out in the kernel.
// Fragment rows: the two 8 x 8 tiles of a 16-row group take the even / the odd rows of the group, so a lane's two
// tiles are adjacent in a column and accumulators and A fragments move as 16-byte accesses (any permutation of the M
// dimension of a matrix product is free).
// Leading dimension 68 (= 4 mod 16: a column starts 8 banks after its neighbour) and the columns of a block taken in the
// order 0 2 1 3 4 6 5 7 by the eight lane groups (any permutation of the M dimension of a product is free): the two
// columns of a quarter-warp's 16-byte accumulator access are then 16 banks apart, and the four panel columns of a
// half-warp's B-fragment load 8 banks apart -- both conflict-free (LD = 72 made the second a two-way conflict, and
// shared-memory wavefronts are what this kernel saturates: ncu l1tex__data_pipe_lsu_wavefronts_mem_shared 73 %).
constexpr int WC2_LD = 68;
__device__ __forceinline__ int wc2_colmap(int lg) { return (lg & 4) | ((lg & 1) << 1) | ((lg >> 1) & 1); }

struct Wc2Shared {
    double W[64 * WC2_LD];         // [column][row], column-major working matrix
    double prow[2][FR_NB + 2];     // [step parity]: the pivot row of the current step as it stands, then 1 / pivot
    int rho[64], rhoinv[64];
    int cell, sing;
    unsigned flip;                 // which of the CTA's two warps runs the pivot chain (factor_wc2_kernel)
};

// Rank-8 update of column block Jb (8 columns) from the panel whose pivot rows are rk0 = R[lq], rk1 = R[4 + lq]:
// W[:, 8 Jb ..] += Z W_old[R, 8 Jb ..], Z = T[:, R] - I[:, R], evaluated TRANSPOSED so that a lane's two accumulators
// are adjacent rows of one column (one 16-byte access): D[i][j] += sum_k A[i][k] B[k][j] with
//   A[i][k] = W_old[R[k]][8 Jb + c(i)] (lane holds A[lg][lq]),  B[k][j] = T[8 I + j][R-column k]   (lane holds B[lq][lg]),
//   D[i][j] = W[8 I + j][8 Jb + c(i)]  (lane holds rows 8 I + 2 lq, + 1 of column 8 Jb + c(lg)), c = wc2_colmap.
// The "- I[:, R]" costs nothing: row r_b of the result is sum_k T[r_b][k] W_old[R[k]][c] WITHOUT its own old value, so
// the eight pivot rows of the block are zeroed (by the lanes that have just read them as A fragments) before the
// accumulators are loaded, and the B fragments are the eliminated panel as it stands in W.
template <int NBLK>
__device__ __forceinline__ void wc2_update_blocks(double *W, const int (&Jb)[NBLK], const double (&zf)[8][2], int rk0, int rk1,
                                                  int lq, int lg)
{
    constexpr int LD = WC2_LD;
    // A fragments of all the blocks first (then they are zeroed, see above): one pair of warp barriers for the lot, and
    // nothing but loads, DMMAs and stores of independent tiles afterwards
    const int cl = wc2_colmap(lg); // this lane group's column of a block
    double a0[NBLK], a1[NBLK];
#pragma unroll
    for (int i = 0; i < NBLK; ++i) {
        a0[i] = W[(8 * Jb[i] + cl) * LD + rk0];
        a1[i] = W[(8 * Jb[i] + cl) * LD + rk1];
    }
    __syncwarp();
#pragma unroll
    for (int i = 0; i < NBLK; ++i) {
        W[(8 * Jb[i] + cl) * LD + rk0] = 0.0;
        W[(8 * Jb[i] + cl) * LD + rk1] = 0.0;
    }
    __syncwarp();
#pragma unroll
    for (int i = 0; i < NBLK; ++i) {
        double2 *cp = reinterpret_cast<double2 *>(&W[(8 * Jb[i] + cl) * LD + 2 * lq]);
#pragma unroll
        for (int I = 0; I < 8; ++I) {
            double2 v = cp[4 * I];
            dmma884(v.x, v.y, a0[i], zf[I][0]);
            dmma884(v.x, v.y, a1[i], zf[I][1]);
            cp[4 * I] = v;
        }
    }
}

// The updates of TWO consecutive panels q, p = q + 1 applied to column blocks Jb in one pass over their accumulators
// (a rank-16 update: four DMMAs per tile instead of two passes of two): with Tq' = block q AFTER update p has been
// applied to it (pivot rows R_p zeroed, += T_p T_q[R_p, :]) the two updates compose to
//   W[:, c] <- W[:, c] (rows R_q and R_p zeroed) + Tq' W_old[R_q, c] + T_p W_old[R_p, c],
// with the ORIGINAL pivot-row entries of both panels as A fragments. zq, zp: B fragments of blocks q (updated) and p;
// rq0/rq1, rp0/rp1: this lane's pivot rows of the two panels. Two tiles at a time: eight DMMAs, four per accumulator.
template <int NBLK>
__device__ __forceinline__ void wc2_update_blocks16(double *W, const int (&Jb)[NBLK], const double (&zq)[8][2], const double (&zp)[8][2],
                                                    int rq0, int rq1, int rp0, int rp1, int lq, int lg)
{
    constexpr int LD = WC2_LD;
    const int cl = wc2_colmap(lg);
    double aq0[NBLK], aq1[NBLK], ap0[NBLK], ap1[NBLK];
#pragma unroll
    for (int i = 0; i < NBLK; ++i) {
        const double *col = &W[(8 * Jb[i] + cl) * LD];
        aq0[i] = col[rq0];
        aq1[i] = col[rq1];
        ap0[i] = col[rp0];
        ap1[i] = col[rp1];
    }
    __syncwarp();
#pragma unroll
    for (int i = 0; i < NBLK; ++i) {
        double *col = &W[(8 * Jb[i] + cl) * LD];
        col[rq0] = 0.0;
        col[rq1] = 0.0;
        col[rp0] = 0.0;
        col[rp1] = 0.0;
    }
    __syncwarp();
#pragma unroll
    for (int i = 0; i < NBLK; ++i) {
        double2 *cp = reinterpret_cast<double2 *>(&W[(8 * Jb[i] + cl) * LD + 2 * lq]);
#pragma unroll
        for (int I = 0; I < 8; I += 2) {
            double2 v0 = cp[4 * I], v1 = cp[4 * I + 4];
            dmma884(v0.x, v0.y, aq0[i], zq[I][0]);
            dmma884(v1.x, v1.y, aq0[i], zq[I + 1][0]);
            dmma884(v0.x, v0.y, aq1[i], zq[I][1]);
            dmma884(v1.x, v1.y, aq1[i], zq[I + 1][1]);
            dmma884(v0.x, v0.y, ap0[i], zp[I][0]);
            dmma884(v1.x, v1.y, ap0[i], zp[I + 1][0]);
            dmma884(v0.x, v0.y, ap1[i], zp[I][1]);
            dmma884(v1.x, v1.y, ap1[i], zp[I + 1][1]);
            cp[4 * I] = v0;
            cp[4 * I + 4] = v1;
        }
    }
}

// B fragments of the eliminated panel in column block `blk`: T[8 I + lg][block column 4 h + lq]
__device__ __forceinline__ void wc2_load_zf(const double *W, int blk, double (&zf)[8][2], int lq, int lg)
{
    constexpr int LD = WC2_LD;
#pragma unroll
    for (int I = 0; I < 8; ++I) {
        zf[I][0] = W[(FR_NB * blk + lq) * LD + 8 * I + lg];
        zf[I][1] = W[(FR_NB * blk + 4 + lq) * LD + 8 * I + lg];
    }
}

// One pivot step (column b of the panel) of warp A: rows {2 lane, 2 lane + 1} as two row vectors in registers.
// 8-byte shared-memory load the compiler may not fuse with its neighbour into a 16-byte one (a 16-byte broadcast
// load costs 2.5 wavefronts, two 8-byte ones 2)
__device__ __forceinline__ double lds_f64(const double *p)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(smem_u32(p)));
    return v;
}

struct WcPanel {
    double t0[FR_NB], t1[FR_NB]; // row 2 lane, row 2 lane + 1
    unsigned m0, m1;             // 0x7fffffff while the row is unused, 0 once it has been a pivot row
};

// FAST = true is the optimistic form the kernel runs first: no branch (the eight steps of a panel are ONE basic block, so
// the scheduler overlaps the tail of a step with the reduction of the next), a tie of the high key words is only
// RECORDED, and the one column the next pivot decision depends on travels by shuffle instead of through shared memory.
// If a panel recorded a tie it is reloaded and eliminated again with FAST = false, which resolves ties exactly (low key
// words, then the lowest row: the first maximal |entry|, as LAPACK's idamax). Same arithmetic in both forms.
template <int b, bool FAST>
__device__ __forceinline__ void wc2_pivot_step(WcPanel &R, double *prow_base, int &myr, int lane, unsigned &bad, unsigned &tie)
{
    constexpr unsigned FULL = 0xffffffffu;
    // |entry| of the unused rows as integer keys (non-negative doubles order like their bit patterns); the low words
    // need no mask: a used row can only win with a zero high word, and that is flagged as singular anyway
    const unsigned h0 = (unsigned)__double2hiint(R.t0[b]) & R.m0, h1 = (unsigned)__double2hiint(R.t1[b]) & R.m1;
    const unsigned l0 = (unsigned)__double2loint(R.t0[b]), l1 = (unsigned)__double2loint(R.t1[b]);
    const bool e1 = h1 > h0 || (h1 == h0 && l1 > l0); // the lane's own winner: the lower row on a tie
    const unsigned khi = e1 ? h1 : h0;
    const unsigned mhi = __reduce_max_sync(FULL, khi);
    const unsigned eball = __ballot_sync(FULL, e1);
    const double linv = rcp_nr(e1 ? R.t1[b] : R.t0[b]); // in the shadow of the reduction: 1 / (the lane's candidate)
    unsigned ball = __ballot_sync(FULL, khi == mhi);
    if (FAST) {
        tie |= ball & (ball - 1u); // more than one lane holds the maximal high word
    } else if (__popc(ball) != 1) { // ties in the high word: low words, then the lowest lane (= the lowest row)
        const unsigned klo = e1 ? l1 : l0;
        const bool cand = khi == mhi;
        const unsigned mlo = __reduce_max_sync(FULL, cand ? klo : 0u);
        ball = __ballot_sync(FULL, cand && klo == mlo);
    }
    const int src = (__ffs(ball) - 1) & 31;
    bad |= (mhi - 1u >= 0x7fefffffu) ? 1u : 0u; // pivot with a zero high word (0 or < 2^-1042), inf, NaN, or no unused row left
    const int esrc = (eball >> src) & 1;
    const bool p0 = lane == src && esrc == 0, p1 = lane == src && esrc != 0;
    const double f0 = R.t0[b], f1 = R.t1[b];
    double ls;
    if (FAST) { // 1 / pivot and, below, column b + 1 of the pivot row by shuffle: nothing else is on the critical path
        ls = __shfl_sync(FULL, linv, src);
        if (b + 1 < FR_NB) {
            const double xn = __shfl_sync(FULL, esrc ? R.t1[b + 1] : R.t0[b + 1], src) * ls;
            const double u0 = fma(-f0, xn, R.t0[b + 1]), u1 = fma(-f1, xn, R.t1[b + 1]);
            R.t0[b + 1] = p0 ? xn : u0;
            R.t1[b + 1] = p1 ? xn : u1;
        }
    }
    double *pr = prow_base + (b & 1) * (FR_NB + 2);
    // the winner publishes its row as it stands (and 1 / pivot for the exact form)
    if (p0) {
#pragma unroll
        for (int c = 0; c < FR_NB / 2; ++c) reinterpret_cast<double2 *>(pr)[c] = make_double2(R.t0[2 * c], R.t0[2 * c + 1]);
        if (!FAST) pr[FR_NB] = linv;
    }
    if (p1) {
#pragma unroll
        for (int c = 0; c < FR_NB / 2; ++c) reinterpret_cast<double2 *>(pr)[c] = make_double2(R.t1[2 * c], R.t1[2 * c + 1]);
        if (!FAST) pr[FR_NB] = linv;
    }
    __syncwarp(); // (two buffers alternate: no second barrier needed)
    if (!FAST) ls = pr[FR_NB];
    double sp[FR_NB]; // pivot row / pivot; column b holds 1 / pivot. 8-byte broadcast loads (one wavefront each) of the
                      // columns that are still needed: shared-memory wavefronts are the resource this kernel saturates
#pragma unroll
    for (int c = 0; c < FR_NB; ++c) {
        if (c == b) sp[c] = ls;
        else if (FAST && c == b + 1) sp[c] = 0.0; // (unused)
        else sp[c] = lds_f64(pr + c) * ls;
    }
#pragma unroll
    for (int c = 0; c < FR_NB; ++c) {
        if (FAST && c == b + 1) continue; // done above (the published row still holds its old value of that column)
        R.t0[c] = (c == b) ? -f0 * ls : fma(-f0, sp[c], R.t0[c]);
        R.t1[c] = (c == b) ? -f1 * ls : fma(-f1, sp[c], R.t1[c]);
    }
    // the pivot row becomes itself / pivot (predicated moves: a divergent branch would add its resolve and
    // reconvergence latency to the chain)
    if (p0) {
#pragma unroll
        for (int c = 0; c < FR_NB; ++c)
            if (!(FAST && c == b + 1)) R.t0[c] = sp[c];
        R.m0 = 0u;
    }
    if (p1) {
#pragma unroll
        for (int c = 0; c < FR_NB; ++c)
            if (!(FAST && c == b + 1)) R.t1[c] = sp[c];
        R.m1 = 0u;
    }
    if (lane == b) myr = 2 * src + esrc; // lane b keeps pivot row b: stored once per panel (wc2_panel)
}

template <bool FAST>
__device__ __forceinline__ void wc2_panel(WcPanel &R, double *prow, int *rho, int *rhoinv, int col0, int lane, unsigned &bad,
                                          unsigned &tie)
{
    int myr = 0;
    wc2_pivot_step<0, FAST>(R, prow, myr, lane, bad, tie);
    wc2_pivot_step<1, FAST>(R, prow, myr, lane, bad, tie);
    wc2_pivot_step<2, FAST>(R, prow, myr, lane, bad, tie);
    wc2_pivot_step<3, FAST>(R, prow, myr, lane, bad, tie);
    wc2_pivot_step<4, FAST>(R, prow, myr, lane, bad, tie);
    wc2_pivot_step<5, FAST>(R, prow, myr, lane, bad, tie);
    wc2_pivot_step<6, FAST>(R, prow, myr, lane, bad, tie);
    wc2_pivot_step<7, FAST>(R, prow, myr, lane, bad, tie);
    if (lane < FR_NB) { // the panel's pivot rows, once per panel
        rho[col0 + lane] = myr;
        rhoinv[myr] = col0 + lane;
    }
}

template <bool DUMP, bool PAIRED>
__global__ void __launch_bounds__(64)
factor_wc2_kernel(ProblemView P, double *__restrict__ Minv, int *info, int *next_cell, double *__restrict__ dumpA, int dump_cell,
                  int /* unused */)
{
    constexpr int n = 64, LD = WC2_LD, NPANEL = n / FR_NB;
    extern __shared__ __align__(16) unsigned char wc_smem[];
    Wc2Shared &sh = *reinterpret_cast<Wc2Shared *>(wc_smem);
    double *W = sh.W;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, lq = lane & 3, lg = lane >> 2;
    // Role: warp A runs the pivot chain, warp B the updates. The two warps of a CTA normally sit on neighbouring SM
    // sub-partitions (warp slots 2 k, 2 k + 1: measured); alternating the roles with bit 2 of the slot puts the six A
    // warps of an SM on all four schedulers instead of two. %warpid is only a scheduling HINT here: thread 0 reads it
    // once and the roles follow from the warp index within the CTA, so the two warps take complementary roles wherever
    // the hardware placed them (the PTX ISA makes no promise about slot numbers).
    if (threadIdx.x == 0) {
        unsigned slot;
        asm volatile("mov.u32 %0, %%warpid;" : "=r"(slot));
        sh.flip = (slot ^ (slot >> 2)) & 1u;
    }
    __syncthreads();
    const bool roleA = (((unsigned)w ^ sh.flip) & 1u) == 0u;

    for (;;) {
        if (threadIdx.x == 0) { sh.cell = DUMP ? dump_cell : atomicAdd(next_cell, 1); sh.sing = 0; }
        __syncthreads();
        const int cell = sh.cell;
        if (cell >= P.J) break;
        assemble_rows2(P, cell, lane, W, LD, w, 2);
        __syncthreads();
        if (DUMP) { // the assembled tile of the production kernel, row-major, for the bit-exactness test
            for (int e = threadIdx.x; e < n * n; e += 64) dumpA[e] = W[(e & 63) * LD + (e >> 6)];
            break;
        }

        WcPanel R;
        R.m0 = R.m1 = 0x7fffffffu;
        bool singular = false;
        for (int pnl = 0; pnl < NPANEL; ++pnl) {
            if (roleA) {
                // ================= phase P (warp A): the 64 x 8 panel in registers, two rows per lane =================
                double *Wp = &W[(FR_NB * pnl) * LD + 2 * lane];
#pragma unroll
                for (int c = 0; c < FR_NB; ++c) {
                    const double2 v = *reinterpret_cast<const double2 *>(Wp + c * LD);
                    R.t0[c] = v.x;
                    R.t1[c] = v.y;
                }
                unsigned bad = 0u, tie = 0u;
                const unsigned m0_in = R.m0, m1_in = R.m1;
                wc2_panel<true>(R, &sh.prow[0][0], sh.rho, sh.rhoinv, FR_NB * pnl, lane, bad, tie);
                if (tie) { // warp-uniform and rare: the panel again, from shared memory, with exact tie resolution
#pragma unroll
                    for (int c = 0; c < FR_NB; ++c) {
                        const double2 v = *reinterpret_cast<const double2 *>(Wp + c * LD);
                        R.t0[c] = v.x;
                        R.t1[c] = v.y;
                    }
                    R.m0 = m0_in;
                    R.m1 = m1_in;
                    bad = 0u;
                    __syncwarp();
                    wc2_panel<false>(R, &sh.prow[0][0], sh.rho, sh.rhoinv, FR_NB * pnl, lane, bad, tie);
                }
                if (bad && lane == 0) sh.sing = 1;
                // the eliminated panel (its columns now hold T e_r) back in place
#pragma unroll
                for (int c = 0; c < FR_NB; ++c) *reinterpret_cast<double2 *>(Wp + c * LD) = make_double2(R.t0[c], R.t1[c]);
            }
            __syncthreads(); // barrier p: Z(p), R(p) visible to B; B has completed update p - 1
            if (sh.sing) { singular = true; break; } // CTA-uniform

            // ================= phase U =================
            const int rk0 = sh.rho[FR_NB * pnl + lq], rk1 = sh.rho[FR_NB * pnl + 4 + lq];
            if (PAIRED) {
                // Panels are paired (q, p = q + 1), q even, and a block that is not needed soon receives the two updates of
                // a pair in ONE pass over its accumulators (wc2_update_blocks16): 9 block passes per pair instead of 14,
                // and the accumulator tiles are what saturates the shared-memory pipe. Who needs what, and when:
                //   A after barrier p': update p' on block p' + 1 (the look-ahead), which therefore must be current
                //     through p' - 1 at that barrier;
                //   B after an even barrier q: the LATE blocks of the pair before (two of its five "other" blocks), then
                //     update q on block q + 2 (A's look-ahead after barrier p applies update p to it);
                //   B after an odd barrier p: update p on block q (which makes Tq'), then the pair on its three EARLY other
                //     blocks p + 2, p + 3, p + 4 (mod 8) -- p + 2 is the one A needs after the next barrier.
                // The other blocks of a pair are p + 2 .. p + 6 (mod 8): everything but q, p and p + 1. The last pair has
                // no p + 1: its six other blocks are shared out between the two warps after the loop.
                const int q = pnl & ~1, pp = q + 1;
                if (roleA) {
                    if (pnl + 1 < NPANEL) {
                        double zf[8][2];
                        wc2_load_zf(W, pnl, zf, lq, lg);
                        const int jb[1] = {pnl + 1};
                        wc2_update_blocks<1>(W, jb, zf, rk0, rk1, lq, lg);
                        __syncwarp();
                    }
                } else if ((pnl & 1) == 0) {
                    if (q >= 2) { // the late blocks of pair (q - 2, q - 1)
                        double zq[8][2], zp[8][2];
                        wc2_load_zf(W, q - 2, zq, lq, lg);
                        wc2_load_zf(W, q - 1, zp, lq, lg);
                        const int jb[2] = {(q + 4) & 7, (q + 5) & 7}; // (p' + 5, p' + 6 with p' = q - 1)
                        wc2_update_blocks16<2>(W, jb, zq, zp, sh.rho[FR_NB * (q - 2) + lq], sh.rho[FR_NB * (q - 2) + 4 + lq],
                                               sh.rho[FR_NB * (q - 1) + lq], sh.rho[FR_NB * (q - 1) + 4 + lq], lq, lg);
                        __syncwarp();
                    }
                    if (q + 2 < NPANEL) {
                        double zf[8][2];
                        wc2_load_zf(W, q, zf, lq, lg);
                        const int jb[1] = {q + 2};
                        wc2_update_blocks<1>(W, jb, zf, rk0, rk1, lq, lg);
                    }
                } else {
                    double zp[8][2];
                    wc2_load_zf(W, pp, zp, lq, lg);
                    {
                        const int jb[1] = {q};
                        wc2_update_blocks<1>(W, jb, zp, rk0, rk1, lq, lg); // block q becomes Tq'
                        __syncwarp();
                    }
                    if (pp + 1 < NPANEL) {
                        double zq[8][2];
                        wc2_load_zf(W, q, zq, lq, lg);
                        const int jb[3] = {(pp + 2) & 7, (pp + 3) & 7, (pp + 4) & 7};
                        wc2_update_blocks16<3>(W, jb, zq, zp, sh.rho[FR_NB * q + lq], sh.rho[FR_NB * q + 4 + lq], rk0, rk1, lq, lg);
                    }
                }
                continue;
            }
            double zf[8][2]; // B fragments: T[8 I + lg][panel column 4 h + lq]
            wc2_load_zf(W, pnl, zf, lq, lg);
            if (pnl + 1 < NPANEL) { // A: the next panel's block only (then straight on to eliminate it); B: the rest
                if (roleA) {
                    const int jb[1] = {pnl + 1};
                    wc2_update_blocks<1>(W, jb, zf, rk0, rk1, lq, lg);
                    __syncwarp();
                } else {
                    int jb[6];
#pragma unroll
                    for (int i = 0; i < 6; ++i) jb[i] = i < pnl ? i : i + 2;
                    wc2_update_blocks<6>(W, jb, zf, rk0, rk1, lq, lg);
                }
            } else { // last panel: blocks 0..6 shared out
                if (w == 0) {
                    const int jb[4] = {0, 2, 4, 6};
                    wc2_update_blocks<4>(W, jb, zf, rk0, rk1, lq, lg);
                } else {
                    const int jb[3] = {1, 3, 5};
                    wc2_update_blocks<3>(W, jb, zf, rk0, rk1, lq, lg);
                }
            }
        }
        __syncthreads(); // update 7 complete (PAIRED: block 6 has received update 7)
        if (PAIRED && !singular) { // the last pair (6, 7) on its six other blocks, three per warp
            double zq[8][2], zp[8][2];
            wc2_load_zf(W, 6, zq, lq, lg);
            wc2_load_zf(W, 7, zp, lq, lg);
            const int jb[3] = {3 * w, 3 * w + 1, 3 * w + 2};
            wc2_update_blocks16<3>(W, jb, zq, zp, sh.rho[48 + lq], sh.rho[52 + lq], sh.rho[56 + lq], sh.rho[60 + lq], lq, lg);
            __syncthreads();
        }

        double *out = Minv + (size_t)cell * n * n;
        if (singular) {
            if (threadIdx.x == 0) atomicMin(info, cell + 1);
            for (int e = threadIdx.x; e < n * n / 2; e += 64) reinterpret_cast<double2 *>(out)[e] = make_double2(0.0, 0.0);
            __syncthreads();
            continue;
        }
        // ---- store A^{-1} column-major: Ainv[rhoinv[i]][rho[j]] = W[i][j]. Column j of W goes to column rho[j] with its
        // rows scattered by rhoinv: conflict-free 16-byte shared-memory reads, and the 64 eight-byte stores of a column
        // fill one 512-byte line between them (the L2 merges them: DRAM traffic stays at the 2.09 GB of the result)
        const int r0 = sh.rhoinv[2 * lane], r1 = sh.rhoinv[2 * lane + 1];
#pragma unroll 4
        for (int j = w; j < n; j += 2) {
            const double2 v = *reinterpret_cast<const double2 *>(&W[j * LD + 2 * lane]);
            double *col = out + (size_t)sh.rho[j] * n;
            col[r0] = v.x;
            col[r1] = v.y;
        }
        __syncthreads(); // everybody is done with W and sh.cell before the next cell
    }
}

// ============================================================================================================
// n = 128: one CTA (one SM) per cell -- the production a1 + a2 kernel of config 3 and of the paper's S16 Table-2 problem.
// ============================================================================================================
// The design of factor_wc2_kernel at the size where one working matrix (132 KB) fills an SM: column-major W in shared
// memory (leading dimension 132 = 4 mod 16, columns of a block in the order 0 2 1 3 4 6 5 7: conflict-free), panels
// of 8 columns, rank-8 updates as transposed m8n8k4 DMMAs with the pivot rows zeroed instead of Z = T - I formed,
// look-ahead, optimistic branch-free panel with an exact replay on a tie of high key words. What differs:
//   * FOUR pivot warps, one row per lane (a single warp with four rows per lane would issue ~200 instructions per
//     pivot step in order). Per step each warp finds its own first maximal |entry| (redux + ballot), its winner
//     publishes {64-bit key, lane, row as it stands with 1 / candidate in the step's column} in a slot (five 16-byte
//     stores: the barrier that follows waits for the stores in flight), one named barrier over the 128 pivot
//     threads, lane ww reads warp ww's key and the arg-max over the warps is a second redux + ballot (the lowest warp
//     = the lowest row wins; the exact replay compares the 64-bit keys one after the other), and every lane eliminates
//     its row. Two slot sets alternate, so one barrier per step; the pivot rows of a panel are stored once per panel.
//   * Look-ahead: the pivot warps update the next panel's block -- warp w the row tiles 4 w .. 4 w + 3, which are the
//     rows it then loads for the next panel, so nothing but one pivot-warp barrier (pivot rows read before anybody
//     stores) separates update and panel -- while the four update warps apply the update to the other 14 blocks.
constexpr int P128_LD = 132, P128_THREADS = 256, P128_AW = 4;

struct alignas(16) P128Slot { // five 16-byte stores per candidate: a barrier waits for the stores in flight
    double row[FR_NB];        // the candidate's panel row as it stands; column b of step b holds 1 / candidate instead
    unsigned long long key;   // |candidate| as an integer key (0: this warp has no unused row)
    int lane;                 // lane of the candidate; bit 8: more lanes of the warp share its high key word
    int pad;
};

struct P128Shared {
    double W[128 * P128_LD];          // [column][row]
    P128Slot slot[2][P128_AW];        // [step parity][pivot warp]
    int rho[128], rhoinv[128];
    int cell, sing, tie;
};

// named barrier over the AW pivot warps of a CTA
template <int AW> __device__ __forceinline__ void pivot_warps_bar() { asm volatile("bar.sync 1, %0;" ::"n"(32 * AW) : "memory"); }
__device__ __forceinline__ void p128_bar_pivot() { pivot_warps_bar<P128_AW>(); }

// One pivot step of a panel shared by AW pivot warps, one row per lane (row 32 w + lane). slots: [2][AW].
template <int b, bool FAST, int AW>
__device__ __forceinline__ void pw_pivot_step(double (&t)[FR_NB], unsigned &m, P128Slot *slots, int &myr, int w, int lane,
                                              unsigned &bad, unsigned &tie)
{
    constexpr unsigned FULL = 0xffffffffu;
    const unsigned h = (unsigned)__double2hiint(t[b]) & m, l = (unsigned)__double2loint(t[b]);
    const unsigned mh = __reduce_max_sync(FULL, h);
    const double linv = rcp_nr(t[b]); // in the shadow of the reduction
    unsigned ball = __ballot_sync(FULL, h == mh);
    const unsigned tied = ball & (ball - 1u); // more than one lane of this warp holds its maximal high word
    if (!FAST && tied) { // low words, then the lowest lane (= the lowest row)
        const bool cand = h == mh;
        const unsigned ml = __reduce_max_sync(FULL, cand ? l : 0u);
        ball = __ballot_sync(FULL, cand && l == ml);
    }
    const int src = (__ffs(ball) - 1) & 31;
    P128Slot *mine = &slots[(b & 1) * AW + w];
    if (lane == src) { // this warp's candidate: key, row as it stands, 1 / candidate
#pragma unroll
        for (int c = 0; c < FR_NB / 2; ++c)
            reinterpret_cast<double2 *>(mine->row)[c] = make_double2(2 * c == b ? linv : t[2 * c], 2 * c + 1 == b ? linv : t[2 * c + 1]);
        // h == 0: no unused row here (loses, or the cell is singular)
        *reinterpret_cast<uint4 *>(&mine->key) = make_uint4(l, h, (unsigned)lane | (tied ? 0x100u : 0u), 0u);
    }
    pivot_warps_bar<AW>();
    int gw, lwv;
    if (FAST) {
        // the AW candidates, one per lane: high key word and lane word of slot `lane` in one 16-byte load, arg-max by
        // redux + ballot (the lowest warp = the lowest row wins). Only high words are compared here: two warps with the
        // same maximal high word, or a winner whose warp recorded a tie of its own, mean "replay the panel exactly"
        // (most warps tie all the time on the identical entries -dx K w / 4 of Eq. 10, far below the pivot: that is
        // why a warp's own tie counts only when its high word is the winning one)
        uint4 v = make_uint4(0u, 0u, 0u, 0u);
        if (lane < AW) v = *reinterpret_cast<const uint4 *>(&slots[(b & 1) * AW + lane].key);
        const unsigned mh2 = __reduce_max_sync(FULL, v.y);
        const bool top = lane < AW && v.y == mh2;
        const unsigned ball2 = __ballot_sync(FULL, top);
        const unsigned tb = __ballot_sync(FULL, top && (v.z & 0x100u));
        gw = (__ffs(ball2) - 1) & 31;
        tie |= ((ball2 & (ball2 - 1u)) | tb) ? 1u : 0u;
        lwv = __shfl_sync(FULL, (int)v.z, gw);
        bad |= (mh2 - 1u >= 0x7fefffffu) ? 1u : 0u; // zero / denormal / inf / NaN pivot
    } else {
        // exact form: 64-bit keys; key and lane word of a slot in one 16-byte broadcast load
        unsigned long long kk[AW];
        int lw4[AW];
#pragma unroll
        for (int ww = 0; ww < AW; ++ww) {
            const uint4 v = *reinterpret_cast<const uint4 *>(&slots[(b & 1) * AW + ww].key);
            kk[ww] = ((unsigned long long)v.y << 32) | v.x;
            lw4[ww] = (int)v.z;
        }
        unsigned long long kmax = kk[0];
        gw = 0;
        lwv = lw4[0];
#pragma unroll
        for (int ww = 1; ww < AW; ++ww) // strict >: a tie goes to the lower warp, i.e. the lower row
            if (kk[ww] > kmax) { kmax = kk[ww]; gw = ww; lwv = lw4[ww]; }
        bad |= ((unsigned)(kmax >> 32) - 1u >= 0x7fefffffu) ? 1u : 0u; // zero / denormal / inf / NaN pivot
    }
    const P128Slot *win = &slots[(b & 1) * AW + gw];
    double sp[FR_NB]; // pivot row / pivot; column b holds 1 / pivot
#pragma unroll
    for (int c = 0; c < FR_NB / 2; ++c) {
        const double2 v = reinterpret_cast<const double2 *>(win->row)[c];
        sp[2 * c] = v.x;
        sp[2 * c + 1] = v.y;
    }
    const double ls = sp[b];
    const int lw = lwv & 31;
#pragma unroll
    for (int c = 0; c < FR_NB; ++c)
        if (c != b) sp[c] *= ls;
    const bool is_p = gw == w && lane == lw;
    const double f = t[b];
#pragma unroll
    for (int c = 0; c < FR_NB; ++c) {
        const double u = (c == b) ? -f * ls : fma(-f, sp[c], t[c]);
        t[c] = is_p ? sp[c] : u;
    }
    m = is_p ? 0u : m;
    if (lane == b) myr = 32 * gw + lw; // lane b keeps pivot row b: stored once per panel (pw_panel)
}

template <bool FAST, int AW>
__device__ __forceinline__ void pw_panel(double (&t)[FR_NB], unsigned &m, P128Slot *slots, int *rho, int *rhoinv, int w, int lane,
                                         int col0, unsigned &bad, unsigned &tie)
{
    int myr = 0;
    pw_pivot_step<0, FAST, AW>(t, m, slots, myr, w, lane, bad, tie);
    pw_pivot_step<1, FAST, AW>(t, m, slots, myr, w, lane, bad, tie);
    pw_pivot_step<2, FAST, AW>(t, m, slots, myr, w, lane, bad, tie);
    pw_pivot_step<3, FAST, AW>(t, m, slots, myr, w, lane, bad, tie);
    pw_pivot_step<4, FAST, AW>(t, m, slots, myr, w, lane, bad, tie);
    pw_pivot_step<5, FAST, AW>(t, m, slots, myr, w, lane, bad, tie);
    pw_pivot_step<6, FAST, AW>(t, m, slots, myr, w, lane, bad, tie);
    pw_pivot_step<7, FAST, AW>(t, m, slots, myr, w, lane, bad, tie);
    if (w == 0 && lane < FR_NB) { // the panel's pivot rows (stores kept out of the steps: the step barrier waits for them)
        rho[col0 + lane] = myr;
        rhoinv[myr] = col0 + lane;
    }
}

// one whole column block by one warp (see wc2_update_blocks): pivot rows read, zeroed, 16 row tiles updated
__device__ __forceinline__ void p128_update_block(double *W, int Jb, const double (&zf)[16][2], int rk0, int rk1, int lq, int lg)
{
    constexpr int LD = P128_LD;
    const int cl = wc2_colmap(lg);
    double *a0p = &W[(8 * Jb + cl) * LD + rk0], *a1p = &W[(8 * Jb + cl) * LD + rk1];
    const double a0 = *a0p, a1 = *a1p;
    __syncwarp();
    *a0p = 0.0;
    *a1p = 0.0;
    __syncwarp();
    double2 *cp = reinterpret_cast<double2 *>(&W[(8 * Jb + cl) * LD + 2 * lq]);
#pragma unroll
    for (int I = 0; I < 16; ++I) {
        double2 v = cp[4 * I];
        dmma884(v.x, v.y, a0, zf[I][0]);
        dmma884(v.x, v.y, a1, zf[I][1]);
        cp[4 * I] = v;
    }
}

template <bool DUMP>
__global__ void __launch_bounds__(P128_THREADS, 1)
factor_p128_kernel(ProblemView P, double *__restrict__ Minv, int *info, int *next_cell, double *__restrict__ dumpA, int dump_cell)
{
    constexpr int n = 128, LD = P128_LD, NPANEL = n / FR_NB;
    extern __shared__ __align__(16) unsigned char p128_smem[];
    P128Shared &sh = *reinterpret_cast<P128Shared *>(p128_smem);
    double *W = sh.W;
    const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5, lq = lane & 3, lg = lane >> 2;
    // pivot warps on two of the SM's four sub-partitions (physical warps 0, 1, 4, 5), update warps on the other two: a
    // DFMA of the pivot chain then never queues behind an update warp's DMMA. w = index within the role (+ 4: update).
    const bool roleA = (wp & 2) == 0;
    const int w = ((wp & 1) | ((wp >> 2) << 1)) + (roleA ? 0 : P128_AW);
    for (;;) {
        if (threadIdx.x == 0) { sh.cell = DUMP ? dump_cell : atomicAdd(next_cell, 1); sh.sing = 0; sh.tie = 0; }
        __syncthreads();
        const int cell = sh.cell;
        if (cell >= P.J) break;
        assemble_rows2(P, cell, lane, W, LD, w >> 1, 4, 64 * (w & 1), 128);
        __syncthreads();
        if (DUMP) { // the assembled tile of the production kernel, row-major, for the bit-exactness test
            for (int e = threadIdx.x; e < n * n; e += P128_THREADS) dumpA[e] = W[(e & 127) * LD + (e >> 7)];
            break;
        }

        double t[FR_NB];            // pivot warps: row 32 w + lane of the current panel
        unsigned m = 0x7fffffffu;   // 0 once that row has been a pivot row
        bool singular = false;
        for (int pnl = 0; pnl < NPANEL; ++pnl) {
            if (roleA) {
                const int r = 32 * w + lane;
                double *Wp = &W[(FR_NB * pnl) * LD + r];
#pragma unroll
                for (int c = 0; c < FR_NB; ++c) t[c] = Wp[c * LD];
                unsigned bad = 0u, tie = 0u;
                const unsigned m_in = m;
                pw_panel<true, P128_AW>(t, m, &sh.slot[0][0], sh.rho, sh.rhoinv, w, lane, FR_NB * pnl, bad, tie);
                if (tie) sh.tie = 1;
                p128_bar_pivot();
                const bool redo = sh.tie != 0;
                p128_bar_pivot();
                if (redo) { // pivot-warp-uniform and rare: the panel again, from shared memory, ties resolved exactly
                    if (threadIdx.x == 0) sh.tie = 0;
#pragma unroll
                    for (int c = 0; c < FR_NB; ++c) t[c] = Wp[c * LD];
                    m = m_in;
                    bad = 0u;
                    pw_panel<false, P128_AW>(t, m, &sh.slot[0][0], sh.rho, sh.rhoinv, w, lane, FR_NB * pnl, bad, tie);
                }
                if (bad && threadIdx.x == 0) sh.sing = 1;
#pragma unroll
                for (int c = 0; c < FR_NB; ++c) Wp[c * LD] = t[c]; // the eliminated panel (T e_r) back in place
            }
            __syncthreads(); // barrier p: T(p), R(p) visible to everybody; update p - 1 is complete
            if (sh.sing) { singular = true; break; } // CTA-uniform

            // ================= phase U: rank-8 update of the other 120 columns =================
            const int rk0 = sh.rho[FR_NB * pnl + lq], rk1 = sh.rho[FR_NB * pnl + 4 + lq];
            if (pnl + 1 < NPANEL && roleA) {
                // look-ahead: the next panel's block, pivot warp w its own 32 rows (row tiles 4 w .. 4 w + 3), on the critical
                // path of the cell: only the B fragments of those four tiles are loaded, all loads before the DMMAs, and
                // the two dependent DMMAs of a tile are four issue slots apart. Z = T - I explicitly (zeroing the pivot
                // rows would cost a second pivot-warp barrier).
                const int Jb = pnl + 1, cl = wc2_colmap(lg);
                const double a0 = W[(8 * Jb + cl) * LD + rk0], a1 = W[(8 * Jb + cl) * LD + rk1];
                double z0[4], z1[4];
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const int row = 8 * (4 * w + i) + lg;
                    z0[i] = W[(FR_NB * pnl + lq) * LD + row] - (rk0 == row ? 1.0 : 0.0);
                    z1[i] = W[(FR_NB * pnl + 4 + lq) * LD + row] - (rk1 == row ? 1.0 : 0.0);
                }
                p128_bar_pivot(); // every pivot warp has read the pivot rows of the block
                double2 *cp = reinterpret_cast<double2 *>(&W[(8 * Jb + cl) * LD + 2 * lq + 32 * w]);
                double2 v[4];
#pragma unroll
                for (int i = 0; i < 4; ++i) v[i] = cp[4 * i];
#pragma unroll
                for (int i = 0; i < 4; ++i) dmma884(v[i].x, v[i].y, a0, z0[i]);
#pragma unroll
                for (int i = 0; i < 4; ++i) dmma884(v[i].x, v[i].y, a1, z1[i]);
#pragma unroll
                for (int i = 0; i < 4; ++i) cp[4 * i] = v[i];
                __syncwarp();
                continue;
            }
            double zf[16][2]; // B fragments: T[8 I + lg][panel column 4 h + lq]
#pragma unroll
            for (int I = 0; I < 16; ++I) {
                zf[I][0] = W[(FR_NB * pnl + lq) * LD + 8 * I + lg];
                zf[I][1] = W[(FR_NB * pnl + 4 + lq) * LD + 8 * I + lg];
            }
            if (pnl + 1 < NPANEL) {
                for (int Jb = w - P128_AW; Jb < NPANEL; Jb += P128_THREADS / 32 - P128_AW)
                    if (Jb != pnl && Jb != pnl + 1) p128_update_block(W, Jb, zf, rk0, rk1, lq, lg);
            } else { // last panel: the other 15 blocks shared out over all eight warps
                for (int Jb = w; Jb < NPANEL - 1; Jb += P128_THREADS / 32) p128_update_block(W, Jb, zf, rk0, rk1, lq, lg);
            }
        }
        __syncthreads(); // the last update is complete

        double *out = Minv + (size_t)cell * n * n;
        if (singular) {
            if (threadIdx.x == 0) atomicMin(info, cell + 1);
            for (int e = threadIdx.x; e < n * n / 2; e += P128_THREADS) reinterpret_cast<double2 *>(out)[e] = make_double2(0.0, 0.0);
            __syncthreads();
            continue;
        }
        // ---- store A^{-1} column-major: Ainv[rhoinv[i]][rho[j]] = W[i][j] (rows scattered on the way out, see wc2)
        int ro[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) ro[q] = sh.rhoinv[64 * (q >> 1) + 2 * lane + (q & 1)];
        for (int j = w; j < n; j += P128_THREADS / 32) {
            const double2 v0 = *reinterpret_cast<const double2 *>(&W[j * LD + 2 * lane]);
            const double2 v1 = *reinterpret_cast<const double2 *>(&W[j * LD + 64 + 2 * lane]);
            double *col = out + (size_t)sh.rho[j] * n;
            col[ro[0]] = v0.x;
            col[ro[1]] = v0.y;
            col[ro[2]] = v1.x;
            col[ro[3]] = v1.y;
        }
        __syncthreads(); // everybody is done with W and sh.cell before the next cell
    }
}

// ============================================================================================================
// n = 64 NS, NS = 3, 4 (n = 192, 256: config 4, Table 2 with S32): a cluster of NQ CTAs per cell, working matrix in the
// DISTRIBUTED shared memory of the cluster.
// ============================================================================================================
// The design of factor_p128_kernel where one working matrix (532 KB at n = 256) no longer fits one SM: the n / 8 column
// blocks are dealt out in contiguous runs to the NQ CTAs of a cluster (cq_bstart), each keeping its columns column-major
// with leading dimension n + 4. NQ is as small as the shared memory allows -- two CTAs of 12 blocks at n = 192 (151 KB),
// three of 10, 11, 11 at n = 256 (183 KB) -- because a cell's time is its chain of n pivot steps whatever the number of
// SMs behind it, and the fewer SMs a cell takes the more cells are in flight (74 / 45 clusters on 148 SMs against 45 /
// 33 with n / 64 CTAs of eight blocks: config 4 8.4 -> 7.1 ms, n = 192 3.8 -> 2.9 ms). Panel p (8 columns) belongs to
// the CTA that holds its block: its n / 32 pivot warps (one row per lane) eliminate it out of their own shared memory exactly as in the
// n = 128 kernel -- nothing in a pivot step leaves the SM. The eliminated panel T (n x 8), the pivot rows R and the
// singular flag then travel ONCE to every other CTA of the cluster: the owner writes them to its own panel buffer and
// one thread issues a bulk asynchronous copy (cp.async.bulk shared::cta -> shared::cluster, completion on the
// receiver's mbarrier) per peer; every CTA then applies the rank-8 update to its own eight column blocks (transposed
// m8n8k4 DMMAs, one warp per block) from its local copy.
// Look-ahead: in the CTA that owns panel p + 1 the pivot warps update only that panel's block (warp w the 32 rows it then
// loads) and go straight on to eliminate it, while the remaining warps apply update p to the CTA's other blocks; the
// other CTAs update all their blocks. The critical path of a cell is its n pivot steps plus n / 8 one-block updates and
// stays inside one SM except at the eight-panel hand-over from CTA to CTA. No cluster barrier inside a cell: the two
// panel buffers are recycled through mbarriers -- `tfull` (the copy of panel p has landed here) and `tempty` (every peer
// has finished reading panel p: each CTA arrives remotely on all its peers' barriers after the CTA barrier that follows
// its update p, so the phase of every barrier is a function of the panel count alone).
constexpr int CQ_THREADS = 384; // 12 warps: the first n / 32 are pivot warps when the CTA owns the panel

template <int NS> struct CqPanelBuf { // NS = n / 64
    double T[FR_NB][64 * NS + 4]; // [panel column][row]
    int R[FR_NB];
    int sing, pad[7];
};

// column blocks [cq_bstart(q), cq_bstart(q + 1)) of the NB = n / 8 belong to CTA q of a cluster of NQ
__host__ __device__ constexpr int cq_bstart(int q, int NB, int NQ) { return (q * NB) / NQ; }

template <int NS, int NQ> struct CqShared { // n = 64 NS, cluster of NQ CTAs
    static constexpr int MAXB = (8 * NS + NQ - 1) / NQ; // column blocks per CTA (at most)
    double W[8 * MAXB * (64 * NS + 4)]; // [local column][row]
    CqPanelBuf<NS> pb[2];             // [panel parity]
    P128Slot slot[2][2 * NS];         // [step parity][pivot warp]
    uint64_t tfull[2];                // panel buffer `parity` holds panel p
    uint64_t tempty[2];               // every peer has finished reading panel buffer `parity`
    int rho[64 * NS], rhoinv[64 * NS];
    int tie;
};

__device__ __forceinline__ uint32_t mapa_u32(uint32_t local_addr, uint32_t cta_rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local_addr), "r"(cta_rank));
    return r;
}
__device__ __forceinline__ void bulk_s2peer(uint32_t dst_cluster, const void *src_smem, uint32_t bytes, uint32_t bar_cluster)
{
    asm volatile("cp.async.bulk.shared::cluster.shared::cta.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst_cluster),
                 "r"(smem_u32(src_smem)), "r"(bytes), "r"(bar_cluster)
                 : "memory");
}
__device__ __forceinline__ void mbar_arrive_peer(uint32_t bar_cluster)
{
    asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(bar_cluster) : "memory");
}
__device__ __forceinline__ void cluster_sync_all()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t cluster_ctarank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}

// one whole column block of a CTA's 64 columns by one warp: pivot rows read, zeroed, n / 8 row tiles updated
template <int NS>
__device__ __forceinline__ void cq_update_block(double *W, const CqPanelBuf<NS> &pb, int Jb, int rk0, int rk1, int lq, int lg)
{
    constexpr int n = 64 * NS, LD = n + 4;
    const int cl = wc2_colmap(lg);
    double *a0p = &W[(8 * Jb + cl) * LD + rk0], *a1p = &W[(8 * Jb + cl) * LD + rk1];
    const double a0 = *a0p, a1 = *a1p;
    __syncwarp();
    *a0p = 0.0;
    *a1p = 0.0;
    __syncwarp();
    dmma_strip<n / 8>(reinterpret_cast<double2 *>(&W[(8 * Jb + cl) * LD + 2 * lq]), &pb.T[lq][lg], &pb.T[4 + lq][lg], a0, a1);
}

template <int NS, int NQ, bool DUMP>
__global__ void __launch_bounds__(CQ_THREADS, 1)
factor_cq_kernel(ProblemView P, double *__restrict__ Minv, int *info, double *__restrict__ dumpA, int dump_cell)
{
    constexpr int n = 64 * NS, LD = n + 4, NPANEL = n / FR_NB, AW = 2 * NS, NWARP = CQ_THREADS / 32, UW = NWARP - AW;
    constexpr int MAXB = CqShared<NS, NQ>::MAXB;
    constexpr int SENDER = CQ_THREADS - 32; // lane 0 of the last warp: never on the pivot chain, least update work
    extern __shared__ __align__(16) unsigned char cq_smem[];
    CqShared<NS, NQ> &sh = *reinterpret_cast<CqShared<NS, NQ> *>(cq_smem);
    double *W = sh.W;
    // (roles by warp index: putting the pivot warps on sub-partitions of their own, as in factor_p128_kernel, was measured
    // slower here -- 8.4 -> 9.6 ms at n = 256, 3.8 -> 4.0 ms at n = 192: three pivot warps per sub-partition, and the update
    // warps' DMMAs on one or two pipes instead of four)
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, lq = lane & 3, lg = lane >> 2;
    const int q = (int)cluster_ctarank();
    const int n_clusters = gridDim.x / NQ, cluster_id = blockIdx.x / NQ;
    const int b0 = cq_bstart(q, NPANEL, NQ), nbq = cq_bstart(q + 1, NPANEL, NQ) - b0; // this CTA's column blocks

    if (threadIdx.x == 0) {
        mbar_init(&sh.tfull[0], 1);
        mbar_init(&sh.tfull[1], 1);
        mbar_init(&sh.tempty[0], NQ - 1);
        mbar_init(&sh.tempty[1], NQ - 1);
        fence_mbar_init();
        sh.tie = 0;
    }
    cluster_sync_all(); // barriers initialised everywhere before any peer copies into this CTA or arrives here
    unsigned gp = 0;    // panels processed so far by this cluster (selects buffer and barrier parities)

    // "this CTA has finished reading panel buffer b": one remote arrival on every peer's tempty[b]
    auto release_panel_buffer = [&](int b) {
#pragma unroll
        for (int peer = 0; peer < NQ; ++peer)
            if (peer != q) mbar_arrive_peer(mapa_u32(smem_u32(&sh.tempty[b]), peer));
    };

    for (int cell = DUMP ? dump_cell : cluster_id; cell < P.J; cell += n_clusters) {
        // ---- a1: this CTA's 8 nbq columns (2 nbq column blocks of 4) x n rows
        {
            double *Wl = W - (size_t)8 * b0 * LD; // so that the global column index addresses the local array
            for (int idx = w; idx < NS * 2 * nbq; idx += NWARP)
                assemble_rows2(P, cell, lane, Wl, LD, 2 * b0 + idx % (2 * nbq), 1 << 20, 64 * (idx / (2 * nbq)), 1 << 20);
        }
        __syncthreads();
        if (DUMP) { // the assembled tile of the production kernel, row-major, for the bit-exactness test
            for (int e = threadIdx.x; e < n * 8 * nbq; e += CQ_THREADS)
                dumpA[(size_t)(e / (8 * nbq)) * n + 8 * b0 + e % (8 * nbq)] = W[(e % (8 * nbq)) * LD + e / (8 * nbq)];
            break;
        }

        unsigned m = 0x7fffffffu; // pivot warps: 0 once row 32 w + lane has been a pivot row (tracked in every CTA)
        bool singular = false;
        for (int pnl = 0; pnl < NPANEL; ++pnl, ++gp) {
            const int buf = gp & 1;
            const uint32_t par = (gp >> 1) & 1;
            const bool own = pnl >= b0 && pnl < b0 + nbq, own_next = pnl + 1 >= b0 && pnl + 1 < b0 + nbq;
            const int lb = pnl - b0; // local index of the panel's block (when this CTA owns it)
            CqPanelBuf<NS> &pb = sh.pb[buf];
            if (own && w < AW) {
                // ================= phase P: the owner's pivot warps eliminate the n x 8 panel, one row per lane =========
                // (its block is up to date: updates < pnl - 1 by the update warps before the last CTA barrier, update
                // pnl - 1 by this very warp, rows 32 w .. 32 w + 31, in the look-ahead below)
                const int r = 32 * w + lane;
                double *Wp = &W[(FR_NB * lb) * LD + r];
                double t[FR_NB];
#pragma unroll
                for (int c = 0; c < FR_NB; ++c) t[c] = Wp[c * LD];
                unsigned bad = 0u, tie = 0u;
                const unsigned m_in = m;
                pw_panel<true, AW>(t, m, &sh.slot[0][0], sh.rho, sh.rhoinv, w, lane, FR_NB * pnl, bad, tie);
                if (tie) sh.tie = 1;
                pivot_warps_bar<AW>();
                const bool redo = sh.tie != 0;
                pivot_warps_bar<AW>();
                if (redo) { // rare: the panel again, from shared memory, ties resolved exactly
                    if (threadIdx.x == 0) sh.tie = 0;
#pragma unroll
                    for (int c = 0; c < FR_NB; ++c) t[c] = Wp[c * LD];
                    m = m_in;
                    bad = 0u;
                    pw_panel<false, AW>(t, m, &sh.slot[0][0], sh.rho, sh.rhoinv, w, lane, FR_NB * pnl, bad, tie);
                }
                // the panel buffer is free once every peer has finished reading the panel before last (which also means
                // that the bulk copies out of it have completed)
                if (gp >= 2) mbar_wait(&sh.tempty[buf], ((gp >> 1) - 1) & 1);
#pragma unroll
                for (int c = 0; c < FR_NB; ++c) { // the eliminated panel: in place, and into the panel buffer
                    Wp[c * LD] = t[c];
                    pb.T[c][r] = t[c];
                }
                if (w == 0 && lane < FR_NB) pb.R[lane] = sh.rho[FR_NB * pnl + lane];
                if (threadIdx.x == 0) pb.sing = bad ? 1 : 0;
            }
            __syncthreads(); // barrier p: update p - 1 is complete in this CTA; in the owner, the panel buffer is complete
            if (threadIdx.x == SENDER) {
                if (own) {
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); // generic-proxy writes -> bulk-copy reads
#pragma unroll
                    for (int peer = 0; peer < NQ; ++peer)
                        if (peer != q)
                            bulk_s2peer(mapa_u32(smem_u32(&pb), peer), &pb, (uint32_t)sizeof(CqPanelBuf<NS>),
                                        mapa_u32(smem_u32(&sh.tfull[buf]), peer));
                    mbar_arrive(&sh.tfull[buf]); // the owner's own copy is already in place
                } else {
                    mbar_arrive_expect_tx(&sh.tfull[buf], (uint32_t)sizeof(CqPanelBuf<NS>));
                }
                if (pnl > 0) release_panel_buffer(buf ^ 1); // nobody here reads the previous panel any more (a cell's last
                                                             // panel is released after the loop)
            }
            if (!own) mbar_wait(&sh.tfull[buf], par);
            if (pb.sing) { singular = true; ++gp; break; } // cluster-uniform
            // every CTA keeps the whole permutation and the used-row masks (any CTA may own a later panel)
            if (!own && threadIdx.x < FR_NB) {
                const int r = pb.R[threadIdx.x];
                sh.rho[FR_NB * pnl + threadIdx.x] = r;
                sh.rhoinv[r] = FR_NB * pnl + threadIdx.x;
            }
            if (!own && w < AW) {
#pragma unroll
                for (int b = 0; b < FR_NB; ++b)
                    if (pb.R[b] == 32 * w + lane) m = 0u;
            }
            // ================= phase U: this CTA's column blocks =================
            const int rk0 = pb.R[lq], rk1 = pb.R[4 + lq];
            const int nb = pnl + 1 - b0; // local index of the next panel's block (when this CTA owns it)
            if (own_next && w < AW) {
                // look-ahead: the next panel's block, pivot warp w its own 32 rows (row tiles 4 w .. 4 w + 3). Every pivot
                // warp reads the pivot-row entries of the block, one barrier over the pivot warps, then each warp zeroes
                // the pivot rows that lie in its own 32 rows (see wc2_update_blocks) and accumulates.
                const int cl = wc2_colmap(lg);
                double *a0p = &W[(8 * nb + cl) * LD + rk0], *a1p = &W[(8 * nb + cl) * LD + rk1];
                const double a0 = *a0p, a1 = *a1p;
                pivot_warps_bar<AW>(); // every pivot warp has read the pivot rows of the block
                if ((rk0 >> 5) == w) *a0p = 0.0;
                if ((rk1 >> 5) == w) *a1p = 0.0;
                __syncwarp();
                dmma_strip<4>(reinterpret_cast<double2 *>(&W[(8 * nb + cl) * LD + 2 * lq + 32 * w]), &pb.T[lq][32 * w + lg],
                              &pb.T[4 + lq][32 * w + lg], a0, a1);
                __syncwarp();
            } else if (own_next) {
                // the update warps while the pivot warps are busy with the next panel: this CTA's other nbq - 2 or nbq - 1
                // blocks as half-blocks (n / 2 rows), shared out round-robin (the last warp, which is also the sender,
                // gets the fewest). The pivot-row entries of a block are read by everybody before anybody stores (named
                // barrier over the update warps); each warp then zeroes the pivot rows that lie in its own half.
                const int wi = w - AW;
                const int s1 = own ? (lb < nb ? lb : nb) : nb, s2 = own ? (lb < nb ? nb : lb) : 99; // skipped blocks, sorted
                const int nitems = 2 * (nbq - (own ? 2 : 1));
                constexpr int MAXIT = (2 * (MAXB - 1) + UW - 1) / UW;
                const int cl = wc2_colmap(lg);
                double a0[MAXIT], a1[MAXIT];
                int jb[MAXIT];
#pragma unroll
                for (int sl = 0; sl < MAXIT; ++sl) {
                    const int it = wi + sl * UW;
                    int Jb = it >> 1;
                    if (Jb >= s1) ++Jb;
                    if (Jb >= s2) ++Jb;
                    jb[sl] = Jb;
                    if (it < nitems) {
                        a0[sl] = W[(8 * Jb + cl) * LD + rk0];
                        a1[sl] = W[(8 * Jb + cl) * LD + rk1];
                    }
                }
                asm volatile("bar.sync 2, %0;" ::"n"(32 * UW) : "memory");
#pragma unroll
                for (int sl = 0; sl < MAXIT; ++sl) {
                    const int it = wi + sl * UW;
                    if (it < nitems) {
                        const int r0 = (it & 1) * (n / 2); // first row of the half
                        double *col = &W[(8 * jb[sl] + cl) * LD];
                        if ((unsigned)(rk0 - r0) < (unsigned)(n / 2)) col[rk0] = 0.0;
                        if ((unsigned)(rk1 - r0) < (unsigned)(n / 2)) col[rk1] = 0.0;
                        __syncwarp();
                        dmma_strip<n / 16>(reinterpret_cast<double2 *>(col + 2 * lq + r0), &pb.T[lq][r0 + lg],
                                                    &pb.T[4 + lq][r0 + lg], a0[sl], a1[sl]);
                    }
                }
            } else {
                // nobody here is on the pivot chain: whole blocks, one per warp
                int k = 0;
                for (int Jb = 0; Jb < nbq; ++Jb) {
                    if (own && Jb == lb) continue;
                    if (k == w) cq_update_block<NS>(W, pb, Jb, rk0, rk1, lq, lg);
                    k = (k + 1 == NWARP) ? 0 : k + 1;
                }
            }
        }
        __syncthreads(); // the last update is complete (or the cell was found singular)
        if (threadIdx.x == SENDER) release_panel_buffer((gp - 1) & 1);

        double *out = Minv + (size_t)cell * n * n;
        if (singular) {
            if (q == 0 && threadIdx.x == 0) atomicMin(info, cell + 1);
            for (int e = threadIdx.x; e < 8 * nbq * n / 2; e += CQ_THREADS)
                reinterpret_cast<double2 *>(out + (size_t)8 * b0 * n)[e] = make_double2(0.0, 0.0);
            __syncthreads();
            continue;
        }
        // ---- store A^{-1} column-major: Ainv[rhoinv[i]][rho[j]] = W[i][j]; this CTA's columns j = 8 b0 + jl
        for (int jl = w; jl < 8 * nbq; jl += NWARP) {
            double *col = out + (size_t)sh.rho[8 * b0 + jl] * n;
#pragma unroll
            for (int s2 = 0; s2 < NS; ++s2) {
                const double2 v = *reinterpret_cast<const double2 *>(&W[jl * LD + 64 * s2 + 2 * lane]);
                col[sh.rhoinv[64 * s2 + 2 * lane]] = v.x;
                col[sh.rhoinv[64 * s2 + 2 * lane + 1]] = v.y;
            }
        }
        __syncthreads(); // everybody is done with W before the next cell's assembly
    }
    cluster_sync_all(); // no CTA exits while a peer may still address its shared memory
}

__global__ void assemble_one_kernel(ProblemView P, int cell, double *__restrict__ A)
{
    const int n = P.n;
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < n * n; e += gridDim.x * blockDim.x)
        A[e] = a_entry(P, cell, e / n, e % n);
}

size_t factor_smem_bytes(int n, bool global_w)
{
    constexpr int NW = FACTOR_THREADS / 32;
    size_t b = (size_t)(2 * n + NW) * sizeof(double) + (size_t)(NW + 3 * n + 1) * sizeof(int);
    b = (b + 15) & ~(size_t)15;
    if (!global_w) b += (size_t)n * (n + 1) * sizeof(double);
    return b;
}

} // namespace

// Scratch the factor path may need: per-CTA n x n working arrays when n is too large for shared memory,
// and at least one n x n matrix for the debug getters.
size_t factor_scratch_bytes(int n, int num_sms, int max_smem_optin)
{
    size_t one = (size_t)n * n * sizeof(double);
    if (factor_smem_bytes(n, false) <= (size_t)max_smem_optin) return one;
    return one * (size_t)num_sms * 4;
}

// n = 64, one warp per cell (factor_wc_kernel). dumpA != nullptr: only assemble `dump_cell` and write the tile there.
static int launch_factor_wc(oci_ctx *ctx, const ProblemView &P, double *dumpA, int dump_cell)
{
    const bool two = ctx->opt_factor_kernel == 1; // 1: two warps per cell with look-ahead; 4: one warp per cell
    const size_t smem = two ? sizeof(Wc2Shared) : sizeof(WcShared);
    const int threads = two ? 64 : 32;
    const bool dmma = ctx->opt_factor_update != 0;
    const void *fn;
    if (two) fn = dumpA ? (const void *)factor_wc2_kernel<true, false>
                        : (ctx->opt_factor_update >= 2 ? (const void *)factor_wc2_kernel<false, true>
                                                       : (const void *)factor_wc2_kernel<false, false>);
    else fn = dumpA ? (const void *)factor_wc_kernel<true, true>
                    : (dmma ? (const void *)factor_wc_kernel<true, false> : (const void *)factor_wc_kernel<false, false>);
    int grid = 1;
    if (dumpA || ctx->factor_fn != fn) { // attributes and occupancy once per (context, kernel)
        OCI_CUDA_TRY(ctx, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        OCI_CUDA_TRY(ctx, cudaFuncSetAttribute(fn, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
        if (!dumpA) {
            int per_sm = 0;
            OCI_CUDA_TRY(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, threads, smem));
            grid = (per_sm < 1 ? 1 : per_sm) * ctx->num_sms;
            if (grid > ctx->J) grid = ctx->J;
            ctx->factor_fn = fn;
            ctx->factor_grid = grid;
        }
    }
    if (!dumpA) {
        grid = ctx->factor_grid;
        OCI_CUDA_TRY(ctx, cudaMemsetAsync(ctx->info + 1, 0, sizeof(int), ctx->stream)); // the cell counter
    }
    int *counter = ctx->info + 1;
    double *Minv = ctx->Minv;
    int *info = ctx->info;
    ProblemView Pv = P;
    int role_mode = 0;
    void *args[] = {&Pv, &Minv, &info, &counter, &dumpA, &dump_cell, &role_mode};
    OCI_CUDA_TRY(ctx, cudaLaunchKernel(fn, dim3(grid), dim3(threads), args, smem, ctx->stream));
    return 1;
}

// n = 192, 256: a cluster of NQ CTAs per cell (factor_cq_kernel). dumpA != nullptr: only assemble `dump_cell`.
template <int NS, int NQ, bool DUMP> static int launch_factor_cq_t(oci_ctx *ctx, const ProblemView &P, double *dumpA, int dump_cell)
{
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.blockDim = dim3(CQ_THREADS, 1, 1);
    cfg.dynamicSmemBytes = sizeof(CqShared<NS, NQ>);
    const void *fn = (const void *)factor_cq_kernel<NS, NQ, DUMP>;
    const bool known = !DUMP && ctx->factor_fn == fn; // attributes and occupancy once per (context, kernel)
    if (!known)
        OCI_CUDA_TRY(ctx, cudaFuncSetAttribute(factor_cq_kernel<NS, NQ, DUMP>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                               (int)sizeof(CqShared<NS, NQ>)));
    cfg.stream = ctx->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = NQ;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    int n_clusters = 1;
    if (known) n_clusters = ctx->factor_grid;
    else if (!DUMP) {
        cfg.gridDim = dim3(NQ * ctx->num_sms, 1, 1); // any multiple of NQ: the query only needs the shape
        OCI_CUDA_TRY(ctx, cudaOccupancyMaxActiveClusters(&n_clusters, factor_cq_kernel<NS, NQ, DUMP>, &cfg));
        if (n_clusters < 1) n_clusters = 1;
        if (n_clusters > ctx->J) n_clusters = ctx->J;
        ctx->factor_fn = fn;
        ctx->factor_grid = n_clusters;
    }
    cfg.gridDim = dim3(NQ * n_clusters, 1, 1);
    OCI_CUDA_TRY(ctx, cudaLaunchKernelEx(&cfg, factor_cq_kernel<NS, NQ, DUMP>, P, ctx->Minv, ctx->info, dumpA, dump_cell));
    return 1;
}

// n = 192: clusters of two CTAs (12 column blocks each), n = 256: of three (10, 11, 11): as few CTAs per cell as hold the
// working matrix -- a cell's time is its chain of n pivot steps whatever the number of SMs behind it, so the cells in
// flight (74 / 45 clusters on 148 SMs; clusters of n / 64 CTAs: 45 / 33) are what counts. factor_cluster = 1 restores
// clusters of n / 64 CTAs with eight column blocks each.
static int launch_factor_cq(oci_ctx *ctx, const ProblemView &P, double *dumpA, int dump_cell)
{
    const bool wide = ctx->opt_factor_cluster == 1;
    if (ctx->n == 192) {
        if (wide) return dumpA ? launch_factor_cq_t<3, 3, true>(ctx, P, dumpA, dump_cell) : launch_factor_cq_t<3, 3, false>(ctx, P, nullptr, 0);
        return dumpA ? launch_factor_cq_t<3, 2, true>(ctx, P, dumpA, dump_cell) : launch_factor_cq_t<3, 2, false>(ctx, P, nullptr, 0);
    }
    if (wide) return dumpA ? launch_factor_cq_t<4, 4, true>(ctx, P, dumpA, dump_cell) : launch_factor_cq_t<4, 4, false>(ctx, P, nullptr, 0);
    return dumpA ? launch_factor_cq_t<4, 3, true>(ctx, P, dumpA, dump_cell) : launch_factor_cq_t<4, 3, false>(ctx, P, nullptr, 0);
}

// n = 128, one CTA per cell (factor_p128_kernel). dumpA != nullptr: only assemble `dump_cell` and write the tile there.
static int launch_factor_p128(oci_ctx *ctx, const ProblemView &P, double *dumpA, int dump_cell)
{
    const size_t smem = sizeof(P128Shared);
    const void *fn = dumpA ? (const void *)factor_p128_kernel<true> : (const void *)factor_p128_kernel<false>;
    if (dumpA || ctx->factor_fn != fn) { // once per (context, kernel)
        OCI_CUDA_TRY(ctx, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        if (!dumpA) ctx->factor_fn = fn;
    }
    int grid = 1;
    if (!dumpA) {
        grid = ctx->num_sms;
        if (grid > ctx->J) grid = ctx->J;
        OCI_CUDA_TRY(ctx, cudaMemsetAsync(ctx->info + 1, 0, sizeof(int), ctx->stream)); // the cell counter
    }
    int *counter = ctx->info + 1;
    double *Minv = ctx->Minv;
    int *info = ctx->info;
    ProblemView Pv = P;
    void *args[] = {&Pv, &Minv, &info, &counter, &dumpA, &dump_cell};
    OCI_CUDA_TRY(ctx, cudaLaunchKernel(fn, dim3(grid), dim3(P128_THREADS), args, smem, ctx->stream));
    return 1;
}

int launch_factor(oci_ctx *ctx)
{
    const int n = ctx->n;
    ProblemView P = make_view(ctx);
    OCI_CUDA_TRY(ctx, cudaMemsetAsync(ctx->info, 0x7f, sizeof(int), ctx->stream)); // 0x7f7f7f7f = "none"
    if ((ctx->opt_factor_kernel == 1 || ctx->opt_factor_kernel == 4) && n == 64) return launch_factor_wc(ctx, P, nullptr, 0);
    if (ctx->opt_factor_kernel == 1 && n == 128) return launch_factor_p128(ctx, P, nullptr, 0);
    if (ctx->opt_factor_kernel == 1 && (n == 192 || n == 256)) return launch_factor_cq(ctx, P, nullptr, 0);
    const bool global_w = factor_smem_bytes(n, false) > (size_t)ctx->max_smem_optin;
    const size_t smem = factor_smem_bytes(n, global_w);
    int grid;
    if (!global_w) {
        const void *fn = (const void *)factor_gj_kernel<false>;
        if (ctx->factor_fn != fn) { // once per (context, kernel)
            OCI_CUDA_TRY(ctx, cudaFuncSetAttribute(factor_gj_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                   (int)smem));
            int per_sm = 1;
            OCI_CUDA_TRY(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, factor_gj_kernel<false>,
                                                                            FACTOR_THREADS, smem));
            if (per_sm < 1) per_sm = 1;
            grid = ctx->num_sms * per_sm;
            if (grid > ctx->J) grid = ctx->J;
            ctx->factor_fn = fn;
            ctx->factor_grid = grid;
        }
        grid = ctx->factor_grid;
        factor_gj_kernel<false><<<grid, FACTOR_THREADS, smem, ctx->stream>>>(P, ctx->Minv, nullptr, n + 1, ctx->info);
    } else {
        grid = ctx->num_sms * 4;
        if (grid > ctx->J) grid = ctx->J;
        if ((size_t)grid * n * n * sizeof(double) > ctx->scratch_bytes) return OCI_E_WORKSPACE;
        factor_gj_kernel<true><<<grid, FACTOR_THREADS, smem, ctx->stream>>>(P, ctx->Minv, ctx->scratch, n, ctx->info);
    }
    OCI_CUDA_TRY(ctx, cudaGetLastError());
    return 1;
}

// The tile the production factor kernel of the current options assembles on chip for `cell`, dumped before the
// elimination (row-major); 0 = that kernel has no such path (it assembles through a_entry(), see launch_assemble_one).
int launch_factor_input(oci_ctx *ctx, int cell, double *A_dev_rowmajor)
{
    ProblemView P = make_view(ctx);
    if ((ctx->opt_factor_kernel == 1 || ctx->opt_factor_kernel == 4) && ctx->n == 64)
        return launch_factor_wc(ctx, P, A_dev_rowmajor, cell);
    if (ctx->opt_factor_kernel == 1 && ctx->n == 128) return launch_factor_p128(ctx, P, A_dev_rowmajor, cell);
    if (ctx->opt_factor_kernel == 1 && (ctx->n == 192 || ctx->n == 256)) return launch_factor_cq(ctx, P, A_dev_rowmajor, cell);
    return 0;
}

int launch_assemble_one(oci_ctx *ctx, int cell, double *A_dev_rowmajor)
{
    ProblemView P = make_view(ctx);
    assemble_one_kernel<<<32, 256, 0, ctx->stream>>>(P, cell, A_dev_rowmajor);
    OCI_CUDA_TRY(ctx, cudaGetLastError());
    return 1;
}
