// si.cu -- a9..a11 of SURVEY.md section 8(a): the source-iteration comparator (Alg. 1, PAPER.md:366-411;
// Appendix A, Eq. 42-46), "parallel over angles x groups and serial in space".
//
// One source iteration:
//   s_{j,g,p} = sum_g' K_j[g][g'] phi^(l)_{j,g',p}                       (all groups lagged, A5/A13)
//   for every (g,m), cells in the direction of mu_m:   L_{c,j,g,m} psi = d + mu * (upstream psi of THIS sweep)
//   phi^(l+1) = sum_m w_m psi_m,  r = max |phi^(l+1) - phi^(l)|
// The 4x4 solve of Eq. 42 is linear in the incident edge flux, and only the two "outgoing" unknowns feed the
// next cell (Eq. 5a-b). The work is therefore split into
//   si_source : (parallel over j,g,m)  base = L^-1 d            -- everything that does not depend on the sweep
//   si_sweep  : (parallel over g,m; SERIAL over j)  in_{j+1} = base_out_j + T_j in_j   (2x2 affine map per cell)
//   si_finish : (parallel over j,g,m)  psi = base + C in,  phi, residual
// which is the same arithmetic as solving cell after cell, re-associated; the serial chain per cell is two
// dependent fused multiply-adds instead of a 4x4 solve.
#include "common.cuh"

namespace {

// Sweep-order record index of (cell j, ordinate gm): chains are grouped `lpc` to a CTA; within a CTA's slab the
// records of one sweep step jj (cell jj for mu > 0, cell J-1-jj for mu < 0) of its lpc chains are contiguous, so a
// tile of consecutive sweep steps is ONE contiguous block that a single bulk copy brings into shared memory.
__device__ __forceinline__ size_t sweep_index(int J, int lpc, size_t j, int gm, bool fwd)
{
    const size_t jj = fwd ? j : (size_t)(J - 1) - j;
    return ((size_t)(gm / lpc) * J + jj) * lpc + (gm % lpc);
}

// Once per (problem, dt): Linv[j][g][m][4][4] = L_{c,j,g,m}^{-1} (Eq. 8b / 42),
// C[j][g][m][p][lev] = |mu_m| Linv[p][row that receives the incident flux of level lev], and the 2x2 part of C
// that maps incident -> outgoing edge flux, T2sw[sweep_index][2][2], in sweep order for si_sweep_kernel.
__global__ void si_setup_kernel(ProblemView P, int lpc, double *__restrict__ Linv, double *__restrict__ C,
                                double *__restrict__ T2sw)
{
    const size_t total = (size_t)P.J * P.G * P.N;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (size_t)gridDim.x * blockDim.x) {
        const int m = (int)(e % P.N);
        const size_t jg = e / P.N;
        const int g = (int)(jg % P.G);
        const size_t j = jg / P.G;
        const double mu = P.mu[m];
        double a[4][4], b[4][4];
#pragma unroll
        for (int p = 0; p < 4; ++p)
#pragma unroll
            for (int pp = 0; pp < 4; ++pp) a[p][pp] = lc_entry(p, pp, P.dx[j], P.sigma_t[jg], P.v[g], P.dt, mu);
        inv4(a, b);
        double *Lo = Linv + e * 16;
#pragma unroll
        for (int p = 0; p < 4; ++p)
#pragma unroll
            for (int pp = 0; pp < 4; ++pp) Lo[p * 4 + pp] = b[p][pp];
        const double am = fabs(mu);
        double *Co = C + e * 8;
#pragma unroll
        for (int p = 0; p < 4; ++p) {
            // mu > 0: rows (k,L)=0 and (k+1/2,L)=2 receive the incident flux; mu < 0: rows 1 and 3 (Eq. 43b-c)
            Co[p * 2 + 0] = am * (mu > 0.0 ? b[p][0] : b[p][1]);
            Co[p * 2 + 1] = am * (mu > 0.0 ? b[p][2] : b[p][3]);
        }
        // outgoing unknowns: (k,R),(k+1/2,R) = rows 1,3 for mu > 0; (k,L),(k+1/2,L) = rows 0,2 for mu < 0 (Eq. 5a-b)
        const bool fwd = mu > 0.0;
        const int o0 = fwd ? 1 : 0;
        double *To = T2sw + sweep_index(P.J, lpc, j, g * P.N + m, fwd) * 4;
        reinterpret_cast<double2 *>(To)[0] = make_double2(Co[o0 * 2], Co[o0 * 2 + 1]);
        reinterpret_cast<double2 *>(To)[1] = make_double2(Co[(o0 + 2) * 2], Co[(o0 + 2) * 2 + 1]);
    }
}

// a9: d_{j,g,m} (Eq. 43b-c, without the incident term) and base = Linv d.
__global__ void si_source_kernel(StopCheck stop, ProblemView P, int lpc, const double *__restrict__ q,
                                 const double *__restrict__ psi_prev, const double *__restrict__ phi,
                                 const double *__restrict__ Linv, double *__restrict__ base,
                                 double *__restrict__ bsw)
{
    if (stop_reached(stop)) return;
    const size_t total = (size_t)P.J * P.G * P.N;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (size_t)gridDim.x * blockDim.x) {
        const size_t jg = e / P.N;
        const int g = (int)(jg % P.G);
        const size_t j = jg / P.G;
        const double dx = P.dx[j];
        const double *Kj = P.transfer + (j * P.G + g) * P.G;
        const double *phij = phi + j * P.G * 4;
        double d[4];
#pragma unroll
        for (int p = 0; p < 4; ++p) {
            double s = 0.0;
            for (int gp = 0; gp < P.G; ++gp) s = fma(Kj[gp], phij[gp * 4 + p], s);
            d[p] = dx * 0.25 * (s + q[jg * 4 + p]);
        }
        const double half_gam = dx / (2.0 * P.v[g] * P.dt);
        d[0] = fma(half_gam, psi_prev[e * 2 + 0], d[0]);
        d[1] = fma(half_gam, psi_prev[e * 2 + 1], d[1]);
        const double *L = Linv + e * 16;
        double bs[4];
#pragma unroll
        for (int p = 0; p < 4; ++p) {
            bs[p] = fma(L[p * 4 + 3], d[3], fma(L[p * 4 + 2], d[2], fma(L[p * 4 + 1], d[1], L[p * 4 + 0] * d[0])));
            base[e * 4 + p] = bs[p];
        }
        // the two outgoing entries of base, in sweep order (the constant term of the sweep's 2x2 affine map)
        const int m = (int)(e % P.N);
        const bool fwd = P.mu[m] > 0.0;
        *reinterpret_cast<double2 *>(bsw + sweep_index(P.J, lpc, j, g * P.N + m, fwd) * 2) =
            fwd ? make_double2(bs[1], bs[3]) : make_double2(bs[0], bs[2]);
    }
}

// a10: the sweep. One CTA per group of LPC chains (ordinates (g,m)), warp-specialised:
//   warp 1, one thread : issues one bulk async copy per tile (TC sweep steps x LPC chains) of the 2x2 maps and one of
//                        the constant terms into a ring of 3-4 shared-memory stages (mbarrier handshake);
//   warp 0, lane = chain: runs the serial chain  in_{jj+1} = b_jj + T_jj in_jj  out of shared memory -- per cell three
//                        conflict-free 16-byte loads, four DFMAs (two dependent), one 16-byte shared-memory store of
//                        the incident flux that si_finish needs. Nothing else is on its instruction stream.
//   warp 2              : copies the finished tiles of incident fluxes from shared memory to in_out[j][gm][2].
// The chain is the latency floor of a sweep "serial in space": J x 2 dependent DFMAs.
constexpr int TC = 64;         // sweep steps per tile
__host__ __device__ constexpr int sw_stages(int lpc) { return lpc >= 16 ? 3 : 4; } // ring depth (227 KB per CTA)
constexpr int SW_THREADS = 96;
constexpr int SW_AHEAD = 4;    // cells of look-ahead of the chain warp's shared-memory loads

template <int LPC>
__global__ void __launch_bounds__(SW_THREADS) si_sweep_kernel(StopCheck stop, int J, int N, int G, int bc_left,
                                                              int bc_right, const double *__restrict__ mu,
                                                              const double *__restrict__ T2sw,
                                                              const double *__restrict__ bsw,
                                                              const double *__restrict__ psi_old,
                                                              const double *__restrict__ inc_left,
                                                              const double *__restrict__ inc_right,
                                                              double *__restrict__ in_out)
{
    constexpr int NST = sw_stages(LPC);
    extern __shared__ __align__(128) unsigned char sw_smem[];
    typedef double (*TsT)[TC][LPC][4];
    typedef double (*BsT)[TC][LPC][2];
    TsT Ts = reinterpret_cast<TsT>(sw_smem);                                              // [NST][TC][LPC][4]
    BsT Bs = reinterpret_cast<BsT>(sw_smem + sizeof(double) * NST * TC * LPC * 4); // [NST][TC][LPC][2]
    BsT Os = reinterpret_cast<BsT>(sw_smem + sizeof(double) * NST * TC * LPC * 6); // incident fluxes found
    uint64_t *full = reinterpret_cast<uint64_t *>(sw_smem + sizeof(double) * NST * TC * LPC * 8);
    uint64_t *empty = full + NST;     // stage free again: chain warp done reading AND writer warp done copying
    uint64_t *outfull = empty + NST;  // chain warp finished the tile: Os[stage] complete
    if (stop_reached(stop)) return;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int GN = G * N, n = 4 * GN;
    const int gm0 = blockIdx.x * LPC;
    const int n_tiles = (J + TC - 1) / TC;
    if (tid == 0) {
        for (int s = 0; s < NST; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 2); mbar_init(&outfull[s], 1); }
        fence_mbar_init();
    }
    __syncthreads();

    if (warp == 1) {
        if (lane == 0) {
            const double *Tsrc = T2sw + (size_t)blockIdx.x * J * LPC * 4;
            const double *Bsrc = bsw + (size_t)blockIdx.x * J * LPC * 2;
            for (int t = 0; t < n_tiles; ++t) {
                const int st = t % NST;
                mbar_wait(&empty[st], ((t / NST) & 1) ^ 1);
                const int cells = min(TC, J - t * TC);
                const uint32_t bt = (uint32_t)(cells * LPC * 4 * sizeof(double));
                const uint32_t bb = (uint32_t)(cells * LPC * 2 * sizeof(double));
                mbar_arrive_expect_tx(&full[st], bt + bb);
                bulk_g2s(&Ts[st][0][0][0], Tsrc + (size_t)t * TC * LPC * 4, bt, &full[st]);
                bulk_g2s(&Bs[st][0][0][0], Bsrc + (size_t)t * TC * LPC * 2, bb, &full[st]);
            }
        }
        return;
    }
    if (warp == 2) { // writer: Os[stage][u][l] -> in_out[cell of sweep step t TC + u][gm0 + l]
        const int l = lane % LPC, u_first = lane / LPC, gmw = gm0 + l;
        const bool on = gmw < GN;
        const bool fwd_w = on ? mu[gmw % N] > 0.0 : true;
        for (int t = 0; t < n_tiles; ++t) {
            const int st = t % NST;
            mbar_wait(&outfull[st], (t / NST) & 1);
            const int cells = min(TC, J - t * TC);
            if (on) {
                for (int u = u_first; u < cells; u += 32 / LPC) {
                    const size_t jj = (size_t)t * TC + u;
                    const size_t j = fwd_w ? jj : (size_t)(J - 1) - jj;
                    *reinterpret_cast<double2 *>(in_out + (j * GN + gmw) * 2) =
                        *reinterpret_cast<const double2 *>(&Os[st][u][l][0]);
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[st]);
        }
        return;
    }

    const int gm = gm0 + lane;
    const bool active = lane < LPC && gm < GN;
    bool fwd = true;
    double in0 = 0.0, in1 = 0.0;
    if (active) {
        const int g = gm / N, m = gm % N;
        fwd = mu[m] > 0.0;
        const int bc = fwd ? bc_left : bc_right;
        if (bc == OCI_BC_REFLECTIVE) { // mirror ordinate of the boundary cell, from iteration l (A12)
            const double *cellp = psi_old + (fwd ? (size_t)0 : (size_t)(J - 1) * n) + (size_t)(g * N + (N - 1 - m)) * 4;
            in0 = cellp[fwd ? 0 : 1];
            in1 = cellp[fwd ? 2 : 3];
        } else if (bc == OCI_BC_PRESCRIBED) {
            const double *ip = (fwd ? inc_left : inc_right) + (size_t)gm * 2;
            in0 = ip[0];
            in1 = ip[1];
        }
    }
    const int l = active ? lane : 0;

    for (int t = 0; t < n_tiles; ++t) {
        const int st = t % NST;
        mbar_wait(&full[st], (t / NST) & 1);
        const int cells = min(TC, J - t * TC);
        if (active) {
            // software-pipelined: the coefficients of cell u + SW_AHEAD are loaded from shared memory while cell u
            // is on the chain, so that the two dependent DFMAs never wait for a shared-memory load
            double2 t0[SW_AHEAD], t1[SW_AHEAD], bb[SW_AHEAD];
#pragma unroll
            for (int d = 0; d < SW_AHEAD; ++d) {
                t0[d] = *reinterpret_cast<const double2 *>(&Ts[st][d][l][0]);
                t1[d] = *reinterpret_cast<const double2 *>(&Ts[st][d][l][2]);
                bb[d] = *reinterpret_cast<const double2 *>(&Bs[st][d][l][0]);
            }
#define OCI_SWEEP_CELL(GUARD)                                                                                      \
    do {                                                                                                           \
        if (!(GUARD) || u0 + d < cells) {                                                                          \
            *reinterpret_cast<double2 *>(&Os[st][u0 + d][l][0]) = make_double2(in0, in1);                          \
            const double o0 = fma(t0[d].x, in0, fma(t0[d].y, in1, bb[d].x));                                       \
            const double o1 = fma(t1[d].x, in0, fma(t1[d].y, in1, bb[d].y));                                       \
            in0 = o0;                                                                                              \
            in1 = o1;                                                                                              \
        }                                                                                                          \
        const int un = min(u0 + d + SW_AHEAD, TC - 1); /* stays inside the stage; unused past `cells` */           \
        t0[d] = *reinterpret_cast<const double2 *>(&Ts[st][un][l][0]);                                             \
        t1[d] = *reinterpret_cast<const double2 *>(&Ts[st][un][l][2]);                                             \
        bb[d] = *reinterpret_cast<const double2 *>(&Bs[st][un][l][0]);                                             \
    } while (0)
            if (cells == TC) {
#pragma unroll 4
                for (int u0 = 0; u0 < TC; u0 += SW_AHEAD) {
#pragma unroll
                    for (int d = 0; d < SW_AHEAD; ++d) OCI_SWEEP_CELL(false);
                }
            } else {
                for (int u0 = 0; u0 < cells; u0 += SW_AHEAD) {
#pragma unroll
                    for (int d = 0; d < SW_AHEAD; ++d) OCI_SWEEP_CELL(true);
                }
            }
#undef OCI_SWEEP_CELL
        }
        __syncwarp();
        if (lane == 0) { mbar_arrive(&outfull[st]); mbar_arrive(&empty[st]); }
    }
}

// ============================================================================================================
// SURVEY 8(f) row f4 (second half): the sweep as a parallel scan -- "si_sweep" = 1. NOT the comparator of north_star
// (which is serial in space, above); it is here because it changes the OCI-vs-SI verdict and that should be known.
// ============================================================================================================
// The per-cell maps in -> T in + b are affine, and composition of affine maps is associative, so the incident flux of
// every cell is a prefix "sum" under composition along the sweep direction. Two kernels, no inter-CTA waiting:
//   si_scan_reduce : per (chain, block of 1024 sweep steps): every thread composes its 4 maps, a block-level scan
//                    (shuffles + shared memory) gives each thread the composition of everything before it in the
//                    block (stored) and the block its aggregate (stored);
//   si_scan_apply  : every block folds the aggregates of the blocks before it onto the boundary value (<= J / 1024 short
//                    steps), every thread applies its stored prefix and walks its 4 cells.
// Layout: the sweep-order arrays with lpc = 1, i.e. chain-major, so consecutive threads read consecutive cells.
constexpr int SCAN_THREADS = 256, SCAN_PER_THREAD = 4, SCAN_BLOCK = SCAN_THREADS * SCAN_PER_THREAD;

struct Affine {            // x -> M x + c, M = [[m00, m01], [m10, m11]]
    double m00, m01, m10, m11, c0, c1;
};
__device__ __forceinline__ Affine affine_identity() { return Affine{1.0, 0.0, 0.0, 1.0, 0.0, 0.0}; }
// second after first: x -> second(first(x))
__device__ __forceinline__ Affine affine_then(const Affine &first, const Affine &second)
{
    Affine r;
    r.m00 = fma(second.m00, first.m00, second.m01 * first.m10);
    r.m01 = fma(second.m00, first.m01, second.m01 * first.m11);
    r.m10 = fma(second.m10, first.m00, second.m11 * first.m10);
    r.m11 = fma(second.m10, first.m01, second.m11 * first.m11);
    r.c0 = fma(second.m00, first.c0, fma(second.m01, first.c1, second.c0));
    r.c1 = fma(second.m10, first.c0, fma(second.m11, first.c1, second.c1));
    return r;
}
__device__ __forceinline__ Affine affine_shfl_up(const Affine &a, int d)
{
    Affine r;
    r.m00 = __shfl_up_sync(0xffffffffu, a.m00, d); r.m01 = __shfl_up_sync(0xffffffffu, a.m01, d);
    r.m10 = __shfl_up_sync(0xffffffffu, a.m10, d); r.m11 = __shfl_up_sync(0xffffffffu, a.m11, d);
    r.c0 = __shfl_up_sync(0xffffffffu, a.c0, d);   r.c1 = __shfl_up_sync(0xffffffffu, a.c1, d);
    return r;
}

__global__ void __launch_bounds__(SCAN_THREADS)
si_scan_reduce_kernel(StopCheck stop, int J, const double *__restrict__ T2, const double *__restrict__ bo,
                      Affine *__restrict__ prefix, Affine *__restrict__ agg)
{
    __shared__ Affine wagg[SCAN_THREADS / 32];
    if (stop_reached(stop)) return;
    const int ch = blockIdx.y, blk = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n_blk = gridDim.x;
    const size_t jj0 = (size_t)blk * SCAN_BLOCK + (size_t)tid * SCAN_PER_THREAD;
    const double *Tp = T2 + ((size_t)ch * J + jj0) * 4;
    const double *bp = bo + ((size_t)ch * J + jj0) * 2;
    Affine a = affine_identity();
#pragma unroll
    for (int u = 0; u < SCAN_PER_THREAD; ++u)
        if (jj0 + u < (size_t)J) {
            const double2 t0 = *reinterpret_cast<const double2 *>(Tp + 4 * u);
            const double2 t1 = *reinterpret_cast<const double2 *>(Tp + 4 * u + 2);
            const double2 bb = *reinterpret_cast<const double2 *>(bp + 2 * u);
            a = affine_then(a, Affine{t0.x, t0.y, t1.x, t1.y, bb.x, bb.y});
        }
    // inclusive scan inside the warp (Hillis-Steele under composition: earlier lanes act first)
    Affine inc = a;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const Affine up = affine_shfl_up(inc, d);
        if (lane >= d) inc = affine_then(up, inc);
    }
    if (lane == 31) wagg[warp] = inc;
    Affine exc = affine_shfl_up(inc, 1);
    if (lane == 0) exc = affine_identity();
    __syncthreads();
    Affine wpre = affine_identity();
    for (int ww = 0; ww < warp; ++ww) wpre = affine_then(wpre, wagg[ww]);
    const Affine pre = affine_then(wpre, exc);              // everything before this thread, inside the block
    prefix[((size_t)ch * n_blk + blk) * SCAN_THREADS + tid] = pre;
    if (tid == SCAN_THREADS - 1) agg[(size_t)ch * n_blk + blk] = affine_then(pre, a);
}

__global__ void __launch_bounds__(SCAN_THREADS)
si_scan_apply_kernel(StopCheck stop, int J, int N, int G, int bc_left, int bc_right, const double *__restrict__ mu,
                     const double *__restrict__ T2, const double *__restrict__ bo, const Affine *__restrict__ prefix,
                     const Affine *__restrict__ agg, const double *__restrict__ psi_old,
                     const double *__restrict__ inc_left, const double *__restrict__ inc_right,
                     double *__restrict__ in_out)
{
    if (stop_reached(stop)) return;
    const int gm = blockIdx.y, blk = blockIdx.x, tid = threadIdx.x, n_blk = gridDim.x;
    const int GN = G * N, n = 4 * GN, g = gm / N, m = gm % N;
    const bool fwd = mu[m] > 0.0;
    double x0 = 0.0, x1 = 0.0;
    const int bc = fwd ? bc_left : bc_right;
    if (bc == OCI_BC_REFLECTIVE) { // mirror ordinate of the boundary cell, from iteration l (A12)
        const double *cellp = psi_old + (fwd ? (size_t)0 : (size_t)(J - 1) * n) + (size_t)(g * N + (N - 1 - m)) * 4;
        x0 = cellp[fwd ? 0 : 1];
        x1 = cellp[fwd ? 2 : 3];
    } else if (bc == OCI_BC_PRESCRIBED) {
        const double *ip = (fwd ? inc_left : inc_right) + (size_t)gm * 2;
        x0 = ip[0];
        x1 = ip[1];
    }
    for (int b = 0; b < blk; ++b) { // the blocks before this one (uniform loads)
        const Affine A = agg[(size_t)gm * n_blk + b];
        const double y0 = fma(A.m00, x0, fma(A.m01, x1, A.c0)), y1 = fma(A.m10, x0, fma(A.m11, x1, A.c1));
        x0 = y0;
        x1 = y1;
    }
    {
        const Affine Pf = prefix[((size_t)gm * n_blk + blk) * SCAN_THREADS + tid];
        const double y0 = fma(Pf.m00, x0, fma(Pf.m01, x1, Pf.c0)), y1 = fma(Pf.m10, x0, fma(Pf.m11, x1, Pf.c1));
        x0 = y0;
        x1 = y1;
    }
    const size_t jj0 = (size_t)blk * SCAN_BLOCK + (size_t)tid * SCAN_PER_THREAD;
    const double *Tp = T2 + ((size_t)gm * J + jj0) * 4;
    const double *bp = bo + ((size_t)gm * J + jj0) * 2;
#pragma unroll
    for (int u = 0; u < SCAN_PER_THREAD; ++u)
        if (jj0 + u < (size_t)J) {
            const size_t jj = jj0 + u, j = fwd ? jj : (size_t)(J - 1) - jj;
            *reinterpret_cast<double2 *>(in_out + (j * GN + gm) * 2) = make_double2(x0, x1);
            const double2 t0 = *reinterpret_cast<const double2 *>(Tp + 4 * u);
            const double2 t1 = *reinterpret_cast<const double2 *>(Tp + 4 * u + 2);
            const double2 bb = *reinterpret_cast<const double2 *>(bp + 2 * u);
            const double y0 = fma(t0.x, x0, fma(t0.y, x1, bb.x)), y1 = fma(t1.x, x0, fma(t1.y, x1, bb.y));
            x0 = y0;
            x1 = y1;
        }
}

// a11 (+ the rest of a10): psi = base + C in for every (j,g,m); phi = sum_m w_m psi_m; residual.
constexpr int FIN_THREADS = 256;
template <bool WANT_L2>
__global__ void __launch_bounds__(FIN_THREADS)
si_finish_kernel(StopCheck stop, int J, int N, int G, const double *__restrict__ w, const double *__restrict__ C,
                 const double *__restrict__ base, const double *__restrict__ in_, double *__restrict__ psi,
                 double *__restrict__ phi, unsigned long long *resid_inf, double *resid_l2)
{
    __shared__ double ws[FIN_THREADS][4];
    if (stop_reached(stop)) return;
    if (blockIdx.x == 0 && threadIdx.x == 0) *stop.executed = stop.slot + 1;
    const int pairs_per_block = FIN_THREADS / N; // (j,g) pairs per block
    const size_t n_pairs = (size_t)J * G;
    const int tid = threadIdx.x, lane = tid & 31;
    double rmax = 0.0, l2 = 0.0;
    for (size_t pair0 = (size_t)blockIdx.x * pairs_per_block; pair0 < n_pairs; pair0 += (size_t)gridDim.x * pairs_per_block) {
        const int local_pair = tid / N, m = tid - local_pair * N;
        const size_t pair = pair0 + local_pair;
        __syncthreads();
        if (local_pair < pairs_per_block && pair < n_pairs) {
            const size_t e = pair * N + m;
            const double i0 = in_[e * 2], i1 = in_[e * 2 + 1];
            const double wm = w[m];
#pragma unroll
            for (int p = 0; p < 4; ++p) {
                const double x = fma(C[e * 8 + p * 2], i0, fma(C[e * 8 + p * 2 + 1], i1, base[e * 4 + p]));
                psi[e * 4 + p] = x;
                ws[tid][p] = wm * x;
            }
        }
        __syncthreads();
        // N = 2 gives 128 pairs per block = 512 (pair, p) entries: stride over them (one pass for N >= 4)
        for (int t = tid; t < pairs_per_block * 4; t += FIN_THREADS) {
            const int lp = t >> 2, p = t & 3;
            if (pair0 + lp >= n_pairs) break;
            double s = 0.0;
            for (int mm = 0; mm < N; ++mm) s += ws[lp * N + mm][p];
            const size_t o = (pair0 + lp) * 4 + p;
            const double d = s - phi[o];
            phi[o] = s;
            const double ad = fabs(d);
            rmax = (ad > rmax || !(ad == ad)) ? ad : rmax;
            if (WANT_L2) l2 = fma(d, d, l2);
        }
    }
    rmax = warp_max(rmax);
    if (lane == 0) atomicMax(resid_inf, resid_bits(rmax));
    if (WANT_L2) {
        l2 = warp_sum(l2);
        if (lane == 0) atomicAdd(resid_l2, l2);
    }
}

inline int grid_for(size_t total, int threads, int num_sms)
{
    size_t g = (total + threads - 1) / threads;
    size_t cap = (size_t)num_sms * 16;
    if (g > cap) g = cap;
    if (g < 1) g = 1;
    return (int)g;
}

} // namespace

// chains (ordinates x groups) per sweep CTA: 4, 8 or 16 ("si_lanes" option; default 8)
static int si_lanes(const oci_ctx *ctx)
{
    if (ctx->opt_si_sweep == 1) return 1; // scan mode: chain-major layout
    const int v = ctx->opt_si_lanes;
    return (v == 4 || v == 16) ? v : 8;
}

int launch_si_setup(oci_ctx *ctx)
{
    ProblemView P = make_view(ctx);
    const size_t total = (size_t)ctx->J * ctx->G * ctx->N;
    si_setup_kernel<<<grid_for(total, 128, ctx->num_sms), 128, 0, ctx->stream>>>(P, si_lanes(ctx), ctx->si_Linv, ctx->si_T,
                                                                                 ctx->si_T2sw);
    OCI_CUDA_TRY(ctx, cudaGetLastError());
    return 1;
}

int launch_si_iteration(oci_ctx *ctx, int hist_slot, bool want_l2, bool check_prev)
{
    ProblemView P = make_view(ctx);
    const StopCheck stop = make_stop(ctx, hist_slot, check_prev);
    const int GN = ctx->G * ctx->N;
    const size_t total = (size_t)ctx->J * GN;
    double *psi = ctx->psi[ctx->cur];
    const int lpc = si_lanes(ctx);
    si_source_kernel<<<grid_for(total, 256, ctx->num_sms), 256, 0, ctx->stream>>>(stop, P, lpc, ctx->q, ctx->psi_prev,
                                                                                   ctx->phi, ctx->si_Linv, ctx->si_base,
                                                                                   ctx->si_bsw);
    OCI_CUDA_TRY(ctx, cudaGetLastError());
    if (ctx->opt_si_sweep == 1) { // f4: the sweep as a parallel scan of the affine edge maps
        const int n_blk = (ctx->J + SCAN_BLOCK - 1) / SCAN_BLOCK;
        if ((size_t)n_blk * GN * (SCAN_THREADS + 1) * sizeof(Affine) > ctx->si_scan_bytes) return OCI_E_WORKSPACE;
        Affine *prefix = reinterpret_cast<Affine *>(ctx->si_scan);
        Affine *agg = prefix + (size_t)n_blk * GN * SCAN_THREADS;
        const dim3 grid(n_blk, GN);
        si_scan_reduce_kernel<<<grid, SCAN_THREADS, 0, ctx->stream>>>(stop, ctx->J, ctx->si_T2sw, ctx->si_bsw, prefix, agg);
        OCI_CUDA_TRY(ctx, cudaGetLastError());
        si_scan_apply_kernel<<<grid, SCAN_THREADS, 0, ctx->stream>>>(stop, ctx->J, ctx->N, ctx->G, ctx->bc_left,
                                                                    ctx->bc_right, ctx->mu, ctx->si_T2sw, ctx->si_bsw, prefix,
                                                                    agg, psi, ctx->inc_left, ctx->inc_right, ctx->si_in);
        OCI_CUDA_TRY(ctx, cudaGetLastError());
    } else {
    const int sweep_grid = (GN + lpc - 1) / lpc;
#define OCI_SWEEP(LPC_)                                                                                            \
    do {                                                                                                           \
        const size_t smem = sizeof(double) * sw_stages(LPC_) * TC * LPC_ * 8 + 3 * sw_stages(LPC_) * sizeof(uint64_t);         \
        OCI_CUDA_TRY(ctx, grant_smem(ctx, SLOT_SWEEP + (LPC_ == 4 ? 0 : (LPC_ == 8 ? 1 : 2)),                       \
                                     (const void *)si_sweep_kernel<LPC_>, smem));                                  \
        si_sweep_kernel<LPC_><<<sweep_grid, SW_THREADS, smem, ctx->stream>>>(                                       \
            stop, ctx->J, ctx->N, ctx->G, ctx->bc_left, ctx->bc_right, ctx->mu, ctx->si_T2sw, ctx->si_bsw, psi,      \
            ctx->inc_left, ctx->inc_right, ctx->si_in);                                                            \
    } while (0)
    if (lpc == 4) OCI_SWEEP(4);
    else if (lpc == 8) OCI_SWEEP(8);
    else OCI_SWEEP(16);
#undef OCI_SWEEP
    OCI_CUDA_TRY(ctx, cudaGetLastError());
    }
    const int pairs_per_block = FIN_THREADS / ctx->N;
    size_t blocks = ((size_t)ctx->J * ctx->G + pairs_per_block - 1) / pairs_per_block;
    if (blocks > (size_t)ctx->num_sms * 16) blocks = (size_t)ctx->num_sms * 16;
    if (want_l2)
        si_finish_kernel<true><<<(int)blocks, FIN_THREADS, 0, ctx->stream>>>(stop, ctx->J, ctx->N, ctx->G, ctx->w, ctx->si_T,
                                                                            ctx->si_base, ctx->si_in, psi, ctx->phi,
                                                                            ctx->resid_inf + hist_slot,
                                                                            ctx->resid_l2 + hist_slot);
    else
        si_finish_kernel<false><<<(int)blocks, FIN_THREADS, 0, ctx->stream>>>(stop, ctx->J, ctx->N, ctx->G, ctx->w, ctx->si_T,
                                                                             ctx->si_base, ctx->si_in, psi, ctx->phi,
                                                                             ctx->resid_inf + hist_slot,
                                                                             ctx->resid_l2 + hist_slot);
    OCI_CUDA_TRY(ctx, cudaGetLastError());
    return ctx->opt_si_sweep == 1 ? 4 : 3;
}
