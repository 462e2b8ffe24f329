// iterate.cu -- a3..a8 of SURVEY.md section 8(a): constant RHS, the fused per-iteration OCI kernel
// (gather incident edge fluxes + RHS + cell solve + scalar flux + residual), advance.
//
// One OCI iteration (Eq. 7; Alg. 2), for every cell j independently:
//   b_j = c_j + incident(Psi^(l))    Eq. 9c-d: rows (k,L),(k+1/2,L) of an ordinate with mu>0 get
//                                    +mu psi^(l)_{j-1,R}; rows (k,R),(k+1/2,R) of mu<0 get +|mu| psi^(l)_{j+1,L}
//   Psi_j^(l+1) = A_j^{-1} b_j       the `_getrs` of Alg. 2, here a streamed matrix-vector product with the
//                                    inverse oci_factor stored (same n^2 doubles, same 2 n^2 flops, no chain)
//   phi_j = sum_m w_m psi_m          Eq. 44
//   r = max |phi^(l+1) - phi^(l)|    (and sum (Psi^(l+1)-Psi^(l))^2 for Eq. 12)
// The kernel is HBM-bound: 8 n^2 bytes of A_j^{-1} per cell-solve against 2 n^2 flops. It therefore runs as
// a persistent, warp-specialised streaming kernel: one producer thread per CTA issues 1-D bulk async copies
// (cp.async.bulk, completion on mbarriers) into multi-stage shared-memory rings and the consumer warps multiply
// the chunks as they land: oci_iterate_wpc_kernel (n = 64, 128, 256: a cell per consumer warp, the production
// kernel of configs 3-5) and oci_iterate_stream_kernel (any other n: a team of threads per cell).
#include "common.cuh"
#include <cooperative_groups.h>

namespace {

constexpr int CONSUMER_WARPS = 8;
constexpr int CONSUMERS = CONSUMER_WARPS * 32;       // 256
constexpr int ITER_THREADS = CONSUMERS + 32;         // + 1 producer warp
constexpr int VEC_SLOTS = 2;
constexpr int MAX_STAGES = 8;

__device__ __forceinline__ void consumer_bar()
{
    asm volatile("bar.sync 1, %0;" ::"n"(CONSUMERS) : "memory");
}

// ---- incident edge flux of entry (cell j, row i) taken from Psi^(l) ------------------------------------------
// `nb` holds Psi^(l) of cells j0-1 .. j0+nc (cell j at nb + (j - j0 + 1) * n); returns coefficient * value.
__device__ __forceinline__ double incident_term(const IterParams &P, const double *nb, int j0, int j, int i,
                                                const double *mu_s)
{
    const int n = P.n, N = P.N;
    const int p = i & 3, bm = i >> 2, m = bm % N, g = bm / N;
    const double mu = mu_s[m];
    const double *self = nb + (size_t)(j - j0 + 1) * n;
    if (mu > 0.0 && !(p & 1)) { // rows (k,L), (k+1/2,L): upstream = (j-1, R), Eq. 5a / 9c
        double val;
        if (j > 0) val = (self - n)[i + 1];
        else if (P.bc_left == OCI_BC_REFLECTIVE) val = self[(g * N + (N - 1 - m)) * 4 + p];
        else if (P.bc_left == OCI_BC_PRESCRIBED) val = P.inc_left[(g * N + m) * 2 + (p >> 1)];
        else val = 0.0;
        return mu * val;
    }
    if (mu < 0.0 && (p & 1)) { // rows (k,R), (k+1/2,R): upstream = (j+1, L), Eq. 5b / 9d
        double val;
        if (j < P.J - 1) val = (self + n)[i - 1];
        else if (P.bc_right == OCI_BC_REFLECTIVE) val = self[(g * N + (N - 1 - m)) * 4 + p];
        else if (P.bc_right == OCI_BC_PRESCRIBED) val = P.inc_right[(g * N + m) * 2 + (p >> 1)];
        else val = 0.0;
        return -mu * val;
    }
    return 0.0;
}

// ============================================================================================================
// Pipelined streaming kernel
// ============================================================================================================
// Work item = `cpb` consecutive cells (cpb > 1 only for small n, where several whole inverses fit one chunk)
// = `nch` chunks of the inverse (column panels of `cw` columns when one cell spans several chunks).
// Consumer thread t of a cell team (team size n*S) owns row r = t % n and the columns c = sub (mod S),
// sub = t / n: with the column-major inverse every step of a team reads S*n consecutive doubles, so shared
// memory reads are conflict-free and the global layout needs no swizzle.
template <bool WANT_L2>
__global__ void __launch_bounds__(ITER_THREADS, 1) oci_iterate_stream_kernel(const IterParams P)
{
    if (stop_reached(P.stop)) return;
    if (blockIdx.x == 0 && threadIdx.x == 0) *P.stop.executed = P.stop.slot + 1;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int n = P.n, N = P.N, G = P.G, J = P.J;
    const int cpb = P.cpb, S = P.S, nch = P.nch, stages = P.stages;
    const int vec_c = cpb * n, vec_nb = (cpb + 2) * n;

    uint64_t *mat_full = reinterpret_cast<uint64_t *>(smem_raw);
    uint64_t *mat_empty = mat_full + MAX_STAGES;
    uint64_t *vec_full = mat_empty + MAX_STAGES;
    uint64_t *vec_empty = vec_full + VEC_SLOTS;
    double *mu_s = reinterpret_cast<double *>(vec_empty + VEC_SLOTS); // [N]
    double *w_s = mu_s + N;                                          // [N]
    double *part = w_s + N;                                          // [CONSUMERS]
    double *xbuf = part + CONSUMERS;                                 // [CONSUMERS]
    size_t off = (size_t)((unsigned char *)(xbuf + CONSUMERS) - smem_raw);
    off = (off + 127) & ~(size_t)127;
    double *vec = reinterpret_cast<double *>(smem_raw + off);        // VEC_SLOTS x (vec_c + vec_nb)
    off += (size_t)VEC_SLOTS * (vec_c + vec_nb) * sizeof(double);
    off = (off + 127) & ~(size_t)127;
    double *mat = reinterpret_cast<double *>(smem_raw + off);        // stages x chunk_doubles

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

    if (tid == 0) {
        for (int s = 0; s < stages; ++s) { mbar_init(&mat_full[s], 1); mbar_init(&mat_empty[s], CONSUMER_WARPS); }
        for (int s = 0; s < VEC_SLOTS; ++s) { mbar_init(&vec_full[s], 1); mbar_init(&vec_empty[s], CONSUMER_WARPS); }
        fence_mbar_init();
    }
    for (int i = tid; i < N; i += ITER_THREADS) { mu_s[i] = P.mu[i]; w_s[i] = P.w[i]; }
    __syncthreads();

    // balanced contiguous split of the items over the CTAs
    const int item0 = (int)(((long long)P.n_items * blockIdx.x) / gridDim.x);
    const int item1 = (int)(((long long)P.n_items * (blockIdx.x + 1)) / gridDim.x);

    if (warp == CONSUMER_WARPS) {
        // ===================== producer: one thread issues every bulk copy ===============================
        if (lane == 0) {
            int ms = 0, vs = 0;
            uint32_t mph = 0, vph = 0;
            for (int item = item0; item < item1; ++item) {
                const int j0 = item * cpb;
                const int nc = min(cpb, J - j0);
                // vectors: c_j of the item's cells, Psi^(l) of the cells and their two neighbours
                mbar_wait(&vec_empty[vs], vph ^ 1);
                {
                    double *cs = vec + (size_t)vs * (vec_c + vec_nb);
                    double *nb = cs + vec_c;
                    const int lo = max(j0 - 1, 0), hi = min(j0 + nc, J - 1);
                    const uint32_t bytes_c = (uint32_t)(nc * n * sizeof(double));
                    const uint32_t bytes_nb = (uint32_t)((hi - lo + 1) * n * sizeof(double));
                    mbar_arrive_expect_tx(&vec_full[vs], bytes_c + bytes_nb);
                    bulk_g2s(cs, P.c + (size_t)j0 * n, bytes_c, &vec_full[vs]);
                    bulk_g2s(nb + (size_t)(lo - (j0 - 1)) * n, P.psi_old + (size_t)lo * n, bytes_nb, &vec_full[vs]);
                }
                if (++vs == VEC_SLOTS) { vs = 0; vph ^= 1; }
                // matrix chunks
                const double *src0 = P.Minv + (size_t)j0 * n * n;
                for (int ch = 0; ch < nch; ++ch) {
                    mbar_wait(&mat_empty[ms], mph ^ 1);
                    uint32_t bytes;
                    const double *src;
                    if (nch == 1) { src = src0; bytes = (uint32_t)((size_t)nc * n * n * sizeof(double)); }
                    else {
                        const int c0 = ch * P.cw, ncol = min(P.cw, n - c0);
                        src = src0 + (size_t)c0 * n;
                        bytes = (uint32_t)((size_t)ncol * n * sizeof(double));
                    }
                    mbar_arrive_expect_tx(&mat_full[ms], bytes);
                    bulk_g2s(mat + (size_t)ms * P.chunk_doubles, src, bytes, &mat_full[ms]);
                    if (++ms == stages) { ms = 0; mph ^= 1; }
                }
            }
        }
        return;
    }

    // ========================= consumers ====================================================================
    const int TS = n * S;                 // threads of one cell team
    const int team = tid / TS;            // cell within the item
    const int tt = tid - team * TS;
    const int sub = tt / n, r = tt - sub * n;
    const bool in_team = team < cpb;      // false: idle in the product phase (n*S*cpb < 256)

    int ms = 0, vs = 0;
    uint32_t mph = 0, vph = 0;
    double rmax = 0.0, l2 = 0.0;

    for (int item = item0; item < item1; ++item) {
        const int j0 = item * cpb;
        const int nc = min(cpb, J - j0);
        double *cs = vec + (size_t)vs * (vec_c + vec_nb);
        const double *nb = cs + vec_c;

        // ---- a4: b = c + incident(Psi^(l)), in place over c
        mbar_wait(&vec_full[vs], vph);
        for (int e = tid; e < nc * n; e += CONSUMERS) {
            const int a = e / n, i = e - a * n;
            cs[e] += incident_term(P, nb, j0, j0 + a, i, mu_s);
        }
        consumer_bar();

        // ---- a5: x = A^{-1} b, chunk by chunk
        double acc0 = 0.0, acc1 = 0.0;
        for (int ch = 0; ch < nch; ++ch) {
            mbar_wait(&mat_full[ms], mph);
            if (in_team && team < nc) {
                int c0 = 0, ncol = n;
                if (nch > 1) { c0 = ch * P.cw; ncol = min(P.cw, n - c0); }
                const double *Mp = mat + (size_t)ms * P.chunk_doubles + (size_t)team * n * n + r;
                const double *bp = cs + team * n + c0;
                int cc = sub;
#pragma unroll 4
                for (; cc + S < ncol; cc += 2 * S) {
                    acc0 = fma(Mp[(size_t)cc * n], bp[cc], acc0);
                    acc1 = fma(Mp[(size_t)(cc + S) * n], bp[cc + S], acc1);
                }
                if (cc < ncol) acc0 = fma(Mp[(size_t)cc * n], bp[cc], acc0);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&mat_empty[ms]);
            if (++ms == stages) { ms = 0; mph ^= 1; }
        }
        part[tid] = acc0 + acc1;
        consumer_bar();

        // ---- combine the column sub-groups; write Psi^(l+1)
        for (int e = tid; e < nc * n; e += CONSUMERS) {
            const int a = e / n, i = e - a * n;
            double x = 0.0;
            for (int s = 0; s < S; ++s) x += part[a * TS + s * n + i];
            xbuf[e] = x;
            P.psi_new[(size_t)j0 * n + e] = x;
            if (WANT_L2) { const double d = x - nb[(a + 1) * n + i]; l2 = fma(d, d, l2); }
        }
        consumer_bar();

        // ---- a6 + a7: phi = sum_m w_m psi_m for the new and the previous iterate, residual
        for (int e = tid; e < nc * G * 4; e += CONSUMERS) {
            const int p = e & 3, ag = e >> 2, g = ag % G, a = ag / G;
            const double *xn = xbuf + a * n + g * N * 4 + p;
            const double *xo = nb + (a + 1) * n + g * N * 4 + p;
            double sn = 0.0, so = 0.0;
            for (int m = 0; m < N; ++m) { sn = fma(w_s[m], xn[m * 4], sn); so = fma(w_s[m], xo[m * 4], so); }
            P.phi[(size_t)j0 * G * 4 + e] = sn;
            const double d = fabs(sn - so);
            rmax = (d > rmax || !(d == d)) ? d : rmax;
        }
        // the slot was written through the generic proxy (b in place of c) and is refilled by bulk copies
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp();
        if (lane == 0) mbar_arrive(&vec_empty[vs]);
        if (++vs == VEC_SLOTS) { vs = 0; vph ^= 1; }
    }

    rmax = warp_max(rmax);
    if (lane == 0 && item1 > item0) atomicMax(P.resid_inf, resid_bits(rmax));
    if (WANT_L2) {
        l2 = warp_sum(l2);
        if (lane == 0 && item1 > item0) atomicAdd(P.resid_l2, l2);
    }
}

// ============================================================================================================
// Warp-per-cell streaming kernel (n = 64, 128, 256): the production path for the large configurations.
// ============================================================================================================
// Every consumer warp owns one cell at a time: lane l holds the rows {64 q + 2 l, 64 q + 2 l + 1}, q < RPL/2, of
// x = A^{-1} b in registers, so a column of the inverse is RPL/2 conflict-free 16-byte shared-memory loads per
// lane and the product needs no cross-warp reduction, no CTA-wide barrier and no shuffles. A cell spans
// NCH = n / CW chunks (column panels of CW = 2048 / n columns, 16 KB each); the producer interleaves the chunks
// of WC consecutive cells (one per consumer warp) so that all warps stream concurrently. The per-cell prologue (b = c + incident) and epilogue (Psi store, phi, residual)
// are warp-local as well, so the only synchronisation is the mbarrier handshake with the bulk-copy engine.
// Every consumer warp has its OWN ring of `spw` stages (single producer, single consumer per mbarrier): a shared
// ring would let a warp test a stage's parity one phase early and read a chunk that has not landed.
constexpr int WPC_WARPS = 4;                      // consumer warps (one per SM sub-partition)
constexpr int WPC_THREADS = (WPC_WARPS + 1) * 32;
constexpr int WPC_VEC_SLOTS = 2;
constexpr int WPC_CHUNK = 2048;                   // doubles per chunk (16 KB)
constexpr int WPC_MAX_STAGES = 16;                // WPC_WARPS x stages per warp

template <int RPL, bool WANT_L2>
__global__ void __launch_bounds__(WPC_THREADS, 1) oci_iterate_wpc_kernel(const IterParams P)
{
    pdl_launch_dependents(); // (see launch_pdl: everything up to pdl_wait() below touches constant inputs only)
    constexpr int n = 32 * RPL;
    constexpr int CW = WPC_CHUNK / n;   // columns per chunk
    constexpr int NCH = n / CW;         // chunks per cell
    constexpr int HQ = RPL / 2;         // 16-byte loads per lane per column
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int N = P.N, G = P.G, J = P.J, spw = P.stages; // stages per consumer warp
    constexpr int vec_c = WPC_WARPS * n, vec_nb = (WPC_WARPS + 2) * n;

    uint64_t *mat_full = reinterpret_cast<uint64_t *>(smem_raw);
    uint64_t *mat_empty = mat_full + WPC_MAX_STAGES;
    uint64_t *vec_full = mat_empty + WPC_MAX_STAGES;
    uint64_t *vec_empty = vec_full + WPC_VEC_SLOTS;
    double *mu_s = reinterpret_cast<double *>(vec_empty + WPC_VEC_SLOTS); // [N]
    double *w_s = mu_s + N;                                              // [N]
    size_t off = (size_t)((unsigned char *)(w_s + N) - smem_raw);
    off = (off + 127) & ~(size_t)127;
    double *vec = reinterpret_cast<double *>(smem_raw + off);            // WPC_VEC_SLOTS x (vec_c + vec_nb)
    off += (size_t)WPC_VEC_SLOTS * (vec_c + vec_nb) * sizeof(double);
    off = (off + 127) & ~(size_t)127;
    double *mat = reinterpret_cast<double *>(smem_raw + off);            // [WPC_WARPS][spw] x WPC_CHUNK

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (tid == 0) {
        for (int s = 0; s < WPC_WARPS * spw; ++s) { mbar_init(&mat_full[s], 1); mbar_init(&mat_empty[s], 1); }
        for (int s = 0; s < WPC_VEC_SLOTS; ++s) { mbar_init(&vec_full[s], 1); mbar_init(&vec_empty[s], WPC_WARPS); }
        fence_mbar_init();
    }
    for (int i = tid; i < N; i += WPC_THREADS) { mu_s[i] = P.mu[i]; w_s[i] = P.w[i]; }
    __syncthreads();
    pdl_wait(); // the previous iteration (or whatever precedes on the stream) is complete from here on
    if (stop_reached(P.stop)) return;
    if (blockIdx.x == 0 && threadIdx.x == 0) *P.stop.executed = P.stop.slot + 1;

    // balanced contiguous split of the cells over the CTAs
    const int cell0 = (int)(((long long)J * blockIdx.x) / gridDim.x);
    const int cell1 = (int)(((long long)J * (blockIdx.x + 1)) / gridDim.x);
    // Successive iterations walk the range in opposite directions (P.reverse = parity of the history slot): a Jacobi
    // iteration does not care about the order of its cells, and the inverses, c and Psi a CTA touched last in iteration l
    // are then the first it asks for in iteration l + 1, while they are still in the L2 (126 MB against 2.1 GB of
    // inverses on config 5: a per cent of the stream, for nothing). Slot 0 walks down: oci_factor writes the inverses
    // in ascending order. Walking down, the groups of WPC_WARPS cells are counted from the top, so that the ragged
    // group is the LAST one in either direction (a warp without a cell skips its ring slots, which is only
    // consistent with the producer's parities when nothing follows).
    const int ngroups = (cell1 - cell0 + WPC_WARPS - 1) / WPC_WARPS;

    if (warp == WPC_WARPS) {
        // ===================== producer ==================================================================
        if (lane == 0) {
            int vs = 0;
            uint32_t vph = 0;
            unsigned it = 0; // chunk round: every warp with a cell gets one chunk per round
            for (int gi = 0; gi < ngroups; ++gi) {
                const int gb = P.reverse ? max(cell0, cell1 - WPC_WARPS * (gi + 1)) : cell0 + WPC_WARPS * gi;
                const int nv = P.reverse ? cell1 - WPC_WARPS * gi - gb : min(WPC_WARPS, cell1 - gb);
                mbar_wait(&vec_empty[vs], vph ^ 1);
                {
                    double *cs = vec + (size_t)vs * (vec_c + vec_nb);
                    double *nb = cs + vec_c;
                    const int lo = max(gb - 1, 0), hi = min(gb + nv, J - 1);
                    const uint32_t bytes_c = (uint32_t)(nv * n * sizeof(double));
                    const uint32_t bytes_nb = (uint32_t)((hi - lo + 1) * n * sizeof(double));
                    mbar_arrive_expect_tx(&vec_full[vs], bytes_c + bytes_nb);
                    bulk_g2s(cs, P.c + (size_t)gb * n, bytes_c, &vec_full[vs]);
                    bulk_g2s(nb + (size_t)(lo - (gb - 1)) * n, P.psi_old + (size_t)lo * n, bytes_nb, &vec_full[vs]);
                }
                if (++vs == WPC_VEC_SLOTS) { vs = 0; vph ^= 1; }
                for (int k = 0; k < NCH; ++k, ++it) {
                    const int slot = it % spw;
                    const uint32_t ph = (it / spw) & 1;
                    for (int w = 0; w < nv; ++w) {
                        const int st = w * spw + slot;
                        mbar_wait(&mat_empty[st], ph ^ 1);
                        mbar_arrive_expect_tx(&mat_full[st], WPC_CHUNK * sizeof(double));
                        bulk_g2s(mat + (size_t)st * WPC_CHUNK, P.Minv + (size_t)(gb + w) * n * n + (size_t)k * CW * n,
                                 WPC_CHUNK * sizeof(double), &mat_full[st]);
                    }
                }
            }
        }
        return;
    }

    // ========================= consumer warps ===============================================================
    int vs = 0;
    uint32_t vph = 0;
    unsigned it = 0;
    double rmax = 0.0, l2 = 0.0;
    for (int gi = 0; gi < ngroups; ++gi) {
        const int gb = P.reverse ? max(cell0, cell1 - WPC_WARPS * (gi + 1)) : cell0 + WPC_WARPS * gi;
        const int nv = P.reverse ? cell1 - WPC_WARPS * gi - gb : min(WPC_WARPS, cell1 - gb);
        double *cs = vec + (size_t)vs * (vec_c + vec_nb);
        const double *nb = cs + vec_c;
        mbar_wait(&vec_full[vs], vph);
        if (warp < nv) {
            const int j = gb + warp;
            double *bs = cs + warp * n;                 // this warp's c_j, turned into b_j in place (a4)
            const double *own = nb + (warp + 1) * n;     // Psi^(l) of this cell
            for (int i = lane; i < n; i += 32) bs[i] += incident_term(P, nb, gb, j, i, mu_s);
            __syncwarp();

            // ---- a5: x = A^{-1} b
            double acc[2][RPL];
#pragma unroll
            for (int r = 0; r < RPL; ++r) { acc[0][r] = 0.0; acc[1][r] = 0.0; }
            for (int k = 0; k < NCH; ++k) {
                const unsigned r = it + (unsigned)k;
                const int st = warp * spw + (int)(r % spw);
                mbar_wait(&mat_full[st], (r / spw) & 1);
                const double2 *Mp = reinterpret_cast<const double2 *>(mat + (size_t)st * WPC_CHUNK) + lane;
                const double2 *bp = reinterpret_cast<const double2 *>(bs + k * CW);
#pragma unroll 4
                for (int cc = 0; cc < CW; cc += 2) {
                    const double2 bv = bp[cc >> 1];
#pragma unroll
                    for (int q = 0; q < HQ; ++q) {
                        const double2 m0 = Mp[(cc * n) / 2 + q * 32];
                        const double2 m1 = Mp[((cc + 1) * n) / 2 + q * 32];
                        acc[0][2 * q] = fma(m0.x, bv.x, acc[0][2 * q]);
                        acc[0][2 * q + 1] = fma(m0.y, bv.x, acc[0][2 * q + 1]);
                        acc[1][2 * q] = fma(m1.x, bv.y, acc[1][2 * q]);
                        acc[1][2 * q + 1] = fma(m1.y, bv.y, acc[1][2 * q + 1]);
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&mat_empty[st]);
            }

            // ---- Psi^(l+1): rows 64 q + 2 lane, + 1; kept in shared memory (over b) for the phi reduction
            double2 *xs2 = reinterpret_cast<double2 *>(bs);
            double2 *out2 = reinterpret_cast<double2 *>(P.psi_new + (size_t)j * n);
#pragma unroll
            for (int q = 0; q < HQ; ++q) {
                const double2 x = make_double2(acc[0][2 * q] + acc[1][2 * q], acc[0][2 * q + 1] + acc[1][2 * q + 1]);
                if (WANT_L2) {
                    const double2 o = reinterpret_cast<const double2 *>(own)[q * 32 + lane];
                    const double d0 = x.x - o.x, d1 = x.y - o.y;
                    l2 = fma(d0, d0, l2);
                    l2 = fma(d1, d1, l2);
                }
                xs2[q * 32 + lane] = x;
                out2[q * 32 + lane] = x;
            }
            __syncwarp();

            // ---- a6 + a7: phi of the new and of the previous iterate, residual
            for (int e = lane; e < G * 4; e += 32) {
                const int p = e & 3, g = e >> 2;
                const double *xn = bs + g * N * 4 + p;
                const double *xo = own + g * N * 4 + p;
                double sn = 0.0, so = 0.0;
                for (int m = 0; m < N; ++m) { sn = fma(w_s[m], xn[m * 4], sn); so = fma(w_s[m], xo[m * 4], so); }
                P.phi[(size_t)j * G * 4 + e] = sn;
                const double d = fabs(sn - so);
                rmax = (d > rmax || !(d == d)) ? d : rmax;
            }
        }
        it += NCH;
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp();
        if (lane == 0) mbar_arrive(&vec_empty[vs]);
        if (++vs == WPC_VEC_SLOTS) { vs = 0; vph ^= 1; }
    }
    rmax = warp_max(rmax);
    if (lane == 0 && cell1 > cell0) atomicMax(P.resid_inf, resid_bits(rmax));
    if (WANT_L2) {
        l2 = warp_sum(l2);
        if (lane == 0 && cell1 > cell0) atomicAdd(P.resid_l2, l2);
    }
}

// ============================================================================================================
// Plain kernel: one CTA per cell, loads straight from global memory. Used for cross-checking the pipelined
// kernel and selectable with oci_set_option("iterate_kernel", 0).
// ============================================================================================================
template <bool WANT_L2>
__global__ void __launch_bounds__(256) oci_iterate_plain_kernel(const IterParams P)
{
    if (stop_reached(P.stop)) return;
    if (blockIdx.x == 0 && threadIdx.x == 0) *P.stop.executed = P.stop.slot + 1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int n = P.n, N = P.N, G = P.G, J = P.J;
    double *b = reinterpret_cast<double *>(smem_raw); // [n]
    double *x = b + n;                                // [n]
    double *nb = x + n;                               // [3n] Psi^(l) of cells j-1, j, j+1
    double *mu_s = nb + 3 * n;                        // [N]
    double *w_s = mu_s + N;
    const int tid = threadIdx.x, lane = tid & 31;
    for (int i = tid; i < N; i += blockDim.x) { mu_s[i] = P.mu[i]; w_s[i] = P.w[i]; }
    double rmax = 0.0, l2 = 0.0;
    for (int j = blockIdx.x; j < J; j += gridDim.x) {
        __syncthreads();
        for (int e = tid; e < 3 * n; e += blockDim.x) {
            const int jj = j - 1 + e / n;
            nb[e] = (jj >= 0 && jj < J) ? P.psi_old[(size_t)jj * n + (e % n)] : 0.0;
        }
        __syncthreads();
        for (int i = tid; i < n; i += blockDim.x) b[i] = P.c[(size_t)j * n + i] + incident_term(P, nb, j, j, i, mu_s);
        __syncthreads();
        const double *M = P.Minv + (size_t)j * n * n;
        for (int i = tid; i < n; i += blockDim.x) {
            double acc = 0.0;
            for (int c = 0; c < n; ++c) acc = fma(M[(size_t)c * n + i], b[c], acc);
            x[i] = acc;
            P.psi_new[(size_t)j * n + i] = acc;
            if (WANT_L2) { const double d = acc - nb[n + i]; l2 = fma(d, d, l2); }
        }
        __syncthreads();
        for (int e = tid; e < G * 4; e += blockDim.x) {
            const int p = e & 3, g = e >> 2;
            double sn = 0.0, so = 0.0;
            for (int m = 0; m < N; ++m) {
                sn = fma(w_s[m], x[(g * N + m) * 4 + p], sn);
                so = fma(w_s[m], nb[n + (g * N + m) * 4 + p], so);
            }
            P.phi[(size_t)j * G * 4 + e] = sn;
            const double d = fabs(sn - so);
            rmax = (d > rmax || !(d == d)) ? d : rmax;
        }
    }
    rmax = warp_max(rmax);
    if (lane == 0) atomicMax(P.resid_inf, resid_bits(rmax));
    if (WANT_L2) {
        l2 = warp_sum(l2);
        if (lane == 0) atomicAdd(P.resid_l2, l2);
    }
}

// ============================================================================================================
// SURVEY 8(f) row f2, dense path: resident multi-iteration kernel for problems whose inverses fit in the shared memory
// of the chip (BASELINE.json configs 1-2: 32 KB and 8.4 MB of A_j^{-1}).
// ============================================================================================================
// PAPER.md:413-415 notes that on small problems the iteration loop is bound by dispatch, not by work. Here ONE
// cooperative launch runs up to n_iters block-Jacobi iterations: every CTA copies the inverses and the constant
// right-hand sides of its contiguous range of cells into shared memory ONCE and keeps them there, an iteration reads
// only Psi^(l) of its cells and their two neighbours (written by other CTAs of the same launch: past the L1), and a
// grid-wide barrier separates the iterations. Same arithmetic per cell as the other dense kernels, same device-side
// stop: after the barrier every thread of the grid reads the same residual slot and takes the same decision.
struct DenseMulti {
    int n_iters, slot0, check_between, rule, cpc; // cpc: cells per CTA
    double tol;
    unsigned long long *resid_inf; // history base (slot 0)
    double *resid_l2;
    int *executed;
};

template <bool WANT_L2>
__global__ void __launch_bounds__(256) oci_iterate_resident_kernel(const IterParams P, const DenseMulti M)
{
    extern __shared__ __align__(16) unsigned char rs_smem[];
    cooperative_groups::grid_group grid = cooperative_groups::this_grid();
    const int n = P.n, N = P.N, G = P.G, J = P.J, cpc = M.cpc;
    const int cell0 = blockIdx.x * cpc, nc = max(0, min(cpc, J - cell0));
    double *Ms = reinterpret_cast<double *>(rs_smem);   // [cpc][n(col)][n(row)]
    double *cs = Ms + (size_t)cpc * n * n;               // [cpc][n]   c_j
    double *bs = cs + (size_t)cpc * n;                   // [cpc][n]   b_j, then Psi^(l+1)
    double *nb = bs + (size_t)cpc * n;                   // [cpc + 2][n] Psi^(l) of cells cell0 - 1 .. cell0 + cpc
    double *mu_s = nb + (size_t)(cpc + 2) * n;           // [N]
    double *w_s = mu_s + N;                              // [N]
    double *red = w_s + N;                               // [8] block reduction scratch
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int i = tid; i < N; i += blockDim.x) { mu_s[i] = P.mu[i]; w_s[i] = P.w[i]; }
    for (size_t e = tid; e < (size_t)nc * n * n; e += blockDim.x) Ms[e] = P.Minv[(size_t)cell0 * n * n + e];
    for (int e = tid; e < nc * n; e += blockDim.x) cs[e] = P.c[(size_t)cell0 * n + e];
    const double *psi_old = P.psi_old;
    double *psi_new = P.psi_new;
    for (int it = 0; it < M.n_iters; ++it) {
        const int slot = M.slot0 + it;
        if (M.check_between && it > 0) {
            StopCheck st;
            st.prev_inf = M.resid_inf + slot - 1;
            st.prev_l2 = M.resid_l2 + slot - 1;
            st.prev2_l2 = slot >= 2 ? M.resid_l2 + slot - 2 : nullptr;
            st.tol = M.tol; st.rule = M.rule; st.slot = slot; st.executed = M.executed;
            if (stop_reached_t<true>(st)) break; // same values everywhere: the whole grid leaves together
        }
        if (blockIdx.x == 0 && tid == 0) *M.executed = slot + 1;
        // Psi^(l) of the own cells and the two neighbours (zeros outside the slab; boundary cells use the BC instead)
        for (int e = tid; e < (nc + 2) * n; e += blockDim.x) {
            const int jj = cell0 - 1 + e / n;
            nb[e] = (jj >= 0 && jj < J) ? __ldcg(psi_old + (size_t)jj * n + (e % n)) : 0.0;
        }
        __syncthreads();
        for (int e = tid; e < nc * n; e += blockDim.x) // a4: b = c + incident(Psi^(l))
            bs[e] = cs[e] + incident_term(P, nb, cell0, cell0 + e / n, e % n, mu_s);
        __syncthreads();
        double rmax = 0.0, l2 = 0.0, x_first = 0.0;
        for (int e = tid; e < nc * n; e += blockDim.x) { // a5: x = A^{-1} b (one entry per thread at the intended sizes)
            const int a = e / n, i = e - a * n;
            const double *Mp = Ms + (size_t)a * n * n + i, *bp = bs + a * n;
            double acc0 = 0.0, acc1 = 0.0, acc2 = 0.0, acc3 = 0.0;
            int c = 0;
            for (; c + 3 < n; c += 4) {
                acc0 = fma(Mp[(size_t)c * n], bp[c], acc0);
                acc1 = fma(Mp[(size_t)(c + 1) * n], bp[c + 1], acc1);
                acc2 = fma(Mp[(size_t)(c + 2) * n], bp[c + 2], acc2);
                acc3 = fma(Mp[(size_t)(c + 3) * n], bp[c + 3], acc3);
            }
            for (; c < n; ++c) acc0 = fma(Mp[(size_t)c * n], bp[c], acc0);
            const double x = (acc0 + acc1) + (acc2 + acc3);
            if (e == tid) x_first = x;
            psi_new[(size_t)cell0 * n + e] = x;
            if (WANT_L2) { const double d = x - nb[n + e]; l2 = fma(d, d, l2); }
        }
        __syncthreads(); // everybody has read bs: it now receives Psi^(l+1) for the phi reduction
        for (int e = tid; e < nc * n; e += blockDim.x) bs[e] = e == tid ? x_first : psi_new[(size_t)cell0 * n + e];
        __syncthreads();
        for (int e = tid; e < nc * G * 4; e += blockDim.x) { // a6 + a7
            const int p = e & 3, ag = e >> 2, g = ag % G, a = ag / G;
            const double *xn = bs + a * n + g * N * 4 + p, *xo = nb + (a + 1) * n + g * N * 4 + p;
            double sn = 0.0, so = 0.0;
            for (int m = 0; m < N; ++m) { sn = fma(w_s[m], xn[m * 4], sn); so = fma(w_s[m], xo[m * 4], so); }
            P.phi[(size_t)cell0 * G * 4 + e] = sn;
            const double d = fabs(sn - so);
            rmax = (d > rmax || !(d == d)) ? d : rmax;
        }
        rmax = warp_max(rmax);
        if (lane == 0) red[warp] = rmax;
        if (WANT_L2) { l2 = warp_sum(l2); if (lane == 0 && nc > 0) atomicAdd(M.resid_l2 + slot, l2); }
        __syncthreads();
        if (tid == 0 && nc > 0) {
            double r = red[0];
            for (int q = 1; q < (int)(blockDim.x >> 5); ++q) r = (red[q] > r || !(red[q] == red[q])) ? red[q] : r;
            atomicMax(M.resid_inf + slot, resid_bits(r));
        }
        grid.sync();
        const double *t = psi_old;
        psi_old = psi_new;
        psi_new = const_cast<double *>(t);
    }
}

// ---- a3: constant part of b_j (Eq. 9c-d without the incident terms; 4th row of 9c restored,
// DESIGN.md A1): rows (k,L),(k,R): dx/4 Q_k + dx/(2 v dt) psi_{k-1/2}; rows (k+1/2,L),(k+1/2,R): dx/4 Q_{k+1/2}
__global__ void const_rhs_kernel(ProblemView P, const double *__restrict__ q, const double *__restrict__ psi_prev,
                                 double *__restrict__ c)
{
    const size_t total = (size_t)P.J * P.n;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (size_t)gridDim.x * blockDim.x) {
        const int p = (int)(e & 3);
        const size_t jgm = e >> 2;
        const size_t jg = jgm / P.N;
        const int g = (int)(jg % P.G);
        const size_t j = jg / P.G;
        const double dx = P.dx[j];
        double val = dx * 0.25 * q[jg * 4 + p];
        if (p < 2) val += dx / (2.0 * P.v[g] * P.dt) * psi_prev[jgm * 2 + p];
        c[e] = val;
    }
}

// ---- a8: psi_{k-1/2} <- psi_{k+1/2} of the converged iterate
__global__ void advance_kernel(size_t n_pairs, const double *__restrict__ psi, double *__restrict__ psi_prev)
{
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n_pairs * 2; e += (size_t)gridDim.x * blockDim.x)
        psi_prev[e] = psi[(e >> 1) * 4 + 2 + (e & 1)];
}

// iterate <- both time levels = psi_{k-1/2} (A11)
__global__ void seed_iterate_kernel(size_t n_pairs, const double *__restrict__ psi_prev, double *__restrict__ psi)
{
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n_pairs * 4; e += (size_t)gridDim.x * blockDim.x)
        psi[e] = psi_prev[(e >> 2) * 2 + (e & 1)];
}

// Eq. 44: phi[j][g][p] = sum_m w_m psi[j][g][m][p]
__global__ void scalar_flux_kernel(int J, int N, int G, const double *__restrict__ w, const double *__restrict__ psi,
                                   double *__restrict__ phi)
{
    const size_t total = (size_t)J * G * 4;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (size_t)gridDim.x * blockDim.x) {
        const int p = (int)(e & 3);
        const size_t jg = e >> 2;
        double s = 0.0;
        for (int m = 0; m < N; ++m) s = fma(w[m], psi[(jg * N + m) * 4 + p], s);
        phi[e] = s;
    }
}

// the launch floor bench.py quotes the per-iteration times of the L2-resident configurations against
__global__ void empty_kernel(int *sink)
{
    if (sink == nullptr && threadIdx.x == 1024) *sink = 0; // never true: keeps the kernel from being optimised away
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

// ------------------------------------------------------------------------------------------------------------
// Work decomposition of the pipelined kernel for a given n (host side)
// ------------------------------------------------------------------------------------------------------------
struct StreamPlan {
    int cpb, S, cw, nch, chunk_doubles, stages, grid;
    size_t smem;
};

static StreamPlan make_plan(const oci_ctx *ctx)
{
    StreamPlan pl;
    const int n = ctx->n;
    const int CH = 4096; // doubles per chunk (32 KB)
    int cpb = CH / (n * n);
    if (cpb < 1) cpb = 1;
    if (cpb > CONSUMERS / n) cpb = CONSUMERS / n;
    if (cpb < 1) cpb = 1;
    pl.cpb = cpb;
    pl.S = CONSUMERS / (cpb * n);
    if (pl.S < 1) pl.S = 1;
    if (cpb > 1 || n * n <= CH) { pl.cw = n; pl.nch = 1; pl.chunk_doubles = cpb * n * n; }
    else {
        pl.cw = CH / n;
        pl.nch = (n + pl.cw - 1) / pl.cw;
        pl.chunk_doubles = pl.cw * n;
    }
    pl.chunk_doubles = (pl.chunk_doubles + 15) & ~15; // keep stages 128-byte aligned
    const int n_items = (ctx->J + cpb - 1) / cpb;
    int ctas_per_sm = ctx->opt_ctas_per_sm > 0 ? ctx->opt_ctas_per_sm : 1;
    const size_t fixed = (size_t)(2 * MAX_STAGES + 2 * VEC_SLOTS) * 8 + (size_t)(2 * ctx->N + 2 * CONSUMERS) * 8 + 256 +
                         (size_t)VEC_SLOTS * ((2 * cpb + 2) * n) * 8 + 128;
    const size_t budget = (size_t)ctx->max_smem_optin / ctas_per_sm - (ctas_per_sm > 1 ? 1024 : 0);
    int stages = (int)((budget - fixed) / ((size_t)pl.chunk_doubles * 8));
    if (stages > MAX_STAGES) stages = MAX_STAGES;
    if (ctx->opt_stages > 0 && ctx->opt_stages < stages) stages = ctx->opt_stages;
    if (stages < 2) stages = 2;
    pl.stages = stages;
    pl.smem = fixed + (size_t)stages * pl.chunk_doubles * 8;
    int grid = ctx->num_sms * ctas_per_sm;
    if (grid > n_items) grid = n_items;
    pl.grid = grid;
    return pl;
}

int launch_oci_iteration(oci_ctx *ctx, int hist_slot, bool want_l2, bool check_prev)
{
    IterParams P;
    P.stop = make_stop(ctx, hist_slot, check_prev);
    P.J = ctx->J; P.N = ctx->N; P.G = ctx->G; P.n = ctx->n;
    P.bc_left = ctx->bc_left; P.bc_right = ctx->bc_right;
    P.Minv = ctx->Minv; P.c = ctx->c;
    P.psi_old = ctx->psi[ctx->cur]; P.psi_new = ctx->psi[ctx->cur ^ 1];
    P.phi = ctx->phi; P.mu = ctx->mu; P.w = ctx->w;
    P.inc_left = ctx->inc_left; P.inc_right = ctx->inc_right;
    P.resid_inf = ctx->resid_inf + hist_slot;
    P.resid_l2 = ctx->resid_l2 + hist_slot;
    P.color = 0; P.ncolors = 1; P.reverse = 0;
    P.reverse = (hist_slot & 1) == 0;
    if (ctx->opt_ordering == 1 && ctx->opt_solve_mode != 1) return OCI_E_UNSUPPORTED; // red-black: structured path only
    const bool wpc_ok = ctx->n == 64 || ctx->n == 128 || ctx->n == 256;
    if (ctx->opt_solve_mode == 1) {
        P.cpb = 1; P.S = 1; P.cw = ctx->n; P.nch = 1; P.n_items = ctx->J; P.stages = 0; P.chunk_doubles = 0;
        const int r = launch_st_iteration(ctx, P, want_l2);
        if (r < 0) return r;
    } else if (ctx->opt_iterate_kernel == 1 && wpc_ok) {
        const int n = ctx->n;
        const size_t fixed = (size_t)(2 * WPC_MAX_STAGES + 2 * WPC_VEC_SLOTS) * 8 + (size_t)(2 * ctx->N) * 8 + 256 +
                             (size_t)WPC_VEC_SLOTS * ((2 * WPC_WARPS + 2) * n) * 8 + 128;
        int stages = (int)(((size_t)ctx->max_smem_optin - fixed) / ((size_t)WPC_CHUNK * 8 * WPC_WARPS)); // per warp
        if (stages > WPC_MAX_STAGES / WPC_WARPS) stages = WPC_MAX_STAGES / WPC_WARPS;
        if (ctx->opt_stages > 0 && ctx->opt_stages < stages) stages = ctx->opt_stages;
        if (stages < 1) stages = 1;
        const size_t smem = fixed + (size_t)stages * WPC_WARPS * WPC_CHUNK * 8;
        P.cpb = 1; P.S = 1; P.cw = WPC_CHUNK / n; P.nch = n / P.cw; P.n_items = ctx->J; P.stages = stages;
        P.chunk_doubles = WPC_CHUNK;
        int grid = ctx->num_sms;
        if (grid > (ctx->J + WPC_WARPS - 1) / WPC_WARPS) grid = (ctx->J + WPC_WARPS - 1) / WPC_WARPS;
#define OCI_WPC_LAUNCH(RPL_, L2_)                                                                                  \
    do {                                                                                                           \
        OCI_CUDA_TRY(ctx, grant_smem(ctx, SLOT_WPC + (RPL_ == 2 ? 0 : (RPL_ == 4 ? 2 : 4)) + (L2_ ? 1 : 0),         \
                                     (const void *)oci_iterate_wpc_kernel<RPL_, L2_>, smem));                      \
        OCI_CUDA_TRY(ctx, launch_pdl(oci_iterate_wpc_kernel<RPL_, L2_>, dim3(grid), dim3(WPC_THREADS), smem,        \
                                     ctx->stream, P));                                                            \
    } while (0)
        if (n == 64) { if (want_l2) OCI_WPC_LAUNCH(2, true); else OCI_WPC_LAUNCH(2, false); }
        else if (n == 128) { if (want_l2) OCI_WPC_LAUNCH(4, true); else OCI_WPC_LAUNCH(4, false); }
        else { if (want_l2) OCI_WPC_LAUNCH(8, true); else OCI_WPC_LAUNCH(8, false); }
#undef OCI_WPC_LAUNCH
    } else if (ctx->opt_iterate_kernel == 0 || ctx->n > CONSUMERS) {
        P.cpb = 1; P.S = 1; P.cw = ctx->n; P.nch = 1; P.n_items = ctx->J; P.stages = 0; P.chunk_doubles = 0;
        const size_t smem = (size_t)(5 * ctx->n + 2 * ctx->N) * sizeof(double);
        int grid = ctx->num_sms * 8;
        if (grid > ctx->J) grid = ctx->J;
        if (want_l2) oci_iterate_plain_kernel<true><<<grid, 256, smem, ctx->stream>>>(P);
        else oci_iterate_plain_kernel<false><<<grid, 256, smem, ctx->stream>>>(P);
    } else {
        const StreamPlan pl = make_plan(ctx);
        P.cpb = pl.cpb; P.S = pl.S; P.cw = pl.cw; P.nch = pl.nch; P.stages = pl.stages;
        P.chunk_doubles = pl.chunk_doubles;
        P.n_items = (ctx->J + pl.cpb - 1) / pl.cpb;
        OCI_CUDA_TRY(ctx, grant_smem(ctx, SLOT_STREAM + (want_l2 ? 1 : 0),
                                     want_l2 ? (const void *)oci_iterate_stream_kernel<true>
                                             : (const void *)oci_iterate_stream_kernel<false>, pl.smem));
        if (want_l2) oci_iterate_stream_kernel<true><<<pl.grid, ITER_THREADS, pl.smem, ctx->stream>>>(P);
        else oci_iterate_stream_kernel<false><<<pl.grid, ITER_THREADS, pl.smem, ctx->stream>>>(P);
    }
    OCI_CUDA_TRY(ctx, cudaGetLastError());
    if (ctx->opt_ordering == 1) return 2; // red-black updates the current iterate in place: no buffer swap
    ctx->cur ^= 1;
    return 1;
}

int launch_empty(oci_ctx *ctx)
{
    empty_kernel<<<ctx->num_sms, 160, 0, ctx->stream>>>(ctx->ctrl);
    OCI_CUDA_TRY(ctx, cudaGetLastError());
    return 1;
}

int launch_const_rhs(oci_ctx *ctx)
{
    ProblemView P = make_view(ctx);
    const size_t total = (size_t)ctx->J * ctx->n;
    const_rhs_kernel<<<grid_for(total, 256, ctx->num_sms), 256, 0, ctx->stream>>>(P, ctx->q, ctx->psi_prev, ctx->c);
    OCI_CUDA_TRY(ctx, cudaGetLastError());
    return 1;
}

int launch_advance(oci_ctx *ctx)
{
    const size_t pairs = (size_t)ctx->J * ctx->G * ctx->N;
    advance_kernel<<<grid_for(pairs * 2, 256, ctx->num_sms), 256, 0, ctx->stream>>>(pairs, ctx->psi[ctx->cur],
                                                                                      ctx->psi_prev);
    OCI_CUDA_TRY(ctx, cudaGetLastError());
    return 1;
}

int launch_seed_iterate(oci_ctx *ctx)
{
    const size_t pairs = (size_t)ctx->J * ctx->G * ctx->N;
    seed_iterate_kernel<<<grid_for(pairs * 4, 256, ctx->num_sms), 256, 0, ctx->stream>>>(pairs, ctx->psi_prev,
                                                                                           ctx->psi[ctx->cur]);
    OCI_CUDA_TRY(ctx, cudaGetLastError());
    return 1;
}

int launch_scalar_flux(oci_ctx *ctx, const double *psi, double *phi)
{
    const size_t total = (size_t)ctx->J * ctx->G * 4;
    scalar_flux_kernel<<<grid_for(total, 256, ctx->num_sms), 256, 0, ctx->stream>>>(ctx->J, ctx->N, ctx->G, ctx->w, psi, phi);
    OCI_CUDA_TRY(ctx, cudaGetLastError());
    return 1;
}

// f2, dense path: k iterations in one cooperative launch with the inverses resident in shared memory. Applies (auto)
// when the problem's inverses fit in the shared memory of the chip with one CTA per SM; "persistent" = 0 disables it.
// Returns 0 when it does not apply (the caller falls back to one launch per iteration).
int launch_dense_multi(oci_ctx *ctx, int slot0, int k, bool want_l2, bool check_between)
{
    if (ctx->opt_solve_mode != 0 || ctx->opt_persistent == 0 || ctx->opt_ordering != 0 || k < 2) return 0;
    if (ctx->opt_iterate_kernel == 0) return 0; // the plain kernel was asked for
    const int n = ctx->n;
    int grid = ctx->num_sms < ctx->J ? ctx->num_sms : ctx->J;
    const int cpc = (ctx->J + grid - 1) / grid;
    grid = (ctx->J + cpc - 1) / cpc;
    const size_t smem = sizeof(double) * ((size_t)cpc * n * n + (size_t)(3 * cpc + 2) * n + 2 * (size_t)ctx->N + 8);
    if (smem > (size_t)ctx->max_smem_optin) return 0;
    int coop = 0;
    if (cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, ctx->device) != cudaSuccess || !coop) return 0;
    const void *fn = want_l2 ? (const void *)oci_iterate_resident_kernel<true> : (const void *)oci_iterate_resident_kernel<false>;
    OCI_CUDA_TRY(ctx, grant_smem(ctx, SLOT_RESIDENT + (want_l2 ? 1 : 0), fn, smem));
    int per_sm = 0;
    OCI_CUDA_TRY(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, 256, smem));
    if (per_sm < 1 || grid > per_sm * ctx->num_sms) return 0; // all CTAs must be co-resident for the grid barrier
    IterParams P;
    P.stop = make_stop(ctx, slot0, false);
    P.J = ctx->J; P.N = ctx->N; P.G = ctx->G; P.n = n;
    P.bc_left = ctx->bc_left; P.bc_right = ctx->bc_right;
    P.Minv = ctx->Minv; P.c = ctx->c;
    P.psi_old = ctx->psi[ctx->cur]; P.psi_new = ctx->psi[ctx->cur ^ 1];
    P.phi = ctx->phi; P.mu = ctx->mu; P.w = ctx->w;
    P.inc_left = ctx->inc_left; P.inc_right = ctx->inc_right;
    P.resid_inf = ctx->resid_inf + slot0; P.resid_l2 = ctx->resid_l2 + slot0;
    P.cpb = 1; P.S = 1; P.cw = n; P.nch = 1; P.n_items = ctx->J; P.stages = 0; P.chunk_doubles = 0;
    P.color = 0; P.ncolors = 1; P.reverse = 0;
    DenseMulti M;
    M.n_iters = k; M.slot0 = slot0; M.check_between = check_between ? 1 : 0; M.rule = ctx->stop_rule; M.tol = ctx->stop_tol;
    M.cpc = cpc;
    M.resid_inf = ctx->resid_inf; M.resid_l2 = ctx->resid_l2; M.executed = ctx->ctrl;
    void *args[] = {&P, &M};
    OCI_CUDA_TRY(ctx, cudaLaunchCooperativeKernel(fn, dim3(grid), dim3(256), args, smem, ctx->stream));
    if (k & 1) ctx->cur ^= 1; // as k single launches would have left it
    return 1;
}
