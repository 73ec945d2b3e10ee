// ea_replica.cuh -- second workload (R24): the paper's own multispin
// coding.  A word holds the spins of the TEMPERATURE REPLICAS of one disorder realization at one
// site ("asynchronous multispin coding"), every replica consumes its own
// random number, and one thread block owns a realization with all its replicas, sweeps them and
// makes the parallel-tempering exchange by itself (PAPER.md:91 Figure 3, :95).  The probability
// table has one row per temperature; a swap exchanges the rows of two replicas, no spin moves
// (PAPER.md:243).
//
//   T storage: spinT[r][c][p][j] uint32, bit b of cube c = slot 32 c + b ("integer cube",
//              more than 32 replicas need several cubes);
//              jbit[r][d][p][NW] packed coupling bits (one bit per bond: the replicas share J).
//
// The library keeps its first layout (bits = realizations) as the exchange format of every
// accessor; k_r2t / k_t2r transpose between the two when a handle in this layout is read or set.
// Draws: PX(g, q, r, ((6+p)<<16)|k)[l] per (site, realization r, slot k); swap draws, tables,
// initial state and couplings are those of the first layout, so both layouts simulate the same
// physical systems with different random numbers.
#pragma once
#include "ea_generic.cuh"
#include "ea_resident.cuh"

namespace ea {

struct ReplicaArgs {
    Params P;
    uint32_t *spinT;          // [Rp][ncube][N]
    uint32_t *jbit;           // [Rp][3][2][NW]
    const uint64_t *acc64;    // [nT][7] acceptance thresholds in [0, 2^32] (row = temperature index)
    int ncube, NW;
    uint32_t g0;
    int n_sweeps, swap_interval;
    uint32_t nswap0;
    uint32_t rk[20];          // Philox round keys (k0 + r*0x9E3779B9, k1 + r*0xBB67AE85), r = 0..9
};

__device__ __forceinline__ int replica_nw(int Nh) { return (Nh + 31) >> 5; }

// first layout -> T storage: thread per (r, c, site word)
__global__ void k_r2t(ReplicaArgs A)
{
    const Params &P = A.P;
    const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t n_spin = (int64_t)P.Rp * A.ncube * P.N;
    if (tid < n_spin) {
        const int i = (int)(tid % P.N), c = (int)((tid / P.N) % A.ncube), r = (int)(tid / ((int64_t)P.N * A.ncube));
        const int w = r >> 5, b = r & 31;
        uint32_t v = 0;
        for (int kb = 0; kb < 32 && 32 * c + kb < P.nT; ++kb)
            v |= ((P.spin[((size_t)(32 * c + kb) * P.W + w) * P.N + i] >> b) & 1u) << kb;
        A.spinT[tid] = v;
        return;
    }
    const int64_t t2 = tid - n_spin;                 // coupling bits: thread per (r, d, p, word)
    const int64_t n_j = (int64_t)P.Rp * 6 * A.NW;
    if (t2 >= n_j) return;
    const int jw = (int)(t2 % A.NW), dp = (int)((t2 / A.NW) % 6), r = (int)(t2 / ((int64_t)A.NW * 6));
    const int w = r >> 5, b = r & 31;
    const uint32_t *cp = P.coup + (size_t)w * 3 * P.N + (size_t)dp * P.Nh;      // [d][p][j] = [dp][j]
    uint32_t v = 0;
    for (int jb = 0; jb < 32 && 32 * jw + jb < P.Nh; ++jb) v |= ((cp[32 * jw + jb] >> b) & 1u) << jb;
    A.jbit[t2] = v;
}

// T storage -> first layout (spins only; couplings never change in this layout): thread per (k, w, site)
__global__ void k_t2r(ReplicaArgs A)
{
    const Params &P = A.P;
    const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= (int64_t)P.nT * P.W * P.N) return;
    const int i = (int)(tid % P.N), w = (int)((tid / P.N) % P.W), k = (int)(tid / ((int64_t)P.N * P.W));
    const int c = k >> 5, kb = k & 31;
    uint32_t v = 0;
    for (int b = 0; b < 32; ++b)
        v |= ((A.spinT[((size_t)(32 * w + b) * A.ncube + c) * P.N + i] >> kb) & 1u) << b;
    P.spin[tid] = v;
}

// n_sat planes of site (p, j) of the block's lattice `lat` ([p][j], one word per site: bit = replica)
// with the realization's packed coupling bits `jb` ([d][p][NW]); the bond bit is the same for all
// replicas, so it enters as an all-ones / all-zeros word.
__device__ __forceinline__ Planes replica_planes(const uint32_t *lat, const uint32_t *jb, int p, int j, int L,
                                                 int Lh, int Nh, int NW, uint32_t *self_out)
{
    const Site c = site_of(j, p, L, Lh);
    const Nbr n = nbr_of(c, L, Lh);
    const uint32_t *so = lat + (1 - p) * Nh;
    const uint32_t s = lat[p * Nh + j];
    auto jm = [&](int d, int pp, int jj) { return 0u - ((jb[(d * 2 + pp) * NW + (jj >> 5)] >> (jj & 31)) & 1u); };
    const uint32_t e0 = xor3(s, jm(0, p, j), so[n.xp]);
    const uint32_t e1 = xor3(s, jm(0, 1 - p, n.xm), so[n.xm]);
    const uint32_t e2 = xor3(s, jm(1, p, j), so[n.yp]);
    const uint32_t e3 = xor3(s, jm(1, 1 - p, n.ym), so[n.ym]);
    const uint32_t e4 = xor3(s, jm(2, p, j), so[n.zp]);
    const uint32_t e5 = xor3(s, jm(2, 1 - p, n.zm), so[n.zm]);
    *self_out = s;
    return nsat_planes(e0, e1, e2, e3, e4, e5);
}

// One block = one realization with all its replicas, for all sweeps of the call.
// Thread = quad of four sites (one Philox call per replica serves them); the lattice (N words per
// cube) and the probability table stay in shared memory; energies by
// bit-sliced counters over the parity-1 sites; one warp takes the swap decisions.
__global__ void __launch_bounds__(256, 2) k_replica_sweep(const ReplicaArgs A)
{
    extern __shared__ __align__(16) uint32_t smem[];
    const Params &P = A.P;
    const int L = P.L, Lh = P.Lh, N = P.N, Nh = P.Nh, nT = P.nT, NW = A.NW, ncube = A.ncube;
    const int r = blockIdx.x, tid = threadIdx.x, lane = tid & 31, NT = blockDim.x;
    uint32_t *lat = smem;                                            // [ncube][N]
    uint32_t *jb = lat + (size_t)ncube * N;                          // [3][2][NW]
    uint64_t *acc = reinterpret_cast<uint64_t *>(jb + 6 * NW + ((6 * NW) & 1));   // [nT][7], 8 B aligned
    int *Ecnt = reinterpret_cast<int *>(acc + 7 * nT);               // [64] satisfied bonds by slot
    int *E = Ecnt + 64;                                              // [64] energies by slot
    uint8_t *tau = reinterpret_cast<uint8_t *>(E + 64);              // [64] slot -> temperature index
    uint8_t *sig = tau + 64;                                         // [64] temperature index -> slot

    for (int a = tid; a < ncube * N; a += NT) lat[a] = A.spinT[(size_t)r * ncube * N + a];
    for (int a = tid; a < 6 * NW; a += NT) jb[a] = A.jbit[(size_t)r * 6 * NW + a];
    for (int a = tid; a < 7 * nT; a += NT) acc[a] = A.acc64[a];
    for (int a = tid; a < nT; a += NT) {
        tau[a] = P.tau[(size_t)r * nT + a];
        sig[a] = P.sigma[(size_t)r * nT + a];
        E[a] = P.E[(size_t)r * nT + a];
    }
    if (tid < 64) Ecnt[tid] = 0;
    __syncthreads();

    const int nq = Nh >> 2;
    const uint32_t gr = P.r0 + (uint32_t)r;
    uint32_t nswap = A.nswap0;
    for (int it = 0; it < A.n_sweeps; ++it) {
        const uint32_t g = A.g0 + (uint32_t)it;
        const bool swap_now = A.swap_interval > 0 && ((uint64_t)g + 1) % (uint64_t)A.swap_interval == 0;
        const bool need_E = swap_now || it == A.n_sweeps - 1;
        for (int p = 0; p < 2; ++p) {
            for (int q = tid; q < nq; q += NT) {
                // counter (g, q, r, tag|k): q is the thread's, everything else the block's -- rounds 0-2 of
                // Philox are partly per-thread constants, partly uniform (philox_quad, ea_resident.cuh)
                const PhiloxQuad PQ = philox_quad_init((uint32_t)q, gr, A.rk);
                for (int c = 0; c < ncube; ++c) {
                    uint32_t *lc = lat + (size_t)c * N;
                    Planes pl[4];
                    uint32_t s[4], flip[4] = {0u, 0u, 0u, 0u};
#pragma unroll
                    for (int l = 0; l < 4; ++l) pl[l] = replica_planes(lc, jb, p, 4 * q + l, L, Lh, Nh, NW, &s[l]);
                    const int kn = min(32, nT - 32 * c);
                    // planes rotated so that replica kb's class bits land on bits 3, 4, 5 of a right
                    // rotation by kb: (rot & 8) | (rot & 16) | (rot & 32) = 8 * n_sat = byte offset of
                    // the 64-bit threshold in the replica's table row
                    uint32_t r0[4], r1[4], r2[4];
#pragma unroll
                    for (int l = 0; l < 4; ++l) {
                        r0[l] = __funnelshift_l(pl[l].b0, pl[l].b0, 3);
                        r1[l] = __funnelshift_l(pl[l].b1, pl[l].b1, 4);
                        r2[l] = __funnelshift_l(pl[l].b2, pl[l].b2, 5);
                    }
                    for (int kb = 0; kb < kn; ++kb) {            // replica by replica ("AMSC1")
                        const int k = 32 * c + kb;
                        const uint4 rnd = philox_quad(PQ, g, ((uint32_t)(6 + p) << 16) | (uint32_t)k, A.rk);
                        const char *row = reinterpret_cast<const char *>(acc + 7 * (int)tau[k]);   // the replica's row of the table
                        const uint32_t u[4] = {rnd.x, rnd.y, rnd.z, rnd.w};
                        const uint32_t kmask = 1u << kb;
#pragma unroll
                        for (int l = 0; l < 4; ++l) {
                            const uint32_t a = __funnelshift_r(r0[l], r0[l], kb), b = __funnelshift_r(r1[l], r1[l], kb);
                            const uint32_t d = __funnelshift_r(r2[l], r2[l], kb);
                            const uint32_t off = (a & 8u) | (b & 16u) | (d & 32u);
                            if ((uint64_t)u[l] < *reinterpret_cast<const uint64_t *>(row + off)) flip[l] |= kmask;
                        }
                    }
#pragma unroll
                    for (int l = 0; l < 4; ++l) lc[p * Nh + 4 * q + l] = s[l] ^ flip[l];
                }
            }
            __syncthreads();
        }
        if (!need_E) continue;
        // ---- energies: every bond has exactly one parity-1 end
        for (int c = 0; c < ncube; ++c) {
            uint32_t cn[22];
#pragma unroll
            for (int i = 0; i < 22; ++i) cn[i] = 0;
            for (int j = tid; j < Nh; j += NT) {
                uint32_t s;
                const Planes pl = replica_planes(lat + (size_t)c * N, jb, 1, j, L, Lh, Nh, NW, &s);
                vadd<22>(cn, pl.b0, 0);
                vadd<22>(cn, pl.b1, 1);
                vadd<22>(cn, pl.b2, 2);
            }
            atomicAdd(&Ecnt[32 * c + lane], warp_positional_sum<22>(cn, lane));
        }
        __syncthreads();
        if (tid < nT) { E[tid] = 3 * N - 2 * Ecnt[tid]; }
        if (tid < 64) Ecnt[tid] = 0;
        __syncthreads();
        if (!swap_now) continue;
        // ---- swap round: lane = temperature pair of this round (disjoint pairs, R4);
        //      an accepted swap exchanges two rows of the table (tau), no spin moves
        if (tid < 32) {
            const int t = (int)(nswap & 1u) + 2 * tid;
            if (t + 1 < nT) {
                const int a = sig[t], b = sig[t + 1];
                const int m = (E[a] - E[b]) / P.ediv;
                const uint4 v = philox4x32_10(g, (uint32_t)t, gr, 2u << 16, P.k0, P.k1);
                if (swap_accept(P, t, m, v.x)) {
                    sig[t] = (uint8_t)b; sig[t + 1] = (uint8_t)a;
                    tau[a] = (uint8_t)(t + 1); tau[b] = (uint8_t)t;
                }
            }
        }
        ++nswap;
        __syncthreads();
    }
    for (int a = tid; a < ncube * N; a += NT) A.spinT[(size_t)r * ncube * N + a] = lat[a];
    for (int a = tid; a < nT; a += NT) {
        P.tau[(size_t)r * nT + a] = tau[a];
        P.sigma[(size_t)r * nT + a] = sig[a];
        P.E[(size_t)r * nT + a] = E[a];
    }
}

}  // namespace ea
