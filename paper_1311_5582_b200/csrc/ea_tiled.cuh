// ea_tiled.cuh -- z-slab tiled half-sweep kernel for lattices that do not fit shared memory
// (L = 32, also 16 and 64).
//
// One launch per half-sweep.  Block = (word w, z-slab, group of SK slots): 512 threads, one
// quad (four x-consecutive same-parity sites = one 128-bit word vector) each.  The couplings
// of the thread's quad stay in registers across the SK slots; the lattice is read and written
// in place in global memory with 128-bit accesses: every neighbour vector is shared by five
// threads of the block, so the tile (slab + two halo planes, 20-24 KiB per slot) is served
// from L1/L2 and HBM sees each word once per half-sweep.  Rank tables live in shared memory.
// Energy: satisfied-bond counts of the parity-1 pass are reduced per warp (bit-sliced adders
// + shuffles), per block (shared-memory atomics) and added to global counters.
#pragma once
#include "ea_resident.cuh"

namespace ea {

struct TiledArgs {
    Params P;
    uint32_t g;              // global sweep index
    int parity;
    int SK;                  // slots per block (multiple of 4)
    int n_kgroups;           // ceil(nT / SK)
    int32_t *Ecnt;           // [Rp][nT] satisfied-bond counters (ENERGY pass), zeroed by k_tiled_finish
    const uint4 *bucket;
    const uchar4 *trip;      // [3 nT + 1] (n4, n5, n6) of every combined rank
    RankKey K;
    uint32_t rk[20];
};

template <int L>
struct TileGeom {
    using Gm = ResGeom<L>;
    static constexpr int QPP = Gm::QR * L;                         // quads per z-plane per parity
    static constexpr int ZS = (512 / QPP) < 1 ? 1 : ((512 / QPP) > L ? L : (512 / QPP));
    static constexpr int NTHR = QPP * ZS;                          // threads per block
    static constexpr int NSLAB = L / ZS;
};

template <int L, bool FAST, bool ENERGY>
__global__ void __launch_bounds__(TileGeom<L>::NTHR, 1) k_tiled_half(const TiledArgs A)
{
    using Gm = ResGeom<L>;
    using Tg = TileGeom<L>;
    constexpr int N = Gm::N, QR = Gm::QR, NT = Tg::NTHR;
    extern __shared__ __align__(16) uint32_t smem[];
    const Params &P = A.P;
    const int nT = P.nT, LTS = P.LTS, SK = A.SK;
    const int p = A.parity;
    int bid = blockIdx.x;
    const int kg = bid % A.n_kgroups; bid /= A.n_kgroups;
    const int slab = bid % Tg::NSLAB;
    const int w = bid / Tg::NSLAB;
    const int k0 = kg * SK;
    const int nk = max(0, min(SK, nT - k0));
    const int tid = threadIdx.x, lane = tid & 31;
    const int q = slab * NT + tid;                // quad index inside a parity array

    const int MTS = 3 * nT + 2;
    uint4 *bucket = reinterpret_cast<uint4 *>(smem);               // [n_bucket]
    uint4 *mt = bucket + A.K.n_bucket;                               // [SK][MTS] mask tables
    uint32_t *lt = reinterpret_cast<uint32_t *>(mt + (size_t)SK * MTS);   // [SK][LTS]
    uint32_t *thr = lt + SK * LTS;                                 // [3][LTS]
    uchar4 *trip = reinterpret_cast<uchar4 *>(thr + 3 * LTS);      // [MTS]
    int32_t *Eacc = (int32_t *)(trip + MTS);                       // [SK][32]

    for (int a = tid; a < A.K.n_bucket; a += NT) bucket[a] = A.bucket[a];
    for (int a = tid; a < nk * LTS; a += NT) lt[a] = P.lt[((size_t)w * nT + k0) * LTS + a];
    for (int a = tid; a < 3 * LTS; a += NT) thr[a] = P.thr32[a];
    for (int a = tid; a < MTS - 1; a += NT) trip[a] = A.trip[a];
    if (ENERGY) for (int a = tid; a < SK * 32; a += NT) Eacc[a] = 0;

    const int qx = q % QR, y = (q / QR) % L, z = q / (QR * L);
    const int qyp = qx + QR * (wrap_inc(y, L) + L * z), qym = qx + QR * (wrap_dec(y, L) + L * z);
    const int qzp = qx + QR * (y + L * wrap_inc(z, L)), qzm = qx + QR * (y + L * wrap_dec(z, L));
    const int s = (y + z + p) & 1;
    const QuadJ J = load_quad_j<L>(P.coup + (size_t)w * 3 * N, p, s, q, qx, qym, qzm);
    // neighbour byte offsets do not fit 16 bits for L = 32, 64: pass quad indices * 16 directly
    RankCtx R;
    R.thr = thr; R.LTS = LTS; R.nT = nT;
    rank_ctx_key(R, A.K, bucket);
    R.z0 = P.z[0]; R.z1 = P.z[1]; R.z2 = P.z[2];
    const uint32_t gw = P.w0 + (uint32_t)w;
    const uint32_t c3 = (uint32_t)p << 16;
    __syncthreads();
    if (FAST) {
        for (int kl = tid >> 5; kl < nk; kl += NT >> 5) build_mt(mt + (size_t)kl * MTS, lt + kl * LTS, trip, nT, lane);
        __syncthreads();
    }

    Planes fin[4];
    if (!ENERGY) {
        for (int kl = 0; kl < nk; ++kl) {
            uint32_t *sp = P.spin + ((size_t)(k0 + kl) * P.W + w) * N;
            const uint4 rnd = philox_rk(A.g, (uint32_t)q, gw, c3 | (uint32_t)(k0 + kl), A.rk);
            update_quad_wide<L, FAST, false>(sp, lt + kl * LTS, mt + (size_t)kl * MTS, R, J, p, s, q, qyp, qym, qzp, qzm, rnd, fin);
        }
    }
    for (int kb = 0; ENERGY && kb < SK; kb += 4) {
        uint32_t en[4][5];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int kl = kb + i;
            if (kl < nk) {
                uint32_t *sp = P.spin + ((size_t)(k0 + kl) * P.W + w) * N;
                const uint4 rnd = philox_rk(A.g, (uint32_t)q, gw, c3 | (uint32_t)(k0 + kl), A.rk);
                update_quad_wide<L, FAST, true>(sp, lt + kl * LTS, mt + (size_t)kl * MTS, R, J, p, s, q, qyp, qym, qzp, qzm, rnd, fin);
                quad_sum(fin, en[i]);
            } else {
#pragma unroll
                for (int j = 0; j < 5; ++j) en[i][j] = 0;
            }
        }
        uint32_t tot[kResPlanes];
        warp_sum4(en, lane, tot);
        const int kl = kb + 2 * (lane >> 4) + ((lane >> 3) & 1);
        if (kl < nk) add_counts(tot, lane & 7, Eacc + kl * 32);
    }
    if (!ENERGY) return;
    __syncthreads();
    for (int a = tid; a < nk * 32; a += NT)
        atomicAdd(A.Ecnt + (size_t)(32 * w + (a & 31)) * nT + k0 + (a >> 5), Eacc[a]);
}

// E[r][k] = 3N - 2 * (satisfied bonds); counters cleared for the next sweep.
__global__ void k_tiled_finish(Params P, int32_t *Ecnt)
{
    const int a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= P.Rp * P.nT) return;
    P.E[a] = 3 * P.N - 2 * Ecnt[a];
    Ecnt[a] = 0;
}

}  // namespace ea
