// ea_stream.cuh -- persistent streaming sweep kernel for lattices that do not fit shared
// memory (L = 32, 64).
//
// One cooperative launch runs all sweeps of a call.  The grid is one block per SM; the work
// items (word w, z-slab, slot k) are dealt out in contiguous ranges, so a block meets at most
// a few (w, slab) groups and re-reads its couplings (registers, one parity at a time) only
// when the group changes.  Per half-sweep a block streams its items through a two-stage ring
// of shared-memory buffers filled by TMA bulk copies (cp.async.bulk + mbarrier): the slab's
// words of the updated parity and the other parity's words of the slab plus one halo plane on
// each side.  Threads compute from shared memory exactly as the resident kernel does (one
// quad = four x-consecutive same-parity sites per thread) and store the new words straight to
// global memory (the state, 35 MiB for config 5, lives in L2).  Two grid-wide barriers per
// sweep separate the half-sweeps (two consecutive stages).  Energies: satisfied
// bonds of the parity-1 pass -> per-block shared atomics -> global counters; after the second
// barrier every block takes the parallel-tempering decisions of the words it works on
// (identical in every block: same counters, same Philox draws) and rebuilds its mask tables.
// No lattice word moves in a swap.
#pragma once
#include <cooperative_groups.h>

#include "ea_generic.cuh"
#include "ea_resident.cuh"

namespace ea {

struct StreamArgs {
    Params P;
    uint32_t g0;             // global index of the first sweep of this call
    int n_sweeps;
    int swap_interval;
    uint32_t nswap0;         // swap rounds done before this call
    int32_t *Ecnt;           // [2][Rp][nT] satisfied-bond counters (zero on entry)
    const uint4 *bucket;
    const uchar4 *trip;
    int n_bucket, key_lo, key_shift;
    uint32_t ones, c48, cm16, c16;
    uint32_t rk[20];
    int MS;                  // most items one block can get = ceil(items / grid)
    int MW;                  // most words one block can meet
};

template <int L>
struct StreamGeom {
    using Gm = ResGeom<L>;
    static constexpr int QPP = Gm::QR * L;                 // quads per z-plane per parity
    static constexpr int NTHR = 512;
    static constexpr int ZS = NTHR / QPP;                  // planes per slab
    static_assert(ZS >= 1 && ZS * QPP == NTHR && L % ZS == 0 && L / ZS >= 2, "slab shape");
    static constexpr int NSLAB = L / ZS;
    static constexpr int OWN_BYTES = NTHR * 16;
    static constexpr int OTH_BYTES = (ZS + 2) * QPP * 16;
    static constexpr int BUF_BYTES = OWN_BYTES + OTH_BYTES;
    static constexpr int NB = BUF_BYTES <= 20480 ? 4 : 2;  // slots per batch
    static constexpr int NS = 2;                           // ring stages
};

// ------------------------------------------------------------------ mbarrier / TMA bulk copy
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }


// Per-block constants of the streaming kernel.
template <int L>
struct StreamCtx {
    int i0, i1;                  // my items [i0, i1), item = (w * NSLAB + slab) * nT + k
    int nT, LTS, MTS;
    int tid, lane, qx, y, zl;
    uint32_t ov, oyp, oym, ozp, ozm;   // byte offsets inside the other-parity buffer
    uint64_t *mbar;
    unsigned char *bufs;
    uint4 *mt;
    uint32_t *lt;
    int32_t *Eacc;               // [2][NB][32]
    RankCtx R;
};

// One half-sweep (parity p) over the block's items.  ENERGY: also count the satisfied bonds of
// the updated (parity-1) sites into A.Ecnt[ebuf].
template <int L, bool FAST, bool ENERGY>
__device__ __forceinline__ void stream_half(const StreamArgs &A, const StreamCtx<L> &C, int p, uint32_t g,
                                            uint32_t &phase, int ebuf)
{
    using Gm = ResGeom<L>;
    using Sg = StreamGeom<L>;
    constexpr int N = Gm::N, Nh = Gm::Nh, QR = Gm::QR, QPP = Sg::QPP, ZS = Sg::ZS, NT = Sg::NTHR;
    constexpr int NB = Sg::NB, NS = Sg::NS, NSLAB = Sg::NSLAB;
    const Params &P = A.P;
    const int nT = C.nT, tid = C.tid;

    auto batch_count = [&](int pos) { return min(min(NB, C.i1 - pos), nT - pos % nT); };
    // TMA bulk loads of one batch into ring stage st (one thread): per slot the slab's own-parity
    // words (contiguous) and the other parity's planes z0-1 .. z0+ZS (periodic wrap = 2 pieces)
    auto issue = [&](int pos, int st) {
        const int cnt = batch_count(pos);
        const int k0 = pos % nT, grp = pos / nT, slab = grp % NSLAB, w = grp / NSLAB;
        const int z0 = slab * ZS;
        fence_proxy_async();
        mbar_expect_tx(&C.mbar[st], (uint32_t)(cnt * Sg::BUF_BYTES));
        for (int i = 0; i < cnt; ++i) {
            const uint32_t *base = P.spin + ((size_t)(k0 + i) * P.W + w) * N;
            unsigned char *dst = C.bufs + (size_t)(st * NB + i) * Sg::BUF_BYTES;
            bulk_g2s(dst, base + p * Nh + (size_t)slab * NT * 4, Sg::OWN_BYTES, &C.mbar[st]);
            const uint32_t *ob = base + (1 - p) * Nh;
            unsigned char *od = dst + Sg::OWN_BYTES;
            constexpr int PLB = QPP * 16;       // bytes per plane and parity
            if (z0 == 0) {
                bulk_g2s(od, ob + (size_t)(L - 1) * QPP * 4, PLB, &C.mbar[st]);
                bulk_g2s(od + PLB, ob, (ZS + 1) * PLB, &C.mbar[st]);
            } else if (z0 + ZS == L) {
                bulk_g2s(od, ob + (size_t)(z0 - 1) * QPP * 4, (ZS + 1) * PLB, &C.mbar[st]);
                bulk_g2s(od + (ZS + 1) * PLB, ob, PLB, &C.mbar[st]);
            } else {
                bulk_g2s(od, ob + (size_t)(z0 - 1) * QPP * 4, (ZS + 2) * PLB, &C.mbar[st]);
            }
        }
    };

    int ld_pos = C.i0;
    for (int st = 0; st < NS && ld_pos < C.i1; ++st) {
        if (tid == 0) issue(ld_pos, st);
        ld_pos += batch_count(ld_pos);
    }
    int cur_grp = -1, s = 0, q = 0;
    QuadJ J;
    Planes fin[4];
    int bi = 0;
    for (int pos = C.i0; pos < C.i1; ++bi) {
        const int cnt = batch_count(pos), st = bi % NS;
        const int k0 = pos % nT, grp = pos / nT, slab = grp % NSLAB, w = grp / NSLAB;
        if (grp != cur_grp) {        // couplings of my quad for this (word, slab) and parity
            cur_grp = grp;
            const int z = slab * ZS + C.zl;
            s = (C.y + z + p) & 1;
            q = slab * NT + tid;
            const int qym = C.qx + QR * (wrap_dec(C.y, L) + L * z);
            const int qzm = C.qx + QR * (C.y + L * wrap_dec(z, L));
            J = load_quad_j<L>(P.coup + (size_t)w * 3 * N, p, s, q, C.qx, qym, qzm);
        }
        const uint32_t gw = P.w0 + (uint32_t)w;
        const uint32_t c3 = (uint32_t)p << 16;
        mbar_wait(&C.mbar[st], (phase >> st) & 1u);
        phase ^= 1u << st;
        const unsigned char *stage = C.bufs + (size_t)(st * NB) * Sg::BUF_BYTES;
        if (!ENERGY) {
            for (int i = 0; i < cnt; ++i) {
                const int li = pos + i - C.i0;
                const char *buf = reinterpret_cast<const char *>(stage + (size_t)i * Sg::BUF_BYTES);
                const uint4 rnd = philox_rk(g, (uint32_t)q, gw, c3 | (uint32_t)(k0 + i), A.rk);
                const uint4 res = update_quad_mem<L, FAST, false, false>(
                    buf + 16 * tid, buf + Sg::OWN_BYTES, C.ov, C.oyp, C.oym, C.ozp, C.ozm, C.qx, C.lt + li * C.LTS,
                    C.mt + (size_t)li * C.MTS, C.R, J, s, rnd, fin);
                reinterpret_cast<uint4 *>(P.spin + ((size_t)(k0 + i) * P.W + w) * N + p * Nh)[q] = res;
            }
        } else {
            uint32_t en[4][5];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                if (i < cnt) {
                    const int li = pos + i - C.i0;
                    const char *buf = reinterpret_cast<const char *>(stage + (size_t)i * Sg::BUF_BYTES);
                    const uint4 rnd = philox_rk(g, (uint32_t)q, gw, c3 | (uint32_t)(k0 + i), A.rk);
                    const uint4 res = update_quad_mem<L, FAST, true, false>(
                        buf + 16 * tid, buf + Sg::OWN_BYTES, C.ov, C.oyp, C.oym, C.ozp, C.ozm, C.qx,
                        C.lt + li * C.LTS, C.mt + (size_t)li * C.MTS, C.R, J, s, rnd, fin);
                    reinterpret_cast<uint4 *>(P.spin + ((size_t)(k0 + i) * P.W + w) * N + p * Nh)[q] = res;
                    quad_sum(fin, en[i]);
                } else {
#pragma unroll
                    for (int j = 0; j < 5; ++j) en[i][j] = 0;
                }
            }
            uint32_t tot[kResPlanes];
            warp_sum4(en, C.lane, tot);
            const int i_mine = 2 * (C.lane >> 4) + ((C.lane >> 3) & 1);
            if (i_mine < cnt) add_counts(tot, C.lane & 7, C.Eacc + ((bi & 1) * NB + i_mine) * 32);
        }
        __syncthreads();             // the stage is free; this batch's shared counters are complete
        if (ld_pos < C.i1) {
            if (tid == 0) issue(ld_pos, st);
            ld_pos += batch_count(ld_pos);
        }
        if (ENERGY) {
            int32_t *acc = C.Eacc + (bi & 1) * NB * 32;
            for (int a = tid; a < cnt * 32; a += NT) {
                const int v = acc[a];
                acc[a] = 0;
                atomicAdd(A.Ecnt + (size_t)ebuf * P.Rp * nT + (size_t)(32 * w + (a & 31)) * nT + k0 + (a >> 5), v);
            }
        }
        pos += cnt;
    }
}

namespace cg = cooperative_groups;

template <int L, bool FAST>
__global__ void __launch_bounds__(StreamGeom<L>::NTHR, 1) k_stream(const StreamArgs A)
{
    using Gm = ResGeom<L>;
    using Sg = StreamGeom<L>;
    constexpr int N = Gm::N, QR = Gm::QR, QPP = Sg::QPP, NT = Sg::NTHR, NB = Sg::NB, NS = Sg::NS;
    constexpr int NSLAB = Sg::NSLAB;
    extern __shared__ __align__(128) unsigned char smraw[];
    const Params &P = A.P;
    const int nT = P.nT, LTS = P.LTS, MTS = 3 * nT + 2, MS = A.MS, MW = A.MW;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarp = NT >> 5;
    cg::grid_group grid = cg::this_grid();

    StreamCtx<L> C;
    const long long T = (long long)P.W * NSLAB * nT;
    C.i0 = (int)(T * blockIdx.x / gridDim.x);
    C.i1 = (int)(T * (blockIdx.x + 1) / gridDim.x);
    const int per_w = NSLAB * nT;
    const int w_first = C.i0 / per_w, nwt = (C.i1 - 1) / per_w - w_first + 1;   // words I meet (<= MW)

    // shared memory
    uint64_t *mbar = reinterpret_cast<uint64_t *>(smraw);                        // [NS], 64 B reserved
    uint4 *bucket = reinterpret_cast<uint4 *>(smraw + 64);                       // [n_bucket]
    unsigned char *bufs = reinterpret_cast<unsigned char *>(bucket + A.n_bucket);   // [NS][NB][BUF_BYTES]
    uint4 *mt = reinterpret_cast<uint4 *>(bufs + (size_t)NS * NB * Sg::BUF_BYTES);  // [MS][MTS]
    uint32_t *lt = reinterpret_cast<uint32_t *>(mt + (size_t)MS * MTS);          // [MS][LTS]
    uint32_t *thr = lt + MS * LTS;                                               // [3][LTS]
    uchar4 *trip = reinterpret_cast<uchar4 *>(thr + 3 * LTS);                    // [MTS]
    int32_t *Eacc = reinterpret_cast<int32_t *>(trip + MTS);                     // [2][NB][32]
    uint8_t *tau8 = reinterpret_cast<uint8_t *>(Eacc + 2 * NB * 32);             // [MW][32][nT]
    uint8_t *sig8 = tau8 + (size_t)MW * 32 * nT;                                 // [MW][32][nT]

    for (int a = tid; a < A.n_bucket; a += NT) bucket[a] = A.bucket[a];
    for (int a = tid; a < 3 * LTS; a += NT) thr[a] = P.thr32[a];
    for (int a = tid; a < MTS - 1; a += NT) trip[a] = A.trip[a];
    for (int a = tid; a < 2 * NB * 32; a += NT) Eacc[a] = 0;
    for (int a = tid; a < nwt * 32 * nT; a += NT) {
        tau8[a] = P.tau[(size_t)32 * w_first * nT + a];
        sig8[a] = P.sigma[(size_t)32 * w_first * nT + a];
    }
    if (tid == 0) {
        for (int i = 0; i < NS; ++i) mbar_init(&mbar[i], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // rank masks and mask tables of my items from the permutation (one warp per item)
    auto rebuild_tables = [&]() {
        for (int li = warp; li < C.i1 - C.i0; li += nwarp) {
            const int item = C.i0 + li, k = item % nT, wl = item / per_w - w_first;
            const int t = tau8[(size_t)(wl * 32 + lane) * nT + k];
            const int pos = P.desc ? t : nT - 1 - t;
            for (int n = 0; n <= nT; ++n) {
                const uint32_t mk = __ballot_sync(0xFFFFFFFFu, pos >= n);
                if (lane == (n & 31)) lt[li * LTS + n] = mk;
            }
            __syncwarp();
            build_mt(mt + (size_t)li * MTS, lt + li * LTS, trip, nT, lane);
        }
    };
    rebuild_tables();

    C.nT = nT; C.LTS = LTS; C.MTS = MTS;
    C.tid = tid; C.lane = lane;
    C.qx = tid % QR; C.y = (tid / QR) % L; C.zl = tid / QPP;
    {
        const int row = QR * C.y + C.qx;
        C.ov = 16u * (uint32_t)((C.zl + 1) * QPP + row);
        C.oyp = 16u * (uint32_t)((C.zl + 1) * QPP + QR * wrap_inc(C.y, L) + C.qx);
        C.oym = 16u * (uint32_t)((C.zl + 1) * QPP + QR * wrap_dec(C.y, L) + C.qx);
        C.ozp = 16u * (uint32_t)((C.zl + 2) * QPP + row);
        C.ozm = 16u * (uint32_t)(C.zl * QPP + row);
    }
    C.mbar = mbar; C.bufs = bufs; C.mt = mt; C.lt = lt; C.Eacc = Eacc;
    C.R.thr = thr; C.R.bucket = bucket; C.R.LTS = LTS; C.R.nT = nT;
    C.R.key_lo = A.key_lo; C.R.key_top = A.n_bucket - 1; C.R.key_shift = A.key_shift;
    C.R.z0 = P.z[0]; C.R.z1 = P.z[1]; C.R.z2 = P.z[2];
    C.R.ones = A.ones; C.R.c48 = A.c48; C.R.cm16 = A.cm16; C.R.c16 = A.c16;
    __syncthreads();

    uint32_t nswap = A.nswap0, phase = 0;
    int ebuf = 0;
    for (int it = 0; it < A.n_sweeps; ++it) {
        const uint32_t g = A.g0 + (uint32_t)it;
        const bool swap_now = A.swap_interval > 0 && ((uint64_t)g + 1) % (uint64_t)A.swap_interval == 0;
        const bool need_E = swap_now || it == A.n_sweeps - 1;
        stream_half<L, FAST, false>(A, C, 0, g, phase, ebuf);
        grid.sync();
        if (need_E) stream_half<L, FAST, true>(A, C, 1, g, phase, ebuf);
        else stream_half<L, FAST, false>(A, C, 1, g, phase, ebuf);
        grid.sync();
        if (!need_E) continue;
        const int32_t *cnt = A.Ecnt + (size_t)ebuf * P.Rp * nT;     // satisfied bonds by [r][k]
        if (swap_now) {
            // swap round: warp per temperature pair, lane = realization; every block that works
            // on a word takes the same decisions.  E_a - E_b = -2 (c_a - c_b).
            for (int wl = 0; wl < nwt; ++wl) {
                const int r = 32 * (w_first + wl) + lane;
                uint8_t *sg_ = sig8 + (size_t)(wl * 32 + lane) * nT, *ta_ = tau8 + (size_t)(wl * 32 + lane) * nT;
                for (int t = (int)(nswap & 1u) + 2 * warp; t + 1 < nT; t += 2 * nwarp) {
                    const int sa = sg_[t], sb = sg_[t + 1];
                    const int ca = __ldcg(cnt + (size_t)r * nT + sa), cb = __ldcg(cnt + (size_t)r * nT + sb);
                    const int m = (cb - ca) / 2;
                    const uint4 v = philox_rk(g, (uint32_t)t, P.r0 + (uint32_t)r, 2u << 16, A.rk);
                    if (swap_accept(P, t, m, v.x)) {
                        sg_[t] = (uint8_t)sb; sg_[t + 1] = (uint8_t)sa;
                        ta_[sa] = (uint8_t)(t + 1); ta_[sb] = (uint8_t)t;
                    }
                }
            }
            ++nswap;
            __syncthreads();
            rebuild_tables();
        }
        // the block that owns item (w, slab 0, slot 0) keeps the word's global state
        for (int wl = 0; wl < nwt; ++wl) {
            const int w = w_first + wl, own = w * per_w;
            if (own < C.i0 || own >= C.i1) continue;
            if (it == A.n_sweeps - 1) {
                for (int a = tid; a < 32 * nT; a += NT) {
                    const size_t idx = (size_t)32 * w * nT + a;
                    P.E[idx] = 3 * N - 2 * __ldcg(cnt + idx);
                    P.tau[idx] = tau8[(size_t)wl * 32 * nT + a];
                    P.sigma[idx] = sig8[(size_t)wl * 32 * nT + a];
                }
                for (int k = warp; k < nT; k += nwarp) {   // rank masks of the whole word
                    const int t = tau8[(size_t)(wl * 32 + lane) * nT + k];
                    const int pos = P.desc ? t : nT - 1 - t;
                    for (int n = 0; n <= nT; ++n) {
                        const uint32_t mk = __ballot_sync(0xFFFFFFFFu, pos >= n);
                        if (lane == (n & 31)) P.lt[((size_t)w * nT + k) * LTS + n] = mk;
                    }
                }
            } else {
                int32_t *other = A.Ecnt + (size_t)(ebuf ^ 1) * P.Rp * nT + (size_t)32 * w * nT;
                for (int a = tid; a < 32 * nT; a += NT) other[a] = 0;   // next energy sweep's counters
            }
        }
        ebuf ^= 1;
        __syncthreads();
    }
}

}  // namespace ea
