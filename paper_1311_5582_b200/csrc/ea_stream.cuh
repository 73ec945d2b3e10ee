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
// (identical in every block: same counters, same Philox draws) and rebuilds its mask tables,
// while the first tiles of the next sweep are already in flight.  No lattice word moves in a
// swap.  Scheduling notes (measured, profiles/): the warp scheduler serves high
// warp ids first, so the block's HIGHEST warps issue the TMA copies, flush the counters and wait
// on the grid barrier; with warp 0 in those roles every batch waited for it.
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
    int Wn;                  // realization words of THIS launch (P's pointers, w0 and r0 are offset to
                             // its first word; P.W and P.Rp stay the strides of the whole problem)
    int32_t *Ecnt;           // [2][Rp][nT] satisfied-bond counters (zero on entry)
    const uint4 *bucket;
    const uchar4 *trip;
    RankKey K;
    uint32_t rk[20];
    int MS;                  // most items one block can get = ceil(items / grid)
    int MW;                  // most words one block can meet
    int swap_win;            // swap thresholds for m in [-swap_win, -1] are staged in smem
    int esm_off;             // byte offset (16 B aligned) of the swap-phase staging area in smem
    int batch_off;           // byte offset (16 B aligned) of the batch list in smem
    unsigned int *gbar;      // grid barrier word (zero before the first launch; self-resetting)
#ifdef EA_TRACE
    unsigned long long *trace;   // builder's aid: [block][8 sweeps][8] globaltimer stamps of the phases, or null
#endif
};

// Phase time stamps exist only in builds with -DEA_TRACE; the product build compiles them away.
__device__ __forceinline__ void trace_stamp(const StreamArgs &A, int it, int slot)
{
#ifdef EA_TRACE
    if (A.trace && threadIdx.x == 0 && it < 8) {
        unsigned long long t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        A.trace[((size_t)blockIdx.x * 8 + it) * 8 + slot] = t;
    }
#else
    (void)A; (void)it; (void)slot;
#endif
}

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
    static constexpr int NB = BUF_BYTES <= 20480 ? 4 : 2;  // slots per batch (same word and slab)
    static constexpr int NST = 2 * NB;                     // ring stages of ONE slot each
    static constexpr int MBAR_BYTES = 192;                 // full[NST], empty[NST], batch count
    static_assert(NST <= 10 && 16 * NST + 8 <= MBAR_BYTES, "stage bookkeeping");
};

// (mbarrier / TMA bulk copy helpers: ea_resident.cuh)


// One batch = up to NB consecutive slots of one (word, slab) group; the block's batch list is
// fixed for the whole launch and sits in shared memory.
struct StreamBatch { int pos, cnt, w, slab; };

// Per-block constants of the streaming kernel.
template <int L>
struct StreamCtx {
    int i0, i1;                  // my items [i0, i1), item = (w * NSLAB + slab) * nT + k
    int nb;                      // my batches
    int nT, LTS, MTS;
    int tid, lane, qx, y, zl;
    uint32_t ov, oyp, oym, ozp, ozm;   // byte offsets inside the other-parity buffer
    uint64_t *full;              // [NST]: the stage's tile has landed (TMA transaction count)
    uint64_t *empty;             // [NST]: all warps have finished reading the stage
    const StreamBatch *batch;
    unsigned char *bufs;
    uint4 *mt;
    uint32_t *lt;
    int32_t *Eacc;               // [items][32] satisfied-bond counts of the running half-sweep
    RankCtx R;
};

// The ring: NST stages of one slot each.  The block's items of a half-sweep are numbered
// li = 0 .. i1-i0-1 in processing order; item li uses stage li % NST.  full[st] counts the TMA
// bytes of a fill, empty[st] the 16 warps that have finished reading it: the only block-wide
// barriers left are those of the grid barrier between half-sweeps, and a warp may run up to
// NST - 1 slots ahead of the slowest one.
//
// TMA bulk loads of item li into stage st, issued by three lanes of one warp (lane = piece):
// the slab's own-parity words (contiguous) and the other parity's planes z0-1 .. z0+ZS
// (periodic wrap = 2 pieces).  `sub` = lane index inside the slot's group of three.
template <int L>
__device__ __forceinline__ void stream_issue_item(const StreamArgs &A, const StreamCtx<L> &C, int p, int li, int piece)
{
    using Gm = ResGeom<L>;
    using Sg = StreamGeom<L>;
    constexpr int N = Gm::N, Nh = Gm::Nh, QPP = Sg::QPP, ZS = Sg::ZS, NT = Sg::NTHR, NSLAB = Sg::NSLAB;
    constexpr uint32_t PLB = QPP * 16;       // bytes per plane and parity
    const Params &P = A.P;
    const int item = C.i0 + li, k = item % C.nT, grp = item / C.nT, w = grp / NSLAB, slab = grp % NSLAB;
    const int st = li % Sg::NST, z0 = slab * ZS;
    if (piece == 0) mbar_expect_tx(&C.full[st], (uint32_t)Sg::BUF_BYTES);
    const uint32_t *base = P.spin + ((size_t)k * P.W + w) * N;
    unsigned char *dst = C.bufs + (size_t)st * Sg::BUF_BYTES;
    const uint32_t *ob = base + (1 - p) * Nh;
    unsigned char *od = dst + Sg::OWN_BYTES;
    const void *src;
    uint32_t bytes;
    if (piece == 0) {
        src = base + p * Nh + (size_t)slab * NT * 4; bytes = Sg::OWN_BYTES;
    } else if (z0 == 0) {
        if (piece == 1) { dst = od; src = ob + (size_t)(L - 1) * QPP * 4; bytes = PLB; }
        else { dst = od + PLB; src = ob; bytes = (ZS + 1) * PLB; }
    } else if (z0 + ZS == L) {
        if (piece == 1) { dst = od; src = ob + (size_t)(z0 - 1) * QPP * 4; bytes = (ZS + 1) * PLB; }
        else { dst = od + (ZS + 1) * PLB; src = ob; bytes = PLB; }
    } else {
        dst = od; src = ob + (size_t)(z0 - 1) * QPP * 4; bytes = piece == 1 ? (ZS + 2) * PLB : 0u;
    }
    if (bytes) bulk_g2s(dst, src, bytes, &C.full[st]);
}

// Start of a half-sweep (every stage is free: the grid barrier has just been passed): the first
// NST items, issued by the lanes of the block's HIGHEST warp in parallel (lane = 3 * item + piece).
// The proxy fence orders the previous phase's global stores (made visible by the grid barrier)
// before the asynchronous-proxy reads.  efill: bit st = parity of the number of fills of stage st.
template <int L>
__device__ __forceinline__ void stream_prime(const StreamArgs &A, const StreamCtx<L> &C, int p, uint32_t &efill)
{
    using Sg = StreamGeom<L>;
    if ((C.tid >> 5) != Sg::NTHR / 32 - 1) return;
    const int n = min(Sg::NST, C.i1 - C.i0);
    fence_proxy_async();
    if (C.lane < 3 * n) stream_issue_item<L>(A, C, p, C.lane / 3, C.lane % 3);
    efill ^= (1u << n) - 1u;
}

// A warp has finished reading item li: release its stage; the block's highest warp (first in the
// scheduler's order, so it runs ahead) then refills the stage of item li - 1, which the slowest
// warp has normally left by now, with item li - 1 + NST.
template <int L>
__device__ __forceinline__ void stream_release(const StreamArgs &A, const StreamCtx<L> &C, int p, int li, uint32_t &efill)
{
    using Sg = StreamGeom<L>;
    __syncwarp();
    if (C.lane == 0) mbar_arrive(&C.empty[li % Sg::NST]);
    if ((C.tid >> 5) != Sg::NTHR / 32 - 1) return;
    const int lj = li - 1;
    if (lj < 0 || lj + Sg::NST >= C.i1 - C.i0) return;
    const int st = lj % Sg::NST;
    mbar_wait(&C.empty[st], ((efill >> st) & 1u) ^ 1u);     // fill n is consumed in phase n - 1
    if (C.lane < 3) stream_issue_item<L>(A, C, p, lj + Sg::NST, C.lane);
    efill ^= 1u << st;
    __syncwarp();
}

// One half-sweep (parity p) over the block's batches; the first NST items are in flight
// (stream_prime).  ENERGY: also count the satisfied bonds of the updated (parity-1) sites.
template <int L, bool FAST, bool ENERGY, int NC = 3>
__device__ __forceinline__ void stream_consume(const StreamArgs &A, const StreamCtx<L> &C, int p, uint32_t g,
                                               uint32_t &phase, uint32_t &efill)
{
    using Gm = ResGeom<L>;
    using Sg = StreamGeom<L>;
    constexpr int N = Gm::N, Nh = Gm::Nh, QR = Gm::QR, ZS = Sg::ZS, NT = Sg::NTHR;
    constexpr int NST = Sg::NST, NSLAB = Sg::NSLAB;
    const Params &P = A.P;
    const int nT = C.nT, tid = C.tid;
    int cur_grp = -1, s = 0, q = 0;
    QuadJ J;
    PhiloxQuad PQ{};
    Planes fin[4];
    for (int b = 0; b < C.nb; ++b) {
        __syncwarp();
        const StreamBatch B = C.batch[b];
        const int cnt = B.cnt, pos = B.pos, w = B.w;
        const int k0 = pos % nT, grp = w * NSLAB + B.slab;
        if (grp != cur_grp) {        // couplings of my quad for this (word, slab) and parity
            cur_grp = grp;
            const int z = B.slab * ZS + C.zl;
            s = (C.y + z + p) & 1;
            q = B.slab * NT + tid;
            const int qym = C.qx + QR * (wrap_dec(C.y, L) + L * z);
            const int qzm = C.qx + QR * (C.y + L * wrap_dec(z, L));
            J = load_quad_j<L>(P.coup + (size_t)w * 3 * N, p, s, q, C.qx, qym, qzm);
            PQ = philox_quad_init((uint32_t)q, P.w0 + (uint32_t)w, A.rk);
        }
        const uint32_t c3 = (uint32_t)p << 16;
        if (!ENERGY) {
            for (int i = 0; i < cnt; ++i) {
                const int li = pos + i - C.i0, st = li % NST;
                const uint4 rnd = philox_quad(PQ, g, c3 | (uint32_t)(k0 + i), A.rk);
                mbar_wait(&C.full[st], (phase >> st) & 1u);
                phase ^= 1u << st;
                const char *buf = reinterpret_cast<const char *>(C.bufs + (size_t)st * Sg::BUF_BYTES);
                const uint4 res = update_quad_mem<L, FAST, false, false, false, NC>(
                    buf + 16 * tid, buf + Sg::OWN_BYTES, C.ov, C.oyp, C.oym, C.ozp, C.ozm, C.qx, C.lt + li * C.LTS,
                    C.mt + (size_t)li * C.MTS, C.R, J, s, rnd, fin);
                reinterpret_cast<uint4 *>(P.spin + ((size_t)(k0 + i) * P.W + w) * N + p * Nh)[q] = res;
                stream_release<L>(A, C, p, li, efill);
            }
        } else {
            for (int i0 = 0; i0 < cnt; i0 += 4) {      // the batch's (up to four) slots share one butterfly
                constexpr int NPE = NC == 4 ? 6 : 5;
                uint32_t en[4][NPE];
#pragma unroll
                for (int h = 0; h < 4; ++h) {
                    const int i = i0 + h;
                    if (i < cnt) {
                        const int li = pos + i - C.i0, st = li % NST;
                        const uint4 rnd = philox_quad(PQ, g, c3 | (uint32_t)(k0 + i), A.rk);
                        mbar_wait(&C.full[st], (phase >> st) & 1u);
                        phase ^= 1u << st;
                        const char *buf = reinterpret_cast<const char *>(C.bufs + (size_t)st * Sg::BUF_BYTES);
                        const uint4 res = update_quad_mem<L, FAST, true, false, false, NC>(
                            buf + 16 * tid, buf + Sg::OWN_BYTES, C.ov, C.oyp, C.oym, C.ozp, C.ozm, C.qx,
                            C.lt + li * C.LTS, C.mt + (size_t)li * C.MTS, C.R, J, s, rnd, fin);
                        reinterpret_cast<uint4 *>(P.spin + ((size_t)(k0 + i) * P.W + w) * N + p * Nh)[q] = res;
                        if constexpr (NC == 4) {
                            // field: T = (satisfied bonds) + |h| (spins that pay the field energy) over my four
                            // parity-1 sites (new words) and the four parity-0 sites of the index-aligned quad
                            // of the tile (every quad of the slab is met once): E = (3 + |h|) N - 2 T
                            const uint4 v4 = *reinterpret_cast<const uint4 *>(buf + Sg::OWN_BYTES + C.ov);
                            stream_release<L>(A, C, p, li, efill);
                            uint32_t e5[5], x4[4], y5[5];
                            quad_sum(fin, e5);
                            const uint32_t inv = P.h > 0 ? 0xFFFFFFFFu : 0u;      // h > 0: down spins pay
                            const uint32_t xs[8] = {res.x ^ inv, res.y ^ inv, res.z ^ inv, res.w ^ inv,
                                                    v4.x ^ inv, v4.y ^ inv, v4.z ^ inv, v4.w ^ inv};
                            count8(xs, x4);
                            const bool two = (P.h & 1) == 0;
                            y5[0] = two ? 0u : x4[0]; y5[1] = two ? x4[0] : x4[1]; y5[2] = two ? x4[1] : x4[2];
                            y5[3] = two ? x4[2] : x4[3]; y5[4] = two ? x4[3] : 0u;
                            vsum<5>(e5, y5, en[h]);
                        } else {
                            stream_release<L>(A, C, p, li, efill);
                            quad_sum(fin, en[h]);
                        }
                    } else {
#pragma unroll
                        for (int j = 0; j < NPE; ++j) en[h][j] = 0;
                    }
                }
                uint32_t tot[NPE + 5];
                warp_sum4_t<NPE>(en, C.lane, tot);
                const int i_mine = i0 + 2 * (C.lane >> 4) + ((C.lane >> 3) & 1);
                if (i_mine < cnt) add_counts_t<NPE + 5>(tot, C.lane & 7, C.Eacc + (pos + i_mine - C.i0) * 32);
            }
        }
    }
}

// End of the parity-1 half-sweep: the block's per-item shared counters go to the global
// satisfied-bond counters [ebuf][r][k] (before the grid barrier, so that every block sees them
// after it) and are cleared for the next energy sweep.
template <int L>
__device__ __forceinline__ void stream_flush_counts(const StreamArgs &A, const StreamCtx<L> &C, int ebuf)
{
    using Sg = StreamGeom<L>;
    const Params &P = A.P;
    __syncthreads();
    for (int a = C.tid; a < (C.i1 - C.i0) * 32; a += Sg::NTHR) {
        const int v = C.Eacc[a];
        C.Eacc[a] = 0;
        const int item = C.i0 + (a >> 5), k = item % C.nT, w = item / (Sg::NSLAB * C.nT);
        atomicAdd(A.Ecnt + (size_t)ebuf * P.Rp * C.nT + (size_t)(32 * w + (a & 31)) * C.nT + k, v);
    }
}

namespace cg = cooperative_groups;

// Grid-wide barrier of a cooperative launch (all blocks co-resident).  Same scheme as
// cooperative_groups::grid_group::sync (block 0 adds 0x80000000 - (G - 1), the others 1; bit 31
// flips when everybody has arrived), but the block's LAST warp waits, all lanes together.  With
// thread 0 as the lone waiter (the library version) warp 0 ran the following batch 2.5 times
// slower than the other warps (measured; the warp scheduler serves high warp ids first).
__device__ __forceinline__ void stream_grid_sync(unsigned int *bar)
{
    __syncthreads();
    if (threadIdx.x >= blockDim.x - 32) {        // the whole last warp waits: no divergence inside it
        unsigned int old = 0;
        if ((threadIdx.x & 31) == 0) {
            const unsigned int add = blockIdx.x == 0 ? 0x80000000u - (gridDim.x - 1) : 1u;
            __threadfence();
            old = atomicAdd(bar, add);
        }
        old = __shfl_sync(0xFFFFFFFFu, old, 0);
        while ((((old ^ *reinterpret_cast<volatile unsigned int *>(bar)) & 0x80000000u) == 0u)) { }
        __threadfence();
    }
    __syncthreads();
}

template <int L, bool FAST, int NC = 3>
__global__ void __launch_bounds__(StreamGeom<L>::NTHR, 1) k_stream(const StreamArgs A)
{
    using Gm = ResGeom<L>;
    using Sg = StreamGeom<L>;
    constexpr int N = Gm::N, QR = Gm::QR, QPP = Sg::QPP, NT = Sg::NTHR, NB = Sg::NB, NST = Sg::NST;
    constexpr int NSLAB = Sg::NSLAB;
    extern __shared__ __align__(128) unsigned char smraw[];
    const Params &P = A.P;
    const int nT = P.nT, LTS = P.LTS, MTS = NC * nT + 2, MS = A.MS, MW = A.MW;
    constexpr int BW = NC == 4 ? 2 : 1;          // 16-byte words per bucket entry (field: 32-byte entries)
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarp = NT >> 5;
    constexpr int NTA = NT;

    StreamCtx<L> C;
    const long long T = (long long)A.Wn * NSLAB * nT;
    C.i0 = (int)(T * blockIdx.x / gridDim.x);
    C.i1 = (int)(T * (blockIdx.x + 1) / gridDim.x);
    const int per_w = NSLAB * nT;
    const int w_first = C.i0 / per_w, nwt = (C.i1 - 1) / per_w - w_first + 1;   // words I meet (<= MW)

    // shared memory
    uint64_t *mbar = reinterpret_cast<uint64_t *>(smraw);                        // full[NST], empty[NST], number of batches
    uint4 *bucket = reinterpret_cast<uint4 *>(smraw + Sg::MBAR_BYTES);           // [n_bucket]
    unsigned char *bufs = reinterpret_cast<unsigned char *>(bucket + BW * A.K.n_bucket);   // [NST][BUF_BYTES]
    uint4 *mt = reinterpret_cast<uint4 *>(bufs + (size_t)NST * Sg::BUF_BYTES);      // [MS][MTS]
    uint32_t *lt = reinterpret_cast<uint32_t *>(mt + (size_t)MS * MTS);          // [MS][LTS]
    uint32_t *thr = lt + MS * LTS;                                               // [3][LTS]
    uchar4 *trip = reinterpret_cast<uchar4 *>(thr + NC * LTS);                   // [MTS]
    int32_t *Eacc = reinterpret_cast<int32_t *>(trip + MTS);                     // [MS][32]
    uint8_t *tau8 = reinterpret_cast<uint8_t *>(Eacc + MS * 32);                 // [MW][32][nT]
    uint8_t *sig8 = tau8 + (size_t)MW * 32 * nT;                                 // [MW][32][nT]
    const int SW = A.swap_win;
    int32_t *Esm = reinterpret_cast<int32_t *>(smraw + A.esm_off);               // [MW][32][nT] bond counts
    StreamBatch *batch = reinterpret_cast<StreamBatch *>(smraw + A.batch_off);   // [MS]
    uint32_t *swwin = reinterpret_cast<uint32_t *>(batch + MS);                  // [nT][SW] thresholds - 1
    int *swlo = reinterpret_cast<int *>(swwin + (size_t)nT * SW);                // [nT] first m of the stored range
    int *swhi = swlo + nT;                                                       // [nT] one past its last m
    int *swk = swhi + nT;                                                        // [nT] decisions left | right << 1 of the range

    for (int a = tid; a < BW * A.K.n_bucket; a += NTA) bucket[a] = A.bucket[a];
    for (int a = tid; a < NC * LTS; a += NTA) thr[a] = NC == 4 ? P.thrF[14 * LTS + a] : P.thr32[a];
    for (int a = tid; a < MTS - 1; a += NTA) trip[a] = A.trip[a];
    for (int a = tid; a < (nT - 1) * SW; a += NTA) {         // window m = -SW + i of row t
        const int t = a / SW, m = -SW + a % SW;
        const int lo = P.swp_lo[t], cn = P.swp_cnt[t];
        swwin[a] = (m >= lo && m < lo + cn) ? P.swp_val[P.swp_off[t] + (m - lo)] : 0u;
    }
    for (int t = tid; t + 1 < nT; t += NTA) {
        swlo[t] = P.swp_lo[t]; swhi[t] = P.swp_lo[t] + P.swp_cnt[t];
        swk[t] = (int)P.swp_kind[2 * t] | ((int)P.swp_kind[2 * t + 1] << 1);
    }
    for (int a = tid; a < MS * 32; a += NTA) Eacc[a] = 0;
    for (int a = tid; a < nwt * 32 * nT; a += NTA) {
        tau8[a] = P.tau[(size_t)32 * w_first * nT + a];
        sig8[a] = P.sigma[(size_t)32 * w_first * nT + a];
    }
    if (tid == 0) {
        for (int i = 0; i < NST; ++i) { mbar_init(&mbar[i], 1); mbar_init(&mbar[NST + i], NT / 32); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        // my batch list: up to NB consecutive slots of one (word, slab) group each
        int nb = 0;
        for (int pos = C.i0; pos < C.i1; ++nb) {
            const int cnt = min(min(NB, C.i1 - pos), nT - pos % nT), grp = pos / nT;
            batch[nb] = StreamBatch{pos, cnt, grp / NSLAB, grp % NSLAB};
            pos += cnt;
        }
        *reinterpret_cast<int *>(smraw + 16 * NST) = nb;
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
            (NC == 4 ? build_mt4 : build_mt)(mt + (size_t)li * MTS, lt + li * LTS, trip, nT, lane);
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
    C.full = mbar; C.empty = mbar + NST; C.batch = batch; C.bufs = bufs; C.mt = mt; C.lt = lt; C.Eacc = Eacc;
    C.nb = *reinterpret_cast<const int *>(smraw + 16 * NST);
    C.R.thr = thr; C.R.LTS = LTS; C.R.nT = nT;
    rank_ctx_key(C.R, A.K, bucket);
    C.R.z0 = P.z[0]; C.R.z1 = P.z[1]; C.R.z2 = P.z[2];
    if (NC == 4) {
        C.R.z0 = P.zF[14]; C.R.z1 = P.zF[15]; C.R.z2 = P.zF[16]; C.R.z3 = P.zF[17]; C.R.h = P.h;
        C.R.bucket0 = reinterpret_cast<const char *>(bucket) - 32 * (ptrdiff_t)A.K.key_lo;
    }
    __syncthreads();

    uint32_t nswap = A.nswap0, phase = 0, efill = 0;
    int ebuf = 0;
    stream_prime<L>(A, C, 0, efill);
    auto bar_compute = [&]() { __syncthreads(); };
    for (int it = 0; it < A.n_sweeps; ++it) {
        const uint32_t g = A.g0 + (uint32_t)it;
        const bool swap_now = A.swap_interval > 0 && ((uint64_t)g + 1) % (uint64_t)A.swap_interval == 0;
        const bool need_E = swap_now || it == A.n_sweeps - 1;
        trace_stamp(A, it, 0);
        stream_consume<L, FAST, false, NC>(A, C, 0, g, phase, efill);
        trace_stamp(A, it, 1);
        stream_grid_sync(A.gbar);
        __syncwarp();   // thread 0 spins inside grid.sync: make its warp converge again before the hot loop
        stream_prime<L>(A, C, 1, efill);
        trace_stamp(A, it, 2);
        if (need_E) {
            stream_consume<L, FAST, true, NC>(A, C, 1, g, phase, efill);
            stream_flush_counts<L>(A, C, ebuf);
        } else {
            stream_consume<L, FAST, false, NC>(A, C, 1, g, phase, efill);
        }
        trace_stamp(A, it, 3);
        stream_grid_sync(A.gbar);
        __syncwarp();   // thread 0 spins inside grid.sync: make its warp converge again before the hot loop
        // the next sweep's first tiles fly while the swap decisions are taken
        if (it + 1 < A.n_sweeps) stream_prime<L>(A, C, 0, efill);
        trace_stamp(A, it, 4);
        if (!need_E) continue;
        const int32_t *cnt = A.Ecnt + (size_t)ebuf * P.Rp * nT;     // satisfied bonds by [r][k]
        for (int a = tid; a < nwt * 32 * nT; a += NT) Esm[a] = __ldcg(cnt + (size_t)32 * w_first * nT + a);
        bar_compute();
        if (swap_now) {
            // swap round: warp per temperature pair, lane = realization; every block that works
            // on a word takes the same decisions.  E_a - E_b = -2 (c_a - c_b).
            for (int wl = 0; wl < nwt; ++wl) {
                const int r = 32 * (w_first + wl) + lane;
                uint8_t *sg_ = sig8 + (size_t)(wl * 32 + lane) * nT, *ta_ = tau8 + (size_t)(wl * 32 + lane) * nT;
                const int32_t *er = Esm + (size_t)(wl * 32 + lane) * nT;
                for (int t = (int)(nswap & 1u) + 2 * warp; t + 1 < nT; t += 2 * nwarp) {
                    const int sa = sg_[t], sb = sg_[t + 1];
                    // counts c: E = E0 - 2 c; h = 0: m = (E_a - E_b) / 4 = (c_b - c_a) / 2; field: (E_a - E_b) / 2 = c_b - c_a
                    const int m = NC == 4 ? er[sb] - er[sa] : (er[sb] - er[sa]) / 2;
                    const uint4 v = philox_rk(g, (uint32_t)t, P.r0 + (uint32_t)r, 2u << 16, A.rk);
                    bool acc;           // everything but the far tail of the stored range is in shared memory
                    if (m < swlo[t]) acc = swk[t] & 1;
                    else if (m >= swhi[t]) acc = (swk[t] >> 1) & 1;
                    else if (m >= -SW && m < 0) acc = v.x <= swwin[t * SW + m + SW];
                    else acc = v.x <= P.swp_val[P.swp_off[t] + (m - swlo[t])];
                    if (acc) {
                        sg_[t] = (uint8_t)sb; sg_[t + 1] = (uint8_t)sa;
                        ta_[sa] = (uint8_t)(t + 1); ta_[sb] = (uint8_t)t;
                    }
                }
            }
            ++nswap;
            bar_compute();
            rebuild_tables();
        }
        // the block that owns item (w, slab 0, slot 0) keeps the word's global state
        for (int wl = 0; wl < nwt; ++wl) {
            const int w = w_first + wl, own = w * per_w;
            if (own < C.i0 || own >= C.i1) continue;
            if (it == A.n_sweeps - 1) {
                for (int a = tid; a < 32 * nT; a += NT) {
                    const size_t idx = (size_t)32 * w * nT + a;
                    P.E[idx] = (3 + (NC == 4 ? abs(P.h) : 0)) * N - 2 * Esm[(size_t)wl * 32 * nT + a];
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
        bar_compute();
        trace_stamp(A, it, 5);
    }
}

}  // namespace ea
