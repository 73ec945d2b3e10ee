// ea_small.cuh -- the shared-memory-resident sweep kernel for ANY even L whose lattices fit
// shared memory (L = 2, 4, 6, 10, 12, 14, ...: the lattices of BASELINE.json's configs 1 and 3).
//
// Same organisation as k_resident (ea_resident.cuh): one thread-block cluster per realization
// word, the slots shared out over its blocks, every slot's lattice in shared memory for all
// sweeps of the call, parallel tempering inside the cluster over distributed
// shared memory (table rows move, no lattice word does).  What differs is the
// geometry: the lattice side is a run-time value and a row of L/2 same-parity sites is not a
// whole number of quads (L = 12: 6 sites), so a thread finds the six neighbours of each of its
// four sites in a table built once per launch (site_of / nbr_of, compare-select wrap) and reads them
// as single words; the word's couplings sit in shared memory next to the lattices.  These
// problems are far too small to fill a B200: what this kernel removes is the per-sweep launch /
// grid-barrier latency of the global-memory path (config 3: 18 -> 4 us per sweep).
#pragma once
#include "ea_resident.cuh"

namespace ea {

// n_sat planes of site (p, j) from shared memory only: lattice `sp` ([2][Nh]), the word's couplings
// `js` ([d][p][j], 3 N words) and the neighbour table `nb` ([3][p][j]: checkerboard indices in the
// other parity's array, + in the low and - in the high 16 bits; built once per launch, so the hot
// loop has no division by the run-time L).  Thread = site: a warp's accesses are stride-1.
__device__ __forceinline__ Planes site_planes_tab(const uint32_t *sp, const uint32_t *js, const uint32_t *nb, int p, int j,
                                                  int Nh, int N, uint32_t *self_out)
{
    const int me = p * Nh + j, ot = (1 - p) * Nh;
    const uint32_t tx = nb[me], ty = nb[N + me], tz = nb[2 * N + me];
    const int xp = (int)(tx & 0xFFFFu), xm = (int)(tx >> 16), yp = (int)(ty & 0xFFFFu), ym = (int)(ty >> 16);
    const int zp = (int)(tz & 0xFFFFu), zm = (int)(tz >> 16);
    const uint32_t *so = sp + ot;
    const uint32_t s = sp[me];
    const uint32_t e0 = xor3(s, js[me], so[xp]);
    const uint32_t e1 = xor3(s, js[ot + xm], so[xm]);
    const uint32_t e2 = xor3(s, js[N + me], so[yp]);
    const uint32_t e3 = xor3(s, js[N + ot + ym], so[ym]);
    const uint32_t e4 = xor3(s, js[2 * N + me], so[zp]);
    const uint32_t e5 = xor3(s, js[2 * N + ot + zm], so[zm]);
    *self_out = s;
    return nsat_planes(e0, e1, e2, e3, e4, e5);
}

// New word of site (p, j) of lattice `sp` for the draw u.  FAST: ranks from the bucket table; the
// rare flagged site is redone with the exact search.
template <bool FAST, bool ENERGY, int NC = 3>
__device__ __forceinline__ void update_site_any(uint32_t *sp, const uint32_t *js, const uint32_t *nb, const uint32_t *lt,
                                                const uint4 *mt, const RankCtx &R, int p, int j, int Nh, int N,
                                                uint32_t u, Planes &fin)
{
    uint32_t s, flag = FAST ? 0u : 0x80000000u, acc = 0u;
    const Planes pl = site_planes_tab(sp, js, nb, p, j, Nh, N, &s);
    if (NC == 4) {                       // field |h| <= 2: four threshold columns, the spin enters the class
        if (FAST) acc = accept_fast4(R, mt, u, pl, s, &flag);
        if ((int)flag < 0) acc = accept_exact4(R, lt, u, pl, s);
    } else {
        if (FAST) acc = accept_fast(R, mt, u, pl, &flag);
        if ((int)flag < 0) acc = accept_exact(R, lt, u, pl);
    }
    sp[p * Nh + j] = s ^ acc;
    if (ENERGY) fin = planes_after(pl, acc);
}

template <bool FAST, int NC = 3, bool MOVE = false>
__global__ void __launch_bounds__(1024, 1) k_resident_any(const ResArgs A)
{
    const int L = A.P.L, Lh = A.P.Lh, N = A.P.N, Nh = A.P.Nh, NSP = A.NQP, G = A.G, NT = NSP * G;
    extern __shared__ __align__(16) uint32_t smem[];
    const Params &P = A.P;
    const int nT = P.nT, LTS = P.LTS, S = A.S, C = A.C;
    const int w = blockIdx.x / C, rank = blockIdx.x % C;
    const int k0 = rank * S;
    const int nk = max(0, min(S, nT - k0));      // slots owned by this block
    const int tid = threadIdx.x, lane = tid & 31;
    // thread = (slot group, site of one parity): a warp's shared-memory accesses are stride-1 and the
    // four sites of a quad, which share a Philox call, sit in adjacent lanes (each computes it).
    // Sites are padded to whole warps (a warp never straddles two slot groups: the energy butterfly
    // sums the 32 lanes of one slot); the padding threads only take part in barriers and shuffles.
    const int sg = tid / NSP, j = tid % NSP, q = j >> 2;
    const bool live = j < Nh;

    // shared memory: the rank table first (fixed offset 0), lattices next (16 B aligned)
    const int MTS = NC * nT + 2, SW = A.swap_win;
    constexpr int BW = NC == 4 ? 2 : 1;                              // 16-byte words per bucket entry
    uint4 *bucket = reinterpret_cast<uint4 *>(smem);                 // [n_bucket] 16 B (field: 32 B) entries
    uint32_t *sp = smem + 4 * (size_t)BW * A.K.n_bucket;             // [S][2][Nh]
    uint4 *mt = reinterpret_cast<uint4 *>(sp + (size_t)S * N);       // [S][MTS] mask tables
    uint32_t *lt = reinterpret_cast<uint32_t *>(mt + (size_t)S * MTS);   // [S][LTS]
    uint32_t *thr = lt + S * LTS;                                    // [3][LTS]
    uchar4 *trip = reinterpret_cast<uchar4 *>(thr + NC * LTS);       // [MTS]
    int32_t *Eacc = (int32_t *)(trip + MTS);                         // [S][32] satisfied-bond counts
    int32_t *swm = Eacc + S * 32;                                    // [nT][4]: lo, cnt, off, kinds
    uint32_t *swwin = (uint32_t *)(swm + 4 * nT);                    // [nT][SW] thresholds - 1
    int16_t *Eall = (int16_t *)(swwin + nT * SW);                    // [2][nT][32], by swap-round parity
    uint8_t *tau8 = (uint8_t *)(Eall + 2 * nT * 32);                 // [32][nT]
    uint8_t *sig8 = tau8 + 32 * nT;                                  // [32][nT]
    uint32_t *mvmask = reinterpret_cast<uint32_t *>(sig8 + 32 * nT);   // [nT] moving swaps: who exchanges in pair t
    uint32_t *js = reinterpret_cast<uint32_t *>(smem) + A.any_off / 4;  // [3][2][Nh] the word's couplings
    uint32_t *nb = js + 3 * N;                                       // [3][2][Nh] neighbour table

    // ---- load state: lattices of my slots, tables, permutation of my 32 realizations
    {   // lattices: eight independent 128-bit loads in flight per thread before the first store
        // (one load per round trip cost ~25 us per launch when the state comes from HBM)
        const int VL = N / 4;
        const int total = nk * VL;
        for (int base = 0; base < total; base += 8 * NT) {
            uint4 v[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const int e = base + u * NT + tid;
                if (e < total)
                    v[u] = reinterpret_cast<const uint4 *>(P.spin + ((size_t)(k0 + e / VL) * P.W + w) * N)[e % VL];
            }
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const int e = base + u * NT + tid;
                if (e < total) reinterpret_cast<uint4 *>(sp)[e] = v[u];
            }
        }
    }
    for (int k = 0; k < nk; ++k)
        for (int a = tid; a < LTS; a += NT) lt[k * LTS + a] = P.lt[((size_t)w * nT + k0 + k) * LTS + a];
    for (int a = tid; a < NC * LTS; a += NT) thr[a] = NC == 4 ? P.thrF[14 * LTS + a] : P.thr32[a];
    for (int a = tid; a < BW * A.K.n_bucket; a += NT) bucket[a] = A.bucket[a];
    for (int a = tid; a < 32 * nT; a += NT) {
        tau8[a] = P.tau[(size_t)32 * w * nT + a];
        sig8[a] = P.sigma[(size_t)32 * w * nT + a];
    }
    for (int a = tid; a < S * 32; a += NT) Eacc[a] = 0;
    for (int a = tid; a < 2 * nT * 32; a += NT)
        Eall[a] = (int16_t)P.E[(size_t)(32 * w + (a & 31)) * nT + ((a >> 5) % nT)];   // |E| <= 3N <= 12288
    for (int a = tid; a < MTS - 1; a += NT) trip[a] = A.trip[a];
    for (int t = tid; t + 1 < nT; t += NT) {
        swm[4 * t] = P.swp_lo[t]; swm[4 * t + 1] = P.swp_cnt[t]; swm[4 * t + 2] = P.swp_off[t];
        swm[4 * t + 3] = (int)P.swp_kind[2 * t] | ((int)P.swp_kind[2 * t + 1] << 1);
    }
    __syncthreads();                                        // swm is complete
    // window m = -SW + i of row t: range constants from shared memory, so that the global loads
    // of the iterations are independent (they were three dependent round trips each: ~12 us)
#pragma unroll 4
    for (int a = tid; a < (nT - 1) * SW; a += NT) {
        const int t = a / SW, m = -SW + a % SW;
        const int lo = swm[4 * t], cnt = swm[4 * t + 1];
        swwin[a] = (m >= lo && m < lo + cnt) ? P.swp_val[swm[4 * t + 2] + (m - lo)] : 0u;
    }

    for (int a = tid; a < 3 * N; a += NT) js[a] = P.coup[(size_t)w * 3 * N + a];
    for (int a = tid; a < N; a += NT) {
        const int pp = a / Nh, ja = a - pp * Nh;
        const Nbr n = nbr_of(site_of(ja, pp, L, Lh), L, Lh);
        nb[a] = (uint32_t)n.xp | ((uint32_t)n.xm << 16);
        nb[N + a] = (uint32_t)n.yp | ((uint32_t)n.ym << 16);
        nb[2 * N + a] = (uint32_t)n.zp | ((uint32_t)n.zm << 16);
    }

    RankCtx R;
    R.thr = thr; R.LTS = LTS; R.nT = nT;
    R.z0 = P.z[0]; R.z1 = P.z[1]; R.z2 = P.z[2];
    rank_ctx_key(R, A.K, bucket);
    if (NC == 4) {
        R.z0 = P.zF[14]; R.z1 = P.zF[15]; R.z2 = P.zF[16]; R.z3 = P.zF[17]; R.h = P.h;
        R.bucket0 = reinterpret_cast<const char *>(bucket) - 32 * (ptrdiff_t)A.K.key_lo;
    }
    const uint32_t gw = P.w0 + (uint32_t)w;
    const PhiloxQuad PQ = philox_quad_init((uint32_t)q, gw, A.rk);
    cg::cluster_group cl = cg::this_cluster();
    __syncthreads();
    for (int kl = tid >> 5; kl < nk; kl += NT >> 5) (NC == 4 ? build_mt4 : build_mt)(mt + (size_t)kl * MTS, lt + kl * LTS, trip, nT, lane);
    if (C > 1) cl.sync(); else __syncthreads();   // every block's shared memory is initialised

    uint32_t nswap = A.nswap0;
    for (int it = 0; it < A.n_sweeps; ++it) {
        const uint32_t g = A.g0 + (uint32_t)it;
        const bool swap_now = A.swap_interval > 0 && ((uint64_t)g + 1) % (uint64_t)A.swap_interval == 0;
        const bool need_E = swap_now || it == A.n_sweeps - 1;
        Planes fin;
        // ---------------- parity 0
        for (int kl = sg; kl < nk; kl += G) {
            if (!live) continue;
            const uint4 rnd = philox_quad(PQ, g, (uint32_t)(k0 + kl), A.rk);
            update_site_any<FAST, false, NC>(sp + (size_t)kl * N, js, nb, lt + kl * LTS, mt + (size_t)kl * MTS, R, 0, j, Nh, N, pick(rnd, j & 3), fin);
        }
        __syncthreads();
        // ---------------- parity 1 (+ satisfied-bond count of the finished sweep)
        if (!need_E) {
            for (int kl = sg; kl < nk; kl += G) {
                if (!live) continue;
                const uint4 rnd = philox_quad(PQ, g, (1u << 16) | (uint32_t)(k0 + kl), A.rk);
                update_site_any<FAST, false, NC>(sp + (size_t)kl * N, js, nb, lt + kl * LTS, mt + (size_t)kl * MTS, R, 1, j, Nh, N, pick(rnd, j & 3), fin);
            }
            __syncthreads();
            continue;
        }
        for (int kb = sg; kb < S; kb += 4 * G) {     // batches of four slots: kb, kb+G, kb+2G, kb+3G
            constexpr int NPE = NC == 4 ? 4 : 3;
            uint32_t en[4][NPE];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int kl = kb + i * G;
                if (kl < nk && live) {
                    const uint4 rnd = philox_quad(PQ, g, (1u << 16) | (uint32_t)(k0 + kl), A.rk);
                    update_site_any<FAST, true, NC>(sp + (size_t)kl * N, js, nb, lt + kl * LTS, mt + (size_t)kl * MTS, R, 1, j, Nh, N, pick(rnd, j & 3), fin);
                    if constexpr (NC == 4) {
                        // field: T = (satisfied bonds) + |h| (spins that pay the field energy) over my parity-1
                        // site and the parity-0 site with the same index (each met once): E = (3 + |h|) N - 2 T
                        const uint32_t inv = P.h > 0 ? 0xFFFFFFFFu : 0u;      // h > 0: down spins pay
                        const uint32_t x1 = sp[(size_t)kl * N + Nh + j] ^ inv, x0 = sp[(size_t)kl * N + j] ^ inv;
                        const uint32_t c0 = x0 ^ x1, c1 = x0 & x1;              // 0..2 paying spins
                        const bool two = (P.h & 1) == 0;
                        const uint32_t a3[3] = {fin.b0, fin.b1, fin.b2};
                        const uint32_t b3[3] = {two ? 0u : c0, two ? c0 : c1, two ? c1 : 0u};
                        vsum<3>(a3, b3, en[i]);
                    } else {
                        en[i][0] = fin.b0; en[i][1] = fin.b1; en[i][2] = fin.b2;
                    }
                } else {
#pragma unroll
                    for (int jj = 0; jj < NPE; ++jj) en[i][jj] = 0;
                }
            }
            uint32_t tot[NPE + 5];
            warp_sum4_t<NPE>(en, lane, tot);
            const int i_mine = 2 * (lane >> 4) + ((lane >> 3) & 1);
            const int kl = kb + i_mine * G;
            if (kl < nk) add_counts_t<NPE + 5>(tot, lane & 7, Eacc + kl * 32);
        }
        __syncthreads();
        // ---- energies of my slots: E = 3N - 2 (satisfied bonds); pushed into every block of
        //      the cluster (distributed shared memory), buffer chosen by the swap-round parity
        int16_t *Ebuf = Eall + (nswap & 1u) * nT * 32;
        for (int a = tid; a < nk * 32; a += NT) {
            const int e = (3 + (NC == 4 ? abs(P.h) : 0)) * N - 2 * Eacc[a];
            Eacc[a] = 0;
            const int dst = k0 * 32 + a;
            if (C > 1) {
                for (int rr = 0; rr < C; ++rr) cl.map_shared_rank(Ebuf, rr)[dst] = (int16_t)e;
            } else {
                Ebuf[dst] = (int16_t)e;
            }
        }
        if (!swap_now) { __syncthreads(); continue; }
        // ---- swap round: warp per temperature pair, lane = realization.  Every block of the
        //      cluster computes all pairs of its word (identical results).  What does not depend on
        //      the energies (the slots of the pair, the draw) is fetched while the barrier completes.
        const int warp = tid >> 5, nwarp = NT >> 5;
        const int t0 = (int)(nswap & 1u) + 2 * warp;
        uint8_t *sg_ = sig8 + lane * nT, *ta_ = tau8 + lane * nT;
        if (C > 1) cluster_arrive();
        int sa0 = 0, sb0 = 0;
        uint32_t v0 = 0;
        if (t0 + 1 < nT) {
            sa0 = sg_[t0]; sb0 = sg_[t0 + 1];
            v0 = philox_rk(g, (uint32_t)t0, P.r0 + (uint32_t)(32 * w + lane), 2u << 16, A.rk).x;
        }
        if (C > 1) cluster_wait(); else __syncthreads();
        for (int t = t0; t + 1 < nT; t += 2 * nwarp) {
            int sa = sa0, sb = sb0;
            uint32_t vx = v0;
            if (t != t0) {
                sa = sg_[t]; sb = sg_[t + 1];
                vx = philox_rk(g, (uint32_t)t, P.r0 + (uint32_t)(32 * w + lane), 2u << 16, A.rk).x;
            }
            const int m = ((int)Ebuf[sa * 32 + lane] - (int)Ebuf[sb * 32 + lane]) / (NC == 4 ? 2 : 4);
            const int lo = swm[4 * t], cnt = swm[4 * t + 1], kinds = swm[4 * t + 3];
            bool acc;
            if (m < lo) acc = kinds & 1;
            else if (m >= lo + cnt) acc = (kinds >> 1) & 1;
            else if (m >= -SW && m < 0) acc = vx <= swwin[t * SW + m + SW];
            else acc = vx <= P.swp_val[swm[4 * t + 2] + (m - lo)];
            if (MOVE) {
                // data-moving swap (ea_set_swap_mode, R26): slots keep their temperatures
                // (sa = t, sb = t + 1 for ever), the accepting realizations exchange their lattices
                // below and their energies here
                const uint32_t mk = __ballot_sync(0xFFFFFFFFu, acc);
                if (acc) {
                    const int16_t x = Ebuf[sa * 32 + lane];
                    Ebuf[sa * 32 + lane] = Ebuf[sb * 32 + lane];
                    Ebuf[sb * 32 + lane] = x;
                }
                if (lane == 0) mvmask[t] = mk;
            } else if (acc) {
                sg_[t] = (uint8_t)sb; sg_[t + 1] = (uint8_t)sa;
                ta_[sa] = (uint8_t)(t + 1); ta_[sb] = (uint8_t)t;
                // rank masks: lt[slot][n] bit r = (pos_r >= n).  The position of a goes from p to p + 1
                // and that of b from p + 1 to p (descending betas; the other way round for ascending),
                // so exactly bit r of row rho toggles in both slots; row rho belongs to this pair alone
                const int rho = P.desc ? t + 1 : nT - 1 - t;
                const int la = sa - k0, lb = sb - k0;
                if ((unsigned)la < (unsigned)nk) atomicXor(&lt[la * LTS + rho], 1u << lane);
                if ((unsigned)lb < (unsigned)nk) atomicXor(&lt[lb * LTS + rho], 1u << lane);
            }
        }
        ++nswap;
        __syncthreads();
        if (MOVE) {
            // pairs (t, t + 1) of this round whose lower slot is mine: x = (a ^ b) & mask, a ^= x, b ^= x on
            // every word of the two lattices; the upper slot may be the first one of the next block
            // of the cluster (distributed shared memory), which does not touch it meanwhile
            const int par = (int)((nswap - 1u) & 1u);
            for (int kl = 0; kl < nk; ++kl) {
                const int t = k0 + kl;
                if ((t & 1) != par || t + 1 >= nT) continue;
                const uint32_t mk = mvmask[t];
                if (mk == 0u) continue;
                uint4 *pa = reinterpret_cast<uint4 *>(sp + (size_t)kl * N);
                uint4 *pb = kl + 1 < nk ? reinterpret_cast<uint4 *>(sp + (size_t)(kl + 1) * N)
                                        : reinterpret_cast<uint4 *>(cl.map_shared_rank(sp, rank + 1));
                for (int i = tid; i < N / 4; i += NT) {
                    uint4 a = pa[i], b = pb[i];
                    const uint4 x = make_uint4((a.x ^ b.x) & mk, (a.y ^ b.y) & mk, (a.z ^ b.z) & mk, (a.w ^ b.w) & mk);
                    a.x ^= x.x; a.y ^= x.y; a.z ^= x.z; a.w ^= x.w;
                    b.x ^= x.x; b.y ^= x.y; b.z ^= x.z; b.w ^= x.w;
                    pa[i] = a; pb[i] = b;
                }
            }
            if (C > 1) cl.sync(); else __syncthreads();
        } else {
            for (int kl = warp; kl < nk; kl += nwarp)     // mask tables of my slots from their rank masks
                (NC == 4 ? build_mt4 : build_mt)(mt + (size_t)kl * MTS, lt + kl * LTS, trip, nT, lane);
            __syncthreads();
        }
    }
    // the energies written last are in the buffer selected by the final nswap parity... the
    // last sweep always computes them; which buffer depends on whether that sweep swapped
    const bool last_swapped = A.swap_interval > 0 &&
                              ((uint64_t)A.g0 + (uint64_t)A.n_sweeps) % (uint64_t)A.swap_interval == 0;
    const int16_t *Elast = Eall + (((last_swapped ? nswap - 1 : nswap) & 1u) * nT * 32);
    if (C > 1) cl.sync();                         // no block exits while others may still push to it

    // ---- write back
    for (int k = 0; k < nk; ++k) {
        uint4 *dst = reinterpret_cast<uint4 *>(P.spin + ((size_t)(k0 + k) * P.W + w) * N);
        const uint4 *src = reinterpret_cast<const uint4 *>(sp + (size_t)k * N);
        for (int a = tid; a < N / 4; a += NT) dst[a] = src[a];
        for (int a = tid; a < LTS; a += NT) P.lt[((size_t)w * nT + k0 + k) * LTS + a] = lt[k * LTS + a];
        for (int a = tid; a < 32; a += NT) P.E[(size_t)(32 * w + a) * nT + k0 + k] = Elast[(k0 + k) * 32 + a];
    }
    if (rank == 0) {
        for (int a = tid; a < 32 * nT; a += NT) {
            P.tau[(size_t)32 * w * nT + a] = tau8[a];
            P.sigma[(size_t)32 * w * nT + a] = sig8[a];
        }
    }
}

}  // namespace ea
