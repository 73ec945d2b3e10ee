// ea_resident.cuh -- shared-memory-resident sweep kernel (L = 8, 16).
//
// One thread-block CLUSTER owns one realization word (32 realizations) for the whole call:
// its C blocks split the n_T slots; every slot's lattice (N words) stays in shared memory
// for all sweeps, the couplings of a thread's two quads stay in registers, and the
// parallel-tempering round exchanges 32 x n_T integer energies through distributed shared
// memory.  HBM/L2 are touched only at kernel entry and exit.  (The paper keeps one "integer
// cube" in the 16 KB scratchpad and swaps LUT rows; this is the same idea
// at sm_100a scale: 192 KB of lattices per SM, rank masks instead of LUT rows.)
//
// Thread t = (slot group sg, quad q): quad q = four x-consecutive same-parity sites
// (one 128-bit word vector); the same q is used for parity 0 and parity 1.
#pragma once
#include <cooperative_groups.h>

#include "ea_device.cuh"

namespace ea {
namespace cg = cooperative_groups;

struct ResArgs {
    Params P;
    uint32_t g0;          // global index of the first sweep of this call
    int n_sweeps;
    int swap_interval;
    uint32_t nswap0;      // swap rounds done before this call
    int C, S;             // cluster size; slots per block (last block may own fewer)
    const uint32_t *bucket;   // fast rank table (FAST variant), device memory
    int n_bucket, key_lo, key_hi, key_shift;
};

constexpr int kResPlanes = 10;   // planes of a warp's per-slot satisfied-bond count (<= 768)

// ------------------------------------------------------------------ small bit-sliced adders
__device__ __forceinline__ uint32_t mux(uint32_t a, uint32_t b, uint32_t m) { return (a & ~m) | (b & m); }

// r[0..NA] = a[0..NA) + b[0..NA)   (bit-sliced, NA planes each, result NA+1 planes)
template <int NA>
__device__ __forceinline__ void vsum(const uint32_t *a, const uint32_t *b, uint32_t *r)
{
    uint32_t c = a[0] & b[0];
    r[0] = a[0] ^ b[0];
#pragma unroll
    for (int i = 1; i < NA; ++i) {
        const uint32_t s = xor3(a[i], b[i], c);
        c = maj3(a[i], b[i], c);
        r[i] = s;
    }
    r[NA] = c;
}

// Sum of four 3-plane numbers (the final n_sat of a quad's four sites) -> 5 planes (<= 24).
__device__ __forceinline__ void quad_sum(const Planes (&f)[4], uint32_t (&o)[5])
{
    // weight 1
    const uint32_t s1 = xor3(f[0].b0, f[1].b0, f[2].b0), c1 = maj3(f[0].b0, f[1].b0, f[2].b0);
    o[0] = s1 ^ f[3].b0;
    const uint32_t c2 = s1 & f[3].b0;
    // weight 2: c1, c2, four b1
    const uint32_t s3 = xor3(c1, c2, f[0].b1), c3 = maj3(c1, c2, f[0].b1);
    const uint32_t s4 = xor3(f[1].b1, f[2].b1, f[3].b1), c4 = maj3(f[1].b1, f[2].b1, f[3].b1);
    o[1] = s3 ^ s4;
    const uint32_t c5 = s3 & s4;
    // weight 4: c3, c4, c5, four b2
    const uint32_t s6 = xor3(c3, c4, c5), c6 = maj3(c3, c4, c5);
    const uint32_t s7 = xor3(f[0].b2, f[1].b2, f[2].b2), c7 = maj3(f[0].b2, f[1].b2, f[2].b2);
    const uint32_t s8 = xor3(s6, s7, f[3].b2), c8 = maj3(s6, s7, f[3].b2);
    o[2] = s8;
    // weight 8: c6, c7, c8
    o[3] = xor3(c6, c7, c8);
    o[4] = maj3(c6, c7, c8);
}

// n_sat of a site AFTER its update: a flipped spin turns every bond around it, n -> 6 - n.
__device__ __forceinline__ Planes planes_after(const Planes &p, uint32_t acc)
{
    Planes f;
    f.b0 = p.b0;
    f.b1 = mux(p.b1, ~(p.b1 ^ p.b0), acc);
    f.b2 = mux(p.b2, ~p.b2 & ~(p.b1 & p.b0), acc);
    return f;
}

// ------------------------------------------------------------------ rank of a draw
// FAST: one look-up keyed by the leading bits of the draw (float exponent + key_shift
// mantissa bits, truncating conversion) gives the rank at the bucket's lower edge for the
// three classes; buckets hold at most one threshold per class, so one compare fixes it.
// Entries with bit 31 set (several thresholds in the bucket, or draw < 2^8) take the exact
// binary search.
struct RankCtx {
    const uint32_t *thr;     // smem [3][LTS]
    const uint32_t *bucket;  // smem
    int LTS, nT, key_lo, key_hi, key_shift;
    int z0, z1, z2;
};

__device__ __forceinline__ uint32_t bucket_entry(const RankCtx &R, uint32_t u)
{
    int key = (int)(__float_as_uint(__uint2float_rz(u)) >> R.key_shift);
    key = min(max(key, R.key_lo), R.key_hi) - R.key_lo;
    return R.bucket[key];
}

__device__ __forceinline__ uint32_t accept_fast(const RankCtx &R, const uint32_t *lt, uint32_t u,
                                                uint32_t e, const Planes &p)
{
    const char *thr = (const char *)R.thr;
    const char *ltb = (const char *)lt;
    uint32_t n4 = e & 0xFFu, n5 = (e >> 8) & 0xFFu, n6 = (e >> 16) & 0xFFu;   // rank * 4
    n4 += (*(const uint32_t *)(thr + n4) < u) ? 4u : 0u;
    n5 += (*(const uint32_t *)(thr + 4 * R.LTS + n5) < u) ? 4u : 0u;
    n6 += (*(const uint32_t *)(thr + 8 * R.LTS + n6) < u) ? 4u : 0u;
    return accept_mask(p, *(const uint32_t *)(ltb + n4), *(const uint32_t *)(ltb + n5),
                       *(const uint32_t *)(ltb + n6));
}

__device__ __forceinline__ uint32_t accept_exact(const RankCtx &R, const uint32_t *lt, uint32_t u,
                                                 const Planes &p)
{
    const uint32_t m4 = lt[rank_of(u, R.thr, R.z0, R.nT)];
    const uint32_t m5 = lt[rank_of(u, R.thr + R.LTS, R.z1, R.nT)];
    const uint32_t m6 = lt[rank_of(u, R.thr + 2 * R.LTS, R.z2, R.nT)];
    return accept_mask(p, m4, m5, m6);
}

}  // namespace ea

namespace ea {

// Per-thread constant geometry + couplings of quad q for one parity.
struct QuadJ {
    uint4 ja;    // J on the x bond whose neighbour vector is v-aligned
    uint4 jb;    // J on the x bond whose neighbour vector is the shifted one
    uint4 jys, jym, jzs, jzm;
};

template <int L>
struct ResGeom {
    static constexpr int Lh = L / 2, N = L * L * L, Nh = N / 2, NQ = Nh / 4, QR = Lh / 4;
    static_assert(Lh % 4 == 0, "resident kernel needs L multiple of 8");
};

// Update the four sites of quad q (parity p) of one slot's lattice `sp` (smem, [2][Nh]).
// Returns the post-update n_sat planes of the four sites through `fin` when ENERGY.
template <int L, bool FAST, bool ENERGY>
__device__ __forceinline__ void update_quad(uint32_t *sp, const uint32_t *lt, const RankCtx &R,
                                            const QuadJ &J, int p, int s, int q, int qyp, int qym,
                                            int qzp, int qzm, const uint4 rnd, Planes (&fin)[4])
{
    using Gm = ResGeom<L>;
    uint4 *self_p = reinterpret_cast<uint4 *>(sp + p * Gm::Nh);
    const uint4 *oth = reinterpret_cast<const uint4 *>(sp + (1 - p) * Gm::Nh);
    const uint4 me = self_p[q];
    const uint4 v = oth[q];
    const uint4 yp = oth[qyp], ym = oth[qym], zp = oth[qzp], zm = oth[qzm];
    uint32_t ext = s ? v.x : v.w;
    if (Gm::QR == 2) ext = __shfl_xor_sync(0xFFFFFFFFu, ext, 1);
    uint4 sh;   // the x neighbour that is not index-aligned: x+1 if s, x-1 otherwise
    sh.x = s ? v.y : ext;
    sh.y = s ? v.z : v.x;
    sh.z = s ? v.w : v.y;
    sh.w = s ? ext : v.z;
    const uint32_t m[4] = {me.x, me.y, me.z, me.w};
    const uint32_t va[4] = {v.x, v.y, v.z, v.w}, vb[4] = {sh.x, sh.y, sh.z, sh.w};
    const uint32_t a_yp[4] = {yp.x, yp.y, yp.z, yp.w}, a_ym[4] = {ym.x, ym.y, ym.z, ym.w};
    const uint32_t a_zp[4] = {zp.x, zp.y, zp.z, zp.w}, a_zm[4] = {zm.x, zm.y, zm.z, zm.w};
    const uint32_t ja[4] = {J.ja.x, J.ja.y, J.ja.z, J.ja.w}, jb[4] = {J.jb.x, J.jb.y, J.jb.z, J.jb.w};
    const uint32_t jys[4] = {J.jys.x, J.jys.y, J.jys.z, J.jys.w}, jym[4] = {J.jym.x, J.jym.y, J.jym.z, J.jym.w};
    const uint32_t jzs[4] = {J.jzs.x, J.jzs.y, J.jzs.z, J.jzs.w}, jzm[4] = {J.jzm.x, J.jzm.y, J.jzm.z, J.jzm.w};
    const uint32_t u[4] = {rnd.x, rnd.y, rnd.z, rnd.w};
    Planes pl[4];
    uint32_t e[4];
#pragma unroll
    for (int l = 0; l < 4; ++l) {
        pl[l] = nsat_planes(xor3(m[l], ja[l], va[l]), xor3(m[l], jb[l], vb[l]),
                            xor3(m[l], jys[l], a_yp[l]), xor3(m[l], jym[l], a_ym[l]),
                            xor3(m[l], jzs[l], a_zp[l]), xor3(m[l], jzm[l], a_zm[l]));
        if (FAST) e[l] = bucket_entry(R, u[l]);
    }
    uint32_t acc[4];
    if (FAST) {
        if ((e[0] | e[1] | e[2] | e[3]) & 0x80000000u) {
#pragma unroll
            for (int l = 0; l < 4; ++l) acc[l] = accept_exact(R, lt, u[l], pl[l]);
        } else {
#pragma unroll
            for (int l = 0; l < 4; ++l) acc[l] = accept_fast(R, lt, u[l], e[l], pl[l]);
        }
    } else {
#pragma unroll
        for (int l = 0; l < 4; ++l) acc[l] = accept_exact(R, lt, u[l], pl[l]);
    }
    self_p[q] = make_uint4(m[0] ^ acc[0], m[1] ^ acc[1], m[2] ^ acc[2], m[3] ^ acc[3]);
    if (ENERGY) {
#pragma unroll
        for (int l = 0; l < 4; ++l) fin[l] = planes_after(pl[l], acc[l]);
    }
}

// Couplings of quad q for parity p from global memory ([d][p][j], 3N words per word w).
template <int L>
__device__ __forceinline__ QuadJ load_quad_j(const uint32_t *cp, int p, int s, int q, int qx, int qym,
                                             int qzm)
{
    using Gm = ResGeom<L>;
    const uint4 *jx_me = reinterpret_cast<const uint4 *>(cp + p * Gm::Nh);
    const uint4 *jx_ot = reinterpret_cast<const uint4 *>(cp + (1 - p) * Gm::Nh);
    const uint4 *jy_me = reinterpret_cast<const uint4 *>(cp + Gm::N + p * Gm::Nh);
    const uint4 *jy_ot = reinterpret_cast<const uint4 *>(cp + Gm::N + (1 - p) * Gm::Nh);
    const uint4 *jz_me = reinterpret_cast<const uint4 *>(cp + 2 * Gm::N + p * Gm::Nh);
    const uint4 *jz_ot = reinterpret_cast<const uint4 *>(cp + 2 * Gm::N + (1 - p) * Gm::Nh);
    QuadJ J;
    const uint4 jxs = jx_me[q];          // bond i -> i + x^ of my sites
    const uint4 jo = jx_ot[q];           // x bonds owned by the index-aligned other-parity sites
    // s = 1: x-1 neighbour is index-aligned (its J is jo), x+1 is shifted (J = mine, jxs)
    // s = 0: x+1 neighbour is index-aligned (J = mine, jxs), x-1 is shifted: J of sites xh-1
    if (s) {
        J.ja = jo;
        J.jb = jxs;
    } else {
        J.ja = jxs;
        const int row = q - qx;
        const int qprev = row + (qx == 0 ? Gm::QR - 1 : qx - 1);
        const uint32_t prev = cp[(1 - p) * Gm::Nh + 4 * qprev + 3];
        J.jb = make_uint4(prev, jo.x, jo.y, jo.z);
    }
    J.jys = jy_me[q];
    J.jym = jy_ot[qym];
    J.jzs = jz_me[q];
    J.jzm = jz_ot[qzm];
    return J;
}

}  // namespace ea

namespace ea {

// Warp-level sum of the per-thread 5-plane counts of four slots at once: two butterfly levels
// that halve the number of slots a lane is responsible for (no redundant work), then three
// plain butterfly levels.  On return every lane of the 8-lane group (lane>>3 ... see below)
// holds the 10-plane sum over the warp's 32 lanes of slot index  2*(lane>>4) + ((lane>>3)&1).
__device__ __forceinline__ void warp_sum4(uint32_t (&en)[4][5], int lane, uint32_t (&out)[kResPlanes])
{
    const uint32_t hi16 = (lane & 16) ? 0xFFFFFFFFu : 0u;
    const uint32_t hi8 = (lane & 8) ? 0xFFFFFFFFu : 0u;
    uint32_t a[2][6];
#pragma unroll
    for (int h = 0; h < 2; ++h) {       // keep slots {0,1} (lanes 0-15) or {2,3} (lanes 16-31)
        uint32_t keep[5], got[5];
#pragma unroll
        for (int i = 0; i < 5; ++i) {
            keep[i] = mux(en[h][i], en[2 + h][i], hi16);
            got[i] = __shfl_xor_sync(0xFFFFFFFFu, mux(en[2 + h][i], en[h][i], hi16), 16);
        }
        vsum<5>(keep, got, a[h]);
    }
    uint32_t b[7];
    {
        uint32_t keep[6], got[6];
#pragma unroll
        for (int i = 0; i < 6; ++i) {
            keep[i] = mux(a[0][i], a[1][i], hi8);
            got[i] = __shfl_xor_sync(0xFFFFFFFFu, mux(a[1][i], a[0][i], hi8), 8);
        }
        vsum<6>(keep, got, b);
    }
    uint32_t c[8], d[9];
    {
        uint32_t got[7];
#pragma unroll
        for (int i = 0; i < 7; ++i) got[i] = __shfl_xor_sync(0xFFFFFFFFu, b[i], 4);
        vsum<7>(b, got, c);
    }
    {
        uint32_t got[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) got[i] = __shfl_xor_sync(0xFFFFFFFFu, c[i], 2);
        vsum<8>(c, got, d);
    }
    {
        uint32_t got[9];
#pragma unroll
        for (int i = 0; i < 9; ++i) got[i] = __shfl_xor_sync(0xFFFFFFFFu, d[i], 1);
        vsum<9>(d, got, out);
    }
}

template <int L, int G, bool FAST>
__global__ void __launch_bounds__(ResGeom<L>::NQ *G, 1) k_resident(const ResArgs A)
{
    using Gm = ResGeom<L>;
    constexpr int N = Gm::N, NQ = Gm::NQ, QR = Gm::QR, NT = NQ * G, NW = NQ / 32;
    extern __shared__ __align__(16) uint32_t smem[];
    const Params &P = A.P;
    const int nT = P.nT, LTS = P.LTS, S = A.S, C = A.C;
    const int w = blockIdx.x / C, rank = blockIdx.x % C;
    const int k0 = rank * S;
    const int nk = max(0, min(S, nT - k0));      // slots owned by this block
    const int tid = threadIdx.x, lane = tid & 31;
    const int q = tid % NQ, sg = tid / NQ, wq = q >> 5;

    uint32_t *sp = smem;                          // [S][2][Nh]
    uint32_t *lt = sp + (size_t)S * N;            // [S][LTS]
    uint32_t *thr = lt + S * LTS;                 // [3][LTS]
    uint32_t *bucket = thr + 3 * LTS;             // [n_bucket]
    int32_t *Eall = (int32_t *)(bucket + A.n_bucket);   // [nT][32]
    uint32_t *wsum = (uint32_t *)(Eall + nT * 32);      // [S][kResPlanes][NW]
    uint8_t *tau8 = (uint8_t *)(wsum + S * kResPlanes * NW);   // [32][nT]
    uint8_t *sig8 = tau8 + 32 * nT;                             // [32][nT]

    // ---- load state: lattices of my slots, tables, permutation of my 32 realizations
    for (int k = 0; k < nk; ++k) {
        const uint4 *src = reinterpret_cast<const uint4 *>(P.spin + ((size_t)(k0 + k) * P.W + w) * N);
        uint4 *dst = reinterpret_cast<uint4 *>(sp + (size_t)k * N);
        for (int a = tid; a < N / 4; a += NT) dst[a] = src[a];
        for (int a = tid; a < LTS; a += NT) lt[k * LTS + a] = P.lt[((size_t)w * nT + k0 + k) * LTS + a];
    }
    for (int a = tid; a < 3 * LTS; a += NT) thr[a] = P.thr32[a];
    for (int a = tid; a < A.n_bucket; a += NT) bucket[a] = A.bucket[a];
    for (int a = tid; a < 32 * nT; a += NT) {
        tau8[a] = P.tau[(size_t)32 * w * nT + a];
        sig8[a] = P.sigma[(size_t)32 * w * nT + a];
    }
    for (int a = tid; a < nT * 32; a += NT) {     // Eall[k][b] <- E[32w+b][k]
        const int k = a >> 5, b = a & 31;
        Eall[a] = P.E[(size_t)(32 * w + b) * nT + k];
    }

    // ---- per-thread geometry and couplings (registers, both parities)
    const int qx = q % QR, y = (q / QR) % L, z = q / (QR * L);
    const int qyp = qx + QR * (wrap_inc(y, L) + L * z), qym = qx + QR * (wrap_dec(y, L) + L * z);
    const int qzp = qx + QR * (y + L * wrap_inc(z, L)), qzm = qx + QR * (y + L * wrap_dec(z, L));
    const int s0 = (y + z) & 1;                   // s for parity 0; parity 1 uses 1 - s0
    const uint32_t *cp = P.coup + (size_t)w * 3 * N;
    const QuadJ J0 = load_quad_j<L>(cp, 0, s0, q, qx, qym, qzm);
    const QuadJ J1 = load_quad_j<L>(cp, 1, 1 - s0, q, qx, qym, qzm);

    RankCtx R;
    R.thr = thr; R.bucket = bucket; R.LTS = LTS; R.nT = nT;
    R.key_lo = A.key_lo; R.key_hi = A.key_hi; R.key_shift = A.key_shift;
    R.z0 = P.z[0]; R.z1 = P.z[1]; R.z2 = P.z[2];
    const uint32_t gw = P.w0 + (uint32_t)w;
    __syncthreads();

    uint32_t nswap = A.nswap0;
    for (int it = 0; it < A.n_sweeps; ++it) {
        const uint32_t g = A.g0 + (uint32_t)it;
        const bool swap_now = A.swap_interval > 0 && ((uint64_t)g + 1) % (uint64_t)A.swap_interval == 0;
        const bool need_E = swap_now || it == A.n_sweeps - 1;
        Planes fin[4];
        // ---------------- parity 0
        for (int kl = sg; kl < nk; kl += G) {
            const uint4 rnd = philox4x32_10(g, (uint32_t)q, gw, (uint32_t)(k0 + kl), P.k0, P.k1);
            update_quad<L, FAST, false>(sp + (size_t)kl * N, lt + kl * LTS, R, J0, 0, s0, q, qyp, qym, qzp,
                                        qzm, rnd, fin);
        }
        __syncthreads();
        // ---------------- parity 1 (+ satisfied-bond count of the finished sweep)
        if (!need_E) {
            for (int kl = sg; kl < nk; kl += G) {
                const uint4 rnd = philox4x32_10(g, (uint32_t)q, gw, (1u << 16) | (uint32_t)(k0 + kl), P.k0, P.k1);
                update_quad<L, FAST, false>(sp + (size_t)kl * N, lt + kl * LTS, R, J1, 1, 1 - s0, q, qyp, qym,
                                            qzp, qzm, rnd, fin);
            }
        } else {
            for (int kb = sg; kb < S; kb += 4 * G) {     // batches of four slots: kb, kb+G, kb+2G, kb+3G
                uint32_t en[4][5];
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const int kl = kb + i * G;
                    if (kl < nk) {
                        const uint4 rnd = philox4x32_10(g, (uint32_t)q, gw, (1u << 16) | (uint32_t)(k0 + kl),
                                                        P.k0, P.k1);
                        update_quad<L, FAST, true>(sp + (size_t)kl * N, lt + kl * LTS, R, J1, 1, 1 - s0, q, qyp,
                                                   qym, qzp, qzm, rnd, fin);
                        quad_sum(fin, en[i]);
                    } else {
#pragma unroll
                        for (int j = 0; j < 5; ++j) en[i][j] = 0;
                    }
                }
                uint32_t tot[kResPlanes];
                warp_sum4(en, lane, tot);
                const int i_mine = 2 * (lane >> 4) + ((lane >> 3) & 1);
                const int kl = kb + i_mine * G;
                if ((lane & 7) == 0 && kl < nk) {
#pragma unroll
                    for (int j = 0; j < kResPlanes; ++j) wsum[(kl * kResPlanes + j) * NW + wq] = tot[j];
                }
            }
        }
        __syncthreads();
        if (need_E) {
            // E[k][b] = 3N - 2 * sum over warps and planes of bit b  (thread = (slot, bit))
            for (int a = tid; a < nk * 32; a += NT) {
                const int kl = a >> 5, b = a & 31;
                int cnt = 0;
                for (int j = 0; j < kResPlanes; ++j) {
                    int cj = 0;
                    for (int x = 0; x < NW; ++x) cj += (int)((wsum[(kl * kResPlanes + j) * NW + x] >> b) & 1u);
                    cnt += cj << j;
                }
                Eall[(k0 + kl) * 32 + b] = 3 * N - 2 * cnt;
            }
        }
        if (swap_now) {
            if (C > 1) {
                cg::cluster_group cl = cg::this_cluster();
                cl.sync();                            // every block's energies are in its Eall
                for (int rr = 0; rr < C; ++rr) {
                    if (rr == rank) continue;
                    const int rk0 = rr * S, rnk = max(0, min(S, nT - rk0));
                    const int32_t *rE = cl.map_shared_rank(Eall, rr);
                    for (int a = tid; a < rnk * 32; a += NT) Eall[rk0 * 32 + a] = rE[rk0 * 32 + a];
                }
                cl.sync();                            // remote reads done before anyone rewrites Eall
            } else {
                __syncthreads();
            }
            // swap round: warp per temperature pair, lane = realization (every block computes all
            // pairs of its word redundantly; results are identical)
            const int warp = tid >> 5, nwarp = NT >> 5;
            for (int t = (int)(nswap & 1u) + 2 * warp; t + 1 < nT; t += 2 * nwarp) {
                uint8_t *sg_ = sig8 + lane * nT, *ta_ = tau8 + lane * nT;
                const int sa = sg_[t], sb = sg_[t + 1];
                const int m = (Eall[sa * 32 + lane] - Eall[sb * 32 + lane]) / 4;
                const uint4 v = philox4x32_10(g, (uint32_t)t, P.r0 + (uint32_t)(32 * w + lane), 2u << 16,
                                              P.k0, P.k1);
                if (swap_accept(P, t, m, v.x)) {
                    sg_[t] = (uint8_t)sb; sg_[t + 1] = (uint8_t)sa;
                    ta_[sa] = (uint8_t)(t + 1); ta_[sb] = (uint8_t)t;
                }
            }
            ++nswap;
            __syncthreads();
            for (int kl = warp; kl < nk; kl += nwarp) {   // rank masks of my slots
                const int t = tau8[lane * nT + k0 + kl];
                const int pos = P.desc ? t : nT - 1 - t;
                for (int n = 0; n <= nT; ++n) {
                    const uint32_t mk = __ballot_sync(0xFFFFFFFFu, pos >= n);
                    if (lane == (n & 31)) lt[kl * LTS + n] = mk;
                }
            }
            __syncthreads();
        }
    }

    // ---- write back
    for (int k = 0; k < nk; ++k) {
        uint4 *dst = reinterpret_cast<uint4 *>(P.spin + ((size_t)(k0 + k) * P.W + w) * N);
        const uint4 *src = reinterpret_cast<const uint4 *>(sp + (size_t)k * N);
        for (int a = tid; a < N / 4; a += NT) dst[a] = src[a];
        for (int a = tid; a < LTS; a += NT) P.lt[((size_t)w * nT + k0 + k) * LTS + a] = lt[k * LTS + a];
        for (int a = tid; a < 32; a += NT) P.E[(size_t)(32 * w + a) * nT + k0 + k] = Eall[(k0 + k) * 32 + a];
    }
    if (rank == 0) {
        for (int a = tid; a < 32 * nT; a += NT) {
            P.tau[(size_t)32 * w * nT + a] = tau8[a];
            P.sigma[(size_t)32 * w * nT + a] = sig8[a];
        }
    }
}

}  // namespace ea
