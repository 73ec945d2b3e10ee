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

// Bucket key of a draw, filled by the host (ea_lib.cu: build_bucket_table / fill_rank_key).
// All of it is data (kernel parameters), opaque to ptxas: the multiplies stay on the FMA pipe.
struct RankKey {
    float kscale, kadd;       // g = sat(float_rz(u) * kscale + kadd): kscale = 2^-E, kadd = 2^(8 - E)
    uint32_t kmul;            // key = hi32(bits(g) * kmul) = bits(g) >> (23 - MB), kmul = 2^(9 + MB)
    uint32_t c16;             // 16
    int key_lo, n_bucket;     // table index = key - key_lo in [0, n_bucket)
};

struct ResArgs {
    Params P;
    uint32_t g0;          // global index of the first sweep of this call
    int n_sweeps;
    int swap_interval;
    uint32_t nswap0;      // swap rounds done before this call
    int C, S;             // cluster size; slots per block (last block may own fewer)
    const uint4 *bucket;      // fast rank table (FAST variant), device memory, 16 B entries
    const uchar4 *trip;       // [3 nT + 1] (n4, n5, n6) of every combined rank
    uint32_t rk[20];          // Philox round keys (k0 + r*0x9E3779B9, k1 + r*0xBB67AE85), r = 0..9
    RankKey K;                // bucket key of a draw (see RankCtx)
    int swap_win;             // swap thresholds for m in [-swap_win, -1] are staged in smem
    int NQP, G;               // k_resident_any (ea_small.cuh): quads per parity padded to whole warps, slot groups
    int any_off;              // ... byte offset (16 B aligned) of its coupling copy and neighbour table in smem
};

// Mask table of one slot from its rank masks (one warp): row n = { lt[n4], lt[n5], lt[n6], 0 },
// n = 0 .. 3 nT; row 3 nT + 1 = slow-path marker.
__device__ __forceinline__ void build_mt(uint4 *mt, const uint32_t *lt, const uchar4 *trip, int nT, int lane)
{
    for (int n = lane; n <= 3 * nT; n += 32) {
        const uchar4 t = trip[n];
        mt[n] = make_uint4(lt[t.x], lt[t.y], lt[t.z], 0u);
    }
    if (lane == 0) mt[3 * nT + 1] = make_uint4(0u, 0u, 0u, 0x80000000u);
}
// Field |h| <= 2 (four threshold columns): row n = the four rank masks of the
// quadruple whose sum is n; the "use the exact search" flag travels in the bucket entry instead.
__device__ __forceinline__ void build_mt4(uint4 *mt, const uint32_t *lt, const uchar4 *trip, int nT, int lane)
{
    for (int n = lane; n <= 4 * nT; n += 32) {
        const uchar4 t = trip[n];
        mt[n] = make_uint4(lt[t.x], lt[t.y], lt[t.z], lt[t.w]);
    }
}

constexpr int kResPlanes = 10;   // planes of a warp's per-slot satisfied-bond count (<= 768)

// Philox4x32-10 with the ten round keys taken from kernel parameters (constant bank): the
// key schedule costs no instruction in the loop.
__device__ __forceinline__ uint4 philox_rk(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                           const uint32_t (&rk)[20])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ rk[2 * r];
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ rk[2 * r + 1];
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
    }
    return make_uint4(c0, c1, c2, c3);
}

// The flip draws of a thread all have the counter (sweep g, quad q, word gw, parity | slot):
// q and gw are fixed per thread, g and the last field are the same for the whole warp.  Round 0
// and half of rounds 1 and 2 therefore depend on per-thread constants only (PhiloxQuad, computed
// once per word) or on warp-uniform values (uniform datapath): per call a thread executes 15
// IMAD.WIDE and 17 LOP3 instead of 20 and 20.  Same function as philox_rk(g, q, gw, c3, rk).
struct PhiloxQuad { uint32_t ph, pl, c1w; };

__device__ __forceinline__ PhiloxQuad philox_quad_init(uint32_t q, uint32_t gw, const uint32_t (&rk)[20])
{
    const uint64_t p1 = (uint64_t)0xCD9E8D57u * gw;
    const uint32_t a0 = (uint32_t)(p1 >> 32) ^ q ^ rk[0];          // c0 after round 0
    const uint64_t p0 = (uint64_t)0xD2511F53u * a0;                // round 1's first product
    PhiloxQuad h;
    h.ph = (uint32_t)(p0 >> 32); h.pl = (uint32_t)p0; h.c1w = (uint32_t)p1;
    return h;
}

__device__ __forceinline__ uint4 philox_quad(const PhiloxQuad &h, uint32_t g, uint32_t ctr3, const uint32_t (&rk)[20])
{
    // round 0 (c0 = g, c1 = q, c2 = gw, c3 = ctr3): everything left is warp-uniform
    const uint64_t pg = (uint64_t)0xD2511F53u * g;
    uint32_t c2 = (uint32_t)(pg >> 32) ^ ctr3 ^ rk[1];
    uint32_t c3 = (uint32_t)pg;
    uint32_t c1 = h.c1w;
    // round 1: p0 = M0 * c0 is the per-thread constant (ph : pl)
    const uint64_t q1 = (uint64_t)0xCD9E8D57u * c2;
    uint32_t c0 = (uint32_t)(q1 >> 32) ^ c1 ^ rk[2];               // uniform
    c2 = h.ph ^ c3 ^ rk[3];
    c1 = (uint32_t)q1;
    c3 = h.pl;
#pragma unroll
    for (int r = 2; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ rk[2 * r];
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ rk[2 * r + 1];
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
    }
    return make_uint4(c0, c1, c2, c3);
}

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
// Three LOP3 written out (ptxas, given the plain expressions, spent six per site here):
// 6 - n >= 4 iff n <= 2, and n >= 3 = b2 | (b1 & b0).
__device__ __forceinline__ Planes planes_after(const Planes &p, uint32_t acc)
{
    Planes f;
    f.b0 = p.b0;
    f.b1 = lop3<0xD2>(p.b1, p.b0, acc);                     // acc ? ~(b1 ^ b0) : b1
    const uint32_t ge3 = lop3<0xF8>(p.b2, p.b1, p.b0);      // b2 | (b1 & b0)
    f.b2 = lop3<0x3A>(acc, ge3, p.b2);                      // acc ? ~ge3 : b2
    return f;
}

// ------------------------------------------------------------------ rank of a draw
// FAST: one 128-bit look-up keyed by the leading bits of the draw, then one 128-bit look-up of the
// three accept masks.
//   key(u)  = bits(g) >> (23 - MB),  g = sat(float_rz(u) * 2^-E + 2^(8-E))   (I2FP, FFMA.SAT, IMAD.HI)
// is a monotone function of u with logarithmic steps (MB mantissa bits per octave); the added
// constant merges all u << 2^8 into the first bucket and the saturation all u >= 2^E (E = number
// of bits of the largest threshold) into the last one, so neither end needs a clamp and most
// draws (86 % for config 4) share ONE shared-memory address (broadcast, no bank conflicts).  The
// host evaluates the same function in double (exactly) to find every bucket's range of u.
//   bucket entry = { ~thr4, n4 + n5 + n6 at the bucket's lower edge, ~thr5, ~thr6 }
// where n_c = number of class-c thresholds <= the lower edge and thr_c = the (threshold - 1)
// of class c inside the bucket, or 0xFFFFFFFF if there is none (at most one per class).
// The COMBINED rank n = n4 + n5 + n6 of the draw is the lower-edge value plus (thr_c < u) for
// the three classes.  As u grows the triple (n4, n5, n6) only ever changes at a threshold, so
// n determines the triple: the per-slot mask table `mt` (3 nT + 2 rows of 16 bytes, rebuilt
// after every swap round) holds in row n the three rank masks { lt[n4], lt[n5], lt[n6], 0 }.
// Buckets with several thresholds of one class, and the first bucket (u < 2^8), point at the last
// row, whose fourth word is 0x80000000: the caller then redoes the quad with the exact binary search.
// The three compares are carries: (thr < u) = carry of u + ~thr (IADD3 with carry-out), summed
// into n by IADD3.X / IMAD.X.  (A 32 x 32 + 64 multiply-add would put them on the FMA pipe, but
// ptxas lowers mad.wide with a register addend to IMAD.WIDE + IADD3 + IADD3.X.)
struct RankCtx {
    const uint32_t *thr;     // smem [3][LTS]  (exact search only)
    const char *bucket0;     // smem: bucket table base - 16 * key_lo (byte address)
    int LTS, nT;
    int z0, z1, z2;
    float kscale, kadd;
    uint32_t kmul, c16;
    int h, z3;               // field variant (four columns): field of Eq. 1, zero count of the fourth column
    uint32_t c32;            // 32: its bucket entries are two 16-byte words
};

__device__ __forceinline__ void rank_ctx_key(RankCtx &R, const RankKey &K, const uint4 *bucket)
{
    R.bucket0 = reinterpret_cast<const char *>(bucket) - 16 * (ptrdiff_t)K.key_lo;
    R.kscale = K.kscale; R.kadd = K.kadd; R.kmul = K.kmul; R.c16 = K.c16;
    R.h = 0; R.z3 = 0; R.c32 = 2u * K.c16;
}

// n + (u + a overflows) + (u + b overflows) + (u + c overflows): three carries (IADD3 with a
// predicate carry-out) and their sum with n (IADD3.X / IMAD.X)
__device__ __forceinline__ uint32_t add3_carries(uint32_t u, uint32_t n, uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t r;
    asm("{\n\t.reg .b32 t, r1, r2;\n\t"
        "add.cc.u32 t, %1, %3;\n\taddc.u32 r1, %2, 0;\n\t"
        "add.cc.u32 t, %1, %4;\n\taddc.u32 r2, r1, 0;\n\t"
        "add.cc.u32 t, %1, %5;\n\taddc.u32 %0, r2, 0;\n\t}"
        : "=r"(r) : "r"(u), "r"(n), "r"(a), "r"(b), "r"(c));
    return r;
}
__device__ __forceinline__ uint32_t mad_lo(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t d;
    asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}

// accept mask of one site from the mask table `mt` of its slot; *flag |= row.w
__device__ __forceinline__ uint32_t accept_fast(const RankCtx &R, const uint4 *mt, uint32_t u,
                                                const Planes &p, uint32_t *flag)
{
    float g;
    asm("fma.rn.sat.f32 %0, %1, %2, %3;" : "=f"(g) : "f"(__uint2float_rz(u)), "f"(R.kscale), "f"(R.kadd));
    const uint32_t key = __umulhi(__float_as_uint(g), R.kmul);
    const uint4 e = *reinterpret_cast<const uint4 *>(R.bucket0 + mad_lo(key, R.c16, 0u));
    const uint32_t n = add3_carries(u, e.y, e.x, e.z, e.w);
    const uint4 row = *reinterpret_cast<const uint4 *>(reinterpret_cast<const char *>(mt) + mad_lo(n, R.c16, 0u));
    *flag |= row.w;
    return accept_mask(p, row.x, row.y, row.z);
}

__device__ __forceinline__ uint32_t accept_exact(const RankCtx &R, const uint32_t *lt, uint32_t u,
                                                 const Planes &p)
{
    const uint32_t m4 = lt[rank_of(u, R.thr, R.z0, R.nT)];
    const uint32_t m5 = lt[rank_of(u, R.thr + R.LTS, R.z1, R.nT)];
    const uint32_t m6 = lt[rank_of(u, R.thr + 2 * R.LTS, R.z2, R.nT)];
    return accept_mask(p, m4, m5, m6);
}

// ---- field |h| <= 2: four threshold columns (shifted class index, accept_mask_field), bucket
// entries of 32 bytes { ~thr_a, n at the lower edge, ~thr_b, ~thr_c | ~thr_d, slow flag, -, - }
__device__ __forceinline__ uint32_t accept_fast4(const RankCtx &R, const uint4 *mt, uint32_t u, const Planes &p,
                                                 uint32_t s, uint32_t *flag)
{
    float g;
    asm("fma.rn.sat.f32 %0, %1, %2, %3;" : "=f"(g) : "f"(__uint2float_rz(u)), "f"(R.kscale), "f"(R.kadd));
    const uint32_t key = __umulhi(__float_as_uint(g), R.kmul);
    const char *ep = R.bucket0 + mad_lo(key, R.c32, 0u);
    const uint4 e = *reinterpret_cast<const uint4 *>(ep);
    const uint2 f = *reinterpret_cast<const uint2 *>(ep + 16);
    uint32_t n = add3_carries(u, e.y, e.x, e.z, e.w);
    n = add3_carries(u, n, f.x, 0u, 0u);
    const uint4 row = *reinterpret_cast<const uint4 *>(reinterpret_cast<const char *>(mt) + mad_lo(n, R.c16, 0u));
    *flag |= f.y;
    return accept_mask_field(p, s, R.h, row.x, row.y, row.z, row.w);
}
__device__ __forceinline__ uint32_t accept_exact4(const RankCtx &R, const uint32_t *lt, uint32_t u, const Planes &p,
                                                  uint32_t s)
{
    const uint32_t m0 = lt[rank_of(u, R.thr, R.z0, R.nT)];
    const uint32_t m1 = lt[rank_of(u, R.thr + R.LTS, R.z1, R.nT)];
    const uint32_t m2 = lt[rank_of(u, R.thr + 2 * R.LTS, R.z2, R.nT)];
    const uint32_t m3 = lt[rank_of(u, R.thr + 3 * R.LTS, R.z3, R.nT)];
    return accept_mask_field(p, s, R.h, m0, m1, m2, m3);
}

// Number of set bits over eight words, per bit lane, as four planes (<= 8).
__device__ __forceinline__ void count8(const uint32_t (&x)[8], uint32_t (&o)[4])
{
    const uint32_t s1 = xor3(x[0], x[1], x[2]), c1 = maj3(x[0], x[1], x[2]);
    const uint32_t s2 = xor3(x[3], x[4], x[5]), c2 = maj3(x[3], x[4], x[5]);
    const uint32_t s3 = x[6] ^ x[7], c3 = x[6] & x[7];
    o[0] = xor3(s1, s2, s3);
    const uint32_t c4 = maj3(s1, s2, s3);
    const uint32_t s5 = xor3(c1, c2, c3), c5 = maj3(c1, c2, c3);
    o[1] = s5 ^ c4;
    const uint32_t c6 = s5 & c4;
    o[2] = c5 ^ c6;
    o[3] = c5 & c6;
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
    static_assert(Lh % 4 == 0 && (QR & (QR - 1)) == 0 && QR <= 8, "needs L in {8,16,32,64}");
};

__device__ __forceinline__ uint4 lds128(uint32_t addr)
{
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr) : "memory");
    return v;
}

// New spin words of the four sites of quad q (parity p) of one slot's lattice `sp` (smem,
// [2][Nh]); nothing is stored.  EXACT = false: ranks from the bucket table; *flag collects
// bit 31 of the entries (set: the caller must redo the quad with EXACT = true).
template <int L, bool EXACT, bool ENERGY, bool UNIS, int NC = 3>
__device__ __forceinline__ uint4 quad_core(const char *self_q, const char *oth_b, uint32_t ov, uint32_t oyp,
                                           uint32_t oym, uint32_t ozp, uint32_t ozm, int qx,
                                           const uint32_t *lt, const uint4 *mt, const RankCtx &R,
                                           const QuadJ &J, int s, const uint4 rnd, Planes (&fin)[4],
                                           uint32_t *flag)
{
    using Gm = ResGeom<L>;
    // self_q: address of the quad's own four words; oth_b: base of the other parity's words;
    // ov, oyp..ozm: byte offsets in oth_b of the index-aligned quad and of the +-y / +-z quads
    uint4 me, v, yp, ym, zp, zm;
    if (UNIS && !EXACT) {
        // resident kernel: the lattice is this block's own shared memory; shared-state-space loads at
        // (uniform slot base) + (per-thread offset) let ptxas use the [R + UR] form instead of adding
        // the cluster window base and the slot base to every one of the six addresses
        const uint32_t ob = (uint32_t)__cvta_generic_to_shared(oth_b);
        me = lds128((uint32_t)__cvta_generic_to_shared(self_q));
        v = lds128(ob + ov); yp = lds128(ob + oyp); ym = lds128(ob + oym);
        zp = lds128(ob + ozp); zm = lds128(ob + ozm);
    } else {
        me = *reinterpret_cast<const uint4 *>(self_q);
        v = *reinterpret_cast<const uint4 *>(oth_b + ov);
        yp = *reinterpret_cast<const uint4 *>(oth_b + oyp);
        ym = *reinterpret_cast<const uint4 *>(oth_b + oym);
        zp = *reinterpret_cast<const uint4 *>(oth_b + ozp);
        zm = *reinterpret_cast<const uint4 *>(oth_b + ozm);
    }
    const uint32_t m[4] = {me.x, me.y, me.z, me.w};
    const uint32_t jb[4] = {J.jb.x, J.jb.y, J.jb.z, J.jb.w};
    // x neighbour that is not index-aligned: x+1 if s, x-1 otherwise; the word beyond the quad
    // (ext) comes from the next (s) / previous (!s) quad of the row
    uint32_t eb[4];
    if (UNIS && !EXACT) {
        // s is warp-uniform (diagonal thread mapping of the resident kernel): a branch instead
        // of five selects; quads of a row sit in adjacent lanes
        const int lane = threadIdx.x & 31;
        const int ln = (lane & ~(Gm::QR - 1)) | ((lane + (s ? 1 : Gm::QR - 1)) & (Gm::QR - 1));
        if (s) {
            const uint32_t ext = Gm::QR > 1 ? __shfl_sync(0xFFFFFFFFu, v.x, ln) : v.x;
            eb[0] = xor3(m[0], jb[0], v.y); eb[1] = xor3(m[1], jb[1], v.z);
            eb[2] = xor3(m[2], jb[2], v.w); eb[3] = xor3(m[3], jb[3], ext);
        } else {
            const uint32_t ext = Gm::QR > 1 ? __shfl_sync(0xFFFFFFFFu, v.w, ln) : v.w;
            eb[0] = xor3(m[0], jb[0], ext); eb[1] = xor3(m[1], jb[1], v.x);
            eb[2] = xor3(m[2], jb[2], v.y); eb[3] = xor3(m[3], jb[3], v.z);
        }
    } else {
        uint32_t ext = s ? v.x : v.w;
        if (Gm::QR > 1) {
            if (EXACT) {   // divergent (rare) path: no shuffle, read the neighbour quad's word
                const uint32_t on = ov - 16u * qx + 16u * ((qx + (s ? 1 : Gm::QR - 1)) & (Gm::QR - 1));
                ext = *reinterpret_cast<const uint32_t *>(oth_b + on + (s ? 0 : 12));
            } else {
                const int lane = threadIdx.x & 31;
                const int ln = (lane & ~(Gm::QR - 1)) | ((lane + (s ? 1 : Gm::QR - 1)) & (Gm::QR - 1));
                ext = __shfl_sync(0xFFFFFFFFu, ext, ln);
            }
        }
        eb[0] = xor3(m[0], jb[0], s ? v.y : ext); eb[1] = xor3(m[1], jb[1], s ? v.z : v.x);
        eb[2] = xor3(m[2], jb[2], s ? v.w : v.y); eb[3] = xor3(m[3], jb[3], s ? ext : v.z);
    }
    const uint32_t va[4] = {v.x, v.y, v.z, v.w};
    const uint32_t a_yp[4] = {yp.x, yp.y, yp.z, yp.w}, a_ym[4] = {ym.x, ym.y, ym.z, ym.w};
    const uint32_t a_zp[4] = {zp.x, zp.y, zp.z, zp.w}, a_zm[4] = {zm.x, zm.y, zm.z, zm.w};
    const uint32_t ja[4] = {J.ja.x, J.ja.y, J.ja.z, J.ja.w};
    const uint32_t jys[4] = {J.jys.x, J.jys.y, J.jys.z, J.jys.w}, jym[4] = {J.jym.x, J.jym.y, J.jym.z, J.jym.w};
    const uint32_t jzs[4] = {J.jzs.x, J.jzs.y, J.jzs.z, J.jzs.w}, jzm[4] = {J.jzm.x, J.jzm.y, J.jzm.z, J.jzm.w};
    const uint32_t u[4] = {rnd.x, rnd.y, rnd.z, rnd.w};
    uint32_t out[4];
    uint32_t fl = 0;
#pragma unroll
    for (int l = 0; l < 4; ++l) {
        const Planes pl = nsat_planes(xor3(m[l], ja[l], va[l]), eb[l],
                                      xor3(m[l], jys[l], a_yp[l]), xor3(m[l], jym[l], a_ym[l]),
                                      xor3(m[l], jzs[l], a_zp[l]), xor3(m[l], jzm[l], a_zm[l]));
        uint32_t acc;
        if (NC == 4) acc = EXACT ? accept_exact4(R, lt, u[l], pl, m[l]) : accept_fast4(R, mt, u[l], pl, m[l], &fl);
        else if (EXACT) acc = accept_exact(R, lt, u[l], pl);
        else acc = accept_fast(R, mt, u[l], pl, &fl);
        out[l] = m[l] ^ acc;
        if (ENERGY) fin[l] = planes_after(pl, acc);
    }
    if (!EXACT) *flag = fl;
    return make_uint4(out[0], out[1], out[2], out[3]);
}

// The exact-search version of a quad update as an out-of-line function: it runs for about one
// quad in 10^7, and keeping it out of the hot loops saves their code size and registers.
struct QuadOut { uint4 res; Planes fin[4]; };

template <int L, bool ENERGY, int NC = 3>
__device__ __noinline__ QuadOut quad_exact(const char *self_q, const char *oth_b, uint32_t ov, uint32_t oyp,
                                           uint32_t oym, uint32_t ozp, uint32_t ozm, int qx, const uint32_t *lt,
                                           const RankCtx R, const QuadJ J, int s, const uint4 rnd)
{
    QuadOut o;
    uint32_t flag;
    o.res = quad_core<L, true, ENERGY, false, NC>(self_q, oth_b, ov, oyp, oym, ozp, ozm, qx, lt, nullptr, R, J, s, rnd,
                                                  o.fin, &flag);
    return o;
}

// New words of a quad (nothing is stored): fast rank path first; rare (or !FAST): the whole
// quad again from memory with the exact search (OOL: through the out-of-line function; measured
// +5 % for the resident kernel, -12 % for the streaming kernel, which then spills more).
template <int L, bool FAST, bool ENERGY, bool UNIS, bool OOL, int NC = 3>
__device__ __forceinline__ uint4 update_quad_mem(const char *self_q, const char *oth_b, uint32_t ov,
                                                 uint32_t oyp, uint32_t oym, uint32_t ozp, uint32_t ozm, int qx,
                                                 const uint32_t *lt, const uint4 *mt, const RankCtx &R,
                                                 const QuadJ &J, int s, const uint4 rnd, Planes (&fin)[4])
{
    uint32_t flag = 0x80000000u;
    uint4 res;
    if (FAST) res = quad_core<L, false, ENERGY, UNIS, NC>(self_q, oth_b, ov, oyp, oym, ozp, ozm, qx, lt, mt, R, J, s, rnd, fin, &flag);
    if (!OOL) {
        if ((int)flag < 0) res = quad_core<L, true, ENERGY, UNIS, NC>(self_q, oth_b, ov, oyp, oym, ozp, ozm, qx, lt, mt, R, J, s, rnd, fin, &flag);
    } else if ((int)flag < 0) {
        const QuadOut o = quad_exact<L, ENERGY, NC>(self_q, oth_b, ov, oyp, oym, ozp, ozm, qx, lt, R, J, s, rnd);
        res = o.res;
        if (ENERGY) {
#pragma unroll
            for (int l = 0; l < 4; ++l) fin[l] = o.fin[l];
        }
    }
    return res;
}

// lattice `sp` = [2][Nh] words (resident and tiled kernels): update quad q of parity p in place
template <int L, bool FAST, bool ENERGY, bool UNIS, int NC = 3>
__device__ __forceinline__ void update_quad_off(uint32_t *sp, const uint32_t *lt, const uint4 *mt, const RankCtx &R,
                                                const QuadJ &J, int p, int s, int q, uint32_t oyp,
                                                uint32_t oym, uint32_t ozp, uint32_t ozm, const uint4 rnd,
                                                Planes (&fin)[4])
{
    using Gm = ResGeom<L>;
    char *self_q = reinterpret_cast<char *>(sp + p * Gm::Nh) + 16 * q;
    const char *oth_b = reinterpret_cast<const char *>(sp + (1 - p) * Gm::Nh);
    const uint4 res = update_quad_mem<L, FAST, ENERGY, UNIS, true, NC>(self_q, oth_b, 16u * q, oyp, oym, ozp, ozm,
                                                                 q & (Gm::QR - 1), lt, mt, R, J, s, rnd, fin);
    *reinterpret_cast<uint4 *>(self_q) = res;
}

// tiled kernel: neighbour quad indices
template <int L, bool FAST, bool ENERGY>
__device__ __forceinline__ void update_quad_wide(uint32_t *sp, const uint32_t *lt, const uint4 *mt, const RankCtx &R,
                                                 const QuadJ &J, int p, int s, int q, int qyp, int qym,
                                                 int qzp, int qzm, const uint4 rnd, Planes (&fin)[4])
{
    update_quad_off<L, FAST, ENERGY, false>(sp, lt, mt, R, J, p, s, q, 16u * qyp, 16u * qym, 16u * qzp, 16u * qzm, rnd, fin);
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

// Two-slot variant (fewer live registers): lanes 0-15 end up with the 10-plane sum over the warp
// of slot 0, lanes 16-31 with that of slot 1.
__device__ __forceinline__ void warp_sum2(uint32_t (&en)[2][5], int lane, uint32_t (&out)[kResPlanes])
{
    const uint32_t hi16 = (lane & 16) ? 0xFFFFFFFFu : 0u;
    uint32_t a[6];
    {
        uint32_t keep[5], got[5];
#pragma unroll
        for (int i = 0; i < 5; ++i) {
            keep[i] = mux(en[0][i], en[1][i], hi16);
            got[i] = __shfl_xor_sync(0xFFFFFFFFu, mux(en[1][i], en[0][i], hi16), 16);
        }
        vsum<5>(keep, got, a);
    }
    uint32_t b[7], c[8], d[9];
    {
        uint32_t got[6];
#pragma unroll
        for (int i = 0; i < 6; ++i) got[i] = __shfl_xor_sync(0xFFFFFFFFu, a[i], 8);
        vsum<6>(a, got, b);
    }
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

__device__ __forceinline__ void cluster_arrive()
{
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
}
__device__ __forceinline__ void cluster_wait()
{
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}


// Turn the warp's 10-plane satisfied-bond count of one slot (all 8 lanes of a group hold the
// same planes) into integers and add them to the block's per-(slot, bit) accumulators: lane i
// of the group takes realization bits i, i+8, i+16, i+24 (two 16-bit fields per word; the
// shift-and-add runs on the FMA pipe).
__device__ __forceinline__ void add_counts(const uint32_t (&tot)[kResPlanes], int i, int *acc_row)
{
    uint32_t lo = 0, hi = 0;
#pragma unroll
    for (int j = 0; j < kResPlanes; ++j) {
        lo += ((tot[j] >> i) & 0x00010001u) * (1u << j);
        hi += ((tot[j] >> (i + 8)) & 0x00010001u) * (1u << j);
    }
    atomicAdd(acc_row + i, (int)(lo & 0xFFFFu));
    atomicAdd(acc_row + i + 16, (int)(lo >> 16));
    atomicAdd(acc_row + i + 8, (int)(hi & 0xFFFFu));
    atomicAdd(acc_row + i + 24, (int)(hi >> 16));
}

// warp_sum4 for NP-plane counts: four slots in flight, two halving levels, three
// plain ones; every lane of the 8-lane group 2 (lane>>4) + ((lane>>3)&1) ends with that slot's sum.
template <int NP>
__device__ __forceinline__ void warp_sum4_t(uint32_t (&en)[4][NP], int lane, uint32_t (&out)[NP + 5])
{
    const uint32_t hi16 = (lane & 16) ? 0xFFFFFFFFu : 0u, hi8 = (lane & 8) ? 0xFFFFFFFFu : 0u;
    uint32_t a[2][NP + 1];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        uint32_t keep[NP], got[NP];
#pragma unroll
        for (int i = 0; i < NP; ++i) {
            keep[i] = mux(en[h][i], en[2 + h][i], hi16);
            got[i] = __shfl_xor_sync(0xFFFFFFFFu, mux(en[2 + h][i], en[h][i], hi16), 16);
        }
        vsum<NP>(keep, got, a[h]);
    }
    uint32_t b[NP + 2], c[NP + 3], d[NP + 4];
    {
        uint32_t keep[NP + 1], got[NP + 1];
#pragma unroll
        for (int i = 0; i < NP + 1; ++i) {
            keep[i] = mux(a[0][i], a[1][i], hi8);
            got[i] = __shfl_xor_sync(0xFFFFFFFFu, mux(a[1][i], a[0][i], hi8), 8);
        }
        vsum<NP + 1>(keep, got, b);
    }
    {
        uint32_t got[NP + 2];
#pragma unroll
        for (int i = 0; i < NP + 2; ++i) got[i] = __shfl_xor_sync(0xFFFFFFFFu, b[i], 4);
        vsum<NP + 2>(b, got, c);
    }
    {
        uint32_t got[NP + 3];
#pragma unroll
        for (int i = 0; i < NP + 3; ++i) got[i] = __shfl_xor_sync(0xFFFFFFFFu, c[i], 2);
        vsum<NP + 3>(c, got, d);
    }
    {
        uint32_t got[NP + 4];
#pragma unroll
        for (int i = 0; i < NP + 4; ++i) got[i] = __shfl_xor_sync(0xFFFFFFFFu, d[i], 1);
        vsum<NP + 4>(d, got, out);
    }
}

// Lane i (0..7) of a slot's eight lanes adds the counts of realizations i, i + 8, i + 16, i + 24 (all eight
// lanes hold the same NPL-plane totals) to the slot's row: the four bits of a plane are gathered as
// four bytes, planes 0..7 weighted into one word (a byte holds up to 255) and the rest into a second.
template <int NPL>
__device__ __forceinline__ void add_counts_t(const uint32_t (&tot)[NPL], int i, int *acc_row)
{
    static_assert(NPL <= 16, "two byte-packed accumulators");
    uint32_t lo = 0, hi = 0;
#pragma unroll
    for (int j = 0; j < (NPL < 8 ? NPL : 8); ++j) lo += ((tot[j] >> i) & 0x01010101u) * (1u << j);
#pragma unroll
    for (int j = 8; j < NPL; ++j) hi += ((tot[j] >> i) & 0x01010101u) * (1u << (j - 8));
#pragma unroll
    for (int b = 0; b < 4; ++b)
        atomicAdd(acc_row + i + 8 * b, (int)(((lo >> (8 * b)) & 0xFFu) + (((hi >> (8 * b)) & 0xFFu) << 8)));
}

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
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
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
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.global;" ::: "memory"); }
// Remote 16-byte store into the shared memory of block `rank` of the cluster that also counts its
// bytes on that block's mbarrier (st.async): the receiver waits on its own barrier, no cluster-wide
// barrier and no fence on the sender's side.
__device__ __forceinline__ void st_async_v4(void *local_dst, uint4 v, uint64_t *local_bar, int rank)
{
    uint32_t ra, rb;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"(smem_u32(local_dst)), "r"(rank));
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(rb) : "r"(smem_u32(local_bar)), "r"(rank));
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v4.b32 [%0], {%1, %2, %3, %4}, [%5];"
                 ::"r"(ra), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w), "r"(rb) : "memory");
}

// Phase clocks of k_resident, only in the -DEA_TRACE build of examples/resident_phases.py (the product
// library has none): thread 0 of block 0 adds the SM cycles between consecutive stamps of a sweep to
// g_res_trace[phase]; ea_debug_res_trace (ea_lib.cu, same build only) reads and clears the sums.
#ifdef EA_TRACE
__device__ unsigned long long g_res_trace[8];
#define RES_STAMP(i) do { if (threadIdx.x == 0 && blockIdx.x == 0) { const long long t_ = clock64(); g_res_trace[i] += (unsigned long long)(t_ - t_last); t_last = t_; } } while (0)
#else
#define RES_STAMP(i) do { } while (0)
#endif

template <int L, int G, bool FAST, int NC = 3, bool MOVE = false>
__global__ void __launch_bounds__(ResGeom<L>::NQ *G, 1) k_resident(const ResArgs A)
{
#ifdef EA_TRACE
    long long t_last = clock64();
#endif
    using Gm = ResGeom<L>;
    constexpr int N = Gm::N, NQ = Gm::NQ, QR = Gm::QR, NT = NQ * G;
    extern __shared__ __align__(16) uint32_t smem[];
    const Params &P = A.P;
    const int nT = P.nT, LTS = P.LTS, S = A.S, C = A.C;
    const int w = blockIdx.x / C, rank = blockIdx.x % C;
    const int k0 = rank * S;
    const int nk = max(0, min(S, nT - k0));      // slots owned by this block
    const int tid = threadIdx.x, lane = tid & 31;
    const int sg = tid / NQ;
    // Diagonal thread mapping: a warp owns whole diagonals y - z = d (mod L) of one parity of d,
    // so s = (y + z + p) & 1 = (d + p) & 1 is warp-uniform, and a quarter-warp's consecutive
    // rows (y+1, z+1) are (L+1) rows apart in memory: its 128-bit accesses hit all 32 banks once.
    constexpr int RW = 32 / QR, DW = RW / L;                       // rows, diagonals per warp
    static_assert(RW % L == 0 && DW >= 1, "a warp must hold whole diagonals (L = 8, 16)");
    const int lw = (tid % NQ) >> 5, rr = lane / QR;
    const int dq = (lw & 1) + 2 * ((lw >> 1) * DW + rr / L);       // my diagonal
    const int z = rr % L, y = (z + dq) % L, qx = lane % QR;
    const int q = qx + QR * (y + L * z);

    // shared memory: the rank table first (fixed offset 0), lattices next (16 B aligned)
    const int MTS = NC * nT + 2, SW = A.swap_win;
    constexpr int BW = NC == 4 ? 2 : 1;                              // 16-byte words per bucket entry
    uint4 *bucket = reinterpret_cast<uint4 *>(smem);                 // [n_bucket] 16 B (field: 32 B) entries
    uint32_t *sp = smem + 4 * (size_t)BW * A.K.n_bucket;             // [S][2][Nh]
    uint4 *mt = reinterpret_cast<uint4 *>(sp + (size_t)S * N);       // [S][MTS] mask tables
    uint32_t *lt = reinterpret_cast<uint32_t *>(mt + (size_t)S * MTS);   // [S][LTS]
    uint32_t *thr = lt + S * LTS;                                    // [NC][LTS]
    uchar4 *trip = reinterpret_cast<uchar4 *>(thr + NC * LTS);       // [MTS]
    int32_t *Eacc = (int32_t *)(trip + MTS);                         // [S][32] satisfied-bond counts
    int32_t *swm = Eacc + S * 32;                                    // [nT][4]: lo, cnt, off, kinds
    uint32_t *swwin = (uint32_t *)(swm + 4 * nT);                    // [nT][SW] thresholds - 1
    int16_t *Eall = (int16_t *)((reinterpret_cast<uintptr_t>(swwin + nT * SW) + 15) & ~(uintptr_t)15);   // [2][nT][32], by swap-round parity; 16 B aligned (st.async.v4)
    uint8_t *tau8 = (uint8_t *)(Eall + 2 * nT * 32);                 // [32][nT]
    uint8_t *sig8 = tau8 + 32 * nT;                                  // [32][nT]
    uint32_t *mvmask = reinterpret_cast<uint32_t *>(sig8 + 32 * nT);   // [nT] moving swaps: who exchanges in pair t
    // the other blocks' energies of a swap round arrive by st.async and are counted here
    uint64_t *ebar = reinterpret_cast<uint64_t *>((reinterpret_cast<uintptr_t>(mvmask + nT) + 7) & ~(uintptr_t)7);
    if (tid == 0) {
        mbar_init(ebar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    uint32_t ephase = 0;

    // ---- load state: lattices of my slots, tables, permutation of my 32 realizations
    {   // lattices: eight independent 128-bit loads in flight per thread before the first store
        // (one load per round trip cost ~25 us per launch when the state comes from HBM)
        constexpr int VL = N / 4;
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

    // ---- per-thread geometry and couplings (registers, both parities)
    const int qyp = qx + QR * (wrap_inc(y, L) + L * z), qym = qx + QR * (wrap_dec(y, L) + L * z);
    const int qzp = qx + QR * (y + L * wrap_inc(z, L)), qzm = qx + QR * (y + L * wrap_dec(z, L));
    const int s0 = __shfl_sync(0xFFFFFFFFu, (y + z) & 1, 0);   // warp-uniform; parity 1 uses 1 - s0
    const uint32_t *cp = P.coup + (size_t)w * 3 * N;
    const QuadJ J0 = load_quad_j<L>(cp, 0, s0, q, qx, qym, qzm);
    const QuadJ J1 = load_quad_j<L>(cp, 1, 1 - s0, q, qx, qym, qzm);
    // neighbour byte offsets: per-thread constants kept in registers (opaque, so that ptxas does
    // not rematerialize them); the loads are [register + uniform slot base + parity immediate]
    uint32_t oyp = 16u * (uint32_t)qyp, oym = 16u * (uint32_t)qym, ozp = 16u * (uint32_t)qzp, ozm = 16u * (uint32_t)qzm;
    asm volatile("" : "+r"(oyp), "+r"(oym), "+r"(ozp), "+r"(ozm));

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
    RES_STAMP(6);                                 // prologue
    for (int it = 0; it < A.n_sweeps; ++it) {
        const uint32_t g = A.g0 + (uint32_t)it;
        const bool swap_now = A.swap_interval > 0 && ((uint64_t)g + 1) % (uint64_t)A.swap_interval == 0;
        const bool need_E = swap_now || it == A.n_sweeps - 1;
        Planes fin[4];
        // ---------------- parity 0
        for (int kl = sg; kl < nk; kl += G) {
            const uint4 rnd = philox_quad(PQ, g, (uint32_t)(k0 + kl), A.rk);
            update_quad_off<L, FAST, false, true, NC>(sp + (size_t)kl * N, lt + kl * LTS, mt + (size_t)kl * MTS, R, J0, 0, s0, q, oyp, oym, ozp, ozm, rnd, fin);
        }
        __syncthreads();
        RES_STAMP(0);
        // ---------------- parity 1 (+ satisfied-bond count of the finished sweep)
        if (!need_E) {
            for (int kl = sg; kl < nk; kl += G) {
                const uint4 rnd = philox_quad(PQ, g, (1u << 16) | (uint32_t)(k0 + kl), A.rk);
                update_quad_off<L, FAST, false, true, NC>(sp + (size_t)kl * N, lt + kl * LTS, mt + (size_t)kl * MTS, R, J1, 1, 1 - s0, q,
                                                      oyp, oym, ozp, ozm, rnd, fin);
            }
            __syncthreads();
            RES_STAMP(5);
            continue;
        }
        for (int kb = sg; kb < S; kb += 4 * G) {     // batches of four slots: kb, kb+G, kb+2G, kb+3G
            constexpr int NPE = NC == 4 ? 6 : 5;
            uint32_t en[4][NPE];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int kl = kb + i * G;
                if (kl < nk) {
                    const uint4 rnd = philox_quad(PQ, g, (1u << 16) | (uint32_t)(k0 + kl), A.rk);
                    update_quad_off<L, FAST, true, true, NC>(sp + (size_t)kl * N, lt + kl * LTS, mt + (size_t)kl * MTS, R, J1, 1, 1 - s0, q,
                                                         oyp, oym, ozp, ozm, rnd, fin);
                    if constexpr (NC == 4) {
                        // field: T = (satisfied bonds) + |h| (sites whose spin pays the field energy), over my
                        // four parity-1 sites and the four parity-0 sites of the index-aligned quad, which
                        // every thread of the lattice meets exactly once: E = (3 + |h|) N - 2 T
                        uint32_t e5[5], x4[4], y5[5];
                        quad_sum(fin, e5);
                        const uint4 me4 = *reinterpret_cast<const uint4 *>(sp + (size_t)kl * N + Gm::Nh + 4 * q);
                        const uint4 v4 = *reinterpret_cast<const uint4 *>(sp + (size_t)kl * N + 4 * q);
                        const uint32_t inv = P.h > 0 ? 0xFFFFFFFFu : 0u;      // h > 0: down spins pay
                        const uint32_t xs[8] = {me4.x ^ inv, me4.y ^ inv, me4.z ^ inv, me4.w ^ inv,
                                                v4.x ^ inv, v4.y ^ inv, v4.z ^ inv, v4.w ^ inv};
                        count8(xs, x4);
                        const bool two = (P.h & 1) == 0;
                        y5[0] = two ? 0u : x4[0]; y5[1] = two ? x4[0] : x4[1]; y5[2] = two ? x4[1] : x4[2];
                        y5[3] = two ? x4[2] : x4[3]; y5[4] = two ? x4[3] : 0u;
                        vsum<5>(e5, y5, en[i]);
                    } else {
                        quad_sum(fin, en[i]);
                    }
                } else {
#pragma unroll
                    for (int j = 0; j < NPE; ++j) en[i][j] = 0;
                }
            }
            uint32_t tot[NPE + 5];
            warp_sum4_t<NPE>(en, lane, tot);
            const int i_mine = 2 * (lane >> 4) + ((lane >> 3) & 1);
            const int kl = kb + i_mine * G;
            if (kl < nk) add_counts_t<NPE + 5>(tot, lane & 7, Eacc + kl * 32);
        }
        __syncthreads();
        RES_STAMP(1);
        // ---- energies of my slots: E = 3N - 2 (satisfied bonds); pushed into every block of
        //      the cluster (distributed shared memory), buffer chosen by the swap-round parity
        int16_t *Ebuf = Eall + (nswap & 1u) * nT * 32;
        // L = 16 (few large blocks per cluster): st.async + the receiver's mbarrier; L = 8 (clusters of up
        // to eight blocks of a few warps): plain DSMEM stores + barrier.cluster, which measured faster there
        // (config 2: 2.77 against 2.85 us per sweep)
        constexpr bool ASYNC = L == 16;
        if (!ASYNC) {
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
        }
        if (ASYNC && C > 1 && swap_now && tid == 0) mbar_expect_tx(ebar, (uint32_t)(nT - nk) * 64u);   // 32 x int16 per foreign slot
        for (int a = NT - 1 - tid; ASYNC && a < nk * 4; a += NT) {    // eight energies = 16 bytes per thread; the last warps do it: with
                                                             // n_T / 2 < NT / 32 they have no pair to prepare below
            const int E0 = (3 + (NC == 4 ? abs(P.h) : 0)) * N;
            int *src = Eacc + 8 * a;
            const int4 c0 = make_int4(src[0], src[1], src[2], src[3]), c1 = make_int4(src[4], src[5], src[6], src[7]);
#pragma unroll
            for (int i = 0; i < 8; ++i) src[i] = 0;
            const uint32_t e0 = (uint32_t)(E0 - 2 * c0.x) & 0xFFFFu, e1 = (uint32_t)(E0 - 2 * c0.y), e2 = (uint32_t)(E0 - 2 * c0.z) & 0xFFFFu,
                           e3 = (uint32_t)(E0 - 2 * c0.w), e4 = (uint32_t)(E0 - 2 * c1.x) & 0xFFFFu, e5 = (uint32_t)(E0 - 2 * c1.y),
                           e6 = (uint32_t)(E0 - 2 * c1.z) & 0xFFFFu, e7 = (uint32_t)(E0 - 2 * c1.w);
            const uint4 v = make_uint4(e0 | (e1 << 16), e2 | (e3 << 16), e4 | (e5 << 16), e6 | (e7 << 16));
            uint4 *dst = reinterpret_cast<uint4 *>(Ebuf + k0 * 32) + a;
            *dst = v;
            if (C > 1 && swap_now)                            // (the last sweep of a call without a swap: own slots only)
                for (int rr = 0; rr < C; ++rr)
                    if (rr != rank) st_async_v4(dst, v, ebar, rr);
        }
        if (!swap_now) { __syncthreads(); continue; }
        // ---- swap round: warp per temperature pair, lane = realization.  Every block of the
        //      cluster computes all pairs of its word (identical results).  What does not depend on
        //      the energies (the slots of the pair, the draw) is fetched while the barrier completes.
        const int warp = tid >> 5, nwarp = NT >> 5;
        const int t0 = (int)(nswap & 1u) + 2 * warp;
        uint8_t *sg_ = sig8 + lane * nT, *ta_ = tau8 + lane * nT;
        int sa0 = 0, sb0 = 0;
        uint32_t v0 = 0;
        if (t0 + 1 < nT) {
            sa0 = sg_[t0]; sb0 = sg_[t0 + 1];
            v0 = philox_rk(g, (uint32_t)t0, P.r0 + (uint32_t)(32 * w + lane), 2u << 16, A.rk).x;
        }
        if (ASYNC) {
            __syncthreads();                                      // my own energies are in Ebuf
            if (C > 1) { mbar_wait(ebar, ephase); ephase ^= 1u; }   // ... and those of the other blocks
        } else if (C > 1) {
            cluster_arrive(); cluster_wait();
        } else {
            __syncthreads();
        }
        RES_STAMP(2);
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
        RES_STAMP(3);
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
        RES_STAMP(4);
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
    RES_STAMP(7);                                 // epilogue (issue of the write-back)
}

}  // namespace ea
