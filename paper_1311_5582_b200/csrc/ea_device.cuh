// ea_device.cuh -- device-side building blocks shared by every kernel of libea_b200.
// Product code: shares nothing with oracle/.  Conventions: DESIGN.md section 2.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace ea {

// Kernel parameters (passed by value).  All pointers are device pointers into the
// handle's workspace; layouts in DESIGN.md section 4.
struct Params {
    int L, Lh, N, Nh;        // Lh = L/2, Nh = N/2 (sites per parity)
    int nT, W, Rp;           // Rp = 32 W (padding realizations are simulated too)
    int LTS;                 // stride of one rank-mask row = nT + 1
    uint32_t k0, k1;         // Philox key
    uint32_t w0, r0;         // global index of word 0 / realization 0 (sharding)
    int desc;                // 1: betas descend with t (pos(t) = t), 0: ascend (pos = nT-1-t)
    int z[3];                // per class c = 4,5,6: number of zero thresholds (coldest first)
    uint32_t *spin;          // [k][w][p][j]
    uint32_t *coup;          // [w][d][p][j]
    uint32_t *lt;            // [w][k][n], n = 0..nT: bits b with pos(tau[32w+b][k]) >= n
    uint8_t *tau;            // [r][k] -> temperature index
    uint8_t *sigma;          // [r][t] -> slot
    int32_t *E;              // [r][k]
    const uint32_t *thr32;   // [3][nT+1]: (threshold - 1) in pos order, sentinel 0xFFFFFFFF
    const int32_t *swp_lo;   // [nT-1] first m stored in swp_val
    const int32_t *swp_cnt;  // [nT-1] number of stored m
    const int32_t *swp_off;  // [nT-1] offset into swp_val
    const uint8_t *swp_kind; // [nT-1][2] decision left / right of the stored range (0 never, 1 always)
    const uint32_t *swp_val; // (threshold - 1) for thresholds in (0, 2^32)
    // external field (ea_set_field; generic kernels only).  Appended last: the offsets of the
    // members above, which the fast kernels read from the constant bank, do not move.
    int h;                   // field of Eq. 1 (integer); 0: zero-field path
    int ediv;                // swap tables are indexed by (E_a - E_b) / ediv: 4 at h = 0, else 2
    const uint32_t *thrF;    // [18][nT+1]: rows 0..13 = class 2 n_sat + (s+1)/2, rows 14..17 = the four
                             // columns of accept_mask_field (|h| <= 2); (threshold - 1) in pos order, sentinel
    int zF[18];              // per row: number of zero thresholds, or -1: dE <= 0, always flips
};

// ---------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al. 2011 = ref. [60]).  Two 32x32->64
// multiplies (IMAD.WIDE on the FMA pipe) and two 3-input XORs (one LOP3 each) per round.
// ---------------------------------------------------------------------------------
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    return make_uint4(c0, c1, c2, c3);
}

__device__ __forceinline__ uint32_t pick(const uint4 &v, int lane)
{
    return lane == 0 ? v.x : lane == 1 ? v.y : lane == 2 ? v.z : v.w;
}

// ---------------------------------------------------------------------------------
// Bit-sliced local field (Eq. 3).  Six bond words e_d = s ^ J ^ s_nb
// (bit = 1: satisfied) are summed per bit lane into three planes n_sat = b0 + 2 b1 + 4 b2
// by a carry-save adder: two full adders, a half adder, a full adder (8 LOP3).
// ---------------------------------------------------------------------------------
// One LOP3 each, pinned with inline PTX so that ptxas keeps the 14-instruction form
// (6 bonds + 8 adder) instead of re-deriving the adder on J ^ s_nb (17-18 LOP3).
template <int LUT>
__device__ __forceinline__ uint32_t lop3(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t d;
    asm("lop3.b32 %0, %1, %2, %3, %4;" : "=r"(d) : "r"(a), "r"(b), "r"(c), "n"(LUT));
    return d;
}
__device__ __forceinline__ uint32_t xor3(uint32_t a, uint32_t b, uint32_t c) { return lop3<0x96>(a, b, c); }
__device__ __forceinline__ uint32_t maj3(uint32_t a, uint32_t b, uint32_t c) { return lop3<0xE8>(a, b, c); }

struct Planes { uint32_t b0, b1, b2; };

__device__ __forceinline__ Planes nsat_planes(uint32_t e0, uint32_t e1, uint32_t e2,
                                              uint32_t e3, uint32_t e4, uint32_t e5)
{
    const uint32_t s1 = xor3(e0, e1, e2), c1 = maj3(e0, e1, e2);
    const uint32_t s2 = xor3(e3, e4, e5), c2 = maj3(e3, e4, e5);
    Planes p;
    p.b0 = s1 ^ s2;
    const uint32_t c3 = s1 & s2;
    p.b1 = xor3(c1, c2, c3);
    p.b2 = maj3(c1, c2, c3);
    return p;
}

// Acceptance mask (Eq. 5 with the sign of DESIGN.md R1).
// m4/m5/m6 = bits whose temperature accepts a flip of class n_sat = 4/5/6 for this draw
// (m6 subset of m5 subset of m4 because thresholds fall with n_sat); n_sat <= 3 always flips.
__device__ __forceinline__ uint32_t accept_mask(const Planes &p, uint32_t m4, uint32_t m5, uint32_t m6)
{
    const uint32_t t1 = m5 | (~p.b0 & m4);
    const uint32_t t2 = m6 | (~p.b1 & t1);
    return ~p.b2 | t2;
}

// Field with |h| <= 2.  dE = 4 n_sat - 12 - 2 h s depends on (n_sat, s) only
// through a shifted index:
//   h = +-1:  c'  = n_sat + x,    dE = 4 (c' - 3) - 2;   h = +-2:  c'' = n_sat + 2 x,  dE = 4 (c'' - 4),
// x = [s = -1] for h > 0, [s = +1] for h < 0 (a one-bit bit-sliced add).  Column j = 0..3 stands for
// dE_j = 4 j + 2 (odd h) or 4 j + 4 (even h); smaller dE always flip.  m_j = bits whose temperature
// accepts a flip of column j for this draw.
__device__ __forceinline__ uint32_t accept_mask_field(const Planes &p, uint32_t s, int h, uint32_t m0,
                                                      uint32_t m1, uint32_t m2, uint32_t m3)
{
    const uint32_t x = h > 0 ? ~s : s;
    if (h & 1) {
        const uint32_t p0 = p.b0 ^ x, c0 = p.b0 & x;
        const uint32_t p1 = p.b1 ^ c0, c1 = p.b1 & c0;
        const uint32_t p2 = p.b2 ^ c1;                       // c' = (p2 p1 p0) in 0..7; columns <-> c' = 4..7
        const uint32_t lo = (m0 & ~p0) | (m1 & p0), hi = (m2 & ~p0) | (m3 & p0);
        return ~p2 | (lo & ~p1) | (hi & p1);
    }
    const uint32_t p0 = p.b0;
    const uint32_t p1 = p.b1 ^ x, c1 = p.b1 & x;
    const uint32_t p2 = p.b2 ^ c1, p3 = p.b2 & c1;           // c'' = (p3 p2 p1 p0) in 0..8; columns <-> 5..8
    const uint32_t in567 = p2 & (p1 | p0);
    const uint32_t sel = (m0 & ~p1) | (p1 & ((m1 & ~p0) | (m2 & p0)));   // c'' = 5: p1 = 0 (and p0 = 1)
    return (p3 & m3) | (~p3 & (~in567 | sel));
}

// n_c(u) = number of pos with threshold <= u = z + #{n in [z, nT): thr32[n] < u};
// thr32 ascending in n with sentinel thr32[nT] = 0xFFFFFFFF.  Generic binary search.
__device__ __forceinline__ int rank_of(uint32_t u, const uint32_t *thr32, int z, int nT)
{
    int lo = z, hi = nT;
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (thr32[mid] < u) lo = mid + 1; else hi = mid;
    }
    return lo;
}

// Positional popcount across a warp.  c[0..PL) are bit-sliced per-thread counters (plane i has
// weight 2^i, bit b of every plane belongs to realization b); the sum over the 32 lanes must stay
// below 2^PL.  Five butterfly levels of bit-sliced ripple adds (2 LOP3 + 1 SHFL per plane and
// level) leave the warp total in every lane; lane b then returns the integer of bit position b.
template <int PL>
__device__ __forceinline__ int warp_positional_sum(uint32_t (&c)[PL], int lane)
{
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) {
        uint32_t carry = 0;
#pragma unroll
        for (int i = 0; i < PL; ++i) {
            const uint32_t g = __shfl_xor_sync(0xFFFFFFFFu, c[i], off);
            const uint32_t s = xor3(c[i], g, carry);
            carry = maj3(c[i], g, carry);
            c[i] = s;
        }
    }
    int v = 0;
#pragma unroll
    for (int i = 0; i < PL; ++i) v += (int)((c[i] >> lane) & 1u) << i;
    return v;
}

// Coordinates of checkerboard index j of parity p:  j = xh + Lh (y + L z), x = 2 xh + ((y+z+p)&1).
struct Site { int xh, y, z, s; };
__device__ __forceinline__ Site site_of(int j, int p, int L, int Lh)
{
    Site c;
    c.xh = j % Lh;
    const int t = j / Lh;
    c.y = t % L;
    c.z = t / L;
    c.s = (c.y + c.z + p) & 1;
    return c;
}
__device__ __forceinline__ int wrap_inc(int a, int n) { return a + 1 == n ? 0 : a + 1; }
__device__ __forceinline__ int wrap_dec(int a, int n) { return a == 0 ? n - 1 : a - 1; }

// Checkerboard indices (in the OTHER parity's array) of the six neighbours of a site.
struct Nbr { int xp, xm, yp, ym, zp, zm; };
__device__ __forceinline__ Nbr nbr_of(const Site &c, int L, int Lh)
{
    Nbr n;
    const int row = Lh * (c.y + L * c.z);
    n.xp = row + (c.s ? wrap_inc(c.xh, Lh) : c.xh);
    n.xm = row + (c.s ? c.xh : wrap_dec(c.xh, Lh));
    n.yp = c.xh + Lh * (wrap_inc(c.y, L) + L * c.z);
    n.ym = c.xh + Lh * (wrap_dec(c.y, L) + L * c.z);
    n.zp = c.xh + Lh * (c.y + L * wrap_inc(c.z, L));
    n.zm = c.xh + Lh * (c.y + L * wrap_dec(c.z, L));
    return n;
}

// n_sat planes of the site (p, j) of lattice `sp` (N words: [p][j]) with couplings `cp`
// ([d][p][j], 3N words).  Scalar loads; used by the generic kernels.
__device__ __forceinline__ Planes site_planes(const uint32_t *sp, const uint32_t *cp, int p, int j,
                                              int L, int Lh, int Nh, int N, uint32_t *self_out)
{
    const Site c = site_of(j, p, L, Lh);
    const Nbr n = nbr_of(c, L, Lh);
    const uint32_t *so = sp + (1 - p) * Nh;   // other parity's spins
    const uint32_t s = sp[p * Nh + j];
    const uint32_t *jx = cp, *jy = cp + N, *jz = cp + 2 * N;
    const int me = p * Nh + j, ot = (1 - p) * Nh;
    const uint32_t e0 = xor3(s, jx[me], so[n.xp]);
    const uint32_t e1 = xor3(s, jx[ot + n.xm], so[n.xm]);
    const uint32_t e2 = xor3(s, jy[me], so[n.yp]);
    const uint32_t e3 = xor3(s, jy[ot + n.ym], so[n.ym]);
    const uint32_t e4 = xor3(s, jz[me], so[n.zp]);
    const uint32_t e5 = xor3(s, jz[ot + n.zm], so[n.zm]);
    *self_out = s;
    // bit 1 <-> +1: J s s' = +1 iff an odd number of the three bits are 1 iff xor3 = 1,
    // so the XOR itself is the "satisfied" bit.
    return nsat_planes(e0, e1, e2, e3, e4, e5);
}

}  // namespace ea
