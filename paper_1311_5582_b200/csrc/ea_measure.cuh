// ea_measure.cuh -- on-device measurements: overlaps of whole
// realization words at equal temperature index, exact integer moments of the overlap and of
// the energy (the inputs of the Binder ratio, Fig. 20), coupling export.
// Product code: shares nothing with oracle/.
#pragma once
#include "ea_device.cuh"

namespace ea {

// Accumulators of one measurement series.  Pair p = (wa, wb) of realization words stands for
// the 32 realization pairs (32 wa + b, 32 wb + b); wb = -1: all-up reference.
struct Moments {
    const int32_t *wpairs;   // [P][2]
    int P, R;
    int64_t *q1;             // [P][32][nT]  sum q
    uint64_t *q2;            // [P][32][nT]  sum q^2
    uint64_t *q4;            // [P][32][nT][2]  sum q^4, 128 bit: (low, high)
    int64_t *e1;             // [R][nT]  sum E by temperature index
    uint64_t *e2;            // [R][nT]  sum E^2
    long long *corr;         // [P][32][nT][L]  sum of C(d) = sum_mu sum_p S_mu(p) S_mu(p + d)  (R23)
    uint8_t *label;          // [R][nT]  by slot: 0 no end touched yet, 1 last at index 0, 2 last at nT-1
    unsigned long long *trips;   // [R]  completed round trips 0 -> nT-1 -> 0 of the realization's replicas
};

// ------------------------------------------------------------------ gather by temperature
// T[t][w][i] = word whose bit b is the spin of realization 32w+b at the slot that currently
// holds temperature index t (i = storage index p Nh + j, the same for every slot):
//   T[t] = OR_k (spin[k] & M[k][t]),  M[k][t] = bits b with tau[32w+b][k] = t.
// After this pass the 32 overlaps of a word pair are one XNOR + positional popcount per site,
// although every bit of a word sits at its own temperature (R14).
// Block = (word w, 1024 consecutive storage words, group of eight temperature indices); a thread
// owns one 128-bit vector: it reads the n_T slots' vectors once and produces eight outputs
// (32 accumulator registers).
constexpr int kGatherThreads = 256;

__global__ void __launch_bounds__(kGatherThreads) k_gather_by_temp(Params P, uint32_t *T)
{
    extern __shared__ uint32_t sm_M[];   // [k][8]: bits of slot k at temperature index t0 + a
    const int nchunk = (P.N / 4 + kGatherThreads - 1) / kGatherThreads, ngrp = (P.nT + 7) / 8;
    const int w = blockIdx.x / (nchunk * ngrp), chunk = (blockIdx.x / ngrp) % nchunk, t0 = 8 * (blockIdx.x % ngrp);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int k = warp; k < P.nT; k += kGatherThreads / 32) {
        const int t_mine = P.tau[(size_t)(32 * w + lane) * P.nT + k];
#pragma unroll
        for (int a = 0; a < 8; ++a) {
            const uint32_t m = __ballot_sync(0xFFFFFFFFu, t_mine == t0 + a);
            if (lane == a) sm_M[k * 8 + a] = m;
        }
    }
    __syncthreads();
    const int v = chunk * kGatherThreads + threadIdx.x;   // vector index inside the lattice
    if (v >= P.N / 4) return;
    const uint4 *src = reinterpret_cast<const uint4 *>(P.spin) + (size_t)w * (P.N / 4) + v;
    uint4 *dst = reinterpret_cast<uint4 *>(T) + (size_t)w * (P.N / 4) + v;
    const size_t slot_stride = (size_t)P.W * (P.N / 4);
    uint4 acc[8];
#pragma unroll
    for (int a = 0; a < 8; ++a) acc[a] = make_uint4(0u, 0u, 0u, 0u);
#pragma unroll 4
    for (int k = 0; k < P.nT; ++k) {
        const uint4 s = src[(size_t)k * slot_stride];
#pragma unroll
        for (int a = 0; a < 8; ++a) {
            const uint32_t m = sm_M[k * 8 + a];      // zero for t0 + a >= nT
            acc[a].x |= s.x & m; acc[a].y |= s.y & m; acc[a].z |= s.z & m; acc[a].w |= s.w & m;
        }
    }
#pragma unroll
    for (int a = 0; a < 8; ++a)
        if (t0 + a < P.nT) dst[(size_t)(t0 + a) * slot_stride] = acc[a];
}

// ------------------------------------------------------------------ word overlaps + moments
// Block = (pair p, temperature index t).  agree = ~(Ta ^ Tb) per site (Tb = all ones for the
// reference), counted per bit lane in vertical (bit-sliced) counters, transposed to 32 integers
// like k_energy; q = 2 agree - N.  Lane b then adds q, q^2, q^4 to the accumulators of
// realization pair (32 wa + b, 32 wb + b): this block is their only writer, so no atomics and a
// fixed summation order.  Padding bits (index >= R) accumulate nothing.  Q (optional): the
// overlaps of this measurement, [P][32][nT].
// PL = planes of the per-thread counters: per-thread count <= 4 ceil(N / 512) < 2^PL.
template <int PL>
__global__ void __launch_bounds__(128) k_overlap_words(Params P, const uint32_t *T, Moments M, int32_t *Q)
{
    constexpr int kOverlapPlanes = PL;
    __shared__ int sm_cnt[32];
    const int p = blockIdx.x / P.nT, t = blockIdx.x % P.nT;
    const int wa = M.wpairs[2 * p], wb = M.wpairs[2 * p + 1];
    const uint32_t *Ta = T + ((size_t)t * P.W + wa) * P.N;
    const uint32_t *Tb = wb >= 0 ? T + ((size_t)t * P.W + wb) * P.N : nullptr;
    if (threadIdx.x < 32) sm_cnt[threadIdx.x] = 0;
    __syncthreads();
    uint32_t c[kOverlapPlanes + 5];          // five more planes for the sum over the warp's lanes
#pragma unroll
    for (int i = 0; i < kOverlapPlanes + 5; ++i) c[i] = 0;
    // 128-bit loads, four vectors of each word in flight per thread before the first add
    const uint4 *Va = reinterpret_cast<const uint4 *>(Ta), *Vb = reinterpret_cast<const uint4 *>(Tb);
    const int nv = P.N / 4;
    for (int i0 = threadIdx.x; i0 < nv; i0 += 4 * blockDim.x) {
        uint4 xa[4], xb[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int i = i0 + u * blockDim.x;
            xa[u] = i < nv ? Va[i] : make_uint4(0u, 0u, 0u, 0u);
            xb[u] = (i < nv && Vb) ? Vb[i] : make_uint4(~0u, ~0u, ~0u, ~0u);   // all-up reference
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            // agree = ~(a ^ b); out-of-range vectors are (0, ~0): agree = 0, counts nothing
            const uint32_t xs[4] = {~(xa[u].x ^ xb[u].x), ~(xa[u].y ^ xb[u].y), ~(xa[u].z ^ xb[u].z), ~(xa[u].w ^ xb[u].w)};
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                uint32_t x = xs[e];
#pragma unroll
                for (int l = 0; l < kOverlapPlanes; ++l) {
                    const uint32_t carry = c[l] & x;
                    c[l] ^= x;
                    x = carry;
                }
            }
        }
    }
    const int lane = threadIdx.x & 31;
    atomicAdd(&sm_cnt[lane], warp_positional_sum<PL + 5>(c, lane));
    __syncthreads();
    if (threadIdx.x >= 32) return;
    const int ra = 32 * wa + lane, rb = wb >= 0 ? 32 * wb + lane : -1;
    const bool valid = ra < M.R && rb < M.R;
    const int64_t q = valid ? 2 * (int64_t)sm_cnt[lane] - P.N : 0;
    const size_t o = ((size_t)p * 32 + lane) * P.nT + t;
    if (Q) Q[o] = (int32_t)q;
    if (!valid) return;
    const uint64_t s = (uint64_t)(q * q);
    const uint64_t lo = s * s, hi = __umul64hi(s, s);
    M.q1[o] += q;
    M.q2[o] += s;
    const uint64_t old = M.q4[2 * o];
    M.q4[2 * o] = old + lo;
    M.q4[2 * o + 1] += hi + (old + lo < old ? 1u : 0u);
}

// ------------------------------------------------------------------ plane-sum correlations
// Block = (pair p, temperature index t).  S_mu(c)[b] = sum of the local overlaps q_i = +-1 of
// realization pair b over the plane (coordinate mu of i) = c; then
//   C(d)[b] += sum_mu sum_c S_mu(c)[b] S_mu((c + d) mod L)[b]
// (R23: all that the wave-vector dependent susceptibility along the axes needs; the
// Fourier sum over the L values is done on the host).  The agreement words ~(Ta ^ Tb) of the
// lattice are staged in shared memory with coalesced 128-bit loads (STAGE; lattices of up to
// 128 KiB, L <= 32), then thread = (axis mu, plane c, sub) walks its share of the plane's L^2
// sites (scattered: the store is checkerboard-ordered) and counts agreeing bits in vertical
// counters.  The nsub threads of a plane (a power of two, adjacent lanes of one warp) add their
// counters with a bit-sliced butterfly and share out the 32 bit positions, so every plane sum has
// one writer.  One block per (p, t) is the only writer of its accumulators: no atomics at all,
// fixed order.
constexpr int kCorrThreads = 512;

template <int PL, bool STAGE>
__global__ void __launch_bounds__(kCorrThreads) k_plane_corr(Params P, const uint32_t *T, Moments M)
{
    extern __shared__ __align__(16) int sm_corr[];
    const int L = P.L;
    // sm_S[b][mu L + c], row stride 3L + 1 (odd): conflict-free both when the lanes of a warp walk
    // the planes (counting) and when they walk the bits (correlation sums)
    const int RS = 3 * L + 1;
    int *sm_S = sm_corr;                                         // [32][RS], padded to a multiple of 4 ints
    uint32_t *sm_A = reinterpret_cast<uint32_t *>(sm_corr + ((32 * RS + 3) & ~3));   // [N] (STAGE)
    const int p = blockIdx.x / P.nT, t = blockIdx.x % P.nT;
    const int wa = M.wpairs[2 * p], wb = M.wpairs[2 * p + 1];
    const uint32_t *Ta = T + ((size_t)t * P.W + wa) * P.N;
    const uint32_t *Tb = wb >= 0 ? T + ((size_t)t * P.W + wb) * P.N : nullptr;
    for (int a = threadIdx.x; a < 32 * RS; a += blockDim.x) sm_S[a] = 0;
    if (STAGE) {
        const uint4 *Va = reinterpret_cast<const uint4 *>(Ta), *Vb = reinterpret_cast<const uint4 *>(Tb);
        for (int i = threadIdx.x; i < P.N / 4; i += blockDim.x) {
            const uint4 a = Va[i];
            const uint4 b = Vb ? Vb[i] : make_uint4(~0u, ~0u, ~0u, ~0u);
            reinterpret_cast<uint4 *>(sm_A)[i] = make_uint4(~(a.x ^ b.x), ~(a.y ^ b.y), ~(a.z ^ b.z), ~(a.w ^ b.w));
        }
    }
    __syncthreads();
    int nsub = 1;                                                // threads per plane: power of two <= 32
    while (2 * nsub <= 32 && 2 * nsub * 3 * L <= (int)blockDim.x) nsub *= 2;
    const int mu = threadIdx.x / (L * nsub), rem = threadIdx.x % (L * nsub);
    const int c = rem / nsub, sub = rem % nsub;                  // the lanes of a warp share a plane: their
                                                                 // sites are neighbours in x (or y for mu = 0)
    {
        uint32_t cnt[PL + 5];                                    // five planes of headroom for the butterfly
#pragma unroll
        for (int l = 0; l < PL + 5; ++l) cnt[l] = 0;
        if (mu < 3) {
        // (u, v) = the two coordinates inside the plane, stepped without divisions
        int u = sub % L, v = sub / L;
        const int du = nsub % L, dv = nsub / L;
        for (int m = sub; m < L * L; m += nsub) {
            const int x = mu == 0 ? c : u, y = mu == 1 ? c : (mu == 0 ? u : v), z = mu == 2 ? c : v;
            const int i = ((x + y + z) & 1) * P.Nh + (x >> 1) + P.Lh * (y + L * z);
            uint32_t w = STAGE ? sm_A[i] : (Tb ? ~(Ta[i] ^ Tb[i]) : Ta[i]);
            u += du; v += dv;
            if (u >= L) { u -= L; ++v; }
#pragma unroll
            for (int l = 0; l < PL; ++l) {
                const uint32_t carry = cnt[l] & w;
                cnt[l] ^= w;
                w = carry;
            }
        }
        }
        for (int off = 1; off < nsub; off <<= 1) {               // sum over the plane's threads (all lanes shuffle)
            uint32_t carry = 0;
#pragma unroll
            for (int l = 0; l < PL + 5; ++l) {
                const uint32_t g = __shfl_xor_sync(0xFFFFFFFFu, cnt[l], off);
                const uint32_t sum = xor3(cnt[l], g, carry);
                carry = maj3(cnt[l], g, carry);
                cnt[l] = sum;
            }
        }
        if (mu < 3)
            for (int b = sub; b < 32; b += nsub) {               // my share of the bit positions
                int v = 0;
#pragma unroll
                for (int l = 0; l < PL + 5; ++l) v += (int)((cnt[l] >> b) & 1u) << l;
                sm_S[b * RS + mu * L + c] = v;
            }
    }
    __syncthreads();
    for (int a = threadIdx.x; a < 32 * RS; a += blockDim.x) sm_S[a] = 2 * sm_S[a] - L * L;   // agree - disagree
    __syncthreads();
    const int b = threadIdx.x & 31;
    const int ra = 32 * wa + b, rb = wb >= 0 ? 32 * wb + b : -1;
    if (ra >= M.R || rb >= M.R) return;
    for (int d = threadIdx.x >> 5; d < L; d += blockDim.x >> 5) {
        long long s = 0;
        for (int a = 0; a < 3; ++a)
            for (int q = 0; q < L; ++q) {
                const int q2 = q + d >= L ? q + d - L : q + d;
                s += (long long)sm_S[b * RS + a * L + q] * (long long)sm_S[b * RS + a * L + q2];
            }
        M.corr[(((size_t)p * 32 + b) * P.nT + t) * L + d] += s;
    }
}

// sum E and sum E^2 by temperature index, and the round-trip bookkeeping of the replica in
// slot k = t (R22: a replica that is back at temperature index 0 after having been at
// nT-1 completes a round trip; observed at measurement times).  One thread per (r, t).
__global__ void k_accum_energy(Params P, Moments M)
{
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= M.R * P.nT) return;
    const int r = tid / P.nT, t = tid % P.nT;
    const int64_t e = P.E[(size_t)r * P.nT + P.sigma[(size_t)r * P.nT + t]];
    M.e1[tid] += e;
    M.e2[tid] += (uint64_t)(e * e);
    const int at = P.tau[tid];            // temperature index of the replica in slot t
    if (at == 0) {
        if (M.label[tid] == 2) atomicAdd(&M.trips[r], 1ull);
        M.label[tid] = 1;
    } else if (at == P.nT - 1) {
        M.label[tid] = 2;
    }
}

// ------------------------------------------------------------------ coupling export
// out[r][d][i] = +-1, canonical site order (the inverse of k_pack mode 1).
__global__ void k_unpack_couplings(Params P, int R, int8_t *out)
{
    const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= (int64_t)R * 3 * P.N) return;
    const int i = (int)(tid % P.N);
    const int d = (int)((tid / P.N) % 3);
    const int r = (int)(tid / ((int64_t)P.N * 3));
    const int x = i % P.L, y = (i / P.L) % P.L, z = i / (P.L * P.L);
    const int p = (x + y + z) & 1, j = (x >> 1) + P.Lh * (y + P.L * z);
    const uint32_t wv = P.coup[((size_t)(r >> 5) * 3 + d) * P.N + p * P.Nh + j];
    out[tid] = ((wv >> (r & 31)) & 1u) ? 1 : -1;
}

}  // namespace ea
