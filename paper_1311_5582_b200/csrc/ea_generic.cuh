// ea_generic.cuh -- kernels that work for every even L: seeding, the global-memory half-sweep,
// the standalone energy reduction, the PT swap round, overlap, pack/unpack.
// The sm_100a fast paths (ea_resident.cuh, ea_tiled.cuh) reuse pt_swap / energy pieces.
#pragma once
#include "ea_device.cuh"

namespace ea {

// ------------------------------------------------------------------ a1: seeding
// spin word (k, i, w) = PX(0, i>>2, w, (3<<16)|k)[i&3];  coupling word (d, i, w) =
// PX(0, i, w, 4<<16)[d].  One thread per (w, canonical site i).
__global__ void k_seed(Params P)
{
    const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= (int64_t)P.W * P.N) return;
    const int i = (int)(tid % P.N), w = (int)(tid / P.N);
    const int x = i % P.L, y = (i / P.L) % P.L, z = i / (P.L * P.L);
    const int p = (x + y + z) & 1;
    const int j = (x >> 1) + P.Lh * (y + P.L * z);
    const uint32_t gw = P.w0 + (uint32_t)w;
    const uint4 c = philox4x32_10(0u, (uint32_t)i, gw, 4u << 16, P.k0, P.k1);
    uint32_t *cp = P.coup + (size_t)w * 3 * P.N + p * P.Nh + j;
    cp[0] = c.x; cp[P.N] = c.y; cp[2 * P.N] = c.z;
    for (int k = 0; k < P.nT; ++k) {
        const uint4 s = philox4x32_10(0u, (uint32_t)(i >> 2), gw, (3u << 16) | (uint32_t)k, P.k0, P.k1);
        P.spin[((size_t)k * P.W + w) * P.N + p * P.Nh + j] = pick(s, i & 3);
    }
}

// +-J couplings with bond concentration p (ea_seed_couplings, R25): bit b of coupling word
// (d, i, w) = [PX(0, i, r, (5<<16)|d)[0] < thr], r = global realization 32 w + b, thr = floor(2^32 p)
// (64-bit compare: p = 1 sets every bit).  One thread per (w, d, canonical site i), 32 draws each.
__global__ void k_seed_couplings(Params P, unsigned long long thr)
{
    const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= (int64_t)P.W * 3 * P.N) return;
    const int i = (int)(tid % P.N), d = (int)((tid / P.N) % 3), w = (int)(tid / ((int64_t)3 * P.N));
    const int x = i % P.L, y = (i / P.L) % P.L, z = i / (P.L * P.L);
    const int p = (x + y + z) & 1;
    const int j = (x >> 1) + P.Lh * (y + P.L * z);
    uint32_t word = 0;
    for (int b = 0; b < 32; ++b) {
        const uint4 c = philox4x32_10(0u, (uint32_t)i, P.r0 + (uint32_t)(32 * w + b), (5u << 16) | (uint32_t)d, P.k0, P.k1);
        word |= (uint32_t)((unsigned long long)c.x < thr) << b;
    }
    P.coup[(size_t)w * 3 * P.N + (size_t)d * P.N + p * P.Nh + j] = word;
}

__global__ void k_identity_perm(Params P)
{
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= P.Rp * P.nT) return;
    const uint8_t k = (uint8_t)(tid % P.nT);
    P.tau[tid] = k;
    P.sigma[tid] = k;
}

// energy[r][t] = E[r][sigma[r][t]] for the first R realizations (ea_energy: north_star (4), by temperature index)
__global__ void k_energy_by_temp(Params P, int R, int32_t *out)
{
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= R * P.nT) return;
    const int r = tid / P.nT;
    out[tid] = P.E[(size_t)r * P.nT + P.sigma[tid]];
}

// sigma = inverse of tau, per realization (after tau was replaced: ea_set_state)
__global__ void k_invert_perm(Params P)
{
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= P.Rp * P.nT) return;
    const int r = tid / P.nT, k = tid % P.nT;
    P.sigma[(size_t)r * P.nT + P.tau[tid]] = (uint8_t)k;
}

// ------------------------------------------------------------------ rank masks
// lt[w][k][n] = bits b whose temperature rank pos(tau[32w+b][k]) >= n, n = 0..nT
// (the paper's "swap the rows of the table, not the lattices", in bit-sliced
// form).  One warp per (w, k), lane = bit.
__device__ __forceinline__ void build_lt_row(const Params &P, int w, int k, int lane)
{
    const int t = P.tau[(size_t)(32 * w + lane) * P.nT + k];
    const int pos = P.desc ? t : P.nT - 1 - t;
    uint32_t *row = P.lt + ((size_t)w * P.nT + k) * P.LTS;
    for (int n = 0; n <= P.nT; ++n) {
        const uint32_t m = __ballot_sync(0xFFFFFFFFu, pos >= n);
        if (lane == (n & 31)) row[n] = m;
    }
}

__global__ void k_build_lt(Params P)
{
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (warp >= P.W * P.nT) return;
    build_lt_row(P, warp / P.nT, warp % P.nT, lane);
}

// ------------------------------------------------------------------ a2-a7: generic half-sweep
// One thread per (slot k, word w, quad q): four sites, one Philox call
// PX(g, q, w, (p<<16)|k) (R17).  Global memory only; any even L.
// work item `tid` in [0, nT W Nh/4) of the zero-field half-sweep; sm_thr = smem copy of thr32
__device__ __forceinline__ void half_sweep_item(const Params &P, int p, uint32_t g, int64_t tid, const uint32_t *sm_thr)
{
    const int nq = P.Nh >> 2;
    const int q = (int)(tid % nq);
    const int w = (int)((tid / nq) % P.W);
    const int k = (int)(tid / ((int64_t)nq * P.W));
    uint32_t *sp = P.spin + ((size_t)k * P.W + w) * P.N;
    const uint32_t *cp = P.coup + (size_t)w * 3 * P.N;
    const uint32_t *lt = P.lt + ((size_t)w * P.nT + k) * P.LTS;
    const uint4 rnd = philox4x32_10(g, (uint32_t)q, P.w0 + (uint32_t)w, ((uint32_t)p << 16) | (uint32_t)k,
                                    P.k0, P.k1);
#pragma unroll
    for (int l = 0; l < 4; ++l) {
        const int j = 4 * q + l;
        uint32_t s;
        const Planes pl = site_planes(sp, cp, p, j, P.L, P.Lh, P.Nh, P.N, &s);
        const uint32_t u = pick(rnd, l);
        const uint32_t m4 = lt[rank_of(u, sm_thr, P.z[0], P.nT)];
        const uint32_t m5 = lt[rank_of(u, sm_thr + P.LTS, P.z[1], P.nT)];
        const uint32_t m6 = lt[rank_of(u, sm_thr + 2 * P.LTS, P.z[2], P.nT)];
        sp[p * P.Nh + j] = s ^ accept_mask(pl, m4, m5, m6);
    }
}

__global__ void __launch_bounds__(128) k_half_sweep_generic(Params P, int p, uint32_t g)
{
    extern __shared__ uint32_t sm_thr[];   // [3][nT+1]
    for (int a = threadIdx.x; a < 3 * P.LTS; a += blockDim.x) sm_thr[a] = P.thr32[a];
    __syncthreads();
    const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= (int64_t)P.nT * P.W * (P.Nh >> 2)) return;
    half_sweep_item(P, p, g, tid, sm_thr);
}

// ------------------------------------------------------------------ f2: half-sweep with a field
// H = -sum J s s + h sum s (Eq. 1; R21): dE = 4 n_sat - 12 - 2 h s_i, so the
// acceptance class of a bit is (n_sat, s_i): the paper's 14 table columns.  Per
// class one rank search and one rank mask; classes with dE <= 0 always flip.  Same thread
// mapping and draws as k_half_sweep_generic.
__device__ __forceinline__ void half_sweep_field_item(const Params &P, int p, uint32_t g, int64_t tid,
                                                      const uint32_t *sm_thr)
{
    const int nq = P.Nh >> 2;
    const int q = (int)(tid % nq);
    const int w = (int)((tid / nq) % P.W);
    const int k = (int)(tid / ((int64_t)nq * P.W));
    uint32_t *sp = P.spin + ((size_t)k * P.W + w) * P.N;
    const uint32_t *cp = P.coup + (size_t)w * 3 * P.N;
    const uint32_t *lt = P.lt + ((size_t)w * P.nT + k) * P.LTS;
    const uint4 rnd = philox4x32_10(g, (uint32_t)q, P.w0 + (uint32_t)w, ((uint32_t)p << 16) | (uint32_t)k,
                                    P.k0, P.k1);
#pragma unroll
    for (int l = 0; l < 4; ++l) {
        const int j = 4 * q + l;
        uint32_t s;
        const Planes pl = site_planes(sp, cp, p, j, P.L, P.Lh, P.Nh, P.N, &s);
        const uint32_t u = pick(rnd, l);
        if (P.h >= -2 && P.h <= 2) {          // four threshold columns instead of fourteen classes
            uint32_t m[4];
#pragma unroll
            for (int jc = 0; jc < 4; ++jc)
                m[jc] = lt[rank_of(u, sm_thr + (14 + jc) * P.LTS, P.zF[14 + jc], P.nT)];
            sp[p * P.Nh + j] = s ^ accept_mask_field(pl, s, P.h, m[0], m[1], m[2], m[3]);
            continue;
        }
        uint32_t acc = 0;
        for (int c = 0; c < 7; ++c) {
            const uint32_t ind = ((c & 1) ? pl.b0 : ~pl.b0) & ((c & 2) ? pl.b1 : ~pl.b1) & ((c & 4) ? pl.b2 : ~pl.b2);
            for (int up = 0; up < 2; ++up) {
                const int cls = 2 * c + up, z = P.zF[cls];
                const uint32_t mine = ind & (up ? s : ~s);
                if (mine == 0u) continue;
                acc |= z < 0 ? mine : mine & lt[rank_of(u, sm_thr + cls * P.LTS, z, P.nT)];
            }
        }
        sp[p * P.Nh + j] = s ^ acc;
    }
}

__global__ void __launch_bounds__(128) k_half_sweep_field(Params P, int p, uint32_t g)
{
    extern __shared__ uint32_t sm_thr[];   // [18][nT+1]
    for (int a = threadIdx.x; a < 18 * P.LTS; a += blockDim.x) sm_thr[a] = P.thrF[a];
    __syncthreads();
    const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= (int64_t)P.nT * P.W * (P.Nh >> 2)) return;
    half_sweep_field_item(P, p, g, tid, sm_thr);
}

// Field term of the energy: E[r][k] += h * (2 * (number of up spins) - N).  One block per (w, k),
// vertical counters like k_energy; runs after it.
// PL planes in all: the per-thread count (<= ceil(N / blockDim)) must stay below 2^(PL-5), the
// warp total below 2^PL.
// item = (w, k) handled by the whole block; sm_cnt = 32 ints of shared memory
template <int PL>
__device__ __forceinline__ void field_energy_item(const Params &P, int item, int *sm_cnt)
{
    constexpr int kFieldPlanes = PL;
    const int w = item / P.nT, k = item % P.nT;
    const uint32_t *sp = P.spin + ((size_t)k * P.W + w) * P.N;
    if (threadIdx.x < 32) sm_cnt[threadIdx.x] = 0;
    __syncthreads();
    uint32_t c[kFieldPlanes];
#pragma unroll
    for (int i = 0; i < kFieldPlanes; ++i) c[i] = 0;
#pragma unroll 4
    for (int i = threadIdx.x; i < P.N; i += blockDim.x) {
        uint32_t x = sp[i];
#pragma unroll
        for (int l = 0; l < kFieldPlanes - 5; ++l) {
            const uint32_t carry = c[l] & x;
            c[l] ^= x;
            x = carry;
        }
    }
    const int lane = threadIdx.x & 31;
    atomicAdd(&sm_cnt[lane], warp_positional_sum<PL>(c, lane));
    __syncthreads();
    if (threadIdx.x < 32)
        P.E[(size_t)(32 * w + threadIdx.x) * P.nT + k] += P.h * (2 * sm_cnt[threadIdx.x] - P.N);
    __syncthreads();
}

template <int PL>
__global__ void __launch_bounds__(128) k_field_energy(Params P)
{
    __shared__ int sm_cnt[32];
    field_energy_item<PL>(P, blockIdx.x, sm_cnt);
}

// ------------------------------------------------------------------ a8: energy from scratch
// E[r][k] = 3N - 2 * (number of satisfied bonds); every bond has exactly one parity-1 end, so
// the satisfied bonds are sum over parity-1 sites of n_sat.  One block per (w, k); per-thread
// bit-sliced (vertical) counters, then a transposition to 32 integers with warp reductions.
// PL planes in all: the per-thread count (<= 6 ceil(Nh / blockDim)) must stay below 2^(PL-5), the
// warp total below 2^PL.
template <int PL>
__device__ __forceinline__ void vadd(uint32_t (&c)[PL], uint32_t x, int from)
{
#pragma unroll
    for (int i = 0; i < PL - 5; ++i) {
        if (i < from) continue;
        const uint32_t t = c[i] & x;
        c[i] ^= x;
        x = t;
    }
}

template <int PL>
__device__ __forceinline__ void energy_item(const Params &P, int item, int *sm_cnt)
{
    constexpr int kEnergyPlanes = PL;
    const int w = item / P.nT, k = item % P.nT;
    const uint32_t *sp = P.spin + ((size_t)k * P.W + w) * P.N;
    const uint32_t *cp = P.coup + (size_t)w * 3 * P.N;
    if (threadIdx.x < 32) sm_cnt[threadIdx.x] = 0;
    __syncthreads();
    uint32_t c[kEnergyPlanes];
#pragma unroll
    for (int i = 0; i < kEnergyPlanes; ++i) c[i] = 0;
    // four sites' loads in flight before the first add
    for (int j0 = threadIdx.x; j0 < P.Nh; j0 += 4 * blockDim.x) {
        Planes pl[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int j = j0 + u * blockDim.x;
            uint32_t s;
            if (j < P.Nh) pl[u] = site_planes(sp, cp, 1, j, P.L, P.Lh, P.Nh, P.N, &s);
            else pl[u].b0 = pl[u].b1 = pl[u].b2 = 0u;
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            vadd<PL>(c, pl[u].b0, 0);
            vadd<PL>(c, pl[u].b1, 1);
            vadd<PL>(c, pl[u].b2, 2);
        }
    }
    const int lane = threadIdx.x & 31;
    atomicAdd(&sm_cnt[lane], warp_positional_sum<PL>(c, lane));
    __syncthreads();
    if (threadIdx.x < 32)
        P.E[(size_t)(32 * w + threadIdx.x) * P.nT + k] = 3 * P.N - 2 * sm_cnt[threadIdx.x];
    __syncthreads();
}

template <int PL>
__global__ void __launch_bounds__(128) k_energy(Params P)
{
    __shared__ int sm_cnt[32];
    energy_item<PL>(P, blockIdx.x, sm_cnt);
}

// ------------------------------------------------------------------ a9: PT swap round
// Decision for temperature pair (t, t+1) of realization r after sweep g_done:
//   a = sigma[t], b = sigma[t+1], m = (E_a - E_b)/4, accept iff PX(g_done,t,r,2<<16)[0] < swp[t][m].
// The swap table is stored trimmed (only thresholds in (0, 2^32), as thr - 1).
__device__ __forceinline__ bool swap_accept(const Params &P, int t, int m, uint32_t v)
{
    const int lo = P.swp_lo[t], cnt = P.swp_cnt[t];
    if (m < lo) return P.swp_kind[2 * t] != 0;
    if (m >= lo + cnt) return P.swp_kind[2 * t + 1] != 0;
    return v <= P.swp_val[P.swp_off[t] + (m - lo)];
}

// One block per word: lane = realization bit, warps stride over the disjoint pairs of this
// round (R4); then the rank masks of the word are rebuilt.  No lattice word moves.
__device__ __forceinline__ void pt_swap_word(const Params &P, int w, uint32_t g_done, uint32_t round)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    const int r = 32 * w + lane;
    uint8_t *sg = P.sigma + (size_t)r * P.nT, *ta = P.tau + (size_t)r * P.nT;
    const int32_t *E = P.E + (size_t)r * P.nT;
    for (int t = (int)(round & 1u) + 2 * warp; t + 1 < P.nT; t += 2 * nwarp) {
        const int a = sg[t], b = sg[t + 1];
        const int m = (E[a] - E[b]) / P.ediv;
        const uint4 v = philox4x32_10(g_done, (uint32_t)t, P.r0 + (uint32_t)r, 2u << 16, P.k0, P.k1);
        if (swap_accept(P, t, m, v.x)) {
            sg[t] = (uint8_t)b; sg[t + 1] = (uint8_t)a;
            ta[a] = (uint8_t)(t + 1); ta[b] = (uint8_t)t;
        }
    }
    __syncthreads();
    for (int k = warp; k < P.nT; k += nwarp) build_lt_row(P, w, k, lane);
}

__global__ void __launch_bounds__(256) k_pt_swap(Params P, uint32_t g_done, uint32_t round)
{
    pt_swap_word(P, blockIdx.x, g_done, round);
}

// Data-moving swap (ea_set_swap_mode, R26): block = (word, pair of this round).  Warp 0
// takes the 32 decisions of the word (lane = realization), the ballot is the exchange mask, then the
// whole block exchanges the masked bits of the two lattices: x = (a ^ b) & m, a ^= x, b ^= x.
// tau stays the identity, so the rank masks never change.
__global__ void __launch_bounds__(256) k_swap_move(Params P, uint32_t g_done, uint32_t round)
{
    __shared__ uint32_t s_mask;
    const int w = blockIdx.x, t = (int)(round & 1u) + 2 * (int)blockIdx.y;
    if (t + 1 >= P.nT) return;
    if (threadIdx.x < 32) {
        const int lane = threadIdx.x, r = 32 * w + lane;
        int32_t *E = P.E + (size_t)r * P.nT;
        const int ea = E[t], eb = E[t + 1];
        const uint4 v = philox4x32_10(g_done, (uint32_t)t, P.r0 + (uint32_t)r, 2u << 16, P.k0, P.k1);
        const bool acc = swap_accept(P, t, (ea - eb) / P.ediv, v.x);
        if (acc) { E[t] = eb; E[t + 1] = ea; }
        const uint32_t m = __ballot_sync(0xFFFFFFFFu, acc);
        if (lane == 0) s_mask = m;
    }
    __syncthreads();
    const uint32_t m = s_mask;
    if (m == 0u) return;
    uint4 *A = reinterpret_cast<uint4 *>(P.spin + ((size_t)t * P.W + w) * P.N);
    uint4 *B = reinterpret_cast<uint4 *>(P.spin + ((size_t)(t + 1) * P.W + w) * P.N);
    for (int i = threadIdx.x; i < P.N / 4; i += blockDim.x) {
        uint4 a = A[i], b = B[i];
        const uint4 x = make_uint4((a.x ^ b.x) & m, (a.y ^ b.y) & m, (a.z ^ b.z) & m, (a.w ^ b.w) & m);
        a.x ^= x.x; a.y ^= x.y; a.z ^= x.z; a.w ^= x.w;
        b.x ^= x.x; b.y ^= x.y; b.z ^= x.z; b.w ^= x.w;
        A[i] = a; B[i] = b;
    }
}

// ------------------------------------------------------------------ persistent generic path
// All sweeps of a call in ONE cooperative launch for lattices that have no shared-memory path
// (L = 2, 4, 6, 12, ... and every L with a field): the same work items as the kernels above,
// dealt out grid-stride, with a grid-wide barrier where the one-launch-per-step path has a
// kernel boundary.  For the small configs (1 and 3) the step time was launch latency (3-4
// launches of ~7 us per sweep); the barrier costs about 1 us.
struct PersistArgs {
    Params P;
    uint32_t g0;          // global index of the first sweep of this call
    int n_sweeps;
    int swap_interval;
    uint32_t nswap0;      // swap rounds done before this call
    unsigned int *gbar;   // grid barrier word, zero before the launch
};

__device__ __forceinline__ void persist_grid_sync(unsigned int *bar)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned int add = blockIdx.x == 0 ? 0x80000000u - (gridDim.x - 1) : 1u;
        __threadfence();
        const unsigned int old = atomicAdd(bar, add);
        while ((((old ^ *reinterpret_cast<volatile unsigned int *>(bar)) & 0x80000000u) == 0u)) { }
        __threadfence();
    }
    __syncthreads();
}

template <bool FIELD>
__global__ void __launch_bounds__(256) k_generic_persistent(const PersistArgs A)
{
    extern __shared__ uint32_t sm_thr[];   // [3 or 18][nT+1]
    __shared__ int sm_cnt[32];
    const Params &P = A.P;
    const int ncls = FIELD ? 18 : 3;
    for (int a = threadIdx.x; a < ncls * P.LTS; a += blockDim.x) sm_thr[a] = FIELD ? P.thrF[a] : P.thr32[a];
    __syncthreads();
    const int64_t n_items = (int64_t)P.nT * P.W * (P.Nh >> 2);
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    uint32_t nswap = A.nswap0;
    for (int it = 0; it < A.n_sweeps; ++it) {
        const uint32_t g = A.g0 + (uint32_t)it;
        for (int p = 0; p < 2; ++p) {
            for (int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; tid < n_items; tid += stride) {
                if (FIELD) half_sweep_field_item(P, p, g, tid, sm_thr);
                else half_sweep_item(P, p, g, tid, sm_thr);
            }
            persist_grid_sync(A.gbar);
        }
        const bool swap_now = A.swap_interval > 0 && ((uint64_t)g + 1) % (uint64_t)A.swap_interval == 0;
        if (!swap_now && it != A.n_sweeps - 1) continue;
        for (int item = blockIdx.x; item < P.W * P.nT; item += gridDim.x) {   // energies of the finished sweep
            energy_item<22>(P, item, sm_cnt);                 // 22 planes: any lattice the library takes
            if (FIELD) field_energy_item<22>(P, item, sm_cnt);
        }
        if (!swap_now) continue;
        persist_grid_sync(A.gbar);
        for (int w = blockIdx.x; w < P.W; w += gridDim.x) pt_swap_word(P, w, g, nswap & 1u);
        ++nswap;
        persist_grid_sync(A.gbar);
    }
}

// ------------------------------------------------------------------ a10: overlap
// Q[pair][t] = sum_i s_i(ra, sigma_a[t]) s_i(rb, sigma_b[t]); rb = -1: all-up reference.
__global__ void __launch_bounds__(256) k_overlap(Params P, const int32_t *pairs, int32_t *Q)
{
    __shared__ int sm_sum[8];
    const int pr = blockIdx.x / P.nT, t = blockIdx.x % P.nT;
    const int ra = pairs[2 * pr], rb = pairs[2 * pr + 1];
    const int ka = P.sigma[(size_t)ra * P.nT + t];
    const uint32_t *sa = P.spin + ((size_t)ka * P.W + (ra >> 5)) * P.N;
    const uint32_t *sb = nullptr;
    if (rb >= 0) sb = P.spin + ((size_t)P.sigma[(size_t)rb * P.nT + t] * P.W + (rb >> 5)) * P.N;
    int agree = 0;
    for (int i = threadIdx.x; i < P.N; i += blockDim.x) {
        const uint32_t a = (sa[i] >> (ra & 31)) & 1u;
        const uint32_t b = sb ? (sb[i] >> (rb & 31)) & 1u : 1u;
        agree += (a == b);
    }
    agree = __reduce_add_sync(0xFFFFFFFFu, agree);
    if ((threadIdx.x & 31) == 0) sm_sum[threadIdx.x >> 5] = agree;
    __syncthreads();
    if (threadIdx.x == 0) {
        int tot = 0;
        for (int i = 0; i < (int)(blockDim.x >> 5); ++i) tot += sm_sum[i];
        Q[blockIdx.x] = 2 * tot - P.N;
    }
}

// ------------------------------------------------------------------ a11: export / import
// out[r][t][i] = +-1 by temperature index (by_slot = 0) or by slot (by_slot = 1).
__global__ void k_unpack_spins(Params P, int R, int by_slot, int8_t *out)
{
    const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= (int64_t)R * P.nT * P.N) return;
    const int i = (int)(tid % P.N);
    const int t = (int)((tid / P.N) % P.nT);
    const int r = (int)(tid / ((int64_t)P.N * P.nT));
    const int k = by_slot ? t : P.sigma[(size_t)r * P.nT + t];
    const int x = i % P.L, y = (i / P.L) % P.L, z = i / (P.L * P.L);
    const int p = (x + y + z) & 1, j = (x >> 1) + P.Lh * (y + P.L * z);
    const uint32_t wv = P.spin[((size_t)k * P.W + (r >> 5)) * P.N + p * P.Nh + j];
    out[tid] = ((wv >> (r & 31)) & 1u) ? 1 : -1;
}

// in[r][outer][i] (+-1 int8, canonical site order) -> words[outer'][w][p][j]; one thread per
// output word.  mode 0: spins (outer = slot k, word index (k W + w) N + ...);
// mode 1: couplings (outer = d, word index (w 3 + d) N + ...).
// *bad is set if any input value is neither +1 nor -1 (the caller then discards `words`).
__global__ void k_pack(Params P, int R, int n_outer, int mode, const int8_t *in, uint32_t *words, int *bad)
{
    const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= (int64_t)n_outer * P.W * P.N) return;
    const int i = (int)(tid % P.N);
    const int w = (int)((tid / P.N) % P.W);
    const int o = (int)(tid / ((int64_t)P.N * P.W));
    const int x = i % P.L, y = (i / P.L) % P.L, z = i / (P.L * P.L);
    const int p = (x + y + z) & 1, j = (x >> 1) + P.Lh * (y + P.L * z);
    uint32_t v = 0;
    bool wrong = false;
    for (int b = 0; b < 32; ++b) {
        const int r = 32 * w + b;
        if (r >= R) break;
        const int8_t v8 = in[((size_t)r * n_outer + o) * P.N + i];
        wrong |= (v8 != 1 && v8 != -1);
        if (v8 > 0) v |= 1u << b;
    }
    if (wrong) *bad = 1;
    const size_t dst = mode == 0 ? ((size_t)o * P.W + w) * P.N : ((size_t)w * 3 + o) * P.N;
    words[dst + p * P.Nh + j] = v;
}

}  // namespace ea
