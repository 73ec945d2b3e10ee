// ea_lib.cu -- host side of libea_b200.so: the C ABI of include/ea.h.
// Product code.  No CPU fallback: every step of the path runs in the CUDA kernels of
// ea_generic.cuh / ea_resident.cuh / ea_tiled.cuh.  Shares nothing with oracle/.
#include "../../include/ea.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "ea_generic.cuh"
#include "ea_resident.cuh"
#include "ea_small.cuh"
#include "ea_tiled.cuh"
#include "ea_stream.cuh"
#include "ea_peak.cuh"
#include "ea_measure.cuh"
#include "ea_replica.cuh"

using ea::Params;

struct ea_handle {
    int L = 0, N = 0, nT = 0, R = 0, W = 0, Rp = 0, r0 = 0;
    uint64_t seed = 0;
    std::vector<double> betas;
    bool desc = true;
    std::vector<uint64_t> acc, swp;   // host copies: acc always; swp only when ea_set_tables gave one (else the
                                      // table is a formula of betas and is written out on demand, ea_get_tables)
    cudaStream_t stream = nullptr;
    bool own_ws = false;
    char *ws = nullptr;
    size_t ws_bytes = 0;
    Params P{};
    uint32_t *d_thr32 = nullptr;
    int32_t *d_swp_lo = nullptr, *d_swp_cnt = nullptr, *d_swp_off = nullptr;
    uint8_t *d_swp_kind = nullptr;
    uint32_t *d_swp_val = nullptr;
    size_t swp_val_cap = 0;
    int32_t *d_Ecnt = nullptr;         // satisfied-bond counters of the tiled path
    uint4 *d_bucket = nullptr;         // fast rank table (ea_resident.cuh), 16 B entries
    int n_bucket = 0;
    ea::RankKey K{};                   // bucket key parameters of the fast rank table
    uchar4 *d_trip = nullptr;          // [3 nT + 1] combined rank -> (n4, n5, n6)
    bool fast_rank = false;
    uint64_t g = 0, nswap = 0;
    bool energy_valid = false;
    int kernel_sel = EA_KERNEL_AUTO;
    int swap_mode = EA_SWAP_PERMUTE;   // ea_set_swap_mode
    bool poisoned = false;             // a launch failed between the word groups of one ea_sweep call: the words
                                       // are no longer at the same sweep; ea_set_state brings the handle back
    int64_t launches = 0;
    int sm_count = 0;
    // measurement series (ea_measure_begin): own allocation, freed by ea_destroy / the next begin
    char *d_meas = nullptr;
    uint32_t *d_T = nullptr;           // spins gathered by temperature index, [t][w][i]
    ea::Moments M{};
    size_t meas_bytes = 0, meas_acc_off = 0;
    uint64_t meas_n = 0;
    bool meas_on = false;
    // external field (ea_set_field): own allocation for the 14-class thresholds and the trimmed
    // field swap table; freed by ea_destroy / the next ea_set_field
    // second layout (ea_set_layout, ea_replica.cuh): own allocation for the T storage (spins by
    // realization, packed coupling bits, the probability table); r_valid / t_valid say which of the
    // two spin stores is current
    int layout = EA_LAYOUT_REALIZATION_BITS;
    char *d_rep = nullptr;
    uint32_t *d_spinT = nullptr, *d_jbit = nullptr;
    uint64_t *d_acc64 = nullptr;
    int ncube = 0, NW = 0;
    bool r_valid = true, t_valid = false;
    // scratch for the host-buffer calls (packing inputs, overlaps, exported spins / couplings, energies
    // by temperature): one allocation that only grows, instead of a cudaMalloc / cudaFree per call
    char *d_scratch = nullptr;
    size_t scratch_bytes = 0;
    int field = 0;
    bool fast_field = false;           // |h| <= 2 and the four-column bucket table exists: the resident kernel runs
    ea::RankKey KF{};
    uint4 *d_bucketF = nullptr;
    uchar4 *d_tripF = nullptr;
    char *d_field = nullptr;
    std::vector<uint64_t> accf;        // host copy [nT][7][2]; the field swap table is a formula (ea_get_field_tables)
    mutable std::string err;
};

static thread_local std::string g_create_err;

static int fail(const ea_handle *h, int code, const std::string &msg)
{
    if (h) h->err = msg; else g_create_err = msg;
    return code;
}
#define CUDA_TRY(h, expr)                                                                   \
    do {                                                                                    \
        cudaError_t e_ = (expr);                                                            \
        if (e_ != cudaSuccess)                                                              \
            return fail(h, EA_ERR_CUDA, std::string(#expr) + ": " + cudaGetErrorString(e_)); \
    } while (0)

// ---------------------------------------------------------------- workspace layout
namespace {
constexpr int kMaxBucket = 1024;
struct Layout {
    size_t spin, coup, lt, tau, sigma, E, thr32, swp_lo, swp_cnt, swp_off, swp_kind, swp_val, bucket, trip, ecnt, total;
    size_t swp_val_cap;
};
size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

bool shape_ok(int L, int nT, int R)
{
    return L >= 2 && (L & 1) == 0 && L <= 128 && nT >= 1 && R >= 1 && R <= (1 << 24);
}

Layout make_layout(int L, int nT, int R)
{
    Layout o{};
    const size_t N = (size_t)L * L * L, W = (size_t)(R + 31) / 32, Rp = 32 * W;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t a = off; off = align256(off + bytes); return a; };
    o.spin = take(4 * (size_t)nT * W * N);
    o.coup = take(4 * 3 * W * N);
    o.lt = take(4 * W * nT * (nT + 1));
    o.tau = take(Rp * nT);
    o.sigma = take(Rp * nT);
    o.E = take(4 * Rp * nT);
    o.thr32 = take(4 * 3 * (size_t)(nT + 1));
    o.swp_lo = take(4 * (size_t)nT);
    o.swp_cnt = take(4 * (size_t)nT);
    o.swp_off = take(4 * (size_t)nT);
    o.swp_kind = take(2 * (size_t)nT);
    o.swp_val_cap = (size_t)(nT > 1 ? nT - 1 : 0) * (3 * N + 1);
    o.swp_val = take(4 * (o.swp_val_cap ? o.swp_val_cap : 1));
    o.bucket = take(16 * (size_t)kMaxBucket);
    o.trip = take(4 * (3 * (size_t)nT + 2));
    o.ecnt = take(2 * 4 * Rp * nT + 256);      // double-buffered by the streaming kernel; + its grid barrier word
    o.total = off;
    return o;
}

uint64_t threshold_of(double x)
{
    if (x >= 0.0) return (uint64_t)1 << 32;
    return (uint64_t)std::floor(std::ldexp(std::exp(x), 32));
}
const uint64_t TWO32 = (uint64_t)1 << 32;

void launch_cfg(int64_t n, int block, int &grid) { grid = (int)((n + block - 1) / block); }
}  // namespace


// ---------------------------------------------------------------- fast rank table
// Buckets of the draw u by a monotone key with logarithmic steps that the kernels evaluate on the
// FMA pipe (ea_resident.cuh, RankCtx):
//   key(u) = bits(g) >> (23 - MB),   g = sat(float_rz(u) * 2^-E + 2^(8-E)),
// E = number of bits of the largest threshold (every larger u takes the same decisions and
// saturates onto the last bucket), the added constant merging all u << 2^8 into the first.  The
// host evaluates the same function exactly (the sum is exact in double, the cast rounds once as
// the device's fused multiply-add does) and finds every bucket's range of u by bisection.
// Entry = { ~thr4, n4 + n5 + n6 at the bucket's lower edge, ~thr5, ~thr6 }: n_c = number of class-c
// thresholds <= the lower edge, thr_c = the class-c (threshold - 1) inside the bucket or
// 0xFFFFFFFF.  Buckets holding several thresholds of one class point at row 3 nT + 1 of the mask
// tables = "use the exact search".  MB is the smallest of 3..6 that leaves < 1e-5 of the draws on
// the slow path.
// trip[n] = the triple (n4, n5, n6) whose sum is n (unique: each n_c is monotone in u).
namespace {
struct KeyFn {
    int E, MB;
    int operator()(uint32_t u) const
    {
        double f = (double)u;                                  // cvt.rz.f32.u32: keep the leading 24 bits
        if (u >> 24) { const int sh = 8 - __builtin_clz(u); f = (double)((u >> sh) << sh); }
        const double x = std::ldexp(f, -E) + std::ldexp(1.0, 8 - E);   // exact in double
        float g = (float)x;                                    // one rounding to nearest even, as fma.rn
        if (g > 1.0f) g = 1.0f;                                // .sat
        uint32_t b;
        std::memcpy(&b, &g, 4);
        return (int)(b >> (23 - MB));
    }
};
}  // namespace

// NC = 3: the zero-field classes n_sat = 4, 5, 6, one 16-byte entry per bucket.  NC = 4: the four
// threshold columns of a field |h| <= 2, 32-byte entries
// { ~thr_a, n, ~thr_b, ~thr_c | ~thr_d, slow flag, 0, 0 }.
static bool build_bucket_table(const std::vector<uint32_t> &thr32, const int *z, int nT, int NC,
                               std::vector<uint4> &tab, std::vector<uchar4> &trip, ea::RankKey &K)
{
    auto rank_c = [&](int c, uint64_t u) {   // n_c(u) = z_c + #{i >= z_c : thr32[c][i] < u}
        int n = z[c];
        for (int i = z[c]; i < nT; ++i) if ((uint64_t)thr32[(size_t)c * (nT + 1) + i] < u) n = i + 1;
        return n;
    };
    trip.assign((size_t)NC * nT + 1, make_uchar4((unsigned char)nT, (unsigned char)nT, (unsigned char)nT, (unsigned char)(NC == 4 ? nT : 0)));
    auto note = [&](uint64_t u) {
        int r[4] = {0, 0, 0, 0}, sum = 0;
        for (int c = 0; c < NC; ++c) { r[c] = rank_c(c, u); sum += r[c]; }
        trip[(size_t)sum] = make_uchar4((unsigned char)r[0], (unsigned char)r[1], (unsigned char)r[2], (unsigned char)r[3]);
    };
    note(0);
    uint32_t tmax = 0;
    for (int c = 0; c < NC; ++c)
        for (int i = z[c]; i < nT; ++i) {
            const uint32_t v = thr32[(size_t)c * (nT + 1) + i];
            note((uint64_t)v + 1);
            if (v != 0xFFFFFFFFu) tmax = std::max(tmax, v);
        }
    int E = 9;
    while (E < 32 && (tmax >> E)) ++E;                     // 2^E > every threshold - 1
    const uint32_t slow_row = (uint32_t)(3 * nT + 1);      // NC = 3 only
    const int BW = NC == 4 ? 2 : 1;
    for (int MB = 3; MB <= 6; ++MB) {
        const KeyFn key{E, MB};
        const int klo = key(0), khi = key(0xFFFFFFFFu);
        const int n = khi - klo + 1;
        if (n > kMaxBucket) continue;      // entries (the field table has its own allocation: 32 B each)
        // first u of every bucket (2^32 for an empty bucket at the top)
        std::vector<uint64_t> first((size_t)n + 1);
        first[0] = 0;
        first[(size_t)n] = (uint64_t)1 << 32;
        for (int b = 1; b < n; ++b) {
            uint64_t lo = first[(size_t)b - 1], hi = (uint64_t)1 << 32;   // smallest u with key(u) - klo >= b
            while (lo < hi) {
                const uint64_t mid = (lo + hi) >> 1;
                if (key((uint32_t)mid) - klo >= b) hi = mid; else lo = mid + 1;
            }
            first[(size_t)b] = lo;
        }
        std::vector<uint4> t((size_t)n * BW);
        auto put = [&](int b, bool slow, uint32_t nsum, const uint32_t *inb) {
            if (NC == 3) {
                t[(size_t)b] = slow ? make_uint4(0u, slow_row, 0u, 0u) : make_uint4(~inb[0], nsum, ~inb[1], ~inb[2]);
            } else {
                t[(size_t)2 * b] = slow ? make_uint4(0u, 0u, 0u, 0u) : make_uint4(~inb[0], nsum, ~inb[1], ~inb[2]);
                t[(size_t)2 * b + 1] = slow ? make_uint4(0u, 0x80000000u, 0u, 0u) : make_uint4(~inb[3], 0u, 0u, 0u);
            }
        };
        double slow_mass = 0.0;
        for (int b = 0; b < n; ++b) {
            const uint64_t lo_u = first[(size_t)b], end_u = first[(size_t)b + 1];
            const uint32_t none[4] = {0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu};
            if (end_u <= lo_u) { put(b, true, 0u, none); continue; }   // empty: never read
            const uint64_t hi_u = end_u - 1;
            uint32_t nsum = 0, inb[4] = {0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu};
            bool slow = false;
            for (int c = 0; c < NC; ++c) {
                const uint32_t *col = thr32.data() + (size_t)c * (nT + 1);
                int nlo = z[c], cnt = 0;
                for (int i = z[c]; i < nT; ++i) {
                    if ((uint64_t)col[i] < lo_u) nlo = i + 1;
                    else if ((uint64_t)col[i] < hi_u) { if (!cnt) inb[c] = col[i]; ++cnt; }
                }
                if (cnt > 1) slow = true;
                nsum += (uint32_t)nlo;
            }
            if (slow) slow_mass += (double)(hi_u - lo_u + 1) / 4294967296.0;
            put(b, slow, nsum, inb);
        }
        if (slow_mass < 1e-5 || MB == 6) {
            if (slow_mass > 1e-3) return false;
            tab = t;
            K.kscale = std::ldexp(1.0f, -E); K.kadd = std::ldexp(1.0f, 8 - E);
            K.kmul = 1u << (9 + MB); K.c16 = 16u;
            K.key_lo = klo; K.n_bucket = n;
            return true;
        }
    }
    return false;
}

// ---------------------------------------------------------------- tables -> device form
// acc: per class c = 4,5,6 a column sorted coldest-first ("pos" order), stored as thr-1 with
// the leading zero thresholds counted in z[c] (R8).  swp: each row trimmed to the
// entries strictly between 0 and 2^32.
// Trimmed form of a swap table with rows [nT-1][2 M + 1], column = index + M: per row the first
// stored index, the number of stored entries, their offset in `val`, the decisions left and right
// of the stored range (0 never, 1 always) and (threshold - 1) for thresholds in (0, 2^32).  Lossless.
struct SwapTrim {
    std::vector<int32_t> lo, cnt, off;
    std::vector<uint8_t> kind;
    std::vector<uint32_t> val;
};
static const uint64_t kTwo32 = (uint64_t)1 << 32;
static int trim_swap_table(ea_handle *h, const uint64_t *swp, int nT, int64_t M, SwapTrim &o)
{
    const int64_t cols = 2 * M + 1;
    o.lo.assign(nT, 0); o.cnt.assign(nT, 0); o.off.assign(nT, 0);
    o.kind.assign((size_t)2 * nT, 0);
    o.val.clear();
    for (int t = 0; t + 1 < nT; ++t) {
        const uint64_t *row = swp + (size_t)t * cols;
        bool inc = true, dec = true;
        for (int64_t a = 0; a < cols; ++a) {
            if (row[a] > kTwo32) return fail(h, EA_ERR_INVALID_ARG, "swp threshold above 2^32");
            if (a && row[a] < row[a - 1]) inc = false;
            if (a && row[a] > row[a - 1]) dec = false;
        }
        if (!inc && !dec) return fail(h, EA_ERR_INVALID_ARG, "swp row not monotone in m");
        int64_t a = 0;
        while (a < cols && (row[a] == 0 || row[a] == kTwo32) && row[a] == row[0]) ++a;
        int64_t b = a;
        while (b < cols && row[b] != 0 && row[b] != kTwo32) ++b;
        for (int64_t c2 = b; c2 < cols; ++c2)
            if (row[c2] != row[cols - 1]) return fail(h, EA_ERR_INVALID_ARG, "swp row not monotone in m");
        o.lo[t] = (int32_t)(a - M); o.cnt[t] = (int32_t)(b - a); o.off[t] = (int32_t)o.val.size();
        o.kind[2 * t] = row[0] == kTwo32;
        o.kind[2 * t + 1] = row[cols - 1] == kTwo32;
        for (int64_t c2 = a; c2 < b; ++c2) o.val.push_back((uint32_t)(row[c2] - 1));
    }
    return EA_OK;
}
// The same trimmed form for a table given by its FORMULA f(t, m), m in [-M, M], without writing the
// table out: every row is monotone in m and constant (0 or 2^32) outside one interval, whose two
// ends are found by bisection; only the thresholds inside it are evaluated.  (A full table is
// (n_temps - 1)(2 M + 1) exp() calls and 8 bytes each: 400 MB at L = 64, n_temps = 64.)
template <class F>
static void trim_swap_generated(int nT, int64_t M, const F &f, SwapTrim &o)
{
    o.lo.assign(nT, 0); o.cnt.assign(nT, 0); o.off.assign(nT, 0);
    o.kind.assign((size_t)2 * nT, 0);
    o.val.clear();
    auto trivial = [](uint64_t v) { return v == 0 || v == kTwo32; };
    for (int t = 0; t + 1 < nT; ++t) {
        const uint64_t v_lo = f(t, -M), v_hi = f(t, M);
        int64_t a = -M, b = M + 1;
        if (trivial(v_lo)) {              // a = first m whose threshold differs from the left constant
            int64_t lo = -M, hi = M + 1;
            while (lo < hi) { const int64_t mid = lo + (hi - lo) / 2; if (f(t, mid) != v_lo) hi = mid; else lo = mid + 1; }
            a = lo;
        }
        if (trivial(v_hi) && a <= M) {    // b = first m >= a whose threshold is the right constant
            int64_t lo = a, hi = M + 1;
            while (lo < hi) { const int64_t mid = lo + (hi - lo) / 2; if (f(t, mid) == v_hi) hi = mid; else lo = mid + 1; }
            b = lo;
        }
        if (a > M) b = a;
        o.lo[t] = (int32_t)a; o.cnt[t] = (int32_t)(b - a); o.off[t] = (int32_t)o.val.size();
        o.kind[2 * t] = v_lo == kTwo32;
        o.kind[2 * t + 1] = v_hi == kTwo32;
        for (int64_t m = a; m < b; ++m) o.val.push_back((uint32_t)(f(t, m) - 1));
    }
}

static int upload_swap_trim(ea_handle *h, const SwapTrim &o, uint32_t *d_val)
{
    const int nT = h->nT;
    cudaStream_t s = h->stream;
    CUDA_TRY(h, cudaMemcpyAsync(h->d_swp_lo, o.lo.data(), 4 * nT, cudaMemcpyHostToDevice, s));
    CUDA_TRY(h, cudaMemcpyAsync(h->d_swp_cnt, o.cnt.data(), 4 * nT, cudaMemcpyHostToDevice, s));
    CUDA_TRY(h, cudaMemcpyAsync(h->d_swp_off, o.off.data(), 4 * nT, cudaMemcpyHostToDevice, s));
    CUDA_TRY(h, cudaMemcpyAsync(h->d_swp_kind, o.kind.data(), 2 * nT, cudaMemcpyHostToDevice, s));
    if (!o.val.empty())
        CUDA_TRY(h, cudaMemcpyAsync(d_val, o.val.data(), 4 * o.val.size(), cudaMemcpyHostToDevice, s));
    CUDA_TRY(h, cudaStreamSynchronize(s));
    return EA_OK;
}

// swp == nullptr: the zero-field swap table of the handle's betas, from its formula
static int upload_tables(ea_handle *h, const std::vector<uint64_t> &acc, const std::vector<uint64_t> *swp)
{
    const int nT = h->nT, M = 3 * h->N / 2;
    for (int t = 0; t < nT; ++t)
        for (int c = 0; c < 7; ++c) {
            const uint64_t v = acc[(size_t)t * 7 + c];
            if (v > TWO32) return fail(h, EA_ERR_INVALID_ARG, "acc threshold above 2^32");
            if (c <= 3 && v != TWO32)
                return fail(h, EA_ERR_UNSUPPORTED, "acc[t][c<=3] must be 2^32 (dE <= 0 always flips)");
        }
    std::vector<uint32_t> thr32((size_t)3 * (nT + 1));
    int z[3];
    for (int c = 4; c <= 6; ++c) {
        uint32_t *col = thr32.data() + (size_t)(c - 4) * (nT + 1);
        uint64_t prev = 0;
        int zc = 0;
        for (int pos = 0; pos < nT; ++pos) {
            const int t = h->desc ? pos : nT - 1 - pos;
            const uint64_t v = acc[(size_t)t * 7 + c];
            if (v < prev) return fail(h, EA_ERR_INVALID_ARG, "acc column not monotone with beta");
            if (c > 4 && v > acc[(size_t)t * 7 + c - 1])
                return fail(h, EA_ERR_INVALID_ARG, "acc row not non-increasing in n_sat");
            prev = v;
            if (v == 0) { zc = pos + 1; col[pos] = 0; }
            else col[pos] = (uint32_t)(v - 1);
        }
        col[nT] = 0xFFFFFFFFu;
        z[c - 4] = zc;
    }
    SwapTrim tr;
    if (swp) {
        int rc = trim_swap_table(h, swp->data(), nT, M, tr);
        if (rc != EA_OK) return rc;
    } else {
        const std::vector<double> &b = h->betas;
        trim_swap_generated(nT, M, [&](int t, int64_t m) { return threshold_of((b[t] - b[t + 1]) * (double)(4 * m)); }, tr);
    }
    if (tr.val.size() > h->swp_val_cap) return fail(h, EA_ERR_ALLOC, "swap table overflow");
    cudaStream_t s = h->stream;
    CUDA_TRY(h, cudaStreamSynchronize(s));
    CUDA_TRY(h, cudaMemcpyAsync(h->d_thr32, thr32.data(), 4 * thr32.size(), cudaMemcpyHostToDevice, s));
    { int rc = upload_swap_trim(h, tr, h->d_swp_val); if (rc != EA_OK) return rc; }
    {
        std::vector<uint4> tab;
        std::vector<uchar4> trip;
        h->fast_rank = build_bucket_table(thr32, z, nT, 3, tab, trip, h->K);
        if (!h->fast_rank) { h->K = ea::RankKey{}; h->K.c16 = 16u; }
        h->n_bucket = h->fast_rank ? (int)tab.size() : 0;
        CUDA_TRY(h, cudaMemcpyAsync(h->d_trip, trip.data(), 4 * trip.size(), cudaMemcpyHostToDevice, s));
        if (h->fast_rank)
            CUDA_TRY(h, cudaMemcpyAsync(h->d_bucket, tab.data(), 16 * tab.size(), cudaMemcpyHostToDevice, s));
        CUDA_TRY(h, cudaStreamSynchronize(s));
    }
    for (int c = 0; c < 3; ++c) h->P.z[c] = z[c];
    h->acc = acc;
    if (swp) h->swp = *swp; else { h->swp.clear(); h->swp.shrink_to_fit(); }
    return EA_OK;
}

// ---------------------------------------------------------------- scratch
static char *scratch(ea_handle *h, size_t bytes)
{
    if (bytes <= h->scratch_bytes) return h->d_scratch;
    if (h->d_scratch) { cudaStreamSynchronize(h->stream); cudaFree(h->d_scratch); h->d_scratch = nullptr; h->scratch_bytes = 0; }
    const size_t want = (bytes + ((size_t)1 << 20)) & ~(((size_t)1 << 20) - 1);
    if (cudaMalloc((void **)&h->d_scratch, want) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    h->scratch_bytes = want;
    return h->d_scratch;
}

// ---------------------------------------------------------------- second layout: which store is current
static ea::ReplicaArgs replica_args(const ea_handle *h)
{
    ea::ReplicaArgs A{};
    A.P = h->P; A.spinT = h->d_spinT; A.jbit = h->d_jbit; A.acc64 = h->d_acc64; A.ncube = h->ncube; A.NW = h->NW;
    return A;
}
// the first layout's spin words are what every accessor and measurement kernel reads
static int ensure_r(ea_handle *h)
{
    if (h->layout != EA_LAYOUT_REPLICA_BITS || h->r_valid) return EA_OK;
    int grid;
    launch_cfg((int64_t)h->nT * h->W * h->N, 256, grid);
    ea::k_t2r<<<grid, 256, 0, h->stream>>>(replica_args(h));
    h->launches++;
    CUDA_TRY(h, cudaGetLastError());
    h->r_valid = true;
    return EA_OK;
}
static int ensure_t(ea_handle *h)
{
    if (h->t_valid) return EA_OK;
    int grid;
    launch_cfg((int64_t)h->Rp * h->ncube * h->N + (int64_t)h->Rp * 6 * h->NW, 256, grid);
    ea::k_r2t<<<grid, 256, 0, h->stream>>>(replica_args(h));
    h->launches++;
    CUDA_TRY(h, cudaGetLastError());
    h->t_valid = true;
    return EA_OK;
}

// ---------------------------------------------------------------- small helpers
static int recompute_energy(ea_handle *h)
{
    { int rc = ensure_r(h); if (rc != EA_OK) return rc; }
    // counter planes: per-thread count (6 Nh / 128 bonds, N / 128 up spins) < 2^(PL - 5)
    const int grid = h->W * h->nT;
    const long long per_thread = 6ll * ((h->N / 2 + 127) / 128);
    if (per_thread < (1 << 8)) ea::k_energy<13><<<grid, 128, 0, h->stream>>>(h->P);
    else if (per_thread < (1 << 12)) ea::k_energy<17><<<grid, 128, 0, h->stream>>>(h->P);
    else ea::k_energy<22><<<grid, 128, 0, h->stream>>>(h->P);
    h->launches++;
    if (h->field != 0) {
        if (per_thread < (1 << 8)) ea::k_field_energy<13><<<grid, 128, 0, h->stream>>>(h->P);
        else if (per_thread < (1 << 12)) ea::k_field_energy<17><<<grid, 128, 0, h->stream>>>(h->P);
        else ea::k_field_energy<22><<<grid, 128, 0, h->stream>>>(h->P);
        h->launches++;
    }
    CUDA_TRY(h, cudaGetLastError());
    h->energy_valid = true;
    return EA_OK;
}
static int rebuild_lt(ea_handle *h)
{
    int grid;
    launch_cfg((int64_t)h->W * h->nT * 32, 128, grid);
    ea::k_build_lt<<<grid, 128, 0, h->stream>>>(h->P);
    h->launches++;
    CUDA_TRY(h, cudaGetLastError());
    return EA_OK;
}

// ---------------------------------------------------------------- create / destroy
extern "C" size_t ea_workspace_bytes(int L, int n_temps, int n_realizations)
{
    if (!shape_ok(L, n_temps, n_realizations) || n_temps > 64) return 0;
    return make_layout(L, n_temps, n_realizations).total;
}

extern "C" ea_handle *ea_create_ex(int L, int n_temps, int n_realizations, const double *betas,
                                   uint64_t seed, void *dev_workspace, size_t workspace_bytes,
                                   void *cuda_stream, int first_realization)
{
    if (!shape_ok(L, n_temps, n_realizations) || !betas || first_realization < 0 ||
        (first_realization & 31)) {
        fail(nullptr, EA_ERR_INVALID_ARG, "ea_create: bad shape (L even >= 2, n_temps >= 1, R >= 1, "
                                          "first_realization multiple of 32)");
        return nullptr;
    }
    if (n_temps > 64) { fail(nullptr, EA_ERR_UNSUPPORTED, "ea_create: n_temps > 64"); return nullptr; }
    bool desc = true, asc = true;
    for (int t = 0; t < n_temps; ++t) {
        if (!std::isfinite(betas[t]) || betas[t] < 0.0) {
            fail(nullptr, EA_ERR_INVALID_ARG, "ea_create: betas must be finite and >= 0");
            return nullptr;
        }
        if (t && betas[t] > betas[t - 1]) desc = false;
        if (t && betas[t] < betas[t - 1]) asc = false;
    }
    if (!desc && !asc) { fail(nullptr, EA_ERR_INVALID_ARG, "ea_create: betas not monotone"); return nullptr; }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        fail(nullptr, EA_ERR_CUDA, "ea_create: no CUDA device (there is no CPU fallback)");
        return nullptr;
    }
    ea_handle *h = new ea_handle();
    h->L = L; h->N = L * L * L; h->nT = n_temps; h->R = n_realizations;
    h->W = (n_realizations + 31) / 32; h->Rp = 32 * h->W; h->r0 = first_realization;
    h->seed = seed; h->betas.assign(betas, betas + n_temps); h->desc = desc;
    h->stream = (cudaStream_t)cuda_stream;
    const Layout lay = make_layout(L, n_temps, n_realizations);
    auto bail = [&](int code, const std::string &m) { fail(nullptr, code, m); ea_destroy(h); return nullptr; };
    if (dev_workspace) {
        if (workspace_bytes < lay.total || ((uintptr_t)dev_workspace & 255))
            return (ea_handle *)bail(EA_ERR_INVALID_ARG, "ea_create_ex: workspace too small or misaligned");
        h->ws = (char *)dev_workspace;
    } else {
        if (cudaMalloc((void **)&h->ws, lay.total) != cudaSuccess)
            return (ea_handle *)bail(EA_ERR_ALLOC, "ea_create: cudaMalloc failed");
        h->own_ws = true;
    }
    h->ws_bytes = lay.total;
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&h->sm_count, cudaDevAttrMultiProcessorCount, dev);
    Params &P = h->P;
    P.L = L; P.Lh = L / 2; P.N = h->N; P.Nh = h->N / 2; P.nT = n_temps; P.W = h->W; P.Rp = h->Rp;
    P.LTS = n_temps + 1;
    P.k0 = (uint32_t)seed; P.k1 = (uint32_t)(seed >> 32);
    P.r0 = (uint32_t)first_realization; P.w0 = (uint32_t)(first_realization >> 5);
    P.desc = desc ? 1 : 0;
    P.h = 0; P.ediv = 4; P.thrF = nullptr;
    for (int c = 0; c < 18; ++c) P.zF[c] = -1;
    P.spin = (uint32_t *)(h->ws + lay.spin);
    P.coup = (uint32_t *)(h->ws + lay.coup);
    P.lt = (uint32_t *)(h->ws + lay.lt);
    P.tau = (uint8_t *)(h->ws + lay.tau);
    P.sigma = (uint8_t *)(h->ws + lay.sigma);
    P.E = (int32_t *)(h->ws + lay.E);
    P.thr32 = h->d_thr32 = (uint32_t *)(h->ws + lay.thr32);
    P.swp_lo = h->d_swp_lo = (int32_t *)(h->ws + lay.swp_lo);
    P.swp_cnt = h->d_swp_cnt = (int32_t *)(h->ws + lay.swp_cnt);
    P.swp_off = h->d_swp_off = (int32_t *)(h->ws + lay.swp_off);
    P.swp_kind = h->d_swp_kind = (uint8_t *)(h->ws + lay.swp_kind);
    P.swp_val = h->d_swp_val = (uint32_t *)(h->ws + lay.swp_val);
    h->swp_val_cap = lay.swp_val_cap;
    h->d_bucket = (uint4 *)(h->ws + lay.bucket);
    h->d_trip = (uchar4 *)(h->ws + lay.trip);
    h->d_Ecnt = (int32_t *)(h->ws + lay.ecnt);

    // threshold tables in double on the host
    const int M = 3 * h->N / 2;
    std::vector<uint64_t> acc((size_t)n_temps * 7);
    for (int t = 0; t < n_temps; ++t)
        for (int c = 0; c < 7; ++c) acc[(size_t)t * 7 + c] = threshold_of(-(betas[t] * (double)(4 * c - 12)));
    if (upload_tables(h, acc, nullptr) != EA_OK) return (ea_handle *)bail(EA_ERR_CUDA, "ea_create: tables: " + h->err);

    int grid;
    launch_cfg((int64_t)h->W * h->N, 128, grid);
    ea::k_seed<<<grid, 128, 0, h->stream>>>(P);
    launch_cfg((int64_t)h->Rp * n_temps, 128, grid);
    ea::k_identity_perm<<<grid, 128, 0, h->stream>>>(P);
    h->launches += 2;
    cudaMemsetAsync(h->d_Ecnt, 0, 2 * 4 * (size_t)h->Rp * n_temps + 256, h->stream);
    if (rebuild_lt(h) != EA_OK || recompute_energy(h) != EA_OK ||
        cudaStreamSynchronize(h->stream) != cudaSuccess || cudaGetLastError() != cudaSuccess)
        return (ea_handle *)bail(EA_ERR_CUDA, "ea_create: initialisation kernels failed: " + h->err);
    return h;
}

extern "C" ea_handle *ea_create(int L, int n_temps, int n_realizations, const double *betas, uint64_t seed)
{
    return ea_create_ex(L, n_temps, n_realizations, betas, seed, nullptr, 0, nullptr, 0);
}

extern "C" void ea_destroy(ea_handle *h)
{
    if (!h) return;
    if (h->ws) cudaStreamSynchronize(h->stream);
    if (h->own_ws && h->ws) cudaFree(h->ws);
    if (h->d_meas) cudaFree(h->d_meas);
    if (h->d_field) cudaFree(h->d_field);
    if (h->d_rep) cudaFree(h->d_rep);
    if (h->d_scratch) cudaFree(h->d_scratch);
    delete h;
}

extern "C" const char *ea_last_error(const ea_handle *h) { return h ? h->err.c_str() : g_create_err.c_str(); }
extern "C" int64_t ea_launch_count(ea_handle *h) { return h ? h->launches : 0; }

extern "C" int ea_synchronize(ea_handle *h)
{
    if (!h) return EA_ERR_INVALID_ARG;
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    CUDA_TRY(h, cudaGetLastError());
    return EA_OK;
}

// ---------------------------------------------------------------- inputs
// Host +-1 array -> packed words.  The values are checked on the device while they are packed into
// a scratch copy; the handle's array is replaced only if all of them are valid (state unchanged on
// error), so the host never walks the input.
static int pack_from_host(ea_handle *h, const int8_t *src, int n_outer, int mode, uint32_t *dst)
{
    const size_t n = (size_t)h->R * n_outer * h->N;
    const size_t nw = (size_t)n_outer * h->W * h->N;
    const size_t off_w = (n + 255) & ~(size_t)255, off_f = off_w + 4 * nw;
    char *tmp = scratch(h, off_f + 256);
    if (!tmp) return fail(h, EA_ERR_ALLOC, "pack: cudaMalloc failed");
    int bad = 0;
    cudaError_t e = cudaMemcpyAsync(tmp, src, n, cudaMemcpyHostToDevice, h->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(tmp + off_f, 0, 4, h->stream);
    if (e == cudaSuccess) {
        int grid;
        launch_cfg((int64_t)nw, 128, grid);
        ea::k_pack<<<grid, 128, 0, h->stream>>>(h->P, h->R, n_outer, mode, (const int8_t *)tmp,
                                                (uint32_t *)(tmp + off_w), (int *)(tmp + off_f));
        h->launches++;
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(&bad, tmp + off_f, 4, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    if (e == cudaSuccess && !bad) {
        e = cudaMemcpyAsync(dst, tmp + off_w, 4 * nw, cudaMemcpyDeviceToDevice, h->stream);
    }
    if (e != cudaSuccess) return fail(h, EA_ERR_CUDA, std::string("pack: ") + cudaGetErrorString(e));
    if (bad) return fail(h, EA_ERR_INVALID_ARG, "values must be +1 or -1");
    return recompute_energy(h);
}

extern "C" int ea_set_couplings(ea_handle *h, const int8_t *J)
{
    if (!h || !J) return fail(h, EA_ERR_INVALID_ARG, "ea_set_couplings: null argument");
    { int rc = ensure_r(h); if (rc != EA_OK) return rc; }
    h->t_valid = false;
    return pack_from_host(h, J, 3, 1, h->P.coup);
}

extern "C" int ea_set_spins(ea_handle *h, const int8_t *s)
{
    if (!h || !s) return fail(h, EA_ERR_INVALID_ARG, "ea_set_spins: null argument");
    { int rc = ensure_r(h); if (rc != EA_OK) return rc; }     // a rejected input leaves the state as it was
    h->t_valid = false;
    return pack_from_host(h, s, h->nT, 0, h->P.spin);
}

extern "C" int ea_set_tables(ea_handle *h, const uint64_t *acc, const uint64_t *swp)
{
    if (!h || !acc || (h->nT > 1 && !swp)) return fail(h, EA_ERR_INVALID_ARG, "ea_set_tables: null argument");
    if (h->field != 0) return fail(h, EA_ERR_UNSUPPORTED, "ea_set_tables: zero-field tables only (field is set)");
    const size_t cols = 3 * (size_t)h->N + 1;
    std::vector<uint64_t> a(acc, acc + (size_t)h->nT * 7);
    std::vector<uint64_t> s;
    if (h->nT > 1) s.assign(swp, swp + (size_t)(h->nT - 1) * cols);
    return upload_tables(h, a, &s);
}

extern "C" int ea_get_tables(ea_handle *h, uint64_t *acc, uint64_t *swp)
{
    if (!h) return EA_ERR_INVALID_ARG;
    if (acc) std::memcpy(acc, h->acc.data(), 8 * h->acc.size());
    if (swp && !h->swp.empty()) {
        std::memcpy(swp, h->swp.data(), 8 * h->swp.size());
    } else if (swp) {                     // the default table, written out from its formula
        const int64_t M = 3 * (int64_t)h->N / 2;
        for (int t = 0; t + 1 < h->nT; ++t) {
            const double db = h->betas[t] - h->betas[t + 1];
            for (int64_t m = -M; m <= M; ++m) swp[(size_t)t * (size_t)(2 * M + 1) + (size_t)(m + M)] = threshold_of(db * (double)(4 * m));
        }
    }
    return EA_OK;
}

// ---------------------------------------------------------------- external field
extern "C" int ea_set_field(ea_handle *h, int field)
{
    if (!h) return EA_ERR_INVALID_ARG;
    if (field < -64 || field > 64) return fail(h, EA_ERR_INVALID_ARG, "ea_set_field: |h| <= 64");
    if (field != 0 && h->layout == EA_LAYOUT_REPLICA_BITS)
        return fail(h, EA_ERR_UNSUPPORTED, "ea_set_field: the replica-bits layout runs at h = 0 only");
    const int nT = h->nT, LTS = nT + 1;
    if (field == 0) {
        if (h->field == 0) return EA_OK;
        CUDA_TRY(h, cudaStreamSynchronize(h->stream));
        h->field = 0;
        h->fast_field = false; h->d_bucketF = nullptr; h->d_tripF = nullptr;
        h->P.h = 0; h->P.ediv = 4; h->P.thrF = nullptr; h->P.swp_val = h->d_swp_val;
        for (int c = 0; c < 18; ++c) h->P.zF[c] = -1;
        const std::vector<uint64_t> acc = h->acc, swp = h->swp;
        int rc = upload_tables(h, acc, swp.empty() ? nullptr : &swp);      // the zero-field swap table again
        if (rc != EA_OK) return rc;
        if (h->d_field) { cudaFree(h->d_field); h->d_field = nullptr; }
        h->accf.clear();
        return recompute_energy(h);
    }
    // tables in double on the host, same formulas as at h = 0 (R21)
    const int64_t Mf = (int64_t)(3 + std::abs(field)) * h->N, cols = 2 * Mf + 1;
    std::vector<uint64_t> accf((size_t)nT * 14);
    (void)cols;
    for (int t = 0; t < nT; ++t)
        for (int c = 0; c < 7; ++c)
            for (int up = 0; up < 2; ++up) {
                const double dE = (double)(4 * c - 12 - 2 * field * (2 * up - 1));
                accf[((size_t)t * 7 + c) * 2 + up] = threshold_of(-(h->betas[t] * dE));
            }
    // class thresholds in pos order (coldest first), as (threshold - 1); classes with dE <= 0 flip always
    std::vector<uint32_t> thrF((size_t)18 * LTS, 0xFFFFFFFFu);
    int zF[18];
    for (int j = 0; j < 4; ++j) {       // |h| <= 2: rows 14..17 = columns dE_j = 4 j + 2 (odd h) / 4 j + 4 (even h)
        const double dE = (double)((field & 1) ? 4 * j + 2 : 4 * j + 4);
        int zc = 0;
        for (int pos = 0; pos < nT; ++pos) {
            const int t = h->desc ? pos : nT - 1 - pos;
            const uint64_t v = threshold_of(-(h->betas[t] * dE));
            if (v == 0) { zc = pos + 1; thrF[(size_t)(14 + j) * LTS + pos] = 0; }
            else thrF[(size_t)(14 + j) * LTS + pos] = (uint32_t)(v - 1);
        }
        zF[14 + j] = zc;
    }
    for (int c = 0; c < 7; ++c)
        for (int up = 0; up < 2; ++up) {
            const int cls = 2 * c + up, dE = 4 * c - 12 - 2 * field * (2 * up - 1);
            if (dE <= 0) { zF[cls] = -1; continue; }
            int zc = 0;
            for (int pos = 0; pos < nT; ++pos) {
                const int t = h->desc ? pos : nT - 1 - pos;
                const uint64_t v = accf[((size_t)t * 7 + c) * 2 + up];
                if (v == 0) { zc = pos + 1; thrF[(size_t)cls * LTS + pos] = 0; }
                else thrF[(size_t)cls * LTS + pos] = (uint32_t)(v - 1);
            }
            zF[cls] = zc;
        }
    SwapTrim tr;
    {   // swpf[t][d2 + Mf] = thr((beta_t - beta_{t+1}) 2 d2), trimmed from the formula
        const std::vector<double> &bt = h->betas;
        trim_swap_generated(nT, Mf, [&](int t, int64_t d2) { return threshold_of((bt[t] - bt[t + 1]) * (double)(2 * d2)); }, tr);
    }
    // |h| <= 2: the four columns also get a bucket table, and the resident kernel runs with the field
    std::vector<uint4> tabF;
    std::vector<uchar4> tripF;
    ea::RankKey KF{};
    bool fastF = false;
    if (field >= -2 && field <= 2) {
        std::vector<uint32_t> col(thrF.begin() + (size_t)14 * LTS, thrF.begin() + (size_t)18 * LTS);
        fastF = build_bucket_table(col, zF + 14, nT, 4, tabF, tripF, KF);
    }
    const size_t o_val = align256(4 * thrF.size());
    const size_t o_tab = align256(o_val + 4 * (tr.val.size() + 1)), o_trip = align256(o_tab + 16 * tabF.size());
    char *d = nullptr;
    if (cudaMalloc((void **)&d, o_trip + 4 * tripF.size() + 16) != cudaSuccess) {
        cudaGetLastError();
        return fail(h, EA_ERR_ALLOC, "ea_set_field: cudaMalloc failed");
    }
    cudaError_t e = cudaStreamSynchronize(h->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d, thrF.data(), 4 * thrF.size(), cudaMemcpyHostToDevice, h->stream);
    if (e == cudaSuccess && fastF) e = cudaMemcpyAsync(d + o_tab, tabF.data(), 16 * tabF.size(), cudaMemcpyHostToDevice, h->stream);
    if (e == cudaSuccess && fastF) e = cudaMemcpyAsync(d + o_trip, tripF.data(), 4 * tripF.size(), cudaMemcpyHostToDevice, h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);       // the vectors live on this stack frame
    if (e != cudaSuccess) { cudaFree(d); return fail(h, EA_ERR_CUDA, std::string("ea_set_field: ") + cudaGetErrorString(e)); }
    { int rc = upload_swap_trim(h, tr, (uint32_t *)(d + o_val)); if (rc != EA_OK) { cudaFree(d); return rc; } }
    if (h->d_field) cudaFree(h->d_field);
    h->d_field = d;
    h->field = field;
    h->fast_field = fastF; h->KF = KF;
    h->d_bucketF = (uint4 *)(d + o_tab); h->d_tripF = (uchar4 *)(d + o_trip);
    h->P.h = field; h->P.ediv = 2; h->P.thrF = (const uint32_t *)d; h->P.swp_val = (const uint32_t *)(d + o_val);
    for (int c = 0; c < 18; ++c) h->P.zF[c] = zF[c];
    h->accf.swap(accf);
    return recompute_energy(h);
}

extern "C" int ea_get_field(ea_handle *h) { return h ? h->field : 0; }

extern "C" int ea_get_field_tables(ea_handle *h, uint64_t *accf, uint64_t *swpf)
{
    if (!h) return EA_ERR_INVALID_ARG;
    if (h->field == 0) return fail(h, EA_ERR_INVALID_ARG, "ea_get_field_tables: no field is set");
    if (accf) std::memcpy(accf, h->accf.data(), 8 * h->accf.size());
    if (swpf) {                           // written out from its formula on demand
        const int64_t Mf = (int64_t)(3 + std::abs(h->field)) * h->N;
        for (int t = 0; t + 1 < h->nT; ++t) {
            const double db = h->betas[t] - h->betas[t + 1];
            for (int64_t d2 = -Mf; d2 <= Mf; ++d2)
                swpf[(size_t)t * (size_t)(2 * Mf + 1) + (size_t)(d2 + Mf)] = threshold_of(db * (double)(2 * d2));
        }
    }
    return EA_OK;
}

// ---------------------------------------------------------------- sweep
// One cooperative launch for all sweeps of the call (k_generic_persistent).  Returns
// cudaErrorCooperativeLaunchTooLarge / NotSupported style errors to the caller, which then falls
// back to one launch per step.
static cudaError_t launch_generic_persistent(ea_handle *h, int n_sweeps, int swap_interval)
{
    int coop = 0, dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
    if (!coop) return cudaErrorNotSupported;
    const void *kern = h->field ? (const void *)ea::k_generic_persistent<true> : (const void *)ea::k_generic_persistent<false>;
    const size_t smem = 4 * (h->field ? 18 : 3) * (size_t)(h->nT + 1);
    int per_sm = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, 256, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorCooperativeLaunchTooLarge;
    // Only problems whose work items all get a thread of their own (one wave): these are the
    // launch-latency-bound ones.  Larger problems are throughput-bound and run faster with one
    // launch per step (measured on config 4 with a field: 1.46 against 1.85 ps per attempt).
    const int64_t n_items = (int64_t)h->nT * h->W * (h->N / 8);
    if ((n_items + 255) / 256 > (int64_t)per_sm * h->sm_count) return cudaErrorCooperativeLaunchTooLarge;
    const int64_t want = std::max<int64_t>((n_items + 255) / 256, std::min<int64_t>((int64_t)h->W * h->nT, h->sm_count));
    const int grid = (int)std::min<int64_t>(want, (int64_t)per_sm * h->sm_count);
    ea::PersistArgs A{};
    A.P = h->P; A.g0 = (uint32_t)h->g; A.n_sweeps = n_sweeps; A.swap_interval = swap_interval;
    A.nswap0 = (uint32_t)h->nswap;
    A.gbar = (unsigned int *)(h->d_Ecnt + 2 * (size_t)h->Rp * h->nT);
    e = cudaMemsetAsync(A.gbar, 0, 4, h->stream);
    if (e != cudaSuccess) return e;
    void *args[] = {(void *)&A};
    return cudaLaunchCooperativeKernel(kern, dim3((unsigned)grid), dim3(256), args, smem, h->stream);
}

static int sweep_generic(ea_handle *h, int64_t n_sweeps, int swap_interval)
{
    // persistent path first (EA_KERNEL_GENERIC_STEPWISE asks for the one-launch-per-step path)
    while (n_sweeps > 0 && h->kernel_sel != EA_KERNEL_GENERIC_STEPWISE) {
        const int chunk = (int)std::min<int64_t>(n_sweeps, 1 << 30);
        const cudaError_t e = launch_generic_persistent(h, chunk, swap_interval);
        if (e == cudaErrorCooperativeLaunchTooLarge || e == cudaErrorNotSupported) { cudaGetLastError(); break; }
        if (e != cudaSuccess) return fail(h, EA_ERR_CUDA, std::string("generic persistent launch: ") + cudaGetErrorString(e));
        h->launches++;
        if (swap_interval > 0) h->nswap += (h->g + (uint64_t)chunk) / (uint64_t)swap_interval - h->g / (uint64_t)swap_interval;
        h->g += (uint64_t)chunk;
        h->energy_valid = true;       // the last sweep of a launch always ends with the energies
        n_sweeps -= chunk;
    }
    if (n_sweeps == 0) return EA_OK;
    const int64_t nthreads = (int64_t)h->nT * h->W * (h->N / 8);
    int grid;
    launch_cfg(nthreads, 128, grid);
    const size_t smem = 4 * (h->field ? 18 : 3) * (size_t)(h->nT + 1);
    for (int64_t it = 0; it < n_sweeps; ++it) {
        if (h->field) {
            ea::k_half_sweep_field<<<grid, 128, smem, h->stream>>>(h->P, 0, (uint32_t)h->g);
            ea::k_half_sweep_field<<<grid, 128, smem, h->stream>>>(h->P, 1, (uint32_t)h->g);
        } else {
            ea::k_half_sweep_generic<<<grid, 128, smem, h->stream>>>(h->P, 0, (uint32_t)h->g);
            ea::k_half_sweep_generic<<<grid, 128, smem, h->stream>>>(h->P, 1, (uint32_t)h->g);
        }
        h->launches += 2;
        h->energy_valid = false;
        h->g++;
        if (swap_interval > 0 && h->g % (uint64_t)swap_interval == 0) {
            int rc = recompute_energy(h);
            if (rc != EA_OK) return rc;
            ea::k_pt_swap<<<h->W, 256, 0, h->stream>>>(h->P, (uint32_t)(h->g - 1), (uint32_t)(h->nswap & 1u));
            h->launches++;
            h->nswap++;
        }
    }
    CUDA_TRY(h, cudaGetLastError());
    return EA_OK;
}


// ---------------------------------------------------------------- resident path (L = 8, 16)
namespace {
struct ResPlan { bool ok; int C, S, G, swap_win; size_t smem; bool any; int NQP; size_t any_off; };

// shared memory of k_resident without the swap-threshold window (layout: ea_resident.cuh)
size_t resident_smem(const ea_handle *h, int S)
{
    const bool f = h->field != 0;                 // field: four columns, 32-byte bucket entries
    const size_t N = (size_t)h->N, nT = (size_t)h->nT, LTS = nT + 1, NC = f ? 4 : 3, MTS = NC * nT + 2;
    const size_t nb = f ? 2 * (size_t)h->KF.n_bucket : (size_t)h->K.n_bucket;
    return 16 * nb + 4 * (size_t)S * N + 16 * (size_t)S * MTS +
           4 * ((size_t)S * LTS + NC * LTS + MTS + (size_t)S * 32 + 4 * nT) +
           2 * (2 * nT * 32) + 64 * nT + 4 * nT + 48;
}

ResPlan plan_resident(const ea_handle *h)
{
    ResPlan pl{false, 1, 0, 1, 0, 0, false, 0, 0};
    // run-time geometry: + the word's couplings (3 N words) and the neighbour table (3 words per site)
    const size_t extra = (h->L != 8 && h->L != 16) ? 24 * (size_t)h->N + 16 : 0;
    pl.any = h->L != 8 && h->L != 16;          // any other even L: run-time geometry (ea_small.cuh)
    if (h->field != 0 && !h->fast_field) return pl;   // field: |h| <= 2 only
    if (pl.any && h->N / 2 > 1024) return pl;  // one thread per site of a parity: L <= 12
    const size_t cap = 227 * 1024;
    int C = 0;
    for (int c = 1; c <= 8; c *= 2) {            // cluster sizes 1, 2, 4, 8 (others fail to launch)
        const int S = (h->nT + c - 1) / c;
        if (resident_smem(h, S) + extra <= cap) { C = c; break; }
    }
    if (!C) return pl;
    // small problems: spread the slots over more SMs (cluster sizes 2, 4, 8)
    while (C < 8 && (int64_t)h->W * C * 2 <= h->sm_count && (h->nT + 2 * C - 1) / (2 * C) >= 1 && 2 * C <= h->nT)
        C *= 2;
    pl.C = C;
    pl.S = (h->nT + C - 1) / C;
    pl.G = 1;
    if (h->L == 8) { pl.G = 8; while (pl.G > 1 && pl.G > pl.S) pl.G >>= 1; }
    if (pl.any) {
        pl.NQP = (h->N / 2 + 31) / 32 * 32;                  // thread = site: sites of a parity, padded to warps
        pl.G = std::max(1, std::min(pl.S, 1024 / pl.NQP));
    }
    // the swap-threshold window takes what is left, up to 128 entries per temperature pair
    const size_t base = resident_smem(h, pl.S);
    pl.swap_win = (int)std::min<size_t>(128, (cap - base - extra) / (4 * (size_t)h->nT));
    pl.any_off = (base + 4 * (size_t)h->nT * pl.swap_win + 15) & ~(size_t)15;
    pl.smem = pl.any_off + extra;
    pl.ok = true;
    return pl;
}

template <int L, int G>
cudaError_t launch_resident_t(const ea_handle *h, const ea::ResArgs &A, const ResPlan &pl, bool fast)
{
    auto kern = h->field != 0 ? ea::k_resident<L, G, true, 4> : fast ? ea::k_resident<L, G, true> : ea::k_resident<L, G, false>;
    if (h->swap_mode == EA_SWAP_MOVE && (h->field != 0 || fast))     // moving swaps inside the kernel: FAST variants only
        kern = h->field != 0 ? ea::k_resident<L, G, true, 4, true> : ea::k_resident<L, G, true, 3, true>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)(h->W * pl.C));
    cfg.blockDim = dim3((unsigned)(ea::ResGeom<L>::NQ * G));
    cfg.dynamicSmemBytes = pl.smem;
    cfg.stream = h->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)pl.C;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, A);
}
cudaError_t launch_resident_any(const ea_handle *h, const ea::ResArgs &A, const ResPlan &pl, bool fast)
{
    auto kern = h->field != 0 ? ea::k_resident_any<true, 4> : fast ? ea::k_resident_any<true> : ea::k_resident_any<false>;
    if (h->swap_mode == EA_SWAP_MOVE && (h->field != 0 || fast))
        kern = h->field != 0 ? ea::k_resident_any<true, 4, true> : ea::k_resident_any<true, 3, true>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)(h->W * pl.C));
    cfg.blockDim = dim3((unsigned)(pl.NQP * pl.G));
    cfg.dynamicSmemBytes = pl.smem;
    cfg.stream = h->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)pl.C;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, A);
}
}  // namespace

static int sweep_resident(ea_handle *h, int64_t n_sweeps, int swap_interval)
{
    const ResPlan pl = plan_resident(h);
    if (!pl.ok) return fail(h, EA_ERR_UNSUPPORTED, "resident kernel: shape not supported");
    int64_t left = n_sweeps;
    while (left > 0) {
        const int chunk = (int)std::min<int64_t>(left, 1 << 30);
        ea::ResArgs A{};
        A.P = h->P;
        A.g0 = (uint32_t)h->g;
        A.n_sweeps = chunk;
        A.swap_interval = swap_interval;
        A.nswap0 = (uint32_t)h->nswap;
        A.C = pl.C; A.S = pl.S;
        A.bucket = h->d_bucket; A.K = h->K; A.trip = h->d_trip;
        if (h->field != 0) { A.bucket = h->d_bucketF; A.K = h->KF; A.trip = h->d_tripF; }
        A.swap_win = pl.swap_win;
        for (int r = 0; r < 10; ++r) {
            A.rk[2 * r] = h->P.k0 + (uint32_t)r * 0x9E3779B9u;
            A.rk[2 * r + 1] = h->P.k1 + (uint32_t)r * 0xBB67AE85u;
        }
        cudaError_t e = cudaErrorInvalidValue;
        const bool fast = h->fast_rank;
        A.NQP = pl.NQP; A.G = pl.G; A.any_off = (int)pl.any_off;
        if (pl.any) e = launch_resident_any(h, A, pl, fast);
        else if (h->L == 16) e = launch_resident_t<16, 1>(h, A, pl, fast);
        else if (pl.G == 8) e = launch_resident_t<8, 8>(h, A, pl, fast);
        else if (pl.G == 4) e = launch_resident_t<8, 4>(h, A, pl, fast);
        else if (pl.G == 2) e = launch_resident_t<8, 2>(h, A, pl, fast);
        else e = launch_resident_t<8, 1>(h, A, pl, fast);
        if (e != cudaSuccess) return fail(h, EA_ERR_CUDA, std::string("resident launch: ") + cudaGetErrorString(e));
        h->launches++;
        if (swap_interval > 0) h->nswap += (h->g + (uint64_t)chunk) / (uint64_t)swap_interval - h->g / (uint64_t)swap_interval;
        h->g += (uint64_t)chunk;
        left -= chunk;
    }
    h->energy_valid = true;
    return EA_OK;
}

// ---------------------------------------------------------------- tiled path (L = 16, 32, 64)
namespace {
struct TilePlan { bool ok; int SK, nkg; size_t smem; int nthr, nslab; };

TilePlan plan_tiled(const ea_handle *h)
{
    TilePlan pl{false, 0, 0, 0, 0, 0};
    if (h->L != 16 && h->L != 32 && h->L != 64) return pl;
    const int qpp = (h->L / 8) * h->L;
    int zs = 512 / qpp; if (zs < 1) zs = 1; if (zs > h->L) zs = h->L;
    pl.nthr = qpp * zs; pl.nslab = h->L / zs;
    // slots per block: amortise the per-block set-up (couplings, tables: ~2.5 slot-times)
    // against wave quantisation on sm_count SMs (one 512-thread block per SM)
    double best = -1.0;
    const int nT4 = (h->nT + 3) / 4 * 4;
    for (int sk = 4; sk <= nT4; sk += 4) {
        const int nkg = (h->nT + sk - 1) / sk;
        const int64_t blocks = (int64_t)h->W * pl.nslab * nkg;
        const int64_t waves = (blocks + h->sm_count - 1) / h->sm_count;
        const double eff = (double)blocks / (double)(waves * h->sm_count) * (double)sk / ((double)sk + 2.5);
        if (eff > best) { best = eff; pl.SK = sk; pl.nkg = nkg; }
    }
    const size_t LTS = (size_t)h->nT + 1;
    const size_t MTS = 3 * (size_t)h->nT + 2;
    pl.smem = 16 * (size_t)h->n_bucket + 16 * (size_t)pl.SK * MTS +
              4 * ((size_t)pl.SK * LTS + 3 * LTS + MTS + (size_t)pl.SK * 32) + 16;
    pl.ok = pl.smem <= 200 * 1024;
    return pl;
}

template <int L>
cudaError_t launch_tiled_t(const ea_handle *h, const ea::TiledArgs &A, const TilePlan &pl, bool fast, bool energy)
{
    void (*kern)(const ea::TiledArgs);
    if (fast) kern = energy ? ea::k_tiled_half<L, true, true> : ea::k_tiled_half<L, true, false>;
    else kern = energy ? ea::k_tiled_half<L, false, true> : ea::k_tiled_half<L, false, false>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem);
    if (e != cudaSuccess) return e;
    kern<<<h->W * pl.nslab * pl.nkg, pl.nthr, pl.smem, h->stream>>>(A);
    return cudaGetLastError();
}
}  // namespace

static int sweep_tiled(ea_handle *h, int64_t n_sweeps, int swap_interval)
{
    const TilePlan pl = plan_tiled(h);
    if (!pl.ok) return fail(h, EA_ERR_UNSUPPORTED, "tiled kernel: shape not supported");
    ea::TiledArgs A{};
    A.P = h->P; A.SK = pl.SK; A.n_kgroups = pl.nkg; A.Ecnt = h->d_Ecnt;
    A.bucket = h->d_bucket; A.K = h->K; A.trip = h->d_trip;
    for (int r = 0; r < 10; ++r) {
        A.rk[2 * r] = h->P.k0 + (uint32_t)r * 0x9E3779B9u;
        A.rk[2 * r + 1] = h->P.k1 + (uint32_t)r * 0xBB67AE85u;
    }
    const bool fast = h->fast_rank;
    for (int64_t it = 0; it < n_sweeps; ++it) {
        const bool swap_now = swap_interval > 0 && (h->g + 1) % (uint64_t)swap_interval == 0;
        A.g = (uint32_t)h->g;
        for (int p = 0; p < 2; ++p) {
            A.parity = p;
            const bool energy = p == 1 && swap_now;
            cudaError_t e = cudaErrorInvalidValue;
            if (h->L == 16) e = launch_tiled_t<16>(h, A, pl, fast, energy);
            else if (h->L == 32) e = launch_tiled_t<32>(h, A, pl, fast, energy);
            else e = launch_tiled_t<64>(h, A, pl, fast, energy);
            if (e != cudaSuccess) return fail(h, EA_ERR_CUDA, std::string("tiled launch: ") + cudaGetErrorString(e));
            h->launches++;
        }
        h->energy_valid = false;
        h->g++;
        if (swap_now) {
            int grid;
            launch_cfg((int64_t)h->Rp * h->nT, 256, grid);
            ea::k_tiled_finish<<<grid, 256, 0, h->stream>>>(h->P, h->d_Ecnt);
            ea::k_pt_swap<<<h->W, 256, 0, h->stream>>>(h->P, (uint32_t)(h->g - 1), (uint32_t)(h->nswap & 1u));
            h->launches += 2;
            h->nswap++;
            h->energy_valid = true;
        }
    }
    CUDA_TRY(h, cudaGetLastError());
    return EA_OK;
}

// ---------------------------------------------------------------- streaming path (L = 32, 64)
namespace {
struct StreamPlan { bool ok; int grid, MS, MW, swap_win; size_t smem, esm_off, batch_off; int Wn; };

// plan for one launch over Wn realization words
template <int L>
StreamPlan plan_stream_words(const ea_handle *h, int Wn)
{
    using Sg = ea::StreamGeom<L>;
    StreamPlan pl{false, 0, 0, 0, 0, 0, 0, 0, Wn};
    const long long T = (long long)Wn * Sg::NSLAB * h->nT;
    if (T >= (1ll << 31)) return pl;
    pl.grid = (int)std::min<long long>(h->sm_count, T);
    pl.MS = (int)((T + pl.grid - 1) / pl.grid);
    const long long per_w = (long long)Sg::NSLAB * h->nT;
    pl.MW = (int)((pl.MS + per_w - 2) / per_w) + 1;
    const bool f = h->field != 0;                 // field |h| <= 2: four columns, 32-byte bucket entries
    const size_t nT = (size_t)h->nT, LTS = nT + 1, NC = f ? 4 : 3, MTS = NC * nT + 2;
    const size_t nbk = f ? 2 * (size_t)h->KF.n_bucket : (size_t)h->n_bucket;
    size_t base = Sg::MBAR_BYTES + 16 * nbk + (size_t)Sg::NST * Sg::BUF_BYTES + 16 * (size_t)pl.MS * MTS +
                  4 * ((size_t)pl.MS * LTS + NC * LTS + MTS + (size_t)pl.MS * 32) + 2 * (size_t)pl.MW * 32 * nT;
    pl.esm_off = (base + 15) & ~(size_t)15;
    pl.batch_off = pl.esm_off + 4 * (size_t)pl.MW * 32 * nT;
    base = pl.batch_off + 16 * (size_t)pl.MS + 12 * nT;
    const size_t cap = 227 * 1024;
    if (base > cap) return pl;
    pl.swap_win = (int)std::min<size_t>(128, (cap - base) / (4 * nT));
    pl.smem = base + 4 * nT * (size_t)pl.swap_win;
    pl.ok = pl.MS < 65536;
    return pl;
}

// Words never interact, so a problem whose per-block tables do not fit shared memory is run as
// several launches over balanced groups of words, each for all sweeps of the call: the fewest
// groups whose plan fits.
template <int L>
StreamPlan plan_stream_t(const ea_handle *h)
{
    for (int groups = 1; groups <= h->W; ++groups) {
        const int Wn = (h->W + groups - 1) / groups;
        const StreamPlan pl = plan_stream_words<L>(h, Wn);
        if (pl.ok) return pl;
        if (Wn == 1) break;
    }
    return StreamPlan{false, 0, 0, 0, 0, 0, 0, 0, 0};
}

StreamPlan plan_stream(const ea_handle *h)
{
    int coop = 0, dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
    if (!coop) return StreamPlan{false, 0, 0, 0, 0, 0, 0, 0, 0};
    if (h->field != 0 && !h->fast_field) return StreamPlan{false, 0, 0, 0, 0, 0, 0, 0, 0};   // field: |h| <= 2 only
    if (h->L == 32) return plan_stream_t<32>(h);
    if (h->L == 64) return plan_stream_t<64>(h);
    return StreamPlan{false, 0, 0, 0, 0, 0, 0, 0, 0};
}

template <int L>
cudaError_t launch_stream_t(const ea_handle *h, ea::StreamArgs &A, const StreamPlan &pl, bool fast)
{
    void (*kern)(const ea::StreamArgs) = h->field != 0 ? ea::k_stream<L, true, 4> : fast ? ea::k_stream<L, true> : ea::k_stream<L, false>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem);
    if (e != cudaSuccess) return e;
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, ea::StreamGeom<L>::NTHR, pl.smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1 || (long long)per_sm * h->sm_count < pl.grid) return cudaErrorCooperativeLaunchTooLarge;
    void *args[] = {(void *)&A};
    return cudaLaunchCooperativeKernel((const void *)kern, dim3((unsigned)pl.grid), dim3(ea::StreamGeom<L>::NTHR),
                                       args, pl.smem, h->stream);
}
}  // namespace

static int sweep_stream(ea_handle *h, int64_t n_sweeps, int swap_interval)
{
    const StreamPlan pl = plan_stream(h);
    if (!pl.ok) return fail(h, EA_ERR_UNSUPPORTED, "stream kernel: shape not supported");
    // every word group must have a plan before the first one is launched (the last group may be smaller)
    if (h->W % pl.Wn) {
        const int Wl = h->W % pl.Wn;
        const StreamPlan pt = h->L == 32 ? plan_stream_words<32>(h, Wl) : plan_stream_words<64>(h, Wl);
        if (!pt.ok) return fail(h, EA_ERR_UNSUPPORTED, "stream kernel: word group does not fit");
    }
    int64_t left = n_sweeps;
    while (left > 0) {
        const int chunk = (int)std::min<int64_t>(left, 1 << 30);
      for (int w_off = 0; w_off < h->W; w_off += pl.Wn) {      // groups of words, each for all sweeps of the chunk
        const int Wg = std::min(pl.Wn, h->W - w_off);
        const StreamPlan pg = Wg == pl.Wn ? pl : (h->L == 32 ? plan_stream_words<32>(h, Wg) : plan_stream_words<64>(h, Wg));
        if (!pg.ok) return fail(h, EA_ERR_UNSUPPORTED, "stream kernel: word group does not fit");
        ea::StreamArgs A{};
        A.P = h->P;
        A.Wn = Wg;
        {   // this group's view of the state: pointers, w0 and r0 move to its first word
            Params &Q = A.P;
            Q.spin += (size_t)w_off * h->N;
            Q.coup += (size_t)w_off * 3 * h->N;
            Q.lt += (size_t)w_off * h->nT * (h->nT + 1);
            Q.tau += (size_t)32 * w_off * h->nT;
            Q.sigma += (size_t)32 * w_off * h->nT;
            Q.E += (size_t)32 * w_off * h->nT;
            Q.w0 += (uint32_t)w_off;
            Q.r0 += 32u * (uint32_t)w_off;
        }
        A.g0 = (uint32_t)h->g;
        A.n_sweeps = chunk;
        A.swap_interval = swap_interval;
        A.nswap0 = (uint32_t)h->nswap;
        A.Ecnt = h->d_Ecnt + (size_t)32 * w_off * h->nT;
        A.gbar = (unsigned int *)(h->d_Ecnt + 2 * (size_t)h->Rp * h->nT);
        A.bucket = h->d_bucket; A.K = h->K; A.trip = h->d_trip;
        if (h->field != 0) { A.bucket = h->d_bucketF; A.K = h->KF; A.trip = h->d_tripF; }
        A.MS = pg.MS; A.MW = pg.MW; A.swap_win = pg.swap_win; A.esm_off = (int)pg.esm_off; A.batch_off = (int)pg.batch_off;
        for (int r = 0; r < 10; ++r) {
            A.rk[2 * r] = h->P.k0 + (uint32_t)r * 0x9E3779B9u;
            A.rk[2 * r + 1] = h->P.k1 + (uint32_t)r * 0xBB67AE85u;
        }
#ifdef EA_TRACE   // builder's aid (nvcc -DEA_TRACE): EA_STREAM_TRACE=<file> dumps per-block phase time stamps
        const char *trace_path = std::getenv("EA_STREAM_TRACE");
        unsigned long long *d_trace = nullptr;
        const size_t trace_n = (size_t)pg.grid * 64;
        if (trace_path && cudaMalloc((void **)&d_trace, 8 * trace_n) == cudaSuccess) {
            cudaMemsetAsync(d_trace, 0, 8 * trace_n, h->stream);
            A.trace = d_trace;
        }
#endif
        // counters and the grid-barrier word start from zero in every launch
        CUDA_TRY(h, cudaMemsetAsync(h->d_Ecnt, 0, 2 * 4 * (size_t)h->Rp * h->nT + 256, h->stream));
        const cudaError_t e = h->L == 32 ? launch_stream_t<32>(h, A, pg, h->fast_rank)
                                         : launch_stream_t<64>(h, A, pg, h->fast_rank);
#ifdef EA_TRACE
        if (d_trace) {
            std::vector<unsigned long long> tr(trace_n);
            cudaMemcpyAsync(tr.data(), d_trace, 8 * trace_n, cudaMemcpyDeviceToHost, h->stream);
            cudaStreamSynchronize(h->stream);
            if (FILE *f = std::fopen(trace_path, "wb")) { std::fwrite(tr.data(), 8, trace_n, f); std::fclose(f); }
            cudaFree(d_trace);
        }
#endif
        if (e == cudaErrorCooperativeLaunchTooLarge && h->kernel_sel == EA_KERNEL_AUTO && w_off == 0) {
            // the SMs are not all free (another context holds some): same result, one launch per
            // half-sweep instead of one cooperative launch
            cudaGetLastError();
            return h->field != 0 ? sweep_generic(h, left, swap_interval) : sweep_tiled(h, left, swap_interval);
        }
        if (e != cudaSuccess) {
            // a later group failed: the earlier groups of this chunk have already advanced, so the
            // handle no longer holds ONE simulation state.  Refuse further work until ea_set_state.
            if (w_off > 0) h->poisoned = true;
            return fail(h, EA_ERR_CUDA, std::string("stream launch: ") + cudaGetErrorString(e) +
                                            (w_off > 0 ? " (between word groups: state invalid, restore it with ea_set_state)" : ""));
        }
        h->launches++;
      }
        if (swap_interval > 0) h->nswap += (h->g + (uint64_t)chunk) / (uint64_t)swap_interval - h->g / (uint64_t)swap_interval;
        h->g += (uint64_t)chunk;
        left -= chunk;
    }
    // the tiled path expects its counters cleared
    CUDA_TRY(h, cudaMemsetAsync(h->d_Ecnt, 0, 2 * 4 * (size_t)h->Rp * h->nT, h->stream));
    h->energy_valid = true;
    return EA_OK;
}


// ---------------------------------------------------------------- second layout
namespace {
size_t replica_smem(const ea_handle *h, int ncube, int NW)
{
    return 4 * ((size_t)ncube * h->N + 6 * (size_t)NW) + 8 * 7 * (size_t)h->nT + 4 * 128 + 128 + 16;
}
}  // namespace

extern "C" int ea_set_layout(ea_handle *h, int layout)
{
    if (!h || (layout != EA_LAYOUT_REALIZATION_BITS && layout != EA_LAYOUT_REPLICA_BITS))
        return fail(h, EA_ERR_INVALID_ARG, "ea_set_layout: bad argument");
    if (layout == h->layout) return EA_OK;
    if (h->swap_mode != EA_SWAP_PERMUTE)
        return fail(h, EA_ERR_UNSUPPORTED, "ea_set_layout: the replica-bits layout has no moving swaps (ea_set_swap_mode)");
    if (layout == EA_LAYOUT_REALIZATION_BITS) {
        { int rc = ensure_r(h); if (rc != EA_OK) return rc; }
        h->layout = layout;
        h->t_valid = false;
        return rebuild_lt(h);                     // the permutation has moved since the masks were built
    }
    if (h->field != 0) return fail(h, EA_ERR_UNSUPPORTED, "ea_set_layout: the replica-bits layout runs at h = 0 only");
    const int ncube = (h->nT + 31) / 32, NW = (h->N / 2 + 31) / 32;
    if (replica_smem(h, ncube, NW) > 227 * 1024)
        return fail(h, EA_ERR_UNSUPPORTED, "ea_set_layout: a realization's replicas do not fit shared memory (L <= 32)");
    if (!h->d_rep) {
        const size_t b_spin = align256(4 * (size_t)h->Rp * ncube * h->N), b_j = align256(4 * (size_t)h->Rp * 6 * NW);
        if (cudaMalloc((void **)&h->d_rep, b_spin + b_j + 8 * 7 * (size_t)h->nT) != cudaSuccess)
            return fail(h, EA_ERR_ALLOC, "ea_set_layout: cudaMalloc failed");
        h->d_spinT = (uint32_t *)h->d_rep;
        h->d_jbit = (uint32_t *)(h->d_rep + b_spin);
        h->d_acc64 = (uint64_t *)(h->d_rep + b_spin + b_j);
    }
    h->ncube = ncube; h->NW = NW;
    h->layout = layout;
    h->r_valid = true; h->t_valid = false;
    return EA_OK;
}
extern "C" int ea_get_layout(ea_handle *h) { return h ? h->layout : EA_ERR_INVALID_ARG; }

static int sweep_replica(ea_handle *h, int64_t n_sweeps, int swap_interval)
{
    if (!h->energy_valid) { int rc = recompute_energy(h); if (rc != EA_OK) return rc; }
    { int rc = ensure_t(h); if (rc != EA_OK) return rc; }
    // the probability table, row = temperature index; h->acc outlives the copy
    CUDA_TRY(h, cudaMemcpyAsync(h->d_acc64, h->acc.data(), 8 * 7 * (size_t)h->nT, cudaMemcpyHostToDevice, h->stream));
    const size_t smem = replica_smem(h, h->ncube, h->NW);
    CUDA_TRY(h, cudaFuncSetAttribute(ea::k_replica_sweep, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int64_t left = n_sweeps;
    while (left > 0) {
        const int chunk = (int)std::min<int64_t>(left, 1 << 30);
        ea::ReplicaArgs A = replica_args(h);
        A.g0 = (uint32_t)h->g; A.n_sweeps = chunk; A.swap_interval = swap_interval; A.nswap0 = (uint32_t)h->nswap;
        for (int r = 0; r < 10; ++r) {
            A.rk[2 * r] = h->P.k0 + (uint32_t)r * 0x9E3779B9u;
            A.rk[2 * r + 1] = h->P.k1 + (uint32_t)r * 0xBB67AE85u;
        }
        ea::k_replica_sweep<<<h->Rp, 256, smem, h->stream>>>(A);
        CUDA_TRY(h, cudaGetLastError());
        h->launches++;
        h->r_valid = false;
        if (swap_interval > 0) h->nswap += (h->g + (uint64_t)chunk) / (uint64_t)swap_interval - h->g / (uint64_t)swap_interval;
        h->g += (uint64_t)chunk;
        left -= chunk;
    }
    h->energy_valid = true;
    return EA_OK;
}

static int pick_kernel(const ea_handle *h)
{
    if (h->layout == EA_LAYOUT_REPLICA_BITS) return EA_KERNEL_REPLICA;
    if (h->kernel_sel == EA_KERNEL_GENERIC_STEPWISE) return EA_KERNEL_GENERIC_STEPWISE;
    if (h->field != 0) {     // with a field: |h| <= 2 on the resident (even L <= 12, 16) and streaming (L = 32, 64) kernels,
                             // else the generic path
        if ((h->kernel_sel == EA_KERNEL_AUTO || h->kernel_sel == EA_KERNEL_RESIDENT) && plan_resident(h).ok) return EA_KERNEL_RESIDENT;
        if ((h->kernel_sel == EA_KERNEL_AUTO || h->kernel_sel == EA_KERNEL_STREAM) && plan_stream(h).ok) return EA_KERNEL_STREAM;
        return EA_KERNEL_GENERIC;
    }
    if (h->kernel_sel != EA_KERNEL_AUTO) return h->kernel_sel;
    if (plan_resident(h).ok) return EA_KERNEL_RESIDENT;
    if (plan_stream(h).ok) return EA_KERNEL_STREAM;
    if (plan_tiled(h).ok) return EA_KERNEL_TILED;
    return EA_KERNEL_GENERIC;
}

extern "C" int ea_set_kernel(ea_handle *h, int kernel)
{
    if (!h) return EA_ERR_INVALID_ARG;
    if (h->layout == EA_LAYOUT_REPLICA_BITS)
        return kernel == EA_KERNEL_AUTO ? EA_OK : fail(h, EA_ERR_UNSUPPORTED, "ea_set_kernel: the replica-bits layout has one kernel");
    if (kernel == EA_KERNEL_AUTO || kernel == EA_KERNEL_GENERIC || kernel == EA_KERNEL_GENERIC_STEPWISE) { h->kernel_sel = kernel; return EA_OK; }
    if (h->field != 0 && !(kernel == EA_KERNEL_RESIDENT && plan_resident(h).ok) && !(kernel == EA_KERNEL_STREAM && plan_stream(h).ok))
        return fail(h, EA_ERR_UNSUPPORTED, "ea_set_kernel: with a field only the generic kernel and, for |h| <= 2, the resident (even L <= 12, L = 16) and streaming (L = 32, 64) ones");
    if (kernel == EA_KERNEL_RESIDENT && plan_resident(h).ok) { h->kernel_sel = kernel; return EA_OK; }
    if (kernel == EA_KERNEL_TILED && plan_tiled(h).ok) { h->kernel_sel = kernel; return EA_OK; }
    if (kernel == EA_KERNEL_STREAM && plan_stream(h).ok) { h->kernel_sel = kernel; return EA_OK; }
    return fail(h, EA_ERR_UNSUPPORTED, "ea_set_kernel: kernel not available for this shape");
}
extern "C" int ea_get_kernel(ea_handle *h) { return h ? pick_kernel(h) : EA_ERR_INVALID_ARG; }

static int sweep_dispatch(ea_handle *h, int64_t n_sweeps, int swap_interval)
{
    const int k = pick_kernel(h);
    if (k == EA_KERNEL_REPLICA) return sweep_replica(h, n_sweeps, swap_interval);
    if (k == EA_KERNEL_RESIDENT) return sweep_resident(h, n_sweeps, swap_interval);
    if (k == EA_KERNEL_TILED) return sweep_tiled(h, n_sweeps, swap_interval);
    if (k == EA_KERNEL_STREAM) return sweep_stream(h, n_sweeps, swap_interval);
    return sweep_generic(h, n_sweeps, swap_interval);
}

extern "C" int ea_sweep(ea_handle *h, int64_t n_sweeps, int swap_interval)
{
    if (!h || n_sweeps < 0 || swap_interval < 0) return fail(h, EA_ERR_INVALID_ARG, "ea_sweep: bad argument");
    if (h->g + (uint64_t)n_sweeps > 0xFFFFFFFFull) return fail(h, EA_ERR_RANGE, "ea_sweep: sweep counter would pass 2^32-1");
    if (n_sweeps == 0) return EA_OK;
    if (h->poisoned) return fail(h, EA_ERR_CUDA, "ea_sweep: an earlier call failed between word groups; restore the state with ea_set_state");
    if (h->swap_mode == EA_SWAP_MOVE && swap_interval > 0 && pick_kernel(h) == EA_KERNEL_RESIDENT && (h->field != 0 || h->fast_rank))
        return sweep_resident(h, n_sweeps, swap_interval);      // the resident kernels exchange in shared memory
    if (h->swap_mode == EA_SWAP_MOVE && swap_interval > 0) {
        // sweeps up to the next swap point on the selected kernel (no swap inside), then the exchange
        while (n_sweeps > 0) {
            const int64_t chunk = std::min<int64_t>(n_sweeps, (int64_t)((uint64_t)swap_interval - h->g % (uint64_t)swap_interval));
            int rc = sweep_dispatch(h, chunk, 0);
            if (rc != EA_OK) return rc;
            n_sweeps -= chunk;
            if (h->g % (uint64_t)swap_interval != 0) continue;
            if (!h->energy_valid && (rc = recompute_energy(h)) != EA_OK) return rc;
            ea::k_swap_move<<<dim3((unsigned)h->W, (unsigned)(h->nT / 2)), 256, 0, h->stream>>>(
                h->P, (uint32_t)(h->g - 1), (uint32_t)(h->nswap & 1u));
            CUDA_TRY(h, cudaGetLastError());
            h->launches++;
            h->nswap++;
        }
        return EA_OK;
    }
    return sweep_dispatch(h, n_sweeps, swap_interval);
}

extern "C" int ea_set_swap_mode(ea_handle *h, int mode)
{
    if (!h || (mode != EA_SWAP_PERMUTE && mode != EA_SWAP_MOVE)) return fail(h, EA_ERR_INVALID_ARG, "ea_set_swap_mode: bad argument");
    if (mode == h->swap_mode) return EA_OK;
    if (h->layout != EA_LAYOUT_REALIZATION_BITS)
        return fail(h, EA_ERR_UNSUPPORTED, "ea_set_swap_mode: only in the realization-bits layout");
    if (h->nT < 2) return fail(h, EA_ERR_UNSUPPORTED, "ea_set_swap_mode: needs at least two temperatures");
    // both directions need slot == temperature index for every realization (moving swaps keep it so)
    std::vector<uint8_t> tau((size_t)h->Rp * h->nT);
    CUDA_TRY(h, cudaMemcpyAsync(tau.data(), h->P.tau, tau.size(), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    for (size_t a = 0; a < tau.size(); ++a)
        if (tau[a] != (uint8_t)(a % (size_t)h->nT))
            return fail(h, EA_ERR_UNSUPPORTED, "ea_set_swap_mode: the temperature permutation is not the identity (call it before the first swap round)");
    h->swap_mode = mode;
    return EA_OK;
}
extern "C" int ea_get_swap_mode(ea_handle *h) { return h ? h->swap_mode : EA_ERR_INVALID_ARG; }

// ---------------------------------------------------------------- observables
extern "C" int ea_energy(ea_handle *h, int32_t *E)
{
    if (!h || !E) return fail(h, EA_ERR_INVALID_ARG, "ea_energy: null argument");
    if (!h->energy_valid) { int rc = recompute_energy(h); if (rc != EA_OK) return rc; }
    const size_t n = (size_t)h->R * h->nT;                 // energy[r][t] = E[r][sigma[r][t]], gathered on the device
    int32_t *d = (int32_t *)scratch(h, 4 * n);
    if (!d) return fail(h, EA_ERR_ALLOC, "ea_energy: cudaMalloc failed");
    int grid;
    launch_cfg((int64_t)n, 256, grid);
    ea::k_energy_by_temp<<<grid, 256, 0, h->stream>>>(h->P, h->R, d);
    h->launches++;
    CUDA_TRY(h, cudaGetLastError());
    CUDA_TRY(h, cudaMemcpyAsync(E, d, 4 * n, cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    return EA_OK;
}

extern "C" int ea_overlap(ea_handle *h, const int32_t *pairs, int n_pairs, int32_t *Q)
{
    if (!h || n_pairs < 0 || (n_pairs && (!pairs || !Q))) return fail(h, EA_ERR_INVALID_ARG, "ea_overlap: bad argument");
    for (int p = 0; p < n_pairs; ++p)
        if (pairs[2 * p] < 0 || pairs[2 * p] >= h->R || pairs[2 * p + 1] < -1 || pairs[2 * p + 1] >= h->R)
            return fail(h, EA_ERR_INVALID_ARG, "ea_overlap: realization index out of range");
    if (n_pairs == 0) return EA_OK;
    { int rc = ensure_r(h); if (rc != EA_OK) return rc; }
    const size_t nb_p = 8 * (size_t)n_pairs, nb_q = 4 * (size_t)n_pairs * h->nT;
    int32_t *d = (int32_t *)scratch(h, nb_p + nb_q);
    if (!d) return fail(h, EA_ERR_ALLOC, "ea_overlap: cudaMalloc failed");
    cudaError_t e = cudaMemcpyAsync(d, pairs, nb_p, cudaMemcpyHostToDevice, h->stream);
    if (e == cudaSuccess) {
        ea::k_overlap<<<n_pairs * h->nT, 256, 0, h->stream>>>(h->P, d, d + 2 * (size_t)n_pairs);
        h->launches++;
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(Q, d + 2 * (size_t)n_pairs, nb_q, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return fail(h, EA_ERR_CUDA, std::string("ea_overlap: ") + cudaGetErrorString(e));
    return EA_OK;
}

// ---------------------------------------------------------------- ea_overlap without any allocation
// Scratch of ea_overlap_static: pairs [n_pairs][2] followed by Q [n_pairs][n_temps], int32.  File-scope
// device array: every GPU that loads the library holds these 256 KiB until the process exits.  In host
// code the NAME below is only a stand-in of the host side; the device address comes from
// cudaGetSymbolAddress, once per device, with that device current (overlap_static_ptr).
static __device__ __align__(256) int32_t g_overlap_static[EA_OVERLAP_STATIC_MAX_INT32];

namespace {
constexpr int kMaxDev = 64;
int32_t *g_overlap_static_ptr[kMaxDev] = {};       // by device ordinal; written once, under the lock
std::mutex g_overlap_static_lock;
}  // namespace

static cudaError_t overlap_static_ptr(int32_t **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDev) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> guard(g_overlap_static_lock);
    if (!g_overlap_static_ptr[dev]) {
        void *ptr = nullptr;
        e = cudaGetSymbolAddress(&ptr, g_overlap_static);
        if (e != cudaSuccess) return e;
        g_overlap_static_ptr[dev] = (int32_t *)ptr;
    }
    if (out) *out = g_overlap_static_ptr[dev];
    return cudaSuccess;
}

extern "C" int ea_overlap_static(ea_handle *h, const int32_t *pairs, int n_pairs, int32_t *Q)
{
    if (!h || n_pairs < 0 || (n_pairs && (!pairs || !Q))) return fail(h, EA_ERR_INVALID_ARG, "ea_overlap_static: bad argument");
    for (int p = 0; p < n_pairs; ++p)
        if (pairs[2 * p] < 0 || pairs[2 * p] >= h->R || pairs[2 * p + 1] < -1 || pairs[2 * p + 1] >= h->R)
            return fail(h, EA_ERR_INVALID_ARG, "ea_overlap_static: realization index out of range");
    if (n_pairs == 0) return EA_OK;
    if ((int64_t)n_pairs * (2 + h->nT) > (int64_t)EA_OVERLAP_STATIC_MAX_INT32)
        return fail(h, EA_ERR_RANGE, "ea_overlap_static: n_pairs * (2 + n_temps) = " + std::to_string((int64_t)n_pairs * (2 + h->nT)) +
                                         " exceeds EA_OVERLAP_STATIC_MAX_INT32 = " + std::to_string(EA_OVERLAP_STATIC_MAX_INT32) +
                                         " (split the pair list, or use ea_overlap)");
    { int rc = ensure_r(h); if (rc != EA_OK) return rc; }
    int32_t *d = nullptr;
    cudaError_t e = overlap_static_ptr(&d);
    if (e != cudaSuccess) return fail(h, EA_ERR_CUDA, std::string("ea_overlap_static: cudaGetSymbolAddress: ") + cudaGetErrorString(e));
    const size_t nb_p = 8 * (size_t)n_pairs, nb_q = 4 * (size_t)n_pairs * h->nT;
    // nothing in the array has to start at zero: the pairs are copied in, and every Q element read back
    // below is written by exactly one block of this launch
    e = cudaMemcpyAsync(d, pairs, nb_p, cudaMemcpyHostToDevice, h->stream);
    if (e == cudaSuccess) {
        ea::k_overlap<<<n_pairs * h->nT, 256, 0, h->stream>>>(h->P, d, d + 2 * (size_t)n_pairs);
        h->launches++;
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(Q, d + 2 * (size_t)n_pairs, nb_q, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return fail(h, EA_ERR_CUDA, std::string("ea_overlap_static: ") + cudaGetErrorString(e));
    return EA_OK;
}

extern "C" int ea_get_spins(ea_handle *h, int8_t *s)
{
    if (!h || !s) return fail(h, EA_ERR_INVALID_ARG, "ea_get_spins: null argument");
    { int rc = ensure_r(h); if (rc != EA_OK) return rc; }
    const size_t n = (size_t)h->R * h->nT * h->N;
    int8_t *d = (int8_t *)scratch(h, n);
    if (!d) return fail(h, EA_ERR_ALLOC, "ea_get_spins: cudaMalloc failed");
    int grid;
    launch_cfg((int64_t)n, 256, grid);
    ea::k_unpack_spins<<<grid, 256, 0, h->stream>>>(h->P, h->R, 0, d);
    h->launches++;
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemcpyAsync(s, d, n, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return fail(h, EA_ERR_CUDA, std::string("ea_get_spins: ") + cudaGetErrorString(e));
    return EA_OK;
}

extern "C" int ea_get_state(ea_handle *h, uint32_t *spin_words, uint8_t *temp_of_slot,
                            int32_t *energy_by_slot, uint64_t *sweeps_done, uint64_t *swap_rounds_done)
{
    if (!h) return EA_ERR_INVALID_ARG;
    if (energy_by_slot && !h->energy_valid) { int rc = recompute_energy(h); if (rc != EA_OK) return rc; }
    { int rc = ensure_r(h); if (rc != EA_OK) return rc; }
    const size_t n = (size_t)h->R * h->nT;
    if (spin_words)
        CUDA_TRY(h, cudaMemcpyAsync(spin_words, h->P.spin, 4 * (size_t)h->nT * h->W * h->N, cudaMemcpyDeviceToHost, h->stream));
    if (temp_of_slot) CUDA_TRY(h, cudaMemcpyAsync(temp_of_slot, h->P.tau, n, cudaMemcpyDeviceToHost, h->stream));
    if (energy_by_slot) CUDA_TRY(h, cudaMemcpyAsync(energy_by_slot, h->P.E, 4 * n, cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    if (sweeps_done) *sweeps_done = h->g;
    if (swap_rounds_done) *swap_rounds_done = h->nswap;
    return EA_OK;
}

// ---------------------------------------------------------------- measurement series
extern "C" int ea_get_couplings(ea_handle *h, int8_t *J)
{
    if (!h || !J) return fail(h, EA_ERR_INVALID_ARG, "ea_get_couplings: null argument");
    const size_t n = (size_t)h->R * 3 * h->N;
    int8_t *d = (int8_t *)scratch(h, n);
    if (!d) return fail(h, EA_ERR_ALLOC, "ea_get_couplings: cudaMalloc failed");
    int grid;
    launch_cfg((int64_t)n, 256, grid);
    ea::k_unpack_couplings<<<grid, 256, 0, h->stream>>>(h->P, h->R, d);
    h->launches++;
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemcpyAsync(J, d, n, cudaMemcpyDeviceToHost, h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) return fail(h, EA_ERR_CUDA, std::string("ea_get_couplings: ") + cudaGetErrorString(e));
    return EA_OK;
}

extern "C" int ea_seed_couplings(ea_handle *h, double p_plus)
{
    if (!h || !(p_plus >= 0.0 && p_plus <= 1.0)) return fail(h, EA_ERR_INVALID_ARG, "ea_seed_couplings: p_plus must lie in [0, 1]");
    { int rc = ensure_r(h); if (rc != EA_OK) return rc; }
    h->t_valid = false;
    const unsigned long long thr = (unsigned long long)std::floor(std::ldexp(p_plus, 32));
    int grid;
    launch_cfg((int64_t)h->W * 3 * h->N, 128, grid);
    ea::k_seed_couplings<<<grid, 128, 0, h->stream>>>(h->P, thr);
    h->launches++;
    CUDA_TRY(h, cudaGetLastError());
    return recompute_energy(h);
}

extern "C" int ea_pair_couplings(ea_handle *h)
{
    if (!h) return EA_ERR_INVALID_ARG;
    if (h->R % 64) return fail(h, EA_ERR_INVALID_ARG, "ea_pair_couplings: n_realizations must be a multiple of 64");
    { int rc = ensure_r(h); if (rc != EA_OK) return rc; }
    h->t_valid = false;
    const size_t half = (size_t)(h->W / 2) * 3 * h->N;   // coup is [w][d][p][j]: each half is contiguous
    CUDA_TRY(h, cudaMemcpyAsync(h->P.coup + half, h->P.coup, 4 * half, cudaMemcpyDeviceToDevice, h->stream));
    return recompute_energy(h);
}

extern "C" int ea_measure_begin(ea_handle *h, const int32_t *word_pairs, int n_word_pairs)
{
    if (!h || n_word_pairs < 0 || (n_word_pairs && !word_pairs))
        return fail(h, EA_ERR_INVALID_ARG, "ea_measure_begin: bad argument");
    for (int p = 0; p < n_word_pairs; ++p)
        if (word_pairs[2 * p] < 0 || word_pairs[2 * p] >= h->W || word_pairs[2 * p + 1] < -1 ||
            word_pairs[2 * p + 1] >= h->W)
            return fail(h, EA_ERR_INVALID_ARG, "ea_measure_begin: word index out of range");
    const size_t nq = (size_t)n_word_pairs * 32 * h->nT, ne = (size_t)h->R * h->nT;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t a = off; off = align256(off + bytes); return a; };
    const size_t o_T = take(4 * (size_t)h->nT * h->W * h->N);
    const size_t o_pairs = take(8 * (size_t)(n_word_pairs ? n_word_pairs : 1));
    const size_t o_q1 = take(8 * nq), o_q2 = take(8 * nq), o_q4 = take(16 * nq);
    const size_t o_e1 = take(8 * ne), o_e2 = take(8 * ne);
    const size_t o_corr = take(8 * nq * (size_t)h->L);
    const size_t o_label = take(ne), o_trips = take(8 * (size_t)h->R);
    char *d = nullptr;
    if (cudaMalloc((void **)&d, off) != cudaSuccess) {
        cudaGetLastError();
        return fail(h, EA_ERR_ALLOC, "ea_measure_begin: cudaMalloc failed");
    }
    cudaError_t e = cudaMemsetAsync(d + o_q1, 0, off - o_q1, h->stream);
    if (e == cudaSuccess && n_word_pairs)
        e = cudaMemcpyAsync(d + o_pairs, word_pairs, 8 * (size_t)n_word_pairs, cudaMemcpyHostToDevice, h->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);   // word_pairs is the caller's: copy done before returning
    if (e != cudaSuccess) {
        cudaFree(d);
        return fail(h, EA_ERR_CUDA, std::string("ea_measure_begin: ") + cudaGetErrorString(e));
    }
    if (h->d_meas) cudaFree(h->d_meas);
    h->d_meas = d;
    h->meas_bytes = off;
    h->meas_acc_off = o_q1;
    h->d_T = (uint32_t *)(d + o_T);
    h->M.wpairs = (const int32_t *)(d + o_pairs);
    h->M.P = n_word_pairs;
    h->M.R = h->R;
    h->M.q1 = (int64_t *)(d + o_q1);
    h->M.q2 = (uint64_t *)(d + o_q2);
    h->M.q4 = (uint64_t *)(d + o_q4);
    h->M.e1 = (int64_t *)(d + o_e1);
    h->M.e2 = (uint64_t *)(d + o_e2);
    h->M.corr = (long long *)(d + o_corr);
    h->M.label = (uint8_t *)(d + o_label);
    h->M.trips = (unsigned long long *)(d + o_trips);
    h->meas_n = 0;
    h->meas_on = true;
    return EA_OK;
}

// one measurement of the current state, enqueued on the handle's stream
static int measure_once(ea_handle *h)
{
    if (!h->energy_valid) { int rc = recompute_energy(h); if (rc != EA_OK) return rc; }
    { int rc = ensure_r(h); if (rc != EA_OK) return rc; }
    if (h->M.P > 0) {
        const int nchunk = (h->N / 4 + ea::kGatherThreads - 1) / ea::kGatherThreads, ngrp = (h->nT + 7) / 8;
        ea::k_gather_by_temp<<<h->W * nchunk * ngrp, ea::kGatherThreads, 4 * 8 * (size_t)h->nT, h->stream>>>(h->P, h->d_T);
        const int per_thread = 4 * ((h->N + 511) / 512), grid = h->M.P * h->nT;      // counts per thread < 2^PL
        if (per_thread < (1 << 6)) ea::k_overlap_words<6><<<grid, 128, 0, h->stream>>>(h->P, h->d_T, h->M, nullptr);
        else if (per_thread < (1 << 9)) ea::k_overlap_words<9><<<grid, 128, 0, h->stream>>>(h->P, h->d_T, h->M, nullptr);
        else if (per_thread < (1 << 12)) ea::k_overlap_words<12><<<grid, 128, 0, h->stream>>>(h->P, h->d_T, h->M, nullptr);
        else ea::k_overlap_words<15><<<grid, 128, 0, h->stream>>>(h->P, h->d_T, h->M, nullptr);
        if (3 * h->L <= ea::kCorrThreads) {     // plane-sum correlations: 3 axes x L planes x nsub threads per block
            int nsub = 1;
            while (2 * nsub <= 32 && 2 * nsub * 3 * h->L <= ea::kCorrThreads) nsub *= 2;
            const int per_thread = (h->L * h->L + nsub - 1) / nsub;            // sites per thread < 2^PL
            const bool stage = 4 * (size_t)h->N <= 128 * 1024;
            const size_t sm = 4 * (size_t)((32 * (3 * h->L + 1) + 3) & ~3) + (stage ? 4 * (size_t)h->N : 0);
            void (*kern)(Params, const uint32_t *, ea::Moments);
            if (per_thread < (1 << 6)) kern = stage ? ea::k_plane_corr<6, true> : ea::k_plane_corr<6, false>;
            else if (per_thread < (1 << 9)) kern = stage ? ea::k_plane_corr<9, true> : ea::k_plane_corr<9, false>;
            else if (per_thread < (1 << 12)) kern = stage ? ea::k_plane_corr<12, true> : ea::k_plane_corr<12, false>;
            else kern = stage ? ea::k_plane_corr<15, true> : ea::k_plane_corr<15, false>;
            CUDA_TRY(h, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
            kern<<<grid, ea::kCorrThreads, sm, h->stream>>>(h->P, h->d_T, h->M);
            h->launches++;
        }
        h->launches += 2;
    }
    int grid;
    launch_cfg((int64_t)h->R * h->nT, 128, grid);
    ea::k_accum_energy<<<grid, 128, 0, h->stream>>>(h->P, h->M);
    h->launches++;
    CUDA_TRY(h, cudaGetLastError());
    h->meas_n++;
    return EA_OK;
}

extern "C" int ea_measure(ea_handle *h, int64_t n_meas, int64_t sweeps_between, int swap_interval)
{
    if (!h || n_meas < 0 || sweeps_between < 0 || swap_interval < 0)
        return fail(h, EA_ERR_INVALID_ARG, "ea_measure: bad argument");
    if (!h->meas_on) return fail(h, EA_ERR_INVALID_ARG, "ea_measure: call ea_measure_begin first");
    const long double total = (long double)n_meas * (long double)sweeps_between;
    if ((long double)h->g + total > 4294967295.0L)
        return fail(h, EA_ERR_RANGE, "ea_measure: sweep counter would pass 2^32-1");
    // sum E^2 <= n 9 N^2 and sum q^2 <= n N^2 must fit 64 bits
    const long double cap = 18446744073709551615.0L / (9.0L * (long double)h->N * (long double)h->N);
    if ((long double)h->meas_n + (long double)n_meas > cap)
        return fail(h, EA_ERR_RANGE, "ea_measure: too many measurements for the 64-bit accumulators");
    for (int64_t m = 0; m < n_meas; ++m) {
        if (sweeps_between > 0) { int rc = ea_sweep(h, sweeps_between, swap_interval); if (rc != EA_OK) return rc; }
        int rc = measure_once(h);
        if (rc != EA_OK) return rc;
    }
    return EA_OK;
}

extern "C" int ea_get_moments(ea_handle *h, uint64_t *n_meas, int64_t *q1, uint64_t *q2, uint64_t *q4,
                              int64_t *e1, uint64_t *e2)
{
    if (!h) return EA_ERR_INVALID_ARG;
    if (!h->meas_on) return fail(h, EA_ERR_INVALID_ARG, "ea_get_moments: call ea_measure_begin first");
    const size_t nq = (size_t)h->M.P * 32 * h->nT, ne = (size_t)h->R * h->nT;
    if (q1 && nq) CUDA_TRY(h, cudaMemcpyAsync(q1, h->M.q1, 8 * nq, cudaMemcpyDeviceToHost, h->stream));
    if (q2 && nq) CUDA_TRY(h, cudaMemcpyAsync(q2, h->M.q2, 8 * nq, cudaMemcpyDeviceToHost, h->stream));
    if (q4 && nq) CUDA_TRY(h, cudaMemcpyAsync(q4, h->M.q4, 16 * nq, cudaMemcpyDeviceToHost, h->stream));
    if (e1) CUDA_TRY(h, cudaMemcpyAsync(e1, h->M.e1, 8 * ne, cudaMemcpyDeviceToHost, h->stream));
    if (e2) CUDA_TRY(h, cudaMemcpyAsync(e2, h->M.e2, 8 * ne, cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    if (n_meas) *n_meas = h->meas_n;
    return EA_OK;
}

extern "C" int ea_get_correlation(ea_handle *h, int64_t *C)
{
    if (!h || !C) return fail(h, EA_ERR_INVALID_ARG, "ea_get_correlation: null argument");
    if (!h->meas_on) return fail(h, EA_ERR_INVALID_ARG, "ea_get_correlation: call ea_measure_begin first");
    const size_t n = (size_t)h->M.P * 32 * h->nT * h->L;
    if (n) CUDA_TRY(h, cudaMemcpyAsync(C, h->M.corr, 8 * n, cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    return EA_OK;
}

extern "C" int ea_get_correlation_length(ea_handle *h, double *xi)
{
    if (!h || !xi) return fail(h, EA_ERR_INVALID_ARG, "ea_get_correlation_length: null argument");
    if (!h->meas_on) return fail(h, EA_ERR_INVALID_ARG, "ea_get_correlation_length: call ea_measure_begin first");
    const int L = h->L, nT = h->nT;
    const size_t n = (size_t)h->M.P * 32 * nT * L;
    std::vector<int64_t> C(n);
    if (n) CUDA_TRY(h, cudaMemcpyAsync(C.data(), h->M.corr, 8 * n, cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    // chi(k) ~ sum_d cos(k d) [<C(d)>]; the common factor 1 / (3 N n M) cancels in chi(0) / chi(k_min).
    // Invalid (padding) pairs hold zeros.  xi = sqrt(chi(0) / chi(k_min) - 1) / (2 sin(pi / L)).
    const long double pi = 3.14159265358979323846264338327950288L;
    for (int t = 0; t < nT; ++t) {
        long double chi0 = 0.0L, chik = 0.0L;
        for (int d = 0; d < L; ++d) {
            long double cd = 0.0L;
            for (size_t pb = 0; pb < (size_t)h->M.P * 32; ++pb) cd += (long double)C[(pb * nT + t) * L + d];
            chi0 += cd;
            chik += std::cos(2.0L * pi * (long double)d / (long double)L) * cd;
        }
        xi[t] = (h->meas_n > 0 && chik > 1e-12L * chi0 && chi0 >= chik)
                    ? (double)(std::sqrt(chi0 / chik - 1.0L) / (2.0L * std::sin(pi / (long double)L)))
                    : std::nan("");
    }
    return EA_OK;
}

extern "C" int ea_get_round_trips(ea_handle *h, uint64_t *trips)
{
    if (!h || !trips) return fail(h, EA_ERR_INVALID_ARG, "ea_get_round_trips: null argument");
    if (!h->meas_on) return fail(h, EA_ERR_INVALID_ARG, "ea_get_round_trips: call ea_measure_begin first");
    CUDA_TRY(h, cudaMemcpyAsync(trips, h->M.trips, 8 * (size_t)h->R, cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    return EA_OK;
}

extern "C" int ea_get_binder(ea_handle *h, double *g)
{
    if (!h || !g) return fail(h, EA_ERR_INVALID_ARG, "ea_get_binder: null argument");
    if (!h->meas_on) return fail(h, EA_ERR_INVALID_ARG, "ea_get_binder: call ea_measure_begin first");
    const size_t nq = (size_t)h->M.P * 32 * h->nT;
    std::vector<uint64_t> q2(nq), q4(2 * nq);
    std::vector<int32_t> wp(2 * (size_t)h->M.P);
    if (nq) {
        CUDA_TRY(h, cudaMemcpyAsync(q2.data(), h->M.q2, 8 * nq, cudaMemcpyDeviceToHost, h->stream));
        CUDA_TRY(h, cudaMemcpyAsync(q4.data(), h->M.q4, 16 * nq, cudaMemcpyDeviceToHost, h->stream));
        CUDA_TRY(h, cudaMemcpyAsync(wp.data(), h->M.wpairs, 8 * (size_t)h->M.P, cudaMemcpyDeviceToHost, h->stream));
    }
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    // g = (3 - [<q^4>] / [<q^2>]^2) / 2 = (3 - S4 n M / S2^2) / 2 with S = sums over measurements and
    // valid pairs, n measurements, M valid pairs; 64-bit-mantissa long double throughout.
    long double M = 0.0L;
    for (int p = 0; p < h->M.P; ++p)
        for (int b = 0; b < 32; ++b)
            if (32 * wp[2 * p] + b < h->R && (wp[2 * p + 1] < 0 || 32 * wp[2 * p + 1] + b < h->R)) M += 1.0L;
    for (int t = 0; t < h->nT; ++t) {
        long double s2 = 0.0L, s4 = 0.0L;
        for (size_t pb = 0; pb < (size_t)h->M.P * 32; ++pb) {   // invalid entries hold zeros
            const size_t o = pb * h->nT + t;
            s2 += (long double)q2[o];
            s4 += (long double)q4[2 * o] + 18446744073709551616.0L * (long double)q4[2 * o + 1];
        }
        g[t] = (h->meas_n == 0 || s2 == 0.0L) ? std::nan("")
                                              : (double)(0.5L * (3.0L - s4 * (long double)h->meas_n * M / (s2 * s2)));
    }
    return EA_OK;
}

// ---------------------------------------------------------------- checkpoint / resume
extern "C" int ea_set_state(ea_handle *h, const uint32_t *spin_words, const uint8_t *temp_of_slot,
                            uint64_t sweeps_done, uint64_t swap_rounds_done)
{
    if (!h || !spin_words || !temp_of_slot) return fail(h, EA_ERR_INVALID_ARG, "ea_set_state: null argument");
    if (sweeps_done > 0xFFFFFFFFull) return fail(h, EA_ERR_RANGE, "ea_set_state: sweep counter above 2^32-1");
    const int nT = h->nT;
    std::vector<uint8_t> tau((size_t)h->Rp * nT);
    for (int r = 0; r < h->Rp; ++r) {
        uint64_t seen = 0;                                   // n_temps <= 64
        for (int k = 0; k < nT; ++k) {
            const int t = r < h->R ? temp_of_slot[(size_t)r * nT + k] : k;   // padding realizations: identity
            if (t >= nT || ((seen >> t) & 1u))
                return fail(h, EA_ERR_INVALID_ARG, "ea_set_state: temp_of_slot is not a permutation");
            if (h->swap_mode == EA_SWAP_MOVE && t != k)
                return fail(h, EA_ERR_INVALID_ARG, "ea_set_state: with moving swaps temp_of_slot must be the identity");
            seen |= (uint64_t)1 << t;
            tau[(size_t)r * nT + k] = (uint8_t)t;
        }
    }
    h->r_valid = true; h->t_valid = false;
    h->poisoned = false;
    CUDA_TRY(h, cudaMemcpyAsync(h->P.spin, spin_words, 4 * (size_t)nT * h->W * h->N, cudaMemcpyHostToDevice, h->stream));
    CUDA_TRY(h, cudaMemcpyAsync(h->P.tau, tau.data(), tau.size(), cudaMemcpyHostToDevice, h->stream));
    int grid;
    launch_cfg((int64_t)h->Rp * nT, 128, grid);
    ea::k_invert_perm<<<grid, 128, 0, h->stream>>>(h->P);
    h->launches++;
    CUDA_TRY(h, cudaGetLastError());
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));           // tau lives on this stack frame
    h->g = sweeps_done;
    h->nswap = swap_rounds_done;
    int rc = rebuild_lt(h);
    if (rc != EA_OK) return rc;
    return recompute_energy(h);
}

// ---------------------------------------------------------------- measurement helper
extern "C" int ea_measure_int_peak(void *cuda_stream, double *out)
{
    if (!out) return EA_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return EA_ERR_CUDA;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    uint32_t *d = nullptr;
    if (cudaMalloc((void **)&d, 256) != cudaSuccess) return EA_ERR_ALLOC;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int iters = 4000, blocks = sms * 8, threads = 256;
    const double lane_ops = (double)blocks * threads * iters * 64.0;
    for (int mode = 0; mode < 3; ++mode) {
        float best = 1e30f;
        for (int rep = 0; rep < 4; ++rep) {
            cudaEventRecord(e0, s);
            if (mode == 0) ea::k_int_peak<0><<<blocks, threads, 0, s>>>(d, iters, 0x9E3779B9u, 0x7F4A7C15u);
            if (mode == 1) ea::k_int_peak<1><<<blocks, threads, 0, s>>>(d, iters, 0x9E3779B9u, 0x7F4A7C15u);
            if (mode == 2) ea::k_int_peak<2><<<blocks, threads, 0, s>>>(d, iters, 0x9E3779B9u, 0x7F4A7C15u);
            cudaEventRecord(e1, s);
            cudaEventSynchronize(e1);
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            if (rep > 0 && ms < best) best = ms;
        }
        out[mode] = lane_ops / (best * 1e-3);
    }
    out[3] = (double)sms;
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaError_t e = cudaGetLastError();
    cudaFree(d);
    return e == cudaSuccess ? EA_OK : EA_ERR_CUDA;
}

// examples/resident_phases.py: cycles per phase of k_resident summed by block 0 (reset != 0: clear)
#ifdef EA_TRACE
extern "C" int ea_debug_res_trace(unsigned long long *out, int reset)
{
    if (reset) { unsigned long long z[8] = {}; return (int)cudaMemcpyToSymbol(ea::g_res_trace, z, sizeof z); }
    return (int)cudaMemcpyFromSymbol(out, ea::g_res_trace, 8 * sizeof(unsigned long long));
}
#endif
