/*
 * ea_oracle.c -- CPU ORACLE (test infrastructure, NOT the product).
 *
 * A plain, slow, one-spin-at-a-time implementation of the hot path of
 * arXiv 1311.5582 (Fang et al.): checkerboard single-spin-flip Metropolis
 * sweeps plus parallel tempering on the 3D +-J Edwards-Anderson model.
 * It exists only so that tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline leg can check / time the CUDA path against it.  Nothing in
 * the product path may import, link or call it, and it shares no code,
 * header, table generator or helper with paper_1311_5582_b200/.
 *
 * Every function cites the PAPER.md passage it follows (line numbers of
 * /root/reference/PAPER.md) or the DESIGN.md reading ("R<n>") that fixes
 * what the paper leaves open.  Spins are int8 +-1, one array element per
 * spin; there is no bit packing, no blocking, no fusion in here.
 *
 * Pinned by tests/test_oracle_*.py:
 *   philox      : cuRAND host generator (library) + independent Python ints
 *   tables      : 50-digit mpmath floor(2^32 exp(x)), closed forms
 *   n_sat / dE  : brute-force flip-and-recompute
 *   energy      : incremental == recomputed, every sweep
 *   chain       : exact enumeration of the 2^3 lattice (256 states)
 *   beta = 0    : every attempt accepted (complement identity)
 *   gauge       : bit-exact gauge covariance
 *   ferromagnet : Binder-cumulant crossing near T = 4.51
 *   PT          : sigma/tau inverse permutations, energy multiset conserved,
 *                 <E>(T) with PT == without PT
 *   replica draws (eao_set_draw_mode 1, the paper's coding): beta = 0 complement, gauge
 *                 covariance, incremental == recomputed, 2^3 enumeration with and without PT,
 *                 composition, independence of realizations (tests/test_oracle_replica.py)
 *   bond concentration (eao_seed_couplings): p = 0, 1 closed forms, bond and frustrated-plaquette
 *                 fractions against p and (1 - (2p-1)^4)/2, independent Python Philox
 *                 (tests/test_oracle_couplings.py)
 *   moving swaps (eao_set_swap_mode 1): beta = 0 closed form of the slot permutation, agreement with
 *                 the index-permuting mode through the first swap round, multiset conservation,
 *                 2^3 enumeration (tests/test_oracle_swapmove.py)
 *   field h     : flip-and-recompute dE, incremental == recomputed, exact
 *                 (s -> -s, h -> -h) symmetry, Boltzmann stationarity on the
 *                 2^3 lattice, saturation at large |h| (tests/test_oracle_field.py)
 * No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------ */
/* Philox4x32-10, ref. [60] of the paper (the paper tried
 * philox4x32_7; R10 fixes 10 rounds).          */
/* ------------------------------------------------------------------ */
void eao_philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                       uint32_t k0, uint32_t k1, uint32_t out[4])
{
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* ------------------------------------------------------------------ */
typedef struct eao {
    int L, N, nT, R;
    int r0;              /* global index of realization 0 (multiple of 32):
                            lets a sub-problem reproduce words r0/32.. of a
                            bigger run exactly */
    uint32_t k0, k1;     /* Philox key = (seed low, seed high) */
    double *beta;        /* [nT] */
    uint64_t *acc;       /* [nT][7]        acceptance thresholds              */
    uint64_t *swp;       /* [nT-1][3N+1]   swap thresholds, column m + 3N/2   */
    int h;               /* external field of Eq. 1 (integer, R21); 0 unless eao_set_field */
    uint64_t *accf;      /* h != 0: [nT][7][2] acceptance thresholds, last index (s+1)/2          */
    uint64_t *swpf;      /* h != 0: [nT-1][2 Mf + 1], Mf = (3+|h|) N, column (E_a-E_b)/2 + Mf     */
    int8_t *s;           /* [slot k][site i][r]  +-1                          */
    int8_t *J;           /* [d][site i][r]       +-1, bond i -> i + d^        */
    int32_t *E;          /* [r][slot k]  incremental energy                   */
    int32_t *tau;        /* [r][slot k] -> temperature index                  */
    int32_t *sigma;      /* [r][temp t] -> slot                               */
    int32_t *nbr;        /* [site i][6]: +x,-x,+y,-y,+z,-z neighbour sites (periodic) */
    uint64_t g;          /* sweeps done  */
    uint64_t nswap;      /* swap rounds done */
    int draw_mode;       /* 0: one draw per (site, word, slot) shared by the word's 32 realizations (R11);
                            1: one draw per (site, realization, slot) -- the paper's own coding, in which the
                            bits of a word are the temperature replicas of one realization (eao_set_draw_mode) */
    int swap_mode;       /* 0: an accepted swap exchanges temperature indices, lattices stay (north_star);
                            1: it exchanges the two lattices, temperatures stay with their slots -- the
                            data-moving swap of the paper's discussion, R26 */
    int check;           /* recompute-and-compare energies every sweep */
    int64_t check_failures;
    int64_t n_attempt, n_accept, n_swap_attempt, n_swap_accept;
} eao;

static inline int wrapi(int a, int L) { return a < 0 ? a + L : (a >= L ? a - L : a); }
static inline int site_of(const eao *o, int x, int y, int z)
{
    int L = o->L;
    return wrapi(x, L) + L * (wrapi(y, L) + L * wrapi(z, L));
}
#define S_(o, k, i, r) ((o)->s[((size_t)(k) * (o)->N + (i)) * (o)->R + (r)])
#define J_(o, d, i, r) ((o)->J[((size_t)(d) * (o)->N + (i)) * (o)->R + (r)])

/* Threshold for probability min(1, e^x) as an integer in [0, 2^32]
 * ("convert the pre-generated probabilities ... to 32 bit
 * unsigned integers"; R7/R8: floor(2^32 p) from double, 2^32 kept). */
static uint64_t threshold_of(double x)
{
    if (x >= 0.0) return (uint64_t)1 << 32;
    return (uint64_t)floor(ldexp(exp(x), 32));
}

/* Probability look-up table, PAPER.md:241-243 (row = temperature, column =
 * local energy), at h = 0: column c = n_sat in 0..6, dE = 4c - 12,
 * P = exp(-beta dE).  Swap table: DESIGN.md R5,
 * P = min(1, exp((beta_t - beta_{t+1}) (E_a - E_b))), E_a - E_b = 4m. */
static void build_tables(eao *o)
{
    int M = 3 * o->N / 2;
    for (int t = 0; t < o->nT; ++t)
        for (int c = 0; c < 7; ++c) {
            double dE = (double)(4 * c - 12);
            o->acc[t * 7 + c] = threshold_of(-(o->beta[t] * dE));
        }
    for (int t = 0; t + 1 < o->nT; ++t)
        for (int m = -M; m <= M; ++m) {
            double db = o->beta[t] - o->beta[t + 1];
            o->swp[(size_t)t * (2 * M + 1) + (m + M)] = threshold_of(db * (double)(4 * m));
        }
}

/* Number of satisfied bonds around site (x,y,z) of replica (r, slot k):
 * e_ij = S_i xor J_ij xor S_j per bond (Eq. 3), written
 * in the +-1 notation: bond satisfied <=> J s_i s_j = +1.  The +d bond uses
 * J_d(i), the -d bond uses J_d(i - d^).  Six bond slots even for L = 2. */
static int n_sat(const eao *o, int k, int r, int i)
{
    const int32_t *nb = o->nbr + 6 * i;
    int si = S_(o, k, i, r);
    int n = 0;
    for (int d = 0; d < 3; ++d) {
        int jp = nb[2 * d], jm = nb[2 * d + 1];
        n += (J_(o, d, i, r) * si * S_(o, k, jp, r) == 1);   /* bond i -> i + d^      */
        n += (J_(o, d, jm, r) * si * S_(o, k, jm, r) == 1);  /* bond (i - d^) -> i    */
    }
    return n;
}
int eao_n_sat(const eao *o, int k, int r, int site) { return n_sat(o, k, r, site); }

/* H = - sum_<ij> J_ij s_i s_j + h sum_i s_i (Eq. 1, sign of the
 * field term as printed; R21), from scratch: every site contributes
 * its three forward bonds and its field term. */
int32_t eao_energy_from_scratch(const eao *o, int r, int k)
{
    int32_t H = 0;
    int L = o->L;
    for (int z = 0; z < L; ++z)
        for (int y = 0; y < L; ++y)
            for (int x = 0; x < L; ++x) {
                int i = site_of(o, x, y, z);
                int si = S_(o, k, i, r);
                H -= J_(o, 0, i, r) * si * S_(o, k, site_of(o, x + 1, y, z), r);
                H -= J_(o, 1, i, r) * si * S_(o, k, site_of(o, x, y + 1, z), r);
                H -= J_(o, 2, i, r) * si * S_(o, k, site_of(o, x, y, z + 1), r);
                H += o->h * si;
            }
    return H;
}

static void recompute_all_energies(eao *o)
{
    for (int r = 0; r < o->R; ++r)
        for (int k = 0; k < o->nT; ++k)
            o->E[r * o->nT + k] = eao_energy_from_scratch(o, r, k);
}

/* Seeded disorder and initial spins (R12, R15): iid p = 1/2 bits
 * of Philox words; bit b of word w is realization 32 w + b; bit 1 <-> +1.
 *   spin word (slot k, site i, word w)  = PX(0, i>>2, w, (3<<16)|k)[i&3]
 *   coupling word (dir d, site i, word w) = PX(0, i, w, 4<<16)[d]          */
static void init_from_seed(eao *o)
{
    uint32_t out[4];
    for (int r = 0; r < o->R; ++r) {
        uint32_t gr = (uint32_t)(o->r0 + r), w = gr >> 5, b = gr & 31;
        for (int i = 0; i < o->N; ++i) {
            eao_philox4x32_10(0u, (uint32_t)i, w, 4u << 16, o->k0, o->k1, out);
            for (int d = 0; d < 3; ++d)
                J_(o, d, i, r) = ((out[d] >> b) & 1u) ? 1 : -1;
            for (int k = 0; k < o->nT; ++k) {
                eao_philox4x32_10(0u, (uint32_t)(i >> 2), w, (3u << 16) | (uint32_t)k,
                                  o->k0, o->k1, out);
                S_(o, k, i, r) = ((out[i & 3] >> b) & 1u) ? 1 : -1;
            }
        }
    }
}

void eao_destroy(eao *o)
{
    if (!o) return;
    free(o->beta); free(o->acc); free(o->swp); free(o->accf); free(o->swpf); free(o->s); free(o->J);
    free(o->E); free(o->tau); free(o->sigma); free(o->nbr); free(o);
}

/* Problem statement PAPER.md:44-59: L^3 periodic cubic lattice, R disorder
 * realizations, nT temperature replicas each.  r0 = global index of the
 * first realization (0 for a whole problem). */
eao *eao_create(int L, int nT, int R, const double *betas, uint64_t seed, int r0)
{
    if (L < 2 || (L & 1) || nT < 1 || R < 1 || !betas || r0 < 0 || (r0 & 31)) return NULL;
    eao *o = (eao *)calloc(1, sizeof(eao));
    if (!o) return NULL;
    o->L = L; o->N = L * L * L; o->nT = nT; o->R = R; o->r0 = r0;
    o->k0 = (uint32_t)seed; o->k1 = (uint32_t)(seed >> 32);
    int M = 3 * o->N / 2;
    o->beta = (double *)malloc(sizeof(double) * nT);
    o->acc = (uint64_t *)malloc(sizeof(uint64_t) * nT * 7);
    o->swp = (uint64_t *)malloc(sizeof(uint64_t) * (size_t)(nT > 1 ? nT - 1 : 1) * (2 * M + 1));
    o->s = (int8_t *)malloc((size_t)nT * o->N * R);
    o->J = (int8_t *)malloc((size_t)3 * o->N * R);
    o->E = (int32_t *)malloc(sizeof(int32_t) * R * nT);
    o->tau = (int32_t *)malloc(sizeof(int32_t) * R * nT);
    o->sigma = (int32_t *)malloc(sizeof(int32_t) * R * nT);
    o->nbr = (int32_t *)malloc(sizeof(int32_t) * 6 * o->N);
    if (!o->beta || !o->acc || !o->swp || !o->s || !o->J || !o->E || !o->tau || !o->sigma || !o->nbr) {
        eao_destroy(o); return NULL;
    }
    memcpy(o->beta, betas, sizeof(double) * nT);
    /* periodic boundary conditions */
    for (int z = 0; z < L; ++z)
        for (int y = 0; y < L; ++y)
            for (int x = 0; x < L; ++x) {
                int32_t *nb = o->nbr + 6 * site_of(o, x, y, z);
                nb[0] = site_of(o, x + 1, y, z); nb[1] = site_of(o, x - 1, y, z);
                nb[2] = site_of(o, x, y + 1, z); nb[3] = site_of(o, x, y - 1, z);
                nb[4] = site_of(o, x, y, z + 1); nb[5] = site_of(o, x, y, z - 1);
            }
    build_tables(o);
    init_from_seed(o);
    for (int r = 0; r < R; ++r)
        for (int k = 0; k < nT; ++k) { o->tau[r * nT + k] = k; o->sigma[r * nT + k] = k; }
    recompute_all_energies(o);
    return o;
}

/* Constant external field h of Eq. 1 ("a constant external
 * field, h, is included in our implementation").  Flipping s_i
 * changes H by dE = (4 n_sat - 12) - 2 h s_i, so the look-up table gets the
 * paper's 14 columns "7 possible local energies E, 2 spins S":
 *   accf[t][c][(s+1)/2] = threshold(-beta_t dE).
 * h is an integer so that H stays an exact integer (R21); E_a - E_b
 * is then even, and the swap table is indexed by (E_a - E_b)/2:
 *   swpf[t][d2 + Mf] = threshold((beta_t - beta_{t+1}) 2 d2),  |d2| <= Mf = (3+|h|) N.
 * h = 0 restores the zero-field tables.  Energies are recomputed. */
int eao_set_field(eao *o, int h)
{
    if (h < -64 || h > 64) return -1;
    free(o->accf); free(o->swpf);
    o->accf = NULL; o->swpf = NULL;
    o->h = h;
    if (h != 0) {
        int64_t Mf = (int64_t)(3 + abs(h)) * o->N;
        o->accf = (uint64_t *)malloc(sizeof(uint64_t) * o->nT * 14);
        o->swpf = (uint64_t *)malloc(sizeof(uint64_t) * (size_t)(o->nT > 1 ? o->nT - 1 : 1) * (size_t)(2 * Mf + 1));
        if (!o->accf || !o->swpf) return -2;
        for (int t = 0; t < o->nT; ++t)
            for (int c = 0; c < 7; ++c)
                for (int sp = 0; sp < 2; ++sp) {
                    int s = 2 * sp - 1;
                    double dE = (double)(4 * c - 12 - 2 * h * s);
                    o->accf[(t * 7 + c) * 2 + sp] = threshold_of(-(o->beta[t] * dE));
                }
        for (int t = 0; t + 1 < o->nT; ++t) {
            double db = o->beta[t] - o->beta[t + 1];
            for (int64_t d2 = -Mf; d2 <= Mf; ++d2)
                o->swpf[(size_t)t * (size_t)(2 * Mf + 1) + (size_t)(d2 + Mf)] = threshold_of(db * (double)(2 * d2));
        }
    }
    recompute_all_energies(o);
    return 0;
}
int eao_get_field(const eao *o) { return o->h; }
/* accf [nT][7][2], swpf [nT-1][2 (3+|h|) N + 1]; only for h != 0. */
int eao_get_field_tables(const eao *o, uint64_t *accf, uint64_t *swpf)
{
    if (o->h == 0) return -1;
    int64_t Mf = (int64_t)(3 + abs(o->h)) * o->N;
    memcpy(accf, o->accf, sizeof(uint64_t) * o->nT * 14);
    if (o->nT > 1) memcpy(swpf, o->swpf, sizeof(uint64_t) * (size_t)(o->nT - 1) * (size_t)(2 * Mf + 1));
    return 0;
}

void eao_set_check(eao *o, int on) { o->check = on; }
int64_t eao_check_failures(const eao *o) { return o->check_failures; }

/* J[r][d][site] in {+1,-1} (canonical order of the C ABI). */
int eao_set_couplings(eao *o, const int8_t *J)
{
    size_t n = (size_t)o->R * 3 * o->N;
    for (size_t a = 0; a < n; ++a) if (J[a] != 1 && J[a] != -1) return -1;
    for (int r = 0; r < o->R; ++r)
        for (int d = 0; d < 3; ++d)
            for (int i = 0; i < o->N; ++i)
                J_(o, d, i, r) = J[((size_t)r * 3 + d) * o->N + i];
    recompute_all_energies(o);
    return 0;
}

/* Other bimodal coupling distributions ("other distributions of the couplings";
 * PAPER.md:44 fixes only the mean): the +-J model with bond concentration p_plus = P(J = +1),
 * each bond independently (R25).  p_plus = 1/2 is the paper's distribution in law (not
 * the same sample as the default seeding), 1 the ferromagnet, 0 the antiferromagnet.
 *   J_d(i) of realization r = +1  iff  PX(0, i, r0 + r, (5<<16)|d)[0] < floor(2^32 p_plus)
 * (64-bit compare, so p_plus = 1 gives +1 everywhere).  Spins, permutation, counters are kept;
 * energies are recomputed. */
int eao_seed_couplings(eao *o, double p_plus)
{
    if (!(p_plus >= 0.0 && p_plus <= 1.0)) return -1;
    uint64_t thr = (uint64_t)floor(ldexp(p_plus, 32));
    uint32_t out[4];
    for (int r = 0; r < o->R; ++r)
        for (int d = 0; d < 3; ++d)
            for (int i = 0; i < o->N; ++i) {
                eao_philox4x32_10(0u, (uint32_t)i, (uint32_t)(o->r0 + r), (5u << 16) | (uint32_t)d,
                                  o->k0, o->k1, out);
                J_(o, d, i, r) = (uint64_t)out[0] < thr ? 1 : -1;
            }
    recompute_all_energies(o);
    return 0;
}

/* s[r][slot][site] in {+1,-1}. */
int eao_set_spins(eao *o, const int8_t *s)
{
    size_t n = (size_t)o->R * o->nT * o->N;
    for (size_t a = 0; a < n; ++a) if (s[a] != 1 && s[a] != -1) return -1;
    for (int r = 0; r < o->R; ++r)
        for (int k = 0; k < o->nT; ++k)
            for (int i = 0; i < o->N; ++i)
                S_(o, k, i, r) = s[((size_t)r * o->nT + k) * o->N + i];
    recompute_all_energies(o);
    return 0;
}

/* Both tables may be replaced by caller-supplied data (north_star: "handed
 * to both paths as input data"). */
void eao_set_tables(eao *o, const uint64_t *acc, const uint64_t *swp)
{
    int M = 3 * o->N / 2;
    memcpy(o->acc, acc, sizeof(uint64_t) * o->nT * 7);
    if (o->nT > 1) memcpy(o->swp, swp, sizeof(uint64_t) * (size_t)(o->nT - 1) * (2 * M + 1));
}
void eao_get_tables(const eao *o, uint64_t *acc, uint64_t *swp)
{
    int M = 3 * o->N / 2;
    memcpy(acc, o->acc, sizeof(uint64_t) * o->nT * 7);
    if (o->nT > 1) memcpy(swp, o->swp, sizeof(uint64_t) * (size_t)(o->nT - 1) * (2 * M + 1));
}

/* One half-sweep: every site of parity p, every slot, every word
 * ("two consecutive stages concentrating independently on each
 * of the sub-lattices").  Random draw: one uint32 per (site, word, slot),
 * shared by the 32 realizations of the word (R11), taken from
 *   PX(g, q, w, (p<<16)|k)[l],  j = (x>>1) + (L/2)(y + L z), q = j>>2, l = j&3
 * (DESIGN.md "RNG convention").  Flip iff draw < acc[tau][n_sat]
 * (Eq. 5 with the sign fixed by R1); with a field
 * the column is (n_sat, s_i) and dE = 4 n_sat - 12 - 2 h s_i (eao_set_field). */
static void half_sweep(eao *o, int p)
{
    int L = o->L, nT = o->nT;
    uint32_t out[4];
    int W0 = o->r0 >> 5, W1 = (o->r0 + o->R + 31) >> 5;
    for (int k = 0; k < nT; ++k)
        for (int z = 0; z < L; ++z)
            for (int y = 0; y < L; ++y)
                for (int x = 0; x < L; ++x) {
                    if (((x + y + z) & 1) != p) continue;
                    int i = x + L * (y + L * z);
                    uint32_t j = (uint32_t)((x >> 1) + (L / 2) * (y + L * z));
                    for (int w = W0; w < W1; ++w) {
                        eao_philox4x32_10((uint32_t)o->g, j >> 2, (uint32_t)w,
                                          ((uint32_t)p << 16) | (uint32_t)k, o->k0, o->k1, out);
                        uint64_t u = out[j & 3];
                        for (int b = 0; b < 32; ++b) {
                            int r = 32 * w + b - o->r0;
                            if (r < 0 || r >= o->R) continue;
                            int c = n_sat(o, k, r, i);
                            int t = o->tau[r * nT + k];
                            o->n_attempt++;
                            int si = S_(o, k, i, r);
                            uint64_t thr = o->h == 0 ? o->acc[t * 7 + c]
                                                     : o->accf[(t * 7 + c) * 2 + (si + 1) / 2];
                            if (u < thr) {
                                S_(o, k, i, r) = (int8_t)(-si);
                                o->E[r * nT + k] += 4 * c - 12 - 2 * o->h * si;
                                o->n_accept++;
                            }
                        }
                    }
                }
}

/* Second workload (R24): the paper packs the spins of the temperature
 * replicas of ONE disorder realization at a site into a word ("spins from different
 * temperature replicas at the same position are encoded into an integer", :186 AMSC, :281 CAMSC),
 * and every replica is "an independent Monte Carlo process" (Figure 3) with its own
 * random number.  Model, tables, sweep order and parallel tempering are unchanged; only the draw is
 * now one uint32 per (site, REALIZATION, slot):
 *   PX(g, q, r, ((6+p)<<16)|k)[l],  r = global realization index, q = j>>2, l = j&3.
 * Flip iff draw < acc[tau][n_sat] exactly as in half_sweep. */
static void half_sweep_replica_draws(eao *o, int p)
{
    int L = o->L, nT = o->nT;
    uint32_t out[4];
    for (int k = 0; k < nT; ++k)
        for (int z = 0; z < L; ++z)
            for (int y = 0; y < L; ++y)
                for (int x = 0; x < L; ++x) {
                    if (((x + y + z) & 1) != p) continue;
                    int i = x + L * (y + L * z);
                    uint32_t j = (uint32_t)((x >> 1) + (L / 2) * (y + L * z));
                    for (int r = 0; r < o->R; ++r) {
                        eao_philox4x32_10((uint32_t)o->g, j >> 2, (uint32_t)(o->r0 + r),
                                          ((uint32_t)(6 + p) << 16) | (uint32_t)k, o->k0, o->k1, out);
                        uint64_t u = out[j & 3];
                        int c = n_sat(o, k, r, i);
                        int t = o->tau[r * nT + k];
                        o->n_attempt++;
                        int si = S_(o, k, i, r);
                        uint64_t thr = o->h == 0 ? o->acc[t * 7 + c]
                                                 : o->accf[(t * 7 + c) * 2 + (si + 1) / 2];
                        if (u < thr) {
                            S_(o, k, i, r) = (int8_t)(-si);
                            o->E[r * nT + k] += 4 * c - 12 - 2 * o->h * si;
                            o->n_accept++;
                        }
                    }
                }
}

int eao_set_draw_mode(eao *o, int mode)
{
    if (mode != 0 && mode != 1) return -1;
    o->draw_mode = mode;
    return 0;
}
int eao_get_draw_mode(const eao *o) { return o->draw_mode; }

/* 0: swaps permute temperature indices; 1: swaps move the lattices (R26). */
int eao_set_swap_mode(eao *o, int mode)
{
    if (mode != 0 && mode != 1) return -1;
    o->swap_mode = mode;
    return 0;
}
int eao_get_swap_mode(const eao *o) { return o->swap_mode; }

/* One parallel-tempering round (temperatures
 * (table rows) are exchanged, lattices stay where they are).  Round n pairs
 * temperature indices (t, t+1) for t = n&1, n&1 + 2, ... (R4);
 * a = slot at t, b = slot at t+1; accept iff
 *   PX(g_done, t, r, 2<<16)[0] < swp[t][(E_a - E_b)/4]      (R5). */
static void swap_round(eao *o, uint64_t g_done)
{
    int nT = o->nT, M = 3 * o->N / 2;
    uint32_t out[4];
    for (int r = 0; r < o->R; ++r) {
        int32_t *sg = o->sigma + r * nT, *ta = o->tau + r * nT, *E = o->E + r * nT;
        for (int t = (int)(o->nswap & 1); t + 1 < nT; t += 2) {
            int a = sg[t], b = sg[t + 1];
            int dE = E[a] - E[b];
            int m = dE / 4;              /* exact at h = 0: dE is a multiple of 4 */
            eao_philox4x32_10((uint32_t)g_done, (uint32_t)t, (uint32_t)(o->r0 + r), 2u << 16,
                              o->k0, o->k1, out);
            uint64_t v = out[0];
            o->n_swap_attempt++;
            uint64_t thr;
            if (o->h == 0) {
                thr = o->swp[(size_t)t * (2 * M + 1) + (m + M)];
            } else {                     /* dE is even: column dE/2 of the field table */
                int64_t Mf = (int64_t)(3 + abs(o->h)) * o->N;
                thr = o->swpf[(size_t)t * (size_t)(2 * Mf + 1) + (size_t)(dE / 2 + Mf)];
            }
            if (v < thr && o->swap_mode == 0) {
                sg[t] = b; sg[t + 1] = a;
                ta[a] = t + 1; ta[b] = t;
                o->n_swap_accept++;
            } else if (v < thr) {        /* R26: the configurations change places, tau stays as it is */
                for (int i = 0; i < o->N; ++i) {
                    int8_t x = S_(o, a, i, r);
                    S_(o, a, i, r) = S_(o, b, i, r);
                    S_(o, b, i, r) = x;
                }
                int32_t e = E[a]; E[a] = E[b]; E[b] = e;
                o->n_swap_accept++;
            }
        }
    }
    o->nswap++;
}

/* n_sweeps full checkerboard sweeps; a swap round follows every sweep whose
 * 1-based global index is a multiple of swap_interval (R6);
 * swap_interval = 0: no parallel tempering. */
int eao_sweep(eao *o, int64_t n_sweeps, int swap_interval)
{
    if (n_sweeps < 0 || swap_interval < 0) return -1;
    if (o->g + (uint64_t)n_sweeps > 0xFFFFFFFFull) return -4;
    for (int64_t it = 0; it < n_sweeps; ++it) {
        if (o->draw_mode == 0) {
            half_sweep(o, 0);
            half_sweep(o, 1);
        } else {
            half_sweep_replica_draws(o, 0);
            half_sweep_replica_draws(o, 1);
        }
        if (o->check) {
            for (int r = 0; r < o->R; ++r)
                for (int k = 0; k < o->nT; ++k)
                    if (o->E[r * o->nT + k] != eao_energy_from_scratch(o, r, k))
                        o->check_failures++;
        }
        o->g++;
        if (swap_interval > 0 && o->g % (uint64_t)swap_interval == 0)
            swap_round(o, o->g - 1);
    }
    return 0;
}

/* E[r][t] by temperature index. */
void eao_energy(const eao *o, int32_t *E)
{
    for (int r = 0; r < o->R; ++r)
        for (int t = 0; t < o->nT; ++t)
            E[r * o->nT + t] = o->E[r * o->nT + o->sigma[r * o->nT + t]];
}

/* Q[p][t] = sum_i s_i^(ra, t) s_i^(rb, t) at equal temperature index
 * (R16); rb = -1: all-up reference, i.e. the magnetization. */
int eao_overlap(const eao *o, const int32_t *pairs, int n_pairs, int32_t *Q)
{
    for (int p = 0; p < n_pairs; ++p) {
        int ra = pairs[2 * p], rb = pairs[2 * p + 1];
        if (ra < 0 || ra >= o->R || rb < -1 || rb >= o->R) return -1;
    }
    for (int p = 0; p < n_pairs; ++p) {
        int ra = pairs[2 * p], rb = pairs[2 * p + 1];
        for (int t = 0; t < o->nT; ++t) {
            int ka = o->sigma[ra * o->nT + t];
            int kb = rb >= 0 ? o->sigma[rb * o->nT + t] : 0;
            int32_t q = 0;
            for (int i = 0; i < o->N; ++i)
                q += S_(o, ka, i, ra) * (rb >= 0 ? S_(o, kb, i, rb) : 1);
            Q[p * o->nT + t] = q;
        }
    }
    return 0;
}

/* s[r][t][site], +-1, by temperature index. */
void eao_get_spins(const eao *o, int8_t *s)
{
    for (int r = 0; r < o->R; ++r)
        for (int t = 0; t < o->nT; ++t) {
            int k = o->sigma[r * o->nT + t];
            for (int i = 0; i < o->N; ++i)
                s[((size_t)r * o->nT + t) * o->N + i] = S_(o, k, i, r);
        }
}
/* s[r][slot][site], by storage slot. */
void eao_get_spins_by_slot(const eao *o, int8_t *s)
{
    for (int r = 0; r < o->R; ++r)
        for (int k = 0; k < o->nT; ++k)
            for (int i = 0; i < o->N; ++i)
                s[((size_t)r * o->nT + k) * o->N + i] = S_(o, k, i, r);
}
void eao_get_couplings(const eao *o, int8_t *J)
{
    for (int r = 0; r < o->R; ++r)
        for (int d = 0; d < 3; ++d)
            for (int i = 0; i < o->N; ++i)
                J[((size_t)r * 3 + d) * o->N + i] = J_(o, d, i, r);
}
void eao_get_perm(const eao *o, int32_t *tau, int32_t *sigma)
{
    memcpy(tau, o->tau, sizeof(int32_t) * o->R * o->nT);
    memcpy(sigma, o->sigma, sizeof(int32_t) * o->R * o->nT);
}
void eao_get_energy_by_slot(const eao *o, int32_t *E)
{
    memcpy(E, o->E, sizeof(int32_t) * o->R * o->nT);
}
/* Resume from a checkpoint ("spin configurations are dumped to the GPU global memory
 * periodically"): spins by slot, the temperature permutation and the two
 * counters that address the random draws.  tau must be a permutation of
 * 0..nT-1 for every realization; energies are recomputed. */
int eao_set_state(eao *o, const int8_t *s, const int32_t *tau, uint64_t g, uint64_t nswap)
{
    int nT = o->nT;
    if (g > 0xFFFFFFFFull) return -4;
    for (int r = 0; r < o->R; ++r) {
        uint64_t seen = 0, seen_hi = 0;
        for (int k = 0; k < nT; ++k) {
            int t = tau[r * nT + k];
            if (t < 0 || t >= nT) return -1;
            if (t < 64) { if ((seen >> t) & 1u) return -1; seen |= (uint64_t)1 << t; }
            else { if ((seen_hi >> (t - 64)) & 1u) return -1; seen_hi |= (uint64_t)1 << (t - 64); }
        }
    }
    if (eao_set_spins(o, s) != 0) return -1;
    for (int r = 0; r < o->R; ++r)
        for (int k = 0; k < nT; ++k) {
            int t = tau[r * nT + k];
            o->tau[r * nT + k] = t;
            o->sigma[r * nT + t] = k;
        }
    o->g = g;
    o->nswap = nswap;
    return 0;
}

void eao_get_counters(const eao *o, uint64_t *g, uint64_t *nswap, int64_t *stats)
{
    *g = o->g; *nswap = o->nswap;
    stats[0] = o->n_attempt; stats[1] = o->n_accept;
    stats[2] = o->n_swap_attempt; stats[3] = o->n_swap_accept;
}
