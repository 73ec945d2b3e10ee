/*
 * ea.h -- C ABI of libea_b200.so: Metropolis sweeps + parallel tempering for the 3D +-J
 * Edwards-Anderson spin glass on one NVIDIA B200 (sm_100a).
 *
 * Method: arXiv 1311.5582 (Fang et al.).  Citations are PAPER.md:<line> (+ section/equation);
 * conventions that the paper leaves open are frozen in DESIGN.md section 2 ("R<n>").
 *
 * General rules
 *   - Every pointer argument is a HOST pointer unless its name starts with dev_.
 *   - The caller owns every input and output buffer; the library copies.  The library owns
 *     the device state of a handle until ea_destroy (inside the caller's workspace if one
 *     was given to ea_create_ex).
 *   - Every call except ea_create* returns 0 (EA_OK) or a negative status.  On error the
 *     simulation state is unchanged, with one exception: a problem larger than one launch can
 *     hold runs as several launches over groups of realization words, and if a LATER group's
 *     launch fails (a CUDA error) the earlier groups have already advanced.  The handle then
 *     refuses ea_sweep / ea_measure (EA_ERR_CUDA) until ea_set_state restores a state.
 *     ea_last_error() gives a message.
 *   - Work is enqueued on the handle's CUDA stream.  ea_sweep returns after enqueueing
 *     (asynchronous); every call that fills a host buffer synchronizes the stream first.
 *   - One handle is not thread-safe; different handles are independent.
 *   - There is no CPU fallback: without a CUDA device ea_create* fails (NULL).
 */
#ifndef EA_B200_H
#define EA_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ea_handle ea_handle;

enum {
    EA_OK = 0,
    EA_ERR_INVALID_ARG = -1,
    EA_ERR_ALLOC = -2,
    EA_ERR_CUDA = -3,
    EA_ERR_RANGE = -4,
    EA_ERR_UNSUPPORTED = -5
};

/* Which sweep implementation ea_sweep uses (ea_set_kernel).  AUTO picks the fastest one
 * that supports the lattice; all produce identical results. */
enum {
    EA_KERNEL_AUTO = 0,
    EA_KERNEL_GENERIC = 1,   /* any even L, global memory: one cooperative launch per call when
                                the work fits one wave, else one launch per half-sweep       */
    EA_KERNEL_RESIDENT = 2,  /* every even L <= 12 and L = 16: lattices resident in shared memory,
                                one launch for all sweeps of the call, PT inside a thread-block
                                cluster (L = 8, 16: quad vectors; other L: run-time geometry)   */
    EA_KERNEL_TILED = 3,     /* L = 16, 32, 64: z-slab tiles, one launch per half-sweep, lattice
                                read in place from global memory (L1/L2)                     */
    EA_KERNEL_STREAM = 4,    /* L = 32, 64: one persistent cooperative launch for all sweeps; z-slab
                                tiles streamed through shared memory by TMA bulk copies, two
                                grid-wide barriers per sweep, PT decided redundantly per block */
    EA_KERNEL_REPLICA = 5,   /* the one kernel of EA_LAYOUT_REPLICA_BITS (ea_set_layout): reported by
                                ea_get_kernel, not selectable                                  */
    EA_KERNEL_GENERIC_STEPWISE = 6   /* the generic kernels with one launch per half-sweep / energy /
                                swap round: what EA_KERNEL_GENERIC falls back to when the
                                cooperative launch is refused or the work exceeds one wave     */
};

/* Multispin coding (ea_set_layout).  Two workloads with the same model, tables, initial state and
 * parallel tempering, different random-number conventions (DESIGN.md section 2 and R24):
 *   REALIZATION_BITS  bit b of word w = disorder realization 32 w + b; one random number per
 *                     (site, word, slot) shared by the word's 32 realizations (the default, and
 *                     the layout of BASELINE.json's configs);
 *   REPLICA_BITS      the paper's own coding: a word = the temperature
 *                     replicas of ONE realization at one site, one random number per
 *                     (site, realization, slot), one thread block per realization. */
enum {
    EA_LAYOUT_REALIZATION_BITS = 0,
    EA_LAYOUT_REPLICA_BITS = 1
};

/*
 * Problem statement: periodic L^3 cubic lattice (L even, >= 2), n_realizations
 * disorder realizations, n_temps temperature replicas of each, betas[n_temps] = inverse
 * temperatures, finite, >= 0, monotone (either direction).  seed = Philox4x32-10 key.
 * Couplings and spins are initialised from the seed, the temperature
 * permutation is the identity, the sweep counter is 0.  Limits: n_temps <= 64
 * (EA_ERR_UNSUPPORTED above).  Returns NULL on failure (see ea_last_error(NULL)).
 */
ea_handle *ea_create(int L, int n_temps, int n_realizations, const double *betas, uint64_t seed);

/* Bytes of device workspace ea_create_ex needs for this shape (0 if the shape is invalid). */
size_t ea_workspace_bytes(int L, int n_temps, int n_realizations);

/*
 * As ea_create, with: dev_workspace = caller-owned device memory of at least
 * ea_workspace_bytes() bytes, 256-byte aligned (NULL: the library allocates);
 * cuda_stream = a cudaStream_t (NULL: the legacy default stream);
 * first_realization = global index of realization 0, a multiple of 32: a handle created with
 * first_realization = 32*w0 reproduces words w0.. of a larger problem bit for bit
 * (sharding by realization word).
 */
ea_handle *ea_create_ex(int L, int n_temps, int n_realizations, const double *betas, uint64_t seed,
                        void *dev_workspace, size_t workspace_bytes, void *cuda_stream,
                        int first_realization);

void ea_destroy(ea_handle *h);

/* J[r][d][site] in {+1,-1}: d = 0,1,2 is the +x,+y,+z bond of that site,
 * site = x + L*(y + L*z) (Eq. 1).  Any other value: EA_ERR_INVALID_ARG.
 * Energies are recomputed. */
int ea_set_couplings(ea_handle *h, const int8_t *J /* [R][3][N] */);

/* s[r][slot][site] in {+1,-1}, by storage slot.  Energies are recomputed. */
int ea_set_spins(ea_handle *h, const int8_t *s /* [R][n_temps][N] */);

/* Replace the threshold tables (north_star: "handed to both paths as input data").
 * acc[t][c] = floor(2^32 min(1, exp(-beta_t (4c-12)))), c = 0..6;
 * swp[t][m + 3N/2] = floor(2^32 min(1, exp((beta_t - beta_{t+1}) 4m))), m in [-3N/2, 3N/2].
 * Values in [0, 2^32].  Each column of acc must be monotone in the same direction as betas
 * and each row of swp monotone in m, else EA_ERR_INVALID_ARG. */
int ea_set_tables(ea_handle *h, const uint64_t *acc /* [n_temps][7] */,
                  const uint64_t *swp /* [n_temps-1][3N+1] */);
int ea_get_tables(ea_handle *h, uint64_t *acc, uint64_t *swp);

/*
 * n_sweeps >= 0 full checkerboard sweeps (parity 0 then parity 1); a
 * parallel-tempering round (R4-R6) follows every sweep whose
 * 1-based GLOBAL index is a multiple of swap_interval; swap_interval = 0: no PT.
 * EA_ERR_RANGE if the global sweep counter would pass 2^32 - 1.  Asynchronous.  Launch
 * configurations of all word groups are checked before the first launch.
 */
int ea_sweep(ea_handle *h, int64_t n_sweeps, int swap_interval);

/* Block until everything enqueued on the handle's stream has finished; reports
 * asynchronous CUDA errors. */
int ea_synchronize(ea_handle *h);

/* E[r][t] = H of realization r at temperature index t. */
int ea_energy(ea_handle *h, int32_t *E /* [R][n_temps] */);

/* Q[p][t] = sum_i s_i(ra, t) s_i(rb, t) for pairs[p] = (ra, rb); rb = -1: all-up reference
 * (magnetization).  Bad realization index: EA_ERR_INVALID_ARG. */
int ea_overlap(ea_handle *h, const int32_t *pairs /* [n_pairs][2] */, int n_pairs,
               int32_t *Q /* [n_pairs][n_temps] */);

/* ea_overlap for callers that must not allocate (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): same arguments (host pointers), same results, but the
 * device copies of pairs and Q live in ONE file-scope device array of the library instead of the
 * handle's growing scratch buffer, and the call makes no cudaMalloc / cudaFree / allocating library
 * call.  The array holds EA_OVERLAP_STATIC_MAX_INT32 32-bit words (256 KiB, held by every GPU that
 * loads the library until the process exits); n_pairs * (2 + n_temps) beyond that: EA_ERR_RANGE, and
 * nothing is launched.  Its address is resolved once per device (cudaGetSymbolAddress, with that
 * device current -- the device of the handle must be current, as for every call).  ALL handles and
 * ALL calls on a device share the array and it keeps the last call's contents (nothing in it needs
 * to start at zero: every element read back is written by the call): calls that overlap on the GPU
 * -- two host threads, two streams -- race; a call returns after its stream has drained, so calls
 * made one after the other from one thread are safe.  In the REPLICA_BITS layout the call may first
 * launch the transposition to the exchange format, as ea_overlap does. */
#define EA_OVERLAP_STATIC_MAX_INT32 65536
int ea_overlap_static(ea_handle *h, const int32_t *pairs /* [n_pairs][2] */, int n_pairs,
                      int32_t *Q /* [n_pairs][n_temps] */);

/* s[r][t][site] = +-1 by temperature index. */
int ea_get_spins(ea_handle *h, int8_t *s /* [R][n_temps][N] */);

/* Raw state, for parity tests and checkpoints.  Any pointer may be NULL.
 * spin_words[k][w][p][j]: bit b = spin of realization 32w+b at slot k, parity p, checkerboard
 * index j; temp_of_slot[r][k]; energy_by_slot[r][k]. */
int ea_get_state(ea_handle *h, uint32_t *spin_words /* [n_temps][W][2][N/2] */,
                 uint8_t *temp_of_slot /* [R][n_temps] */, int32_t *energy_by_slot /* [R][n_temps] */,
                 uint64_t *sweeps_done, uint64_t *swap_rounds_done);

/* Resume from a checkpoint taken with ea_get_state ("spin configurations are dumped ...
 * periodically"): packed spins by slot, the temperature permutation and the two
 * counters that address the random draws.  The handle must have been created with the same
 * shape, betas and seed (and given the same couplings / field) as the one that was saved.
 * temp_of_slot[r] must be a permutation of 0..n_temps-1 (EA_ERR_INVALID_ARG), sweeps_done
 * <= 2^32-1 (EA_ERR_RANGE).  Padding bits of the last word are taken as given.  Rank masks and
 * energies are recomputed. */
int ea_set_state(ea_handle *h, const uint32_t *spin_words /* [n_temps][W][2][N/2] */,
                 const uint8_t *temp_of_slot /* [R][n_temps] */, uint64_t sweeps_done,
                 uint64_t swap_rounds_done);

/*
 * ---- Measurement series (the observables of PAPER.md:317-339) ----
 * The paper's spin-glass order parameter is the overlap q between two copies of one disorder
 * realization (Binder ratio of the EA model, Fig. 20); it never prints the
 * definitions, R16/R20 fix them.  All sums are exact integers accumulated on the
 * device; no host round trip between measurements.
 */

/* J[r][d][site] = +-1, the inverse of ea_set_couplings. */
int ea_get_couplings(ea_handle *h, int8_t *J /* [R][3][N] */);

/* Two-copy set-up: realizations R/2 .. R-1 get the couplings of 0 .. R/2-1.  n_realizations must
 * be a multiple of 64 so that the two copies of a realization sit in different words and hence
 * see different random draws (R11); else EA_ERR_INVALID_ARG.  Spins are untouched
 * (the halves were seeded differently); energies are recomputed. */
int ea_pair_couplings(ea_handle *h);

/* Start (or restart) a series: zero accumulators for n_word_pairs pairs of realization words.
 * Pair p = (wa, wb) stands for the 32 realization pairs (32 wa + b, 32 wb + b), b = 0..31;
 * wb = -1: all-up reference (q = magnetization).  Word index outside [0, W): EA_ERR_INVALID_ARG.
 * Allocates device memory of its own (one more copy of the spin store), freed by ea_destroy
 * or the next ea_measure_begin. */
int ea_measure_begin(ea_handle *h, const int32_t *word_pairs /* [n_word_pairs][2] */, int n_word_pairs);

/* n_meas times: ea_sweep(sweeps_between, swap_interval), then one measurement at equal
 * temperature index t: q = sum_i s_i(ra, t) s_i(rb, t) for every realization pair of the series
 * and E = ea_energy's value for every (r, t); adds 1, q, q^2, q^4, E, E^2 to the accumulators,
 * and updates the plane-sum correlations and the round-trip counters (below).
 * Pairs that touch a padding bit (realization index >= R) accumulate nothing.  Asynchronous.
 * EA_ERR_RANGE if the sweep counter would pass 2^32-1 or the number of measurements would pass
 * 2^64 / (9 N^2) (64-bit sums of q^2 and E^2; the q^4 sums are 128-bit). */
int ea_measure(ea_handle *h, int64_t n_meas, int64_t sweeps_between, int swap_interval);

/* Copy the accumulators out (any pointer may be NULL).  q4[..][0] = low, [1] = high 64 bits. */
int ea_get_moments(ea_handle *h, uint64_t *n_meas, int64_t *q1 /* [P][32][n_temps] */,
                   uint64_t *q2 /* [P][32][n_temps] */, uint64_t *q4 /* [P][32][n_temps][2] */,
                   int64_t *e1 /* [R][n_temps] */, uint64_t *e2 /* [R][n_temps] */);

/* Plane-sum correlations of the local overlap q_i = s_i(ra, t) s_i(rb, t), accumulated by every
 * measurement: C[p][b][t][d] = sum over measurements, over the three axes mu and over the planes c
 * of S_mu(c) S_mu((c + d) mod L), S_mu(c) = sum of q_i over the plane (coordinate mu of i) = c
 * (R23).  sum_d C = 3 * (sum of q^2). */
int ea_get_correlation(ea_handle *h, int64_t *C /* [P][32][n_temps][L] */);

/* Second-moment correlation length by temperature index (the quantity of the paper's Fig. 19,
 * PAPER.md:329): chi(k) = sum_d cos(k d) [<C(d)>] / (3 N), xi = sqrt(chi(0)/chi(k_min) - 1) /
 * (2 sin(k_min/2)), k_min = 2 pi / L, [.] = average over the series' valid realization pairs.
 * Host arithmetic in long double from the integer sums.  NaN where nothing was measured,
 * chi(k_min) <= 1e-12 chi(0) or chi(0) < chi(k_min). */
int ea_get_correlation_length(ea_handle *h, double *xi /* [n_temps] */);

/* Round trips in temperature space, the parallel-tempering diagnostic behind "the choice of
 * temperatures is crucial", observed at the measurements of the series: a replica
 * that is at temperature index 0 after having been at index n_temps-1 completes one round trip
 * (R22).  trips[r] = round trips completed by the n_temps replicas of realization r
 * since ea_measure_begin. */
int ea_get_round_trips(ea_handle *h, uint64_t *trips /* [R] */);

/* Binder ratio by temperature index, g[t] = (3 - [<q^4>] / [<q^2>]^2) / 2: <.> = average over the
 * measurements of one realization pair, [.] = average over the series' valid realization pairs
 * (disorder average).  Computed on the host from the integer sums in long double; agrees with
 * the exact rational value to ~1e-18 relative.  NaN where no measurement was taken or [<q^2>] = 0. */
int ea_get_binder(ea_handle *h, double *g /* [n_temps] */);

/*
 * ---- External field ----
 * Constant field h of Eq. 1 ("a constant external field, h, is included in our
 * implementation"), sign as printed: H = -sum J s s + h sum_i s_i.  Flipping s_i costs
 * dE = 4 n_sat - 12 - 2 h s_i, so the acceptance table has the paper's 14 columns (7 local energies
 * x 2 spins).  h is an integer, |h| <= 64 (R21: H stays an exact
 * integer; the swap table is then indexed by (E_a - E_b)/2).  Tables are rebuilt on the host in
 * double from betas, energies are recomputed, the sweep counter is kept.  With 1 <= |h| <= 2 the
 * resident (even L <= 12, L = 16) and streaming (L = 32, 64) kernels run (four threshold columns of the
 * shifted class index); every other case runs on EA_KERNEL_GENERIC.
 * ea_set_kernel of a kernel that cannot run the field -> EA_ERR_UNSUPPORTED; ea_set_tables ->
 * EA_ERR_UNSUPPORTED; ea_get_tables keeps returning the zero-field tables; h = 0 restores the
 * zero-field path.  Not available in EA_LAYOUT_REPLICA_BITS.
 */
int ea_set_field(ea_handle *h, int field);
int ea_get_field(ea_handle *h);
/* accf[t][c][(s+1)/2] = floor(2^32 min(1, exp(-beta_t (4c - 12 - 2 h s)))), c = n_sat, s = +-1;
 * swpf[t][d2 + Mf] = floor(2^32 min(1, exp((beta_t - beta_{t+1}) 2 d2))), |d2| <= Mf = (3+|h|) N.
 * EA_ERR_INVALID_ARG when no field is set. */
int ea_get_field_tables(ea_handle *h, uint64_t *accf /* [n_temps][7][2] */,
                        uint64_t *swpf /* [n_temps-1][2 (3+|h|) N + 1] */);

/* Other bimodal coupling distributions (R25):
 * replace the couplings by +-J bonds with concentration p_plus = P(J = +1), 0 <= p_plus <= 1,
 * drawn independently per bond from the handle's seed (p_plus = 1: ferromagnet, as used for the
 * Ising check of PAPER.md:329).  Spins, permutation and counters are kept, energies recomputed.
 * Any other +-1 disorder can be given explicitly with ea_set_couplings. */
int ea_seed_couplings(ea_handle *h, double p_plus);

/* Switch the multispin coding of the handle (EA_LAYOUT_*).  The physical state (spins, couplings,
 * permutation, energies, counters) is kept: only the random numbers consumed by later sweeps
 * follow the other convention, so ea_set_layout is normally called right after ea_create.
 * Accessors keep their formats (ea_get_state returns words in the REALIZATION_BITS packing).
 * REPLICA_BITS needs L <= 32 (a realization's replicas stay in shared memory), n_temps <= 64,
 * h = 0: otherwise EA_ERR_UNSUPPORTED and nothing changes. */
int ea_set_layout(ea_handle *h, int layout);
int ea_get_layout(ea_handle *h);

/* What an accepted parallel-tempering swap exchanges.  EA_SWAP_PERMUTE (default, north_star): the
 * temperature indices of the two slots; lattices stay ("swap rows, not lattices").
 * EA_SWAP_MOVE: the two lattices (per realization: the masked bits of every word of the two slots)
 * and their energies; slot k keeps temperature index k for every realization, so the 32 realizations
 * of a word are always at the same temperature.  The draws keep their counters (flip: by slot;
 * swap: by temperature pair), which makes MOVE a different, equally valid, Markov chain: its oracle
 * is the oracle's swap mode 1 (R26).  Allowed only while the permutation is the identity
 * (before the first swap round, or after ea_set_state with identity temp_of_slot) and in the
 * REALIZATION_BITS layout: else EA_ERR_UNSUPPORTED and nothing changes.  ea_get_round_trips counts
 * movements of temperature indices and therefore stays at zero in MOVE mode.  The resident kernels
 * exchange inside shared memory (one launch per ea_sweep, as in PERMUTE mode); the other kernels are
 * launched once per swap round, followed by an exchange kernel. */
#define EA_SWAP_PERMUTE 0
#define EA_SWAP_MOVE 1
int ea_set_swap_mode(ea_handle *h, int mode);
int ea_get_swap_mode(ea_handle *h);

/* Select the sweep implementation (EA_KERNEL_*); EA_ERR_UNSUPPORTED if it cannot run this shape. */
int ea_set_kernel(ea_handle *h, int kernel);
/* The implementation ea_sweep would use now (EA_KERNEL_GENERIC/RESIDENT/TILED/STREAM). */
int ea_get_kernel(ea_handle *h);
/* Number of kernels this handle has launched so far. */
int64_t ea_launch_count(ea_handle *h);

/* Measurement helper: issue-rate microbenchmark on the current device.
 * out[0] = LOP3 lane-operations per second (ALU pipe), out[1] = IMAD lane-operations per second
 * (FMA pipe), out[2] = a 1:1 LOP3/IMAD mix, out[3] = number of SMs.  The roofline denominator
 * of the sweep kernel is out[0]. */
int ea_measure_int_peak(void *cuda_stream, double *out /* [4] */);

/* Message for the last failure on h (h = NULL: last ea_create* failure on this thread). */
const char *ea_last_error(const ea_handle *h);

#ifdef __cplusplus
}
#endif
#endif /* EA_B200_H */
