/*
 * potts_oracle.c -- CPU ORACLE for the checkerboard Metropolis sweep of the 2D q-state Potts
 * model (arXiv 1101.0876, Ferrero / De Francesco / Wolovick / Cannas).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares no
 * code, header, table or constant generator with the CUDA path under
 * paper_1101_0876_b200/csrc/, and it is deliberately plain: a scalar loop over the lattice in
 * the paper's order, one statement per rule, so that it can be checked against the paper by
 * eye.  It is never tuned for speed.
 *
 * Rules (R1..R9 are the readings recorded in DESIGN.md section 3 / SURVEY.md section 8(c)):
 *   R1 model        H = -J sum_<ij> delta(s_i,s_j), J = k_B = 1, s in {0..q-1}, L x L periodic
 *                   square lattice, 4 nearest neighbours          (PAPER.md:46 Eq. 1; :94 sec. 3)
 *   R2 order        sweep t = all sites with (i+j) even ("white"), then all with (i+j) odd
 *                   ("black")
 *   R3 randomness   (w0,w1,w2,w3) = Philox4x32-10(counter = (j, i, t, colour), key = seed);
 *                   one independent stream per site                (north_star)
 *   R4 proposal     s' = floor(w0 * q / 2^32), uniform on all q states
 *   R5 energy diff  d = n_old - n_new, n_x = #neighbours equal to x  (Eq. 1)
 *   R6 acceptance   accept iff d <= 0 or w1 < floor(2^32 exp(-d/T))   (Metropolis)
 *   R7 bookkeeping  on accept s <- s', E_inc += d
 *   R8 measures     E = -(number of satisfied bonds), N_k = #{s = k}  (sec. 3.4)
 *   R9 init         ordered: all 0; random: s(i,j) = floor(w0 * q / 2^32) with counter (j,i,0,2)
 *                                                                   (PAPER.md:96 start states)
 *
 * Parity pins (tests/test_oracle_*.py, all -m "not gpu"): Philox known-answer vectors, the
 * threshold table, exact enumeration of the 4x4 lattice (q = 2, 3), Kaufman/Onsager exact
 * Ising energies and specific heat at q = 2, bookkeeping invariants, degenerate temperatures,
 * proposal uniformity, and the SURVEY's independently computed golden trajectories.
 * No function in this file is "parity unpinned".
 *
 * Stream-spec v2 (R3', reading S15; off unless oracle_set_stream(o, 2)): the same-colour
 * sites of a row are numbered k = j >> 1; sites k = 2m and 2m+1 share ONE Philox block, the one R3 gives site 2m
 * (counter (j of site 2m, i, t, colour)); site 2m takes (w0, w1) for (proposal, acceptance), site 2m+1 takes
 * (w2, w3).  Everything else (R1, R2, R4..R9) is unchanged, so even-k sites draw exactly what they draw in v1.
 * Needs L % 4 == 0.
 *
 * Optional row parallelism (-fopenmp, oracle_set_threads): rows of one colour are independent
 * (a colour reads only the other colour; the random words are a pure function of the site), so
 * the threaded loop produces the same bits as the serial one; tests check that.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int32_t L;       /* linear size, even, >= 2 */
    int32_t q;       /* number of states, 2..256 */
    uint64_t seed;   /* Philox key */
    uint64_t t;      /* sweeps done since creation (Philox counter word 2) */
    int64_t E_inc;   /* energy tracked incrementally: E(0) + sum of accepted d (R7) */
    uint8_t *s;      /* spins, row-major s[i*L + j] */
    int threads;     /* 1 = serial */
    int stream;      /* random-stream definition: 1 = one Philox block per site (R3), 2 = per pair of sites (R3') */
} oracle_potts;

/* ---- R3: Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), written out from its definition:
 * ten rounds of
 *     (c0,c1,c2,c3) <- (hi(M1*c2) ^ c1 ^ k0,  lo(M1*c2),  hi(M0*c0) ^ c3 ^ k1,  lo(M0*c0))
 * with the key bumped by the Weyl constants (W0,W1) between rounds. */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)M0 * c0;
        uint64_t p1 = (uint64_t)M1 * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* ---- R6: thr[d] = floor(2^32 * exp(-d/T)) for d = 1..4; thr[0] is unused (d <= 0 accepts). */
void oracle_thresholds(double T, uint32_t thr[5])
{
    thr[0] = 0xFFFFFFFFu;
    for (int d = 1; d <= 4; ++d)
        thr[d] = (uint32_t)floor(ldexp(exp(-(double)d / T), 32));
}

/* ---- R4 */
static uint32_t propose(uint32_t w0, uint32_t q)
{
    return (uint32_t)(((uint64_t)w0 * (uint64_t)q) >> 32);
}

/* ---- R8 (Eq. 1): E = - sum_{i,j} [ delta(s_ij, s_i,j+1) + delta(s_ij, s_i+1,j) ] */
int64_t oracle_energy(const oracle_potts *o)
{
    const int32_t L = o->L;
    int64_t bonds = 0;
    for (int32_t i = 0; i < L; ++i)
        for (int32_t j = 0; j < L; ++j) {
            uint8_t s = o->s[(size_t)i * L + j];
            bonds += (s == o->s[(size_t)i * L + (j + 1) % L]);
            bonds += (s == o->s[(size_t)((i + 1) % L) * L + j]);
        }
    return -bonds;
}

/* ---- R8: N_k */
void oracle_histogram(const oracle_potts *o, int64_t *counts)
{
    for (int32_t k = 0; k < o->q; ++k) counts[k] = 0;
    for (size_t n = 0; n < (size_t)o->L * o->L; ++n) counts[o->s[n]] += 1;
}

oracle_potts *oracle_create(int32_t L, int32_t q, uint64_t seed, int32_t init)
{
    if (L < 2 || (L & 1) || q < 2 || q > 256 || (init != 0 && init != 1)) return NULL;
    oracle_potts *o = (oracle_potts *)calloc(1, sizeof *o);
    if (!o) return NULL;
    o->L = L; o->q = q; o->seed = seed; o->t = 0; o->threads = 1; o->stream = 1;
    o->s = (uint8_t *)calloc((size_t)L * L, 1);
    if (!o->s) { free(o); return NULL; }
    if (init == 1) {                                   /* R9 */
        const uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
        for (int32_t i = 0; i < L; ++i)
            for (int32_t j = 0; j < L; ++j) {
                const uint32_t ctr[4] = { (uint32_t)j, (uint32_t)i, 0u, 2u };
                uint32_t w[4];
                oracle_philox4x32_10(ctr, key, w);
                o->s[(size_t)i * L + j] = (uint8_t)propose(w[0], (uint32_t)q);
            }
    }
    o->E_inc = oracle_energy(o);
    return o;
}

void oracle_destroy(oracle_potts *o)
{
    if (o) { free(o->s); free(o); }
}

void oracle_set_threads(oracle_potts *o, int threads)
{
    o->threads = threads < 1 ? 1 : threads;
}

/* choose the random-stream definition (1 or 2, see the header); returns 1 on a bad argument */
int oracle_set_stream(oracle_potts *o, int stream)
{
    if (!o || (stream != 1 && stream != 2) || (stream == 2 && (o->L & 3))) return 1;
    o->stream = stream;
    return 0;
}

int oracle_get_threads(const oracle_potts *o)
{
#ifdef _OPENMP
    return o->threads;
#else
    (void)o;
    return 1;
#endif
}

/* ---- R2..R7 for one colour of sweep t. Returns the sum of accepted d. */
static int64_t half_sweep(oracle_potts *o, uint32_t colour, const uint32_t thr[5])
{
    const int32_t L = o->L;
    const uint32_t q = (uint32_t)o->q;
    const uint32_t key[2] = { (uint32_t)(o->seed & 0xFFFFFFFFu), (uint32_t)(o->seed >> 32) };
    const uint32_t t32 = (uint32_t)o->t;
    uint8_t *S = o->s;
    int64_t dE = 0;
#ifdef _OPENMP
#pragma omp parallel for reduction(+ : dE) num_threads(o->threads) schedule(static)
#endif
    for (int32_t i = 0; i < L; ++i) {
        for (int32_t j = (int32_t)((i + colour) & 1u); j < L; j += 2) {
            /* R3: the site's own block, words 0 and 1.  R3': the block of the first site of its pair,
             * words 0, 1 for the first site and 2, 3 for the second. */
            const int second = o->stream == 2 && ((j >> 1) & 1);
            const uint32_t ctr[4] = { (uint32_t)(second ? j - 2 : j), (uint32_t)i, t32, colour };
            uint32_t w[4];
            oracle_philox4x32_10(ctr, key, w);
            const uint32_t w_prop = second ? w[2] : w[0], w_acc = second ? w[3] : w[1];
            const uint8_t s_old = S[(size_t)i * L + j];
            const uint8_t s_new = (uint8_t)propose(w_prop, q);          /* R4 */
            const uint8_t nb[4] = {
                S[(size_t)((i + L - 1) % L) * L + j],
                S[(size_t)((i + 1) % L) * L + j],
                S[(size_t)i * L + (j + L - 1) % L],
                S[(size_t)i * L + (j + 1) % L],
            };
            int n_old = 0, n_new = 0;
            for (int k = 0; k < 4; ++k) { n_old += (nb[k] == s_old); n_new += (nb[k] == s_new); }
            const int d = n_old - n_new;                                /* R5 */
            if (d <= 0 || w_acc < thr[d]) {                             /* R6 */
                S[(size_t)i * L + j] = s_new;                           /* R7 */
                dE += d;
            }
        }
    }
    return dE;
}

/* n sweeps at temperature T.  Returns 0, or 1 on bad arguments. */
int oracle_sweep(oracle_potts *o, double T, int64_t nsweeps)
{
    if (!o || !(T > 0.0) || !isfinite(T) || nsweeps < 0) return 1;
    if (o->t + (uint64_t)nsweeps > 0xFFFFFFFFull) return 1;             /* R3: t < 2^32 */
    uint32_t thr[5];
    oracle_thresholds(T, thr);
    for (int64_t n = 0; n < nsweeps; ++n) {
        o->E_inc += half_sweep(o, 0u, thr);                             /* R2: white first */
        o->E_inc += half_sweep(o, 1u, thr);
        o->t += 1;
    }
    return 0;
}

/* n sweeps, sampling (E, N_0..N_{q-1}) after every `every`-th sweep of this call (R8).
 * E_series has n/every entries, hist_series n/every rows of q (may be NULL).
 * The recorded E is the recomputed Eq. 1 energy; returns 2 if it ever differs from E_inc
 * or a histogram does not sum to L^2 (bookkeeping invariants), else 0. */
int oracle_sweep_measured(oracle_potts *o, double T, int64_t nsweeps, int64_t every,
                          int64_t *E_series, int64_t *hist_series)
{
    if (!o || every < 1 || nsweeps < 0 || nsweeps % every != 0) return 1;
    int bad = 0;
    for (int64_t k = 0; k < nsweeps / every; ++k) {
        int rc = oracle_sweep(o, T, every);
        if (rc) return rc;
        const int64_t E = oracle_energy(o);
        if (E != o->E_inc) bad = 2;
        if (E_series) E_series[k] = E;
        if (hist_series) {
            oracle_histogram(o, hist_series + k * o->q);
            int64_t tot = 0;
            for (int32_t b = 0; b < o->q; ++b) tot += hist_series[k * o->q + b];
            if (tot != (int64_t)o->L * o->L) bad = 2;
        }
    }
    return bad;
}

/* accessors for the ctypes wrapper */
uint8_t *oracle_spins(oracle_potts *o) { return o->s; }
uint64_t oracle_sweep_count(const oracle_potts *o) { return o->t; }
int64_t oracle_energy_incremental(const oracle_potts *o) { return o->E_inc; }

/* restore a state (spins + sweep counter): the counter-based RNG has no other state */
int oracle_set_state(oracle_potts *o, const uint8_t *spins, uint64_t t)
{
    if (!o || !spins) return 1;
    for (size_t n = 0; n < (size_t)o->L * o->L; ++n)
        if (spins[n] >= o->q) return 1;
    memcpy(o->s, spins, (size_t)o->L * o->L);
    o->t = t;
    o->E_inc = oracle_energy(o);
    return 0;
}

/* One site of one half-sweep computed on its own from an explicit neighbourhood (used by the
 * full-size sampled parity checks): returns the new spin.  Same rules, same order. */
uint8_t oracle_update_site_s(uint32_t i, uint32_t j, uint32_t t32, uint32_t colour, uint64_t seed,
                             uint32_t q, double T, uint8_t s_old, const uint8_t nb[4], int stream)
{
    const uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
    const int second = stream == 2 && ((j >> 1) & 1u);
    const uint32_t ctr[4] = { second ? j - 2u : j, i, t32, colour };
    uint32_t w[4], thr[5];
    oracle_philox4x32_10(ctr, key, w);
    oracle_thresholds(T, thr);
    const uint8_t s_new = (uint8_t)propose(second ? w[2] : w[0], q);
    int n_old = 0, n_new = 0;
    for (int k = 0; k < 4; ++k) { n_old += (nb[k] == s_old); n_new += (nb[k] == s_new); }
    const int d = n_old - n_new;
    return (d <= 0 || (second ? w[3] : w[1]) < thr[d]) ? s_new : s_old;
}

uint8_t oracle_update_site(uint32_t i, uint32_t j, uint32_t t32, uint32_t colour, uint64_t seed,
                           uint32_t q, double T, uint8_t s_old, const uint8_t nb[4])
{
    return oracle_update_site_s(i, j, t32, colour, seed, q, T, s_old, nb, 1);
}
