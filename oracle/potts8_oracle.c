/*
 * potts8_oracle.c -- CPU ORACLE for the 2D generalisation with first AND second neighbour interactions
 * (arXiv 1101.0876 sec. 7: "For the 2D case with first and second neighbors interactions, there are
 * nine independent sub-networks to update instead of two").
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT (see potts_oracle.c: same rules of use).  It shares no code with
 * paper_1101_0876_b200/csrc/.  Inside oracle/ it reuses oracle_philox4x32_10 of potts_oracle.c (the routine pinned
 * by the known-answer vectors) and nothing else.
 *
 * Rules = R1..R9 of potts_oracle.c with the neighbourhood enlarged (reading S17):
 *   R1" model       s in {0..q-1} on an L x L periodic square lattice; every site interacts with its 4 first
 *                   neighbours (i+-1, j), (i, j+-1) and its 4 second (diagonal) neighbours (i+-1, j+-1), all with
 *                   the same coupling J = 1:
 *                   E = - sum_{i,j} [ d(s, s_{i,j+1}) + d(s, s_{i+1,j}) + d(s, s_{i+1,j+1}) + d(s, s_{i+1,j-1}) ]
 *   R2" order       sweep t = the nine sub-networks c = 3 (i mod 3) + (j mod 3), c = 0, 1, ..., 8 in this order; two
 *                   sites of one sub-network differ by a multiple of 3 in both coordinates, so they never interact
 *   R3" randomness  Philox4x32-10(counter = (j, i, t, 16 + c), key = seed)
 *   R4  proposal    s' = floor(w0 q / 2^32)
 *   R5" energy diff d = n_old - n_new over the 8 neighbours, d in -8..8
 *   R6" acceptance  accept iff d <= 0 or w1 < floor(2^32 exp(-d/T)), d = 1..8
 *   R7  bookkeeping on accept s <- s', E_inc += d
 *   R9  init        as in potts_oracle.c: ordered all 0; random floor(w0 q / 2^32) with counter (j, i, 0, 2)
 * L a multiple of 3, L >= 3 (at L = 3 every site neighbours the 8 others once: the complete graph on 9 sites).
 *
 * Parity pins (tests/test_oracle_nnn.py, -m "not gpu"): exact enumeration of the 3 x 3 lattice (q = 2, 3), the
 * single-bond high-temperature energy, invariants against a recount written with numpy rolls in the test, the
 * degenerate temperatures, a sweep rebuilt site by site from the KAT-pinned Philox words.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);   /* potts_oracle.c */

typedef struct {
    int32_t L, q;
    uint64_t seed, t;
    int64_t E_inc;
    uint8_t *s;
    int threads;
} oracle_potts8;

void oracle8_thresholds(double T, uint32_t thr[9])
{
    thr[0] = 0xFFFFFFFFu;
    for (int d = 1; d <= 8; ++d)
        thr[d] = (uint32_t)floor(ldexp(exp(-(double)d / T), 32));
}

static size_t at8(const oracle_potts8 *o, int32_t i, int32_t j)
{
    const int32_t L = o->L;
    return (size_t)((i + L) % L) * L + (size_t)((j + L) % L);
}

/* R1" */
int64_t oracle8_energy(const oracle_potts8 *o)
{
    const int32_t L = o->L;
    int64_t bonds = 0;
    for (int32_t i = 0; i < L; ++i)
        for (int32_t j = 0; j < L; ++j) {
            const uint8_t s = o->s[at8(o, i, j)];
            bonds += (s == o->s[at8(o, i, j + 1)]);
            bonds += (s == o->s[at8(o, i + 1, j)]);
            bonds += (s == o->s[at8(o, i + 1, j + 1)]);
            bonds += (s == o->s[at8(o, i + 1, j - 1)]);
        }
    return -bonds;
}

void oracle8_histogram(const oracle_potts8 *o, int64_t *counts)
{
    for (int32_t k = 0; k < o->q; ++k) counts[k] = 0;
    for (size_t n = 0; n < (size_t)o->L * o->L; ++n) counts[o->s[n]] += 1;
}

oracle_potts8 *oracle8_create(int32_t L, int32_t q, uint64_t seed, int32_t init)
{
    if (L < 3 || (L % 3) || q < 2 || q > 256 || (init != 0 && init != 1)) return NULL;
    oracle_potts8 *o = (oracle_potts8 *)calloc(1, sizeof *o);
    if (!o) return NULL;
    o->L = L; o->q = q; o->seed = seed; o->t = 0; o->threads = 1;
    o->s = (uint8_t *)calloc((size_t)L * L, 1);
    if (!o->s) { free(o); return NULL; }
    if (init == 1) {   /* R9 */
        const uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32)};
        for (int32_t i = 0; i < L; ++i)
            for (int32_t j = 0; j < L; ++j) {
                const uint32_t ctr[4] = {(uint32_t)j, (uint32_t)i, 0u, 2u};
                uint32_t w[4];
                oracle_philox4x32_10(ctr, key, w);
                o->s[at8(o, i, j)] = (uint8_t)(((uint64_t)w[0] * (uint64_t)q) >> 32);
            }
    }
    o->E_inc = oracle8_energy(o);
    return o;
}

void oracle8_destroy(oracle_potts8 *o) { if (o) { free(o->s); free(o); } }
void oracle8_set_threads(oracle_potts8 *o, int n) { o->threads = n < 1 ? 1 : n; }
uint8_t *oracle8_spins(oracle_potts8 *o) { return o->s; }
uint64_t oracle8_sweep_count(const oracle_potts8 *o) { return o->t; }
int64_t oracle8_energy_incremental(const oracle_potts8 *o) { return o->E_inc; }

/* R3"-R7 for one site; returns the accepted d (0 if rejected) */
static int update_site8(oracle_potts8 *o, int32_t i, int32_t j, uint32_t t, uint32_t c, const uint32_t thr[9])
{
    const uint32_t key[2] = {(uint32_t)(o->seed & 0xFFFFFFFFu), (uint32_t)(o->seed >> 32)};
    const uint32_t ctr[4] = {(uint32_t)j, (uint32_t)i, t, 16u + c};
    uint32_t w[4];
    oracle_philox4x32_10(ctr, key, w);
    const uint8_t s_old = o->s[at8(o, i, j)];
    const uint8_t s_new = (uint8_t)(((uint64_t)w[0] * (uint64_t)o->q) >> 32);             /* R4 */
    int n_old = 0, n_new = 0;
    for (int di = -1; di <= 1; ++di)
        for (int dj = -1; dj <= 1; ++dj) {
            if (di == 0 && dj == 0) continue;
            const uint8_t nb = o->s[at8(o, i + di, j + dj)];
            n_old += (nb == s_old);
            n_new += (nb == s_new);
        }
    const int d = n_old - n_new;                                                          /* R5" */
    if (d <= 0 || w[1] < thr[d]) {                                                        /* R6" */
        o->s[at8(o, i, j)] = s_new;                                                       /* R7 */
        return d;
    }
    return 0;
}

int oracle8_sweep(oracle_potts8 *o, double T, int64_t nsweeps)
{
    if (!(T > 0.0) || nsweeps < 0 || o->t + (uint64_t)nsweeps > 0xFFFFFFFFull) return 1;
    uint32_t thr[9];
    oracle8_thresholds(T, thr);
    const int32_t L = o->L;
    for (int64_t n = 0; n < nsweeps; ++n) {
        for (uint32_t c = 0; c < 9; ++c) {                                                /* R2" */
            const int32_t a = (int32_t)(c / 3), b = (int32_t)(c % 3);
            int64_t dsum = 0;
#ifdef _OPENMP
#pragma omp parallel for reduction(+ : dsum) num_threads(o->threads) schedule(static)
#endif
            for (int32_t i = a; i < L; i += 3)
                for (int32_t j = b; j < L; j += 3) dsum += update_site8(o, i, j, (uint32_t)o->t, c, thr);
            o->E_inc += dsum;
        }
        o->t += 1;
    }
    return 0;
}

int oracle8_sweep_measured(oracle_potts8 *o, double T, int64_t nsweeps, int64_t every, int64_t *E_series, int64_t *hist_series)
{
    if (every < 1 || nsweeps % every) return 1;
    for (int64_t k = 0; k < nsweeps / every; ++k) {
        if (oracle8_sweep(o, T, every)) return 1;
        if (E_series) E_series[k] = oracle8_energy(o);
        if (hist_series) oracle8_histogram(o, hist_series + k * o->q);
    }
    return 0;
}

int oracle8_set_state(oracle_potts8 *o, const uint8_t *spins, uint64_t t)
{
    const size_t n = (size_t)o->L * o->L;
    for (size_t k = 0; k < n; ++k)
        if (spins[k] >= o->q) return 1;
    memcpy(o->s, spins, n);
    o->t = t;
    o->E_inc = oracle8_energy(o);
    return 0;
}
