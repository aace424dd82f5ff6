/*
 * potts3d_oracle.c -- CPU ORACLE for the 3D generalisation of the checkerboard Metropolis sweep
 * (arXiv 1101.0876 sec. 7: "For the generalization to the 3D case, the checkerboard scheme
 * defining two independent sub-networks persists").
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT (see potts_oracle.c: same rules of use).  It shares no code
 * with paper_1101_0876_b200/csrc/.  Inside oracle/ it reuses oracle_philox4x32_10 of potts_oracle.c (the
 * routine pinned by the known-answer vectors) and nothing else.
 *
 * Rules = R1..R9 of potts_oracle.c with the lattice made cubic (reading S16):
 *   R1' model       s in {0..q-1} on an L x L x L periodic simple-cubic lattice, 6 nearest neighbours,
 *                   E = - sum_{x,y,z} [ delta(s, s_{x+1}) + delta(s, s_{y+1}) + delta(s, s_{z+1}) ]   (Eq. 1)
 *   R2' order       sweep t = all sites with (x+y+z) even, then all with (x+y+z) odd
 *   R3' randomness  Philox4x32-10(counter = (x, y, t, colour + 4 z), key = seed): the 2D counter (j, i, t, colour)
 *                   with the plane index z in the bits of word 3 above the colour / domain bits
 *   R4  proposal    s' = floor(w0 q / 2^32)
 *   R5' energy diff d = n_old - n_new over the 6 neighbours, d in -6..6
 *   R6' acceptance  accept iff d <= 0 or w1 < floor(2^32 exp(-d/T)), d = 1..6
 *   R7  bookkeeping on accept s <- s', E_inc += d
 *   R9' init        ordered: all 0; random: floor(w0 q / 2^32) with counter (x, y, 0, 2 + 4 z)
 * L even (the two sub-networks exist only then), L < 2^30.  Spins are stored s[(z L + y) L + x].
 *
 * Parity pins (tests/test_oracle_3d.py, -m "not gpu"): exact enumeration of the 2 x 2 x 2 lattice (q = 2, 3),
 * the single-bond high-temperature energy at L = 8, the degenerate temperatures, bookkeeping invariants against
 * an energy recount written with numpy rolls in the test, the counter layout against the KAT-pinned Philox.
 * Plane parallelism (oracle3_set_threads): planes of one colour are independent, same bits as serial.
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
} oracle_potts3;

/* R6': thr[d], d = 1..6 */
void oracle3_thresholds(double T, uint32_t thr[7])
{
    thr[0] = 0xFFFFFFFFu;
    for (int d = 1; d <= 6; ++d)
        thr[d] = (uint32_t)floor(ldexp(exp(-(double)d / T), 32));
}

static size_t at(const oracle_potts3 *o, int32_t x, int32_t y, int32_t z)
{
    const int32_t L = o->L;
    return ((size_t)((z + L) % L) * L + (size_t)((y + L) % L)) * L + (size_t)((x + L) % L);
}

/* R1' */
int64_t oracle3_energy(const oracle_potts3 *o)
{
    const int32_t L = o->L;
    int64_t bonds = 0;
    for (int32_t z = 0; z < L; ++z)
        for (int32_t y = 0; y < L; ++y)
            for (int32_t x = 0; x < L; ++x) {
                const uint8_t s = o->s[at(o, x, y, z)];
                bonds += (s == o->s[at(o, x + 1, y, z)]);
                bonds += (s == o->s[at(o, x, y + 1, z)]);
                bonds += (s == o->s[at(o, x, y, z + 1)]);
            }
    return -bonds;
}

void oracle3_histogram(const oracle_potts3 *o, int64_t *counts)
{
    for (int32_t k = 0; k < o->q; ++k) counts[k] = 0;
    for (size_t n = 0; n < (size_t)o->L * o->L * o->L; ++n) counts[o->s[n]] += 1;
}

oracle_potts3 *oracle3_create(int32_t L, int32_t q, uint64_t seed, int32_t init)
{
    if (L < 2 || (L & 1) || q < 2 || q > 256 || (init != 0 && init != 1)) return NULL;
    oracle_potts3 *o = (oracle_potts3 *)calloc(1, sizeof *o);
    if (!o) return NULL;
    o->L = L; o->q = q; o->seed = seed; o->t = 0; o->threads = 1;
    o->s = (uint8_t *)calloc((size_t)L * L * L, 1);
    if (!o->s) { free(o); return NULL; }
    if (init == 1) {   /* R9' */
        const uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32)};
        for (int32_t z = 0; z < L; ++z)
            for (int32_t y = 0; y < L; ++y)
                for (int32_t x = 0; x < L; ++x) {
                    const uint32_t ctr[4] = {(uint32_t)x, (uint32_t)y, 0u, 2u + 4u * (uint32_t)z};
                    uint32_t w[4];
                    oracle_philox4x32_10(ctr, key, w);
                    o->s[at(o, x, y, z)] = (uint8_t)(((uint64_t)w[0] * (uint64_t)q) >> 32);
                }
    }
    o->E_inc = oracle3_energy(o);
    return o;
}

void oracle3_destroy(oracle_potts3 *o) { if (o) { free(o->s); free(o); } }
void oracle3_set_threads(oracle_potts3 *o, int n) { o->threads = n < 1 ? 1 : n; }
uint8_t *oracle3_spins(oracle_potts3 *o) { return o->s; }
uint64_t oracle3_sweep_count(const oracle_potts3 *o) { return o->t; }
int64_t oracle3_energy_incremental(const oracle_potts3 *o) { return o->E_inc; }

/* R3'-R7 for one site; returns the accepted d (0 if rejected) and stores the new spin */
static int update_site3(oracle_potts3 *o, int32_t x, int32_t y, int32_t z, uint32_t t, uint32_t colour, const uint32_t thr[7])
{
    const uint32_t key[2] = {(uint32_t)(o->seed & 0xFFFFFFFFu), (uint32_t)(o->seed >> 32)};
    const uint32_t ctr[4] = {(uint32_t)x, (uint32_t)y, t, colour + 4u * (uint32_t)z};
    uint32_t w[4];
    oracle_philox4x32_10(ctr, key, w);
    const uint8_t s_old = o->s[at(o, x, y, z)];
    const uint8_t s_new = (uint8_t)(((uint64_t)w[0] * (uint64_t)o->q) >> 32);             /* R4 */
    const uint8_t nb[6] = {o->s[at(o, x - 1, y, z)], o->s[at(o, x + 1, y, z)], o->s[at(o, x, y - 1, z)],
                           o->s[at(o, x, y + 1, z)], o->s[at(o, x, y, z - 1)], o->s[at(o, x, y, z + 1)]};
    int n_old = 0, n_new = 0;
    for (int k = 0; k < 6; ++k) { n_old += (nb[k] == s_old); n_new += (nb[k] == s_new); }
    const int d = n_old - n_new;                                                          /* R5' */
    if (d <= 0 || w[1] < thr[d]) {                                                        /* R6' */
        o->s[at(o, x, y, z)] = s_new;                                                     /* R7 */
        return d;
    }
    return 0;
}

int oracle3_sweep(oracle_potts3 *o, double T, int64_t nsweeps)
{
    if (!(T > 0.0) || nsweeps < 0 || o->t + (uint64_t)nsweeps > 0xFFFFFFFFull) return 1;
    uint32_t thr[7];
    oracle3_thresholds(T, thr);
    const int32_t L = o->L;
    for (int64_t n = 0; n < nsweeps; ++n) {
        for (uint32_t colour = 0; colour < 2; ++colour) {                                 /* R2' */
            int64_t dsum = 0;
#ifdef _OPENMP
#pragma omp parallel for reduction(+ : dsum) num_threads(o->threads) schedule(static)
#endif
            for (int32_t z = 0; z < L; ++z)
                for (int32_t y = 0; y < L; ++y)
                    for (int32_t x = 0; x < L; ++x)
                        if ((uint32_t)((x + y + z) & 1) == colour) dsum += update_site3(o, x, y, z, (uint32_t)o->t, colour, thr);
            o->E_inc += dsum;
        }
        o->t += 1;
    }
    return 0;
}

/* series sample k (k = 1..nsweeps/every) after sweep k*every of the call (R8) */
int oracle3_sweep_measured(oracle_potts3 *o, double T, int64_t nsweeps, int64_t every, int64_t *E_series, int64_t *hist_series)
{
    if (every < 1 || nsweeps % every) return 1;
    for (int64_t k = 0; k < nsweeps / every; ++k) {
        if (oracle3_sweep(o, T, every)) return 1;
        if (E_series) E_series[k] = oracle3_energy(o);
        if (hist_series) oracle3_histogram(o, hist_series + k * o->q);
    }
    return 0;
}

int oracle3_set_state(oracle_potts3 *o, const uint8_t *spins, uint64_t t)
{
    const size_t n = (size_t)o->L * o->L * o->L;
    for (size_t k = 0; k < n; ++k)
        if (spins[k] >= o->q) return 1;
    memcpy(o->s, spins, n);
    o->t = t;
    o->E_inc = oracle3_energy(o);
    return 0;
}
