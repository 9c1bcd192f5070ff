/* ORACLE (test infrastructure).  Counter-based RNG and track identity.
 * Paper: PAPER.md:189 uses XORWOW; BASELINE.json north_star replaces it with a
 * "counter-based Philox RNG keyed by track id and step" -> DESIGN.md R5/R6.
 * Algorithm: Philox4x32-10 as published by Salmon, Moraes, Dror, Shaw (SC'11),
 * restated here from the definition: 10 rounds of two 32x32->64 multiplies with
 * a Weyl key schedule.
 */
#include "emo.h"

void emo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)M0 * c0;
        uint64_t p1 = (uint64_t)M1 * c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* 52-bit uniform strictly inside (0,1): (k + 1/2) * 2^-52, k in [0, 2^52). */
double emo_u01(uint32_t wa, uint32_t wb) {
    uint64_t k = (((uint64_t)wa << 32) | (uint64_t)wb) >> 12;
    return ((double)k + 0.5) * (1.0 / 4503599627370496.0);
}

/* draw number n of (prim, tid, step): block n/2, words 2(n%2), 2(n%2)+1.
 * key = (seed32, prim); counter = (block, step, tid_lo, tid_hi). */
double emo_draw(uint64_t seed, uint32_t prim, uint64_t tid, uint32_t step, uint32_t n) {
    uint32_t ctr[4] = { n >> 1, step, (uint32_t)tid, (uint32_t)(tid >> 32) };
    uint32_t key[2] = { (uint32_t)seed, prim };
    uint32_t o[4];
    emo_philox4x32_10(ctr, key, o);
    uint32_t h = 2u * (n & 1u);
    return emo_u01(o[h], o[h + 1]);
}

/* child number `ordinal` created by (prim, tid) at `step`:
 * first 64 bits of Philox(counter = (0xFFFFFFFF - ordinal, step, tid_lo, tid_hi)). */
uint64_t emo_child_tid(uint64_t seed, uint32_t prim, uint64_t tid, uint32_t step, uint32_t ordinal) {
    uint32_t ctr[4] = { 0xFFFFFFFFu - ordinal, step, (uint32_t)tid, (uint32_t)(tid >> 32) };
    uint32_t key[2] = { (uint32_t)seed, prim };
    uint32_t o[4];
    emo_philox4x32_10(ctr, key, o);
    return ((uint64_t)o[0] << 32) | (uint64_t)o[1];
}

double emo_next(emo_rng *r) {
    double v = emo_draw(r->seed, r->prim, r->tid, r->step, r->n);
    r->n += 1;
    return v;
}
