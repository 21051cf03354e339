/*
 * gmgq.c -- oracle for the torus-ensemble generators GM19, GM29, GM31, GM55, GM61, GQ58.1,
 * GQ58.3, GQ58.4 (TEST INFRASTRUCTURE ONLY, see oracle.h).
 *
 * PAPER.md:281-284 (section 5.1, eq. 1):
 *     x_i^(n) = k x_i^(n-1) - q x_i^(n-2)  (mod g),   i = 0, 1, ..., s-1.
 * Parameters (k, q, g, v): Table 2, PAPER.md:232-244:
 *     GM19 (15, 28, 2^19-1, 1)   GM29 (4, 2, 2^29-3, 1)      GM31 (11, 14, 2^31-1, 1)
 *     GM55 (256, 176, 16(2^51-129), 4)                        GM61 (24, 74, 2^61-1, 1)
 *     GQ58.1/.3/.4 (8, 48, 2^29(2^29-3), v = 1/3/4).
 * Jump-ahead: any exact method reaching x^(n); here the n-th power of the companion matrix
 * [[k,-q],[1,0]] mod g.  The paper's own relations (eqs. 2-4) are used as
 * independent pins in tests/test_oracle_gmgq.py.
 *
 * Readings (the paper defers these to its refs [1],[5],[6],[8]):
 *  G1  ensemble size s = "threads per array section" of Table 5:
 *      32 (GM19, GM29, GM31, GM61, GQ58.1), 8 (GM55, GQ58.4), 12 (GQ58.3).
 *  G2  output: after the step, point i contributes the digit d_i = floor(2^v x_i / g) and the
 *      word is sum_i d_i 2^(v i) (point 0 least significant).  GQ58.3 has 12*3 = 36 > 32 bits:
 *      points 0..9 give floor(8x/g) at bits 3i..3i+2, points 10 and 11 give floor(2x/g) at
 *      bits 30 and 31.
 *  G3  seeding: base orbit w(0) = 0, w(1) = seed mod g (must be non-zero),
 *      w(n+1) = k w(n) - q w(n-1) mod g.  At position P point i holds
 *      (x^(n-1), x^(n)) = (w(P + (i+1) D), w(P + (i+1) D + 1)),  D = 2^d,
 *      d = 32 (GM19), 52 (GM29), 56 (GM31), 98 (GM55), 116 (GM61), 52 (GQ58.1),
 *      54 (GQ58.3), 54 (GQ58.4); (s+1) D < period for every generator (Table 2).
 * PRAND's real packing and seeding are not in the paper: parity with the original binary is
 * unpinned; oracle and CUDA library share this written definition only.
 */
#include "oracle.h"
#include <string.h>

typedef unsigned __int128 u128;

static const o_gm_params PARAMS[O_NGEN] = {
    [O_GM19]   = {15, 28, (1ull << 19) - 1, 1, 32, 32},
    [O_GM29]   = {4, 2, (1ull << 29) - 3, 1, 32, 52},
    [O_GM31]   = {11, 14, (1ull << 31) - 1, 1, 32, 56},
    [O_GM55]   = {256, 176, 16ull * ((1ull << 51) - 129), 4, 8, 98},
    [O_GM61]   = {24, 74, (1ull << 61) - 1, 1, 32, 116},
    [O_GQ58_1] = {8, 48, (1ull << 29) * ((1ull << 29) - 3), 1, 32, 52},
    [O_GQ58_3] = {8, 48, (1ull << 29) * ((1ull << 29) - 3), 3, 12, 54},
    [O_GQ58_4] = {8, 48, (1ull << 29) * ((1ull << 29) - 3), 4, 8, 54},
};

int o_gm_params_get(int gen, o_gm_params *p)
{
    if (gen < O_GM19 || gen > O_GQ58_4) return -1;
    *p = PARAMS[gen];
    return 0;
}

/* eq. 1 for one point: (xP, xN) <- (xN, k xN - q xP mod g) */
static void point_step(const o_gm_params *p, uint64_t *xP, uint64_t *xN)
{
    u128 pos = (u128)p->k * *xN + (u128)p->q * (p->g - *xP);   /* -q xP == q (g - xP) mod g */
    uint64_t nw = (uint64_t)(pos % p->g);
    *xP = *xN;
    *xN = nw;
}

/* 2x2 matrices mod g, row-major; the companion matrix maps (x^(n), x^(n-1)) to (x^(n+1), x^(n)) */
static void mm2(uint64_t o[4], const uint64_t a[4], const uint64_t b[4], uint64_t g)
{
    uint64_t t[4];
    for (int i = 0; i < 2; i++)
        for (int j = 0; j < 2; j++) {
            u128 acc = (u128)a[2 * i] * b[j] % g + (u128)a[2 * i + 1] * b[2 + j] % g;
            t[2 * i + j] = (uint64_t)(acc % g);
        }
    memcpy(o, t, sizeof t);
}

static void companion_pow(const o_gm_params *p, const uint8_t *exp, size_t nbytes, uint64_t acc[4])
{
    const uint64_t base[4] = {p->k % p->g, p->g - p->q % p->g, 1, 0};
    acc[0] = 1; acc[1] = 0; acc[2] = 0; acc[3] = 1;
    for (size_t i = nbytes; i-- > 0;)
        for (int b = 7; b >= 0; b--) {
            mm2(acc, acc, acc, p->g);
            if ((exp[i] >> b) & 1u) mm2(acc, base, acc, p->g);
        }
}

static void point_apply(const uint64_t m[4], uint64_t g, uint64_t *xP, uint64_t *xN)
{
    u128 n = (u128)m[0] * *xN % g + (u128)m[1] * *xP % g;
    u128 o = (u128)m[2] * *xN % g + (u128)m[3] * *xP % g;
    *xN = (uint64_t)(n % g);
    *xP = (uint64_t)(o % g);
}

void o_gm_orbit(int gen, uint64_t seed, const uint8_t *exp, size_t nbytes,
                uint64_t *w_n, uint64_t *w_n1)
{
    const o_gm_params *p = &PARAMS[gen];
    uint64_t m[4];
    uint64_t xP = 0, xN = seed % p->g;            /* (w(0), w(1)) */
    companion_pow(p, exp, nbytes, m);
    point_apply(m, p->g, &xP, &xN);
    *w_n = xP; *w_n1 = xN;
}

int o_gm_seed(int gen, o_gm *st, uint64_t seed)
{
    o_gm_params p;
    if (o_gm_params_get(gen, &p)) return -1;
    if (seed % p.g == 0) return -1;
    memset(st, 0, sizeof *st);
    for (unsigned i = 0; i < p.s; i++) {
        /* exponent (i+1) * 2^d as a little-endian byte string (G3) */
        uint8_t e[24];
        memset(e, 0, sizeof e);
        unsigned mant = i + 1;                    /* <= 32: fits 6 bits */
        unsigned byte = p.d / 8, sh = p.d % 8;
        e[byte] = (uint8_t)(mant << sh);
        e[byte + 1] = (uint8_t)((mant << sh) >> 8);
        o_gm_orbit(gen, seed, e, sizeof e, &st->xP[i], &st->xN[i]);
    }
    return 0;
}

uint32_t o_gm_next(int gen, o_gm *st)
{
    const o_gm_params *p = &PARAMS[gen];
    uint32_t word = 0;
    for (unsigned i = 0; i < p->s; i++) {
        point_step(p, &st->xP[i], &st->xN[i]);
        unsigned v = p->v, pos = v * i;
        if (gen == O_GQ58_3 && i >= 10) { v = 1; pos = 30 + (i - 10); }   /* G2, GQ58.3 tail */
        uint32_t digit = (uint32_t)(((u128)st->xN[i] << v) / p->g);       /* floor(2^v x / g) */
        word |= digit << pos;
    }
    return word;
}

void o_gm_jump(int gen, o_gm *st, const uint8_t *exp, size_t nbytes)
{
    const o_gm_params *p = &PARAMS[gen];
    uint64_t m[4];
    companion_pow(p, exp, nbytes, m);
    for (unsigned i = 0; i < p->s; i++) point_apply(m, p->g, &st->xP[i], &st->xN[i]);
}

/* canonical export: xP_0, xN_0, ..., xP_{s-1}, xN_{s-1}; u32 words when g < 2^32, else u64 */
void o_gm_export(int gen, const o_gm *st, void *out)
{
    const o_gm_params *p = &PARAMS[gen];
    for (unsigned i = 0; i < p->s; i++) {
        if (p->g < (1ull << 32)) {
            ((uint32_t *)out)[2 * i] = (uint32_t)st->xP[i];
            ((uint32_t *)out)[2 * i + 1] = (uint32_t)st->xN[i];
        } else {
            ((uint64_t *)out)[2 * i] = st->xP[i];
            ((uint64_t *)out)[2 * i + 1] = st->xN[i];
        }
    }
}
