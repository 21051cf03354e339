/*
 * lfsr113.c -- oracle for LFSR113 (TEST INFRASTRUCTURE ONLY, see oracle.h).
 *
 * PAPER.md:351-361 (section 5.3): LFSR113 combines four shift-register sequences.  Each obeys
 *     x_n = x_{n-p} + x_{n-p+q}  (mod 2)                                   (eq. 7)
 * and emits the 32-bit fraction
 *     u_n = sum_{i=1..32} x_{ns+i-1} 2^-i                                   (eq. 8)
 * i.e. the word whose most significant bit is x_{ns}, next bit x_{ns+1}, ...  The four
 * parameter sets are (p,q,s) = (31,6,18), (29,2,2), (28,13,7), (25,3,13);
 * the generator's output is the bitwise sum (XOR) of the four words.
 *
 * Word form used here, derived from eq. 7-8.  Let the component state word z hold the bits
 * x_{ns} .. x_{ns+31}, MSB first.  Only its top p bits are free (the remaining 32-p follow
 * from eq. 7).  The next word needs bits x_{ns+s} .. x_{ns+s+31}:
 *   - the first p-s of them are bits s..p-1 of z: (z & mask_p) << s puts them on top, where
 *     mask_p keeps the top p bits (the low 32-p bits of z are *not* trusted, reading L1);
 *   - bit number p+j of the stream is x_j + x_{j+q} (eq. 7 with n = p+j), i.e. bit j of
 *     (z ^ (z << q)); the word needs j = 0 .. 32-(p-s)-1 of these placed below the first
 *     p-s bits: ((z << q) ^ z) >> (p - s).  All bits of (z << q) used are inside the top p
 *     bits of z because j + q <= 32-(p-s)-1+q < p for all four parameter sets.
 * Hence  z' = ((z & mask_p) << s) ^ (((z << q) ^ z) >> (p - s)).
 * tests/test_oracle_lfsr113.py pins this against a literal bit-by-bit eq. 7-8 program.
 *
 * Readings: L1 the seed's low 32-p bits are ignored; L2 output number i of a
 * state at position P is u_{P+i+1} (step, then output); L3 canonical export masks the low bits.
 */
#include "oracle.h"
#include <string.h>

static const unsigned LP[4] = {31, 29, 28, 25};
static const unsigned LQ[4] = {6, 2, 13, 3};
static const unsigned LS[4] = {18, 2, 7, 13};

static uint32_t mask_top(unsigned p) { return (uint32_t)(0xFFFFFFFFu << (32 - p)); }

static uint32_t comp_step(uint32_t z, unsigned c)
{
    unsigned p = LP[c], q = LQ[c], s = LS[c];
    uint32_t b = ((z << q) ^ z) >> (p - s);
    return ((z & mask_top(p)) << s) ^ b;
}

/* Seed: all four words = seed (SURVEY.md 8(b) seed convention, BASELINE.json config 1).
 * A component whose top p bits are all zero is stuck at zero: reject (z1<2, z2<8, z3<16, z4<128). */
int o_lfsr113_seed(o_lfsr113 *st, uint32_t seed)
{
    for (int c = 0; c < 4; c++) {
        if ((seed & mask_top(LP[c])) == 0) return -1;
        st->z[c] = seed;
    }
    return 0;
}

uint32_t o_lfsr113_next(o_lfsr113 *st)
{
    uint32_t u = 0;
    for (int c = 0; c < 4; c++) {
        st->z[c] = comp_step(st->z[c], c);
        u ^= st->z[c];
    }
    return u;
}

/* Jump-ahead: one step of a component is linear over GF(2) on the 32-bit word, so n steps are
 * the n-th power of a 32x32 bit matrix (the "natural linear operator"; the paper's own table
 * method, reaches the same state).  A matrix is stored by columns:
 * col[j] = image of the unit word 1<<j. */
typedef struct { uint32_t col[32]; } bm32;

static uint32_t bm_apply(const bm32 *m, uint32_t v)
{
    uint32_t r = 0;
    for (int j = 0; j < 32; j++)
        if ((v >> j) & 1u) r ^= m->col[j];
    return r;
}

static void bm_mul(bm32 *out, const bm32 *a, const bm32 *b) /* out = a*b (apply b first) */
{
    bm32 t;
    for (int j = 0; j < 32; j++) t.col[j] = bm_apply(a, b->col[j]);
    *out = t;
}

void o_lfsr113_jump(o_lfsr113 *st, const uint8_t *exp, size_t nbytes)
{
    for (int c = 0; c < 4; c++) {
        bm32 step, acc;
        for (int j = 0; j < 32; j++) {
            step.col[j] = comp_step(1u << j, c);
            acc.col[j] = 1u << j;               /* identity */
        }
        /* left-to-right square and multiply over the bits of exp */
        for (size_t i = nbytes; i-- > 0;) {
            for (int b = 7; b >= 0; b--) {
                bm_mul(&acc, &acc, &acc);
                if ((exp[i] >> b) & 1u) bm_mul(&acc, &step, &acc);
            }
        }
        st->z[c] = bm_apply(&acc, st->z[c]);
    }
}

void o_lfsr113_export(const o_lfsr113 *st, uint32_t out[4])
{
    for (int c = 0; c < 4; c++) out[c] = st->z[c] & mask_top(LP[c]);
}
