/*
 * mt19937.c -- oracle for MT19937 (TEST INFRASTRUCTURE ONLY, see oracle.h).
 *
 * PAPER.md:374-378 (section 5.4): "The general algorithm for MT19937 is presented in [2]";
 * it is linear over F_2, Y_{n+1} = A Y_n, and jump-ahead uses
 *     A^v Y_0 = g_v(A) Y_0 = a_k Y_{k-1} + ... + a_2 Y_1 + a_1 Y_0,  k = 19937   (eq. 10)
 * with g_v(x) = x^v mod phi(x), phi the characteristic polynomial of A.
 *
 * Reading T1 (the paper prints no constants; they are those of its ref. [2], which is the
 * parameter set of ISO C++ std::mt19937): w=32, n=624, m=397, r=31, a=0x9908B0DF,
 * tempering (u,s,b,t,c,l) = (11, 7, 0x9D2C5680, 15, 0xEFC60000, 18), seeding
 * x_0 = seed, x_i = 1812433253*(x_{i-1} ^ (x_{i-1} >> 30)) + i.
 * Recurrence: x_{i+624} = x_{i+397} ^ (y >> 1) ^ (a if y odd),
 *             y = (x_i & 0x80000000) | (x_{i+1} & 0x7FFFFFFF).
 * Position convention (paper silent): the state at position P is the window x_P..x_{P+623};
 * output number P is temper(x_{P+624}).  BASELINE.json pins seed 5489 -> output #9999
 * (the 10000th) = 4123659995.
 * Reading T2: only the top bit of window word 0 belongs to the 19937-bit state; the
 * canonical export zeroes its low 31 bits.
 * Reading T4: PRAND's precomputed polynomial table is not available;
 * g_v is computed as x^v mod phi for any v.
 *
 * phi is obtained as the minimal polynomial (Berlekamp-Massey) of one output bit-plane of
 * x_t; it is pinned in tests by its degree (19937), by phi(A) W = 0, by
 * x^(2^19937) = x (mod phi) (period 2^19937-1) and through jump = stepping.
 */
#include "oracle.h"
#include <stdlib.h>
#include <string.h>

#define NW 624
#define MW 397
#define DEG 19937
#define PW 312                 /* 64-bit words holding a polynomial of degree < 19968 */

void o_mt19937_seed(o_mt19937 *st, uint32_t seed)
{
    st->w[0] = seed;
    for (uint32_t i = 1; i < NW; i++)
        st->w[i] = 1812433253u * (st->w[i - 1] ^ (st->w[i - 1] >> 30)) + i;
}

static uint32_t recur(uint32_t xi, uint32_t xi1, uint32_t xim)
{
    uint32_t y = (xi & 0x80000000u) | (xi1 & 0x7FFFFFFFu);
    return xim ^ (y >> 1) ^ ((y & 1u) ? 0x9908B0DFu : 0u);
}

static uint32_t temper(uint32_t y)
{
    y ^= y >> 11;
    y ^= (y << 7) & 0x9D2C5680u;
    y ^= (y << 15) & 0xEFC60000u;
    y ^= y >> 18;
    return y;
}

/* one step: window x_P.. -> x_{P+1}..; returns the new word x_{P+624} */
static uint32_t step_window(o_mt19937 *st)
{
    uint32_t nw = recur(st->w[0], st->w[1], st->w[MW]);
    memmove(&st->w[0], &st->w[1], (NW - 1) * sizeof(uint32_t));
    st->w[NW - 1] = nw;
    return nw;
}

uint32_t o_mt19937_next(o_mt19937 *st) { return temper(step_window(st)); }

/* ---------------- polynomials over F_2, bit i of word i/64 = coefficient of x^i -------- */

static int pbit(const uint64_t *p, size_t i) { return (int)((p[i >> 6] >> (i & 63)) & 1u); }

/* p ^= q << sh, q has qw words, p must be large enough */
static void pxor_shifted(uint64_t *p, const uint64_t *q, size_t qw, size_t sh)
{
    size_t ws = sh >> 6, bs = sh & 63;
    for (size_t i = 0; i < qw; i++) {
        p[i + ws] ^= q[i] << bs;
        if (bs) p[i + ws + 1] ^= q[i] >> (64 - bs);
    }
}

static uint64_t PHI[PW + 1];
static int PHI_READY = 0;

/* Berlekamp-Massey over F_2 on N = 2*DEG + 64 bits of the least significant bit of x_t. */
static void build_phi(void)
{
    enum { N = 2 * DEG + 64 };
    uint8_t *s = malloc(N), *C = calloc(N + 1, 1), *B = calloc(N + 1, 1), *T = malloc(N + 1);
    o_mt19937 st;
    o_mt19937_seed(&st, 5489u);
    for (int n = 0; n < N; n++) s[n] = (uint8_t)(step_window(&st) & 1u);
    int L = 0, m = 1;
    C[0] = B[0] = 1;
    for (int n = 0; n < N; n++) {
        int d = s[n];
        for (int i = 1; i <= L; i++) d ^= C[i] & s[n - i];
        if (d == 0) { m++; continue; }
        if (2 * L <= n) {
            memcpy(T, C, N + 1);
            for (int i = 0; i + m <= N; i++) C[i + m] ^= B[i];
            L = n + 1 - L;
            memcpy(B, T, N + 1);
            m = 1;
        } else {
            for (int i = 0; i + m <= N; i++) C[i + m] ^= B[i];
            m++;
        }
    }
    /* s[t+L] = sum_{i=1..L} C[i] s[t+L-i]  =>  phi(x) = x^L + sum_{j<L} C[L-j] x^j */
    memset(PHI, 0, sizeof PHI);
    for (int j = 0; j <= L && j < 64 * (PW + 1); j++)
        if (C[L - j]) PHI[j >> 6] |= 1ull << (j & 63);
    PHI_READY = L;
    free(s); free(C); free(B); free(T);
}

int o_mt19937_charpoly(uint64_t phi[312])
{
    if (!PHI_READY) build_phi();
    memcpy(phi, PHI, PW * sizeof(uint64_t));   /* bits 0..19967; bit 19937 is the leading one */
    return PHI_READY;
}

/* r (PW words) = a*b mod phi, schoolbook: shift-and-xor product, then bitwise long division */
static void pmulmod(uint64_t *r, const uint64_t *a, const uint64_t *b)
{
    uint64_t prod[2 * PW + 2];
    memset(prod, 0, sizeof prod);
    for (size_t i = 0; i < DEG; i++)
        if (pbit(a, i)) pxor_shifted(prod, b, PW, i);
    for (size_t d = 2 * DEG - 2; d >= DEG; d--)
        if (pbit(prod, d)) pxor_shifted(prod, PHI, PW, d - DEG);
    memcpy(r, prod, PW * sizeof(uint64_t));
}

/* g = x^e mod phi, left-to-right square and multiply */
void o_mt19937_jump_poly(const uint8_t *exp, size_t nbytes, uint64_t g[312])
{
    if (!PHI_READY) build_phi();
    uint64_t acc[PW], x[PW];
    memset(acc, 0, sizeof acc); acc[0] = 1;      /* 1 */
    memset(x, 0, sizeof x);     x[0] = 2;        /* x */
    int started = 0;
    for (size_t i = nbytes; i-- > 0;)
        for (int b = 7; b >= 0; b--) {
            int bit = (exp[i] >> b) & 1;
            if (!started && !bit) continue;      /* leading zeros: acc stays 1 */
            started = 1;
            pmulmod(acc, acc, acc);
            if (bit) pmulmod(acc, acc, x);
        }
    memcpy(g, acc, sizeof acc);
}

/* eq. 10: window <- sum_i a_i * (window advanced i steps), a_i = coefficient of x^i in g. */
void o_mt19937_apply_poly(o_mt19937 *st, const uint64_t g[312])
{
    uint32_t *x = malloc((DEG + NW) * sizeof(uint32_t));
    memcpy(x, st->w, NW * sizeof(uint32_t));
    for (size_t t = 0; t + NW < DEG + NW; t++) x[t + NW] = recur(x[t], x[t + 1], x[t + MW]);
    uint32_t acc[NW];
    memset(acc, 0, sizeof acc);
    for (size_t i = 0; i < DEG; i++)
        if (pbit(g, i))
            for (size_t j = 0; j < NW; j++) acc[j] ^= x[i + j];
    memcpy(st->w, acc, sizeof acc);
    st->w[0] &= 0x80000000u;                      /* T2: bits outside the 19937-bit state */
    free(x);
}

void o_mt19937_jump(o_mt19937 *st, const uint8_t *exp, size_t nbytes)
{
    uint64_t g[PW];
    o_mt19937_jump_poly(exp, nbytes, g);
    o_mt19937_apply_poly(st, g);
}

void o_mt19937_export(const o_mt19937 *st, uint32_t out[624])
{
    memcpy(out, st->w, NW * sizeof(uint32_t));
    out[0] &= 0x80000000u;
}
