/*
 * mrg32k3a.c -- oracle for MRG32K3A (TEST INFRASTRUCTURE ONLY, see oracle.h).
 *
 * PAPER.md:336-347 (section 5.2, eqs. 5-6):
 *     X_{n+1} = A X_n (mod m1),  Y_{n+1} = B Y_n (mod m2),
 *     X_n = (x_n, x_{n-1}, x_{n-2})^T,  Y_n = (y_n, y_{n-1}, y_{n-2})^T,
 *     A = [[0 a b],[1 0 0],[0 1 0]],  B = [[c 0 d],[1 0 0],[0 1 0]],
 *     a = 1403580, b = -810728, c = 527612, d = -1370589,
 *     m1 = 2^32 - 209, m2 = 2^32 - 22853.
 * Jump-ahead: A^n mod m1, B^n mod m2 in O(log n).
 *
 * Readings:
 *  M1  the printed output "(x_n + y_n) (mod g)" has an undefined g; the
 *      generator the paper says it implements is ref [3]'s, whose combination is
 *      z_n = (x_n - y_n) mod m1.  That is what is computed here.
 *  M2  the u32 output is z_n in [0, m1).
 *  M3  f64 in (0,1): u = z_n * norm with norm = 1/(m1+1) = 2.328306549295727688e-10 and
 *      z_n = 0 mapped to m1*norm; one IEEE-754 double multiply, round to nearest.
 *  M4  f32 is the generic conversion applied to z_n.
 *  M5  seed: all six state words = seed; export order x_n,x_{n-1},x_{n-2},y_n,y_{n-1},y_{n-2}.
 */
#include "oracle.h"

#define M1 4294967087ull   /* 2^32 - 209   */
#define M2 4294944443ull   /* 2^32 - 22853 */

typedef unsigned __int128 u128;

/* row-major 3x3 matrices of residues */
static const uint64_t A_MAT[9] = {0, 1403580ull, M1 - 810728ull, 1, 0, 0, 0, 1, 0};
static const uint64_t B_MAT[9] = {527612ull, 0, M2 - 1370589ull, 1, 0, 0, 0, 1, 0};

int o_mrg32k3a_seed(o_mrg32k3a *st, uint32_t seed)
{
    if (seed == 0 || (uint64_t)seed >= M2) return -1;  /* valid residue for both moduli, not all-zero */
    for (int i = 0; i < 3; i++) { st->x[i] = seed; st->y[i] = seed; }
    return 0;
}

static void matvec(const uint64_t m[9], uint32_t v[3], uint64_t mod)
{
    uint64_t r[3];
    for (int i = 0; i < 3; i++) {
        u128 acc = 0;
        for (int j = 0; j < 3; j++) acc += (u128)m[3 * i + j] * v[j];
        r[i] = (uint64_t)(acc % mod);
    }
    for (int i = 0; i < 3; i++) v[i] = (uint32_t)r[i];
}

static void matmul(uint64_t out[9], const uint64_t a[9], const uint64_t b[9], uint64_t mod)
{
    uint64_t t[9];
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            u128 acc = 0;
            for (int l = 0; l < 3; l++) acc += (u128)a[3 * i + l] * b[3 * l + j];
            t[3 * i + j] = (uint64_t)(acc % mod);
        }
    for (int i = 0; i < 9; i++) out[i] = t[i];
}

uint32_t o_mrg32k3a_next(o_mrg32k3a *st)
{
    matvec(A_MAT, st->x, M1);                      /* eq. 5 with the matrices of eq. 6 */
    matvec(B_MAT, st->y, M2);
    uint64_t x = st->x[0], y = st->y[0];
    return (uint32_t)((x + M1 - y % M1) % M1);     /* z_n = (x_n - y_n) mod m1 (M1, M2) */
}

double o_mrg32k3a_to_f64(uint32_t z)
{
    const double norm = 2.328306549295727688e-10;  /* 1/(m1+1) (M3) */
    volatile double u = (z == 0 ? (double)M1 : (double)z) * norm;
    return u;
}

static void matpow(uint64_t out[9], const uint64_t base[9], uint64_t mod,
                   const uint8_t *exp, size_t nbytes)
{
    uint64_t acc[9] = {1, 0, 0, 0, 1, 0, 0, 0, 1};
    for (size_t i = nbytes; i-- > 0;)
        for (int b = 7; b >= 0; b--) {
            matmul(acc, acc, acc, mod);
            if ((exp[i] >> b) & 1u) matmul(acc, base, acc, mod);
        }
    for (int i = 0; i < 9; i++) out[i] = acc[i];
}

void o_mrg32k3a_jump(o_mrg32k3a *st, const uint8_t *exp, size_t nbytes)
{
    uint64_t an[9], bn[9];
    matpow(an, A_MAT, M1, exp, nbytes);
    matpow(bn, B_MAT, M2, exp, nbytes);
    matvec(an, st->x, M1);
    matvec(bn, st->y, M2);
}

void o_mrg32k3a_export(const o_mrg32k3a *st, uint32_t out[6])
{
    for (int i = 0; i < 3; i++) { out[i] = st->x[i]; out[3 + i] = st->y[i]; }
}
