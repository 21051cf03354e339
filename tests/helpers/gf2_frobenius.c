/*
 * gf2_frobenius.c -- test helper (compiled by tests/test_oracle_mt19937.py, not part of the
 * oracle or of the product).  Reads the exponents of a sparse polynomial phi over F_2 from
 * stdin (first number = degree n, then the lower exponents) and prints "1" if
 * x^(2^n) == x (mod phi), else "0".  Own arithmetic: squaring by bit spreading, reduction one
 * 64-bit word at a time against the sparse terms (valid because the gap between n and the next
 * exponent is >= 64, which is checked).
 */
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

int main(void)
{
    int n, terms[4096], nt = 0, e;
    if (scanf("%d", &n) != 1) return 2;
    while (scanf("%d", &e) == 1 && nt < 4096) terms[nt++] = e;
    for (int i = 0; i < nt; i++) if (n - terms[i] < 64 || terms[i] < 0) return 3;
    int words = (2 * n + 63) / 64 + 1;
    uint64_t *a = calloc(words, 8), *b = calloc(words, 8);
    a[0] = 2;                                           /* x */
    for (int it = 0; it < n; it++) {
        memset(b, 0, words * 8);
        for (int i = 0; i < n; i++)                     /* b = a^2 */
            if ((a[i >> 6] >> (i & 63)) & 1) b[(2 * i) >> 6] |= 1ull << ((2 * i) & 63);
        for (int w = words - 1; w >= n / 64; w--) {     /* fold everything at or above x^n */
            uint64_t W = b[w];
            if (w == n / 64) W &= ~((1ull << (n & 63)) - 1);
            if (!W) continue;
            b[w] ^= W;
            long base = (long)w * 64 - n;               /* W*x^(64w) = W*x^base*x^n */
            for (int t = 0; t < nt; t++) {
                long pos = base + terms[t];
                long ws = pos >> 6; int bs = (int)(pos & 63);
                b[ws] ^= W << bs;
                if (bs) b[ws + 1] ^= W >> (64 - bs);
            }
        }
        uint64_t *tmp = a; a = b; b = tmp;
    }
    int ok = a[0] == 2;
    for (int i = 1; i < words; i++) ok &= a[i] == 0;
    printf("%d\n", ok);
    return 0;
}
