/*
 * prand_ops.h -- layouts of the skip operators of libprand (plain C structs).
 *
 * A skip operator is the n-step map of one generator; the host
 * side of the library prepares them (step a0 of the hot path), the jump kernels and the device-callable
 * API of include/prand_device.cuh apply them.  prand_device_ops() (prand.h) returns a DEVICE array of
 * them for distances dist * 2^j, j = 0 .. levels-1, so that a stream index s is reached by applying the
 * operators of the set bits of s ("block splitting").
 */
#ifndef PRAND_OPS_H
#define PRAND_OPS_H

#include <stdint.h>

/* LFSR113: one step of a component is GF(2)-linear on its 32-bit word;
 * col[c][j] = image of the unit word 1 << j under the n-step map of component c. */
typedef struct prand_lfsr113_op { uint32_t col[4][32]; } prand_lfsr113_op;

/* MRG32K3A: A^n mod m1, B^n mod m2 (eqs. 5-6), row-major 3x3 residues acting on the
 * columns (x_n, x_{n-1}, x_{n-2}) and (y_n, y_{n-1}, y_{n-2}). */
typedef struct prand_mrg32k3a_op { uint32_t a[9]; uint32_t b[9]; } prand_mrg32k3a_op;

/* GM/GQ: n-th power of the companion matrix [[k, -q], [1, 0]] mod g, row-major, acting
 * on the column (x(n), x(n-1)) = (xN, xP) of every ensemble point. */
typedef struct prand_gm_op { uint64_t m[4]; } prand_gm_op;

/* MT19937: g_n(x) = x^n mod phi(x) (eq. 10); bit (i & 31) of w[i >> 5] = a_i. */
typedef struct prand_mt19937_op { uint32_t w[624]; } prand_mt19937_op;

#endif /* PRAND_OPS_H */
