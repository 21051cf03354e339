/*
 * prand_host.h -- host-only hooks of libprand (no CUDA call, usable on a machine without a GPU).
 *
 * They expose the host logic of step a0 (preparation of the skip operators,
 * PAPER.md:296, 347, 370, 378) and the launch policy so that CPU tests can check them against the
 * oracle.  None of them is needed to use the library; nothing here generates random numbers.
 * All pointers are HOST pointers; return value 0 or a negative prand_error code (prand.h).
 */
#ifndef PRAND_HOST_H
#define PRAND_HOST_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/*
 * Size in bytes / content of the skip operator of generator `gen` for distance mant * 2^log2:
 *   LFSR113   4 x 32 u32: col[c][j] = image of the unit word 1<<j of component c (GF(2)-linear map)
 *   MRG32K3A  18 u32: A^n mod m1 then B^n mod m2, row-major 3x3, acting on (x_n, x_{n-1}, x_{n-2})^T
 *   GM/GQ     4 u64: [[k,-q],[1,0]]^n mod g, row-major, acting on (x(n), x(n-1))^T
 *   MT19937   624 u32: coefficients of x^n mod phi(x), bit (i & 31) of word i >> 5 = a_i (eq. 10)
 */
size_t prand_host_skip_op_bytes(int gen);
int prand_host_skip_op(int gen, uint64_t mant, unsigned log2, void *buf, size_t bytes);

/* Canonical seed state of one stream at position 0 (layout of prand_get_state, not masked). */
size_t prand_host_state_bytes(int gen);
int prand_host_seed_state(int gen, uint64_t seed, void *buf, size_t bytes);

/* MT19937 characteristic polynomial phi, 624 u32 words, bit 19937 is the leading coefficient. */
int prand_host_mt19937_phi(uint32_t *words624);

/* The check prand_init makes once per process before it accepts MT19937: phi(A) annihilates a window of the
 * recurrence (Cayley-Hamilton).  0, or PRAND_ERR_INTERNAL. */
int prand_host_mt19937_phi_selfcheck(void);

/* r = a b mod phi on 624-word coefficient arrays (the product used to combine level polynomials). */
int prand_host_mt19937_mulmod(const uint32_t *a624, const uint32_t *b624, uint32_t *r624);

/*
 * PRAND ships the MT19937 jump polynomials x^v mod phi for v = 2^n (n = 0..511) and
 * v = m 2^i (m = 15..24, i = 0..127) precomputed; libprand's build step writes the same table
 * (csrc/mt_table_gen.cpp -> mt19937_polys.bin next to the library).  Copies the record of
 * v = mant * 2^log2 (624 u32 words, layout of prand_mt19937_op) or returns PRAND_ERR_ARG if v is not of a
 * tabulated form or the table file is missing.
 */
int prand_host_mt19937_table(uint64_t mant, unsigned log2, uint32_t *words624);

/*
 * Launch policy of prand_generate_* on a device with `sm_count` multiprocessors: a stream's range
 * of n_per_stream outputs is cut into n_chunks sub-sections of chunk_len reached by jump-ahead
 * when there are too few streams to fill the GPU.  dtype: 0 u32, 1 f32, 2 f64.
 */
int prand_host_plan(int gen, uint64_t n_streams, uint64_t n_per_stream, int dtype, int sm_count,
                    uint64_t *chunk_len, uint64_t *n_chunks);

/*
 * GM/GQ: the coefficients (k_n, q_n) of the paper's jump relation x(2n+w) = k_n x(n+w) - q_n x(w)
 * (eq. 2) for n = mant * 2^log2, computed by eq. 3-4 (Lucas ladder, no matrix);
 * prand_init fills a family of >= 64 streams with them.
 */
int prand_host_gm_kq(int gen, uint64_t mant, unsigned log2, uint64_t *k_n, uint64_t *q_n);

/*
 * Section plan of prand_generate_seq_* (Table 5): `length` outputs of one sequence are
 * cut into n_sections sections of sec_len (a multiple of 32; the last one may be shorter).
 */
int prand_host_plan_sections(int gen, uint64_t length, uint64_t *n_sections, uint64_t *sec_len);
/* The plan above is the one of a device with 148 multiprocessors (B200).  prand_generate_seq_* plans with the
 * multiprocessor count of the device it runs on (MT19937 takes at most 4 sections per multiprocessor); this variant
 * takes that count, so that the cuts can be located on any device. */
int prand_host_plan_sections_sm(int gen, uint64_t length, int sm_count, uint64_t *n_sections, uint64_t *sec_len);

#ifdef __cplusplus
}
#endif
#endif /* PRAND_HOST_H */
