/*
 * oracle.h -- CPU oracle for the PRAND hot path (arXiv 1307.5869, Barash & Shchur).
 *
 * TEST INFRASTRUCTURE ONLY.  This is the plain, slow, scalar reference that the CUDA
 * library is checked against.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load it.  It shares no code, header, table
 * or helper with paper_1307_5869_b200/ (the product) and never calls into it.
 *
 * Every function cites the PAPER.md passage it follows ("PAPER.md:<line>").  Where the
 * paper is silent or garbled the reading of SURVEY.md section 8(c) is taken; those
 * readings are labelled (L1..L4, M1..M5, T1..T4, G1..G3, CONV) here and in DESIGN.md.
 *
 * Parity status: every function below is pinned by tests/test_oracle_*.py against
 * something other than itself (bit-level definitions, library routines, period
 * invariants printed in the paper's Table 2, brute force).  What stays "parity
 * unpinned" against the *original PRAND binary* (not available): the GM/GQ output
 * packing (G2), the GM/GQ seeding (G3) and the MRG32K3A combination sign (M1).
 *
 * Positional convention used for all generators ("step-then-output"):
 *   a state at position P produces output number P by first advancing one step and
 *   then reading the output from the new state.  Stream s of a block-split family
 *   starts at position s*block_len of the single base sequence.
 *
 * Jump exponents are arbitrary-precision non-negative integers passed as little-endian
 * byte strings (exp, nbytes), because block lengths such as 2^76 or
 * period tests (2^19937) do not fit a machine word.
 */
#ifndef PRAND_ORACLE_H
#define PRAND_ORACLE_H

#include <stddef.h>
#include <stdint.h>

enum {
    O_LFSR113 = 0, O_MRG32K3A = 1, O_MT19937 = 2,
    O_GM19 = 3, O_GM29 = 4, O_GM31 = 5, O_GM55 = 6, O_GM61 = 7,
    O_GQ58_1 = 8, O_GQ58_3 = 9, O_GQ58_4 = 10, O_NGEN = 11
};

enum { O_U32 = 0, O_F32 = 1, O_F64 = 2 };

/* ---- LFSR113 ------------------------------------------------ */
typedef struct { uint32_t z[4]; } o_lfsr113;
int      o_lfsr113_seed(o_lfsr113 *st, uint32_t seed);           /* 0 ok, -1 invalid   */
uint32_t o_lfsr113_next(o_lfsr113 *st);                          /* step, then output  */
void     o_lfsr113_jump(o_lfsr113 *st, const uint8_t *exp, size_t nbytes);
void     o_lfsr113_export(const o_lfsr113 *st, uint32_t out[4]); /* masked top-p bits  */

/* ---- MRG32K3A ----------------------------------------------- */
typedef struct { uint32_t x[3]; uint32_t y[3]; } o_mrg32k3a;     /* x[0]=x_n, x[1]=x_{n-1}, x[2]=x_{n-2} */
int      o_mrg32k3a_seed(o_mrg32k3a *st, uint32_t seed);
uint32_t o_mrg32k3a_next(o_mrg32k3a *st);                        /* z_n in [0,m1)      */
double   o_mrg32k3a_to_f64(uint32_t z);                          /* (0,1), reading M3  */
void     o_mrg32k3a_jump(o_mrg32k3a *st, const uint8_t *exp, size_t nbytes);
void     o_mrg32k3a_export(const o_mrg32k3a *st, uint32_t out[6]);

/* ---- MT19937 ------------------------------------------------ */
typedef struct { uint32_t w[624]; } o_mt19937;                   /* window x_P..x_{P+623} */
void     o_mt19937_seed(o_mt19937 *st, uint32_t seed);
uint32_t o_mt19937_next(o_mt19937 *st);
void     o_mt19937_jump(o_mt19937 *st, const uint8_t *exp, size_t nbytes);
void     o_mt19937_export(const o_mt19937 *st, uint32_t out[624]);
/* pieces exposed so that tests can pin them one by one */
int      o_mt19937_charpoly(uint64_t phi[312]);                  /* returns degree      */
void     o_mt19937_jump_poly(const uint8_t *exp, size_t nbytes, uint64_t g[312]);
void     o_mt19937_apply_poly(o_mt19937 *st, const uint64_t g[312]);

/* ---- GM / GQ family (Table 2) ---------------- */
typedef struct { uint64_t xP[32]; uint64_t xN[32]; } o_gm;       /* points 0..s-1       */
typedef struct { uint64_t k, q, g; unsigned v, s, d; } o_gm_params;
int      o_gm_params_get(int gen, o_gm_params *p);
int      o_gm_seed(int gen, o_gm *st, uint64_t seed);
uint32_t o_gm_next(int gen, o_gm *st);
void     o_gm_jump(int gen, o_gm *st, const uint8_t *exp, size_t nbytes);
void     o_gm_export(int gen, const o_gm *st, void *out);        /* u32 or u64 words    */
/* single orbit point: (w(n), w(n+1)) of the base orbit w(0)=0, w(1)=seed mod g         */
void     o_gm_orbit(int gen, uint64_t seed, const uint8_t *exp, size_t nbytes,
                    uint64_t *w_n, uint64_t *w_n1);

/* ---- conversions (reading CONV) ------------------------------ */
float    o_u32_to_f32(uint32_t u);   /* (u >> 8) * 2^-24, in [0,1)   */
double   o_u32_to_f64(uint32_t u);   /* u * 2^-32, in [0,1)          */

/* ---- generic driver ------------------------------------------------------------ */
size_t oracle_internal_bytes(int gen);          /* sizeof internal state struct        */
size_t oracle_state_bytes(int gen);             /* canonical export bytes per stream   */
int    oracle_seed(int gen, uint64_t seed, void *st);
int    oracle_jump(int gen, void *st, const uint8_t *exp, size_t nbytes);
void   oracle_export(int gen, const void *st, void *canon);
int    oracle_import(int gen, void *st, const void *canon);
/* Advance `st` by `count` steps writing output j to out[j*stride] in `dtype`. */
int    oracle_fill(int gen, void *st, uint64_t count, int dtype, void *out, uint64_t stride);
/* Streams [s_first, s_first+s_count): seed, jump by stream_exp[s] (s_count byte strings
 * of nbytes each, = s*block_len), then fill n_per_stream outputs in the canonical layout
 * out[i*row_stride + (s - s_first) + col0] and export the final canonical states.       */
int    oracle_streams(int gen, uint64_t seed, uint64_t s_count,
                      const uint8_t *stream_exp, size_t nbytes,
                      uint64_t n_per_stream, int dtype, void *out,
                      uint64_t row_stride, uint64_t col0, void *canon_states);

#endif
