/*
 * driver.c -- generic entry points of the oracle (TEST INFRASTRUCTURE ONLY, see oracle.h).
 *
 * Conversions, reading CONV (PAPER.md:443-446 only says "uniformly distributed in the interval
 * [0,1)" and gives no formula): f32 = (u >> 8) * 2^-24 (exact, < 1); f64 = u * 2^-32 (exact);
 * MRG32K3A f64 is reading M3 (mrg32k3a.c).
 *
 * Block splitting: stream s = the base sequence advanced s*block_len.
 * oracle_streams() takes the per-stream exponents s*block_len as byte strings computed by the
 * caller (plain integer arithmetic in Python), seeds, jumps, and then generates by single steps.
 */
#include "oracle.h"
#include <string.h>

float o_u32_to_f32(uint32_t u) { return (float)(u >> 8) * (1.0f / 16777216.0f); }
double o_u32_to_f64(uint32_t u) { return (double)u * (1.0 / 4294967296.0); }

static int is_gm(int gen) { return gen >= O_GM19 && gen <= O_GQ58_4; }

size_t oracle_internal_bytes(int gen)
{
    if (gen == O_LFSR113) return sizeof(o_lfsr113);
    if (gen == O_MRG32K3A) return sizeof(o_mrg32k3a);
    if (gen == O_MT19937) return sizeof(o_mt19937);
    if (is_gm(gen)) return sizeof(o_gm);
    return 0;
}

size_t oracle_state_bytes(int gen)
{
    if (gen == O_LFSR113) return 16;
    if (gen == O_MRG32K3A) return 24;
    if (gen == O_MT19937) return 2496;
    if (is_gm(gen)) {
        o_gm_params p;
        o_gm_params_get(gen, &p);
        return (size_t)2 * p.s * (p.g < (1ull << 32) ? 4 : 8);
    }
    return 0;
}

int oracle_seed(int gen, uint64_t seed, void *st)
{
    if (gen == O_LFSR113) return seed > 0xFFFFFFFFull ? -1 : o_lfsr113_seed(st, (uint32_t)seed);
    if (gen == O_MRG32K3A) return seed > 0xFFFFFFFFull ? -1 : o_mrg32k3a_seed(st, (uint32_t)seed);
    if (gen == O_MT19937) {
        if (seed > 0xFFFFFFFFull) return -1;
        o_mt19937_seed(st, (uint32_t)seed);
        return 0;
    }
    if (is_gm(gen)) return o_gm_seed(gen, st, seed);
    return -1;
}

int oracle_jump(int gen, void *st, const uint8_t *exp, size_t nbytes)
{
    if (gen == O_LFSR113) o_lfsr113_jump(st, exp, nbytes);
    else if (gen == O_MRG32K3A) o_mrg32k3a_jump(st, exp, nbytes);
    else if (gen == O_MT19937) o_mt19937_jump(st, exp, nbytes);
    else if (is_gm(gen)) o_gm_jump(gen, st, exp, nbytes);
    else return -1;
    return 0;
}

void oracle_export(int gen, const void *st, void *canon)
{
    if (gen == O_LFSR113) o_lfsr113_export(st, canon);
    else if (gen == O_MRG32K3A) o_mrg32k3a_export(st, canon);
    else if (gen == O_MT19937) o_mt19937_export(st, canon);
    else if (is_gm(gen)) o_gm_export(gen, st, canon);
}

int oracle_import(int gen, void *st, const void *canon)
{
    if (gen == O_LFSR113) memcpy(st, canon, 16);
    else if (gen == O_MRG32K3A) memcpy(st, canon, 24);
    else if (gen == O_MT19937) memcpy(st, canon, 2496);
    else if (is_gm(gen)) {
        o_gm_params p;
        o_gm *g = st;
        o_gm_params_get(gen, &p);
        memset(g, 0, sizeof *g);
        for (unsigned i = 0; i < p.s; i++) {
            if (p.g < (1ull << 32)) {
                g->xP[i] = ((const uint32_t *)canon)[2 * i];
                g->xN[i] = ((const uint32_t *)canon)[2 * i + 1];
            } else {
                g->xP[i] = ((const uint64_t *)canon)[2 * i];
                g->xN[i] = ((const uint64_t *)canon)[2 * i + 1];
            }
        }
    } else return -1;
    return 0;
}

static uint32_t next_u32(int gen, void *st)
{
    if (gen == O_LFSR113) return o_lfsr113_next(st);
    if (gen == O_MRG32K3A) return o_mrg32k3a_next(st);
    if (gen == O_MT19937) return o_mt19937_next(st);
    return o_gm_next(gen, st);
}

int oracle_fill(int gen, void *st, uint64_t count, int dtype, void *out, uint64_t stride)
{
    if (oracle_internal_bytes(gen) == 0) return -1;
    for (uint64_t j = 0; j < count; j++) {
        uint32_t u = next_u32(gen, st);
        if (dtype == O_U32) ((uint32_t *)out)[j * stride] = u;
        else if (dtype == O_F32) ((float *)out)[j * stride] = o_u32_to_f32(u);
        else if (dtype == O_F64)
            ((double *)out)[j * stride] = gen == O_MRG32K3A ? o_mrg32k3a_to_f64(u) : o_u32_to_f64(u);
        else return -1;
    }
    return 0;
}

int oracle_streams(int gen, uint64_t seed, uint64_t s_count,
                   const uint8_t *stream_exp, size_t nbytes,
                   uint64_t n_per_stream, int dtype, void *out,
                   uint64_t row_stride, uint64_t col0, void *canon_states)
{
    union { o_lfsr113 l; o_mrg32k3a m; o_mt19937 t; o_gm g; } st;
    size_t esz = dtype == O_F64 ? 8 : 4, cb = oracle_state_bytes(gen);
    if (cb == 0) return -1;
    for (uint64_t s = 0; s < s_count; s++) {
        if (oracle_seed(gen, seed, &st)) return -2;
        oracle_jump(gen, &st, stream_exp + s * nbytes, nbytes);
        if (n_per_stream && out) {
            int rc = oracle_fill(gen, &st, n_per_stream, dtype, (char *)out + (col0 + s) * esz, row_stride);
            if (rc) return rc;
        }
        if (canon_states) oracle_export(gen, &st, (char *)canon_states + s * cb);
    }
    return 0;
}
