// skip_ops.h -- host-side preparation of the skip operators.
//
// For a distance n = mant * 2^log2 the library needs the n-step map of every generator:
//   LFSR113   four 32x32 GF(2) matrices
//   MRG32K3A  A^n mod m1, B^n mod m2 (3x3)
//   GM/GQ     [[k,-q],[1,0]]^n mod g (2x2)
//   MT19937   g_n(x) = x^n mod phi(x)             (eq. 10)
// and, for block splitting, the "level" family n * 2^j, j = 0..levels-1, so that
// stream s is reached by multiplying the operators of the set bits of s.
// Product code: shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <vector>
#include "internal.h"

namespace prand {
namespace host {

// distance mant * 2^log2
struct Dist { uint64_t mant; unsigned log2; };

// ---- LFSR113 -------------------------------------------------------------------------------------
uint32_t lfsr113_component_step(int c, uint32_t z);   // one output step of component c (0..3)
void lfsr113_levels(Dist n, unsigned levels, std::vector<LfsrOp> &out);

// ---- MRG32K3A ------------------------------------------------------------------------------------
void mrg32k3a_levels(Dist n, unsigned levels, std::vector<MrgOp> &out);

// ---- GM/GQ ---------------------------------------------------------------------------------------
void gm_levels(const GmParams &p, Dist n, unsigned levels, std::vector<GmOp> &out);
// seed state of the ensemble (reading G3): words xP_0, xN_0, ..., xP_{s-1}, xN_{s-1} with
// (xP_i, xN_i) = (w((i+1) 2^d), w((i+1) 2^d + 1)), w(0) = 0, w(1) = seed mod g.  false if seed = 0 mod g.
// (k_n, q_n) of the paper's eq. 2-4 for n * 2^j, j < levels
void gm_kq_levels(const GmParams &p, Dist n, unsigned levels, std::vector<uint64_t> &kn, std::vector<uint64_t> &qn);
bool gm_seed_state(const GmParams &p, uint64_t seed, uint64_t *words);

// ---- MT19937 -------------------------------------------------------------------------------------
constexpr int MT_N = 624, MT_M = 397, MT_DEG = 19937;
constexpr int MT_PW = 312;                         // 64-bit words of a polynomial of degree < 19968
struct MtPoly { uint64_t w[MT_PW]; };              // bit (i & 63) of w[i >> 6] = coefficient of x^i
const MtPoly &mt19937_phi();                       // characteristic polynomial (closed form of ref. [2])
bool mt19937_phi_selfcheck();                      // phi(A) annihilates a generated window (checked once per process)
void mt19937_mulmod(MtPoly &r, const MtPoly &a, const MtPoly &b);   // r = a b mod phi
void mt19937_sqrmod(MtPoly &r, const MtPoly &a);                     // r = a^2 mod phi
void mt19937_xpow(Dist n, MtPoly &out);                              // x^n mod phi (table entries where they apply)
void mt19937_xpow_raw(Dist n, MtPoly &out);                          // x^n mod phi by square-and-multiply only

// The precomputed table of: x^v mod phi for v = 2^n (n < 512) and v = m 2^i (m = 15..24, i < 128),
// written by csrc/mt_table_gen.cpp at build time and loaded from the file next to the library.
constexpr int MT_TABLE_POW2 = 512, MT_TABLE_M0 = 15, MT_TABLE_M1 = 24, MT_TABLE_SHIFTS = 128;
constexpr int MT_TABLE_ENTRIES = MT_TABLE_POW2 + (MT_TABLE_M1 - MT_TABLE_M0 + 1) * MT_TABLE_SHIFTS;   // 1792
const MtPoly *mt19937_table();                    // MT_TABLE_ENTRIES records, or nullptr (no file / hook PRAND_MT_POLY=host)
int mt19937_table_index(Dist v);                  // record of x^v, or -1 if v is not of a tabulated form
// v as a sum of tabulated distances (binary decomposition of the mantissa): record indices in
// `idx`; false if some term is not tabulated (2^n with n >= 512)
bool mt19937_table_terms(Dist v, std::vector<int> &idx);
void mt19937_levels(Dist n, unsigned levels, std::vector<MtPoly> &out);
void mt19937_to_op(const MtPoly &p, MtOp &op);                       // repack as 32-bit words
void mt19937_seed_state(uint32_t seed, uint32_t *w624);              // ref.-[2] initialiser

}  // namespace host
}  // namespace prand
