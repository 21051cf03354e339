/* prand_device_gm.cuh -- the GM/GQ torus-ensemble generators' step and output functions
 * (eq. 1, Table 2, Table 5; readings G1-G3
 * and section 6.4).  Included by prand_device.cuh (device-callable API) and by libprand's bulk kernels
 * (paper_1307_5869_b200/csrc/k_gmgq.cu): one definition of the arithmetic for both.
 * Product code: shares nothing with oracle/.
 */
#pragma once
#include <stdint.h>
#include "prand.h"
#include "prand_ops.h"

namespace prand_dev {

/* ---- skip-ahead: 2x2 companion-matrix powers mod g, Barrett reduction ----------
 * g < 2^61; mu = floor(2^(2 nb) / g) with nb = bit length of g. */
struct Barrett { uint64_t g, mu; unsigned nb; };

__host__ __device__ constexpr unsigned gm_bit_length(uint64_t x) { return x ? 1u + gm_bit_length(x >> 1) : 0u; }
__host__ __device__ constexpr Barrett gm_barrett(uint64_t g)
{
    return Barrett{g, (uint64_t)((((unsigned __int128)1) << (2 * gm_bit_length(g))) / g), gm_bit_length(g)};
}
__device__ __forceinline__ uint64_t bmulmod(uint64_t a, uint64_t b, const Barrett &B)
{
    uint64_t lo = a * b, hi = __umul64hi(a, b);                      // x = a b < g^2 < 2^(2 nb)
    uint64_t q1 = (hi << (65 - B.nb)) | (lo >> (B.nb - 1));          // x >> (nb-1) < 2^(nb+1)
    uint64_t l2 = q1 * B.mu, h2 = __umul64hi(q1, B.mu);
    uint64_t q3 = (h2 << (63 - B.nb)) | (l2 >> (B.nb + 1));          // floor(q1 mu / 2^(nb+1))
    uint64_t r = lo - q3 * B.g;                                      // 0 <= x - q3 g < 3 g < 2^64
    while (r >= B.g) r -= B.g;
    return r;
}
__device__ __forceinline__ uint64_t baddmod(uint64_t a, uint64_t b, const Barrett &B)
{
    uint64_t t = a + b;                                              // < 2^62
    return t >= B.g ? t - B.g : t;
}
// (xN, xP) <- product of ops[b] over the set bits b of idx, applied to the column (x(n), x(n-1)).
// noinline: callers invoke it once per register-resident point (static indexing keeps the ensemble
// out of local memory) and it is cold
static __device__ __noinline__ void gm_apply_bits(const prand_gm_op *__restrict__ ops, uint64_t idx, uint64_t &xP,
                                           uint64_t &xN, const Barrett &B)
{
    for (int lev = 0; idx != 0; lev++, idx >>= 1)
        if (idx & 1) {
            uint64_t m0 = __ldg(&ops[lev].m[0]), m1 = __ldg(&ops[lev].m[1]);
            uint64_t m2 = __ldg(&ops[lev].m[2]), m3 = __ldg(&ops[lev].m[3]);
            uint64_t n = baddmod(bmulmod(m0, xN, B), bmulmod(m1, xP, B), B);
            uint64_t o = baddmod(bmulmod(m2, xN, B), bmulmod(m3, xP, B), B);
            xN = n; xP = o;
        }
}

// Traits of one generator.  W = canonical state word in HBM (a residue mod g), R = the word the
// generation loop keeps in registers, load/store convert between them at the ends of a call.
//   step(xP, xN) -> the new point k xN - q xP (mod g), canonical in the R representation
//   pack<J>(word, x): word |= digit(x) << bitpos(J); GM61 instead shifts the accumulator (points are
//   fed in descending order there, PACK_DESCENDING)
// The B200 has two integer pipes of 64 lanes/clk/SM each: the ALU pipe (LOP3, SHF, IADD3, VIMNMX,
// LEA, ISETP) and the FMA-heavy pipe (IMAD 1 slot, IMAD.WIDE / IMAD.HI 2 slots).  Every step below is
// arranged so that the negation, the fold of the high part (r = t - (t >> b) p is one IMAD) and
// where possible the packing run on the FMA pipe; DESIGN.md 6.4 lists the per-point counts.
template <int GEN> struct Gm;

__device__ __forceinline__ uint32_t umin_sub(uint32_t r, uint32_t g) { return min(r, r - g); }   // r < 2g -> r mod g
// word + (d << sh) as one multiply-add (FMA pipe) instead of a shift, a mask and an add (ALU pipe)
__device__ __forceinline__ uint32_t pack_mad(uint32_t word, uint32_t d, const int sh)
{
    uint32_t r;
    asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(r) : "r"(d), "r"(1u << sh), "r"(word));
    return r;
}

template <> struct Gm<PRAND_GM19> {
    typedef uint32_t W;
    typedef uint32_t R;
    static constexpr int S = 32;
    static constexpr bool PACK_DESCENDING = false, NEEDS_CLEAN = false, HAS_FAST = false;
    static constexpr uint32_t G = (1u << 19) - 1;
    static constexpr uint64_t MODULUS = G;
    __device__ static __forceinline__ R load(W x) { return x; }
    __device__ static __forceinline__ W store(R x) { return x; }
    __device__ static __forceinline__ R step(R xP, R xN)
    {
        uint32_t t = xP * (0u - 28u) + 28u * G;            // 28 (g - xP)
        t = xN * 15u + t;                                  // < 43 * 2^19
        uint32_t r = (t >> 19) * (0u - G) + t;             // t - (t >> 19) g = (t & g) + (t >> 19) < 2^19 + 43
        return umin_sub(r, G);
    }
    __device__ static __forceinline__ void pack(uint32_t &word, R x, const int J) { word = pack_mad(word, x >> 18, J); }
};

static __constant__ uint32_t gm29_c[3] = {0u - 2u, 2u * ((1u << 29) - 3), 4u};

template <> struct Gm<PRAND_GM29> {
    typedef uint32_t W;
    typedef uint32_t R;
    static constexpr int S = 32;
    static constexpr bool PACK_DESCENDING = false, NEEDS_CLEAN = false, HAS_FAST = false;
    static constexpr uint32_t G = (1u << 29) - 3;
    static constexpr uint64_t MODULUS = G;
    __device__ static __forceinline__ R load(W x) { return x; }
    __device__ static __forceinline__ W store(R x) { return x; }
    __device__ static __forceinline__ R step(R xP, R xN)
    {
        // multipliers from constant memory: two IMADs (as literals the compiler turns them into three
        // shift/add instructions)
        uint32_t t = xP * gm29_c[0] + gm29_c[1];           // 2 (g - xP)
        t = xN * gm29_c[2] + t;                            // + 4 xN < 6 g < 2^32
        uint32_t r = (t >> 29) * (0u - G) + t;             // 2^29 = 3 (mod g): (t & (2^29-1)) + 3 (t >> 29) < 2^29 + 15
        return umin_sub(r, G);
    }
    // floor(2x/g) = [2x >= 2^29 - 3] = [x >= 2^28 - 1]: not a plain shift of x
    __device__ static __forceinline__ void pack(uint32_t &word, R x, const int J)
    {
        word = pack_mad(word, (x + 1u) >> 28, J);
    }
};

template <> struct Gm<PRAND_GM31> {
    typedef uint32_t W;
    typedef uint32_t R;
    static constexpr int S = 32;
    static constexpr bool PACK_DESCENDING = false, NEEDS_CLEAN = false, HAS_FAST = false;
    static constexpr uint32_t G = (1u << 31) - 1;
    static constexpr uint64_t MODULUS = G;
    __device__ static __forceinline__ R load(W x) { return x; }
    __device__ static __forceinline__ W store(R x) { return x; }
    __device__ static __forceinline__ R step(R xP, R xN)
    {
        // t = 11 xN + 14 (g - xP) < 25 * 2^31: g - xP = xP ^ g (g is all ones), two chained 32x32+64
        // multiply-adds (a 64-bit constant addend would cost two more adds)
        const uint64_t t = (uint64_t)(xP ^ G) * 14u + (uint64_t)xN * 11u;
        uint32_t h = (uint32_t)(t >> 31);                  // < 25
        uint32_t r = h * 0x80000001u + (uint32_t)t;        // lo - h 2^31 + h = (t & g) + (t >> 31) < 2^31 + 25
        return umin_sub(r, G);
    }
    __device__ static __forceinline__ void pack(uint32_t &word, R x, const int J) { word = pack_mad(word, x >> 30, J); }
};

// GM61: the register word is X = 8 x (the 61-bit residue in the top bits of a 64-bit word), i.e.
// arithmetic mod M = 8 g = 2^64 - 8.  Then T = 24 XN + 74 (M - XP) < 98 * 2^64 is a 3-limb number
// whose top limb A is t >> 61 and whose low 64 bits are 8 (t mod 2^61) with no shift or mask, and
// 2^64 = 8 (mod M): X' = lo64 + 8 A, minus M if that reaches M.  S = lo64 + 8 A + 8 carries out of 64
// bits exactly when X' >= M, and then S mod 2^64 = X' - M; otherwise X' = S - 8.  M - XP = ~XP with the
// three low bits cleared (two LOP3); the digit (bit 60 of x) is bit 63 of X, shifted into the output
// word by one funnel shift.
static __constant__ uint32_t gm61_eight[1] = {8u};        // from constant memory: keeps 8 A an IMAD (FMA pipe)

template <> struct Gm<PRAND_GM61> {
    typedef uint64_t W;
    typedef uint64_t R;
    static constexpr int S = 32;
    static constexpr bool PACK_DESCENDING = true, NEEDS_CLEAN = false, HAS_FAST = true;
    static constexpr uint64_t MODULUS = (1ull << 61) - 1;
    __device__ static __forceinline__ R load(W x) { return x << 3; }
    __device__ static __forceinline__ W store(R x) { return x >> 3; }
    __device__ static __forceinline__ R step(R XP, R XN)
    {
        uint64_t S;
        asm("{\n\t.reg .u32 pl, ph, nl, nh, yl, yh, c0l, c0h, c1l, c1h, a8, sl, sh, cy;\n\t"
            ".reg .u64 c0, c1;\n\t.reg .pred p;\n\t"
            "mov.b64 {pl, ph}, %1;\n\t"
            "mov.b64 {nl, nh}, %2;\n\t"
            "xor.b32 yl, pl, 0xFFFFFFF8;\n\t"             // M - XP = ~XP with the low three bits cleared
            "not.b32 yh, ph;\n\t"
            "mul.wide.u32 c0, nl, 24;\n\t"
            "mad.wide.u32 c0, yl, 74, c0;\n\t"            // < 98 * 2^32
            "mov.b64 {c0l, c0h}, c0;\n\t"
            "mov.b64 c1, {c0h, 0};\n\t"
            "mad.wide.u32 c1, nh, 24, c1;\n\t"
            "mad.wide.u32 c1, yh, 74, c1;\n\t"            // top limb A < 98
            "mov.b64 {c1l, c1h}, c1;\n\t"
            "mad.lo.u32 a8, c1h, 8, 8;\n\t"
            "add.cc.u32 sl, c0l, a8;\n\t"
            "addc.cc.u32 sh, c1l, 0;\n\t"
            "addc.u32 cy, 0, 0;\n\t"
            "setp.eq.u32 p, cy, 0;\n\t"
            "@p sub.cc.u32 sl, sl, 8;\n\t"
            "@p subc.u32 sh, sh, 0;\n\t"
            "mov.b64 %0, {sl, sh};\n\t}"
            : "=l"(S) : "l"(XP), "l"(XN));
        return S;
    }
    // Optimistic form of the same step for the bulk kernels: X' = lo64 + 8 A without the test against
    // M.  If the middle limb c1l of T is at most 2^32 - 3, the sum neither carries out of 64 bits nor
    // reaches M, so the result is already canonical; otherwise (probability 2^-31 per point) the
    // caller must discard it and call step().  `watch` collects the maximum of c1l over a group of points.
    __device__ static __forceinline__ R step_fast(R XP, R XN, uint32_t &watch)
    {
        uint64_t S;
        uint32_t mid;
        asm("{\n\t.reg .u32 pl, ph, nl, nh, yl, yh, c0l, c0h, c1l, c1h, a8, sl, sh;\n\t"
            ".reg .u64 c0, c1;\n\t"
            "mov.b64 {pl, ph}, %2;\n\t"
            "mov.b64 {nl, nh}, %3;\n\t"
            "xor.b32 yl, pl, 0xFFFFFFF8;\n\t"
            "not.b32 yh, ph;\n\t"
            "mul.wide.u32 c0, nl, 24;\n\t"
            "mad.wide.u32 c0, yl, 74, c0;\n\t"
            "mov.b64 {c0l, c0h}, c0;\n\t"
            "mov.b64 c1, {c0h, 0};\n\t"
            "mad.wide.u32 c1, nh, 24, c1;\n\t"
            "mad.wide.u32 c1, yh, 74, c1;\n\t"
            "mov.b64 {c1l, c1h}, c1;\n\t"
            "mul.lo.u32 a8, c1h, %4;\n\t"
            "add.cc.u32 sl, c0l, a8;\n\t"
            "addc.u32 sh, c1l, 0;\n\t"
            "mov.b64 %0, {sl, sh};\n\t"
            "mov.u32 %1, c1l;\n\t}"
            : "=l"(S), "=r"(mid) : "l"(XP), "l"(XN), "r"(gm61_eight[0]));
        watch = max(watch, mid);
        return S;
    }
    static constexpr uint32_t WATCH_LIMIT = 0xFFFFFFFEu;      // watch >= limit: redo the group with step()
    __device__ static __forceinline__ void pack(uint32_t &word, R X, const int J)
    {
        word = __funnelshift_l((uint32_t)(X >> 32), word, 1);     // (word << 1) | bit 63 of X
    }
};

// g = 2^t p (GM55: 16 (2^51 - 129); GQ58: 2^29 (2^29 - 3)).  k and q are multiples of 2^3 resp. 2^4,
// so every point of the orbit is a multiple of 2^t after at most 16 steps (GM55: one step), and for
// such states x = 2^t y the recurrence is y' = k y - q y' (mod p) and floor(2^v x / g) =
// floor(2^v y / p): the hot loop works on y.  Stream initialisation places every point at least 2^32
// steps into its orbit, so the states the library creates are always of this form ("clean");
// the library runs them only on such states;  for imported states that are not, and those run the plain mod-g
// traits GmPlain<> until they have advanced 16 steps.

// GM55: register word Y = 2^13 y (the 51-bit residue mod p in the top bits), arithmetic mod
// M = 2^13 p = 2^64 - C, C = 129 * 2^13, exactly as for GM61.
// The multipliers are read from constant memory so that the compiler keeps 256 * YN as a 32x32+64
// multiply-add on the FMA pipe instead of a chain of 64-bit shifts and masks on the ALU pipe.
static __constant__ uint32_t gm55_kq[3] = {256u, 176u, 129u << 13};

template <> struct Gm<PRAND_GM55> {
    typedef uint64_t W;
    typedef uint64_t R;
    static constexpr int S = 8;
    static constexpr bool PACK_DESCENDING = false, NEEDS_CLEAN = true, HAS_FAST = true;
    static constexpr uint32_t WATCH_LIMIT = 0xFFFFFFFEu;
    static constexpr uint32_t C = 129u << 13;
    static constexpr uint64_t M = 0ull - C;
    __device__ static __forceinline__ R load(W x) { return x << 9; }               // x = 16 y
    __device__ static __forceinline__ W store(R Y) { return (Y >> 13) << 4; }
    __device__ static __forceinline__ R step(R YP, R YN)
    {
        const uint32_t K = gm55_kq[0], Q = gm55_kq[1];
        const uint64_t D = M - YP;
        const uint32_t dl = (uint32_t)D, dh = (uint32_t)(D >> 32);
        const uint32_t nl = (uint32_t)YN, nh = (uint32_t)(YN >> 32);
        uint64_t c0 = (uint64_t)nl * K + (uint64_t)dl * Q;                           // < 432 * 2^32
        uint64_t c1 = (uint64_t)nh * K + (c0 >> 32);
        c1 = (uint64_t)dh * Q + c1;                                                  // top limb A < 432
        const uint32_t ac = (uint32_t)(c1 >> 32) * C + C;                            // (A + 1) C < 2^29
        uint32_t sl, sh, cy;
        asm("add.cc.u32 %0, %3, %4;\n\t"
            "addc.cc.u32 %1, %5, 0;\n\t"
            "addc.u32 %2, 0, 0;"
            : "=r"(sl), "=r"(sh), "=r"(cy) : "r"((uint32_t)c0), "r"(ac), "r"((uint32_t)c1));
        uint64_t Sx = ((uint64_t)sh << 32) | sl;
        if (cy == 0) Sx -= C;
        return Sx;
    }
    // Optimistic form (see GM61): Y' = lo64 + A C is canonical whenever the middle limb of T is at most
    // 2^32 - 3; `watch` collects the maximum of that limb, the caller falls back to step() otherwise.
    __device__ static __forceinline__ R step_fast(R YP, R YN, uint32_t &watch)
    {
        const uint32_t K = gm55_kq[0], Q = gm55_kq[1];
        const uint64_t D = M - YP;
        const uint32_t dl = (uint32_t)D, dh = (uint32_t)(D >> 32);
        const uint32_t nl = (uint32_t)YN, nh = (uint32_t)(YN >> 32);
        uint64_t c0 = (uint64_t)nl * K + (uint64_t)dl * Q;
        uint64_t c1 = (uint64_t)nh * K + (c0 >> 32);
        c1 = (uint64_t)dh * Q + c1;
        watch = max(watch, (uint32_t)c1);
        const uint64_t lo64 = (c1 << 32) | (uint32_t)c0;
        return lo64 + (uint64_t)((uint32_t)(c1 >> 32) * gm55_kq[2]);
    }
    // floor(16 y / p) = floor(16 Y / M): with h = Y >> 60, 16 Y = h 2^64 + L = h M + (h C + L), so the
    // digit is h + [L + (h + 1) C >= 2^64] = floor((16 Y + (h + 1) C) / 2^64) = (Y + (h + 1) C / 16) >> 60
    __device__ static __forceinline__ void pack(uint32_t &word, R Y, const int J)
    {
        const uint32_t h = (uint32_t)(Y >> 60);
        const uint64_t t = Y + (uint64_t)(h * (C / 16) + (C / 16));
        word = pack_mad(word, (uint32_t)(t >> 60), 4 * J);
    }
};

template <int VB, int SS> struct Gq58 {
    typedef uint64_t W;
    typedef uint32_t R;
    static constexpr int S = SS;
    static constexpr bool PACK_DESCENDING = false, NEEDS_CLEAN = true, HAS_FAST = false;
    static constexpr uint32_t P = (1u << 29) - 3;
    __device__ static __forceinline__ R load(W x) { return (uint32_t)(x >> 29); }  // x = 2^29 y
    __device__ static __forceinline__ W store(R y) { return (uint64_t)y << 29; }
    __device__ static __forceinline__ R step(R yP, R yN)
    {
        uint32_t u = yP * (0u - 6u) + yN + 6u * P;         // yN + 6 (p - yP) in (0, 7 p)
        uint32_t h = u >> 26;                              // (8 u) >> 29 < 56
        uint32_t r = h * (0u - P) + (u << 3);              // (8 u mod 2^29) + 3 h < 2^29 + 168
        return umin_sub(r, P);
    }
    // floor(2 y / p) = [y >= 2^28 - 1]
    __device__ static __forceinline__ uint32_t digit1(R y) { return (y + 1u) >> 28; }
    // floor(2^v y / p), N = 2^v y = h 2^29 + l = h p + (3 h + l): h plus one possible carry
    __device__ static __forceinline__ uint32_t digit3(R y)
    {
        uint32_t h = y >> 26;
        return (h * 3u + (y * 8u + 3u)) >> 29;             // N < 2^32
    }
    __device__ static __forceinline__ uint32_t digit4(R y)
    {
        uint32_t h = y >> 25;
        uint32_t l3 = (y * 16u + 3u) & ((1u << 29) - 1);   // (N mod 2^29) + 3
        return h + ((h * 3u + l3) >> 29);
    }
    __device__ static __forceinline__ void pack(uint32_t &word, R y, const int J)
    {
        if (VB == 1) word += digit1(y) << J;
        else if (VB == 4) word += digit4(y) << (4 * J);
        else if (J < 10) word += digit3(y) << (3 * J);     // GQ58.3: ten 3-bit digits, then two 1-bit digits
        else word += digit1(y) << (20 + J);
    }
};
template <> struct Gm<PRAND_GQ58_1> : Gq58<1, 32> {};
template <> struct Gm<PRAND_GQ58_3> : Gq58<3, 12> {};
template <> struct Gm<PRAND_GQ58_4> : Gq58<4, 8> {};

// ---- plain mod-g traits for states that are not (yet) multiples of 2^t ------------------------------
template <int GEN> struct GmPlain;

template <> struct GmPlain<PRAND_GM55> {
    typedef uint64_t W;
    typedef uint64_t R;
    static constexpr int S = 8;
    static constexpr bool PACK_DESCENDING = false, NEEDS_CLEAN = false, HAS_FAST = false;
    static constexpr uint64_t P = (1ull << 51) - 129;
    static constexpr uint64_t G = 16ull * P;
    static constexpr uint64_t MODULUS = G;
    __device__ static __forceinline__ R load(W x) { return x; }
    __device__ static __forceinline__ W store(R x) { return x; }
    __device__ static __forceinline__ R step(R xP, R xN)
    {
        uint64_t t = 256ull * xN + 176ull * (G - xP);      // < 432 * 2^55 < 2^64
        uint64_t u = t >> 4;                               // t mod 16p = 16 (u mod p) + (t & 15)
        uint64_t r = (u & ((1ull << 51) - 1)) + 129ull * (u >> 51);   // 2^51 = 129 (mod p); r < 2p
        r = r >= P ? r - P : r;
        return (r << 4) | (t & 15ull);
    }
    // floor(16x/g) = floor(x/p): with h = x >> 51, x = h p + (129 h + low), one possible carry
    __device__ static __forceinline__ void pack(uint32_t &word, R x, const int J)
    {
        uint64_t h = x >> 51;
        word |= (uint32_t)((x + 129ull * (h + 1)) >> 51) << (4 * J);
    }
};

template <int VB, int SS> struct Gq58Plain {
    typedef uint64_t W;
    typedef uint64_t R;
    static constexpr int S = SS;
    static constexpr bool PACK_DESCENDING = false, NEEDS_CLEAN = false, HAS_FAST = false;
    static constexpr uint64_t P = (1ull << 29) - 3;
    static constexpr uint64_t G = P << 29;
    static constexpr uint64_t MODULUS = G;
    __device__ static __forceinline__ R load(W x) { return x; }
    __device__ static __forceinline__ W store(R x) { return x; }
    __device__ static __forceinline__ R step(R xP, R xN)
    {
        uint64_t t = 8ull * xN + 48ull * (G - xP);         // < 56 * 2^58 < 2^64
        uint32_t low = (uint32_t)t & ((1u << 29) - 1);     // t mod 2^29 p = 2^29 (u mod p) + low
        uint64_t u = t >> 29;                              // < 2^35
        uint32_t r = ((uint32_t)u & ((1u << 29) - 1)) + 3u * (uint32_t)(u >> 29);   // < 2^29 + 168 < 2p
        r = min(r, r - (uint32_t)P);
        return ((uint64_t)r << 29) | low;
    }
    // floor(2^v x / g) = floor(N / p), N = x >> (29 - v) < 2^v p; h = N >> 29, one possible carry
    __device__ static __forceinline__ uint32_t digit(R x, int v)
    {
        uint64_t N = x >> (29 - v);
        uint64_t h = N >> 29;
        return (uint32_t)((N + 3ull * (h + 1ull)) >> 29);
    }
    __device__ static __forceinline__ void pack(uint32_t &word, R x, const int J)
    {
        if (VB == 1) word |= digit(x, 1) << J;
        else if (VB == 4) word |= digit(x, 4) << (4 * J);
        else if (J < 10) word |= digit(x, 3) << (3 * J);
        else word |= digit(x, 1) << (20 + J);
    }
};
template <> struct GmPlain<PRAND_GQ58_1> : Gq58Plain<1, 32> {};
template <> struct GmPlain<PRAND_GQ58_3> : Gq58Plain<3, 12> {};
template <> struct GmPlain<PRAND_GQ58_4> : Gq58Plain<4, 8> {};

/* ---- device-callable wrappers: all s points of one stream in the calling thread ------------------- */
template <class Tr> struct GmGen {
    typedef typename Tr::W W;
    typename Tr::R xP[Tr::S], xN[Tr::S];
    __device__ void load(const void *base, uint64_t ns, uint64_t s)
    {
        const W *b = static_cast<const W *>(base);
#pragma unroll
        for (int i = 0; i < Tr::S; i++) {
            xP[i] = Tr::load(b[(uint64_t)(2 * i) * ns + s]);
            xN[i] = Tr::load(b[(uint64_t)(2 * i + 1) * ns + s]);
        }
    }
    __device__ void store(void *base, uint64_t ns, uint64_t s) const
    {
        W *b = static_cast<W *>(base);
#pragma unroll
        for (int i = 0; i < Tr::S; i++) {
            b[(uint64_t)(2 * i) * ns + s] = Tr::store(xP[i]);
            b[(uint64_t)(2 * i + 1) * ns + s] = Tr::store(xN[i]);
        }
    }
    /* every ensemble point advanced by idx * dist (ops from prand_device_ops(dist, levels)) */
    __device__ void skipahead(const prand_gm_op *ops, uint64_t idx)
    {
        const Barrett B = gm_barrett(Tr::MODULUS);
#pragma unroll
        for (int i = 0; i < Tr::S; i++) {
            uint64_t a = Tr::store(xP[i]), b = Tr::store(xN[i]);
            gm_apply_bits(ops, idx, a, b, B);
            xP[i] = Tr::load((W)a);
            xN[i] = Tr::load((W)b);
        }
    }
    __device__ uint32_t next_u32()
    {
        uint32_t word = 0;
#pragma unroll
        for (int jj = 0; jj < Tr::S; jj++) {
            const int j = Tr::PACK_DESCENDING ? Tr::S - 1 - jj : jj;
            const typename Tr::R nw = Tr::step(xP[j], xN[j]);
            xP[j] = xN[j];
            xN[j] = nw;
            Tr::pack(word, nw, j);
        }
        return word;
    }
    __device__ float next_f32() { return __uint2float_rn(next_u32() >> 8) * 5.9604644775390625e-08f; }
    __device__ double next_f64() { return __hiloint2double(0x41300000, (int)next_u32()) - 1048576.0; }
};
template <int GEN> struct Gen;
template <> struct Gen<PRAND_GM19> : GmGen<Gm<PRAND_GM19> > {};
template <> struct Gen<PRAND_GM29> : GmGen<Gm<PRAND_GM29> > {};
template <> struct Gen<PRAND_GM31> : GmGen<Gm<PRAND_GM31> > {};
template <> struct Gen<PRAND_GM61> : GmGen<Gm<PRAND_GM61> > {};
/* g = 2^t p: a user's state may be inside the 2-adic transient, so the plain mod-g forms */
template <> struct Gen<PRAND_GM55> : GmGen<GmPlain<PRAND_GM55> > {};
template <> struct Gen<PRAND_GQ58_1> : GmGen<GmPlain<PRAND_GQ58_1> > {};
template <> struct Gen<PRAND_GQ58_3> : GmGen<GmPlain<PRAND_GQ58_3> > {};
template <> struct Gen<PRAND_GQ58_4> : GmGen<GmPlain<PRAND_GQ58_4> > {};

}  /* namespace prand_dev */
