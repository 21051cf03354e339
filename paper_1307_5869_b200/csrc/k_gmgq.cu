// k_gmgq.cu -- GM19/29/31/55/61 and GQ58.1/3/4 jump and generation kernels
// (SURVEY.md 8(a) a1, a2, a6, a7, a8).
//
// PAPER.md:281-284 (eq. 1): x_i(n) = k x_i(n-1) - q x_i(n-2) (mod g), i = 0..s-1, an ensemble of s
// torus points; parameters (k, q, g, v) from Table 2, ensemble sizes from Table 5
// (PAPER.md:390-397).  Output (reading G2): after the step point i contributes the digit
// floor(2^v x_i / g) at bits v*i.. (GQ58.3: points 0..9 three bits, points 10, 11 one bit at 30, 31).
// Jump-ahead: powers of the companion matrix mod g (GmOp), reduced with Barrett's method here.
// State layout (SoA): word (2*i + h) of stream s at st[(2*i + h) * n_streams + s], h = 0: x_i(n-1)
// ("xP"), h = 1: x_i(n) ("xN"); u32 words for g < 2^32, u64 otherwise.
//
// Every modular step below exploits the shape of g (Mersenne, pseudo-Mersenne, or 2^t times such a
// prime) so that no division is executed in the hot loop; the digit is an exact floor computed from
// the same shape (derivations in DESIGN.md section "GM/GQ arithmetic").
#include <cstdlib>
#include <type_traits>
#include "k_common.cuh"

namespace prand {
namespace {

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
    static constexpr bool PACK_DESCENDING = false, NEEDS_CLEAN = false;
    static constexpr uint32_t G = (1u << 19) - 1;
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

template <> struct Gm<PRAND_GM29> {
    typedef uint32_t W;
    typedef uint32_t R;
    static constexpr int S = 32;
    static constexpr bool PACK_DESCENDING = false, NEEDS_CLEAN = false;
    static constexpr uint32_t G = (1u << 29) - 3;
    __device__ static __forceinline__ R load(W x) { return x; }
    __device__ static __forceinline__ W store(R x) { return x; }
    __device__ static __forceinline__ R step(R xP, R xN)
    {
        uint32_t t = xP * (0u - 2u) + 2u * G;
        t = xN * 4u + t;                                   // < 6 g < 2^32
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
    static constexpr bool PACK_DESCENDING = false, NEEDS_CLEAN = false;
    static constexpr uint32_t G = (1u << 31) - 1;
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
template <> struct Gm<PRAND_GM61> {
    typedef uint64_t W;
    typedef uint64_t R;
    static constexpr int S = 32;
    static constexpr bool PACK_DESCENDING = true, NEEDS_CLEAN = false;
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
// GmArgs::clean is false only for imported states that are not, and those run the plain mod-g
// traits GmPlain<> until they have advanced 16 steps.

// GM55: register word Y = 2^13 y (the 51-bit residue mod p in the top bits), arithmetic mod
// M = 2^13 p = 2^64 - C, C = 129 * 2^13, exactly as for GM61.
template <> struct Gm<PRAND_GM55> {
    typedef uint64_t W;
    typedef uint64_t R;
    static constexpr int S = 8;
    static constexpr bool PACK_DESCENDING = false, NEEDS_CLEAN = true;
    static constexpr uint32_t C = 129u << 13;
    static constexpr uint64_t M = 0ull - C;
    __device__ static __forceinline__ R load(W x) { return x << 9; }               // x = 16 y
    __device__ static __forceinline__ W store(R Y) { return (Y >> 13) << 4; }
    __device__ static __forceinline__ R step(R YP, R YN)
    {
        const uint64_t D = M - YP;
        const uint32_t dl = (uint32_t)D, dh = (uint32_t)(D >> 32);
        const uint32_t nl = (uint32_t)YN, nh = (uint32_t)(YN >> 32);
        uint64_t c0 = (uint64_t)nl * 256u + (uint64_t)dl * 176u;                     // < 432 * 2^32
        uint64_t c1 = (uint64_t)nh * 256u + (c0 >> 32);
        c1 = (uint64_t)dh * 176u + c1;                                               // top limb A < 432
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
    // floor(16 y / p) = floor(16 Y / M): with h = Y >> 60 and L = 16 Y mod 2^64, 16 Y = h M + h C + L,
    // so the digit is h plus the carry out of L + (h + 1) C
    __device__ static __forceinline__ void pack(uint32_t &word, R Y, const int J)
    {
        const uint32_t yl = (uint32_t)Y, yh = (uint32_t)(Y >> 32);
        const uint32_t h = yh >> 28;
        const uint32_t ll = yl << 4, lh = __funnelshift_l(yl, yh, 4);
        const uint32_t hc = h * C + C;
        uint32_t t0, t1, d;
        asm("add.cc.u32 %0, %3, %4;\n\t"
            "addc.cc.u32 %1, %5, 0;\n\t"
            "addc.u32 %2, %6, 0;"
            : "=r"(t0), "=r"(t1), "=r"(d) : "r"(ll), "r"(hc), "r"(lh), "r"(h));
        word += d << (4 * J);
    }
};

template <int VB, int SS> struct Gq58 {
    typedef uint64_t W;
    typedef uint32_t R;
    static constexpr int S = SS;
    static constexpr bool PACK_DESCENDING = false, NEEDS_CLEAN = true;
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
    static constexpr bool PACK_DESCENDING = false, NEEDS_CLEAN = false;
    static constexpr uint64_t P = (1ull << 51) - 129;
    static constexpr uint64_t G = 16ull * P;
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
    static constexpr bool PACK_DESCENDING = false, NEEDS_CLEAN = false;
    static constexpr uint64_t P = (1ull << 29) - 3;
    static constexpr uint64_t G = P << 29;
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

// ---- cold path: Barrett a*b mod g for the jump kernels ------------------------------------------
struct Barrett { uint64_t g, mu; unsigned nb; };

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
// noinline: the generation kernels call it once per register-resident point (static indexing keeps
// the ensemble out of local memory) and it is cold
__device__ __noinline__ void gm_apply_bits(const GmOp *__restrict__ ops, uint64_t idx, uint64_t &xP,
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

// one thread per (stream, point)
template <class W>
__global__ void __launch_bounds__(256)
gm_jump_kernel(const W *__restrict__ base, const W *st_in, W *st_out,
               uint64_t ns, int S, const GmOp *__restrict__ ops, uint64_t idx0, uint64_t idx_stride,
               Barrett B)
{
    uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= ns * (uint64_t)S) return;
    uint64_t pt = t / ns, s = t - pt * ns;
    uint64_t xP, xN;
    if (base) { xP = base[2 * pt]; xN = base[2 * pt + 1]; }
    else { xP = st_in[(2 * pt) * ns + s]; xN = st_in[(2 * pt + 1) * ns + s]; }
    gm_apply_bits(ops, idx0 + s * idx_stride, xP, xN, B);
    st_out[(2 * pt) * ns + s] = (W)xP;
    st_out[(2 * pt + 1) * ns + s] = (W)xN;
}

// Generation.  LP lanes share one stream, each holding S/LP ensemble points in registers.
//   LP = 1: lane = stream; a warp stores 32 adjacent streams of a row (128 B for u32/f32).
//   LP = 2, 4 (one-bit digits only): the partial words are OR-combined with butterfly shuffles; the
//           group then buffers LP rows so that lane q stores row i+q.
template <class Tr, int LP, int DT, int MINB>
__global__ void __launch_bounds__(128, MINB)
gm_gen_kernel(const typename Tr::W *st_in, typename Tr::W *st_out,
              typename OutElem<DT>::type *__restrict__ out, uint64_t ns, uint64_t n, uint64_t chunk_len,
              uint64_t n_chunks, const GmOp *__restrict__ chunk_ops, Barrett B)
{
    typedef typename Tr::W W;
    typedef typename Tr::R R;
    typedef typename OutElem<DT>::type T;
    constexpr int PPL = Tr::S / LP;
    static_assert(Tr::S % LP == 0, "points must divide evenly over lanes");

    const uint64_t lane_id = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int q = (int)(lane_id % LP);
    const uint64_t vs = lane_id / LP;
    const bool valid = vs < ns * n_chunks;
    const uint64_t c = valid ? vs / ns : 0, s = valid ? vs - c * ns : 0;

    R xP[PPL], xN[PPL];
#pragma unroll
    for (int j = 0; j < PPL; j++) {
        int pt = q * PPL + j;
        W a = valid ? st_in[(uint64_t)(2 * pt) * ns + s] : (W)0;
        W b = valid ? st_in[(uint64_t)(2 * pt + 1) * ns + s] : (W)0;
        if (c != 0) {
            uint64_t a64 = a, b64 = b;
            gm_apply_bits(chunk_ops + (c - 1), 1, a64, b64, B);   // operator of c * chunk_len
            a = (W)a64; b = (W)b64;
        }
        xP[j] = Tr::load(a);
        xN[j] = Tr::load(b);
    }
    const uint64_t row0 = valid ? c * chunk_len : 0;
    const uint64_t row1 = valid ? ((row0 + chunk_len < n) ? row0 + chunk_len : n) : 0;

    // One step of all points of this lane -> their packed digits.  The two state arrays swap roles
    // every step (PAR = 0: xA holds x(n-1) and receives x(n+1)) instead of being rotated.
    auto step_word = [&](auto par) -> uint32_t {
        constexpr bool PAR = decltype(par)::value;
        uint32_t word = 0;
#pragma unroll
        for (int jj = 0; jj < PPL; jj++) {
            const int j = Tr::PACK_DESCENDING ? PPL - 1 - jj : jj;
            if (!PAR) { xP[j] = Tr::step(xP[j], xN[j]); Tr::pack(word, xP[j], j); }
            else { xN[j] = Tr::step(xN[j], xP[j]); Tr::pack(word, xN[j], j); }
        }
        return word;
    };
    typedef std::integral_constant<bool, false> Even;
    typedef std::integral_constant<bool, true> Odd;
    bool odd = false;                                        // an odd number of steps so far: roles swapped

    if constexpr (LP == 1) {
        T *p = out + row0 * ns + s;
        uint64_t i = row0;
#pragma unroll 1
        for (; i + 2 <= row1; i += 2) {
            store1(p, convert<DT>(step_word(Even())));
            p += ns;
            store1(p, convert<DT>(step_word(Odd())));
            p += ns;
        }
        if (i < row1) {
            store1(p, convert<DT>(step_word(Even())));
            odd = true;
        }
    } else {
        static_assert(LP == 2 || LP == 4, "LP must be 1, 2 or 4");
        const unsigned gmask = (LP == 4 ? 0xFu : 0x3u) << (threadIdx.x & (32 - LP));
        T *p = out + (row0 + q) * ns + s;
#pragma unroll 1
        for (uint64_t i = row0; i < row1; i += LP) {
            uint32_t keep = 0;
#pragma unroll
            for (int r = 0; r < LP; r++) {
                if (i + r < row1) {                          // uniform within the lane group
                    uint32_t w = (r & 1) ? step_word(Odd()) : step_word(Even());
                    odd = !(r & 1);
                    w <<= q * PPL;
                    w |= __shfl_xor_sync(gmask, w, 1);
                    if (LP == 4) w |= __shfl_xor_sync(gmask, w, 2);
                    if (q == r) keep = w;
                }
            }
            if (i + q < row1) store1(p, convert<DT>(keep));
            p += LP * ns;
        }
    }
    if (odd) {
#pragma unroll
        for (int j = 0; j < PPL; j++) { R tmp = xP[j]; xP[j] = xN[j]; xN[j] = tmp; }
    }
    if (valid && c == n_chunks - 1) {
#pragma unroll
        for (int j = 0; j < PPL; j++) {
            int pt = q * PPL + j;
            st_out[(uint64_t)(2 * pt) * ns + s] = Tr::store(xP[j]);
            st_out[(uint64_t)(2 * pt + 1) * ns + s] = Tr::store(xN[j]);
        }
    }
}

template <class Tr, int LP, int DT, int MINB>
cudaError_t launch_gen(cudaStream_t stream, const GenArgs &a, const Barrett &B)
{
    typedef typename Tr::W W;
    typedef typename OutElem<DT>::type T;
    uint64_t lanes = a.n_streams * a.n_chunks * LP;
    unsigned blocks = (unsigned)ceil_div_u64(lanes, 128);
    gm_gen_kernel<Tr, LP, DT, MINB><<<blocks, 128, 0, stream>>>((const W *)a.st_in, (W *)a.st_out, (T *)a.out,
                                                                a.n_streams, a.n, a.chunk_len, a.n_chunks,
                                                                (const GmOp *)a.chunk_ops, B);
    return cudaGetLastError();
}

template <class Tr, int LP, int MINB = 1>
cudaError_t dispatch_dt(cudaStream_t stream, const GenArgs &a, const Barrett &B)
{
    switch (a.dtype) {
    case DT_U32: return launch_gen<Tr, LP, DT_U32, MINB>(stream, a, B);
    case DT_F32: return launch_gen<Tr, LP, DT_F32, MINB>(stream, a, B);
    default: return launch_gen<Tr, LP, DT_F64, MINB>(stream, a, B);
    }
}

Barrett barrett_of(const GmParams *p) { Barrett B; B.g = p->g; B.mu = p->mu; B.nb = p->nbits; return B; }

}  // namespace

cudaError_t gm_jump(cudaStream_t stream, int gen, const JumpArgs &a, LaunchInfo *li)
{
    const GmParams *p = gm_params(gen);
    if (!p) return cudaErrorInvalidValue;
    Barrett B = barrett_of(p);
    uint64_t threads = a.n_streams * p->s;
    unsigned blocks = (unsigned)ceil_div_u64(threads, 256);
    if (p->wide)
        gm_jump_kernel<uint64_t><<<blocks, 256, 0, stream>>>((const uint64_t *)a.base, (const uint64_t *)a.st_in,
                                                             (uint64_t *)a.st_out, a.n_streams, (int)p->s,
                                                             (const GmOp *)a.ops, a.idx0, a.idx_stride, B);
    else
        gm_jump_kernel<uint32_t><<<blocks, 256, 0, stream>>>((const uint32_t *)a.base, (const uint32_t *)a.st_in,
                                                             (uint32_t *)a.st_out, a.n_streams, (int)p->s,
                                                             (const GmOp *)a.ops, a.idx0, a.idx_stride, B);
    li->kernel = "gm_jump";
    li->launches = 1;
    return cudaGetLastError();
}

cudaError_t gm_generate(cudaStream_t stream, int gen, const GenArgs &a, LaunchInfo *li)
{
    const GmParams *p = gm_params(gen);
    if (!p) return cudaErrorInvalidValue;
    Barrett B = barrett_of(p);
    li->launches = 1;
    int lp = 0;                                              // test / tuning hook: lanes per stream
    if (const char *env = std::getenv("PRAND_GM_LP")) lp = std::atoi(env);
    switch (gen) {
    case PRAND_GM19: li->kernel = "gm19_gen<LP=1>"; return dispatch_dt<Gm<PRAND_GM19>, 1>(stream, a, B);
    case PRAND_GM29: li->kernel = "gm29_gen<LP=1>"; return dispatch_dt<Gm<PRAND_GM29>, 1>(stream, a, B);
    case PRAND_GM31: li->kernel = "gm31_gen<LP=1>"; return dispatch_dt<Gm<PRAND_GM31>, 1>(stream, a, B);
    case PRAND_GM61:
        if (lp == 2) { li->kernel = "gm61_gen<LP=2>"; return dispatch_dt<Gm<PRAND_GM61>, 2>(stream, a, B); }
        if (lp == 4) { li->kernel = "gm61_gen<LP=4>"; return dispatch_dt<Gm<PRAND_GM61>, 4>(stream, a, B); }
        li->kernel = "gm61_gen<LP=1>"; return dispatch_dt<Gm<PRAND_GM61>, 1, 2>(stream, a, B);
    case PRAND_GM55:
        if (!a.clean) { li->kernel = "gm55_gen<plain>"; return dispatch_dt<GmPlain<PRAND_GM55>, 1>(stream, a, B); }
        li->kernel = "gm55_gen<LP=1>"; return dispatch_dt<Gm<PRAND_GM55>, 1>(stream, a, B);
    case PRAND_GQ58_1:
        if (!a.clean) { li->kernel = "gq58.1_gen<plain,LP=4>"; return dispatch_dt<GmPlain<PRAND_GQ58_1>, 4>(stream, a, B); }
        if (lp == 2) { li->kernel = "gq58.1_gen<LP=2>"; return dispatch_dt<Gm<PRAND_GQ58_1>, 2>(stream, a, B); }
        li->kernel = "gq58.1_gen<LP=1>"; return dispatch_dt<Gm<PRAND_GQ58_1>, 1>(stream, a, B);
    case PRAND_GQ58_3:
        if (!a.clean) { li->kernel = "gq58.3_gen<plain>"; return dispatch_dt<GmPlain<PRAND_GQ58_3>, 1>(stream, a, B); }
        li->kernel = "gq58.3_gen<LP=1>"; return dispatch_dt<Gm<PRAND_GQ58_3>, 1>(stream, a, B);
    case PRAND_GQ58_4:
        if (!a.clean) { li->kernel = "gq58.4_gen<plain>"; return dispatch_dt<GmPlain<PRAND_GQ58_4>, 1>(stream, a, B); }
        li->kernel = "gq58.4_gen<LP=1>"; return dispatch_dt<Gm<PRAND_GQ58_4>, 1>(stream, a, B);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace prand
