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
#include "k_common.cuh"

namespace prand {
namespace {

template <int GEN> struct Gm;

template <> struct Gm<PRAND_GM19> {
    typedef uint32_t W;
    static constexpr int S = 32, NDIG = 32;
    static constexpr uint32_t G = (1u << 19) - 1;
    __device__ static __forceinline__ W step(W xP, W xN)
    {
        uint32_t t = 15u * xN + 28u * (G - xP);            // < 43 * 2^19
        uint32_t r = (t & G) + (t >> 19);                  // < 2^19 + 2^6
        return min(r, r - G);                              // r - G wraps unless r >= G
    }
    __device__ static __forceinline__ uint32_t digit(W x, int) { return x >> 18; }
};

template <> struct Gm<PRAND_GM29> {
    typedef uint32_t W;
    static constexpr int S = 32;
    static constexpr uint32_t G = (1u << 29) - 3;
    __device__ static __forceinline__ W step(W xP, W xN)
    {
        uint32_t t = 4u * xN + 2u * (G - xP);              // < 6 g < 2^32
        uint32_t r = (t & ((1u << 29) - 1)) + 3u * (t >> 29);   // 2^29 = 3 (mod g); r < 2^29 + 15
        return min(r, r - G);
    }
    // floor(2x/g) = [2x >= 2^29 - 3] = [x >= 2^28 - 1]: not a plain shift of x
    __device__ static __forceinline__ uint32_t digit(W x, int) { return (x + 1u) >> 28; }
};

template <> struct Gm<PRAND_GM31> {
    typedef uint32_t W;
    static constexpr int S = 32;
    static constexpr uint32_t G = (1u << 31) - 1;
    __device__ static __forceinline__ W step(W xP, W xN)
    {
        uint64_t t = (uint64_t)11u * xN + (uint64_t)14u * (G - xP);   // < 25 * 2^31
        uint32_t r = ((uint32_t)t & G) + (uint32_t)(t >> 31);        // < 2^31 + 25
        return min(r, r - G);
    }
    __device__ static __forceinline__ uint32_t digit(W x, int) { return x >> 30; }
};

template <> struct Gm<PRAND_GM61> {
    typedef uint64_t W;
    static constexpr int S = 32;
    static constexpr uint64_t G = (1ull << 61) - 1;
    __device__ static __forceinline__ W step(W xP, W xN)
    {
        // t = 24 xN + 74 (g - xP) < 98 * 2^61 needs 68 bits: 96-bit column sums of 32-bit limbs
        uint64_t y = G - xP;
        uint64_t c0 = (uint64_t)(uint32_t)xN * 24u + (uint64_t)(uint32_t)y * 74u;
        uint64_t c1 = (uint64_t)(uint32_t)(xN >> 32) * 24u + (uint64_t)(uint32_t)(y >> 32) * 74u + (c0 >> 32);
        uint64_t lo = (c1 << 32) | (uint32_t)c0;           // low 64 bits of t
        uint64_t top = c1 >> 29;                           // t >> 61  (c1 < 2^36)
        uint64_t r = (lo & G) + top;                       // 2^61 = 1 (mod g); r < 2^61 + 2^7
        return r >= G ? r - G : r;
    }
    __device__ static __forceinline__ uint32_t digit(W x, int) { return (uint32_t)(x >> 60); }
};

template <> struct Gm<PRAND_GM55> {
    typedef uint64_t W;
    static constexpr int S = 8;
    static constexpr uint64_t P = (1ull << 51) - 129;
    static constexpr uint64_t G = 16ull * P;
    __device__ static __forceinline__ W step(W xP, W xN)
    {
        uint64_t t = 256ull * xN + 176ull * (G - xP);      // < 432 * 2^55 < 2^64
        uint64_t u = t >> 4;                               // t mod 16p = 16 (u mod p) + (t & 15)
        uint64_t r = (u & ((1ull << 51) - 1)) + 129ull * (u >> 51);   // 2^51 = 129 (mod p); r < 2p
        r = r >= P ? r - P : r;
        return (r << 4) | (t & 15ull);
    }
    // floor(16x/g) = floor(x/p): with h = x >> 51, x = h p + (129 h + low), one possible carry
    __device__ static __forceinline__ uint32_t digit(W x, int)
    {
        uint64_t h = x >> 51;
        return (uint32_t)((x + 129ull * (h + 1)) >> 51);
    }
};

template <int VB, int SS> struct Gq58 {
    typedef uint64_t W;
    static constexpr int S = SS;
    static constexpr uint64_t P = (1ull << 29) - 3;
    static constexpr uint64_t G = P << 29;
    __device__ static __forceinline__ W step(W xP, W xN)
    {
        uint64_t t = 8ull * xN + 48ull * (G - xP);         // < 56 * 2^58 < 2^64
        uint32_t low = (uint32_t)t & ((1u << 29) - 1);     // t mod 2^29 p = 2^29 (u mod p) + low
        uint64_t u = t >> 29;                              // < 2^35
        uint32_t r = ((uint32_t)u & ((1u << 29) - 1)) + 3u * (uint32_t)(u >> 29);   // < 2^29 + 168 < 2p
        r = min(r, r - (uint32_t)P);
        return ((uint64_t)r << 29) | low;
    }
    // floor(2^v x / g) = floor(N / p), N = x >> (29 - v) < 2^v p; h = N >> 29, one possible carry
    __device__ static __forceinline__ uint32_t digit(W x, int v)
    {
        uint32_t N = (uint32_t)(x >> (29 - v));            // < 2^(29+v) <= 2^32 for v <= 3 ...
        uint32_t h = N >> 29;
        return (N + 3u * (h + 1u)) >> 29;
    }
};
// v = 4: N < 16 p needs 33 bits
template <> __device__ __forceinline__ uint32_t Gq58<4, 8>::digit(W x, int)
{
    uint64_t N = x >> 25;
    uint64_t h = N >> 29;
    return (uint32_t)((N + 3ull * (h + 1ull)) >> 29);
}
template <> struct Gm<PRAND_GQ58_1> : Gq58<1, 32> {};
template <> struct Gm<PRAND_GQ58_3> : Gq58<3, 12> {};
template <> struct Gm<PRAND_GQ58_4> : Gq58<4, 8> {};

// digit width and bit position of point i in the output word (reading G2)
template <int GEN> __device__ __forceinline__ constexpr int gm_vbits(int i)
{
    if (GEN == PRAND_GM55 || GEN == PRAND_GQ58_4) return 4;
    if (GEN == PRAND_GQ58_3) return i < 10 ? 3 : 1;
    return 1;
}
template <int GEN> __device__ __forceinline__ constexpr int gm_bitpos(int i)
{
    if (GEN == PRAND_GM55 || GEN == PRAND_GQ58_4) return 4 * i;
    if (GEN == PRAND_GQ58_3) return i < 10 ? 3 * i : 20 + i;
    return i;
}

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
//   LP = 4: the four partial words are OR-combined with two butterfly shuffles; the group then
//           buffers four rows so that lane q stores row i+q (8 adjacent streams = 32 B per row).
template <int GEN, int LP, int DT>
__global__ void __launch_bounds__(128)
gm_gen_kernel(const typename Gm<GEN>::W *st_in, typename Gm<GEN>::W *st_out,
              typename OutElem<DT>::type *__restrict__ out, uint64_t ns, uint64_t n, uint64_t chunk_len,
              uint64_t n_chunks, const GmOp *__restrict__ chunk_ops, Barrett B)
{
    typedef Gm<GEN> Tr;
    typedef typename Tr::W W;
    typedef typename OutElem<DT>::type T;
    constexpr int PPL = Tr::S / LP;
    static_assert(Tr::S % LP == 0, "points must divide evenly over lanes");

    const uint64_t lane_id = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int q = (int)(lane_id % LP);
    const uint64_t vs = lane_id / LP;
    const bool valid = vs < ns * n_chunks;
    const uint64_t c = valid ? vs / ns : 0, s = valid ? vs - c * ns : 0;

    W xP[PPL], xN[PPL];
#pragma unroll
    for (int j = 0; j < PPL; j++) {
        int pt = q * PPL + j;
        xP[j] = valid ? st_in[(uint64_t)(2 * pt) * ns + s] : (W)0;
        xN[j] = valid ? st_in[(uint64_t)(2 * pt + 1) * ns + s] : (W)0;
    }
    if (c != 0) {
#pragma unroll
        for (int j = 0; j < PPL; j++) {
            uint64_t a = xP[j], b = xN[j];
            gm_apply_bits(chunk_ops + (c - 1), 1, a, b, B);   // operator of c * chunk_len
            xP[j] = (W)a; xN[j] = (W)b;
        }
    }
    const uint64_t row0 = valid ? c * chunk_len : 0;
    const uint64_t row1 = valid ? ((row0 + chunk_len < n) ? row0 + chunk_len : n) : 0;

    auto step_word = [&]() -> uint32_t {
        uint32_t word = 0;
#pragma unroll
        for (int j = 0; j < PPL; j++) {
            W nw = Tr::step(xP[j], xN[j]);
            xP[j] = xN[j]; xN[j] = nw;
            if constexpr (LP == 1) {
                word |= Tr::digit(nw, gm_vbits<GEN>(j)) << gm_bitpos<GEN>(j);
            } else {
                word |= Tr::digit(nw, 1) << j;               // LP > 1 only for v = 1 generators
            }
        }
        return word;
    };

    if constexpr (LP == 1) {
        T *p = out + row0 * ns + s;
#pragma unroll 1
        for (uint64_t i = row0; i < row1; i++) {
            store1(p, convert<DT>(step_word()));
            p += ns;
        }
    } else {
        static_assert(LP == 4, "LP must be 1 or 4");
        const unsigned gmask = 0xFu << (threadIdx.x & 28u);
        T *p = out + (row0 + q) * ns + s;
#pragma unroll 1
        for (uint64_t i = row0; i < row1; i += 4) {
            uint32_t keep = 0;
#pragma unroll
            for (int r = 0; r < 4; r++) {
                if (i + r < row1) {                          // uniform within the 4-lane group
                    uint32_t w = step_word() << (q * PPL);
                    w |= __shfl_xor_sync(gmask, w, 1);
                    w |= __shfl_xor_sync(gmask, w, 2);
                    if (q == r) keep = w;
                }
            }
            if (i + q < row1) store1(p, convert<DT>(keep));
            p += 4 * ns;
        }
    }
    if (valid && c == n_chunks - 1) {
#pragma unroll
        for (int j = 0; j < PPL; j++) {
            int pt = q * PPL + j;
            st_out[(uint64_t)(2 * pt) * ns + s] = xP[j];
            st_out[(uint64_t)(2 * pt + 1) * ns + s] = xN[j];
        }
    }
}

template <int GEN, int LP, int DT>
cudaError_t launch_gen(cudaStream_t stream, const GenArgs &a, const Barrett &B)
{
    typedef typename Gm<GEN>::W W;
    typedef typename OutElem<DT>::type T;
    uint64_t lanes = a.n_streams * a.n_chunks * LP;
    unsigned blocks = (unsigned)ceil_div_u64(lanes, 128);
    gm_gen_kernel<GEN, LP, DT><<<blocks, 128, 0, stream>>>((const W *)a.st_in, (W *)a.st_out, (T *)a.out,
                                                          a.n_streams, a.n, a.chunk_len, a.n_chunks,
                                                          (const GmOp *)a.chunk_ops, B);
    return cudaGetLastError();
}

template <int GEN, int LP>
cudaError_t dispatch_dt(cudaStream_t stream, const GenArgs &a, const Barrett &B)
{
    switch (a.dtype) {
    case DT_U32: return launch_gen<GEN, LP, DT_U32>(stream, a, B);
    case DT_F32: return launch_gen<GEN, LP, DT_F32>(stream, a, B);
    default: return launch_gen<GEN, LP, DT_F64>(stream, a, B);
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
    switch (gen) {
    case PRAND_GM19: li->kernel = "gm19_gen<LP=1>"; return dispatch_dt<PRAND_GM19, 1>(stream, a, B);
    case PRAND_GM29: li->kernel = "gm29_gen<LP=1>"; return dispatch_dt<PRAND_GM29, 1>(stream, a, B);
    case PRAND_GM31: li->kernel = "gm31_gen<LP=1>"; return dispatch_dt<PRAND_GM31, 1>(stream, a, B);
    case PRAND_GM55: li->kernel = "gm55_gen<LP=1>"; return dispatch_dt<PRAND_GM55, 1>(stream, a, B);
    case PRAND_GM61: li->kernel = "gm61_gen<LP=4>"; return dispatch_dt<PRAND_GM61, 4>(stream, a, B);
    case PRAND_GQ58_1: li->kernel = "gq58.1_gen<LP=4>"; return dispatch_dt<PRAND_GQ58_1, 4>(stream, a, B);
    case PRAND_GQ58_3: li->kernel = "gq58.3_gen<LP=1>"; return dispatch_dt<PRAND_GQ58_3, 1>(stream, a, B);
    case PRAND_GQ58_4: li->kernel = "gq58.4_gen<LP=1>"; return dispatch_dt<PRAND_GQ58_4, 1>(stream, a, B);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace prand
