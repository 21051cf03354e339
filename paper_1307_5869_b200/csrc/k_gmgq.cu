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
#include "../../include/prand_device_gm.cuh"

namespace prand {
namespace {

// The traits Gm<GEN> / GmPlain<GEN> (state word types, load/store, step, pack) live in
// include/prand_device_gm.cuh: the device-callable API and these bulk kernels share one definition.
using namespace prand_dev;

// ---- cold path: Barrett a*b mod g for the jump kernels ------------------------------------------
// Barrett reduction mod g and the 2x2 skip are the device-callable API's (include/prand_device_gm.cuh)
using prand_dev::Barrett;
using prand_dev::bmulmod;
using prand_dev::baddmod;
using prand_dev::gm_apply_bits;

// one thread per (stream, point)
template <class W>
__global__ void __launch_bounds__(256)
gm_jump_kernel(const W *__restrict__ base, const W *st_in, W *st_out,
               uint64_t ns, int S, const GmOp *__restrict__ ops, uint64_t idx0, uint64_t idx_stride,
               Barrett B, uint64_t count)
{
    uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= count * (uint64_t)S) return;
    uint64_t pt = t / count, s = t - pt * count;
    uint64_t xP, xN;
    if (base) { xP = base[2 * pt]; xN = base[2 * pt + 1]; }
    else { xP = st_in[(2 * pt) * ns + s]; xN = st_in[(2 * pt + 1) * ns + s]; }
    gm_apply_bits(ops, idx0 + s * idx_stride, xP, xN, B);
    st_out[(2 * pt) * ns + s] = (W)xP;
    st_out[(2 * pt + 1) * ns + s] = (W)xN;
}

// Stream initialisation by the paper's relation (eq. 2): for any w,
// x(w + 2n) = k_n x(w + n) - q_n x(w), and block splitting puts stream s at offset s L, so with n = 2^j L
//     state(s) = k_n state(s - 2^j) - q_n state(s - 2^(j+1))        (every state word alike).
// One launch fills streams [s_begin, s_end) from already filled ones: two modular products per word
// instead of one 2x2 matrix product per set bit of the stream index.  One thread per (word, stream).
template <class W>
__global__ void __launch_bounds__(256)
gm_tree_kernel(W *st, uint64_t ns, uint64_t s_begin, uint64_t s_end, uint64_t back, int words, uint64_t kn,
               uint64_t qneg, Barrett B)
{
    const uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const uint64_t count = s_end - s_begin;
    if (t >= count * (uint64_t)words) return;
    const uint64_t w = t / count, s = s_begin + (t - w * count);
    const uint64_t a = st[w * ns + s - back], b = st[w * ns + s - 2 * back];
    st[w * ns + s] = (W)baddmod(bmulmod(kn, a, B), bmulmod(qneg, b, B), B);
}

// Generation.  LP lanes share one stream, each holding S/LP ensemble points in registers.
//   LP = 1: lane = stream; a warp stores 32 adjacent streams of a row (128 B for u32/f32).
//   LP = 2, 4 (one-bit digits only): the partial words are OR-combined with butterfly shuffles; the
//           group then buffers LP rows so that lane q stores row i+q.
template <class Tr, int LP, int DT, int MINB>
__global__ void __launch_bounds__(128, MINB)
gm_gen_kernel(const typename Tr::W *st_in, typename Tr::W *st_out,
              typename OutElem<DT>::type *__restrict__ out, uint64_t ns, uint64_t n, uint64_t chunk_len,
              uint64_t n_chunks, const GmOp *__restrict__ chunk_ops, Barrett B, uint32_t watch_limit)
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
        if constexpr (Tr::HAS_FAST) {
            // optimistic steps in groups of (up to) 8 points; a group whose watch value reaches the
            // limit (probability ~2^-28) is recomputed with the exact step before it is committed
            constexpr int GRP = PPL < 8 ? PPL : 8;
#pragma unroll
            for (int g0 = 0; g0 < PPL; g0 += GRP) {
                R nw[GRP];
                uint32_t watch = 0;
#pragma unroll
                for (int jj = 0; jj < GRP; jj++) {
                    const int j = Tr::PACK_DESCENDING ? PPL - 1 - (g0 + jj) : g0 + jj;
                    nw[jj] = PAR ? Tr::step_fast(xN[j], xP[j], watch) : Tr::step_fast(xP[j], xN[j], watch);
                }
                if (watch >= watch_limit) {
#pragma unroll
                    for (int jj = 0; jj < GRP; jj++) {
                        const int j = Tr::PACK_DESCENDING ? PPL - 1 - (g0 + jj) : g0 + jj;
                        nw[jj] = PAR ? Tr::step(xN[j], xP[j]) : Tr::step(xP[j], xN[j]);
                    }
                }
#pragma unroll
                for (int jj = 0; jj < GRP; jj++) {
                    const int j = Tr::PACK_DESCENDING ? PPL - 1 - (g0 + jj) : g0 + jj;
                    if (!PAR) xP[j] = nw[jj]; else xN[j] = nw[jj];
                    Tr::pack(word, nw[jj], j);
                }
            }
        } else {
#pragma unroll
            for (int jj = 0; jj < PPL; jj++) {
                const int j = Tr::PACK_DESCENDING ? PPL - 1 - jj : jj;
                if (!PAR) { xP[j] = Tr::step(xP[j], xN[j]); Tr::pack(word, xP[j], j); }
                else { xN[j] = Tr::step(xN[j], xP[j]); Tr::pack(word, xN[j], j); }
            }
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

// ---- GM31: some of the 32 points on the FP64 pipe ----------------------------------------------------
// The integer step of GM31 is bound by the FMA-heavy pipe (two half-rate 32x32+64 multiply-adds per
// point) while the FP64 pipe (64 lanes/clk/SM) idles.  NF of the 32 points are therefore kept as
// doubles and stepped there, exactly (g = 2^31 - 1):
//   p = 11 xN + 14 (g - xP) in [0, 25 * 2^31)       two DFMA, integers below 2^36: exact
//   k = floor(p / g) = rint(p * (1/g) - 0.5 + 2^-33)   p/g is an integer or at least 1/g = 2^-31 away from
//                                                   one, the product is off by < 2^-47: the rounding can
//                                                   never go the wrong way; rint as +- 1.5 * 2^52
//   x' = p - k g in [0, g)                          one DFMA, exact and already canonical
// The digit (bit 30) is read from the low mantissa word of x' + 1.5 * 2^52.  Seven FP64 instructions,
// one shift and one multiply-add per point, against four ALU and six FMA-pipe slots for the integer
// step; with NF = 14 the three pipes are about evenly loaded.
template <int NF, int DT>
__global__ void __launch_bounds__(128)
gm31_hybrid_kernel(const uint32_t *st_in, uint32_t *st_out, typename OutElem<DT>::type *__restrict__ out,
                   uint64_t ns, uint64_t n, uint64_t chunk_len, uint64_t n_chunks,
                   const GmOp *__restrict__ chunk_ops, Barrett B)
{
    typedef Gm<PRAND_GM31> Tr;
    typedef typename OutElem<DT>::type T;
    constexpr int NI = 32 - NF;
    constexpr double GD = 2147483647.0, MAGIC = 6755399441055744.0;
    const uint64_t vs = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool valid = vs < ns * n_chunks;
    const uint64_t c = valid ? vs / ns : 0, s = valid ? vs - c * ns : 0;
    double dA[NF], dB[NF];                                  // points 0 .. NF-1
    uint32_t iA[NI], iB[NI];                                // points NF .. 31
#pragma unroll
    for (int j = 0; j < 32; j++) {
        uint32_t a = valid ? st_in[(uint64_t)(2 * j) * ns + s] : 0u;
        uint32_t b = valid ? st_in[(uint64_t)(2 * j + 1) * ns + s] : 0u;
        if (c != 0) {
            uint64_t a64 = a, b64 = b;
            gm_apply_bits(chunk_ops + (c - 1), 1, a64, b64, B);
            a = (uint32_t)a64; b = (uint32_t)b64;
        }
        if (j < NF) { dA[j] = (double)a; dB[j] = (double)b; }
        else { iA[j - NF] = a; iB[j - NF] = b; }
    }
    const uint64_t row0 = valid ? c * chunk_len : 0;
    const uint64_t row1 = valid ? ((row0 + chunk_len < n) ? row0 + chunk_len : n) : 0;

    auto step_d = [&](double xP, double xN, uint32_t &word, const int j) -> double {
        const double t = __fma_rn(-14.0, xP, 14.0 * GD);
        const double p = __fma_rn(11.0, xN, t);
        const double sq = __fma_rn(p, 4.6566128752457969e-10, -0.5 + 1.1641532182693481e-10);   // 1/g, 2^-33
        const double kk = __dadd_rn(__dadd_rn(sq, MAGIC), -MAGIC);
        const double r = __fma_rn(-kk, GD, p);
        const uint32_t v = (uint32_t)__double2loint(__dadd_rn(r, MAGIC));
        word = pack_mad(word, v >> 30, j);
        return r;
    };
    // PAR = false: (A, B) = (x(n-1), x(n)) and A receives x(n+1); PAR = true: roles swapped
    auto step_word = [&](auto par) -> uint32_t {
        constexpr bool PAR = decltype(par)::value;
        uint32_t word = 0;
#pragma unroll
        for (int j = 0; j < 32; j++) {
            if (j < NF) {
                const int q = j < NF ? j : 0;
                if (!PAR) dA[q] = step_d(dA[q], dB[q], word, j); else dB[q] = step_d(dB[q], dA[q], word, j);
            } else {
                const int q = j >= NF ? j - NF : 0;
                if (!PAR) { iA[q] = Tr::step(iA[q], iB[q]); Tr::pack(word, iA[q], j); }
                else { iB[q] = Tr::step(iB[q], iA[q]); Tr::pack(word, iB[q], j); }
            }
        }
        return word;
    };
    T *p = out + row0 * ns + s;
    uint64_t i = row0;
    bool odd = false;
#pragma unroll 1
    for (; i + 2 <= row1; i += 2) {
        store1(p, convert<DT>(step_word(std::false_type())));
        p += ns;
        store1(p, convert<DT>(step_word(std::true_type())));
        p += ns;
    }
    if (i < row1) {
        store1(p, convert<DT>(step_word(std::false_type())));
        odd = true;
    }
    if (valid && c == n_chunks - 1) {
#pragma unroll
        for (int j = 0; j < 32; j++) {
            uint32_t a, b;
            if (j < NF) { a = (uint32_t)__double2uint_rn(dA[j < NF ? j : 0]); b = (uint32_t)__double2uint_rn(dB[j < NF ? j : 0]); }
            else { a = iA[j >= NF ? j - NF : 0]; b = iB[j >= NF ? j - NF : 0]; }
            st_out[(uint64_t)(2 * j) * ns + s] = odd ? b : a;
            st_out[(uint64_t)(2 * j + 1) * ns + s] = odd ? a : b;
        }
    }
}

template <int NF> cudaError_t launch_gm31_hybrid(cudaStream_t stream, const GenArgs &a, const Barrett &B)
{
    const uint64_t lanes = a.n_streams * a.n_chunks;
    const unsigned blocks = (unsigned)ceil_div_u64(lanes, 128);
    const uint32_t *si = (const uint32_t *)a.st_in;
    uint32_t *so = (uint32_t *)a.st_out;
    const GmOp *co = (const GmOp *)a.chunk_ops;
    switch (a.dtype) {
    case DT_U32: gm31_hybrid_kernel<NF, DT_U32><<<blocks, 128, 0, stream>>>(si, so, (uint32_t *)a.out, a.n_streams, a.n, a.chunk_len, a.n_chunks, co, B); break;
    case DT_F32: gm31_hybrid_kernel<NF, DT_F32><<<blocks, 128, 0, stream>>>(si, so, (float *)a.out, a.n_streams, a.n, a.chunk_len, a.n_chunks, co, B); break;
    default: gm31_hybrid_kernel<NF, DT_F64><<<blocks, 128, 0, stream>>>(si, so, (double *)a.out, a.n_streams, a.n, a.chunk_len, a.n_chunks, co, B); break;
    }
    return cudaGetLastError();
}

// Limit of the optimistic steps' watch value (Tr::WATCH_LIMIT); the test hook PRAND_GM_WATCH lowers it
// so that the exact fallback runs often (0: always).
template <class Tr> uint32_t gm_watch_limit()
{
    if constexpr (Tr::HAS_FAST) {
        return debug_hooks().gm_watch_set ? debug_hooks().gm_watch : Tr::WATCH_LIMIT;
    } else {
        return 0xFFFFFFFFu;
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
                                                                (const GmOp *)a.chunk_ops, B, gm_watch_limit<Tr>());
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
    const uint64_t count = a.count ? a.count : a.n_streams;
    uint64_t threads = count * p->s;
    unsigned blocks = (unsigned)ceil_div_u64(threads, 256);
    if (p->wide)
        gm_jump_kernel<uint64_t><<<blocks, 256, 0, stream>>>((const uint64_t *)a.base, (const uint64_t *)a.st_in,
                                                             (uint64_t *)a.st_out, a.n_streams, (int)p->s,
                                                             (const GmOp *)a.ops, a.idx0, a.idx_stride, B, count);
    else
        gm_jump_kernel<uint32_t><<<blocks, 256, 0, stream>>>((const uint32_t *)a.base, (const uint32_t *)a.st_in,
                                                             (uint32_t *)a.st_out, a.n_streams, (int)p->s,
                                                             (const GmOp *)a.ops, a.idx0, a.idx_stride, B, count);
    li->kernel = "gm_jump";
    li->launches = 1;
    return cudaGetLastError();
}

cudaError_t gm_tree_fill(cudaStream_t stream, int gen, void *st, uint64_t ns, uint64_t s_begin, uint64_t s_end,
                         uint64_t back, uint64_t kn, uint64_t qn, LaunchInfo *li)
{
    const GmParams *p = gm_params(gen);
    if (!p) return cudaErrorInvalidValue;
    li->kernel = "gm_tree";
    li->launches = 0;
    if (s_end <= s_begin) return cudaSuccess;
    Barrett B = barrett_of(p);
    const int words = 2 * (int)p->s;
    const uint64_t threads = (s_end - s_begin) * (uint64_t)words;
    const unsigned blocks = (unsigned)ceil_div_u64(threads, 256);
    const uint64_t qneg = (p->g - qn % p->g) % p->g;
    if (p->wide)
        gm_tree_kernel<uint64_t><<<blocks, 256, 0, stream>>>((uint64_t *)st, ns, s_begin, s_end, back, words, kn, qneg, B);
    else
        gm_tree_kernel<uint32_t><<<blocks, 256, 0, stream>>>((uint32_t *)st, ns, s_begin, s_end, back, words, kn, qneg, B);
    li->launches = 1;
    return cudaGetLastError();
}

cudaError_t gm_generate(cudaStream_t stream, int gen, const GenArgs &a, LaunchInfo *li)
{
    const GmParams *p = gm_params(gen);
    if (!p) return cudaErrorInvalidValue;
    Barrett B = barrett_of(p);
    li->launches = 1;
    const int lp = debug_hooks().gm_lp;                      // test / tuning hook: lanes per stream
    switch (gen) {
    case PRAND_GM19: li->kernel = "gm19_gen<LP=1>"; return dispatch_dt<Gm<PRAND_GM19>, 1>(stream, a, B);
    case PRAND_GM29: li->kernel = "gm29_gen<LP=1>"; return dispatch_dt<Gm<PRAND_GM29>, 1>(stream, a, B);
    case PRAND_GM31: {
        const int nf = debug_hooks().gm31_nf < 0 ? 14 : debug_hooks().gm31_nf;   // points on the FP64 pipe (test / tuning hook)
        if (nf == 12) { li->kernel = "gm31_gen<fp64 x12>"; return launch_gm31_hybrid<12>(stream, a, B); }
        if (nf == 14) { li->kernel = "gm31_gen<fp64 x14>"; return launch_gm31_hybrid<14>(stream, a, B); }
        if (nf == 16) { li->kernel = "gm31_gen<fp64 x16>"; return launch_gm31_hybrid<16>(stream, a, B); }
        if (nf == 10) { li->kernel = "gm31_gen<fp64 x10>"; return launch_gm31_hybrid<10>(stream, a, B); }
        li->kernel = "gm31_gen<LP=1>"; return dispatch_dt<Gm<PRAND_GM31>, 1>(stream, a, B);
    }
    case PRAND_GM61:
        if (lp == 1) { li->kernel = "gm61_gen<LP=1>"; return dispatch_dt<Gm<PRAND_GM61>, 1, 2>(stream, a, B); }
        if (lp == 2) { li->kernel = "gm61_gen<LP=2>"; return dispatch_dt<Gm<PRAND_GM61>, 2>(stream, a, B); }
        li->kernel = "gm61_gen<LP=4>"; return dispatch_dt<Gm<PRAND_GM61>, 4>(stream, a, B);
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
