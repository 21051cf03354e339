// k_mt19937.cu -- MT19937 jump-polynomial application and generation kernels
// (SURVEY.md 8(a) a1, a2, a5, a7, a8).
//
// MT19937 (algorithm of the paper's ref. [2]) is linear over F_2, Y_{n+1} = A Y_n;
// jump-ahead is A^v Y_0 = g_v(A) Y_0 = a_k Y_{k-1} + ... + a_1 Y_0, k = 19937 (eq. 10), with
// g_v(x) = x^v mod phi(x).  Recurrence (ref. [2] parameters, reading T1):
//   x_{i+624} = x_{i+397} ^ (y >> 1) ^ (y odd ? 0x9908B0DF : 0),  y = (x_i & 0x80000000) | (x_{i+1} & 0x7FFFFFFF),
// output number P = temper(x_{P+624}); the state at position P is the window x_P..x_{P+623}.
// State layout: [stream][624] u32 (one stream's window is contiguous: a warp loads it coalesced).
#include <cstdlib>
#include <cuda.h>                                         // CUtensorMap (types only: the encoder comes through the runtime)
#include "k_common.cuh"
#include "../../include/prand_device.cuh"

namespace prand {
namespace {

constexpr int NW = 624, MW = 397, DEG = 19937;

using prand_dev::mt_recur;

__device__ __forceinline__ uint32_t xor3(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t d;
    asm("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}

// ---- eq. 10 in correlation form -----------------------------------------------------------------
// One CTA per destination stream runs the device-callable API's CTA-cooperative skip-ahead
// (include/prand_device.cuh, mt19937_skipahead_cta: window extension + position-list accumulation).
constexpr int APPLY_XWORDS = prand_dev::MT_SKIP_XWORDS;     // 20561
constexpr int APPLY_ZERO = APPLY_XWORDS;                    // x[APPLY_ZERO .. +APPLY_ZPAD) = 0
constexpr int APPLY_ZPAD = prand_dev::MT_SKIP_ZPAD;
constexpr size_t APPLY_SMEM = prand_dev::MT_SKIP_WORK_BYTES;

// NT = 256: three output words per thread, two CTAs per SM (throughput: many streams); NT = 640: one
// output word per thread, a third of the loads per thread (latency: the first levels of a doubling tree
// and other launches with fewer CTAs than SMs).
// SPLIT > 1: SPLIT CTAs share one application, each extending the window itself (cheap) and
// accumulating 624 / SPLIT of the output words -- for launches with far fewer applications than SMs
// (the first levels of a doubling tree), where the time of a level is the latency of one application.
// Only for src != dst streams (src_back != 0): the parts of one stream run concurrently.
template <int NT, int SPLIT>
__global__ void __launch_bounds__(NT)
mt19937_apply_kernel(const uint32_t *st_src, uint32_t *st_dst, uint64_t dst0,
                     uint64_t src_back, const MtOp *__restrict__ op)
{
    static_assert(NW % SPLIT == 0, "SPLIT must divide 624");
    constexpr int NOUT = NW / SPLIT;
    extern __shared__ __align__(16) uint32_t smem[];
    const uint64_t dst = dst0 + blockIdx.x / SPLIT;
    prand_dev::mt19937_skipahead_cta<NT, NOUT>(smem, op, st_src + (dst - src_back) * NW, st_dst + dst * NW,
                                               (int)(blockIdx.x % SPLIT) * NOUT);
}

// Latency form of the same application (a handful of destination streams: the first levels of a doubling tree,
// where a level lasts as long as ONE application and 140 SMs idle).  An application is cut into 39 CTAs of 16
// output words; every CTA extends the window itself (88 rounds of 227 words, 4.5 us) and thread (word j, slice s)
// of its 256 threads XORs the words selected by the polynomial words s, s + 16, ...: 39 coefficient words per
// thread, every coefficient visited branch-free (a bit scan was latency-bound: 58 us), then the 16 slices of a
// word are folded through shared memory.  src != dst only.
constexpr int AW_OUT = 16, AW_SL = 16, AW_THREADS = AW_OUT * AW_SL, AW_PARTS = NW / AW_OUT;

__global__ void __launch_bounds__(AW_THREADS)
mt19937_apply_wide_kernel(const uint32_t *st_src, uint32_t *st_dst, uint64_t dst0, uint64_t src_back,
                          const MtOp *__restrict__ op)
{
    extern __shared__ __align__(16) uint32_t smem[];
    uint32_t *x = smem;                                    // APPLY_XWORDS, then AW_SL * AW_OUT partial sums
    uint32_t *red = smem + APPLY_XWORDS + 3;
    const int tid = threadIdx.x;
    const uint64_t dst = dst0 + blockIdx.x / AW_PARTS;
    const int out0 = (int)(blockIdx.x % AW_PARTS) * AW_OUT;
    const uint32_t *src = st_src + (dst - src_back) * NW;
    for (int j = tid; j < NW; j += AW_THREADS) x[j] = src[j];
    __syncthreads();
    for (int r0 = 0; r0 < DEG; r0 += NW - MW) {
        const int k = r0 + tid;
        if (tid < NW - MW && k < DEG) x[NW + k] = mt_recur(x[k], x[k + 1], x[k + MW]);
        __syncthreads();
    }
    const int j = tid % AW_OUT, sl = tid / AW_OUT;
    const uint32_t *xo = x + out0 + j;
    // no bit scan, no branch: every coefficient is visited, its word loaded at a compile-time offset and masked
    // (a load and two logic operations per coefficient, all independent: the loop runs at issue rate)
    uint32_t acc0 = 0, acc1 = 0;
#pragma unroll 1
    for (int wi = sl; wi < NW; wi += AW_SL) {
        const uint32_t pw = __ldg(&op->w[wi]);
        const uint32_t *xw = xo + 32 * wi;
#pragma unroll
        for (int b = 0; b < 32; b += 2) {
            acc0 ^= xw[b] & (uint32_t)((int32_t)(pw << (31 - b)) >> 31);
            acc1 ^= xw[b + 1] & (uint32_t)((int32_t)(pw << (30 - b)) >> 31);
        }
    }
    red[sl * AW_OUT + j] = acc0 ^ acc1;
    __syncthreads();
    if (tid < AW_OUT) {
        uint32_t a = 0;
#pragma unroll
        for (int q = 0; q < AW_SL; q++) a ^= red[q * AW_OUT + tid];
        const int w = out0 + tid;
        st_dst[dst * NW + w] = w == 0 ? (a & 0x80000000u) : a;   // only the top bit of word 0 is state (T2)
    }
}
constexpr size_t AW_SMEM = (size_t)(APPLY_XWORDS + 3 + AW_SL * AW_OUT) * sizeof(uint32_t);

// Throughput form of the same application (many destination streams).  Thread t accumulates the four
// consecutive output words 4t .. 4t+3.  For the 32 coefficients of one polynomial word pw (positions
// 32 wi + b) they read x[32 wi + 4t + b + c], c < 4: a window of 35 consecutive words, loaded as nine
// aligned 16-byte shared loads into registers; bit b of pw (the same for all threads) then predicates
// four register XORs.  36 words loaded per 64 XORs on average instead of one load per XOR.
constexpr int APPLYW_THREADS = 160;                         // 156 active in the accumulation

// NSL > 1: the coefficient words are dealt to NSL slices of 160 threads whose partial sums are folded through
// shared memory -- the same work in 1 / NSL of the time for launches of a few hundred applications, where a
// level of the tree lasts as long as one CTA (NSL = 4: one CTA per SM, NSL = 2: two).
template <int NSL>
__global__ void __launch_bounds__(APPLYW_THREADS * NSL)
mt19937_apply_win_kernel(const uint32_t *st_src, uint32_t *st_dst, uint64_t dst0,
                         uint64_t src_back, const MtOp *__restrict__ op)
{
    constexpr int NT = APPLYW_THREADS * NSL;
    constexpr int EXT = NT < NW - MW ? NT : NW - MW;       // at most 227 new words are independent
    static_assert((NW / 2) % NSL == 0, "the slices take whole pairs of coefficient words");
    extern __shared__ __align__(16) uint32_t smem[];
    uint32_t *x = smem;                                    // APPLY_XWORDS + APPLY_ZPAD, then [NSL][624] partial sums
    uint32_t *red = smem + (APPLY_XWORDS + APPLY_ZPAD + 3) / 4 * 4;
    const int tid = threadIdx.x;
    const uint64_t dst = dst0 + blockIdx.x;
    const uint32_t *src = st_src + (dst - src_back) * NW;
    for (int j = tid; j < NW; j += NT) x[j] = src[j];
    for (int j = tid; j < APPLY_ZPAD; j += NT) x[APPLY_ZERO + j] = 0;
    __syncthreads();
    for (int r0 = 0; r0 < DEG; r0 += EXT) {
        int k = r0 + tid;
        if (tid < EXT && k < DEG) x[NW + k] = mt_recur(x[k], x[k + 1], x[k + MW]);
        __syncthreads();
    }
    const int q = tid / APPLYW_THREADS, t = tid % APPLYW_THREADS;
    const bool accum = t < NW / 4;
    uint32_t r[4] = {0u, 0u, 0u, 0u};
    if (accum) {
        uint32_t acc[4][4] = {};                           // four interleaved sets: independent XOR chains
        const uint4 *xw = reinterpret_cast<const uint4 *>(x) + t;     // window of wi starts at xw[8 wi]
        // two register windows in ping-pong: the nine loads of the next polynomial word are issued before
        // the 128 predicated XORs of the current one
        uint4 wa[9], wb[9];
        auto load_win = [&](uint4 (&w)[9], int wi) {
#pragma unroll
            for (int m = 0; m < 9; m++) w[m] = xw[8 * wi + m];
        };
        auto accumulate = [&](const uint4 (&w)[9], uint32_t pw) {
            uint32_t v[36];
#pragma unroll
            for (int m = 0; m < 9; m++) { v[4 * m] = w[m].x; v[4 * m + 1] = w[m].y; v[4 * m + 2] = w[m].z; v[4 * m + 3] = w[m].w; }
#pragma unroll
            for (int b = 0; b < 32; b++) {
                if (pw & (1u << b)) {
                    acc[b & 3][0] ^= v[b]; acc[b & 3][1] ^= v[b + 1]; acc[b & 3][2] ^= v[b + 2]; acc[b & 3][3] ^= v[b + 3];
                }
            }
        };
        constexpr int STEP = 2 * NSL;                      // slice q takes the word pairs 2q, 2q + 2 NSL, ...
        load_win(wa, 2 * q);
        uint32_t pw0 = __ldg(&op->w[2 * q]), pw1 = __ldg(&op->w[2 * q + 1]);
#pragma unroll 1
        for (int wi = 2 * q; wi < NW; wi += STEP) {
            load_win(wb, wi + 1);
            const uint32_t p0 = pw0, p1 = pw1;
            if (wi + STEP < NW) { pw0 = __ldg(&op->w[wi + STEP]); pw1 = __ldg(&op->w[wi + STEP + 1]); }
            accumulate(wa, p0);
            load_win(wa, wi + STEP < NW ? wi + STEP : wi);
            accumulate(wb, p1);
        }
#pragma unroll
        for (int c = 0; c < 4; c++) r[c] = acc[0][c] ^ acc[1][c] ^ acc[2][c] ^ acc[3][c];
    }
    if (NSL > 1) {
        if (accum) *reinterpret_cast<uint4 *>(red + q * NW + 4 * t) = make_uint4(r[0], r[1], r[2], r[3]);
        __syncthreads();
        if (q != 0 || !accum) return;
#pragma unroll
        for (int o = 1; o < NSL; o++) {
            const uint4 v = *reinterpret_cast<const uint4 *>(red + o * NW + 4 * t);
            r[0] ^= v.x; r[1] ^= v.y; r[2] ^= v.z; r[3] ^= v.w;
        }
    } else if (!accum) return;
    uint32_t *d = st_dst + dst * NW + 4 * t;
    *reinterpret_cast<uint4 *>(d) = make_uint4(t == 0 ? (r[0] & 0x80000000u) : r[0], r[1], r[2], r[3]);
}
template <int NSL> constexpr size_t applyw_smem() { return ((APPLY_XWORDS + APPLY_ZPAD + 3) / 4 * 4 + (NSL > 1 ? NSL * NW : 0)) * sizeof(uint32_t); }

// Many destination streams, second form: FOUR streams per CTA share the control flow.  The coefficient word
// is the same for every thread and every stream, so its bits are consumed two at a time through warp-uniform
// branches -- nothing is issued for a zero pair, one XOR per output word for a single bit and one three-input
// XOR for a set pair: 0.75 LOP3 per pair and output word on average instead of the 2 predicated ones above, and
// the branch instructions are shared by the 16 output words (4 streams x 4 words) of a thread.  Four extended
// sequences of 82 KB do not fit a CTA, so x is not tabulated: each stream keeps a ring of 1024 words that
// holds x_{32 wi} .. x_{32 wi + 655}, the part the 156 threads' windows touch at coefficient word wi, and the
// next 32 words of every stream are generated (by 128 of the threads, recurrence of PAPER.md:374) while word wi
// is accumulated; one CTA barrier per coefficient word.
constexpr int AM_S = 4, AM_THREADS = 160, AM_RING = 1024, AM_WB = 8;

// PARAM: the polynomial travels as a kernel argument (2496 bytes of the constant bank): its words, the pair
// codes and the branch conditions then live on the uniform datapath and cost the ALU pipe nothing.
template <bool PARAM>
__global__ void __launch_bounds__(AM_THREADS, 4)
mt19937_apply_multi_kernel(const uint32_t *st_src, uint32_t *st_dst, uint64_t dst0, uint64_t count,
                           uint64_t src_back, const MtOp *__restrict__ op, const __grid_constant__ MtOp opv)
{
    __shared__ __align__(16) uint32_t ring[AM_S][AM_RING];
    const int tid = threadIdx.x;
    const uint64_t d0 = dst0 + (uint64_t)blockIdx.x * AM_S;
    const int n_live = (int)(dst0 + count - d0 < (uint64_t)AM_S ? dst0 + count - d0 : AM_S);
    for (int i = tid; i < AM_S * NW; i += AM_THREADS) {
        const int q = i / NW, j = i % NW;
        ring[q][j] = st_src[(d0 + (q < n_live ? q : 0) - src_back) * NW + j];
    }
    __syncthreads();
    // thread g = (stream gq, lane gj) of the generator group extends every ring by 32 words per step
    const int gq = tid >> 5, gj = tid & 31;
    auto generate = [&](int k0) {                          // x_{k0 + 624 + gj} from x_{k0 + gj}, +1, +397
        if (tid < 32 * AM_S) {
            const int k = k0 + gj;
            ring[gq][(k + NW) & (AM_RING - 1)] =
                mt_recur(ring[gq][k & (AM_RING - 1)], ring[gq][(k + 1) & (AM_RING - 1)], ring[gq][(k + MW) & (AM_RING - 1)]);
        }
    };
    generate(0);                                           // x_624 .. x_655
    __syncthreads();
    const bool accum = tid < NW / 4;
    uint32_t acc[AM_S][4] = {};
    // The window of a piece (AM_WB = 8 coefficients: words 4 tid + h .. + 11 of each stream) slides by 8 words from
    // one piece to the next, so 4 of its 12 words are the last 4 of the previous piece's: the windows are a ring of
    // four 4-word groups per stream and a piece loads only TWO new groups (two 16-byte shared loads per stream
    // instead of three) -- shared-memory bandwidth is what bounds this kernel (ncu: L1TEX 88 %, ALU pipe 62 %).
    // Two pieces are unrolled so that the groups rotate by renaming: piece A uses groups (0, 1, 2), piece B (2, 3, 0).
    uint32_t G[AM_S][4][4];
    auto load_group = [&](int g, int pos) {                // group g <- words pos .. pos + 3 (pos = 0 mod 4)
#pragma unroll
        for (int q = 0; q < AM_S; q++) {
            const uint4 t = *reinterpret_cast<const uint4 *>(&ring[q][pos & (AM_RING - 1)]);
            G[q][g][0] = t.x; G[q][g][1] = t.y; G[q][g][2] = t.z; G[q][g][3] = t.w;
        }
    };
    auto piece = [&](uint32_t ph, int g0, int g1, int g2) {   // window word i = group (g0, g1, g2)[i / 4], word i % 4
        auto W = [&](int q, int i) -> uint32_t { return G[q][i < 4 ? g0 : i < 8 ? g1 : g2][i & 3]; };
#pragma unroll
        for (int b = 0; b < AM_WB; b += 2) {
            const bool lo = ph & (1u << b), hi = ph & (2u << b);     // warp-uniform
            if (lo) {
                if (hi) {
#pragma unroll
                    for (int q = 0; q < AM_S; q++)
#pragma unroll
                        for (int o = 0; o < 4; o++) acc[q][o] = xor3(acc[q][o], W(q, b + o), W(q, b + 1 + o));
                } else {
#pragma unroll
                    for (int q = 0; q < AM_S; q++)
#pragma unroll
                        for (int o = 0; o < 4; o++) acc[q][o] ^= W(q, b + o);
                }
            } else if (hi) {
#pragma unroll
                for (int q = 0; q < AM_S; q++)
#pragma unroll
                    for (int o = 0; o < 4; o++) acc[q][o] ^= W(q, b + 1 + o);
            }
        }
    };
    if (accum) load_group(0, 4 * tid);                     // the first piece's first group
    uint32_t pw = PARAM ? 0u : __ldg(&op->w[0]);
#pragma unroll 1
    for (int wi = 0; wi < NW; wi++) {
        const uint32_t p = PARAM ? opv.w[wi] : pw;
        if (!PARAM && wi + 1 < NW) pw = __ldg(&op->w[wi + 1]);
        generate(32 * wi + 32);                            // x_{32 wi + 656} .. : the words step wi + 1 adds to the windows
        if (accum) {
            // the word's 32 coefficients in four pieces of AM_WB (the code of two pieces is executed twice per word
            // instead of being unrolled further)
#pragma unroll 1
            for (int h = 0; h < 32; h += 2 * AM_WB) {
                const int pos = 32 * wi + h + 4 * tid;
                load_group(1, pos + 4);
                load_group(2, pos + 8);
                piece(p >> h, 0, 1, 2);
                load_group(3, pos + 12);
                load_group(0, pos + 16);                   // (the last one of a word is the next word's first group)
                piece(p >> (h + AM_WB), 2, 3, 0);
            }
        }
        __syncthreads();
    }
    if (accum) {
#pragma unroll
        for (int q = 0; q < AM_S; q++)
            if (q < n_live)
                *reinterpret_cast<uint4 *>(st_dst + (d0 + q) * NW + 4 * tid) =
                    make_uint4(tid == 0 ? (acc[q][0] & 0x80000000u) : acc[q][0], acc[q][1], acc[q][2], acc[q][3]);
    }
}

// ---- generation ----------------------------------------------------------------------------------
// CTA = S adjacent streams x T word slices (thread = (slice t, stream ls), ls fastest).  Thread
// (t, ls) owns the K = 624/T words w = T j + t, j = 0..K-1, of stream ls and keeps them in registers.
// One *round* regenerates the whole window (624 new numbers per stream): word w of the new window is
//     x'_w = x_{w+397} ^ twist(x_w, x_{w+1})            for w < 227  (all inputs from the old window)
//     x'_w = x'_{w-227} ^ twist(x_w, x_{w+1})           for w >= 227 (x_{w+1} = x'_0 for w = 623)
// so any 227 consecutive words are independent of each other (the 227 of PAPER.md:400, Table 5):
// M waves of T words (T M <= 227) run between two CTA barriers, every thread is busy in every wave.
// The neighbour words come from shared memory, which holds the old and the new window
// ([2][S][P] words, P = 624 + pad chosen so that both the generation pattern -- a warp reads 32/S
// consecutive words of S streams -- and the coalesced state load/store pattern are bank-conflict
// free).  A warp's store covers 32/S rows x S adjacent streams: full 32-byte sectors for S = 8.
// With few streams (C3: 512) S = 4 keeps 128 CTAs busy; the two CTAs that share a 32-byte sector form
// a cluster and meet at a cluster barrier once per round so that L2 merges their half-sector writes.
template <int S> struct MtPitch { static constexpr int value = 624 + 16 + (32 / S) % 32; };   // = 32/S mod 32, multiple of 4
template <> struct MtPitch<1> { static constexpr int value = 640; };

// Arithmetic of one number, arranged for the B200 pipes.  The ALU pipe (LOP3, SHF:
// 64 lanes/clk/SM) is the binding one, so everything that is not a logic operation runs on the
// FMA-heavy pipe: with rot = rotr(y, 1) the twist is
//     (y >> 1) ^ (y odd ? 0x9908B0DF : 0) = rot ^ (y odd ? 0x1908B0DF : 0)
// (the rotation already puts y's low bit into bit 31), and the second term is
// mul.hi(x1 << 31, 2 * 0x1908B0DF): IMAD.SHL + IMAD.HI.  Right shifts of the tempering can run as
// mul.hi by 2^(32-r) (HI bit 1: >> 11, bit 2: >> 18).  The multipliers are kernel arguments so that
// ptxas cannot turn them back into shifts or selects.  Per number: 3 + 4 LOP3/SHF, 1 address add.
struct MtMul { uint32_t a2, m31, m21, m14; };

__device__ __forceinline__ uint32_t lop3_e4(uint32_t a, uint32_t b, uint32_t c)   // (a & c) | (b & ~c)
{
    uint32_t d;
    asm("lop3.b32 %0, %1, %2, %3, 0xE4;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}

template <int HI, int BIT> __device__ __forceinline__ uint32_t mt_shr(uint32_t x, int r, uint32_t mul)
{
    return ((HI >> BIT) & 1) ? __umulhi(x, mul) : (x >> r);
}

template <int HI> __device__ __forceinline__ uint32_t mt_recur2(uint32_t x0, uint32_t x1, uint32_t xm, const MtMul &c)
{
    const uint32_t y = lop3_e4(x0, x1, 0x80000000u);
    const uint32_t rot = __funnelshift_r(y, y, 1);
    const uint32_t h = __umulhi(x1 * c.m31, c.a2);
    return xor3(xm, rot, h);
}
template <int HI> __device__ __forceinline__ uint32_t mt_temper2(uint32_t y, const MtMul &c)
{
    y ^= mt_shr<HI, 1>(y, 11, c.m21);
    y ^= (y << 7) & 0x9D2C5680u;
    y ^= (y << 15) & 0xEFC60000u;
    y ^= mt_shr<HI, 2>(y, 18, c.m14);
    return y;
}

__device__ __forceinline__ void cluster_arrive()
{
    asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory");
}
__device__ __forceinline__ void cluster_wait()
{
    asm volatile("barrier.cluster.wait.aligned;" ::: "memory");
}

// One round (FULL) or the first `rem` words of one (the tail of a call).  ob = this thread's byte
// offset (row t, stream s) from the uniform row-block pointer `rows`.
// In full rounds the tempering and the global store of a number are deferred until the shared loads
// of the thread's next number have been issued: after a barrier every warp of the CTA waits for
// shared memory at the same time, and the deferred work (half of a number's instructions, with no
// consumer) is what fills that wait.  pend / pend_p carry the deferred number across barriers and
// rounds; FIRST marks the call's first round, whose first step has nothing pending.
template <int S, int T, int M, int DT, int HI, bool FULL, bool ALL, bool FIRST>
__device__ __forceinline__ void mt_round(uint32_t *smem, const uint32_t ia, const uint32_t ib, const int t,
                                         uint32_t (&r)[NW / T], char *rows, const uint32_t ob,
                                         const uint64_t wave_bytes, const bool live, const int rem,
                                         const MtMul &c, uint32_t &pend, typename OutElem<DT>::type *&pend_p)
{
    typedef typename OutElem<DT>::type E;
    constexpr int K = NW / T;
#pragma unroll
    for (int j = 0; j < K; j++) {
        const int w = T * j + t;
        if (FULL || w < rem) {
            const uint32_t x1 = smem[ia + T * j + 1];
            uint32_t xm;
            if (T * (j + 1) <= NW - MW) xm = smem[ia + T * j + MW];
            else if (T * j >= NW - MW) xm = smem[ib + T * j - (NW - MW)];
            else xm = smem[(w < NW - MW ? ia + MW : ib - (NW - MW)) + T * j];
            if (FULL && !(FIRST && j == 0)) {
                const E v = convert<DT>(mt_temper2<HI>(pend, c));
                if (ALL || live) store1(pend_p, v);
            }
            const uint32_t nw = mt_recur2<HI>(r[j], x1, xm, c);
            r[j] = nw;
            smem[ib + T * j] = nw;
            if (j == 0 && t == 0) smem[ia + NW] = nw;       // x_{w+1} of word 623 is the new word 0
            E *q = reinterpret_cast<E *>(rows + j * wave_bytes + ob);
            if (FULL) {
                pend = nw;
                pend_p = q;
            } else {
                const E v = convert<DT>(mt_temper2<HI>(nw, c));
                if (ALL || live) store1(q, v);
            }
        }
        if ((j + 1) % M == 0) __syncthreads();
    }
}

template <int S, int T, int M, int DT, int HI, bool PAIR>
__global__ void __launch_bounds__(S * T)
mt19937_gen_kernel(const uint32_t *st_in, uint32_t *st_out,
                   typename OutElem<DT>::type *__restrict__ out, uint64_t ns, uint64_t n, const MtMul c)
{
    typedef typename OutElem<DT>::type E;
    constexpr int K = NW / T, P = MtPitch<S>::value, NT = S * T;
    static_assert(NW % T == 0 && K % M == 0 && T * M <= NW - MW, "bad MT19937 tiling");
    static_assert(P % 4 == 0 && P > NW, "bad pitch");
    extern __shared__ __align__(16) uint32_t smem[];     // [2][S][P]
    const int tid = threadIdx.x, ls = tid % S, t = tid / S;
    const uint64_t s0 = (uint64_t)blockIdx.x * S;
    const uint64_t s = s0 + ls;
    const bool live = s < ns;
    const int n_live = s0 >= ns ? 0 : (ns - s0 < (uint64_t)S ? (int)(ns - s0) : S);

    // state load: the CTA's S windows are one contiguous piece of st_in
    for (int i = tid; i < S * (NW / 4); i += NT) {
        const int q = i / (NW / 4), w4 = i % (NW / 4);
        if (q < n_live) {
            const uint4 v = __ldg(reinterpret_cast<const uint4 *>(st_in + (s0 + q) * NW) + w4);
            *reinterpret_cast<uint4 *>(smem + q * P + 4 * w4) = v;
        }
    }
    __syncthreads();
    uint32_t ia = ls * P + t, ib = ia + S * P;
    uint32_t r[K];
#pragma unroll
    for (int j = 0; j < K; j++) r[j] = smem[ia + T * j];
    // the launcher guarantees (T * ns + S) * sizeof(E) < 2^32
    const uint32_t ob = (uint32_t)(((uint64_t)t * ns + ls) * sizeof(E));
    char *rows = reinterpret_cast<char *>(out + s0);
    const uint64_t wave_bytes = (uint64_t)T * ns * sizeof(E);
    const uint64_t round_bytes = (uint64_t)NW * ns * sizeof(E);
    uint64_t left = n;
    uint32_t cur = 0;                                     // buffer that holds the old window
    bool pending = false;
    uint32_t pend = 0;
    E *pend_p = nullptr;
#define PRAND_MT_ROUNDS(ALLV, LIVEV)                                                                         \
    if (left >= NW) {                                                                                        \
        mt_round<S, T, M, DT, HI, true, ALLV, true>(smem, ia, ib, t, r, rows, ob, wave_bytes, LIVEV, NW, c,  \
                                                    pend, pend_p);                                           \
        for (;;) {                                                                                           \
            if (PAIR) {                                   /* stay within one round of the sector partner */ \
                if (pending) cluster_wait();                                                                 \
                cluster_arrive();                                                                            \
                pending = true;                                                                              \
            }                                                                                                \
            const uint32_t tmp = ia; ia = ib; ib = tmp;                                                      \
            cur ^= 1;                                                                                        \
            rows += round_bytes;                                                                             \
            left -= NW;                                                                                      \
            if (left < NW) break;                                                                            \
            mt_round<S, T, M, DT, HI, true, ALLV, false>(smem, ia, ib, t, r, rows, ob, wave_bytes, LIVEV,    \
                                                         NW, c, pend, pend_p);                               \
        }                                                                                                    \
        if (ALLV || LIVEV) store1(pend_p, convert<DT>(mt_temper2<HI>(pend, c)));                             \
    }
    if (n_live == S) {
        PRAND_MT_ROUNDS(true, true)
    } else {
        PRAND_MT_ROUNDS(false, live)
    }
#undef PRAND_MT_ROUNDS
    if (PAIR && pending) cluster_wait();
    const int rem = (int)left;
    if (rem) mt_round<S, T, M, DT, HI, false, false, false>(smem, ia, ib, t, r, rows, ob, wave_bytes, live, rem, c, pend, pend_p);
    // final window x_{P+n}..x_{P+n+623}: words [rem, 624) of the old buffer, then [0, rem) of the new
    const uint32_t *a0 = smem + cur * (S * P), *b0 = smem + (cur ^ 1) * (S * P);
    for (int i = tid; i < S * NW; i += NT) {
        const int q = i / NW, j = i % NW;
        if (q < n_live) {
            const int p = j + rem;
            st_out[(s0 + q) * NW + j] = p < NW ? a0[q * P + p] : b0[q * P + p - NW];
        }
    }
}

template <int S, int T, int M, int DT, int HI, bool PAIR> cudaError_t launch_gen(cudaStream_t stream, const GenArgs &a)
{
    typedef typename OutElem<DT>::type E;
    auto kern = mt19937_gen_kernel<S, T, M, DT, HI, PAIR>;
    const size_t smem = (size_t)2 * S * MtPitch<S>::value * sizeof(uint32_t);
    // per launch, not once per process: the attribute belongs to the current device's context
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    uint64_t blocks = ceil_div_u64(a.n_streams, S);
    if (PAIR) blocks += blocks & 1;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)blocks);
    cfg.blockDim = dim3(S * T);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = PAIR ? 2 : 1;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    const MtMul c = {2u * 0x1908B0DFu, 1u << 31, 1u << 21, 1u << 14};
    return cudaLaunchKernelEx(&cfg, kern, (const uint32_t *)a.st_in, (uint32_t *)a.st_out, (E *)a.out,
                              a.n_streams, a.n, c);
}

template <int S, int T, int M, int HI, bool PAIR> cudaError_t dispatch_dt(cudaStream_t stream, const GenArgs &a)
{
    switch (a.dtype) {
    case DT_U32: return launch_gen<S, T, M, DT_U32, HI, PAIR>(stream, a);
    case DT_F32: return launch_gen<S, T, M, DT_F32, HI, PAIR>(stream, a);
    default: return launch_gen<S, T, M, DT_F64, HI, PAIR>(stream, a);
    }
}

// ---- generation, few streams: rows leave through TMA tensor stores ------------------------------------
// Same CTA = S streams x T word slices and the same rounds as above, but a number is not stored to global
// memory by its thread: a CTA that writes 16-byte pieces of a row (S = 4, four-byte outputs) is bound by the
// SM's store path -- measured on C3's geometry (128 CTAs, 2048-byte rows, profiles/r02_store_pieces.md):
// STG 2.0 TB/s, TMA tensor stores of [rows x 16 bytes] boxes 3.3 TB/s.  The tempered number goes to a
// shared-memory tile [M T rows][S streams] instead (tile index = thread index: conflict-free), and once the
// CTA barrier that the recurrence needs anyway has passed, one thread sends the tile with a single
// cp.async.bulk.tensor.2d store (box = S elements x M T rows).  Tiles: two rounds' worth (2 K/M buffers);
// the issuing thread waits (wait_group.read) until the store that last used the next buffer has read it.
__device__ __forceinline__ void tma_store_2d(const CUtensorMap *tm, uint32_t src, int x, int y)
{
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%1, %2}], [%3];"
                 :: "l"(tm), "r"(x), "r"(y), "r"(src) : "memory");
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
}

template <int S, int T, int M, int DT, int HI, bool PAIR>
__global__ void __launch_bounds__(S * T)
mt19937_tgen_kernel(const uint32_t *st_in, uint32_t *st_out, typename OutElem<DT>::type *__restrict__ out,
                    uint64_t ns, uint64_t n, const MtMul c, const __grid_constant__ CUtensorMap tmap)
{
    typedef typename OutElem<DT>::type E;
    constexpr int K = NW / T, P = MtPitch<S>::value, NT = S * T, NG = K / M, TILE = M * NT;
    constexpr int W32 = (int)(sizeof(E) / 4);             // 32-bit words per element (the tensor map counts words)
    static_assert(NW % T == 0 && K % M == 0 && T * M <= NW - MW && M * T <= 256, "bad MT19937 tiling");
    static_assert((2 * S * P * 4) % 128 == 0 && (TILE * sizeof(E)) % 128 == 0, "tiles must be 128-byte aligned");
    extern __shared__ __align__(128) uint32_t smem[];     // windows [2][S][P], tiles [2 NG][TILE] of E
    E *tiles = reinterpret_cast<E *>(smem + 2 * S * P);
    const int tid = threadIdx.x, ls = tid % S, t = tid / S;
    const uint64_t s0 = (uint64_t)blockIdx.x * S;
    const uint64_t s = s0 + ls;
    const bool live = s < ns;
    const int n_live = s0 >= ns ? 0 : (ns - s0 < (uint64_t)S ? (int)(ns - s0) : S);
    const bool issuer = tid == 0 && n_live > 0;

    for (int i = tid; i < S * (NW / 4); i += NT) {
        const int q = i / (NW / 4), w4 = i % (NW / 4);
        if (q < n_live) {
            const uint4 v = __ldg(reinterpret_cast<const uint4 *>(st_in + (s0 + q) * NW) + w4);
            *reinterpret_cast<uint4 *>(smem + q * P + 4 * w4) = v;
        }
    }
    __syncthreads();
    uint32_t ia = ls * P + t, ib = ia + S * P;
    uint32_t r[K];
#pragma unroll
    for (int j = 0; j < K; j++) r[j] = smem[ia + T * j];
    const uint32_t tile_s = (uint32_t)__cvta_generic_to_shared(tiles);
    uint32_t ta = 0, tb = NG * TILE;                      // element offsets of this round's / the other round's tiles
    const int x = (int)(s0 * W32);
    const uint32_t rounds = (uint32_t)(n / NW);           // the launcher keeps n below 2^31
    const int rem = (int)(n % NW);
    uint32_t pend = 0;
    bool pending = false;
    int y = 0;                                            // first row of the round
    for (uint32_t rd = 0; rd < rounds; rd++) {
#pragma unroll
        for (int j = 0; j < K; j++) {
            const uint32_t x1 = smem[ia + T * j + 1];
            uint32_t xm;
            if (T * (j + 1) <= NW - MW) xm = smem[ia + T * j + MW];
            else if (T * j >= NW - MW) xm = smem[ib + T * j - (NW - MW)];
            else xm = smem[(T * j + t < NW - MW ? ia + MW : ib - (NW - MW)) + T * j];
            // the previous wave's number: tempering and tile store fill the wait for this wave's operands
            if (j != 0 || rd != 0) {
                const int q = (j + K - 1) % K;
                tiles[(j == 0 ? tb : ta) + (q / M) * TILE + (q % M) * NT + tid] = convert<DT>(mt_temper2<HI>(pend, c));
            }
            const uint32_t nw = mt_recur2<HI>(r[j], x1, xm, c);
            r[j] = nw;
            smem[ib + T * j] = nw;
            if (j == 0 && t == 0) smem[ia + NW] = nw;       // x_{w+1} of word 623 is the new word 0
            pend = nw;
            if ((j + 1) % M == 0) {
                const int gg = j / M;
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // tile writes -> visible to the TMA engine
                if (issuer) asm volatile("cp.async.bulk.wait_group.read %0;" :: "n"(2 * NG - 3) : "memory");
                __syncthreads();
                // the tile of the previous group is complete
                if (issuer && (gg != 0 || rd != 0)) {
                    const int pg = (gg + NG - 1) % NG;
                    tma_store_2d(&tmap, tile_s + (uint32_t)(((gg == 0 ? tb : ta) + pg * TILE) * sizeof(E)), x,
                                 y + (gg == 0 ? -NW : 0) + pg * M * T);
                }
            }
        }
        if (PAIR) {                                       // stay within one round of the sector partner
            if (pending) cluster_wait();
            cluster_arrive();
            pending = true;
        }
        { const uint32_t tmp = ia; ia = ib; ib = tmp; }
        { const uint32_t tmp = ta; ta = tb; tb = tmp; }
        y += NW;
    }
    if (rounds) {                                         // the last wave's number and the last tile
        tiles[tb + (NG - 1) * TILE + ((K - 1) % M) * NT + tid] = convert<DT>(mt_temper2<HI>(pend, c));
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads();
        if (issuer) tma_store_2d(&tmap, tile_s + (uint32_t)((tb + (NG - 1) * TILE) * sizeof(E)), x, y - NW + (NG - 1) * M * T);
    }
    if (PAIR && pending) cluster_wait();
    // ragged tail (< 624 rows): straight to global memory
    if (rem) {
        const uint32_t ob = (uint32_t)(((uint64_t)t * ns + ls) * sizeof(E));
        char *rows = reinterpret_cast<char *>(out + s0) + (uint64_t)rounds * NW * ns * sizeof(E);
        E *pend_p = nullptr;
        mt_round<S, T, M, DT, HI, false, false, false>(smem, ia, ib, t, r, rows, ob, (uint64_t)T * ns * sizeof(E), live,
                                                       rem, c, pend, pend_p);
    }
    // final window x_{P+n}..x_{P+n+623}: words [rem, 624) of the old buffer, then [0, rem) of the new
    const uint32_t cur = rounds & 1;
    const uint32_t *a0 = smem + cur * (S * P), *b0 = smem + (cur ^ 1) * (S * P);
    for (int i = tid; i < S * NW; i += NT) {
        const int q = i / NW, j = i % NW;
        if (q < n_live) {
            const int p = j + rem;
            st_out[(s0 + q) * NW + j] = p < NW ? a0[q * P + p] : b0[q * P + p - NW];
        }
    }
    if (issuer) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");     // the tiles outlive the stores' reads
}

typedef CUresult (*TensorMapEncodeFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                      const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                      CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// cuTensorMapEncodeTiled through the runtime (libprand does not link libcuda); nullptr if the driver has none
TensorMapEncodeFn tensor_map_encoder()
{
    static TensorMapEncodeFn fn = [] {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
            q != cudaDriverEntryPointSuccess)
            p = nullptr;
        return (TensorMapEncodeFn)p;
    }();
    return fn;
}

// the TMA path needs 16-byte aligned rows of at most 2^31 - 1 and at least one full round
bool tgen_ok(const GenArgs &a)
{
    return a.n_streams % 4 == 0 && (uintptr_t)a.out % 16 == 0 && a.n >= NW && a.n < (1ull << 31) && tensor_map_encoder();
}

template <int S, int T, int M, int DT, int HI, bool PAIR> cudaError_t launch_tgen(cudaStream_t stream, const GenArgs &a)
{
    typedef typename OutElem<DT>::type E;
    auto kern = mt19937_tgen_kernel<S, T, M, DT, HI, PAIR>;
    constexpr int K = NW / T, NG = K / M;
    const size_t smem = (size_t)2 * S * MtPitch<S>::value * sizeof(uint32_t) + (size_t)2 * NG * M * S * T * sizeof(E);
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    // the output as a 2-D tensor of 32-bit words: [rows of full rounds][n_streams * words per element]
    const uint32_t w32 = (uint32_t)(sizeof(E) / 4);
    CUtensorMap tm;
    const cuuint64_t dims[2] = {a.n_streams * w32, (a.n / NW) * NW};
    const cuuint64_t strides[1] = {a.n_streams * sizeof(E)};
    const cuuint32_t box[2] = {S * w32, (cuuint32_t)(M * T)};
    const cuuint32_t es[2] = {1, 1};
    if (tensor_map_encoder()(&tm, CU_TENSOR_MAP_DATA_TYPE_UINT32, 2, a.out, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                             CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return cudaErrorInvalidValue;
    uint64_t blocks = ceil_div_u64(a.n_streams, S);
    if (PAIR) blocks += blocks & 1;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)blocks);
    cfg.blockDim = dim3(S * T);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = PAIR ? 2 : 1;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    const MtMul c = {2u * 0x1908B0DFu, 1u << 31, 1u << 21, 1u << 14};
    return cudaLaunchKernelEx(&cfg, kern, (const uint32_t *)a.st_in, (uint32_t *)a.st_out, (E *)a.out, a.n_streams, a.n, c, tm);
}

template <int S, int T, int M, int HI, bool PAIR> cudaError_t dispatch_tdt(cudaStream_t stream, const GenArgs &a)
{
    switch (a.dtype) {
    case DT_U32: return launch_tgen<S, T, M, DT_U32, HI, PAIR>(stream, a);
    case DT_F32: return launch_tgen<S, T, M, DT_F32, HI, PAIR>(stream, a);
    default: return launch_tgen<S, T, M, DT_F64, HI, PAIR>(stream, a);
    }
}

// ---- generation, many streams: lane = stream, one CTA per 32 streams --------------------------------
// With thousands of streams a CTA can own 32 whole streams.  A window is a circular buffer in shared
// memory regenerated *in place*: cell c always holds the latest x_n with n = c (mod 624), so x_{n+397}
// is cell (c + 397) mod 624 whether it belongs to the old or the new window.  One round = three
// intervals of 208 consecutive words (at most 227, see above); the CTA's 8 warps take the 8 slices of
// an interval, warp u the 26 consecutive words base + 26 u ... of its 32 streams (lane = stream): x_w
// of step i+1 is x_{w+1} of step i (a register), so a number costs two shared loads and one shared
// store at compile-time offsets, each one conflict-free wavefront (pitch 625 is odd), and a warp
// store is one full 128-byte line of a row: 4 L1 wavefronts per 32 numbers (the S = 8 kernels above
// need 7, which is what bounds them).  Warps meet at a CTA barrier between intervals; inside one a
// thread runs 2 x 13 independent recurrences.  80 KB of shared memory per CTA, two CTAs per SM.
constexpr int WCH = 13;                                   // steps per chunk (operands staged in registers)

// 13 consecutive steps of one slice.  a = cell of the first word, am = a + (397 or -227) for the
// lanes' x_{w+397} cell; LAST: the chunk ends the slice, whose last x_{w+1} is the saved xb.
template <int DT, int HI, bool GUARD, bool ALL, bool LAST>
__device__ __forceinline__ void mt_chunk(uint32_t *a, const uint32_t *am, const uint32_t *am2, const int k2,
                                         uint32_t &x0, const uint32_t xb, typename OutElem<DT>::type *&p,
                                         const uint64_t ns, const bool live, const int left, const MtMul &c)
{
    typedef typename OutElem<DT>::type E;
    // all operands first (none of these cells is written during the chunk before it is read), so that
    // the 26 shared loads overlap and the 13 recurrences are independent instruction streams
    uint32_t x[WCH + 1], xm[WCH];
    x[0] = x0;
#pragma unroll
    for (int k = 0; k < WCH; k++) {
        x[k + 1] = (LAST && k == WCH - 1) ? xb : a[k + 1];
        xm[k] = (k >= k2 ? am2 : am)[k];
    }
#pragma unroll
    for (int k = 0; k < WCH; k++) xm[k] = mt_recur2<HI>(x[k], x[k + 1], xm[k], c);
#pragma unroll
    for (int k = 0; k < WCH; k++)
        if (!GUARD || k < left) a[k] = xm[k];
#pragma unroll
    for (int k = 0; k < WCH; k++) {
        const E v = convert<DT>(mt_temper2<HI>(xm[k], c));
        if ((!GUARD || k < left) && (ALL || live)) store1(p, v);
        p += ns;
    }
    x0 = x[WCH];
}

// One interval: words [BASE + 39 u, BASE + 39 u + 39) for slice u.  GUARD: only words < rem are real (tail).
template <bool CTA> __device__ __forceinline__ void mt_sync()
{
    if (CTA) __syncthreads(); else __syncwarp();
}

template <int BASE, int WB, int NSL, bool CTA, int DT, int HI, bool GUARD, bool ALL>
__device__ __forceinline__ void mt_interval(uint32_t *A, const int u, typename OutElem<DT>::type *rowp,
                                            const uint64_t ns, const bool live, const int rem, const MtMul &c)
{
    typedef typename OutElem<DT>::type E;
    static_assert(WB % WCH == 0 && NSL * WB <= NW - MW && BASE + NSL * WB <= NW, "bad interval");
    constexpr int NCH = WB / WCH, SW = NW - MW;           // x_{w+397} wraps to cell w - 227 from w = 227 on
    const int w0 = BASE + WB * u;
    // x_{w+1} of the slice's last word belongs to the next slice: read it before that slice overwrites it
    const int wb = w0 + WB;
    const uint32_t xb = A[wb == NW ? 0 : wb];
    mt_sync<CTA>();
    E *p = rowp + (uint64_t)w0 * ns;
    asm("" : "+l"(p));                                    // one running pointer, not rowp + two offsets
    uint32_t *a = A + w0;
    uint32_t x0 = a[0];
    // Only the interval that contains word 227 needs per-lane offsets, and only one slice of it switches
    // inside its words: offsets are per-lane registers, the switch position is a compile-time step of
    // the last chunk (u1 = the slice that contains word 227, k1 = its step within the last chunk).
    constexpr bool STRADDLE = BASE < SW && BASE + NSL * WB > SW;
    constexpr int u1 = STRADDLE ? (SW - BASE) / WB : 0, i1 = STRADDLE ? (SW - BASE) % WB : 0;
    static_assert(!STRADDLE || i1 >= (NCH - 1) * WCH, "the switch must fall into the slice's last chunk");
    const uint32_t *am, *am2;
    int k2 = WCH;
    if (!STRADDLE) {
        am = am2 = a + (BASE < SW ? MW : -SW);
    } else {
        am = a + (u <= u1 ? MW : -SW);
        am2 = a + (u < u1 ? MW : -SW);
        k2 = i1 - (NCH - 1) * WCH;
    }
    int left = rem - w0;
#pragma unroll 1
    for (int ch = 0; ch < NCH - 1; ch++) {
        mt_chunk<DT, HI, GUARD, ALL, false>(a, am, am, WCH, x0, xb, p, ns, live, left, c);
        a += WCH; am += WCH; am2 += WCH; left -= WCH;
    }
    mt_chunk<DT, HI, GUARD, ALL, true>(a, am, am2, k2, x0, xb, p, ns, live, left, c);
    mt_sync<CTA>();
}

constexpr int BP = 625;                                   // window pitch (odd: lane = stream is conflict-free)
constexpr int BW = 8;                                     // warps per CTA = slices per interval
constexpr int BSL = 26;                                   // words per slice per interval

template <int DT, int HI, bool GUARD, bool ALL>
__device__ __forceinline__ void mt_bround(uint32_t *A, const int u, typename OutElem<DT>::type *rowp,
                                          const uint64_t ns, const bool live, const int rem, const MtMul &c)
{
    mt_interval<0, BSL, BW, true, DT, HI, GUARD, ALL>(A, u, rowp, ns, live, rem, c);
    mt_interval<208, BSL, BW, true, DT, HI, GUARD, ALL>(A, u, rowp, ns, live, rem, c);
    mt_interval<416, BSL, BW, true, DT, HI, GUARD, ALL>(A, u, rowp, ns, live, rem, c);
}

template <int DT, int HI>
__global__ void __launch_bounds__(BW * 32, 2)
mt19937_bgen_kernel(const uint32_t *st_in, uint32_t *st_out,
                    typename OutElem<DT>::type *__restrict__ out, uint64_t ns, uint64_t n, const MtMul c)
{
    typedef typename OutElem<DT>::type E;
    extern __shared__ __align__(16) uint32_t smem[];     // [32][BP]
    const int lane = threadIdx.x & 31, u = threadIdx.x >> 5;
    const uint64_t s0 = (uint64_t)blockIdx.x * 32;
    const int n_live = ns - s0 < 32 ? (int)(ns - s0) : 32;
    const bool live = lane < n_live;
    {
        const uint32_t smem_s = (uint32_t)__cvta_generic_to_shared(smem);
        for (int q = u; q < n_live; q += BW) {             // warp u loads windows u, u + 8, ...
            const uint32_t *src = st_in + (s0 + q) * NW;
#pragma unroll 5
            for (int k = 0; k < 20; k++) {
                const int j = k * 32 + lane;
                if (j < NW)
                    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::
                                 "r"(smem_s + (uint32_t)(q * BP + j) * 4u), "l"(src + j));
            }
        }
        asm volatile("cp.async.commit_group;\n\tcp.async.wait_group 0;" ::: "memory");
    }
    __syncthreads();
    uint32_t *A = smem + lane * BP;
    E *rowp = out + s0 + lane;
    uint64_t left = n;
    if (n_live == 32) {
        for (; left >= NW; left -= NW, rowp += (uint64_t)NW * ns)
            mt_bround<DT, HI, false, true>(A, u, rowp, ns, true, NW, c);
    } else {
        for (; left >= NW; left -= NW, rowp += (uint64_t)NW * ns)
            mt_bround<DT, HI, false, false>(A, u, rowp, ns, live, NW, c);
    }
    const int rem = (int)left;
    if (rem) mt_bround<DT, HI, true, false>(A, u, rowp, ns, live, rem, c);
    __syncthreads();
    for (int q = u; q < n_live; q += BW) {
        uint32_t *dst = st_out + (s0 + q) * NW;
#pragma unroll 4
        for (int k = 0; k < 20; k++) {
            const int j = k * 32 + lane;
            if (j < NW) {
                int p = j + rem;
                if (p >= NW) p -= NW;
                dst[j] = smem[q * BP + p];
            }
        }
    }
}

template <int DT, int HI> cudaError_t launch_bgen(cudaStream_t stream, const GenArgs &a)
{
    typedef typename OutElem<DT>::type E;
    auto kern = mt19937_bgen_kernel<DT, HI>;
    const size_t smem = (size_t)32 * BP * sizeof(uint32_t);
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);   // per device
    if (e != cudaSuccess) return e;
    const uint64_t blocks = ceil_div_u64(a.n_streams, 32);
    const MtMul c = {2u * 0x1908B0DFu, 1u << 31, 1u << 21, 1u << 14};
    kern<<<(unsigned)blocks, BW * 32, smem, stream>>>((const uint32_t *)a.st_in, (uint32_t *)a.st_out, (E *)a.out,
                                                      a.n_streams, a.n, c);
    return cudaGetLastError();
}

template <int HI> cudaError_t dispatch_bdt(cudaStream_t stream, const GenArgs &a)
{
    switch (a.dtype) {
    case DT_U32: return launch_bgen<DT_U32, HI>(stream, a);
    case DT_F32: return launch_bgen<DT_F32, HI>(stream, a);
    default: return launch_bgen<DT_F64, HI>(stream, a);
    }
}

// ---- generation, few streams: output gathered across a cluster of 4 CTAs ----------------------------
// With a few hundred streams (C3: 512) a CTA can hold only ~4 of them, and a CTA that writes 16-byte
// pieces of a row is bound by the SM's store path: measured 7.4 B/clk/SM for 16-byte pieces against
// 17 B/clk/SM for 32-byte and ~21 B/clk/SM for 64-byte and longer ones (the request rate, about one
// per two clocks, is what limits; TMA tensor stores of such narrow boxes are slower still).  So the
// four CTAs of a cluster (16 adjacent streams) exchange their outputs through distributed shared
// memory: CTA r computes the full recurrence of its own 4 streams, as above, but CTA d writes rows
// [156 d, 156 d + 156) of every round (624 rows) for all 16 streams, i.e. 64-byte pieces, as 128-bit
// stores.  Thread = (stream, word slice) with the stream index slowest: the threads of one stream meet
// at their own named barrier, so the four streams of a CTA drift apart and fill each other's waits.
//
// Exchange: a round's numbers go to a local staging tile (one column per (destination, stream), 156
// rows); a helper warp sends the 16 columns with bulk asynchronous copies (cp.async.bulk shared::cta ->
// shared::cluster) that signal the destination's mbarrier by transaction bytes -- no release fence (a
// cluster-scope fence is a MEMBAR.ALL.GPU, ~800 clocks per round when tried), no spinning on the data
// path.  NB = 4 tile buffers, read-out LAG = 2 rounds behind: every wait has a full round of slack.
//   full[b]   (count 1 + tx)  destination: all 16 columns of a tile have landed
//   empty[b]  (count 4)       source: all four destinations have written tile b out (its staging and
//                             gather buffers may be reused)
//   prod[b] / cons[b] (count 28) local: the compute warps have staged / read tile b
constexpr int CG_CS = 4, CG_S = 4;
constexpr int CG_T = 208;                                 // words per wave (three waves per round)
constexpr int CG_U = CG_T / 2;                            // a thread owns two adjacent words of a wave: 104 threads per stream
constexpr int CG_GT = 128;                                // threads per group = one stream (104) rounded up to whole warps
constexpr int CG_GROUPS = CG_S;
constexpr int CG_COLS = CG_CS * CG_S;                     // streams per cluster
constexpr int CG_ROWS = NW / CG_CS;                       // rows of a round written by one CTA
constexpr int CG_CP = 192;                                // column pitch in words (768 B: a bulk copy)
constexpr int CG_ROT = 2;                                 // column c starts CG_ROT * c words into its slot: conflict-free read-out
constexpr int CG_NB = 4, CG_LAG = 2;
constexpr int CG_P = 628;                                 // window pitch
constexpr int CG_TILE = CG_COLS * CG_CP;                  // words per tile buffer
constexpr int CG_CT = CG_GROUPS * CG_GT;                  // compute threads (448)
constexpr int CG_WARPS = CG_CT / 32;                      // compute warps (14); the next warp is the helper
constexpr int CG_THREADS = CG_CT + 32;
constexpr int CG_PIECES = CG_ROWS * (CG_COLS / 4);        // 16-byte pieces of a gathered tile (624)
constexpr uint32_t CG_TILE_BYTES = CG_TILE * 4;
constexpr size_t CG_SMEM = (size_t)(2 * CG_S * CG_P + 2 * CG_NB * CG_TILE) * sizeof(uint32_t) + 4 * CG_NB * 8;
static_assert(NW % CG_CS == 0 && CG_ROWS % 2 == 0 && CG_ROWS + CG_ROT * (CG_COLS - 1) <= CG_CP && CG_T * 3 == NW, "bad cluster tiling");
static_assert(CG_LAG < CG_NB && (CG_NB & (CG_NB - 1)) == 0 && CG_CP % 4 == 0 && CG_P % 2 == 0 && CG_ROT % 2 == 0, "bad pipeline");

__device__ __forceinline__ uint32_t smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t map_to_cta(uint32_t addr, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
    return r;
}
__device__ __forceinline__ void mbar_init(uint32_t a, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(a), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t a, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(a), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t a)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(a) : "memory");
}
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_addr)
{
    asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" :: "r"(cluster_addr) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t a, uint32_t parity)
{
    asm volatile("{\n\t.reg .pred p;\n\tWAIT_%=:\n\t"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t@!p bra WAIT_%=;\n\t}"
                 :: "r"(a), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_copy_to_cta(uint32_t dst_cluster, uint32_t src, uint32_t bytes, uint32_t mbar_cluster)
{
    asm volatile("cp.async.bulk.shared::cluster.shared::cta.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(dst_cluster), "r"(src), "r"(bytes), "r"(mbar_cluster) : "memory");
}
__device__ __forceinline__ void cluster_sync_all()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ void group_barrier(int g)
{
    // compile-time barrier numbers: a register operand would reserve all 16 hardware barriers for the CTA
    switch (g) {
    case 0: asm volatile("bar.sync 1, %0;" :: "n"(CG_GT) : "memory"); break;
    case 1: asm volatile("bar.sync 2, %0;" :: "n"(CG_GT) : "memory"); break;
    case 2: asm volatile("bar.sync 3, %0;" :: "n"(CG_GT) : "memory"); break;
    default: asm volatile("bar.sync 4, %0;" :: "n"(CG_GT) : "memory"); break;
    }
}
template <int DT> __device__ __forceinline__ uint32_t out_bits(uint32_t u)
{
    if constexpr (DT == DT_F32) return __float_as_uint(u32_to_f32(u));
    else return u;
}

// One wave for one thread: words w = 208 J + 2u and w + 1 of its stream.  x_w, x_{w+1} are registers,
// x_{w+2} and the two x_{w+397} (old window) resp. new x_{w-227} come from shared memory.  The cell after
// the old window's last word holds the new word 0 (written in wave 0), so a pair never needs a special
// case: for w <= 226 both operands are old[w + 397 ..] (old[624] = new[0]), else new[w - 227 ..].
template <int J>
__device__ __forceinline__ void cg_operands(const uint32_t *smem, const uint32_t ia, const uint32_t ib, const int u,
                                            uint32_t &x2, uint32_t &m0, uint32_t &m1)
{
    x2 = smem[ia + CG_T * J + 2];
    if (CG_T * (J + 1) <= NW - MW) { m0 = smem[ia + CG_T * J + MW]; m1 = smem[ia + CG_T * J + MW + 1]; }
    else if (CG_T * J > NW - MW) { m0 = smem[ib + CG_T * J - (NW - MW)]; m1 = smem[ib + CG_T * J - (NW - MW) + 1]; }
    else {
        const uint32_t q = (CG_T * J + 2 * u <= NW - MW - 1 ? ia + MW : ib - (NW - MW)) + CG_T * J;
        m0 = smem[q]; m1 = smem[q + 1];
    }
}
// The two recurrences of a wave from their operands; (p0, p1) receive the new words.
template <int J>
__device__ __forceinline__ void cg_step(uint32_t *smem, const uint32_t ia, const uint32_t ib, const int u, uint32_t (&r)[6],
                                        const MtMul &c, const uint32_t x2, const uint32_t m0, const uint32_t m1,
                                        uint32_t &p0, uint32_t &p1)
{
    const uint32_t n0 = mt_recur2<0>(r[2 * J], r[2 * J + 1], m0, c);
    const uint32_t n1 = mt_recur2<0>(r[2 * J + 1], x2, m1, c);
    r[2 * J] = n0;
    r[2 * J + 1] = n1;
    *reinterpret_cast<uint2 *>(smem + ib + CG_T * J) = make_uint2(n0, n1);
    if (J == 0 && u == 0) smem[ia + NW] = n0;
    p0 = n0;
    p1 = n1;
}
// Full wave.  (p0, p1) carry the previous wave's two new words, whose tempering and staging store (slot
// pend_slot of tile sb) run here, after this wave's loads have been issued, if `pending`.
template <int J, int DT>
__device__ __forceinline__ void cg_wave(uint32_t *smem, const uint32_t ia, const uint32_t ib, const int u,
                                        uint32_t (&r)[6], const MtMul &c, uint32_t &p0, uint32_t &p1, uint32_t *sb,
                                        const uint32_t pend_slot, const bool pending)
{
    uint32_t x2, m0, m1;
    cg_operands<J>(smem, ia, ib, u, x2, m0, m1);
    if (pending)
        *reinterpret_cast<uint2 *>(sb + pend_slot) = make_uint2(out_bits<DT>(mt_temper2<0>(p0, c)), out_bits<DT>(mt_temper2<0>(p1, c)));
    cg_step<J>(smem, ia, ib, u, r, c, x2, m0, m1, p0, p1);
}
// Ragged tail: only words below `rem` are produced; (o0, o1) = the converted outputs.
template <int J, int DT>
__device__ __forceinline__ void cg_tail_wave(uint32_t *smem, const uint32_t ia, const uint32_t ib, const int u,
                                             uint32_t (&r)[6], const MtMul &c, uint32_t &o0, uint32_t &o1, const int rem)
{
    const int w = CG_T * J + 2 * u;
    if (w >= rem) return;
    uint32_t x2, m0, m1;
    cg_operands<J>(smem, ia, ib, u, x2, m0, m1);
    const uint32_t n0 = mt_recur2<0>(r[2 * J], r[2 * J + 1], m0, c);
    const uint32_t n1 = mt_recur2<0>(r[2 * J + 1], x2, m1, c);
    smem[ib + CG_T * J] = n0;
    if (w + 1 < rem) smem[ib + CG_T * J + 1] = n1;
    if (J == 0 && u == 0) smem[ia + NW] = n0;
    o0 = out_bits<DT>(mt_temper2<0>(n0, c));
    o1 = out_bits<DT>(mt_temper2<0>(n1, c));
}

template <int DT>
__global__ void __launch_bounds__(CG_THREADS)
mt19937_cgen_kernel(const uint32_t *st_in, uint32_t *st_out, uint32_t *__restrict__ out, uint64_t ns, uint64_t n,
                    const MtMul c)
{
    static_assert(DT == DT_U32 || DT == DT_F32, "4-byte outputs only");
    extern __shared__ __align__(128) uint32_t smem[];    // windows [2][S][P], staging [NB][COLS][CP], gather [NB][COLS][CP], mbarriers
    uint32_t *stage = smem + 2 * CG_S * CG_P;
    uint32_t *gat = stage + CG_NB * CG_TILE;
    const uint32_t bars = smem_addr(gat + CG_NB * CG_TILE);           // full, empty, prod, cons: [NB] each
    const uint32_t full = bars, empty = bars + 8 * CG_NB, prod = bars + 16 * CG_NB, cons = bars + 24 * CG_NB;
    const int tid = threadIdx.x, lane = tid & 31;
    const bool helper = tid >= CG_CT;
    const int g = helper ? 0 : tid / CG_GT, tg = tid % CG_GT;         // group = stream within the CTA, thread in group
    const bool act = !helper && tg < CG_U;
    const int ls = g, u = act ? tg : 0;                               // word pair
    uint32_t rank;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(rank));
    const uint64_t sc0 = (uint64_t)(blockIdx.x / CG_CS) * CG_COLS;       // first stream of the cluster
    const uint64_t s0 = sc0 + rank * CG_S;                                // first stream of this CTA
    const uint64_t s = s0 + ls;
    const bool live = s < ns;
    const int n_live = s0 >= ns ? 0 : (ns - s0 < (uint64_t)CG_S ? (int)(ns - s0) : CG_S);
    const uint32_t rounds = (uint32_t)(n / NW);           // the launcher keeps n / 624 below 2^32
    const int rem = (int)(n % NW);

    if (tid == 0) {
        for (int b = 0; b < CG_NB; b++) {
            mbar_init(full + 8 * b, 1);
            mbar_init(empty + 8 * b, CG_CS);
            mbar_init(prod + 8 * b, CG_WARPS);
            mbar_init(cons + 8 * b, CG_WARPS);
            if ((uint32_t)b < rounds) mbar_expect_tx(full + 8 * b, CG_TILE_BYTES);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int i = tid; i < CG_S * (NW / 4); i += CG_THREADS) {
        const int q = i / (NW / 4), w4 = i % (NW / 4);
        uint4 v = make_uint4(0u, 0u, 0u, 0u);
        if (q < n_live) v = __ldg(reinterpret_cast<const uint4 *>(st_in + (s0 + q) * NW) + w4);
        *reinterpret_cast<uint4 *>(smem + q * CG_P + 4 * w4) = v;
    }
    __syncthreads();
    cluster_sync_all();                                   // every CTA's barriers are initialised
    uint32_t ia = ls * CG_P + 2 * u, ib = ia + CG_S * CG_P;
    const uint32_t cur = rounds & 1;                      // window buffer that is "old" after the full rounds
    uint32_t r[6] = {0u, 0u, 0u, 0u, 0u, 0u};

    if (helper) {
        // ---- helper warp: forwards staged tiles, returns buffers -------------------------------------
        const uint32_t copy_dst = map_to_cta(smem_addr(gat + (rank * CG_S + (lane & 3)) * CG_CP), (uint32_t)(lane >> 2) & 3u);
        const uint32_t copy_bar = map_to_cta(full, (uint32_t)(lane >> 2) & 3u);
        const uint32_t copy_src = smem_addr(stage + (lane & 15) * CG_CP);
        const uint32_t free_bar = map_to_cta(empty, (uint32_t)lane & 3u);
        for (uint32_t rd = 0; rd < rounds + CG_LAG; rd++) {
            if (rd < rounds) {
                const uint32_t b = rd & (CG_NB - 1), ph = (rd / CG_NB) & 1u;
                mbar_wait(prod + 8 * b, ph);
                // column (destination lane / 4, own stream lane % 4) -> column (rank, stream) of that CTA's tile
                if (lane < CG_COLS)
                    bulk_copy_to_cta(copy_dst + b * CG_TILE_BYTES, copy_src + b * CG_TILE_BYTES, CG_CP * 4, copy_bar + 8 * b);
            }
            if (rd >= CG_LAG) {
                const uint32_t q = rd - CG_LAG;
                const uint32_t b = q & (CG_NB - 1), ph = (q / CG_NB) & 1u;
                mbar_wait(cons + 8 * b, ph);
                if (lane == 0 && q + CG_NB < rounds) mbar_expect_tx(full + 8 * b, CG_TILE_BYTES);
                __syncwarp();
                if (lane < CG_CS) mbar_arrive_cluster(free_bar + 8 * b);
            }
        }
    } else {
        // ---- compute warps --------------------------------------------------------------------------------
        if (act) {
#pragma unroll
            for (int j = 0; j < 3; j++) { r[2 * j] = smem[ia + CG_T * j]; r[2 * j + 1] = smem[ia + CG_T * j + 1]; }
        }
        // staging slots of this thread's words w = 208 j + 2u, w + 1: column (destination w / 156, own stream),
        // rows w % 156 and the next one (same destination: 156 is even)
        uint32_t so[3];
#pragma unroll
        for (int j = 0; j < 3; j++) {
            const int w = CG_T * j + 2 * u;
            so[j] = (uint32_t)(((w / CG_ROWS) * CG_S + ls) * CG_CP + CG_ROT * (rank * CG_S + ls) + w % CG_ROWS);
        }
        // read-out of a gathered tile: 156 rows x 16 streams as 624 pieces of 16 bytes, piece = (row, 4 streams);
        // thread tid takes pieces tid and tid + CG_CT (the shared-memory pattern is conflict-free: 8 rows x 4 column
        // groups per warp, column pitch = 2 mod 32)
        constexpr int RO = (CG_PIECES + CG_CT - 1) / CG_CT;
        uint32_t ro_src[RO];
        uint64_t ro_dst[RO];
        bool ro_on[RO];
#pragma unroll
        for (int k = 0; k < RO; k++) {
            const int i = tid + k * CG_CT, row = i >> 2, cq = i & 3;
            ro_on[k] = i < CG_PIECES && sc0 + 4 * cq < ns;
            ro_src[k] = (uint32_t)((4 * cq) * (CG_CP + CG_ROT) + row);
            ro_dst[k] = ((uint64_t)rank * CG_ROWS + row) * ns + sc0 + 4 * cq;
        }
        const uint64_t round_elems = (uint64_t)NW * ns;
        uint32_t *ro_out = out;                           // row 0 of the next round to be read out
        auto read_out = [&](uint32_t q) {
            const uint32_t b = q & (CG_NB - 1), ph = (q / CG_NB) & 1u;
            mbar_wait(full + 8 * b, ph);
            const uint32_t *gb = gat + b * CG_TILE;
#pragma unroll
            for (int k = 0; k < RO; k++) {
                if (ro_on[k]) {
                    const uint32_t *gp = gb + ro_src[k];
                    const uint4 v = make_uint4(gp[0], gp[CG_CP + CG_ROT], gp[2 * (CG_CP + CG_ROT)], gp[3 * (CG_CP + CG_ROT)]);
                    __stcs(reinterpret_cast<uint4 *>(ro_out + ro_dst[k]), v);
                }
            }
            ro_out += round_elems;
            __syncwarp();
            if (lane == 0) mbar_arrive(cons + 8 * b);
        };
        // The tempering and the staging store of a wave's two numbers are deferred until the next wave's shared
        // loads have been issued: after a barrier every warp of the group waits for shared memory at the same
        // time, and the deferred half of the work is what fills that wait.
        uint32_t p0 = 0, p1 = 0;
        for (uint32_t rd = 0; rd < rounds; rd++) {
            const uint32_t b = rd & (CG_NB - 1), ph = (rd / CG_NB) & 1u;
            if (rd >= CG_NB) mbar_wait(empty + 8 * b, ph ^ 1u);           // tile rd - NB has been written out everywhere
            uint32_t *sb = stage + b * CG_TILE;
            if (act) cg_wave<0, DT>(smem, ia, ib, u, r, c, p0, p1, sb, 0u, false);
            group_barrier(g);
            if (act) cg_wave<1, DT>(smem, ia, ib, u, r, c, p0, p1, sb, so[0], true);
            group_barrier(g);
            if (act) cg_wave<2, DT>(smem, ia, ib, u, r, c, p0, p1, sb, so[1], true);
            group_barrier(g);
            if (act) *reinterpret_cast<uint2 *>(sb + so[2]) = make_uint2(out_bits<DT>(mt_temper2<0>(p0, c)), out_bits<DT>(mt_temper2<0>(p1, c)));
            { const uint32_t tmp = ia; ia = ib; ib = tmp; }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");    // staged numbers -> visible to the bulk copy
            __syncwarp();
            if (lane == 0) mbar_arrive(prod + 8 * b);
            if (rd >= CG_LAG) read_out(rd - CG_LAG);
        }
        for (uint32_t q = rounds > CG_LAG ? rounds - CG_LAG : 0; q < rounds; q++) read_out(q);
    }
    // nobody leaves while a peer may still send it a tile or a signal
    cluster_sync_all();
    // ragged tail (< 624 rows): straight to global memory
    if (rem && !helper) {
        uint32_t *p = out + (uint64_t)rounds * NW * ns + s;
        uint32_t o0 = 0, o1 = 0;
#define PRAND_CG_TAIL(J)                                                                      \
        if (act) {                                                                            \
            const int w = CG_T * J + 2 * u;                                                   \
            cg_tail_wave<J, DT>(smem, ia, ib, u, r, c, o0, o1, rem);                         \
            if (live && w < rem) __stcs(p + (uint64_t)w * ns, o0);                            \
            if (live && w + 1 < rem) __stcs(p + (uint64_t)(w + 1) * ns, o1);                  \
        }                                                                                     \
        group_barrier(g);
        PRAND_CG_TAIL(0)
        PRAND_CG_TAIL(1)
        PRAND_CG_TAIL(2)
#undef PRAND_CG_TAIL
    }
    __syncthreads();
    // final window x_{P+n}..x_{P+n+623}: words [rem, 624) of the old buffer, then [0, rem) of the new
    const uint32_t *a0 = smem + cur * (CG_S * CG_P), *b0 = smem + (cur ^ 1) * (CG_S * CG_P);
    for (int i = tid; i < CG_S * NW; i += CG_THREADS) {
        const int q = i / NW, j = i % NW;
        if (q < n_live) {
            const int pp = j + rem;
            st_out[(s0 + q) * NW + j] = pp < NW ? a0[q * CG_P + pp] : b0[q * CG_P + pp - NW];
        }
    }
}

// ---- generation, few streams: warp = stream, window in registers, rows leave through TMA ----------------
// With a few hundred streams (C3: 512 = 4 per SM on 128 SMs) the slice kernels above are bound by their own
// instruction stream and by latency, not by any pipe: a wave of 208 words per stream is one shared-memory
// round trip, a dozen dependent instructions and a CTA barrier, every warp of the CTA waits for the same thing
// at the same time, and the per-wave bookkeeping costs more issue slots than the arithmetic (ncu: 1.09 ms on
// C3 even with the stores removed).  And a CTA that holds 4 streams writes 16-byte pieces, HALF sectors: L2
// merges the two halves of a sector only if they arrive within a few hundred clocks of each other (measured,
// profiles/r02_store_pieces.md: 128 CTAs storing [rows x 16 bytes] boxes by TMA take 0.65 ms in lock step,
// 1.28 ms when every second CTA runs 500 clocks late, 2.7 ms when the partners drift freely -- each lone half
// costs a DRAM read-modify-write), which ties sector partners into lock step.  Full sectors do not care (32-byte
// pieces: no change up to 10,000 clocks of skew).
//
// So: a WARP owns a stream and the recurrence shares nothing.  The window lives in registers, word i of the
// sequence in lane i mod 32 of ring slot (i / 32) mod 20 (640 words: the window and the 16 words that complete
// its last slot).  A step produces the 32 words of one slot, lane l from x_{i-624}, x_{i-623}, x_{i-227} --
// lanes l+16, l+17, l+29 (mod 32) of slots k / k+1 resp. k+12 / k+13: three selects and three shuffles, no
// shared memory, no barrier; the seven steps before a step are independent of it (227 > 7 * 32), which is the
// instruction-level parallelism a lone warp needs.  One turn of the ring (20 steps, 640 rows) is unrolled.
// A lone warp issues only every other clock (measured 2.1 clocks per instruction at best), so the work of a
// number is split over two warps on the same scheduler: the COMPUTE warp of a stream runs the recurrence alone
// (12 instructions per 32 numbers) and drops the raw words into staging columns; HELPER warps read the words of
// a row, temper and convert them and build the row's piece in a tile of their own, which the same warp sends
// with one TMA tensor store (bulk groups are per thread: a helper waits only for its own stores).
// Two CTAs (8 adjacent streams) form a cluster and trade halves: rows [0, 320) of every turn are written by CTA
// 0, rows [320, 640) by CTA 1, each for all 8 streams = full 32-byte sectors.  A compute warp writes the steps
// that belong to its own CTA with plain shared stores and the others straight into the partner's staging
// columns with st.async, which counts the bytes on the partner's "full" mbarrier (no fence, no flag); a buffer
// comes back through one "empty" mbarrier on which the helpers of both CTAs arrive (the partner's remotely).  Nothing on the compute warps' path
// waits for a TMA store or a proxy fence.  Rows outside whole turns of the ring (the first 16, the last < 640)
// take a plain warp-level path on a shared-memory copy of the ring.
constexpr int WG_S = 4;                                   // streams = compute warps = helper warps per CTA
constexpr int WG_COLS = 2 * WG_S;                         // streams per cluster
constexpr int WG_RING = 20;                               // ring slots (registers per lane)
constexpr int WG_XS = 32 * WG_RING;                       // 640 words = rows per turn
constexpr int WG_HALF = WG_XS / 2;                        // rows per CTA and turn
constexpr int WG_HSTEPS = WG_RING / 2;                    // steps per CTA and turn
constexpr int WG_BOX = WG_HALF / WG_S;                    // rows per helper and turn: one TMA box of 80 rows x 8 streams
constexpr int WG_CP = WG_HALF + 4;                        // staging column pitch: the two CTAs' columns 16 banks apart
constexpr int WG_NSB = 6;                                 // staging buffers (even: the compute warps wait for two at a time)
constexpr int WG_HW = 2 * WG_S;                           // helper warps: two per row block, taking turns
constexpr int WG_NTB = 2;                                 // tile buffers per helper
constexpr int WG_THREADS = 32 * (WG_S + WG_HW);
constexpr uint32_t WG_TX = WG_HSTEPS * 32 * 4;            // bytes one partner warp sends per turn
static_assert(WG_BOX % 16 == 0 && WG_BOX <= 256 && (WG_BOX * WG_COLS * 4) % 128 == 0 && (4 * WG_CP) % 32 == 16, "bad tile");

// A waiting warp shares its scheduler with the warp it waits for: it must not spin (ncu: a bare try_wait loop took
// 45 % of all issue slots), so it sleeps between polls.
__device__ __forceinline__ void mbar_wait_sleep(uint32_t a, uint32_t parity)
{
    for (;;) {
        uint32_t done;
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(a), "r"(parity) : "memory");
        if (done) break;
        __nanosleep(40);
    }
}
// two barriers at once: the polls are issued back to back, so their latencies overlap
__device__ __forceinline__ void mbar_wait_sleep2(uint32_t a0, uint32_t p0, uint32_t a1, uint32_t p1)
{
    for (;;) {
        uint32_t d0, d1;
        asm volatile("{\n\t.reg .pred p, q;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%2], %3;\n\t"
                     "mbarrier.try_wait.parity.shared::cta.b64 q, [%4], %5;\n\tselp.u32 %0, 1, 0, p;\n\tselp.u32 %1, 1, 0, q;\n\t}"
                     : "=r"(d0), "=r"(d1) : "r"(a0), "r"(p0), "r"(a1), "r"(p1) : "memory");
        if (d0 & d1) break;
        __nanosleep(40);
    }
}
__device__ __forceinline__ void st_async_u32(uint32_t dst_cluster, uint32_t v, uint32_t mbar_cluster)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b32 [%0], %1, [%2];"
                 :: "r"(dst_cluster), "r"(v), "r"(mbar_cluster) : "memory");
}

// rows [ra, rb) of one stream by its warp, ring in shared memory (word i of the call at xs[i mod 640])
template <int DT>
__device__ __forceinline__ void wg_slow_rows(uint32_t *xs, uint64_t ra, uint64_t rb, typename OutElem<DT>::type *col,
                                             uint64_t ns, int lane, const MtMul &c)
{
    uint32_t pos = (uint32_t)(ra % WG_XS);
    for (uint64_t r0 = ra; r0 < rb; r0 += 32) {
        const bool on = r0 + lane < rb;
        uint32_t a0 = pos + lane;
        a0 -= a0 >= WG_XS ? WG_XS : 0;
        uint32_t a1 = a0 + 1, am = a0 + MW, aw = a0 + NW;
        a1 -= a1 >= WG_XS ? WG_XS : 0;
        am -= am >= WG_XS ? WG_XS : 0;
        aw -= aw >= WG_XS ? WG_XS : 0;
        uint32_t nw = 0;
        if (on) nw = mt_recur2<0>(xs[a0], xs[a1], xs[am], c);
        __syncwarp();                                      // every operand read before any cell is rewritten
        if (on) {
            xs[aw] = nw;
            store1(col + (r0 + lane) * ns, convert<DT>(mt_temper2<0>(nw, c)));
        }
        __syncwarp();
        pos += 32;
        pos -= pos >= WG_XS ? WG_XS : 0;
    }
}

__device__ __forceinline__ void wg_store_piece(uint32_t *p, const uint32_t (&v)[4])
{
    *reinterpret_cast<uint4 *>(p) = make_uint4(v[0], v[1], v[2], v[3]);
}
__device__ __forceinline__ void wg_store_piece(float *p, const float (&v)[4])
{
    *reinterpret_cast<float4 *>(p) = make_float4(v[0], v[1], v[2], v[3]);
}
__device__ __forceinline__ void wg_store_piece(double *p, const double (&v)[4])
{
    *reinterpret_cast<double2 *>(p) = make_double2(v[0], v[1]);
    *reinterpret_cast<double2 *>(p + 2) = make_double2(v[2], v[3]);
}

// One turn of the ring for the compute warp of CTA RANK: the steps of the first half of the rows belong to CTA 0,
// the others to CTA 1; the words of the partner's steps go straight into its staging column (st.async).
template <int RANK, int HI>
__device__ __forceinline__ void wg_turn(uint32_t (&r)[WG_RING], uint32_t *sp, const uint32_t rp, const uint32_t rbar,
                                        const bool ge16, const bool ge17, const bool ge29, const int l17, const int l29,
                                        const MtMul &c)
{
#pragma unroll
    for (int k = 0; k < WG_RING; k++) {                    // k = ring slot of the step (compile-time after unrolling)
        const uint32_t v0 = ge16 ? r[k] : r[(k + 1) % WG_RING];
        const uint32_t v1 = ge17 ? r[k] : r[(k + 1) % WG_RING];
        const uint32_t vm = ge29 ? r[(k + 12) % WG_RING] : r[(k + 13) % WG_RING];
        const uint32_t x0 = __shfl_xor_sync(0xffffffffu, v0, 16);
        const uint32_t x1 = __shfl_sync(0xffffffffu, v1, l17);
        const uint32_t xm = __shfl_sync(0xffffffffu, vm, l29);
        const uint32_t nw = mt_recur2<HI>(x0, x1, xm, c);
        r[k] = nw;
        if (k / WG_HSTEPS == RANK) sp[32 * (k % WG_HSTEPS)] = nw;
        else st_async_u32(rp + 128u * (k % WG_HSTEPS), nw, rbar);
    }
}

template <int DT, int HI>
__global__ void __launch_bounds__(WG_THREADS, 1)
mt19937_wgen_kernel(const uint32_t *st_in, uint32_t *st_out, typename OutElem<DT>::type *__restrict__ out,
                    uint64_t ns, uint64_t n, const MtMul c, const __grid_constant__ CUtensorMap tmap)
{
    typedef typename OutElem<DT>::type E;
    constexpr int W32 = (int)(sizeof(E) / 4);
    constexpr int TILE = WG_BOX * WG_COLS;                // elements per helper tile
    constexpr int SBUF = WG_COLS * WG_CP;                 // words per staging buffer
    // tiles [helper][NTB][TILE] of E, staging [NSB][8 columns][CP], rings [stream][640],
    // mbarriers sfull[NSB], sempty[NSB]
    extern __shared__ __align__(128) uint32_t smem[];
    E *tiles = reinterpret_cast<E *>(smem);
    uint32_t *staging = smem + WG_HW * WG_NTB * TILE * W32;
    uint32_t *rings = staging + WG_NSB * SBUF;
    const uint32_t bars = smem_addr(rings + WG_S * WG_XS);
    const uint32_t sfull = bars, sempty = bars + 8 * WG_NSB;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    uint32_t rank;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(rank));
    const uint32_t peer = rank ^ 1u;
    const uint64_t sc0 = (uint64_t)(blockIdx.x / 2) * WG_COLS;           // first stream of the cluster
    const uint64_t s0 = sc0 + rank * WG_S;                                // first stream of this CTA
    if (threadIdx.x == 0) {
        for (int b = 0; b < WG_NSB; b++) {
            mbar_init(sfull + 8 * b, WG_S);
            mbar_init(sempty + 8 * b, 2 * WG_S);             // our four helper blocks and the partner's four
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    cluster_sync_all();                                   // both CTAs' barriers are initialised
    const uint32_t turns = n >= 16 ? (uint32_t)((n - 16) / WG_XS) : 0;   // whole turns of the ring after the first 16 rows

    if (warp >= WG_S) {
        // ---- helper warp h: rows [80 h, 80 h + 80) of this CTA's half of every turn, all eight streams -------
        // lane = (row, half): 16 rows per pass, the even lanes take the four streams of CTA 0, the odd ones CTA 1's
        // (helper warps h and h + 4 share the rows and alternate turns: three warps per scheduler keep it busy)
        const int h = (warp - WG_S) % WG_S, par = (warp - WG_S) / WG_S;
        E *my = tiles + (warp - WG_S) * WG_NTB * TILE;
        const uint32_t my_s = smem_addr(my);
        const uint32_t peer_sempty = map_to_cta(sempty, peer);
        const int x = (int)(sc0 * W32);
        const int y0 = 16 + WG_HALF * (int)rank + WG_BOX * h;
        const uint32_t *sp0 = staging + (lane & 1) * (WG_S * WG_CP) + h * WG_BOX + (lane >> 1);
        for (uint32_t u = par; u < turns; u += 2) {
            const uint32_t b = u % WG_NSB, tb = (u / 2) % WG_NTB;
            // (all lanes poll the barrier: no divergence to reconverge)
            mbar_wait_sleep(sfull + 8 * b, (u / WG_NSB) & 1u);
            // bulk groups belong to the thread that committed them: lane 0 issued the stores, so lane 0 waits until the
            // store that last used tile buffer tb has read it, and the warp barrier holds the other lanes' tile writes back
            if (u / 2 >= WG_NTB) {
                if (lane == 0) asm volatile("cp.async.bulk.wait_group.read %0;" :: "n"(WG_NTB - 1) : "memory");
                __syncwarp();
            }
            const uint32_t *sp = sp0 + b * SBUF;
            E *tp = my + tb * TILE + lane * 4;
#pragma unroll
            for (int i = 0; i < WG_BOX / 16; i++) {
                E v[4];
#pragma unroll
                for (int q = 0; q < 4; q++) v[q] = convert<DT>(mt_temper2<HI>(sp[q * WG_CP + 16 * i], c));
                wg_store_piece(tp + 16 * i * WG_COLS, v);
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // tile writes -> visible to the TMA engine
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(sempty + 8 * b);
                mbar_arrive_cluster(peer_sempty + 8 * b);
                tma_store_2d(&tmap, my_s + tb * (uint32_t)(TILE * sizeof(E)), x, y0 + WG_XS * (int)u);
            }
        }
        if (lane == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    } else {
        // ---- compute warp g: stream s0 + g ------------------------------------------------------------------
        const int g = warp;
        uint32_t *xs = rings + g * WG_XS;
        {
            const uint32_t *src = st_in + (s0 + g) * NW;
            for (int i = lane; i < NW; i += 32) xs[i] = __ldg(src + i);
        }
        __syncwarp();
        E *col = out + s0 + g;
        wg_slow_rows<DT>(xs, 0, n < 16 ? n : 16, col, ns, lane, c);
        if (turns) {
            uint32_t r[WG_RING];
#pragma unroll
            for (int q = 0; q < WG_RING; q++) r[q] = xs[32 * q + lane];
            const bool ge16 = lane >= 16, ge17 = lane >= 17, ge29 = lane >= 29;
            const int l17 = (lane + 17) & 31, l29 = (lane + 29) & 31;
            // this warp's staging column (rank, g): here and in the partner CTA
            uint32_t *lcol = staging + (rank * WG_S + g) * WG_CP + lane;
            const uint32_t rcol = map_to_cta(smem_addr(lcol), peer);
            const uint32_t rfull = map_to_cta(sfull, peer);
            for (uint32_t u = 0; u < turns; u++) {
                const uint32_t b = u % WG_NSB, ph = ((u / WG_NSB) - 1u) & 1u;
                // both staging columns of this turn must have been read out, here by our helpers and there by the partner's:
                // ONE barrier counts all eight (every mbarrier operation costs the compute warp ~100 clocks)
                if (u >= WG_NSB && (u & 1u) == 0) {         // this turn's buffer and the next one's
                    const uint32_t u1 = u + 1;
                    mbar_wait_sleep2(sempty + 8 * b, ph, sempty + 8 * (u1 % WG_NSB), ((u1 / WG_NSB) - 1u) & 1u);
                }
                if (rank == 0) wg_turn<0, HI>(r, lcol + b * SBUF, rcol + b * (uint32_t)(SBUF * 4), rfull + 8 * b, ge16, ge17, ge29, l17, l29, c);
                else wg_turn<1, HI>(r, lcol + b * SBUF, rcol + b * (uint32_t)(SBUF * 4), rfull + 8 * b, ge16, ge17, ge29, l17, l29, c);
                __syncwarp();
                if (lane == 0) mbar_expect_tx(sfull + 8 * b, WG_TX);
            }
#pragma unroll
            for (int q = 0; q < WG_RING; q++) xs[32 * q + lane] = r[q];
            __syncwarp();
        }
        wg_slow_rows<DT>(xs, n < 16 ? n : 16 + (uint64_t)turns * WG_XS, n, col, ns, lane, c);
        // the window after n numbers: words n .. n + 623 of the call
        uint32_t *dst = st_out + (s0 + g) * NW;
        uint32_t pos = (uint32_t)(n % WG_XS) + lane;
        for (int i = lane; i < NW; i += 32) {
            pos -= pos >= WG_XS ? WG_XS : 0;
            dst[i] = xs[pos];
            pos += 32;
        }
    }
    // nobody leaves while the partner may still send it words or signals
    cluster_sync_all();
}

// the cluster kernel needs whole clusters of 8 streams on top of the TMA conditions
bool wgen_ok(const GenArgs &a) { return a.n_streams % WG_COLS == 0 && tgen_ok(a); }

template <int DT, int HI> cudaError_t launch_wgen(cudaStream_t stream, const GenArgs &a)
{
    typedef typename OutElem<DT>::type E;
    auto kern = mt19937_wgen_kernel<DT, HI>;
    const size_t smem = (size_t)WG_HW * WG_NTB * WG_BOX * WG_COLS * sizeof(E) + (size_t)WG_NSB * WG_COLS * WG_CP * 4 +
                        (size_t)WG_S * WG_XS * 4 + 2 * WG_NSB * 8;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const uint32_t w32 = (uint32_t)(sizeof(E) / 4);
    CUtensorMap tm;
    const cuuint64_t dims[2] = {a.n_streams * w32, a.n};
    const cuuint64_t strides[1] = {a.n_streams * sizeof(E)};
    const cuuint32_t box[2] = {WG_COLS * w32, WG_BOX};
    const cuuint32_t es[2] = {1, 1};
    if (tensor_map_encoder()(&tm, CU_TENSOR_MAP_DATA_TYPE_UINT32, 2, a.out, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                             CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return cudaErrorInvalidValue;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(a.n_streams / WG_S));
    cfg.blockDim = dim3(WG_THREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    const MtMul c = {2u * 0x1908B0DFu, 1u << 31, 1u << 21, 1u << 14};
    return cudaLaunchKernelEx(&cfg, kern, (const uint32_t *)a.st_in, (uint32_t *)a.st_out, (E *)a.out, a.n_streams, a.n, c, tm);
}

template <int HI> cudaError_t dispatch_wdt(cudaStream_t stream, const GenArgs &a)
{
    switch (a.dtype) {
    case DT_U32: return launch_wgen<DT_U32, HI>(stream, a);
    case DT_F32: return launch_wgen<DT_F32, HI>(stream, a);
    default: return launch_wgen<DT_F64, HI>(stream, a);
    }
}

// ---- sections of a single sequence (prand_generate_seq_*; Table 5) ----------------------
// Section c = stream c of the family, its numbers contiguous in memory: out[c * sec_len + i].  With the
// per-stream thread groups of the kernel above (thread = two adjacent words of a wave, 104 threads per
// stream) a warp's store is 64 consecutive rows of ONE section: 256 (u32, f32) or 512 (f64) contiguous
// bytes straight from registers -- no exchange, no staging, no transposition.  Four sections per CTA,
// each group running at its own pace (named barriers); the last section of the array may be shorter
// and its final window, the state of the sequence after `length` numbers, goes to st_last.
template <int DT> __device__ __forceinline__ void sg_store2(typename OutElem<DT>::type *p, uint32_t a, uint32_t b)
{
    store2(p, convert<DT>(a), convert<DT>(b));
}

template <int DT>
__global__ void __launch_bounds__(CG_CT, 2)
mt19937_sgen_kernel(const uint32_t *st_in, uint32_t *st_last, typename OutElem<DT>::type *__restrict__ out,
                    uint64_t n_sections, uint64_t sec_len, uint64_t length, const MtMul c)
{
    typedef typename OutElem<DT>::type E;
    extern __shared__ __align__(16) uint32_t smem[];     // windows [2][S][P]
    const int tid = threadIdx.x;
    const int g = tid / CG_GT, tg = tid % CG_GT;
    const uint64_t sec0 = (uint64_t)blockIdx.x * CG_S, sec = sec0 + g;
    const bool live = sec < n_sections;
    const bool act = live && tg < CG_U;
    const int u = act ? tg : 0;
    const int n_live = sec0 >= n_sections ? 0 : (n_sections - sec0 < (uint64_t)CG_S ? (int)(n_sections - sec0) : CG_S);
    for (int i = tid; i < CG_S * (NW / 4); i += CG_CT) {
        const int q = i / (NW / 4), w4 = i % (NW / 4);
        if (q < n_live) {
            const uint4 v = __ldg(reinterpret_cast<const uint4 *>(st_in + (sec0 + q) * NW) + w4);
            *reinterpret_cast<uint4 *>(smem + q * CG_P + 4 * w4) = v;
        }
    }
    __syncthreads();
    const uint64_t last = n_sections - 1;
    const uint64_t rows = !live ? 0 : (sec == last ? length - last * sec_len : sec_len);
    const uint32_t rounds = (uint32_t)(rows / NW);
    const int rem = (int)(rows % NW);
    uint32_t ia = g * CG_P + 2 * u, ib = ia + CG_S * CG_P;
    uint32_t r[6] = {0u, 0u, 0u, 0u, 0u, 0u};
    if (act) {
#pragma unroll
        for (int j = 0; j < 3; j++) { r[2 * j] = smem[ia + CG_T * j]; r[2 * j + 1] = smem[ia + CG_T * j + 1]; }
    }
    E *p = out + sec * sec_len + 2 * u;
    // as in the cluster kernel the tempering and the store of a wave's two numbers are deferred until the next
    // wave's shared loads have been issued (they fill the wait after the barrier)
    uint32_t p0 = 0, p1 = 0;
    for (uint32_t rd = 0; rd < rounds; rd++, p += NW) {
        if (act) {
            uint32_t x2, m0, m1;
            cg_operands<0>(smem, ia, ib, u, x2, m0, m1);
            if (rd) sg_store2<DT>(p - NW + 2 * CG_T, mt_temper2<0>(p0, c), mt_temper2<0>(p1, c));
            cg_step<0>(smem, ia, ib, u, r, c, x2, m0, m1, p0, p1);
        }
        group_barrier(g);
        if (act) {
            uint32_t x2, m0, m1;
            cg_operands<1>(smem, ia, ib, u, x2, m0, m1);
            sg_store2<DT>(p, mt_temper2<0>(p0, c), mt_temper2<0>(p1, c));
            cg_step<1>(smem, ia, ib, u, r, c, x2, m0, m1, p0, p1);
        }
        group_barrier(g);
        if (act) {
            uint32_t x2, m0, m1;
            cg_operands<2>(smem, ia, ib, u, x2, m0, m1);
            sg_store2<DT>(p + CG_T, mt_temper2<0>(p0, c), mt_temper2<0>(p1, c));
            cg_step<2>(smem, ia, ib, u, r, c, x2, m0, m1, p0, p1);
        }
        group_barrier(g);
        { const uint32_t tmp = ia; ia = ib; ib = tmp; }
    }
    if (act && rounds) sg_store2<DT>(p - NW + 2 * CG_T, mt_temper2<0>(p0, c), mt_temper2<0>(p1, c));
    if (rem) {                                             // only the last section of the array is ragged
        uint32_t o0 = 0, o1 = 0;
#define PRAND_SG_TAIL(J)                                                                      \
        if (act) {                                                                            \
            const int w = CG_T * J + 2 * u;                                                   \
            cg_tail_wave<J, DT_U32>(smem, ia, ib, u, r, c, o0, o1, rem);                      \
            if (w < rem) store1(p + CG_T * J, convert<DT>(o0));                               \
            if (w + 1 < rem) store1(p + CG_T * J + 1, convert<DT>(o1));                       \
        }                                                                                     \
        group_barrier(g);
        PRAND_SG_TAIL(0)
        PRAND_SG_TAIL(1)
        PRAND_SG_TAIL(2)
#undef PRAND_SG_TAIL
    }
    // the sequence after `length` numbers: final window of the last section = words [rem, 624) of its old
    // buffer, then [0, rem) of the new one (written by that section's own group)
    if (live && sec == last) {
        const uint32_t cur = rounds & 1;
        const uint32_t *a0 = smem + cur * (CG_S * CG_P) + g * CG_P, *b0 = smem + (cur ^ 1) * (CG_S * CG_P) + g * CG_P;
        for (int j = tg; j < NW; j += CG_GT) {
            const int pp = j + rem;
            st_last[j] = pp < NW ? a0[pp] : b0[pp - NW];
        }
    }
}

template <int DT> cudaError_t launch_sgen(cudaStream_t stream, const void *st_in, void *st_last, void *out,
                                          uint64_t n_sections, uint64_t sec_len, uint64_t length)
{
    typedef typename OutElem<DT>::type E;
    auto kern = mt19937_sgen_kernel<DT>;
    const size_t smem = (size_t)2 * CG_S * CG_P * sizeof(uint32_t);
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const MtMul c = {2u * 0x1908B0DFu, 1u << 31, 1u << 21, 1u << 14};
    kern<<<(unsigned)ceil_div_u64(n_sections, CG_S), CG_CT, smem, stream>>>((const uint32_t *)st_in, (uint32_t *)st_last,
                                                                           (E *)out, n_sections, sec_len, length, c);
    return cudaGetLastError();
}

template <int DT> cudaError_t launch_cgen(cudaStream_t stream, const GenArgs &a)
{
    auto kern = mt19937_cgen_kernel<DT>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)CG_SMEM);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(ceil_div_u64(a.n_streams, CG_COLS) * CG_CS));
    cfg.blockDim = dim3(CG_THREADS);
    cfg.dynamicSmemBytes = CG_SMEM;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CG_CS;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    const MtMul c = {2u * 0x1908B0DFu, 1u << 31, 1u << 21, 1u << 14};
    return cudaLaunchKernelEx(&cfg, kern, (const uint32_t *)a.st_in, (uint32_t *)a.st_out, (uint32_t *)a.out,
                              a.n_streams, a.n, c);
}

}  // namespace

cudaError_t mt19937_apply(cudaStream_t stream, const uint32_t *st_src, uint32_t *st_dst, uint64_t dst0,
                          uint64_t count, uint64_t src_back, const MtOp *d_op, const MtOp *h_op, LaunchInfo *li)
{
    // the opt-in belongs to the current device's context: set it per call (a microsecond), not once per process
    cudaError_t e = cudaFuncSetAttribute(mt19937_apply_kernel<256, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)APPLY_SMEM);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(mt19937_apply_kernel<640, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)APPLY_SMEM);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(mt19937_apply_kernel<160, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)APPLY_SMEM);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(mt19937_apply_win_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)applyw_smem<1>());
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(mt19937_apply_win_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)applyw_smem<2>());
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(mt19937_apply_win_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)applyw_smem<4>());
    if (e != cudaSuccess) return e;
    li->kernel = "mt19937_apply";
    li->launches = 0;
    // grid.x is limited to 2^31-1 blocks; streams beyond that would not fit device memory anyway
    if (count == 0) return cudaSuccess;
    const uint64_t sms = (uint64_t)sm_count();
    const DebugHooks &hk = debug_hooks();
    auto win = [&](int nsl) {
        if (nsl == 4) mt19937_apply_win_kernel<4><<<(unsigned)count, 4 * APPLYW_THREADS, applyw_smem<4>(), stream>>>(st_src, st_dst, dst0, src_back, d_op);
        else if (nsl == 2) mt19937_apply_win_kernel<2><<<(unsigned)count, 2 * APPLYW_THREADS, applyw_smem<2>(), stream>>>(st_src, st_dst, dst0, src_back, d_op);
        else mt19937_apply_win_kernel<1><<<(unsigned)count, APPLYW_THREADS, applyw_smem<1>(), stream>>>(st_src, st_dst, dst0, src_back, d_op);
    };
    if (hk.mt_apply_list) {                                  // test hook: the position-list kernels
        if (src_back != 0 && 4 * count <= 2 * sms)
            mt19937_apply_kernel<160, 4><<<(unsigned)(4 * count), 160, APPLY_SMEM, stream>>>(st_src, st_dst, dst0, src_back, d_op);
        else if (count <= sms)
            mt19937_apply_kernel<640, 1><<<(unsigned)count, 640, APPLY_SMEM, stream>>>(st_src, st_dst, dst0, src_back, d_op);
        else
            mt19937_apply_kernel<256, 1><<<(unsigned)count, 256, APPLY_SMEM, stream>>>(st_src, st_dst, dst0, src_back, d_op);
    } else if (hk.mt_apply_win) {                            // test hook: a window kernel at any size
        win(hk.mt_apply_nsl);
    } else if (hk.mt_apply_nsl >= 0 && src_back != 0 && count * AW_PARTS <= 5 * sms) {
        // a handful of applications: the launch is as long as one application, spread each over 39 CTAs
        e = cudaFuncSetAttribute(mt19937_apply_wide_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)AW_SMEM);
        if (e != cudaSuccess) return e;
        mt19937_apply_wide_kernel<<<(unsigned)(count * AW_PARTS), AW_THREADS, AW_SMEM, stream>>>(st_src, st_dst, dst0, src_back, d_op);
    } else if (hk.mt_apply_nsl >= 0 && count <= 5 * sms) {
        // up to a few hundred applications a level lasts as long as a CTA: four slices per CTA (measured: 148
        // applications 0.137 ms against 0.203 ms with one slice, 0.162 ms for the position list and 0.65 ms for the
        // four-streams-per-CTA kernel; 592: 0.49 against 0.66 ms; 1024: 0.85 against 0.77 ms)
        win(4);
    } else if (h_op) {
        mt19937_apply_multi_kernel<true><<<(unsigned)ceil_div_u64(count, AM_S), AM_THREADS, 0, stream>>>(
            st_src, st_dst, dst0, count, src_back, d_op, *h_op);
    } else {
        static const MtOp none = {};
        mt19937_apply_multi_kernel<false><<<(unsigned)ceil_div_u64(count, AM_S), AM_THREADS, 0, stream>>>(
            st_src, st_dst, dst0, count, src_back, d_op, none);
    }
    li->launches = 1;
    return cudaGetLastError();
}

cudaError_t mt19937_seq(cudaStream_t stream, const void *st_in, void *st_last, void *out, int dtype, uint64_t n_sections,
                        uint64_t sec_len, uint64_t length, LaunchInfo *li)
{
    li->kernel = "mt19937_sgen<S=4>";
    li->launches = 1;
    switch (dtype) {
    case DT_U32: return launch_sgen<DT_U32>(stream, st_in, st_last, out, n_sections, sec_len, length);
    case DT_F32: return launch_sgen<DT_F32>(stream, st_in, st_last, out, n_sections, sec_len, length);
    default: return launch_sgen<DT_F64>(stream, st_in, st_last, out, n_sections, sec_len, length);
    }
}

cudaError_t mt19937_generate(cudaStream_t stream, const GenArgs &a, LaunchInfo *li)
{
    li->launches = 1;
    // a thread's byte offset inside a row block must fit 32 bits (wave of 208 rows, 8-byte elements);
    // prand_init refuses larger families (PRAND_MT19937_MAX_STREAMS, prand.h)
    if (a.n_streams > PRAND_MT19937_MAX_STREAMS) return cudaErrorInvalidValue;
    // Kernel choice by stream count (measured on B200): 32 streams per CTA need >= ~128
    // CTAs; below that 8 streams per CTA; below ~1000 streams the warp-per-stream cluster kernel if the rows are
    // long enough to amortise its start-up (whole clusters of 8 streams, 16-byte aligned rows), else 4 streams
    // per CTA in sector-sharing cluster pairs.
    int cfg = a.n_streams >= 4096 ? 0 : a.n_streams >= 1024 ? 1 : (a.n >= 65536 && wgen_ok(a)) ? 6 : 2;
    // 4-byte outputs, 16-byte aligned rows: the cluster-gather kernel writes 64-byte pieces
    const bool gather_ok = a.dtype != DT_F64 && a.n_streams % 4 == 0 && (uintptr_t)a.out % 16 == 0 && a.n / NW < (1ull << 32);
    // (not the default: measured 1.29 ms on C3 against 1.00 ms for the cluster-pair kernel -- the exchange is
    // bound by the ~10-13 B/clk/SM that distributed shared memory moves between four CTAs)
    if (debug_hooks().mt_cfg >= 0) {                                          // test hook: force a variant
        const int want = debug_hooks().mt_cfg;
        if ((want != 3 || gather_ok) && (want < 4 || tgen_ok(a)) && (want < 6 || wgen_ok(a))) cfg = want;
    }
    switch (cfg) {
    case 0: li->kernel = "mt19937_bgen<S=32>"; return dispatch_bdt<0>(stream, a);
    case 1: li->kernel = "mt19937_gen<S=8,T=104>"; return dispatch_dt<8, 104, 2, 0, false>(stream, a);
    case 3:
        li->kernel = "mt19937_cgen<CS=4>";
        return a.dtype == DT_U32 ? launch_cgen<DT_U32>(stream, a) : launch_cgen<DT_F32>(stream, a);
    case 6: {
        // (a tensor map the driver refuses is not an error of the call: the cluster-pair kernel takes over)
        li->kernel = "mt19937_wgen<CS=2>";
        const cudaError_t e = dispatch_wdt<0>(stream, a);
        if (e != cudaErrorInvalidValue || debug_hooks().mt_cfg >= 0) return e;
        (void)cudaGetLastError();
        li->kernel = "mt19937_gen<S=4,T=208,pair>";
        return dispatch_dt<4, 208, 1, 6, true>(stream, a);
    }
    case 4: li->kernel = "mt19937_tgen<S=4,T=208,pair>"; return dispatch_tdt<4, 208, 1, 6, true>(stream, a);
    case 5: li->kernel = "mt19937_tgen<S=8,T=104>"; return dispatch_tdt<8, 104, 2, 0, false>(stream, a);
    default: li->kernel = "mt19937_gen<S=4,T=208,pair>"; return dispatch_dt<4, 208, 1, 6, true>(stream, a);
    }
}

}  // namespace prand
